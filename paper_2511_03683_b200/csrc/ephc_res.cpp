// ephc_res.cpp -- host side of the resident-tile store (variant 3): once-stored directed entries, tile images that
// a CTA fetches with bulk copies and processes in place (see ephc_internal.h "resident-tile store" and DESIGN.md).
// Performed once on the CPU.  The diagonal (q = 0, n == m) terms are left out: they contribute
// exactly 0 to the collision integral; this store serves ephc_collision / ephc_rt_step.
//
// Product code: shares nothing with oracle/.
#include <algorithm>
#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <cstring>

#include "ephc_internal.h"

namespace ephc {

namespace {

struct DEnt {          // entry: T = |w| F_em or F_abs (sign of w)(f_out, f_in, N[iq, nu]); I[out] -= T; I[in] += T
    int32_t out, in;   // compact rows of the channel's first end a and second end b
    int32_t ip;        // candidate pair (-> iq)
    int32_t nu;
    double w;
};

struct Image {
    ResTile dir;
    std::vector<unsigned char> blob;
    std::vector<uint32_t> iqn;
    int64_t smem = 0;   // blob + zero + N rows
    int64_t work = 0;
};

struct ImgParams {
    int32_t a_row0, a_rows, b_row0, b_rows;
    int nnu, nwarp;
    int hcap;           // pieces of at most this many elements (0: automatic)
    bool stats;         // EPHC_DEBUG: count the gather wavefronts of the layout
    bool bank_aware;    // order a lane's entries so that the gathers of a column spread over the shared-memory banks
    int32_t nq_cap;     // pairs per tile (bounds the iq list that rides in the previous tile's image)
    int64_t budget;     // bytes available for image (without that list) + zero + N rows
    const int32_t *pair_iq;
};

struct Scratch {
    std::vector<int32_t> cnt, start, idx, pos_of, in_start, in_list;
    std::vector<uint32_t> pair_local;
};

// working statistics (EPHC_DEBUG): shared-memory wavefronts of the 8-byte gathers as laid out, and their lower bound
static long long g_wf_f = 0, g_wf_n = 0, g_wf_t = 0, g_wf_ideal1 = 0, g_wf_ideal2 = 0;

struct Piece {
    int32_t row, start, len;   // local row; first element in the row-sorted list; elements
};

struct Slab {
    int32_t base, H;           // first position; columns
    bool multi;                // some row owns more than one lane
    int32_t piece[32];         // piece per lane, -1 = none
};

// Cuts the lists [start[r], start[r+1]) of the rows r0 .. r1 into pieces of at most hcap elements (equal parts), sorts
// them by descending length with the pieces of one row adjacent, and deals them 32 per slab; the pieces of one row never
// straddle two slabs (a row has at most 32 pieces).  With keep_empty, rows without elements get a lane too (a piece
// of length 0).  The slabs are then dealt to nwarp warps, longest first to the least loaded warp, and come out warp by
// warp (wptr[w] .. wptr[w+1]), each warp's slabs by descending height.
static void make_slabs(const std::vector<int32_t> &start, int32_t r0, int32_t r1, bool keep_empty, int32_t hcap, int nwarp,
                       std::vector<Piece> &pieces, std::vector<Slab> &slabs, std::vector<int32_t> &wptr, int32_t &npos) {
    pieces.clear();
    std::vector<Slab> tmp;
    std::vector<std::pair<int32_t, int32_t>> rows;  // (first piece, pieces) per row
    for (int32_t r = r0; r < r1; ++r) {
        const int32_t c = start[r + 1] - start[r];
        if (c == 0 && !keep_empty) continue;
        int32_t npc = 1;  // a power of two, so that the lanes of whole rows fill a slab exactly
        while (npc * hcap < c) npc *= 2;
        const int32_t base = c / npc, rem = c % npc;
        rows.push_back({(int32_t)pieces.size(), npc});
        int32_t s = start[r];
        for (int32_t k = 0; k < npc; ++k) {
            const int32_t len = base + (k < rem ? 1 : 0);
            pieces.push_back(Piece{r, s, len});
            s += len;
        }
    }
    // rows by the length of their longest piece (the first), descending; ties by row
    std::stable_sort(rows.begin(), rows.end(), [&](const std::pair<int32_t, int32_t> &x, const std::pair<int32_t, int32_t> &y) {
        return pieces[x.first].len > pieces[y.first].len;
    });
    int32_t used = 32;
    for (const auto &rw : rows) {
        if (used + rw.second > 32) {
            Slab sl;
            sl.base = 0;
            sl.H = pieces[rw.first].len;
            sl.multi = false;
            std::fill(sl.piece, sl.piece + 32, -1);
            tmp.push_back(sl);
            used = 0;
        }
        Slab &sl = tmp.back();
        if (rw.second > 1) sl.multi = true;
        for (int32_t k = 0; k < rw.second; ++k) sl.piece[used++] = rw.first + k;
    }
    // tmp is sorted by descending height: longest first to the least loaded warp (cost: columns + a prologue)
    std::vector<std::vector<int32_t>> mine((size_t)nwarp);
    std::vector<int64_t> load((size_t)nwarp, 0);
    for (size_t i = 0; i < tmp.size(); ++i) {
        int best = 0;
        for (int w = 1; w < nwarp; ++w)
            if (load[w] < load[best]) best = w;
        mine[best].push_back((int32_t)i);
        load[best] += tmp[i].H + 2;
    }
    slabs.clear();
    wptr.assign((size_t)nwarp + 1, 0);
    npos = 0;
    for (int w = 0; w < nwarp; ++w) {
        for (int32_t i : mine[w]) {
            slabs.push_back(tmp[i]);
            slabs.back().base = npos;
            npos += 32 * tmp[i].H;
        }
        wptr[w + 1] = (int32_t)slabs.size();
    }
}

// Builds the image of one tile from entries e[0..n) (sorted by pair).  Returns false when a format limit or the
// shared-memory budget is exceeded (the caller then splits the entry range).
static bool build_image(const DEnt *e, int64_t n, const ImgParams &P, Scratch &S, Image &out) {
    const int32_t R = P.a_rows + P.b_rows;
    if (n > kResXMax - 32 || R > kResRowMax) return false;
    auto loc = [&](int32_t row) {
        return (row >= P.a_row0 && row < P.a_row0 + P.a_rows) ? row - P.a_row0 : P.a_rows + (row - P.b_row0);
    };
    // pairs
    S.pair_local.resize((size_t)n);
    out.iqn.clear();
    for (int64_t i = 0; i < n; ++i) {
        if (i == 0 || e[i].ip != e[i - 1].ip) out.iqn.push_back((uint32_t)P.pair_iq[e[i].ip] * (uint32_t)P.nnu);
        S.pair_local[i] = (uint32_t)out.iqn.size() - 1u;
    }
    const int32_t nq = (int32_t)out.iqn.size();
    if ((int64_t)nq * P.nnu > kResSlotMax || nq > P.nq_cap) return false;
    // ---- phase 1: entries by a row (inside a row by b row, then canonical order) ------------------------------------
    S.cnt.assign((size_t)R + 1, 0);
    for (int64_t i = 0; i < n; ++i) S.cnt[loc(e[i].out) + 1]++;
    S.start.assign((size_t)R + 1, 0);
    int32_t longest = 0;
    for (int32_t r = 0; r < R; ++r) {
        S.start[r + 1] = S.start[r] + S.cnt[r + 1];
        longest = std::max(longest, S.cnt[r + 1]);
    }
    S.idx.resize((size_t)n);
    {
        std::vector<int32_t> &cur = S.cnt;  // reuse as cursor
        for (int32_t r = 0; r < R; ++r) cur[r] = S.start[r];
        for (int64_t i = 0; i < n; ++i) S.idx[cur[loc(e[i].out)]++] = (int32_t)i;
    }
    for (int32_t r = 0; r < R; ++r)
        std::sort(S.idx.begin() + S.start[r], S.idx.begin() + S.start[r + 1], [&](int32_t x, int32_t y) {
            if (e[x].in != e[y].in) return e[x].in < e[y].in;
            return x < y;
        });
    // b-row lists (an upper bound on their lengths for the piece length: one term per entry)
    S.in_start.assign((size_t)R + 1, 0);
    for (int64_t i = 0; i < n; ++i) S.in_start[loc(e[i].in) + 1]++;
    for (int32_t r = 0; r < R; ++r) {
        longest = std::max(longest, S.in_start[r + 1]);
        S.in_start[r + 1] += S.in_start[r];
    }
    const int32_t hmin = (longest + 31) / 32;  // a row owns at most 32 lanes
    if (hmin > kResHMax) return false;
    std::vector<Piece> pc1, pc2;
    std::vector<Slab> sl1, sl2;
    std::vector<int32_t> wp1, wp2;
    int32_t ne_pad = 0, ng_pad = 0;
    // piece length: the candidate with the least padding and fewest slabs (positions + a prologue per slab)
    int32_t hcap = std::max(P.hcap, hmin);
    if (P.hcap <= 0) {
        int64_t best = -1;
        for (int32_t cand : {6, 8, 10, 12, 16, 20, 24, 32, 48, 64, 96, 128, 256, kResHMax}) {
            if (cand < hmin) continue;
            int32_t np1 = 0, np2 = 0;
            make_slabs(S.start, 0, R, false, cand, P.nwarp, pc1, sl1, wp1, np1);
            if (P.b_rows > 0)
                make_slabs(S.in_start, P.a_rows, R, true, cand, P.nwarp, pc2, sl2, wp2, np2);
            else
                make_slabs(S.in_start, 0, R, false, cand, P.nwarp, pc2, sl2, wp2, np2);
            // the slowest warp of each phase sets the pace
            int64_t cost = 0;
            for (int ph = 0; ph < 2; ++ph) {
                const std::vector<Slab> &sl = ph ? sl2 : sl1;
                const std::vector<int32_t> &wp = ph ? wp2 : wp1;
                int64_t worst = 0;
                for (int w = 0; w < P.nwarp; ++w) {
                    int64_t ld = 0;
                    for (int32_t k = wp[w]; k < wp[w + 1]; ++k) ld += (ph ? 2 : 5) * (int64_t)sl[k].H + 8;
                    worst = std::max(worst, ld);
                }
                cost += worst * P.nwarp;
            }
            cost += 2 * ((int64_t)np1 + np2) / 3;  // and the bytes moved
            if (best < 0 || cost < best) {
                best = cost;
                hcap = cand;
            }
        }
    }
    make_slabs(S.start, 0, R, false, hcap, P.nwarp, pc1, sl1, wp1, ne_pad);
    if (ne_pad > kResXMax - 1 || ne_pad / 32 > 1023) return false;
    // Order of a lane's entries.  The entries of one (owner, partner) state pair inside a piece -- a COMBO: its modes and
    // kinds -- stay adjacent: the kernel sums their weights and forms ONE term at the combo's last entry, so f_b is
    // gathered, T stored and T gathered again once per combo.  Inside that constraint the order is free (combos as
    // blocks, entries inside a combo): a warp gathers N (every entry) and f_b (combo ends) of a column with 8-byte loads,
    // 16 lanes per shared-memory wavefront, and every extra lane on a bank pair (address / 8 mod 16) costs another
    // wavefront.  Column by column, lanes with the fewest entries left choose first: an entry of the lane's open combo,
    // or of any combo if none is open, that lands on the least used bank pairs.
    if (P.bank_aware) {
        auto bank_f = [&](int32_t ei) { return loc(e[ei].in) & 15; };
        auto bank_n = [&](int32_t ei) { return (int32_t)((S.pair_local[ei] * (uint32_t)P.nnu + (uint32_t)e[ei].nu) & 15u); };
        int32_t order[16];
        for (const Slab &sl : sl1)
            for (int32_t j = 0; j + 1 < sl.H; ++j)
                for (int half = 0; half < 2; ++half) {
                    int32_t cf[16] = {0}, cn[16] = {0}, nl = 0;
                    for (int l = 16 * half; l < 16 * half + 16; ++l)
                        if (sl.piece[l] >= 0 && pc1[sl.piece[l]].len > j) order[nl++] = l;
                    std::sort(order, order + nl, [&](int32_t x, int32_t y) { return pc1[sl.piece[x]].len < pc1[sl.piece[y]].len; });
                    for (int32_t k = 0; k < nl; ++k) {
                        const Piece &pc = pc1[sl.piece[order[k]]];
                        // the open combo: entries left with the partner of the entry just placed
                        int32_t open_in = -1;
                        if (j > 0) {
                            const int32_t pin = e[S.idx[pc.start + j - 1]].in;
                            for (int32_t m = j; m < pc.len && open_in < 0; ++m)
                                if (e[S.idx[pc.start + m]].in == pin) open_in = pin;
                        }
                        int32_t best = -1, bc = 1 << 30;
                        for (int32_t m = j; m < pc.len; ++m) {
                            const int32_t ei = S.idx[pc.start + m];
                            if (open_in >= 0 && e[ei].in != open_in) continue;
                            int32_t left = 0;  // entries of this combo still to place (including this one)
                            for (int32_t m2 = j; m2 < pc.len; ++m2) left += e[S.idx[pc.start + m2]].in == e[ei].in;
                            const int32_t c = cn[bank_n(ei)] + (left == 1 ? cf[bank_f(ei)] : 0);
                            if (c < bc) bc = c, best = m;
                        }
                        std::swap(S.idx[pc.start + j], S.idx[pc.start + best]);
                        const int32_t ei = S.idx[pc.start + j];
                        cn[bank_n(ei)]++;
                        bool last = true;
                        for (int32_t m2 = j + 1; m2 < pc.len; ++m2) last &= e[S.idx[pc.start + m2]].in != e[ei].in;
                        if (last) cf[bank_f(ei)]++;
                    }
                }
    }
    // combo ends: the last entry of a piece, or the next entry has another partner
    std::vector<uint8_t> is_end((size_t)n, 0);
    int32_t ncombo = 0;
    for (const Piece &pc : pc1)
        for (int32_t k = 0; k < pc.len; ++k)
            if (k + 1 == pc.len || e[S.idx[pc.start + k + 1]].in != e[S.idx[pc.start + k]].in) {
                is_end[S.idx[pc.start + k]] = 1;
                ++ncombo;
            }
    if (P.stats) {  // wavefronts of the f_b and N gathers: per column and half-warp, the largest number of DISTINCT addresses on a bank pair
        long long wf = 0, wn = 0, wi = 0;
        for (const Slab &sl : sl1)
            for (int32_t j = 0; j < sl.H; ++j)
                for (int half = 0; half < 2; ++half) {
                    int32_t af[16][16], an[16][16], cf[16] = {0}, cn[16] = {0};
                    bool any = false;
                    for (int l = 16 * half; l < 16 * half + 16; ++l) {
                        if (sl.piece[l] < 0 || pc1[sl.piece[l]].len <= j) continue;
                        any = true;
                        const int32_t ei = S.idx[pc1[sl.piece[l]].start + j];
                        const int32_t fa = loc(e[ei].in), na = (int32_t)(S.pair_local[ei] * (uint32_t)P.nnu + (uint32_t)e[ei].nu);
                        bool dup = !is_end[ei];  // f_b is read at combo ends only
                        for (int k = 0; k < cf[fa & 15]; ++k) dup |= af[fa & 15][k] == fa;
                        if (!dup) af[fa & 15][cf[fa & 15]++] = fa;
                        dup = false;
                        for (int k = 0; k < cn[na & 15]; ++k) dup |= an[na & 15][k] == na;
                        if (!dup) an[na & 15][cn[na & 15]++] = na;
                    }
                    if (!any) continue;
                    wf += *std::max_element(cf, cf + 16);
                    wn += *std::max_element(cn, cn + 16);
                    wi += 1;
                }
#pragma omp critical
        {
            g_wf_f += wf;
            g_wf_n += wn;
            g_wf_ideal1 += wi;
        }
    }
    S.pos_of.resize((size_t)n);
    for (const Slab &sl : sl1)
        for (int l = 0; l < 32; ++l) {
            if (sl.piece[l] < 0) continue;
            const Piece &pc = pc1[sl.piece[l]];
            for (int32_t k = 0; k < pc.len; ++k) S.pos_of[S.idx[pc.start + k]] = sl.base + 32 * k + l;
        }
    // ---- phase 2: positions of the combo terms of every b row, ascending; off the diagonal every B row gets a lane ---
    S.in_start.assign((size_t)R + 1, 0);
    for (int64_t i = 0; i < n; ++i)
        if (is_end[i]) S.in_start[loc(e[i].in) + 1]++;
    for (int32_t r = 0; r < R; ++r) S.in_start[r + 1] += S.in_start[r];
    S.in_list.resize((size_t)ncombo);
    {
        std::vector<int32_t> cur(S.in_start.begin(), S.in_start.end() - 1);
        for (int64_t i = 0; i < n; ++i)
            if (is_end[i]) S.in_list[cur[loc(e[i].in)]++] = S.pos_of[i];
        for (int32_t r = 0; r < R; ++r) std::sort(S.in_list.begin() + S.in_start[r], S.in_list.begin() + S.in_start[r + 1]);
    }
    if (P.b_rows > 0)
        make_slabs(S.in_start, P.a_rows, R, true, hcap, P.nwarp, pc2, sl2, wp2, ng_pad);
    else
        make_slabs(S.in_start, 0, R, false, hcap, P.nwarp, pc2, sl2, wp2, ng_pad);
    if (ng_pad / 32 > 1023) return false;
    if (P.bank_aware) {  // the same for the T values a lane of phase 2 gathers: bank pair = position mod 16
        int32_t order[16];
        for (const Slab &sl : sl2)
            for (int32_t j = 0; j + 1 < sl.H; ++j)
                for (int half = 0; half < 2; ++half) {
                    int32_t cx[16] = {0}, nl = 0;
                    for (int l = 16 * half; l < 16 * half + 16; ++l)
                        if (sl.piece[l] >= 0 && pc2[sl.piece[l]].len > j) order[nl++] = l;
                    std::sort(order, order + nl, [&](int32_t x, int32_t y) { return pc2[sl.piece[x]].len < pc2[sl.piece[y]].len; });
                    for (int32_t k = 0; k < nl; ++k) {
                        const Piece &pc = pc2[sl.piece[order[k]]];
                        int32_t best = j, bc = 1 << 30;
                        for (int32_t m = j; m < pc.len; ++m) {
                            const int32_t c = cx[S.in_list[pc.start + m] & 15];
                            if (c < bc) bc = c, best = m;
                        }
                        std::swap(S.in_list[pc.start + j], S.in_list[pc.start + best]);
                        cx[S.in_list[pc.start + j] & 15]++;
                    }
                }
    }
    if (P.stats) {
        long long wt = 0, wi = 0;
        for (const Slab &sl : sl2)
            for (int32_t j = 0; j < sl.H; ++j)
                for (int half = 0; half < 2; ++half) {
                    int32_t cx[16] = {0};
                    bool any = false;
                    for (int l = 16 * half; l < 16 * half + 16; ++l) {
                        if (sl.piece[l] < 0 || pc2[sl.piece[l]].len <= j) continue;
                        any = true;
                        cx[S.in_list[pc2[sl.piece[l]].start + j] & 15]++;
                    }
                    if (!any) continue;
                    wt += *std::max_element(cx, cx + 16);
                    wi += 1;
                }
#pragma omp critical
        {
            g_wf_t += wt;
            g_wf_ideal2 += wi;
        }
    }
    ResTile &D = out.dir;
    std::memset(&D, 0, sizeof(D));
    D.ne = (int32_t)n;
    D.ncombo = ncombo;
    D.ne_pad = ne_pad;
    D.ng_pad = ng_pad;
    D.nslab1 = (int32_t)sl1.size();
    D.nslab2 = (int32_t)sl2.size();
    D.nq = nq;
    D.nq_next = 0;
    D.b_row0 = P.b_row0;
    D.b_rows = P.b_rows;
    D.b_slot = -1;
    res_set_layout(D, P.nwarp);
    out.smem = res_tile_smem(D, P.nnu);
    if (out.smem > P.budget) return false;
    // ---- fill the blob ---------------------------------------------------------------------------------------------
    out.blob.assign((size_t)D.blob_bytes, 0);
    uint32_t *code = reinterpret_cast<uint32_t *>(out.blob.data());
    uint16_t *perm = reinterpret_cast<uint16_t *>(out.blob.data() + D.o_perm);
    uint16_t *srow1 = reinterpret_cast<uint16_t *>(out.blob.data() + D.o_srow1);
    uint32_t *shdr1 = reinterpret_cast<uint32_t *>(out.blob.data() + D.o_shdr1);
    uint16_t *srow2 = reinterpret_cast<uint16_t *>(out.blob.data() + D.o_srow2);
    uint32_t *shdr2 = reinterpret_cast<uint32_t *>(out.blob.data() + D.o_shdr2);
    uint16_t *wptr = reinterpret_cast<uint16_t *>(out.blob.data() + D.o_wptr);
    double *w = reinterpret_cast<double *>(out.blob.data() + D.o_w);
    // padding entries: w = 0, partner row 0, N slot 0 (both always staged)
    for (int64_t i = 0; i < n; ++i) {
        const int32_t pos = S.pos_of[i];
        code[pos] = ((uint32_t)loc(e[i].in) << 3) | ((S.pair_local[i] * (uint32_t)P.nnu + (uint32_t)e[i].nu) << 19) | is_end[i];
        w[pos] = e[i].w;
    }
    for (size_t s = 0; s < sl1.size(); ++s) {
        shdr1[s] = (uint32_t)(sl1[s].base / 32) | ((uint32_t)sl1[s].H << kResHdrHShift) | (sl1[s].multi ? kResHdrMulti : 0u);
        for (int l = 0; l < 32; ++l) srow1[32 * s + l] = sl1[s].piece[l] < 0 ? kResNoRow : (uint16_t)pc1[sl1[s].piece[l]].row;
    }
    for (int32_t g = 0; g < ng_pad; ++g) perm[g] = (uint16_t)ne_pad;  // the zero
    for (size_t s = 0; s < sl2.size(); ++s) {
        shdr2[s] = (uint32_t)(sl2[s].base / 32) | ((uint32_t)sl2[s].H << kResHdrHShift) | (sl2[s].multi ? kResHdrMulti : 0u);
        for (int l = 0; l < 32; ++l) {
            srow2[32 * s + l] = kResNoRow;
            if (sl2[s].piece[l] < 0) continue;
            const Piece &pc = pc2[sl2[s].piece[l]];
            srow2[32 * s + l] = (uint16_t)pc.row;
            for (int32_t k = 0; k < pc.len; ++k) perm[sl2[s].base + 32 * k + l] = (uint16_t)S.in_list[pc.start + k];
        }
    }
    for (int w_ = 0; w_ <= P.nwarp; ++w_) {
        wptr[w_] = (uint16_t)wp1[w_];
        wptr[P.nwarp + 1 + w_] = (uint16_t)wp2[w_];
    }
    // cost model of a tile for the shares, in phase-1 positions: positions, gathers, per-slab prologues, staged N rows
    out.work = ne_pad + (2 * (int64_t)ng_pad) / 5 + 45 * (int64_t)(D.nslab1 + D.nslab2) + 3 * (int64_t)nq + 600;
    return true;
}

static int build_images(const DEnt *e, int64_t n, const ImgParams &P, Scratch &S, std::vector<Image> &outs) {
    if (n <= 0) return EPHC_OK;
    Image img;
    if (build_image(e, n, P, S, img)) {
        outs.push_back(std::move(img));
        return EPHC_OK;
    }
    if (n == 1) return EPHC_ELIMIT;
    int64_t mid = n / 2, lo = mid, hi = mid;  // prefer a pair boundary near the middle
    while (lo > n / 4 && e[lo].ip == e[lo - 1].ip) --lo;
    while (hi < n - n / 4 && e[hi].ip == e[hi - 1].ip) ++hi;
    if (lo > 0 && e[lo].ip != e[lo - 1].ip)
        mid = lo;
    else if (hi < n && e[hi].ip != e[hi - 1].ip)
        mid = hi;
    int rc = build_images(e, mid, P, S, outs);
    if (rc == EPHC_OK) rc = build_images(e + mid, n - mid, P, S, outs);
    return rc;
}

static int env_int(const char *name, int dflt) {
    const char *e = std::getenv(name);
    return e ? std::atoi(e) : dflt;
}

}  // namespace

int build_res(const ephc_problem *p, const Dims &d, const Canonical &c, int ncta, int64_t smem_cap, int nwarp, ResHost &t,
              std::string &err) {
    const int nb = d.nb, nnu = d.nnu;
    const int64_t npair = p->npair;
    t = ResHost();
    t.nnu = nnu;
    t.smem_cap = smem_cap;
    if (ncta < 1) ncta = 1;
    try {
        t.state_row.assign((size_t)d.ns, -1);
        for (int64_t s = 0; s < d.ns; ++s)
            if (p->E[s] >= p->emin && p->E[s] <= p->emax) {
                t.state_row[s] = (int32_t)t.row_state.size();
                t.row_state.push_back((int32_t)s);
            }
        t.nrows = (int32_t)t.row_state.size();
        const int64_t nent = c.nw;
        t.nent = nent;
        // ---- geometry: strips of Ra rows, B ranges of <= RbMax rows in units of fine blocks of Rf rows --------------
        int Ra = env_int("EPHC_RES_ROWS", 1024), RbMax = env_int("EPHC_RES_ROWS_B", 512);
        const int hcap = std::max(0, env_int("EPHC_RES_HCAP", 0));
        Ra = std::max(1, std::min(Ra, kResRowMax / 2));
        RbMax = std::max(1, std::min(RbMax, kResRowMax / 2));
        const double rho = (double)std::max<int64_t>(nent, 1) / (0.5 * (double)t.nrows * (double)t.nrows + 1.0);  // entries per row pair
        const double bytes_per_entry = 15.5 + 8.0 * nnu / std::max(1.0, (double)nent / std::max<int64_t>(1, c.npair_active));
        if (!std::getenv("EPHC_RES_ROWS")) {
            // square tiles give both ends of a channel equally long rows: Ra = Rb = sqrt(entries that fit / density); the
            // f values of both row ranges may take a quarter of a buffer
            Ra = 1024;
            for (int iter = 0; iter < 3; ++iter) {
                const double buf = (double)(smem_cap - res_fixed_bytes(Ra)) / 2 - 8.0 * 3.0 * Ra - 256;
                const double rstar = std::sqrt(std::max(64.0, buf) / bytes_per_entry / rho);
                Ra = (int)std::max(32.0, std::min({rstar, 2048.0, (double)smem_cap / (2 * 4 * 8 * 3.0)}));
            }
            RbMax = std::min(2 * Ra, kResRowMax / 2);
            // small problems: enough strips that every CTA gets a few runs
            while (Ra > 16 && (int64_t)(t.nrows / Ra) * (t.nrows / Ra) < 8 * (int64_t)ncta) Ra /= 2;
        }
        // two tile buffers: f of the A and B rows, image + zero + N rows; three fifths of a buffer may hold N rows of pairs
        // (few channels per pair: the N rows outweigh the entries), which bounds the next tile's iq list that an image carries
        const int64_t per_buf = (smem_cap - res_fixed_bytes(Ra)) / 2 - 8 * (int64_t)(Ra + RbMax) - 256;
        const int32_t nq_cap = (int32_t)std::max<int64_t>(1, std::min<int64_t>(kResSlotMax / nnu, (per_buf * 3 / 5) / (8 * (int64_t)nnu)));
        const int64_t budget = per_buf - 4 * (int64_t)nq_cap - 16;
        if (budget < 2048) {
            t.why = "resident-tile store: shared-memory budget too small";
            return EPHC_OK;
        }
        int Rf = env_int("EPHC_RES_FINE", 0);
        if (Rf <= 0) {
            // an atom (strip x fine block) should hold about a sixth of what fits in a tile
            const double per_row = std::max(1e-9, rho * Ra) * bytes_per_entry;
            Rf = 128;
            while (Rf > 4 && Rf * per_row > (double)budget / 6.0) Rf /= 2;
        }
        Rf = std::max(2, std::min(Rf, Ra) & ~1);  // even: bulk copies of f need 16-byte aligned row ranges
        Ra = std::max(Rf, Ra / Rf * Rf);
        RbMax = std::max(Rf, RbMax / Rf * Rf);
        t.Ra = Ra;
        t.rf = Rf;
        t.nblk = std::max(1, (t.nrows + Rf - 1) / Rf);
        t.blk_row0.resize((size_t)t.nblk + 1);
        for (int32_t b = 0; b <= t.nblk; ++b) t.blk_row0[b] = std::min(t.nrows, b * Rf);
        t.state_blk.assign((size_t)d.ns, -1);
        for (int64_t s = 0; s < d.ns; ++s)
            if (t.state_row[s] >= 0) t.state_blk[s] = t.state_row[s] / Rf;
        const int32_t bps = Ra / Rf;
        const int32_t nstrip = (t.nblk + bps - 1) / bps;
        std::vector<int64_t> atom0((size_t)nstrip + 1, 0);  // atoms of strip I: diagonal, then the fine blocks after it
        for (int32_t I = 0; I < nstrip; ++I) atom0[I + 1] = atom0[I] + 1 + std::max(0, t.nblk - (I + 1) * bps);
        const int64_t natom = atom0[nstrip];
        auto atom_of = [&](int32_t a, int32_t b) {  // a < b compact rows
            const int32_t I = a / Ra, j = b / Rf;
            return (j < (I + 1) * bps) ? atom0[I] : atom0[I] + 1 + (j - (I + 1) * bps);
        };
        // entries and pairs per atom
        std::vector<int64_t> atom_ne((size_t)natom + 1, 0);
        std::vector<int32_t> atom_np((size_t)natom + 1, 0);
        {
            std::vector<int64_t> seen;
            for (int64_t ip = 0; ip < npair; ++ip) {
                const int64_t sa = (int64_t)p->pair_ik[ip] * nb, sb = (int64_t)p->pair_ikq[ip] * nb;
                seen.clear();
                for (int64_t j = c.pair_ch0[ip]; j < c.pair_ch0[ip + 1]; ++j) {
                    const int n = c.ch_code[j] & 15, m = (c.ch_code[j] >> 4) & 15;
                    const int64_t at = atom_of(t.state_row[sa + n], t.state_row[sb + m]);
                    atom_ne[at + 1] += (c.ch_wabs[j] != 0.0) + (c.ch_wem[j] != 0.0);
                    if (std::find(seen.begin(), seen.end(), at) == seen.end()) {  // a pair touches very few atoms
                        seen.push_back(at);
                        atom_np[at + 1]++;
                    }
                }
            }
        }
        for (int64_t i = 0; i < natom; ++i) atom_ne[i + 1] += atom_ne[i];  // prefix sums from here on
        // initial tiles: consecutive atoms of a strip while the estimated image fits.  The estimate is an upper bound
        // (every row of the tile has a piece and a task); `scale` (<= 1) is the measured ratio of the real size.
        struct Init {
            int64_t at0, at1;
            int32_t strip;
            int64_t est;
        };
        auto est_bytes = [&](int64_t E, int64_t Pq, int64_t rows_) {
            return 15 * E + 8 * (int64_t)nnu * Pq + 5 * std::min<int64_t>(rows_, 2 * E) + 1024;
        };
        auto make_inits = [&](int32_t I, double scale, std::vector<Init> &inits) {
            const int32_t a_rows = std::min(t.nrows, (I + 1) * Ra) - std::min(t.nrows, I * Ra);
            if (atom_ne[atom0[I] + 1] > atom_ne[atom0[I]]) inits.push_back(Init{atom0[I], atom0[I] + 1, I, 0});
            int64_t a0 = atom0[I] + 1;
            while (a0 < atom0[I + 1]) {
                if (atom_ne[a0 + 1] == atom_ne[a0]) {
                    ++a0;
                    continue;
                }
                int64_t a1 = a0, Pq = 0, est_last = 0;
                while (a1 < atom0[I + 1] && (a1 + 1 - a0) * Rf <= RbMax) {
                    const int64_t E2 = atom_ne[a1 + 1] - atom_ne[a0], P2 = Pq + atom_np[a1 + 1];
                    const int64_t est = est_bytes(E2, P2, a_rows + (a1 + 1 - a0) * Rf);
                    if (a1 > a0 && ((double)est * scale > (double)budget || E2 > kResXMax * 3 / 4 || (double)P2 * scale > nq_cap)) break;
                    Pq = P2;
                    est_last = est;
                    ++a1;
                }
                while (a1 - 1 > a0 && atom_ne[a1] == atom_ne[a1 - 1]) --a1;
                inits.push_back(Init{a0, a1, I, est_last});
                a0 = a1;
            }
        };
        std::vector<int32_t> atom_init((size_t)natom, -1);
        // entries of the given initial tiles -> images (bucket by tile in canonical order, then build in parallel)
        auto build_inits = [&](const std::vector<Init> &inits, std::vector<std::vector<Image>> &imgs) -> int {
            const int64_t ninit = (int64_t)inits.size();
            std::vector<int64_t> init_e0((size_t)ninit + 1, 0);
            std::fill(atom_init.begin(), atom_init.end(), -1);
            std::vector<uint8_t> strip_on((size_t)nstrip, 0);
            for (int64_t it = 0; it < ninit; ++it) {
                for (int64_t at = inits[it].at0; at < inits[it].at1; ++at) atom_init[at] = (int32_t)it;
                init_e0[it + 1] = init_e0[it] + (atom_ne[inits[it].at1] - atom_ne[inits[it].at0]);
                strip_on[inits[it].strip] = 1;
            }
            std::vector<DEnt> ents((size_t)init_e0[ninit]);
            {
                std::vector<int64_t> cur(init_e0.begin(), init_e0.end() - 1);
                for (int64_t ip = 0; ip < npair; ++ip) {
                    const int64_t sa = (int64_t)p->pair_ik[ip] * nb, sb = (int64_t)p->pair_ikq[ip] * nb;
                    for (int64_t j = c.pair_ch0[ip]; j < c.pair_ch0[ip + 1]; ++j) {
                        const int n = c.ch_code[j] & 15, m = (c.ch_code[j] >> 4) & 15, nu = c.ch_code[j] >> 8;
                        const int32_t a = t.state_row[sa + n], b = t.state_row[sb + m];
                        if (!strip_on[a / Ra]) continue;
                        const int64_t it = atom_init[atom_of(a, b)];
                        if (it < 0) continue;
                        // owner a, partner b; emission weight stored as +w, absorption weight as -w
                        if (c.ch_wem[j] != 0.0) ents[cur[it]++] = DEnt{a, b, (int32_t)ip, nu, c.ch_wem[j]};
                        if (c.ch_wabs[j] != 0.0) ents[cur[it]++] = DEnt{a, b, (int32_t)ip, nu, -c.ch_wabs[j]};
                    }
                }
                for (int64_t it = 0; it < ninit; ++it)
                    if (cur[it] != init_e0[it + 1]) return EPHC_ESTATE;
            }
            imgs.assign((size_t)ninit, {});
            int rc_all = EPHC_OK;
#pragma omp parallel
            {
                Scratch S;
#pragma omp for schedule(dynamic, 4)
                for (int64_t it = 0; it < ninit; ++it) {
                    const Init &in = inits[it];
                    ImgParams P;
                    P.a_row0 = std::min(t.nrows, in.strip * Ra);
                    P.a_rows = std::min(t.nrows, (in.strip + 1) * Ra) - P.a_row0;
                    if (in.at0 == atom0[in.strip]) {
                        P.b_row0 = P.a_row0;
                        P.b_rows = 0;
                    } else {
                        const int32_t j0 = (in.strip + 1) * bps + (int32_t)(in.at0 - atom0[in.strip] - 1);
                        const int32_t j1 = (in.strip + 1) * bps + (int32_t)(in.at1 - 1 - atom0[in.strip] - 1);
                        P.b_row0 = t.blk_row0[j0];
                        P.b_rows = t.blk_row0[j1 + 1] - P.b_row0;
                    }
                    P.nnu = nnu;
                    P.nwarp = nwarp;
                    P.hcap = hcap;
                    P.bank_aware = !std::getenv("EPHC_RES_NO_BANKS");
                    P.stats = std::getenv("EPHC_DEBUG") != nullptr;
                    P.nq_cap = nq_cap;
                    P.budget = budget;
                    P.pair_iq = c.pair_iq.data();
                    const int rc = build_images(ents.data() + init_e0[it], init_e0[it + 1] - init_e0[it], P, S, imgs[it]);
                    if (rc != EPHC_OK) {
#pragma omp critical
                        rc_all = rc;
                    }
                }
            }
            return rc_all;
        };
        // calibration on a few strips: how much of the upper bound do real images use?
        double scale = 1.0;
        if (!std::getenv("EPHC_RES_NO_CALIB")) {
            std::vector<Init> sample;
            const int nsample = std::min(nstrip, 6);
            for (int k = 0; k < nsample; ++k) make_inits((int32_t)((int64_t)k * nstrip / nsample), 1.0, sample);
            std::vector<std::vector<Image>> simg;
            const int rc = build_inits(sample, simg);
            if (rc != EPHC_OK) {
                err = rc == EPHC_ESTATE ? "internal: resident-tile store lost entries" : "resident-tile store: a single entry does not fit the shared-memory budget";
                return rc;
            }
            double worst = 0.0;
            for (size_t it = 0; it < sample.size(); ++it)
                if (simg[it].size() == 1 && sample[it].est > budget / 2)  // well filled, not split
                    worst = std::max(worst, (double)simg[it][0].smem / (double)sample[it].est);
            if (worst > 0.0) scale = std::min(1.0, worst * 1.03);
        }
        std::vector<Init> inits;
        for (int32_t I = 0; I < nstrip; ++I) make_inits(I, scale, inits);
        const int64_t ninit = (int64_t)inits.size();
        std::vector<std::vector<Image>> imgs;
        {
            const int rc = build_inits(inits, imgs);
            if (rc != EPHC_OK) {
                err = rc == EPHC_ESTATE ? "internal: resident-tile store lost entries" : "resident-tile store: a single entry does not fit the shared-memory budget";
                return rc;
            }
        }
        // ---- runs, static schedule, images in schedule order, slots -----------------------------------------------
        int64_t total_work = 0;
        for (auto &v : imgs)
            for (Image &im : v) total_work += im.work;
        // static schedule: the tiles in strip-major order are cut into ncta contiguous shares of equal work; inside a
        // share, consecutive tiles of one strip form a run
        struct RunTmp {
            std::vector<std::pair<int64_t, int32_t>> tl;  // (initial tile, image)
            int32_t strip;
            int64_t work;
        };
        std::vector<RunTmp> rt;
        std::vector<std::vector<int32_t>> cta_runs((size_t)ncta);
        {
            int32_t cur_strip = -1, cta = 0;
            int64_t done = 0;
            for (int64_t it = 0; it < ninit; ++it)
                for (size_t k = 0; k < imgs[it].size(); ++k) {
                    const int64_t wk = imgs[it][k].work;
                    bool cut = false;
                    while (cta + 1 < ncta && done + wk / 2 > total_work * (int64_t)(cta + 1) / ncta) {
                        ++cta;
                        cut = true;
                    }
                    if (cut || inits[it].strip != cur_strip) {
                        rt.push_back(RunTmp{{}, inits[it].strip, 0});
                        cta_runs[cta].push_back((int32_t)rt.size() - 1);
                        cur_strip = inits[it].strip;
                    }
                    rt.back().tl.push_back({it, (int32_t)k});
                    rt.back().work += wk;
                    done += wk;
                }
        }
        t.ncta = ncta;
        int64_t rows = 0;
        auto new_slot = [&](int32_t row0, int32_t nrows_) {
            const int32_t sl = (int32_t)t.slot_off.size();
            t.slot_off.push_back(rows);
            t.slot_row0.push_back(row0);
            t.slot_rows.push_back(nrows_);
            rows += nrows_;
            return sl;
        };
        t.cta_ptr.assign((size_t)ncta + 1, 0);
        std::vector<std::pair<int64_t, int32_t>> src;  // image of every scheduled tile
        for (int32_t cta = 0; cta < ncta; ++cta) {
            for (int32_t ir : cta_runs[cta]) {
                const RunTmp &r = rt[ir];
                const int32_t a_row0 = std::min(t.nrows, r.strip * Ra), a_rows = std::min(t.nrows, (r.strip + 1) * Ra) - a_row0;
                ResRun run{(int32_t)t.tiles.size(), (int32_t)r.tl.size(), a_row0, a_rows, new_slot(a_row0, a_rows), cta};
                t.runs.push_back(run);
                for (size_t k = 0; k < r.tl.size(); ++k) {
                    ResTile D = imgs[r.tl[k].first][r.tl[k].second].dir;
                    D.a_row0 = a_row0;
                    D.a_rows = a_rows;
                    D.a_slot = run.a_slot;
                    D.a_off = (uint32_t)t.slot_off[run.a_slot];
                    D.flags = (k == 0 ? 1 : 0) | (k + 1 == r.tl.size() ? 2 : 0);
                    if (D.b_rows > 0) {
                        D.b_slot = new_slot(D.b_row0, D.b_rows);
                        D.b_off = (uint32_t)t.slot_off[D.b_slot];
                    }
                    t.tiles.push_back(D);
                    t.tile_work.push_back((double)imgs[r.tl[k].first][r.tl[k].second].work);
                    src.push_back(r.tl[k]);
                }
            }
            t.cta_ptr[cta + 1] = (int32_t)t.tiles.size();
        }
        const int64_t ntile = (int64_t)t.tiles.size();
        int64_t boff = 0, nqtot = 0;
        t.Rcap = 2;
        for (int64_t i = 0; i < ntile; ++i) {
            ResTile &D = t.tiles[i];
            D.nq_next = 0;
            D.q0 = (int32_t)nqtot;
            nqtot += D.nq;
            if (nqtot > 0x7fffffffLL) {
                err = "resident-tile store: more than 2^31 tile pairs";
                return EPHC_ELIMIT;
            }
        }
        // the pair list of the NEXT tile in storage order rides in every image (the shares are contiguous pieces of that
        // order, wherever their boundaries are: res_reschedule may move them)
        for (int64_t i = 0; i + 1 < ntile; ++i) t.tiles[i].nq_next = t.tiles[i + 1].nq;
        for (int64_t i = 0; i < ntile; ++i) {
            ResTile &D = t.tiles[i];
            res_set_layout(D, nwarp);
            D.blob_off = boff;
            boff += (D.blob_bytes + 127) & ~127;
            t.smem_tile = std::max(t.smem_tile, res_tile_smem(D, nnu));
            t.Rcap = std::max(t.Rcap, D.a_rows + D.b_rows);
        }
        for (int64_t i = 0; i + 1 < ntile; ++i) t.tiles[i].o_sn_next = res_o_sn(t.tiles[i + 1]);
        if (t.smem_tile > per_buf) {
            err = "internal: resident tile exceeds its shared-memory budget";
            return EPHC_ESTATE;
        }
        t.Rcap = (t.Rcap + 1) & ~1;
        t.RbMax = RbMax;
        t.nwarp = nwarp;
        t.iqn.resize((size_t)nqtot);
        t.blob.assign((size_t)boff + 128, 0);
#pragma omp parallel for schedule(dynamic, 16)
        for (int64_t i = 0; i < ntile; ++i) {
            const ResTile &D = t.tiles[i];
            Image &im = imgs[src[i].first][src[i].second];
            const ResTile &D0 = im.dir;  // layout without the next tile's iq list: only w moves
            unsigned char *dst = t.blob.data() + D.blob_off;
            std::memcpy(dst, im.blob.data(), (size_t)D0.o_w);
            std::memcpy(dst + D.o_w, im.blob.data() + D0.o_w, (size_t)(D0.blob_bytes - (int32_t)D0.o_w));
            std::copy(im.iqn.begin(), im.iqn.end(), t.iqn.begin() + D.q0);
        }
        for (int64_t i = 0; i + 1 < ntile; ++i) {  // the next tile's iq list rides in the image of its predecessor
            const ResTile &D = t.tiles[i], &Dn = t.tiles[i + 1];
            std::memcpy(t.blob.data() + D.blob_off + D.o_nxt, t.iqn.data() + Dn.q0, (size_t)Dn.nq * 4);
        }
        imgs.clear();
        t.part_rows = rows;
        if (rows > 0xffffffffLL) {
            err = "resident-tile store: partial-sum buffer exceeds 2^32 rows";
            return EPHC_ELIMIT;
        }
        t.blk_ent_ptr.assign((size_t)t.nblk + 1, 0);
        const int64_t nslot = (int64_t)t.slot_off.size();
        for (int64_t sl = 0; sl < nslot; ++sl)
            for (int32_t b = t.slot_row0[sl] / Rf; b * Rf < t.slot_row0[sl] + t.slot_rows[sl]; ++b) t.blk_ent_ptr[b + 1]++;
        for (int32_t b = 0; b < t.nblk; ++b) t.blk_ent_ptr[b + 1] += t.blk_ent_ptr[b];
        t.blk_ent_off.assign((size_t)t.blk_ent_ptr[t.nblk], 0);
        {
            std::vector<int32_t> cur(t.blk_ent_ptr.begin(), t.blk_ent_ptr.end() - 1);
            for (int64_t sl = 0; sl < nslot; ++sl)
                for (int32_t b = t.slot_row0[sl] / Rf; b * Rf < t.slot_row0[sl] + t.slot_rows[sl]; ++b)
                    t.blk_ent_off[cur[b]++] = t.slot_off[sl] + (t.blk_row0[b] - t.slot_row0[sl]);
        }
        for (const ResTile &D : t.tiles) {
            t.nent_pad += D.ne_pad;
            t.ngather_pad += D.ng_pad;
            t.nslab += D.nslab1 + D.nslab2;
        }
        if (std::getenv("EPHC_DEBUG")) {
            double nq = 0, bb = 0, br = 0, sm = 0;
            for (const ResTile &D : t.tiles) {
                sm += (double)res_tile_smem(D, nnu);
                nq += D.nq;
                bb += D.blob_bytes;
                br += D.b_rows;
            }
            {
                double mn = 1e30, mx = 0;
                for (int32_t cta = 0; cta < ncta; ++cta) {
                    double wk = 0;
                    for (int32_t i = t.cta_ptr[cta]; i < t.cta_ptr[cta + 1]; ++i)
                        wk += t.tiles[i].ne_pad + 0.4 * t.tiles[i].ng_pad + 45.0 * (t.tiles[i].nslab1 + t.tiles[i].nslab2) + 3.0 * t.tiles[i].nq + 600;
                    mn = std::min(mn, wk);
                    mx = std::max(mx, wk);
                }
                std::fprintf(stderr, "res schedule: %d CTAs, work %.0f .. %.0f\n", ncta, mn, mx);
            }
            std::fprintf(stderr, "res gathers (wavefronts per half-warp column, 1 = conflict-free; calibration tiles included): f_b %.3f, N %.3f, T %.3f\n",
                         (double)g_wf_f / std::max<long long>(g_wf_ideal1, 1), (double)g_wf_n / std::max<long long>(g_wf_ideal1, 1),
                         (double)g_wf_t / std::max<long long>(g_wf_ideal2, 1));
            g_wf_f = g_wf_n = g_wf_t = g_wf_ideal1 = g_wf_ideal2 = 0;
            const double n = (double)std::max<size_t>(t.tiles.size(), 1), ne = (double)std::max<int64_t>(nent, 1);
            std::fprintf(stderr,
                         "res store: Ra %d Rf %d RbMax %d budget %lld scale %.3f | %zu tiles in %zu runs, per tile: %.0f entries (+%.1f%% padding), "
                         "%.0f gathers (+%.1f%%), %.1f slabs, %.0f pairs, %.0f B rows, %.0f blob bytes (%.2f B/entry), smem avg %.0f max %lld, part rows %lld\n",
                         Ra, Rf, RbMax, (long long)budget, scale, t.tiles.size(), t.runs.size(), ne / n, 100.0 * (t.nent_pad - ne) / ne,
                         (double)t.ngather_pad / n, 100.0 * (t.ngather_pad - ne) / ne, (double)t.nslab / n, nq / n, br / n, bb / n, bb / ne,
                         sm / n, (long long)t.smem_tile, (long long)t.part_rows);
        }
    } catch (const std::bad_alloc &) {
        err = "host allocation failed (resident-tile store)";
        return EPHC_ENOMEM;
    }
    t.supported = true;
    return EPHC_OK;
}

// Re-cuts the static schedule: the tiles keep their storage order and images; the contiguous shares get new boundaries
// of equal cost (cost[i] per stored tile, e.g. cycles measured on the device), and what depends on the boundaries -- the
// runs (consecutive tiles of one strip inside a share), their flags, the partial-sum slots and the per-block slot
// lists of the finish kernel -- is rebuilt.  Order of additions: per state still fixed by the tables, so a handle is
// bit-reproducible from call to call; two handles with different boundaries group the partial sums differently.
int res_reschedule(ResHost &t, const std::vector<double> &cost, std::string &err) {
    const int64_t ntile = (int64_t)t.tiles.size();
    const int32_t ncta = t.ncta, Rf = t.rf;
    if ((int64_t)cost.size() != ntile || ncta < 1 || Rf < 1) {
        err = "internal: res_reschedule arguments";
        return EPHC_ESTATE;
    }
    try {
        double total = 0.0;
        for (double c : cost) total += std::max(c, 0.0);
        t.cta_ptr.assign((size_t)ncta + 1, 0);
        t.runs.clear();
        t.slot_off.clear();
        t.slot_row0.clear();
        t.slot_rows.clear();
        int64_t rows = 0;
        auto new_slot = [&](int32_t row0, int32_t nrows_) {
            const int32_t sl = (int32_t)t.slot_off.size();
            t.slot_off.push_back(rows);
            t.slot_row0.push_back(row0);
            t.slot_rows.push_back(nrows_);
            rows += nrows_;
            return sl;
        };
        int32_t cta = 0, cur_strip = -1;
        double done = 0.0;
        for (int64_t i = 0; i < ntile; ++i) {
            ResTile &D = t.tiles[i];
            const double wk = std::max(cost[i], 0.0);
            bool cut = false;
            while (cta + 1 < ncta && done + 0.5 * wk > total * (double)(cta + 1) / ncta) {
                ++cta;
                t.cta_ptr[cta] = (int32_t)i;
                cut = true;
            }
            if (cut || D.a_row0 != cur_strip || i == 0) {
                if (!t.runs.empty()) t.tiles[i - 1].flags |= 2;  // the previous tile was the last of its run
                t.runs.push_back(ResRun{(int32_t)i, 0, D.a_row0, D.a_rows, new_slot(D.a_row0, D.a_rows), cta});
                cur_strip = D.a_row0;
                D.flags = 1;
            } else {
                D.flags = 0;
            }
            ResRun &run = t.runs.back();
            run.nt++;
            D.a_slot = run.a_slot;
            D.a_off = (uint32_t)t.slot_off[run.a_slot];
            D.b_slot = -1;
            D.b_off = 0;
            if (D.b_rows > 0) {
                D.b_slot = new_slot(D.b_row0, D.b_rows);
                D.b_off = (uint32_t)t.slot_off[D.b_slot];
            }
            done += wk;
        }
        if (ntile > 0) t.tiles[ntile - 1].flags |= 2;
        while (cta + 1 <= ncta) t.cta_ptr[++cta] = (int32_t)ntile;  // shares left without tiles
        t.part_rows = rows;
        if (rows > 0xffffffffLL) {
            err = "resident-tile store: partial-sum buffer exceeds 2^32 rows";
            return EPHC_ELIMIT;
        }
        t.blk_ent_ptr.assign((size_t)t.nblk + 1, 0);
        const int64_t nslot = (int64_t)t.slot_off.size();
        for (int64_t sl = 0; sl < nslot; ++sl)
            for (int32_t b = t.slot_row0[sl] / Rf; b * Rf < t.slot_row0[sl] + t.slot_rows[sl]; ++b) t.blk_ent_ptr[b + 1]++;
        for (int32_t b = 0; b < t.nblk; ++b) t.blk_ent_ptr[b + 1] += t.blk_ent_ptr[b];
        t.blk_ent_off.assign((size_t)t.blk_ent_ptr[t.nblk], 0);
        std::vector<int32_t> cur(t.blk_ent_ptr.begin(), t.blk_ent_ptr.end() - 1);
        for (int64_t sl = 0; sl < nslot; ++sl)
            for (int32_t b = t.slot_row0[sl] / Rf; b * Rf < t.slot_row0[sl] + t.slot_rows[sl]; ++b)
                t.blk_ent_off[cur[b]++] = t.slot_off[sl] + (t.blk_row0[b] - t.slot_row0[sl]);
    } catch (const std::bad_alloc &) {
        err = "host allocation failed (resident-tile schedule)";
        return EPHC_ENOMEM;
    }
    return EPHC_OK;
}

}  // namespace ephc
