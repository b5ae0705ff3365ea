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

struct DEnt {          // directed entry: T = w F_em(f_out, f_in, N[iq, nu]); I[out] -= T; I[in] += T
    int32_t out, in;   // compact rows
    int32_t ip;        // candidate pair (-> iq)
    int32_t nu;
    double w;
};

struct Image {
    ResTile dir;
    std::vector<unsigned char> blob;
    std::vector<uint32_t> iqn;
    int64_t smem = 0;   // blob + X tail + N rows
    int64_t work = 0;
};

struct ImgParams {
    int32_t a_row0, a_rows, b_row0, b_rows;
    int nnu, nl;
    int qmul, lmul;     // longest piece / gather task in units of a lane's average load
    int32_t nq_cap;     // pairs per tile (bounds the iq list that rides in the previous tile's image)
    int64_t budget;     // bytes available for image (without that list) + X tail + N rows
    const int32_t *pair_iq;
};

struct Scratch {
    std::vector<int32_t> cnt, start, idx, pos_of, in_cnt, in_start, in_list;
    std::vector<uint32_t> pair_local;
};

struct Item {
    int32_t key, start, len;   // piece: out row / task: destination; first element; elements
};

// Column tables of a set of lists sorted by descending length: col[j] = (number of lists longer than j) | (first
// element of column j) << 16.
static void make_cols(const std::vector<int32_t> &lens_desc, std::vector<uint32_t> &cols, int32_t &ncol) {
    ncol = lens_desc.empty() ? 0 : lens_desc[0];
    cols.assign((size_t)ncol, 0);
    size_t n = lens_desc.size();
    int32_t base = 0;
    for (int32_t j = 0; j < ncol; ++j) {
        while (n > 0 && lens_desc[n - 1] <= j) --n;
        cols[j] = (uint32_t)n | ((uint32_t)base << 16);
        base += (int32_t)n;
    }
}

// Packs items into nl lanes of (almost) equal load, longest item first (every item goes to the lane with the least
// load so far); lanes are then sorted by descending load.  lanes[l] = the items of lane l in the order it walks them.
static void pack_lanes(const std::vector<Item> &items, int nl, std::vector<std::vector<int32_t>> &lanes,
                       std::vector<int32_t> &loads) {
    std::vector<int32_t> order(items.size());
    for (size_t i = 0; i < items.size(); ++i) order[i] = (int32_t)i;
    std::stable_sort(order.begin(), order.end(), [&](int32_t x, int32_t y) { return items[x].len > items[y].len; });
    std::vector<std::vector<int32_t>> bins((size_t)nl);
    std::vector<std::pair<int32_t, int32_t>> heap;  // (-load, -bin): the top is the least loaded, lowest bin
    for (int32_t b = 0; b < nl; ++b) heap.push_back({0, -b});
    std::make_heap(heap.begin(), heap.end());
    for (int32_t it : order) {
        std::pop_heap(heap.begin(), heap.end());
        auto top = heap.back();
        bins[(size_t)(-top.second)].push_back(it);
        heap.back() = {top.first - items[it].len, top.second};
        std::push_heap(heap.begin(), heap.end());
    }
    std::vector<int32_t> bl((size_t)nl, 0), bo((size_t)nl);
    for (int32_t b = 0; b < nl; ++b) {
        for (int32_t it : bins[b]) bl[b] += items[it].len;
        bo[b] = b;
    }
    std::stable_sort(bo.begin(), bo.end(), [&](int32_t x, int32_t y) { return bl[x] > bl[y]; });
    lanes.assign((size_t)nl, {});
    loads.assign((size_t)nl, 0);
    for (int32_t l = 0; l < nl; ++l) {
        lanes[l].swap(bins[bo[l]]);
        loads[l] = bl[bo[l]];
    }
}

// Builds the image of one tile from entries e[0..n) (sorted by pair).  Returns false when a format limit or the
// shared-memory budget is exceeded (the caller then splits the entry range).
static bool build_image(const DEnt *e, int64_t n, const ImgParams &P, Scratch &S, Image &out) {
    const int32_t R = P.a_rows + P.b_rows;
    const int nl = P.nl;
    if (n > kResXMax || R > kResRowMax) return false;
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
    // ---- phase 1: out rows -> pieces of at most ceil(n / nl) entries -> lanes ------------------------------------------
    S.cnt.assign((size_t)R + 1, 0);
    for (int64_t i = 0; i < n; ++i) S.cnt[loc(e[i].out) + 1]++;
    S.start.assign((size_t)R + 1, 0);
    for (int32_t r = 0; r < R; ++r) S.start[r + 1] = S.start[r] + S.cnt[r + 1];
    S.idx.resize((size_t)n);
    {
        std::vector<int32_t> &cur = S.cnt;  // reuse as cursor
        for (int32_t r = 0; r < R; ++r) cur[r] = S.start[r];
        for (int64_t i = 0; i < n; ++i) S.idx[cur[loc(e[i].out)]++] = (int32_t)i;
    }
    // inside an out row: by in row, so that the entries of one (out, in) combo (same rows, different modes) are adjacent
    for (int32_t r = 0; r < R; ++r)
        std::sort(S.idx.begin() + S.start[r], S.idx.begin() + S.start[r + 1], [&](int32_t x, int32_t y) {
            if (e[x].in != e[y].in) return e[x].in < e[y].in;
            return x < y;
        });
    const int32_t Q1 = (int32_t)std::max<int64_t>(1, P.qmul * ((n + nl - 1) / nl));
    std::vector<Item> pieces;
    for (int32_t r = 0; r < R; ++r) {
        const int32_t c = S.start[r + 1] - S.start[r];
        if (c == 0) continue;
        const int32_t npc = (c + Q1 - 1) / Q1, base = c / npc, rem = c % npc;
        int32_t s = S.start[r];
        for (int32_t k = 0; k < npc; ++k) {
            const int32_t len = base + (k < rem ? 1 : 0);
            pieces.push_back(Item{r, s, len});
            s += len;
        }
    }
    const int32_t npiece = (int32_t)pieces.size();
    std::vector<std::vector<int32_t>> lanes1, lanes2;
    std::vector<int32_t> loads1, loads2;
    pack_lanes(pieces, nl, lanes1, loads1);
    std::vector<uint32_t> cols1, cols2, cols3;
    int32_t nc1 = 0, nc2 = 0, nc3 = 0;
    make_cols(loads1, cols1, nc1);
    while (nc1 % 4) {  // the kernel reads four columns at a time
        cols1.push_back((uint32_t)n << 16);
        ++nc1;
    }
    // pieces are numbered in the order the lanes walk them; entry positions; END flags
    std::vector<int32_t> piece_no((size_t)npiece), pf((size_t)nl), prow((size_t)npiece + 4, 0);
    std::vector<uint8_t> is_end((size_t)n, 0);  // bit 0: last entry of its piece; bit 1: the next entry of the piece has the same in row
    S.pos_of.resize((size_t)n);
    {
        int32_t no = 0;
        for (int32_t l = 0; l < nl; ++l) {
            pf[l] = no;
            int32_t j = 0;
            for (int32_t ip : lanes1[l]) {
                piece_no[ip] = no;
                prow[no] = pieces[ip].key;
                ++no;
                for (int32_t k = 0; k < pieces[ip].len; ++k, ++j) {
                    const int32_t ei = S.idx[pieces[ip].start + k];
                    S.pos_of[ei] = (int32_t)(cols1[j] >> 16) + l;
                    if (k + 1 == pieces[ip].len)
                        is_end[ei] = 1;
                    else if (e[S.idx[pieces[ip].start + k + 1]].in == e[ei].in)
                        is_end[ei] = 2;
                }
            }
        }
    }
    // ---- phase 2: inputs of every row: positions of its in-entries (ascending), then of its out pieces --------------------
    S.in_cnt.assign((size_t)R + 1, 0);
    int32_t ncombo = 0;
    for (int64_t i = 0; i < n; ++i)
        if (!(is_end[i] & 2)) {  // the term of a combo sits at its last entry
            S.in_cnt[loc(e[i].in) + 1]++;
            ++ncombo;
        }
    for (int32_t p = 0; p < npiece; ++p) S.in_cnt[pieces[p].key + 1]++;
    S.in_start.assign((size_t)R + 1, 0);
    for (int32_t r = 0; r < R; ++r) S.in_start[r + 1] = S.in_start[r] + S.in_cnt[r + 1];
    S.in_list.resize((size_t)ncombo + npiece);
    int32_t nrow_in = 0;
    {
        std::vector<int32_t> &cur = S.in_cnt;
        for (int32_t r = 0; r < R; ++r) cur[r] = S.in_start[r];
        for (int64_t i = 0; i < n; ++i)
            if (!(is_end[i] & 2)) S.in_list[cur[loc(e[i].in)]++] = S.pos_of[i];
        for (int32_t r = 0; r < R; ++r) std::sort(S.in_list.begin() + S.in_start[r], S.in_list.begin() + cur[r]);
        for (int32_t p = 0; p < npiece; ++p) S.in_list[cur[pieces[p].key]++] = (int32_t)n + piece_no[p];
        for (int32_t r = 0; r < R; ++r) nrow_in += S.in_start[r + 1] > S.in_start[r];
    }
    // gather tasks: a row with at most Lcap inputs is one final task; longer rows are cut into partial tasks whose
    // sums a round-2 task adds
    const int32_t Lcap = (int32_t)std::max<int64_t>(2, P.lmul * (((int64_t)ncombo + npiece + nl - 1) / nl));
    std::vector<Item> t1, t2;
    std::vector<int32_t> list2;
    int32_t npart = 0;
    for (int32_t r = 0; r < R; ++r) {
        const int32_t L = S.in_start[r + 1] - S.in_start[r];
        if (L == 0) continue;
        if (L <= Lcap) {
            t1.push_back(Item{r, S.in_start[r], L});
            continue;
        }
        const int32_t nchunk = (L + Lcap - 1) / Lcap, base = L / nchunk, rem = L % nchunk;
        int32_t s = S.in_start[r];
        t2.push_back(Item{r, (int32_t)list2.size(), nchunk});
        for (int32_t k = 0; k < nchunk; ++k) {
            const int32_t len = base + (k < rem ? 1 : 0);
            t1.push_back(Item{0x8000 | npart, s, len});
            list2.push_back((int32_t)n + npiece + npart);
            ++npart;
            s += len;
        }
    }
    if (npart > 0x7fff || n + npiece + npart > kResXMax) return false;
    const int32_t ntask1 = (int32_t)t1.size(), ntask2 = (int32_t)t2.size();
    pack_lanes(t1, nl, lanes2, loads2);
    make_cols(loads2, cols2, nc2);
    while (nc2 % 4) {
        cols2.push_back((uint32_t)(ncombo + npiece) << 16);
        ++nc2;
    }
    std::stable_sort(t2.begin(), t2.end(), [](const Item &x, const Item &y) { return x.len > y.len; });
    {
        std::vector<int32_t> lens((size_t)ntask2);
        for (int32_t t = 0; t < ntask2; ++t) lens[t] = t2[t].len;
        make_cols(lens, cols3, nc3);
    }
    ResTile &D = out.dir;
    std::memset(&D, 0, sizeof(D));
    D.ne = (int32_t)n;
    D.npiece = npiece;
    D.npart = npart;
    D.ntask1 = ntask1;
    D.ntask2 = ntask2;
    D.nc1 = nc1;
    D.nc2 = nc2;
    D.nc3 = nc3;
    D.ngl1 = ncombo + npiece;
    D.ngl2 = (int32_t)list2.size();
    D.nq = nq;
    D.nq_next = 0;
    D.b_row0 = P.b_row0;
    D.b_rows = P.b_rows;
    D.b_slot = -1;
    res_set_layout(D, nl, P.nnu);
    out.smem = res_tile_smem(D, P.nnu);
    if (out.smem > P.budget) return false;
    // ---- fill the blob ---------------------------------------------------------------------------------------------
    out.blob.assign((size_t)D.blob_bytes, 0);
    uint32_t *code = reinterpret_cast<uint32_t *>(out.blob.data());
    uint16_t *perm = reinterpret_cast<uint16_t *>(out.blob.data() + D.o_perm);
    uint16_t *prow_o = reinterpret_cast<uint16_t *>(out.blob.data() + D.o_prow);
    uint16_t *pf_o = reinterpret_cast<uint16_t *>(out.blob.data() + D.o_pf);
    uint16_t *tf_o = reinterpret_cast<uint16_t *>(out.blob.data() + D.o_tf);
    uint16_t *d1 = reinterpret_cast<uint16_t *>(out.blob.data() + D.o_d1);
    uint16_t *d2 = reinterpret_cast<uint16_t *>(out.blob.data() + D.o_d2);
    uint32_t *cols = reinterpret_cast<uint32_t *>(out.blob.data() + D.o_cols);
    double *w = reinterpret_cast<double *>(out.blob.data() + D.o_w);
    for (int64_t i = 0; i < n; ++i) {
        const int32_t pos = S.pos_of[i];
        code[pos] = ((uint32_t)loc(e[i].in) << 3) | ((S.pair_local[i] * (uint32_t)P.nnu + (uint32_t)e[i].nu) << 19) | is_end[i];
        w[pos] = e[i].w;
    }
    for (int32_t p = 0; p < npiece + 4; ++p) prow_o[p] = (uint16_t)prow[p];  // four pad entries: the kernel reads three pieces ahead
    for (int32_t l = 0; l < nl; ++l) pf_o[l] = (uint16_t)pf[l];
    {
        int32_t no = 0;
        for (int32_t l = 0; l < nl; ++l) {
            tf_o[l] = (uint16_t)no;
            int32_t j = 0;
            for (int32_t it : lanes2[l]) {
                d1[no++] = (uint16_t)t1[it].key;
                for (int32_t k = 0; k < t1[it].len; ++k, ++j)
                    perm[(cols2[j] >> 16) + l] = (uint16_t)(S.in_list[t1[it].start + k] | (k + 1 == t1[it].len ? 0x8000 : 0));
            }
        }
    }
    for (int32_t t = 0; t < ntask2; ++t) {
        d2[t] = (uint16_t)t2[t].key;
        for (int32_t j = 0; j < t2[t].len; ++j) perm[D.ngl1 + (cols3[j] >> 16) + t] = (uint16_t)list2[t2[t].start + j];
    }
    std::copy(cols1.begin(), cols1.end(), cols);
    std::copy(cols2.begin(), cols2.end(), cols + nc1);
    std::copy(cols3.begin(), cols3.end(), cols + nc1 + nc2);
    // cost model of a tile for the shares (entries, row pieces / tasks, staged N rows, fixed)
    out.work = n + 2 * (int64_t)(npiece + ntask1 + ntask2) + 3 * (int64_t)nq + 600;
    (void)nrow_in;
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

int build_res(const ephc_problem *p, const Dims &d, const Canonical &c, int ncta, int64_t smem_cap, ResHost &t,
              std::string &err) {
    const int nb = d.nb, nnu = d.nnu;
    const int64_t npair = p->npair;
    t = ResHost();
    t.nnu = nnu;
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
        const int nl = kResLanes;
        const int qmul = std::max(1, env_int("EPHC_RES_QMUL", 1)), lmul = std::max(1, env_int("EPHC_RES_LMUL", 1));
        Ra = std::max(1, std::min(Ra, kResRowMax / 2));
        RbMax = std::max(1, std::min(RbMax, kResRowMax / 2));
        if (!std::getenv("EPHC_RES_ROWS")) {
            // small problems: enough strips that every CTA gets a few runs
            while (Ra > 16 && (int64_t)(t.nrows / Ra) * (t.nrows / Ra) < 8 * (int64_t)ncta) Ra /= 2;
        }
        // two tile buffers: f of the A and B rows, accumulators of the B rows, image + X tail + N rows; a tenth of what
        // is left may hold N rows of pairs, which bounds the next tile's iq list that an image carries
        const int64_t per_buf = (smem_cap - res_fixed_bytes(Ra)) / 2 - 8 * (int64_t)(Ra + RbMax) - 8 * (int64_t)RbMax - 256;
        const int32_t nq_cap = (int32_t)std::max<int64_t>(1, std::min<int64_t>(kResSlotMax / nnu, per_buf / (3 * 8 * (int64_t)nnu)));
        const int64_t budget = per_buf - 4 * (int64_t)nq_cap - 16;
        if (budget < 2048) {
            t.why = "resident-tile store: shared-memory budget too small";
            return EPHC_OK;
        }
        int Rf = env_int("EPHC_RES_FINE", 0);
        if (Rf <= 0) {
            // an atom (strip x fine block) should hold about a sixth of what fits in a tile
            const double rho = (double)std::max<int64_t>(nent, 1) / (0.5 * (double)t.nrows * (double)t.nrows + 1.0);
            const double per_row = std::max(1e-9, rho * Ra) * (14.5 + 8.0 * nnu / std::max(1.0, (double)nent / std::max<int64_t>(1, c.npair_active)));
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
            return 14 * E + 8 * (int64_t)nnu * Pq + 16 * std::min<int64_t>(rows_, 2 * E) + 16 * (int64_t)nl + 512;
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
                        // emission weight: out = a, in = b; absorption weight: out = b, in = a (F_abs(a,b) = -F_em(b,a))
                        if (c.ch_wem[j] != 0.0) ents[cur[it]++] = DEnt{a, b, (int32_t)ip, nu, c.ch_wem[j]};
                        if (c.ch_wabs[j] != 0.0) ents[cur[it]++] = DEnt{b, a, (int32_t)ip, nu, c.ch_wabs[j]};
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
                    P.nl = nl;
                    P.qmul = qmul;
                    P.lmul = lmul;
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
        for (int32_t cta = 0; cta < ncta; ++cta)
            for (int32_t i = t.cta_ptr[cta]; i + 1 < t.cta_ptr[cta + 1]; ++i) t.tiles[i].nq_next = t.tiles[i + 1].nq;
        for (int64_t i = 0; i < ntile; ++i) {
            ResTile &D = t.tiles[i];
            res_set_layout(D, nl, nnu);
            D.blob_off = boff;
            boff += (D.blob_bytes + 127) & ~127;
            t.smem_tile = std::max(t.smem_tile, res_tile_smem(D, nnu));
            t.Rcap = std::max(t.Rcap, D.a_rows + D.b_rows);
        }
        if (t.smem_tile > per_buf) {
            err = "internal: resident tile exceeds its shared-memory budget";
            return EPHC_ESTATE;
        }
        t.Rcap = (t.Rcap + 1) & ~1;
        t.RbMax = RbMax;
        t.nl = nl;
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
        for (int32_t cta = 0; cta < ncta; ++cta)  // the next tile's iq list rides in the image of its predecessor
            for (int32_t i = t.cta_ptr[cta]; i + 1 < t.cta_ptr[cta + 1]; ++i) {
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
        if (std::getenv("EPHC_DEBUG")) {
            double ne = 0, np = 0, nt1 = 0, nt2 = 0, nq = 0, bb = 0, br = 0, sm = 0;
            for (const ResTile &D : t.tiles) {
                sm += (double)res_tile_smem(D, nnu);
                ne += D.ne;
                np += D.npiece;
                nt1 += D.ntask1;
                nt2 += D.ntask2;
                nq += D.nq;
                bb += D.blob_bytes;
                br += D.b_rows;
            }
            {
                double mn = 1e30, mx = 0;
                for (int32_t cta = 0; cta < ncta; ++cta) {
                    double wk = 0;
                    for (int32_t i = t.cta_ptr[cta]; i < t.cta_ptr[cta + 1]; ++i)
                        wk += t.tiles[i].ne + 2.0 * (t.tiles[i].npiece + t.tiles[i].ntask1 + t.tiles[i].ntask2) + 3.0 * t.tiles[i].nq + 600;
                    mn = std::min(mn, wk);
                    mx = std::max(mx, wk);
                }
                std::fprintf(stderr, "res schedule: %d CTAs, work %.0f .. %.0f\n", ncta, mn, mx);
            }
            const double n = (double)std::max<size_t>(t.tiles.size(), 1);
            std::fprintf(stderr,
                         "res store: Ra %d Rf %d RbMax %d budget %lld scale %.3f | %zu tiles in %zu runs, per tile: %.0f entries, %.0f pieces, "
                         "%.0f + %.0f tasks, %.0f pairs, %.0f B rows, %.0f blob bytes (%.2f B/entry), smem avg %.0f max %lld, part rows %lld\n",
                         Ra, Rf, RbMax, (long long)budget, scale, t.tiles.size(), t.runs.size(), ne / n, np / n, nt1 / n, nt2 / n,
                         nq / n, br / n, bb / n, bb / std::max(ne, 1.0), sm / n, (long long)t.smem_tile, (long long)t.part_rows);
        }
    } catch (const std::bad_alloc &) {
        err = "host allocation failed (resident-tile store)";
        return EPHC_ENOMEM;
    }
    t.supported = true;
    return EPHC_OK;
}

}  // namespace ephc
