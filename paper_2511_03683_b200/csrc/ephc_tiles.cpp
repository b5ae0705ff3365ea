// ephc_tiles.cpp -- host side of the tile store (variant 1): every active channel is stored ONCE and both of its
// ends, I(n,k) and I(m,k+q), are updated from that one copy ("contributes to two elements of I ...
// equal in magnitude but opposite in sign").  This is the "transposed index over the mk+q side" of north_star
// folded into the layout itself: pairs are grouped into (k-block, k'-block) tiles so that both ends of every
// channel of a tile live in the shared memory of the CTA that walks the tile; see ephc_internal.h for the
// formats and DESIGN.md "Tile store" for the reasoning.  Performed once on the CPU.
//
// Product code: shares nothing with oracle/.
#include <algorithm>
#include <cmath>
#include <cstdlib>
#include <cstring>

#include "ephc_internal.h"

namespace ephc {

namespace {

struct Piece {      // one pair record before it is laid out
    int32_t ip;     // candidate pair
    int32_t first;  // first entry of the pair covered by this piece
    int32_t len;    // entries
};

struct Ent {
    uint16_t code;
    double w;
};

// entries of candidate pair ip in canonical order (nu, m, n), absorption before emission, then the diagonal
// (q = 0, n == m) terms; rank[] maps (k, band) to the compact band rank.
inline int pair_entries(const ephc_problem *p, const Dims &d, const Canonical &c, const uint8_t *rank, int64_t ip,
                        Ent *out) {
    const int nb = d.nb;
    const int32_t ik = p->pair_ik[ip], ikq = p->pair_ikq[ip];
    const uint8_t *ra = rank + (int64_t)ik * nb, *rb = rank + (int64_t)ikq * nb;
    int cnt = 0;
    for (int64_t j = c.pair_ch0[ip]; j < c.pair_ch0[ip + 1]; ++j) {
        const int n = c.ch_code[j] & 15, m = (c.ch_code[j] >> 4) & 15, nu = c.ch_code[j] >> 8;
        const uint16_t base = (uint16_t)(ra[n] | (rb[m] << kTcM) | (nu << kTcNu));
        if (c.ch_wabs[j] != 0.0) out[cnt++] = Ent{base, c.ch_wabs[j]};
        if (c.ch_wem[j] != 0.0) out[cnt++] = Ent{(uint16_t)(base | (1u << kTcKind)), c.ch_wem[j]};
    }
    for (int64_t j = c.pair_dg0[ip]; j < c.pair_dg0[ip + 1]; ++j) {
        const int n = c.dg_s[j] % nb, nu = c.dg_nu[j];
        const uint16_t base = (uint16_t)(ra[n] | (ra[n] << kTcM) | (nu << kTcNu) | (1u << kTcDiag));
        if (c.dg_wabs[j] != 0.0) out[cnt++] = Ent{base, c.dg_wabs[j]};
        if (c.dg_wem[j] != 0.0) out[cnt++] = Ent{(uint16_t)(base | (1u << kTcKind)), c.dg_wem[j]};
    }
    return cnt;
}

inline int pair_len(const Canonical &c, int64_t ip) {
    int cnt = 0;
    for (int64_t j = c.pair_ch0[ip]; j < c.pair_ch0[ip + 1]; ++j)
        cnt += (c.ch_wabs[j] != 0.0) + (c.ch_wem[j] != 0.0);
    for (int64_t j = c.pair_dg0[ip]; j < c.pair_dg0[ip + 1]; ++j)
        cnt += (c.dg_wabs[j] != 0.0) + (c.dg_wem[j] != 0.0);
    return cnt;
}

}  // namespace

int build_tiles(const ephc_problem *p, const Dims &d, const Canonical &c, int ncta, TileHost &t, std::string &err) {
    const int nb = d.nb, nnu = d.nnu;
    const int64_t npair = p->npair;
    t = TileHost();
    if (nb > kTileNbMax || nnu > kTileNnuMax) {
        t.why = "tile store handles nb <= 4 and nnu <= 8 in registers";
        return EPHC_OK;
    }
    if (d.nq > (1LL << 24)) {
        t.why = "tile store packs iq into 24 bits";
        return EPHC_OK;
    }
    if (ncta < 1) ncta = 1;
    try {
        // ---- compact rows: states inside the window (R-7), in state order -------------------------------------
        std::vector<uint8_t> rank((size_t)d.ns, 0), nin((size_t)d.nk, 0);
        std::vector<int32_t> krow0((size_t)d.nk + 1, 0);
        t.state_row.assign((size_t)d.ns, -1);
        t.state_blk.assign((size_t)d.ns, -1);
        for (int32_t k = 0; k < d.nk; ++k) {
            int r = 0;
            for (int n = 0; n < nb; ++n) {
                const int64_t s = (int64_t)k * nb + n;
                if (p->E[s] >= p->emin && p->E[s] <= p->emax) {
                    rank[s] = (uint8_t)r;
                    t.state_row[s] = krow0[k] + r;
                    ++r;
                }
            }
            nin[k] = (uint8_t)r;
            krow0[k + 1] = krow0[k] + r;
        }
        t.nrows = krow0[d.nk];
        t.row_state.resize((size_t)t.nrows);
        for (int64_t s = 0; s < d.ns; ++s)
            if (t.state_row[s] >= 0) t.row_state[t.state_row[s]] = (int32_t)s;

        // ---- blocks of <= R compact rows (whole k points) ---------------------------------------------------------
        // aim at ~8 tiles per CTA so that the contiguous partition below balances; R <= 1024 keeps the transport
        // kernel (4 arrays x R rows x 3 components x 8 B) at two CTAs per SM.
        int R = 1024;
        {
            const double nblk_t = std::sqrt(2.0 * 8.0 * ncta);
            const int r_bal = (int)std::ceil((double)std::max(t.nrows, 1) / nblk_t);
            R = std::max(std::min(R, r_bal), 32);
            if (const char *e = std::getenv("EPHC_TILE_ROWS")) R = std::max(nb, std::min(1536, std::atoi(e)));  // 1536: transport_iter fits 227 KB
            R = std::max(R, nb);
        }
        t.R = R;
        std::vector<int32_t> blk_of_k((size_t)d.nk, 0);
        t.blk_row0.assign(1, 0);
        {
            int rows = 0;
            for (int32_t k = 0; k < d.nk; ++k) {
                if (rows + nin[k] > R) {
                    t.blk_row0.push_back(krow0[k]);
                    rows = 0;
                }
                rows += nin[k];
                blk_of_k[k] = (int32_t)t.blk_row0.size() - 1;
            }
            t.blk_row0.push_back(krow0[d.nk]);
        }
        t.nblk = (int32_t)t.blk_row0.size() - 1;
        for (int64_t s = 0; s < d.ns; ++s)
            if (t.state_row[s] >= 0) t.state_blk[s] = blk_of_k[s / nb];
        const int64_t nblk = t.nblk;
        const int64_t ntile_all = nblk * (nblk + 1) / 2;
        auto tile_id = [&](int64_t I, int64_t J) { return I * nblk - I * (I - 1) / 2 + (J - I); };

        // ---- pieces per tile (canonical order inside a tile, then stable sort by length) ----------------------------
        std::vector<int32_t> plen((size_t)npair, 0);
#pragma omp parallel for schedule(dynamic, 4096)
        for (int64_t ip = 0; ip < npair; ++ip) plen[ip] = pair_len(c, ip);
        // a pair longer than piece_max entries is cut into pieces (separate pair records, consecutive tickets): the
        // longest slice bounds the idle tail of a tile
        int piece_max = 24;
        if (const char *e = std::getenv("EPHC_TILE_PIECE")) piece_max = std::atoi(e);
        piece_max = std::max(1, std::min(kTilePieceMax, piece_max));
        std::vector<int64_t> tile_p0((size_t)ntile_all + 1, 0);
        for (int64_t ip = 0; ip < npair; ++ip) {
            if (plen[ip] == 0) continue;
            const int64_t tid = tile_id(blk_of_k[p->pair_ik[ip]], blk_of_k[p->pair_ikq[ip]]);
            tile_p0[tid + 1] += (plen[ip] + piece_max - 1) / piece_max;
        }
        for (int64_t i = 0; i < ntile_all; ++i) tile_p0[i + 1] += tile_p0[i];
        const int64_t npiece = tile_p0[ntile_all];
        if (npiece > 0x7fffffffLL) {
            err = "more than 2^31-1 pair records";
            return EPHC_ELIMIT;
        }
        std::vector<Piece> pieces((size_t)npiece);
        {
            std::vector<int64_t> cur(tile_p0.begin(), tile_p0.end() - 1);
            for (int64_t ip = 0; ip < npair; ++ip) {
                if (plen[ip] == 0) continue;
                const int64_t tid = tile_id(blk_of_k[p->pair_ik[ip]], blk_of_k[p->pair_ikq[ip]]);
                for (int32_t f = 0; f < plen[ip]; f += piece_max)
                    pieces[cur[tid]++] = Piece{(int32_t)ip, f, std::min(piece_max, plen[ip] - f)};
            }
        }
        // non-empty tiles in row-major (I, J) order
        std::vector<int64_t> live;      // tile ids
        std::vector<int32_t> live_bi, live_bj;
        for (int64_t I = 0; I < nblk; ++I)
            for (int64_t J = I; J < nblk; ++J) {
                const int64_t tid = tile_id(I, J);
                if (tile_p0[tid + 1] > tile_p0[tid]) {
                    live.push_back(tid);
                    live_bi.push_back((int32_t)I);
                    live_bj.push_back((int32_t)J);
                }
            }
        const int64_t ntile = (int64_t)live.size();
        std::vector<int64_t> tile_e0((size_t)ntile + 1, 0), tile_s0((size_t)ntile + 1, 0), tile_r0((size_t)ntile + 1, 0);
#pragma omp parallel for schedule(dynamic, 8)
        for (int64_t it = 0; it < ntile; ++it) {
            Piece *b = pieces.data() + tile_p0[live[it]], *e = pieces.data() + tile_p0[live[it] + 1];
            // slices in ASCENDING length (a slice that starts earlier also ends earlier, so a lane rarely waits for
            // the ticket of a pair in an earlier slice); lanes of one slice in descending length (the active lanes
            // of every column are a prefix)
            std::stable_sort(b, e, [](const Piece &x, const Piece &y) { return x.len < y.len; });
            for (Piece *q = b; q < e; q += 32) std::reverse(q, std::min(q + 32, e));
            int64_t ne = 0;
            for (Piece *q = b; q != e; ++q) ne += q->len;
            tile_e0[it + 1] = ne;
            tile_r0[it + 1] = e - b;
            tile_s0[it + 1] = ((e - b) + 31) / 32;
        }
        for (int64_t it = 0; it < ntile; ++it) {
            tile_e0[it + 1] += tile_e0[it];
            tile_s0[it + 1] += tile_s0[it];
            tile_r0[it + 1] += tile_r0[it];
        }
        const int64_t nent = tile_e0[ntile], nslice = tile_s0[ntile];
        if (nslice > 0x7fffffffLL) {
            err = "more than 2^31-1 slices";
            return EPHC_ELIMIT;
        }
        t.npiece = npiece;
        t.w.resize((size_t)nent);
        t.code.resize((size_t)nent);
        t.prec.resize((size_t)npiece * 3);
        t.slices.resize((size_t)nslice);
        t.tiles.resize((size_t)ntile);

        // ---- fill: slices, pair records with tickets, entries column-major per slice ---------------------------------
        int over = 0;
#pragma omp parallel reduction(| : over)
        {
            std::vector<Ent> buf((size_t)2 * nnu * nb * nb + 4 * nnu * nb + 8);
            std::vector<int32_t> tick_a((size_t)R), tick_b((size_t)R);
#pragma omp for schedule(dynamic, 4)
            for (int64_t it = 0; it < ntile; ++it) {
                const int32_t bi = live_bi[it], bj = live_bj[it];
                const bool dg = (bi == bj);
                std::fill(tick_a.begin(), tick_a.end(), 0);
                std::fill(tick_b.begin(), tick_b.end(), 0);
                std::vector<int32_t> &tb = dg ? tick_a : tick_b;
                const Piece *pc = pieces.data() + tile_p0[live[it]];
                const int64_t np_t = tile_r0[it + 1] - tile_r0[it];
                int64_t e0 = tile_e0[it];
                TileHdr &th = t.tiles[it];
                th.s0 = (int32_t)tile_s0[it];
                th.ns = (int32_t)(tile_s0[it + 1] - tile_s0[it]);
                th.bi = bi;
                th.bj = bj;
                th.a_slot = th.b_slot = -1;
                th.flags = 0;
                th.pad = 0;
                for (int64_t s = 0; s < th.ns; ++s) {
                    const int64_t q0 = s * 32;
                    const int np_s = (int)std::min<int64_t>(32, np_t - q0);
                    TileSlice &sl = t.slices[th.s0 + s];
                    sl.e0 = e0;
                    sl.p0 = (int32_t)(tile_r0[it] + q0);
                    sl.np = (int16_t)np_s;
                    sl.maxlen = (int16_t)pc[q0].len;
                    // column offsets: cnt_i lanes have more than i entries (a prefix, lengths descend)
                    int colstart[kTilePieceMax + 1];
                    {
                        int off = 0, cnt = np_s;
                        for (int i = 0; i < sl.maxlen; ++i) {
                            while (cnt > 0 && pc[q0 + cnt - 1].len <= i) --cnt;
                            colstart[i] = off;
                            off += cnt;
                        }
                        colstart[sl.maxlen] = off;
                    }
                    for (int l = 0; l < np_s; ++l) {
                        const Piece &pp = pc[q0 + l];
                        const int32_t ik = p->pair_ik[pp.ip], ikq = p->pair_ikq[pp.ip];
                        const int32_t ra = krow0[ik] - t.blk_row0[bi], rb = krow0[ikq] - t.blk_row0[bj];
                        const int32_t ta = tick_a[ra]++;
                        const int32_t tbk = tb[rb]++;
                        if (ta > kTileTicketMax || tbk > kTileTicketMax) over = 1;
                        uint32_t *rec = t.prec.data() + (size_t)(sl.p0 + l);  // structure of arrays: [3][npiece]
                        rec[0] = (uint32_t)ra | ((uint32_t)rb << 16);
                        rec[npiece] = (uint32_t)c.pair_iq[pp.ip] | ((uint32_t)pp.len << 24);
                        rec[2 * npiece] = (uint32_t)(ta & 0xfff) | ((uint32_t)(nin[ik] - 1) << 12) |
                                          ((uint32_t)(tbk & 0xfff) << 16) | ((uint32_t)(nin[ikq] - 1) << 28);
                        const int cnt = pair_entries(p, d, c, rank.data(), pp.ip, buf.data());
                        (void)cnt;
                        for (int i = 0; i < pp.len; ++i) {
                            const int64_t o = e0 + colstart[i] + l;
                            t.code[o] = buf[pp.first + i].code;
                            t.w[o] = buf[pp.first + i].w;
                        }
                    }
                    e0 += colstart[sl.maxlen];
                }
            }
        }
        if (over) {
            t = TileHost();
            t.why = "more than 4096 pair records of one k point in a tile";
            return EPHC_OK;
        }

        // ---- contiguous partition of the tile sequence over the CTAs, balanced by work ----------------------------------
        t.ncta = ncta;
        t.ctas.assign((size_t)ncta, TileCta{0, 0});
        {
            std::vector<double> work((size_t)ntile);
            double total = 0.0;
            for (int64_t it = 0; it < ntile; ++it) {
                work[it] = (double)(tile_e0[it + 1] - tile_e0[it]) + 8.0 * (double)(tile_r0[it + 1] - tile_r0[it]) + 256.0;
                total += work[it];
            }
            double acc = 0.0;
            int64_t it = 0;
            for (int cta = 0; cta < ncta; ++cta) {
                const double goal = total * (double)(cta + 1) / (double)ncta;
                t.ctas[cta].t0 = (int32_t)it;
                while (it < ntile && (cta == ncta - 1 || acc + 0.5 * work[it] <= goal)) acc += work[it++];
                t.ctas[cta].t1 = (int32_t)it;
            }
        }
        // ---- partial-sum slots: one per a-run (consecutive tiles of a CTA with the same block I) and one per
        //      off-diagonal tile for block J; per block the list of its slots in a fixed order -----------------------------
        std::vector<std::pair<int32_t, int32_t>> bs;  // (block, slot)
        t.slot_off.clear();
        int64_t rows = 0;
        auto new_slot = [&](int32_t blk) {
            const int32_t sl = (int32_t)t.slot_off.size();
            t.slot_off.push_back(rows);
            rows += t.blk_row0[blk + 1] - t.blk_row0[blk];
            bs.emplace_back(blk, sl);
            return sl;
        };
        for (int cta = 0; cta < ncta; ++cta)
            for (int32_t it = t.ctas[cta].t0; it < t.ctas[cta].t1; ++it) {
                TileHdr &th = t.tiles[it];
                const bool first = (it == t.ctas[cta].t0) || (t.tiles[it - 1].bi != th.bi);
                const bool last = (it + 1 == t.ctas[cta].t1) || (t.tiles[it + 1].bi != th.bi);
                th.a_slot = first ? new_slot(th.bi) : t.tiles[it - 1].a_slot;
                th.flags = (first ? 1 : 0) | (last ? 2 : 0);
                th.b_slot = (th.bi != th.bj) ? new_slot(th.bj) : -1;
            }
        t.part_rows = rows;
        std::stable_sort(bs.begin(), bs.end(), [](const std::pair<int32_t, int32_t> &x, const std::pair<int32_t, int32_t> &y) {
            return x.first < y.first;
        });
        t.blk_slot_ptr.assign((size_t)t.nblk + 1, 0);
        t.blk_slots.resize(bs.size());
        for (size_t i = 0; i < bs.size(); ++i) {
            t.blk_slot_ptr[bs[i].first + 1]++;
            t.blk_slots[i] = bs[i].second;
        }
        for (int32_t b = 0; b < t.nblk; ++b) t.blk_slot_ptr[b + 1] += t.blk_slot_ptr[b];
    } catch (const std::bad_alloc &) {
        err = "host allocation failed (tile store)";
        return EPHC_ENOMEM;
    }
    t.supported = true;
    return EPHC_OK;
}

}  // namespace ephc
