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

        // ---- fine blocks (whole k points, <= Rf rows) and strips of fine blocks (<= Ra rows) ---------------------------
        // Ra, Rb: rows of the k side / k' side a tile may span.  Defaults keep the collision kernel (4 x 8 B per row,
        // 48 KB of per-thread rows) at two CTAs per SM and the transport kernel (4 x 24 B per row) at one.
        int Ra = 1536, Rb = 1536, Rf = 128;
        if (const char *e = std::getenv("EPHC_TILE_ROWS")) Ra = Rb = std::atoi(e);
        if (const char *e = std::getenv("EPHC_TILE_ROWS_B")) Rb = std::atoi(e);
        if (const char *e = std::getenv("EPHC_TILE_FINE")) Rf = std::atoi(e);
        Ra = std::max(nb, std::min(1536, Ra));
        Rb = std::max(nb, std::min(1536, Rb));
        // small problems: keep at least ~4 fine column blocks per CTA share so that the partition can balance
        {
            const double want = std::sqrt((double)std::max(t.nrows, 1) * (double)std::max(t.nrows, 1) / (8.0 * ncta));
            Rf = std::min(Rf, std::max(nb, (int)want));
        }
        Rf = std::max(nb, std::min(Rf, std::min(Ra, Rb)));
        std::vector<int32_t> blk_of_k((size_t)d.nk, 0);
        t.blk_row0.assign(1, 0);
        {
            int rows = 0;
            for (int32_t k = 0; k < d.nk; ++k) {
                if (rows + nin[k] > Rf) {
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
        const int32_t nblk = t.nblk;
        std::vector<int32_t> strip_b0(1, 0), strip_of_blk((size_t)nblk, 0);  // strip -> first fine block
        for (int32_t b = 0; b < nblk; ++b) {
            if (t.blk_row0[b + 1] - t.blk_row0[strip_b0.back()] > Ra) strip_b0.push_back(b);
            strip_of_blk[b] = (int32_t)strip_b0.size() - 1;
        }
        strip_b0.push_back(nblk);
        const int32_t nstrip = (int32_t)strip_b0.size() - 1;
        // atoms in row-major order: (strip I, diagonal), then (strip I, fine block j) for every j after the strip
        std::vector<int64_t> atom0((size_t)nstrip + 1, 0);
        for (int32_t I = 0; I < nstrip; ++I) atom0[I + 1] = atom0[I] + 1 + (nblk - strip_b0[I + 1]);
        const int64_t natom = atom0[nstrip];
        auto atom_of = [&](int32_t ik, int32_t ikq) {
            const int32_t I = strip_of_blk[blk_of_k[ik]], j = blk_of_k[ikq];
            return (j < strip_b0[I + 1]) ? atom0[I] : atom0[I] + 1 + (j - strip_b0[I + 1]);
        };

        // ---- pair records ("pieces") and work per atom ---------------------------------------------------------------
        std::vector<int32_t> plen((size_t)npair, 0);
#pragma omp parallel for schedule(dynamic, 4096)
        for (int64_t ip = 0; ip < npair; ++ip) plen[ip] = pair_len(c, ip);
        // a pair longer than piece_max entries is cut into pieces (separate pair records, consecutive tickets): the
        // longest slice bounds the idle tail of a tile
        int piece_max = 24;
        if (const char *e = std::getenv("EPHC_TILE_PIECE")) piece_max = std::atoi(e);
        piece_max = std::max(1, std::min(kTilePieceMax, piece_max));
        std::vector<int64_t> atom_np((size_t)natom + 1, 0);
        std::vector<double> atom_work((size_t)natom, 0.0);
        for (int64_t ip = 0; ip < npair; ++ip) {
            if (plen[ip] == 0) continue;
            const int64_t at = atom_of(p->pair_ik[ip], p->pair_ikq[ip]);
            const int64_t np_ = (plen[ip] + piece_max - 1) / piece_max;
            atom_np[at + 1] += np_;
            atom_work[at] += (double)plen[ip] + 12.0 * (double)np_;
        }
        for (int64_t i = 0; i < natom; ++i) atom_np[i + 1] += atom_np[i];
        const int64_t npiece = atom_np[natom];
        if (npiece > 0x7fffffffLL) {
            err = "more than 2^31-1 pair records";
            return EPHC_ELIMIT;
        }
        // ---- contiguous partition of the atom sequence over the CTAs, balanced by work; inside a CTA's share,
        //      consecutive atoms of one strip merge into tiles of <= Rb rows on the k' side ----------------------------------
        t.ncta = ncta;
        t.ctas.assign((size_t)ncta, TileCta{0, 0});
        std::vector<int64_t> tile_at0, tile_at1;  // atom range of a tile
        std::vector<int32_t> tile_strip;
        {
            double total = 0.0;
            for (double wv : atom_work) total += wv;
            double acc = 0.0;
            int64_t at = 0;
            for (int cta = 0; cta < ncta; ++cta) {
                const double goal = total * (double)(cta + 1) / (double)ncta;
                t.ctas[cta].t0 = (int32_t)tile_at0.size();
                const int64_t first = at;
                while (at < natom && (cta == ncta - 1 || acc + 0.5 * atom_work[at] <= goal)) acc += atom_work[at++];
                // tiles of [first, at)
                int64_t a0 = first;
                while (a0 < at) {
                    if (atom_np[a0 + 1] == atom_np[a0]) {  // empty atom
                        ++a0;
                        continue;
                    }
                    const int32_t I = (int32_t)(std::upper_bound(atom0.begin(), atom0.end(), a0) - atom0.begin()) - 1;
                    int64_t a1 = a0 + 1;
                    if (a0 != atom0[I]) {  // off-diagonal: extend over following fine blocks of the same strip
                        const int32_t j0 = strip_b0[I + 1] + (int32_t)(a0 - atom0[I] - 1);
                        while (a1 < at && a1 < atom0[I + 1]) {
                            const int32_t j1 = strip_b0[I + 1] + (int32_t)(a1 - atom0[I] - 1);
                            if (t.blk_row0[j1 + 1] - t.blk_row0[j0] > Rb) break;
                            ++a1;
                        }
                        while (a1 - 1 > a0 && atom_np[a1] == atom_np[a1 - 1]) --a1;  // drop empty atoms at the end
                    }
                    tile_at0.push_back(a0);
                    tile_at1.push_back(a1);
                    tile_strip.push_back(I);
                    a0 = a1;
                }
                t.ctas[cta].t1 = (int32_t)tile_at0.size();
            }
        }
        const int64_t ntile = (int64_t)tile_at0.size();
        t.tiles.resize((size_t)ntile);
        std::vector<int64_t> tile_p0((size_t)ntile + 1, 0);
        std::vector<int32_t> atom_tile((size_t)natom, -1);
        t.Ra = t.Rb = nb;
        for (int64_t it = 0; it < ntile; ++it) {
            TileHdr &th = t.tiles[it];
            const int32_t I = tile_strip[it];
            const bool dg = (tile_at0[it] == atom0[I]);
            th.a_row0 = t.blk_row0[strip_b0[I]];
            th.a_rows = t.blk_row0[strip_b0[I + 1]] - th.a_row0;
            if (dg) {
                th.b_row0 = th.a_row0;
                th.b_rows = th.a_rows;
            } else {
                const int32_t j0 = strip_b0[I + 1] + (int32_t)(tile_at0[it] - atom0[I] - 1);
                const int32_t j1 = strip_b0[I + 1] + (int32_t)(tile_at1[it] - 1 - atom0[I] - 1);
                th.b_row0 = t.blk_row0[j0];
                th.b_rows = t.blk_row0[j1 + 1] - th.b_row0;
            }
            th.flags = dg ? 4 : 0;
            th.a_slot = th.b_slot = -1;
            th.pad = 0;
            t.Ra = std::max(t.Ra, th.a_rows);
            t.Rb = std::max(t.Rb, th.b_rows);
            for (int64_t at = tile_at0[it]; at < tile_at1[it]; ++at) atom_tile[at] = (int32_t)it;
            tile_p0[it + 1] = tile_p0[it] + (atom_np[tile_at1[it]] - atom_np[tile_at0[it]]);
        }
        // bucket the pieces by tile, canonical order inside a tile
        std::vector<Piece> pieces((size_t)npiece);
        {
            std::vector<int64_t> cur(tile_p0.begin(), tile_p0.end() - 1);
            for (int64_t ip = 0; ip < npair; ++ip) {
                if (plen[ip] == 0) continue;
                const int64_t it = atom_tile[atom_of(p->pair_ik[ip], p->pair_ikq[ip])];
                for (int32_t f = 0; f < plen[ip]; f += piece_max)
                    pieces[cur[it]++] = Piece{(int32_t)ip, f, std::min(piece_max, plen[ip] - f)};
            }
        }
        std::vector<int64_t> tile_e0((size_t)ntile + 1, 0), tile_s0((size_t)ntile + 1, 0);
        const std::vector<int64_t> &tile_r0 = tile_p0;
#pragma omp parallel for schedule(dynamic, 8)
        for (int64_t it = 0; it < ntile; ++it) {
            Piece *b = pieces.data() + tile_p0[it], *e = pieces.data() + tile_p0[it + 1];
            // slices in ASCENDING length (a slice that starts earlier also ends earlier, so a lane rarely waits for
            // the ticket of a pair in an earlier slice); lanes of one slice in descending length (the active lanes
            // of every column are a prefix)
            std::stable_sort(b, e, [](const Piece &x, const Piece &y) { return x.len < y.len; });
            for (Piece *q = b; q < e; q += 32) std::reverse(q, std::min(q + 32, e));
            int64_t ne = 0;
            for (Piece *q = b; q != e; ++q) ne += q->len;
            tile_e0[it + 1] = ne;
            tile_s0[it + 1] = ((e - b) + 31) / 32;
        }
        for (int64_t it = 0; it < ntile; ++it) {
            tile_e0[it + 1] += tile_e0[it];
            tile_s0[it + 1] += tile_s0[it];
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

        // ---- fill: slices, pair records with tickets, entries column-major per slice ---------------------------------
        // Tickets count the pair records of one k point on one side; on the k side they run on through all tiles
        // of an a-run (the accumulators of the strip stay in shared memory), on the k' side they restart per tile.
        std::vector<uint8_t> run_first((size_t)ntile, 0), run_last((size_t)ntile, 0);
        for (int cta = 0; cta < ncta; ++cta)
            for (int32_t it = t.ctas[cta].t0; it < t.ctas[cta].t1; ++it) {
                run_first[it] = (it == t.ctas[cta].t0) || (tile_strip[it - 1] != tile_strip[it]);
                run_last[it] = (it + 1 == t.ctas[cta].t1) || (tile_strip[it + 1] != tile_strip[it]);
            }
        std::vector<int64_t> runs;  // first tile of every a-run
        for (int64_t it = 0; it < ntile; ++it)
            if (run_first[it]) runs.push_back(it);
        runs.push_back(ntile);
        const int64_t nruns = (int64_t)runs.size() - 1;
        int over = 0;
#pragma omp parallel reduction(| : over)
        {
            std::vector<Ent> buf((size_t)2 * nnu * nb * nb + 4 * nnu * nb + 8);
            std::vector<int32_t> tick_a((size_t)t.Ra), tick_b((size_t)t.Rb);
#pragma omp for schedule(dynamic, 1)
            for (int64_t ir = 0; ir < nruns; ++ir) {
                std::fill(tick_a.begin(), tick_a.end(), 0);
                for (int64_t it = runs[ir]; it < runs[ir + 1]; ++it) {
                    TileHdr &th = t.tiles[it];
                    const bool dg = (th.flags & 4) != 0;
                    std::fill(tick_b.begin(), tick_b.end(), 0);
                    std::vector<int32_t> &tb = dg ? tick_a : tick_b;
                    const Piece *pc = pieces.data() + tile_p0[it];
                    const int64_t np_t = tile_r0[it + 1] - tile_r0[it];
                    int64_t e0 = tile_e0[it];
                    th.p0 = (int32_t)tile_r0[it];
                    th.npc = (int32_t)np_t;
                    th.s0 = (int32_t)tile_s0[it];
                    th.ns = (int32_t)(tile_s0[it + 1] - tile_s0[it]);
                    th.flags |= (run_first[it] ? 1 : 0) | (run_last[it] ? 2 : 0);
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
                            const int32_t ra = krow0[ik] - th.a_row0, rb = krow0[ikq] - th.b_row0;
                            const int32_t ta = tick_a[ra]++;
                            const int32_t tbk = tb[rb]++;
                            if (ta > kTileTicketMax || tbk > kTileTicketMax) over = 1;
                            uint32_t *rec = t.prec.data() + (size_t)(sl.p0 + l);  // structure of arrays: [3][npiece]
                            rec[0] = (uint32_t)ra | ((uint32_t)rb << 16);
                            rec[npiece] = (uint32_t)c.pair_iq[pp.ip] | ((uint32_t)pp.len << 24);
                            rec[2 * npiece] = (uint32_t)(ta & 0xfff) | ((uint32_t)(nin[ik] - 1) << 12) |
                                              ((uint32_t)(tbk & 0xfff) << 16) | ((uint32_t)(nin[ikq] - 1) << 28);
                            pair_entries(p, d, c, rank.data(), pp.ip, buf.data());
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
        }
        if (over) {
            t = TileHost();
            t.why = "more than 4096 pair records of one k point in a run of tiles";
            return EPHC_OK;
        }

        // ---- partial-sum slots: one per a-run (rows of the strip) and one per off-diagonal tile (its k' rows);
        //      per fine block the list of the slots that cover it, in a fixed order -------------------------------------
        t.slot_off.clear();
        int64_t rows = 0;
        auto new_slot = [&](int32_t row0, int32_t nrows) {
            const int32_t sl = (int32_t)t.slot_off.size();
            t.slot_off.push_back(rows);
            t.slot_row0.push_back(row0);
            t.slot_rows.push_back(nrows);
            rows += nrows;
            return sl;
        };
        for (int64_t it = 0; it < ntile; ++it) {
            TileHdr &th = t.tiles[it];
            th.a_slot = (th.flags & 1) ? new_slot(th.a_row0, th.a_rows) : t.tiles[it - 1].a_slot;
            th.b_slot = (th.flags & 4) ? -1 : new_slot(th.b_row0, th.b_rows);
        }
        t.part_rows = rows;
        {
            std::vector<int32_t> blk_of_row0;  // fine block whose first row is a given row: by binary search
            t.blk_ent_ptr.assign((size_t)t.nblk + 1, 0);
            const int64_t nslot = (int64_t)t.slot_off.size();
            auto blk_range = [&](int64_t sl, int32_t &b0, int32_t &b1) {
                b0 = (int32_t)(std::lower_bound(t.blk_row0.begin(), t.blk_row0.end(), t.slot_row0[sl]) - t.blk_row0.begin());
                b1 = (int32_t)(std::lower_bound(t.blk_row0.begin(), t.blk_row0.end(), t.slot_row0[sl] + t.slot_rows[sl]) -
                               t.blk_row0.begin());
            };
            for (int64_t sl = 0; sl < nslot; ++sl) {
                int32_t b0, b1;
                blk_range(sl, b0, b1);
                for (int32_t b = b0; b < b1; ++b) t.blk_ent_ptr[b + 1]++;
            }
            for (int32_t b = 0; b < t.nblk; ++b) t.blk_ent_ptr[b + 1] += t.blk_ent_ptr[b];
            t.blk_ent_off.assign((size_t)t.blk_ent_ptr[t.nblk], 0);
            std::vector<int32_t> cur(t.blk_ent_ptr.begin(), t.blk_ent_ptr.end() - 1);
            for (int64_t sl = 0; sl < nslot; ++sl) {
                int32_t b0, b1;
                blk_range(sl, b0, b1);
                for (int32_t b = b0; b < b1; ++b)
                    t.blk_ent_off[cur[b]++] = t.slot_off[sl] + (t.blk_row0[b] - t.slot_row0[sl]);
            }
        }
    } catch (const std::bad_alloc &) {
        err = "host allocation failed (tile store)";
        return EPHC_ENOMEM;
    }
    t.supported = true;
    return EPHC_OK;
}

}  // namespace ephc
