// ephc_stream.cpp -- host side of the stream store (variant 2): once-stored channels, one lane per entry, tile-local
// reductions for both ends (see ephc_internal.h "stream store" and DESIGN.md).  Performed once on the CPU
// (PAPER.md:94).  The diagonal (q = 0, n == m) terms are left out: they contribute exactly 0 to the collision
// integral and this store is used by ephc_collision / ephc_rt_step only.
//
// Product code: shares nothing with oracle/.
#include <algorithm>
#include <cmath>
#include <cstdio>
#include <cstdlib>

#include "ephc_internal.h"

namespace ephc {

namespace {
struct SEnt {
    int32_t a, b;      // compact rows, a < b
    int32_t ip;        // candidate pair (-> iq)
    uint16_t nu, kind;
    double w;
};
}  // namespace

int build_stream(const ephc_problem *p, const Dims &d, const Canonical &c, int ncta, StreamHost &t, std::string &err) {
    const int nb = d.nb, nnu = d.nnu;
    const int64_t npair = p->npair;
    t = StreamHost();
    if (nnu > 64 || c.nw > 0x7fffffffLL) {
        t.why = "stream store: nnu <= 64 and fewer than 2^31 weights";
        return EPHC_OK;
    }
    if (ncta < 1) ncta = 1;
    try {
        // compact rows (states inside the window, R-7)
        t.state_row.assign((size_t)d.ns, -1);
        for (int64_t s = 0; s < d.ns; ++s)
            if (p->E[s] >= p->emin && p->E[s] <= p->emax) {
                t.state_row[s] = (int32_t)t.row_state.size();
                t.row_state.push_back((int32_t)s);
            }
        t.nrows = (int32_t)t.row_state.size();
        // fine blocks of Rf rows, strips of Ra rows (multiples of Rf), k' ranges of <= Rb rows
        int Rf = 128, Ra = 1024, Rb = 1536;
        if (const char *e = std::getenv("EPHC_STREAM_FINE")) Rf = std::atoi(e);
        if (const char *e = std::getenv("EPHC_STREAM_ROWS")) Ra = std::atoi(e);
        if (const char *e = std::getenv("EPHC_STREAM_ROWS_B")) Rb = std::atoi(e);
        {
            const double want = std::sqrt((double)std::max(t.nrows, 1) * (double)std::max(t.nrows, 1) / (8.0 * ncta));
            Rf = std::min(Rf, std::max(1, (int)want));
        }
        Rf = std::max(1, Rf);
        if (!std::getenv("EPHC_STREAM_ROWS")) {
            // small problems: enough strips for a few tiles per CTA (about nstrip^2 / 2 x fine blocks per strip tiles)
            const int ra_small = (int)((double)std::max(t.nrows, 1) / std::sqrt(2.0 * ncta * 3.0)) * 8;
            Ra = std::min(Ra, std::max(Rf, ra_small));
        }
        Ra = std::max(Rf, std::min(2048, Ra) / Rf * Rf);
        Rb = std::max(Rf, std::min(kStreamRbMax, Rb) / Rf * Rf);
        t.rf = Rf;
        t.nblk = std::max(1, (t.nrows + Rf - 1) / Rf);
        t.blk_row0.resize((size_t)t.nblk + 1);
        for (int32_t b = 0; b <= t.nblk; ++b) t.blk_row0[b] = std::min(t.nrows, b * Rf);
        t.state_blk.assign((size_t)d.ns, -1);
        for (int64_t s = 0; s < d.ns; ++s)
            if (t.state_row[s] >= 0) t.state_blk[s] = t.state_row[s] / Rf;
        const int32_t bps = Ra / Rf;  // fine blocks per strip
        const int32_t nstrip = (t.nblk + bps - 1) / bps;
        std::vector<int64_t> atom0((size_t)nstrip + 1, 0);  // atoms of strip I: diagonal, then fine blocks after it
        for (int32_t I = 0; I < nstrip; ++I) atom0[I + 1] = atom0[I] + 1 + std::max(0, t.nblk - (I + 1) * bps);
        const int64_t natom = atom0[nstrip];
        auto atom_of = [&](int32_t a, int32_t b) {
            const int32_t I = a / Ra, j = b / Rf;
            return (j < (I + 1) * bps) ? atom0[I] : atom0[I] + 1 + (j - (I + 1) * bps);
        };
        // entries and work per atom
        // work of an atom: its entries plus a per-pair cost (N[iq,:] staging, chunks cut by the slot limit)
        int pair_cost = 4;  // measured on B200 (Si workload): 0 -> 155 us, 4 -> 141 us, 8 -> 146 us
        if (const char *e = std::getenv("EPHC_STREAM_PAIR_COST")) pair_cost = std::max(0, std::atoi(e));
        std::vector<int64_t> atom_ne((size_t)natom + 1, 0), atom_wk((size_t)natom + 1, 0);
        for (int64_t ip = 0; ip < npair; ++ip) {
            const int64_t sa = (int64_t)p->pair_ik[ip] * nb, sb = (int64_t)p->pair_ikq[ip] * nb;
            for (int64_t j = c.pair_ch0[ip]; j < c.pair_ch0[ip + 1]; ++j) {
                const int n = c.ch_code[j] & 15, m = (c.ch_code[j] >> 4) & 15;
                const int64_t at = atom_of(t.state_row[sa + n], t.state_row[sb + m]);
                const int ne = (c.ch_wabs[j] != 0.0) + (c.ch_wem[j] != 0.0);
                atom_ne[at + 1] += ne;
                atom_wk[at + 1] += ne + (j == c.pair_ch0[ip] ? pair_cost : 0);
            }
        }
        for (int64_t i = 0; i < natom; ++i) {
            atom_ne[i + 1] += atom_ne[i];
            atom_wk[i + 1] += atom_wk[i];
        }
        const int64_t nent = atom_ne[natom], nwork = atom_wk[natom];
        // contiguous shares of equal work; tiles = consecutive atoms of one strip inside a share, <= Rb rows
        // Tiles are cut so that a CTA gets about `tiles_per_cta` of them; the kernel hands them out dynamically,
        // largest first (t.order), so every tile is self-contained (own partial-sum slots for both row ranges).
        int tiles_per_cta = 3;
        if (const char *e = std::getenv("EPHC_STREAM_TILES_PER_CTA")) tiles_per_cta = std::max(1, std::atoi(e));
        t.ncta = ncta;
        const int nshare = ncta * tiles_per_cta;
        t.ctas.assign((size_t)nshare, TileCta{0, 0});
        std::vector<int64_t> tile_at0, tile_at1;
        std::vector<int32_t> tile_strip;
        {
            int64_t at = 0;
            for (int cta = 0; cta < nshare; ++cta) {
                const int64_t goal = nwork * (int64_t)(cta + 1) / nshare;
                t.ctas[cta].t0 = (int32_t)tile_at0.size();
                const int64_t first = at;
                while (at < natom && (cta == nshare - 1 || (atom_wk[at] + atom_wk[at + 1]) / 2 <= goal)) ++at;
                int64_t a0 = first;
                while (a0 < at) {
                    if (atom_ne[a0 + 1] == atom_ne[a0]) {
                        ++a0;
                        continue;
                    }
                    const int32_t I = (int32_t)(std::upper_bound(atom0.begin(), atom0.end(), a0) - atom0.begin()) - 1;
                    int64_t a1 = a0 + 1;
                    if (a0 != atom0[I]) {
                        while (a1 < at && a1 < atom0[I + 1] && (a1 + 1 - a0) * Rf <= Rb) ++a1;
                        while (a1 - 1 > a0 && atom_ne[a1] == atom_ne[a1 - 1]) --a1;
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
        std::vector<int64_t> tile_e0((size_t)ntile + 1, 0);
        std::vector<int32_t> atom_tile((size_t)natom, -1);
        t.Ra = t.Rb = 1;
        for (int64_t it = 0; it < ntile; ++it) {
            StreamTile &th = t.tiles[it];
            const int32_t I = tile_strip[it];
            const bool dg = (tile_at0[it] == atom0[I]);
            th.a_row0 = std::min(t.nrows, I * Ra);
            th.a_rows = std::min(t.nrows, (I + 1) * Ra) - th.a_row0;
            if (dg) {
                th.b_row0 = th.a_row0;
                th.b_rows = th.a_rows;
            } else {
                const int32_t j0 = (I + 1) * bps + (int32_t)(tile_at0[it] - atom0[I] - 1);
                const int32_t j1 = (I + 1) * bps + (int32_t)(tile_at1[it] - 1 - atom0[I] - 1);
                th.b_row0 = t.blk_row0[j0];
                th.b_rows = t.blk_row0[j1 + 1] - th.b_row0;
            }
            th.flags = dg ? 4 : 0;
            th.a_slot = th.b_slot = -1;
            th.pad = 0;
            t.Ra = std::max(t.Ra, th.a_rows);
            t.Rb = std::max(t.Rb, th.b_rows);
            for (int64_t at = tile_at0[it]; at < tile_at1[it]; ++at) atom_tile[at] = (int32_t)it;
            tile_e0[it + 1] = tile_e0[it] + (atom_ne[tile_at1[it]] - atom_ne[tile_at0[it]]);
        }
        // bucket the entries by tile
        std::vector<SEnt> ents((size_t)nent);
        {
            std::vector<int64_t> cur(tile_e0.begin(), tile_e0.end() - 1);
            for (int64_t ip = 0; ip < npair; ++ip) {
                const int64_t sa = (int64_t)p->pair_ik[ip] * nb, sb = (int64_t)p->pair_ikq[ip] * nb;
                for (int64_t j = c.pair_ch0[ip]; j < c.pair_ch0[ip + 1]; ++j) {
                    const int n = c.ch_code[j] & 15, m = (c.ch_code[j] >> 4) & 15, nu = c.ch_code[j] >> 8;
                    const int32_t a = t.state_row[sa + n], b = t.state_row[sb + m];
                    const int64_t it = atom_tile[atom_of(a, b)];
                    if (c.ch_wabs[j] != 0.0) ents[cur[it]++] = SEnt{a, b, (int32_t)ip, (uint16_t)nu, 0, c.ch_wabs[j]};
                    if (c.ch_wem[j] != 0.0) ents[cur[it]++] = SEnt{a, b, (int32_t)ip, (uint16_t)nu, 1, c.ch_wem[j]};
                }
            }
        }
        // per tile: sort by (k row, k' row, pair, mode, kind), cut into chunks, build the chunk-local tables
        struct TileOut {
            std::vector<StreamChunk> chunks;
            std::vector<uint32_t> code, iq;
            std::vector<uint16_t> perm, aid, ast, bid, bst;
        };
        std::vector<TileOut> outs((size_t)ntile);
        const int pair_cap = std::max(1, kStreamNSlots / nnu);
#pragma omp parallel
        {
            std::vector<int32_t> slot_of((size_t)npair, -1);
            std::vector<int32_t> touched;
            std::vector<uint16_t> order;
#pragma omp for schedule(dynamic, 1)
            for (int64_t it = 0; it < ntile; ++it) {
                SEnt *eb = ents.data() + tile_e0[it], *ee = ents.data() + tile_e0[it + 1];
                std::sort(eb, ee, [](const SEnt &x, const SEnt &y) {
                    if (x.a != y.a) return x.a < y.a;
                    if (x.b != y.b) return x.b < y.b;
                    if (x.ip != y.ip) return x.ip < y.ip;
                    if (x.nu != y.nu) return x.nu < y.nu;
                    return x.kind < y.kind;
                });
                const StreamTile &th = t.tiles[it];
                TileOut &o = outs[it];
                const int64_t n_t = ee - eb;
                o.code.resize((size_t)n_t);
                o.perm.clear();
                int64_t s = 0;
                while (s < n_t) {
                    // greedy chunk [s, e)
                    touched.clear();
                    int64_t e = s;
                    const int32_t a0 = eb[s].a - th.a_row0;
                    while (e < n_t && e - s < kStreamChunk) {
                        if (eb[e].a - th.a_row0 - a0 > 255) break;
                        if (slot_of[eb[e].ip] < 0) {
                            if ((int)touched.size() >= pair_cap) break;
                            slot_of[eb[e].ip] = (int32_t)touched.size();
                            touched.push_back(eb[e].ip);
                        }
                        ++e;
                    }
                    StreamChunk ch;
                    ch.e0 = s;  // tile-relative for now
                    ch.ne = (int32_t)(e - s);
                    ch.a0 = a0;
                    ch.ar0 = (int32_t)o.aid.size();
                    ch.br0 = (int32_t)o.bid.size();
                    ch.q0 = (int32_t)o.iq.size();
                    ch.nq = (int32_t)touched.size();
                    ch.pad0 = ch.pad1 = 0;  // pad0: offset of the chunk's permutation in units of 4 elements
                    for (int32_t ipq : touched) o.iq.push_back((uint32_t)c.pair_iq[ipq]);
                    int nar = 0;
                    for (int64_t i = s; i < e; ++i) {
                        const SEnt &x = eb[i];
                        o.code[i] = (uint32_t)(x.a - th.a_row0 - a0) | ((uint32_t)(x.b - th.b_row0) << 8) |
                                    ((uint32_t)(slot_of[x.ip] * nnu + x.nu) << 19) | ((uint32_t)x.kind << 31);
                        if (i == s || x.a != eb[i - 1].a) {
                            o.aid.push_back((uint16_t)(x.a - th.a_row0));
                            o.ast.push_back((uint16_t)(i - s));
                            ++nar;
                        }
                    }
                    o.aid.push_back(0);
                    o.ast.push_back((uint16_t)(e - s));  // sentinel (ne <= 4096 fits)
                    ch.nar = nar;
                    order.resize((size_t)(e - s));
                    for (int64_t i = 0; i < e - s; ++i) order[i] = (uint16_t)i;
                    std::stable_sort(order.begin(), order.end(), [&](uint16_t x, uint16_t y) { return eb[s + x].b < eb[s + y].b; });
                    int nbr = 0;
                    ch.pad0 = (int32_t)(o.perm.size() / 4);  // permutation of this chunk starts at a multiple of 4
                    for (int64_t i = 0; i < e - s; ++i) {
                        o.perm.push_back(order[i]);
                        if (i == 0 || eb[s + order[i]].b != eb[s + order[i - 1]].b) {
                            o.bid.push_back((uint16_t)(eb[s + order[i]].b - th.b_row0));
                            o.bst.push_back((uint16_t)i);
                            ++nbr;
                        }
                    }
                    while (o.perm.size() % 4) o.perm.push_back(0);
                    o.bid.push_back(0);
                    o.bst.push_back((uint16_t)(e - s));
                    ch.nbr = nbr;
                    o.chunks.push_back(ch);
                    for (int32_t ipq : touched) slot_of[ipq] = -1;
                    s = e;
                }
            }
        }
        // concatenate
        t.w.resize((size_t)nent);
        t.code.resize((size_t)nent);
        t.perm.clear();
#pragma omp parallel for schedule(static)
        for (int64_t e = 0; e < nent; ++e) t.w[e] = ents[e].w;
        for (int64_t it = 0; it < ntile; ++it) {
            TileOut &o = outs[it];
            StreamTile &th = t.tiles[it];
            th.c0 = (int32_t)t.chunks.size();
            th.nc = (int32_t)o.chunks.size();
            const int64_t a_base = (int64_t)t.arow_id.size(), b_base = (int64_t)t.brow_id.size(), q_base = (int64_t)t.iq.size();
            if (a_base + (int64_t)o.aid.size() > 0x7fffffffLL || b_base + (int64_t)o.bid.size() > 0x7fffffffLL) {
                err = "stream store: more than 2^31 row tasks";
                return EPHC_ELIMIT;
            }
            const int64_t p_base = (int64_t)t.perm.size() / 4;
            for (StreamChunk ch : o.chunks) {
                ch.e0 += tile_e0[it];
                if (p_base + ch.pad0 > 0x7fffffffLL) {
                    err = "stream store: permutation offset overflow";
                    return EPHC_ELIMIT;
                }
                ch.pad0 += (int32_t)p_base;
                ch.ar0 += (int32_t)a_base;
                ch.br0 += (int32_t)b_base;
                ch.q0 += (int32_t)q_base;
                t.chunks.push_back(ch);
            }
            std::copy(o.code.begin(), o.code.end(), t.code.begin() + tile_e0[it]);
            t.perm.insert(t.perm.end(), o.perm.begin(), o.perm.end());
            t.arow_id.insert(t.arow_id.end(), o.aid.begin(), o.aid.end());
            t.arow_start.insert(t.arow_start.end(), o.ast.begin(), o.ast.end());
            t.brow_id.insert(t.brow_id.end(), o.bid.begin(), o.bid.end());
            t.brow_start.insert(t.brow_start.end(), o.bst.begin(), o.bst.end());
            t.iq.insert(t.iq.end(), o.iq.begin(), o.iq.end());
            o = TileOut();
        }
        // a-runs, partial-sum slots and the per-fine-block lists (as in the tile store)
        for (int64_t it = 0; it < ntile; ++it) t.tiles[it].flags |= 3;  // every tile stages and flushes both row ranges
        t.order.resize((size_t)ntile);
        for (int64_t it = 0; it < ntile; ++it) t.order[it] = (int32_t)it;
        std::stable_sort(t.order.begin(), t.order.end(), [&](int32_t x, int32_t y) {
            return atom_wk[tile_at1[x]] - atom_wk[tile_at0[x]] > atom_wk[tile_at1[y]] - atom_wk[tile_at0[y]];
        });
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
            StreamTile &th = t.tiles[it];
            th.a_slot = (th.flags & 1) ? new_slot(th.a_row0, th.a_rows) : t.tiles[it - 1].a_slot;
            th.b_slot = (th.flags & 4) ? -1 : new_slot(th.b_row0, th.b_rows);
        }
        t.part_rows = rows;
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
    } catch (const std::bad_alloc &) {
        err = "host allocation failed (stream store)";
        return EPHC_ENOMEM;
    }
    if (std::getenv("EPHC_DEBUG")) {
        double ne = 0, nar = 0, nbr = 0, nq = 0;
        for (const StreamChunk &ch : t.chunks) {
            ne += ch.ne;
            nar += ch.nar;
            nbr += ch.nbr;
            nq += ch.nq;
        }
        {
            double mn[4] = {1e30, 1e30, 1e30, 1e30}, mx[4] = {0, 0, 0, 0};
            for (const TileCta &ct : t.ctas) {
                double v[4] = {0, 0, 0, 0};
                for (int32_t it = ct.t0; it < ct.t1; ++it) {
                    v[3] += 1;
                    for (int32_t ci = t.tiles[it].c0; ci < t.tiles[it].c0 + t.tiles[it].nc; ++ci) {
                        v[0] += t.chunks[ci].ne;
                        v[1] += 1;
                        v[2] += t.chunks[ci].nq;
                    }
                }
                for (int j = 0; j < 4; ++j) {
                    mn[j] = std::min(mn[j], v[j]);
                    mx[j] = std::max(mx[j], v[j]);
                }
            }
            std::fprintf(stderr, "stream shares: entries %.0f..%.0f, chunks %.0f..%.0f, pairs %.0f..%.0f, tiles %.0f..%.0f\n", mn[0], mx[0],
                         mn[1], mx[1], mn[2], mx[2], mn[3], mx[3]);
        }
        const double n = (double)std::max<size_t>(t.chunks.size(), 1);
        std::fprintf(stderr, "stream store: %zu tiles, %zu chunks, per chunk: %.0f entries, %.0f k rows, %.0f k' rows, %.0f pairs; Ra %d Rb %d\n",
                     t.tiles.size(), t.chunks.size(), ne / n, nar / n, nbr / n, nq / n, t.Ra, t.Rb);
    }
    t.supported = true;
    return EPHC_OK;
}

}  // namespace ephc
