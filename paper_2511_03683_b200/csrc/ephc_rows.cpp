// ephc_rows.cpp -- host side of the row store used by ephc_transport_iter (see ephc_internal.h "row store").
// Built once from the two-sided gather store ("performed only once on CPUs"): the same ordered terms,
// regrouped by (strip of destination rows, range of partner rows, destination row).
//
// Product code: shares nothing with oracle/.
#include <algorithm>
#include <cstdlib>
#include <numeric>

#include "ephc_internal.h"

namespace ephc {

int build_rows(const ephc_problem *p, const Dims &d, const GatherHost &g, int nstrip, RowHost &r, std::string &err) {
    const int nb = d.nb;
    const int64_t nent = (int64_t)g.code.size();
    r = RowHost();
    if (nent >= 0xffffffffLL) {
        err = "row store: more than 2^32-1 ordered entries";
        return EPHC_ELIMIT;
    }
    if (nstrip < 1) nstrip = 1;
    try {
        // compact rows: states inside the window (R-7), in state order
        r.state_row.assign((size_t)d.ns, -1);
        for (int64_t s = 0; s < d.ns; ++s)
            if (p->E[s] >= p->emin && p->E[s] <= p->emax) {
                r.state_row[s] = (int32_t)r.row_state.size();
                r.row_state.push_back((int32_t)s);
            }
        r.nrows = (int32_t)r.row_state.size();
        int Rb = 6144;
        if (const char *e = std::getenv("EPHC_ROW_RANGE")) Rb = std::atoi(e);
        Rb = std::max(32, std::min(8192, Rb)) & ~1;  // even: 16-byte aligned staging copies
        r.Rb = Rb;
        const int32_t nrange = std::max(1, (r.nrows + Rb - 1) / Rb);

        // destination / partner row of every gather entry (walk work units -> rounds -> tasks as the kernels do)
        std::vector<int32_t> drow((size_t)nent), prow((size_t)nent);
        std::vector<uint32_t> pmeta((size_t)nent);  // (iq * nnu + mode) | kind << 31: what transport_setup needs besides w
        if ((int64_t)d.nq * d.nnu >= 0x80000000LL) {
            err = "row store: N table with 2^31 or more elements";
            return EPHC_ELIMIT;
        }
        const int64_t nwu = (int64_t)g.wus.size();
#pragma omp parallel for schedule(dynamic, 16)
        for (int64_t iw = 0; iw < nwu; ++iw) {
            const WorkUnit &wu = g.wus[iw];
            for (int32_t rr = wu.r0; rr < wu.r1; ++rr) {
                const Round &rd = g.rounds[rr];
                for (int32_t t = rd.t0; t < rd.t0 + rd.nt; ++t) {
                    const Task &tk = g.tasks[t];
                    for (int64_t e = tk.e0; e < tk.e0 + tk.len; ++e) {
                        const uint32_t c = g.code[e];
                        const int32_t ps = g.hp_k[rd.hp0 + (c & kPairMask)] * nb + (int32_t)((c >> kBandShift) & 15);
                        drow[e] = r.state_row[tk.row];
                        prow[e] = r.state_row[ps];
                        pmeta[e] = ((uint32_t)g.hp_q[rd.hp0 + (c & kPairMask)] * (uint32_t)d.nnu + ((c >> kModeShift) & 63u)) |
                                   (((c >> kKindBit) & 1u) << 31);
                    }
                }
            }
        }
        for (int64_t e = 0; e < nent; ++e)
            if (drow[e] < 0 || prow[e] < 0) {
                err = "internal: ordered entry with a state outside the window";
                return EPHC_ESTATE;
            }
        // entries per (row, range) and per row
        std::vector<uint32_t> cnt((size_t)r.nrows * nrange, 0);
        for (int64_t e = 0; e < nent; ++e) cnt[(size_t)drow[e] * nrange + prow[e] / Rb]++;
        // work of a row for the strip balance: a segment is walked in steps of 32 entries (8 lanes x 4 entries) and
        // costs a fixed overhead (header fetch, shuffle reduction, accumulator update) on top
        int seg_step = 32, seg_cost = 16;
        if (const char *e = std::getenv("EPHC_ROW_SEG_STEP")) seg_step = std::max(1, std::atoi(e));
        if (const char *e = std::getenv("EPHC_ROW_SEG_COST")) seg_cost = std::max(0, std::atoi(e));
        std::vector<int64_t> row_cnt((size_t)r.nrows + 1, 0);
        for (int32_t i = 0; i < r.nrows; ++i) {
            int64_t sum = 0;
            for (int32_t c = 0; c < nrange; ++c) {
                const int64_t n = cnt[(size_t)i * nrange + c];
                if (n) sum += (n + seg_step - 1) / seg_step * seg_step + seg_cost;
            }
            row_cnt[i + 1] = row_cnt[i] + sum;
        }
        const int64_t work_total = row_cnt[r.nrows];
        // strips of equal entry count (row granularity)
        int Ra_cap = 2048;
        std::vector<int32_t> strip_row0(1, 0);
        for (int s = 1; s <= nstrip; ++s) {
            const int64_t goal = work_total * (int64_t)s / nstrip;
            int32_t r1 = (int32_t)(std::lower_bound(row_cnt.begin(), row_cnt.end(), goal) - row_cnt.begin());
            r1 = std::max(r1, strip_row0.back());
            if (s == nstrip) r1 = r.nrows;
            while (r1 - strip_row0.back() > Ra_cap) {  // an (almost) empty stretch of rows: cut it
                strip_row0.push_back(strip_row0.back() + Ra_cap);
            }
            if (r1 > strip_row0.back() || s == nstrip) strip_row0.push_back(r1);
        }
        if (strip_row0.back() != r.nrows) strip_row0.push_back(r.nrows);
        const int32_t ns_real = (int32_t)strip_row0.size() - 1;
        r.strips.resize((size_t)ns_real);
        r.Ra = 1;
        // Sparse staging: a strip needs F of the partner rows its entries reference only.  When that is less than half
        // of all (strip, partner row) combinations (few partner k per k: large cells), a strip's tiles run over ITS sorted
        // list of referenced partner rows (cols[]: chunks of Rb list positions) instead of over all rows, the kernels
        // stage those rows only, and the partner index of an entry is its position in the tile's chunk of the list.
        std::vector<int32_t> row_strip((size_t)r.nrows, 0);
        for (int32_t s2 = 0; s2 < ns_real; ++s2)
            for (int32_t i = strip_row0[s2]; i < strip_row0[s2 + 1]; ++i) row_strip[i] = s2;
        std::vector<int64_t> cols_off((size_t)ns_real + 1, 0);
        {
            // referenced (strip, partner row) combinations: a bitmap per strip
            const size_t wpr = ((size_t)r.nrows + 63) / 64;
            std::vector<uint64_t> bits((size_t)ns_real * wpr, 0);
            for (int64_t e = 0; e < nent; ++e) bits[(size_t)row_strip[drow[e]] * wpr + ((size_t)prow[e] >> 6)] |= 1ull << (prow[e] & 63);
            int64_t total = 0;
            for (int32_t s2 = 0; s2 < ns_real; ++s2) {
                int64_t m = 0;
                for (size_t k = 0; k < wpr; ++k) m += __builtin_popcountll(bits[(size_t)s2 * wpr + k]);
                cols_off[s2 + 1] = cols_off[s2] + m;
                total += m;
            }
            const char *force = std::getenv("EPHC_ROW_SPARSE");
            const bool sparse = force ? std::atoi(force) != 0 : 2 * total < (int64_t)ns_real * r.nrows;
            if (sparse) {
                r.cols.resize((size_t)total);
                for (int32_t s2 = 0; s2 < ns_real; ++s2) {
                    int64_t o = cols_off[s2];
                    for (size_t k = 0; k < wpr; ++k)
                        for (uint64_t wbits = bits[(size_t)s2 * wpr + k]; wbits; wbits &= wbits - 1)
                            r.cols[o++] = (int32_t)(k * 64 + (size_t)__builtin_ctzll(wbits));
                }
            }
        }
        const bool sparse = !r.cols.empty();
        // position of an entry's partner: (chunk of Rb rows, index inside the chunk)
        auto place = [&](int64_t e, int32_t &c, int32_t &j) {
            int32_t p = prow[e];
            if (sparse) {
                const int32_t s2 = row_strip[drow[e]];
                const int32_t *b0 = r.cols.data() + cols_off[s2], *b1 = r.cols.data() + cols_off[s2 + 1];
                p = (int32_t)(std::lower_bound(b0, b1, p) - b0);
            }
            c = p / Rb;
            j = p - c * Rb;
        };
        if (sparse) {  // entries per (row, chunk) on the strips' own lists
            std::fill(cnt.begin(), cnt.end(), 0u);
            for (int64_t e = 0; e < nent; ++e) {
                int32_t c, j;
                place(e, c, j);
                cnt[(size_t)drow[e] * nrange + c]++;
            }
        }
        // per strip: tiles and segments (sorted by descending length), entry offsets
        std::vector<int64_t> seg_abs((size_t)r.nrows * nrange, 0);  // absolute first entry of (row, range)
        int64_t e_run = 0;
        for (int32_t s = 0; s < ns_real; ++s) {
            RowStrip &st = r.strips[s];
            st.row0 = strip_row0[s];
            st.nrows = strip_row0[s + 1] - strip_row0[s];
            st.e0 = e_run;
            st.t0 = (int32_t)r.tiles.size();
            r.Ra = std::max(r.Ra, st.nrows);
            for (int32_t c = 0; c < nrange; ++c) {
                std::vector<std::pair<uint32_t, int32_t>> rows;  // (len, row)
                for (int32_t i = st.row0; i < st.row0 + st.nrows; ++i) {
                    const uint32_t n = cnt[(size_t)i * nrange + c];
                    if (n) rows.emplace_back(n, i);
                }
                if (rows.empty()) continue;
                std::stable_sort(rows.begin(), rows.end(),
                                 [](const std::pair<uint32_t, int32_t> &x, const std::pair<uint32_t, int32_t> &y) { return x.first > y.first; });
                RowTile tl;
                tl.seg0 = (int32_t)r.segs.size();
                tl.nseg = (int32_t)rows.size();
                if (sparse) {  // rows cols[col0 .. col0 + ncols) of the strip's list
                    const int64_t m = cols_off[s + 1] - cols_off[s];
                    if (cols_off[s] + (int64_t)c * Rb > 0x7fffffffLL) {
                        err = "row store: partner lists with more than 2^31 rows";
                        return EPHC_ELIMIT;
                    }
                    tl.col0 = (int32_t)(cols_off[s] + (int64_t)c * Rb);
                    tl.ncols = (int32_t)std::min<int64_t>(Rb, m - (int64_t)c * Rb);
                } else {
                    tl.col0 = c * Rb;
                    tl.ncols = std::min(Rb, r.nrows - tl.col0);
                }
                for (const auto &q : rows) {
                    if (e_run - st.e0 > 0xffffffffLL) {
                        err = "row store: strip with more than 2^32 entries";
                        return EPHC_ELIMIT;
                    }
                    r.segs.push_back(RowSeg{(uint32_t)(e_run - st.e0), q.first, (uint32_t)(q.second - st.row0), 0u});
                    seg_abs[(size_t)q.second * nrange + c] = e_run;
                    e_run += q.first;
                }
                r.tiles.push_back(tl);
            }
            st.t1 = (int32_t)r.tiles.size();
        }
        // scatter the entries (gather order inside a segment)
        r.idx.resize((size_t)nent);
        r.perm.resize((size_t)nent);
        r.wst.resize((size_t)nent);
        r.meta.resize((size_t)nent);
        for (int64_t e = 0; e < nent; ++e) {
            int32_t c, j;
            place(e, c, j);
            const int64_t o = seg_abs[(size_t)drow[e] * nrange + c]++;
            r.idx[o] = (uint16_t)j;
            r.perm[o] = (uint32_t)e;
            r.wst[o] = g.w[e];
            r.meta[o] = pmeta[e];
        }
        // inside a segment: by partner row (stable), so that the ordered terms of one (destination, partner) state pair --
        // its modes and kinds -- are adjacent (the mode-collapsed specialisation sums them)
        if (!std::getenv("EPHC_ROW_NO_SORT")) {
            const int64_t nstrips = (int64_t)r.strips.size();
#pragma omp parallel
            {
                std::vector<uint32_t> ord;
                std::vector<uint16_t> t_idx;
                std::vector<uint32_t> t_perm, t_meta;
                std::vector<double> t_w;
#pragma omp for schedule(dynamic, 1)
                for (int64_t is = 0; is < nstrips; ++is) {
                    const RowStrip &st = r.strips[is];
                    for (int32_t t = st.t0; t < st.t1; ++t)
                        for (int32_t sg = r.tiles[t].seg0; sg < r.tiles[t].seg0 + r.tiles[t].nseg; ++sg) {
                            const uint32_t len = r.segs[sg].len;
                            const int64_t e0 = st.e0 + r.segs[sg].start;
                            ord.resize(len);
                            for (uint32_t i = 0; i < len; ++i) ord[i] = i;
                            std::stable_sort(ord.begin(), ord.end(), [&](uint32_t x, uint32_t y) { return r.idx[e0 + x] < r.idx[e0 + y]; });
                            t_idx.resize(len);
                            t_perm.resize(len);
                            t_meta.resize(len);
                            t_w.resize(len);
                            for (uint32_t i = 0; i < len; ++i) {
                                t_idx[i] = r.idx[e0 + ord[i]];
                                t_perm[i] = r.perm[e0 + ord[i]];
                                t_meta[i] = r.meta[e0 + ord[i]];
                                t_w[i] = r.wst[e0 + ord[i]];
                            }
                            for (uint32_t i = 0; i < len; ++i) {
                                r.idx[e0 + i] = t_idx[i];
                                r.perm[e0 + i] = t_perm[i];
                                r.meta[e0 + i] = t_meta[i];
                                r.wst[e0 + i] = t_w[i];
                            }
                        }
                }
            }
        }
    } catch (const std::bad_alloc &) {
        err = "host allocation failed (row store)";
        return EPHC_ENOMEM;
    }
    return EPHC_OK;
}

int build_rows_collapsed(const RowHost &r, RowCollapsed &c, std::string &err) {
    c = RowCollapsed();
    try {
        c.strips.resize(r.strips.size());
        int64_t e_run = 0;
        std::vector<std::pair<uint32_t, int32_t>> order;  // (collapsed length, segment) of a tile
        std::vector<uint32_t> clen(r.segs.size(), 0);
        for (size_t is = 0; is < r.strips.size(); ++is) {  // collapsed length of every segment
            const RowStrip &st = r.strips[is];
            for (int32_t t = st.t0; t < st.t1; ++t)
                for (int32_t sg = r.tiles[t].seg0; sg < r.tiles[t].seg0 + r.tiles[t].nseg; ++sg) {
                    const int64_t e0 = st.e0 + r.segs[sg].start;
                    uint32_t n = 0;
                    for (uint32_t i = 0; i < r.segs[sg].len; ++i) n += (i == 0 || r.idx[e0 + i] != r.idx[e0 + i - 1]);
                    clen[sg] = n;
                }
        }
        for (size_t is = 0; is < r.strips.size(); ++is) {
            const RowStrip &st = r.strips[is];
            RowStrip &cs = c.strips[is];
            cs = st;
            cs.e0 = e_run;
            cs.t0 = (int32_t)c.tiles.size();
            for (int32_t t = st.t0; t < st.t1; ++t) {
                RowTile tl = r.tiles[t];
                order.clear();
                for (int32_t sg = tl.seg0; sg < tl.seg0 + tl.nseg; ++sg) order.emplace_back(clen[sg], sg);
                std::stable_sort(order.begin(), order.end(),
                                 [](const std::pair<uint32_t, int32_t> &x, const std::pair<uint32_t, int32_t> &y) { return x.first > y.first; });
                tl.seg0 = (int32_t)c.segs.size();
                for (const auto &q : order) {
                    const RowSeg &sg = r.segs[q.second];
                    const int64_t e0 = st.e0 + sg.start;
                    if (e_run - cs.e0 > 0xffffffffLL || e0 + sg.len > 0xffffffffLL) {
                        err = "collapsed row store: more than 2^32 entries";
                        return EPHC_ELIMIT;
                    }
                    c.segs.push_back(RowSeg{(uint32_t)(e_run - cs.e0), q.first, sg.row, 0u});
                    for (uint32_t i = 0; i < sg.len;) {
                        uint32_t j = i + 1;
                        while (j < sg.len && r.idx[e0 + j] == r.idx[e0 + i]) ++j;
                        if (j - i > 0xffffu) {
                            err = "collapsed row store: more than 65535 terms on one state pair";
                            return EPHC_ELIMIT;
                        }
                        c.idx.push_back(r.idx[e0 + i]);
                        c.first.push_back((uint32_t)(e0 + i));
                        c.count.push_back((uint16_t)(j - i));
                        ++e_run;
                        i = j;
                    }
                }
                c.tiles.push_back(tl);
            }
            cs.t1 = (int32_t)c.tiles.size();
        }
    } catch (const std::bad_alloc &) {
        err = "host allocation failed (collapsed row store)";
        return EPHC_ENOMEM;
    }
    return EPHC_OK;
}

}  // namespace ephc
