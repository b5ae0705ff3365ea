// ephc_build.cpp -- host side of ephc_build_channels: channel selection, the canonical
// unordered channel list, and the destination-k-segmented two-sided ("gather") store with its launch
// geometry (work units / rounds / warp tasks).  "This step is not computationally intensive and is
// performed only once on CPUs"; it is OpenMP-parallel over candidate pairs / rounds.
//
// Product code: shares nothing with oracle/.
#include <algorithm>
#include <cmath>
#include <cstdlib>
#include <cstring>

#include "ephc_internal.h"

namespace ephc {

namespace {

// Gaussian energy-conservation factor, reading R-3/R-4: normalised normal density of standard
// deviation sigma, exactly zero unless |x| < ncut*sigma (strict).
inline double delta_sigma(double x, double sigma, double cut) {
    if (!(std::fabs(x) < cut)) return 0.0;
    return std::exp(-(x * x) / (2.0 * sigma * sigma)) / (sigma * std::sqrt(2.0 * kPi));
}

// index of (k' - k) mod grid from two full-grid indices (R-20)
inline int32_t q_of(const int32_t g[3], int32_t kf, int32_t kqf) {
    const int32_t n23 = g[1] * g[2];
    int32_t d1 = kqf / n23 - kf / n23;
    int32_t d2 = (kqf / g[2]) % g[1] - (kf / g[2]) % g[1];
    int32_t d3 = kqf % g[2] - kf % g[2];
    if (d1 < 0) d1 += g[0];
    if (d2 < 0) d2 += g[1];
    if (d3 < 0) d3 += g[2];
    return (d1 * g[1] + d2) * g[2] + d3;
}

struct Sel {  // one selected (nu, m, n) of a pair
    uint16_t code;
    bool diag;
    double wabs, wem;
};

// Selection of the active channels of candidate pair p in canonical order (nu, m, n).  Returns the number
// of selected entries written to out (capacity nnu*nb*nb).
inline int select_pair(const ephc_problem *p, const Dims &d, const uint8_t *inwin, int64_t ip, int32_t iq,
                       double cut, Sel *out) {
    const int32_t ik = p->pair_ik[ip], ikq = p->pair_ikq[ip];
    const int nb = d.nb, nnu = d.nnu;
    const bool self = (ik == ikq);
    const double *Ea = p->E + (int64_t)ik * nb, *Eb = p->E + (int64_t)ikq * nb;
    const uint8_t *wa = inwin + (int64_t)ik * nb, *wb = inwin + (int64_t)ikq * nb;
    const double *hw = p->hw + (int64_t)iq * nnu;
    const double *g2 = p->g2 + ip * (int64_t)nnu * nb * nb;
    int cnt = 0;
    for (int nu = 0; nu < nnu; ++nu) {
        const double w = hw[nu];
        for (int m = 0; m < nb; ++m) {
            if (!wb[m]) continue;
            for (int n = 0; n < nb; ++n) {
                if (!wa[n]) continue;
                if (self && n > m) continue;  // mirror image of the stored (n < m) entry
                const double gg = g2[((int64_t)nu * nb + m) * nb + n];
                if (!(gg >= p->g2_cut)) continue;
                const double dE = Ea[n] - Eb[m];
                const double da = delta_sigma(dE + w, p->sigma, cut);
                const double de = delta_sigma(dE - w, p->sigma, cut);
                if (da == 0.0 && de == 0.0) continue;
                Sel s;
                s.code = (uint16_t)(n | (m << 4) | (nu << 8));
                s.diag = self && n == m;
                s.wabs = d.C * gg * da;
                s.wem = d.C * gg * de;
                out[cnt++] = s;
            }
        }
    }
    return cnt;
}

}  // namespace

int validate_problem(const ephc_problem *p, const Dims &d, std::string &err) {
    const int nb = d.nb, nnu = d.nnu;
    const int64_t npair = p->npair;
    for (int32_t k = 0; k < d.nk; ++k) {
        if (p->kfull[k] < 0 || p->kfull[k] >= d.nq || (k > 0 && p->kfull[k] <= p->kfull[k - 1])) {
            err = "kfull must be strictly ascending full-grid indices";
            return EPHC_EINVAL;
        }
    }
    if (!(p->sigma > 0.0) || !std::isfinite(p->sigma) || !(p->ncut > 0.0) || !std::isfinite(p->ncut) ||
        !(p->g2_cut >= 0.0) || !std::isfinite(p->g2_cut) || !(p->emin <= p->emax)) {
        err = "sigma, ncut must be > 0 and finite, g2_cut >= 0, emin <= emax";
        return EPHC_EINVAL;
    }
    int bad = 0;
#pragma omp parallel for reduction(| : bad) schedule(static)
    for (int64_t i = 0; i < d.ns; ++i) bad |= !std::isfinite(p->E[i]);
#pragma omp parallel for reduction(| : bad) schedule(static)
    for (int64_t i = 0; i < d.nq * nnu; ++i) bad |= !(std::isfinite(p->hw[i]) && p->hw[i] > 0.0);
    if (bad) {
        err = "E must be finite; hw must be finite and > 0";
        return EPHC_EINVAL;
    }
#pragma omp parallel for reduction(| : bad) schedule(static)
    for (int64_t ip = 0; ip < npair; ++ip) {
        const int32_t ik = p->pair_ik[ip], ikq = p->pair_ikq[ip];
        int b = (ik < 0 || ikq < ik || ikq >= d.nk);
        if (ip > 0) {
            const int32_t jk = p->pair_ik[ip - 1], jkq = p->pair_ikq[ip - 1];
            b |= !(jk < ik || (jk == ik && jkq < ikq));
        }
        bad |= b;
    }
    if (bad) {
        err = "pair list: need 0 <= ik <= ikq < nk, strictly ascending in (ik, ikq)";
        return EPHC_EINVAL;
    }
    const int64_t blk = (int64_t)nnu * nb * nb;
#pragma omp parallel for reduction(| : bad) schedule(static)
    for (int64_t i = 0; i < npair * blk; ++i) bad |= !(std::isfinite(p->g2[i]) && p->g2[i] >= 0.0);
    if (bad) {
        err = "g2 must be finite and >= 0";
        return EPHC_EINVAL;
    }
    return EPHC_OK;
}

int build_canonical(const ephc_problem *p, const Dims &d, Canonical &c, std::string &err) {
    const int nb = d.nb, nnu = d.nnu;
    const int64_t npair = p->npair;
    {
        const int rc = validate_problem(p, d, err);
        if (rc != EPHC_OK) return rc;
    }
    const int64_t blk = (int64_t)nnu * nb * nb;
    // ---- window flags (R-7: inclusive, state level) -------------------------------------------------
    std::vector<uint8_t> inwin((size_t)d.ns);
    for (int64_t i = 0; i < d.ns; ++i) inwin[i] = (p->E[i] >= p->emin && p->E[i] <= p->emax) ? 1 : 0;
    const double cut = p->ncut * p->sigma;

    // ---- pass 1: count per pair -----------------------------------------------------------------------
    try {
        c.pair_ch0.assign((size_t)npair + 1, 0);
        c.pair_dg0.assign((size_t)npair + 1, 0);
        c.pair_iq.assign((size_t)npair, 0);
    } catch (const std::bad_alloc &) {
        err = "host allocation failed (pair tables)";
        return EPHC_ENOMEM;
    }
#pragma omp parallel
    {
        std::vector<Sel> buf((size_t)blk);
#pragma omp for schedule(dynamic, 1024)
        for (int64_t ip = 0; ip < npair; ++ip) {
            const int32_t iq = q_of(d.grid, p->kfull[p->pair_ik[ip]], p->kfull[p->pair_ikq[ip]]);
            c.pair_iq[ip] = iq;
            const int cnt = select_pair(p, d, inwin.data(), ip, iq, cut, buf.data());
            int nd = 0;
            for (int j = 0; j < cnt; ++j) nd += buf[j].diag;
            c.pair_ch0[ip + 1] = cnt - nd;
            c.pair_dg0[ip + 1] = nd;
        }
    }
    int64_t npa = 0;
    for (int64_t ip = 0; ip < npair; ++ip) {
        npa += (c.pair_ch0[ip + 1] + c.pair_dg0[ip + 1]) > 0;
        c.pair_ch0[ip + 1] += c.pair_ch0[ip];
        c.pair_dg0[ip + 1] += c.pair_dg0[ip];
    }
    c.nch = c.pair_ch0[npair];
    c.ndiag = c.pair_dg0[npair];
    c.npair_active = npa;
    try {
        c.ch_code.resize((size_t)c.nch);
        c.ch_wabs.resize((size_t)c.nch);
        c.ch_wem.resize((size_t)c.nch);
        c.dg_s.resize((size_t)c.ndiag);
        c.dg_nu.resize((size_t)c.ndiag);
        c.dg_wabs.resize((size_t)c.ndiag);
        c.dg_wem.resize((size_t)c.ndiag);
    } catch (const std::bad_alloc &) {
        err = "host allocation failed (canonical channel list)";
        return EPHC_ENOMEM;
    }
    // ---- pass 2: fill ------------------------------------------------------------------------------------
    int64_t nw = 0;
#pragma omp parallel reduction(+ : nw)
    {
        std::vector<Sel> buf((size_t)blk);
#pragma omp for schedule(dynamic, 1024)
        for (int64_t ip = 0; ip < npair; ++ip) {
            if (c.pair_ch0[ip + 1] == c.pair_ch0[ip] && c.pair_dg0[ip + 1] == c.pair_dg0[ip]) continue;
            const int cnt = select_pair(p, d, inwin.data(), ip, c.pair_iq[ip], cut, buf.data());
            int64_t oc = c.pair_ch0[ip], od = c.pair_dg0[ip];
            for (int j = 0; j < cnt; ++j) {
                const Sel &s = buf[j];
                if (s.diag) {
                    c.dg_s[od] = p->pair_ik[ip] * nb + (s.code & 15);
                    c.dg_nu[od] = s.code >> 8;
                    c.dg_wabs[od] = s.wabs;
                    c.dg_wem[od] = s.wem;
                    ++od;
                } else {
                    c.ch_code[oc] = s.code;
                    c.ch_wabs[oc] = s.wabs;
                    c.ch_wem[oc] = s.wem;
                    nw += (s.wabs != 0.0) + (s.wem != 0.0);
                    ++oc;
                }
            }
        }
    }
    c.nw = nw;
    c.iq0 = 0;
    return EPHC_OK;
}

// ---------------------------------------------------------------------------------------------------------
// Two-sided store.  For every destination k: the half-pairs (k <- k') in ascending k', i.e. every candidate
// pair that touches k in either orientation.  An ordered entry of destination state a = (n,k) with partner
// b = (m,k') carries the weight of ONE delta and the occupation factor seen from a:
//     canonical side (a on pair_ik):   w_abs -> F_abs,  w_em -> F_em
//     mirrored  side (a on pair_ikq):  w_abs -> F_em,   w_em -> F_abs      (x_abs' = -x_em, x_em' = -x_abs)
// and I[a] = - sum over a's entries of w * F_kind(f_a, f_b, N[iq,nu]) with iq the canonical q of the pair for
// both sides (literal Eq. 2 uses one symbol N_nu,q; R-10).
// ---------------------------------------------------------------------------------------------------------
namespace {

struct HalfPair {
    int64_t ip;     // candidate pair
    int32_t side;   // 0: destination = pair_ik, 1: destination = pair_ikq, 2: self pair (both roles + diagonal)
};

}  // namespace

int build_gather(const ephc_problem *p, const Dims &d, const Canonical &c, GatherHost &g, std::string &err) {
    const int nb = d.nb, nnu = d.nnu;
    const int64_t npair = p->npair;
    const int vpp = std::max(nb + nnu, 3 * nb);  // staged doubles per half-pair (collision / transport)
    int pmax = std::max(1, std::min<int>(kVMax / vpp, (int)kPairMask));
    int64_t etarget = kEntriesTarget;
    // tuning knobs (sweeps, and tests that force multi-round segments): they can only tighten the limits
    if (const char *e = std::getenv("EPHC_ROUND_PAIRS")) pmax = std::max(1, std::min(pmax, std::atoi(e)));
    if (const char *e = std::getenv("EPHC_WU_ENTRIES")) etarget = std::max(1, std::min<int>((kTasksMax - kRowsMax) * kTaskLen, std::atoi(e)));

    // ---- half-pairs per destination k, ascending partner ---------------------------------------------
    std::vector<int64_t> seg_hp0((size_t)d.nk + 1, 0);
    std::vector<int32_t> n_mirror((size_t)d.nk, 0);
    auto active = [&](int64_t ip) {
        return (c.pair_ch0[ip + 1] > c.pair_ch0[ip]) || (c.pair_dg0[ip + 1] > c.pair_dg0[ip]);
    };
    // k-sharded handles keep only the half-pairs whose DESTINATION k they own (k points are distributed
    // over the processes); every ordered term then lives on exactly one rank
    auto owned = [&](int32_t k) { return k >= d.k_lo && k < d.k_hi; };
    for (int64_t ip = 0; ip < npair; ++ip) {
        if (!active(ip)) continue;
        const int32_t ik = p->pair_ik[ip], ikq = p->pair_ikq[ip];
        if (owned(ik)) seg_hp0[ik + 1]++;
        if (ikq != ik && owned(ikq)) {
            seg_hp0[ikq + 1]++;
            n_mirror[ikq]++;
        }
    }
    for (int32_t k = 0; k < d.nk; ++k) seg_hp0[k + 1] += seg_hp0[k];
    const int64_t nhp = seg_hp0[d.nk];
    if (nhp > 0x7fffffffLL) {
        err = "more than 2^31-1 half-pairs";
        return EPHC_ELIMIT;
    }
    std::vector<HalfPair> hps;
    try {
        hps.resize((size_t)nhp);
        g.hp_k.resize((size_t)nhp);
        g.hp_q.resize((size_t)nhp);
    } catch (const std::bad_alloc &) {
        err = "host allocation failed (half-pairs)";
        return EPHC_ENOMEM;
    }
    {
        std::vector<int64_t> cur_m((size_t)d.nk), cur_f((size_t)d.nk);
        for (int32_t k = 0; k < d.nk; ++k) {
            cur_m[k] = seg_hp0[k];
            cur_f[k] = seg_hp0[k] + n_mirror[k];
        }
        for (int64_t ip = 0; ip < npair; ++ip) {
            if (!active(ip)) continue;
            const int32_t ik = p->pair_ik[ip], ikq = p->pair_ikq[ip];
            int64_t o = 0;
            if (owned(ik)) {
                o = cur_f[ik]++;
                hps[o] = HalfPair{ip, ik == ikq ? 2 : 0};
                g.hp_k[o] = ikq;
                g.hp_q[o] = c.pair_iq[ip];
            }
            if (ikq != ik && owned(ikq)) {
                o = cur_m[ikq]++;
                hps[o] = HalfPair{ip, 1};
                g.hp_k[o] = ik;
                g.hp_q[o] = c.pair_iq[ip];
            }
        }
    }

    // entries emitted by one half-pair, per destination band
    auto walk = [&](const HalfPair &hp, auto &&fn) {
        for (int64_t j = c.pair_ch0[hp.ip]; j < c.pair_ch0[hp.ip + 1]; ++j) {
            const int n = c.ch_code[j] & 15, m = (c.ch_code[j] >> 4) & 15, nu = c.ch_code[j] >> 8;
            const double wa = c.ch_wabs[j], we = c.ch_wem[j];
            if (hp.side != 1) {
                if (wa != 0.0) fn(n, m, nu, 0u, 0u, wa);
                if (we != 0.0) fn(n, m, nu, 1u, 0u, we);
            }
            if (hp.side != 0) {
                if (wa != 0.0) fn(m, n, nu, 1u, 0u, wa);
                if (we != 0.0) fn(m, n, nu, 0u, 0u, we);
            }
        }
        if (hp.side == 2) {
            for (int64_t j = c.pair_dg0[hp.ip]; j < c.pair_dg0[hp.ip + 1]; ++j) {
                const int n = c.dg_s[j] % nb, nu = c.dg_nu[j];
                if (c.dg_wabs[j] != 0.0) fn(n, n, nu, 0u, 1u, c.dg_wabs[j]);
                if (c.dg_wem[j] != 0.0) fn(n, n, nu, 1u, 1u, c.dg_wem[j]);
            }
        }
    };

    // ---- entries per segment (for work-unit sizing) ------------------------------------------------------
    std::vector<int64_t> seg_ent((size_t)d.nk, 0);
#pragma omp parallel for schedule(dynamic, 64)
    for (int32_t k = 0; k < d.nk; ++k) {
        int64_t e = 0;
        for (int64_t h = seg_hp0[k]; h < seg_hp0[k + 1]; ++h) walk(hps[h], [&](int, int, int, unsigned, unsigned, double) { ++e; });
        seg_ent[k] = e;
    }

    // ---- work units and rounds ------------------------------------------------------------------------------
    // A work unit owns whole k segments.  Small segments are packed into one round while the staged pair data,
    // the row count and the task count fit; a segment whose half-pairs alone exceed the staging buffer gets a
    // work unit of its own with several rounds.
    struct RoundSeg { int32_t k; int64_t h0, h1; };
    std::vector<std::vector<RoundSeg>> round_segs;  // per round: the segment pieces it holds
    g.wus.clear();
    g.rounds.clear();
    const int segs_max = std::max(1, kRowsMax / nb);
    {
        int32_t k = 0;
        while (k < d.nk) {
            const int64_t nh = seg_hp0[k + 1] - seg_hp0[k];
            WorkUnit wu;
            wu.r0 = (int32_t)round_segs.size();
            wu.row0 = k * nb;
            if (nh > pmax || seg_ent[k] > (int64_t)(kTasksMax - nb) * kTaskLen) {
                // split by half-pair range: even pieces, bounded pairs and entries
                int64_t pieces = (nh + pmax - 1) / pmax;
                const int64_t emax = (int64_t)(kTasksMax - nb) * kTaskLen / 2;
                pieces = std::max<int64_t>(pieces, (seg_ent[k] + emax - 1) / emax);
                pieces = std::max<int64_t>(pieces, 1);
                // walk half-pairs, closing a piece when either bound would be exceeded
                const int64_t per = (nh + pieces - 1) / pieces;
                int64_t h = seg_hp0[k];
                while (h < seg_hp0[k + 1]) {
                    int64_t h1 = h, e = 0;
                    while (h1 < seg_hp0[k + 1] && (h1 - h) < per) {
                        int64_t eh = 0;
                        walk(hps[h1], [&](int, int, int, unsigned, unsigned, double) { ++eh; });
                        if (h1 > h && e + eh > emax) break;
                        e += eh;
                        ++h1;
                    }
                    round_segs.push_back({RoundSeg{k, h, h1}});
                    h = h1;
                }
                wu.nrows = nb;
                ++k;
            } else {
                std::vector<RoundSeg> rs;
                int64_t pairs = 0, ents = 0;
                int32_t k1 = k;
                while (k1 < d.nk) {
                    const int64_t nh1 = seg_hp0[k1 + 1] - seg_hp0[k1];
                    if (k1 > k) {
                        if (pairs + nh1 > pmax || ents + seg_ent[k1] > etarget || (k1 - k) >= segs_max) break;
                        if (nh1 > pmax || seg_ent[k1] > (int64_t)(kTasksMax - nb) * kTaskLen) break;
                    }
                    rs.push_back(RoundSeg{k1, seg_hp0[k1], seg_hp0[k1 + 1]});
                    pairs += nh1;
                    ents += seg_ent[k1];
                    ++k1;
                }
                round_segs.push_back(std::move(rs));
                wu.nrows = (k1 - k) * nb;
                k = k1;
            }
            wu.r1 = (int32_t)round_segs.size();
            g.wus.push_back(wu);
        }
    }
    const int64_t nrounds = (int64_t)round_segs.size();

    // ---- per round: entries per (segment piece, destination band) -> tasks -------------------------------------
    std::vector<std::vector<int64_t>> rcnt((size_t)nrounds);
#pragma omp parallel for schedule(dynamic, 16)
    for (int64_t r = 0; r < nrounds; ++r) {
        const auto &rs = round_segs[r];
        rcnt[r].assign(rs.size() * nb, 0);
        for (size_t s = 0; s < rs.size(); ++s)
            for (int64_t h = rs[s].h0; h < rs[s].h1; ++h)
                walk(hps[h], [&](int nd, int, int, unsigned, unsigned, double) { rcnt[r][s * nb + nd]++; });
    }
    g.rounds.resize((size_t)nrounds);
    std::vector<int64_t> round_e0((size_t)nrounds + 1, 0);
    g.tasks.clear();
    for (int64_t r = 0; r < nrounds; ++r) {
        const auto &rs = round_segs[r];
        Round rd;
        rd.hp0 = (int32_t)rs.front().h0;
        rd.nhp = (int32_t)(rs.back().h1 - rs.front().h0);
        rd.t0 = (int32_t)g.tasks.size();
        int64_t e = round_e0[r];
        for (size_t s = 0; s < rs.size(); ++s) {
            for (int n = 0; n < nb; ++n) {
                int64_t left = rcnt[r][s * nb + n];
                while (left > 0) {
                    const int32_t len = (int32_t)std::min<int64_t>(left, kTaskLen);
                    g.tasks.push_back(Task{e, len, rs[s].k * nb + n});
                    e += len;
                    left -= len;
                }
            }
        }
        rd.nt = (int32_t)g.tasks.size() - rd.t0;
        if (rd.nt > kTasksMax || rd.nhp > pmax) {
            err = "internal: round exceeds task or staging limit";
            return EPHC_ELIMIT;
        }
        round_e0[r + 1] = e;
        g.rounds[r] = rd;
        if (g.tasks.size() > 0x7fffff00ULL) {
            err = "more than 2^31 warp tasks";
            return EPHC_ELIMIT;
        }
    }
    const int64_t nent = round_e0[nrounds];
    try {
        g.code.resize((size_t)nent);
        g.w.resize((size_t)nent);
    } catch (const std::bad_alloc &) {
        err = "host allocation failed (gather store)";
        return EPHC_ENOMEM;
    }
    // ---- fill: rows of a round are contiguous, ordered (segment piece, band); inside a row ascending k' -----------
#pragma omp parallel for schedule(dynamic, 16)
    for (int64_t r = 0; r < nrounds; ++r) {
        const auto &rs = round_segs[r];
        std::vector<int64_t> cur(rs.size() * nb);
        int64_t e = round_e0[r];
        for (size_t i = 0; i < cur.size(); ++i) {
            cur[i] = e;
            e += rcnt[r][i];
        }
        const int64_t hp0 = rs.front().h0;
        for (size_t s = 0; s < rs.size(); ++s)
            for (int64_t h = rs[s].h0; h < rs[s].h1; ++h) {
                const uint32_t pl = (uint32_t)(h - hp0);
                walk(hps[h], [&](int nd, int mp, int nu, unsigned kind, unsigned diag, double w) {
                    const int64_t o = cur[s * nb + nd]++;
                    g.code[o] = pl | ((uint32_t)mp << kBandShift) | ((uint32_t)nu << kModeShift) |
                                (kind << kKindBit) | (diag << kDiagBit);
                    g.w[o] = w;
                });
            }
    }
    return EPHC_OK;
}

}  // namespace ephc
