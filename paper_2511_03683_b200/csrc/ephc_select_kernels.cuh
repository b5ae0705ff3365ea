// ephc_select_kernels.cuh -- channel selection on the GPU (energy window, Gaussian delta, |g| cut-off;
// SURVEY.md 8(f) NEXT-3).  The same canonical list as the host builder (ephc_build.cpp: reading R-12, order
// (pair, nu, m, n)), produced by a count pass, a prefix sum over the candidate pairs and a fill pass: one thread per
// candidate pair.  The keep / drop decisions are the same fp64 comparisons as on the host; the weights differ from the
// host's by the two exp implementations (<= 2 ulp).
#pragma once
#include <cuda_runtime.h>

#include "ephc_internal.h"

namespace ephc {

struct SelectParams {
    const int32_t *pair_ik, *pair_ikq, *kfull;
    const double *E, *hw, *g2;
    int32_t nb, nnu, g0, g1, g2n;
    double emin, emax, sigma, cut, g2_cut, C;
    int64_t npair;
    // count pass: written; fill pass: read
    uint32_t *cnt_ch, *cnt_dg;
    int32_t *pair_iq;
    const int64_t *ch0, *dg0;
    // fill pass
    uint16_t *ch_code;
    double *ch_wabs, *ch_wem;
    int32_t *dg_s, *dg_nu;
    double *dg_wabs, *dg_wem;
};

// Gaussian energy-conservation factor, readings R-3 / R-4: normal density of standard deviation sigma, exactly zero
// unless |x| < ncut * sigma (strict)
__device__ __forceinline__ double select_delta(double x, double sigma, double cut) {
    if (!(fabs(x) < cut)) return 0.0;
    return exp(-(x * x) / (2.0 * sigma * sigma)) / (sigma * sqrt(2.0 * kPi));
}

template <bool FILL>
__global__ void __launch_bounds__(128) select_kernel(const SelectParams P) {
    const int64_t ip = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (ip >= P.npair) return;
    const int32_t ik = P.pair_ik[ip], ikq = P.pair_ikq[ip];
    const int nb = P.nb, nnu = P.nnu;
    // index of (k' - k) mod grid from the two full-grid indices (reading R-20)
    const int32_t kf = P.kfull[ik], kqf = P.kfull[ikq], n23 = P.g1 * P.g2n;
    int32_t d1 = kqf / n23 - kf / n23, d2 = (kqf / P.g2n) % P.g1 - (kf / P.g2n) % P.g1, d3 = kqf % P.g2n - kf % P.g2n;
    if (d1 < 0) d1 += P.g0;
    if (d2 < 0) d2 += P.g1;
    if (d3 < 0) d3 += P.g2n;
    const int32_t iq = (d1 * P.g1 + d2) * P.g2n + d3;
    const bool self = ik == ikq;
    const double *Ea = P.E + (int64_t)ik * nb, *Eb = P.E + (int64_t)ikq * nb;
    const double *hw = P.hw + (int64_t)iq * nnu;
    const double *g2 = P.g2 + ip * (int64_t)nnu * nb * nb;
    uint32_t nch = 0, ndg = 0;
    int64_t oc = 0, od = 0;
    if (FILL) {
        oc = P.ch0[ip];
        od = P.dg0[ip];
        if (P.ch0[ip + 1] == oc && P.dg0[ip + 1] == od) return;
    }
    for (int nu = 0; nu < nnu; ++nu) {
        const double w = hw[nu];
        for (int m = 0; m < nb; ++m) {
            const double eb = Eb[m];
            if (!(eb >= P.emin && eb <= P.emax)) continue;
            for (int n = 0; n < nb; ++n) {
                const double ea = Ea[n];
                if (!(ea >= P.emin && ea <= P.emax)) continue;
                if (self && n > m) continue;  // mirror image of the stored (n < m) entry
                const double gg = g2[((int64_t)nu * nb + m) * nb + n];
                if (!(gg >= P.g2_cut)) continue;
                const double dE = ea - eb;
                const double da = select_delta(dE + w, P.sigma, P.cut), de = select_delta(dE - w, P.sigma, P.cut);
                if (da == 0.0 && de == 0.0) continue;
                const bool diag = self && n == m;
                if (FILL) {
                    const double wabs = __dmul_rn(__dmul_rn(P.C, gg), da), wem = __dmul_rn(__dmul_rn(P.C, gg), de);
                    if (diag) {
                        P.dg_s[od] = ik * nb + n;
                        P.dg_nu[od] = nu;
                        P.dg_wabs[od] = wabs;
                        P.dg_wem[od] = wem;
                        ++od;
                    } else {
                        P.ch_code[oc] = (uint16_t)(n | (m << 4) | (nu << 8));
                        P.ch_wabs[oc] = wabs;
                        P.ch_wem[oc] = wem;
                        ++oc;
                    }
                } else {
                    nch += diag ? 0u : 1u;
                    ndg += diag ? 1u : 0u;
                }
            }
        }
    }
    if (!FILL) {
        P.cnt_ch[ip] = nch;
        P.cnt_dg[ip] = ndg;
        P.pair_iq[ip] = iq;
    }
}

}  // namespace ephc
