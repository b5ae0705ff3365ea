// ephc_paper_kernels.cuh -- the paper's own GPU data structure and algorithm (Fig. 2), written out as
// two plain kernels (variant 4).  It exists to put a measured number on "this library's stores vs the paper's layout"
// on the same B200; it is not the default of any call.
//   scatter            one row per (k,q) pair: ik, ikq (and iq, the row of N)                 PAPER.md:84, Fig. 2a
//   scatter_channels   one row per active channel weight: eph_g2*delta (fp64), bnds_idx (joint n, m, nu index and
//                      which delta), kq_idx (row in scatter); channels of a pair are contiguous
//   sc_col             per-channel scratch written by step 2 and read by step 3
//   stargets_sources   two rows per channel (index into sc_col and the sign of its contribution), sorted so that
//                      equal (n,k) are adjacent;  targets: (src, len, nk_index) per distinct (n,k)
//   step 2  one thread per channel: gathers f_nk, f_mk+q, N_nu,q and stores the summand of Eq. 2 to sc_col
//   step 3  one thread per target: adds its len signed sc_col values, one owner per I(n,k), no atomics
#pragma once
#include <cuda_runtime.h>

#include "ephc_internal.h"

namespace ephc {

struct PaperChannel {   // 16 bytes
    double w;           // (2 pi / hbar N_q) |g|^2 delta_sigma(.) of ONE delta
    uint32_t bnds_idx;  // n | m << 4 | nu << 8 | kind << 14 (0: F_abs, 1: F_em)
    uint32_t kq_idx;    // row in scatter
};
struct PaperTarget {    // 16 bytes
    int64_t src;        // first row in stargets_sources
    int32_t len;
    int32_t nk_index;   // state s = ik * nb + n
};

__global__ void __launch_bounds__(256) paper_step2_kernel(const PaperChannel *__restrict__ ch, const int32_t *__restrict__ sc_ik,
                                                          const int32_t *__restrict__ sc_ikq, const int32_t *__restrict__ sc_iq,
                                                          const double *__restrict__ f, const double *__restrict__ N,
                                                          double *__restrict__ sc_col, int64_t nrow, int nb, int nnu) {
    const int64_t c = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (c >= nrow) return;
    const PaperChannel r = ch[c];
    const int n = r.bnds_idx & 15, m = (r.bnds_idx >> 4) & 15, nu = (r.bnds_idx >> 8) & 63;
    const double fa = f[(int64_t)sc_ik[r.kq_idx] * nb + n], fb = f[(int64_t)sc_ikq[r.kq_idx] * nb + m];
    const double Nq = N[(int64_t)sc_iq[r.kq_idx] * nnu + nu];
    const double out = fa * (1.0 - fb), in = fb * (1.0 - fa);  // reading R-1
    const double F = (r.bnds_idx >> 14) ? out * (Nq + 1.0) - in * Nq : out * Nq - in * (Nq + 1.0);
    sc_col[c] = r.w * F;
}

// src_idx: channel << 1 | 1 for the (m,k+q) side, which receives +T; the (n,k) side receives -T
__global__ void __launch_bounds__(256) paper_step3_kernel(const PaperTarget *__restrict__ targets, const uint32_t *__restrict__ src_idx,
                                                          const double *__restrict__ sc_col, double *__restrict__ I, int64_t ntarget) {
    const int64_t t = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= ntarget) return;
    const PaperTarget tg = targets[t];
    double sum = 0.0;
    for (int32_t i = 0; i < tg.len; ++i) {
        const uint32_t s = src_idx[tg.src + i];
        const double v = sc_col[s >> 1];
        sum += (s & 1u) ? v : -v;
    }
    I[tg.nk_index] = sum;
}

}  // namespace ephc
