// ephc_row_kernels.cuh -- sm_100a kernels of the row store: the transport iteration
//     F'[al][a] = tau[a] ( v[al][a] + sum_b W(a<-b) F[al][b] ),  al = x, y, z           (reading R-16)
// One CTA = one strip of destination rows and their single owner (no atomics).  The partner rows
// are walked in ranges; per range the CTA stages F[0..3)[partner] in shared memory ([row][3], 24 B per row), then
// groups of 8 lanes take one destination row each: the lanes stream that row's (weight, partner) entries of this
// range from HBM (contiguous, every byte used once), multiply by the staged F and reduce with three shuffles;
// the group's first lane adds the three sums to the row's accumulators in shared memory (one owner per row and
// range, fixed order: bit-reproducible).  The epilogue tau (v + sum) is fused ("additional loop over
// the directions of the field").
#pragma once
#include <cuda_runtime.h>

#include "ephc_internal.h"

namespace ephc {

constexpr int kRowThreads = 1024;  // one CTA per SM: the staging traffic is (number of strips) x |F|
constexpr int kRowGroup = 8;  // lanes per destination row

struct RowParams {
    const double *W;        // per entry, row-store order
    const uint16_t *idx;
    const RowSeg *segs;
    const RowTile *tiles;
    const RowStrip *strips;
    const int32_t *row_state, *state_row;
    int32_t Rb, Ra, nstrip;
    int64_t ns;
    const double *F, *v, *tau;
    double *out;
};

inline size_t row_smem_bytes(int Rb, int Ra) { return ((size_t)Rb + (size_t)Ra) * 3 * sizeof(double); }

// weights of the gather store (written by its transport_setup kernel) -> row-store order
__global__ void __launch_bounds__(256) row_permute_kernel(const double *gW, const uint32_t *perm, double *W, int64_t n) {
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n) W[i] = __ldg(gW + __ldcs(perm + i));
}

__global__ void __launch_bounds__(kRowThreads, 1) row_iter_kernel(const RowParams P) {
    extern __shared__ double smem[];
    double *sF = smem;               // [Rb][3]
    double *sAcc = smem + P.Rb * 3;  // [Ra][3]
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int sub = lane / kRowGroup, gl = lane % kRowGroup;
    constexpr int NW = kRowThreads / 32, GPW = 32 / kRowGroup;  // warps, row groups per warp

    // states outside the window receive no contribution: F' = tau v (grid-stride over all states)
    for (int64_t s = (int64_t)blockIdx.x * kRowThreads + tid; s < P.ns; s += (int64_t)gridDim.x * kRowThreads)
        if (P.state_row[s] < 0) {
            const double ta = P.tau[s];
#pragma unroll
            for (int c = 0; c < 3; ++c) P.out[(int64_t)c * P.ns + s] = ta * P.v[(int64_t)c * P.ns + s];
        }
    if ((int)blockIdx.x >= P.nstrip) return;
    const RowStrip st = P.strips[blockIdx.x];
    for (int i = tid; i < st.nrows * 3; i += kRowThreads) sAcc[i] = 0.0;
    const double *Wb = P.W + st.e0;
    const uint16_t *Ib = P.idx + st.e0;

    for (int t = st.t0; t < st.t1; ++t) {
        const RowTile tl = P.tiles[t];
        __syncthreads();  // previous tile done with sF (and sAcc zeroed)
        for (int i = tid; i < tl.ncols; i += kRowThreads) {
            const int64_t s = P.row_state[tl.col0 + i];
#pragma unroll
            for (int c = 0; c < 3; ++c) sF[i * 3 + c] = P.F[(int64_t)c * P.ns + s];
        }
        __syncthreads();
        for (int sg0 = warp * GPW; sg0 < tl.nseg; sg0 += NW * GPW) {
            const int sg = sg0 + sub;
            uint32_t start = 0, len = 0, row = 0;
            if (sg < tl.nseg) {
                const uint4 q = __ldg(reinterpret_cast<const uint4 *>(P.segs + tl.seg0 + sg));
                start = q.x;
                len = q.y;
                row = q.z;
            }
            const double *w = Wb + start;
            const uint16_t *ix = Ib + start;
            double a0 = 0.0, a1 = 0.0, a2 = 0.0;
            // four entries per lane in flight
            for (uint32_t i = gl; i < len; i += 4 * kRowGroup) {
                double wv[4];
                unsigned jv[4];
#pragma unroll
                for (int u = 0; u < 4; ++u) {
                    const uint32_t ii = i + u * kRowGroup;
                    wv[u] = 0.0;
                    jv[u] = 0;
                    if (ii < len) {
                        wv[u] = __ldcs(w + ii);
                        jv[u] = __ldcs(ix + ii);
                    }
                }
#pragma unroll
                for (int u = 0; u < 4; ++u) {
                    const double *f = sF + jv[u] * 3;
                    a0 = fma(wv[u], f[0], a0);
                    a1 = fma(wv[u], f[1], a1);
                    a2 = fma(wv[u], f[2], a2);
                }
            }
#pragma unroll
            for (int o = kRowGroup / 2; o > 0; o >>= 1) {
                a0 += __shfl_xor_sync(0xffffffffu, a0, o);
                a1 += __shfl_xor_sync(0xffffffffu, a1, o);
                a2 += __shfl_xor_sync(0xffffffffu, a2, o);
            }
            if (gl == 0 && sg < tl.nseg) {  // the only writer of this row in this tile
                sAcc[row * 3 + 0] += a0;
                sAcc[row * 3 + 1] += a1;
                sAcc[row * 3 + 2] += a2;
            }
        }
    }
    __syncthreads();
    for (int i = tid; i < st.nrows; i += kRowThreads) {
        const int64_t s = P.row_state[st.row0 + i];
        const double ta = P.tau[s];
#pragma unroll
        for (int c = 0; c < 3; ++c) P.out[(int64_t)c * P.ns + s] = ta * (P.v[(int64_t)c * P.ns + s] + sAcc[i * 3 + c]);
    }
}

}  // namespace ephc
