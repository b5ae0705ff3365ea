// ephc_row_kernels.cuh -- sm_100a kernels of the row store: the transport iteration
//     F'[al][a] = tau[a] ( v[al][a] + sum_b W(a<-b) F[al][b] ),  al = x, y, z           (reading R-16)
// One CTA = one strip of destination rows and their single owner (no atomics).  The partner rows
// are walked in ranges; per range the CTA stages F[0..3)[partner] in shared memory ([row][3], 24 B per row; copied
// asynchronously one range ahead from a compact copy of F), then
// groups of 8 lanes take one destination row each: the lanes stream that row's (weight, partner) entries of this
// range from HBM (contiguous, every byte used once), multiply by the staged F and reduce with three shuffles;
// the group's first lane adds the three sums to the row's accumulators in shared memory (one owner per row and
// range, fixed order: bit-reproducible).  The epilogue tau (v + sum) is fused ("additional loop over
// the directions of the field").
#pragma once
#include <cuda_runtime.h>

#include "ephc_internal.h"

namespace ephc {

#ifndef EPHC_ROW_THREADS
#define EPHC_ROW_THREADS 1024
#endif
constexpr int kRowThreads = EPHC_ROW_THREADS;  // 1024: one CTA per SM (the staging traffic is (number of strips) x |F|)
constexpr int kRowGroup = 8;  // lanes per destination row
#ifndef EPHC_ROW_BATCH
#define EPHC_ROW_BATCH 4
#endif
constexpr int kRowBatch = EPHC_ROW_BATCH;

struct RowParams {
    double *W;              // per entry, row-store order: written by row_setup_kernel, read by row_iter_kernel
    const double *wst;      // per entry: channel weight (setup)
    const uint32_t *meta;   // per entry: (iq * nnu + mode) | kind << 31 (setup)
    const double *N;        // setup: phonon occupations [nq][nnu]
    const uint16_t *idx;
    const RowSeg *segs;
    const RowTile *tiles;
    const RowStrip *strips;
    const int32_t *row_state, *state_row;
    const int32_t *cols;    // sparse staging: the strips' lists of referenced partner rows (null: tiles cover row ranges)
    int32_t Rb, Ra, nstrip;
    int64_t ns;
    const double *Fc;       // F of the compact rows, [nrows][3] (row_compact_kernel), padded by 2 doubles
    const double *v, *tau;
    double *out;            // API layout [3][ns] (Gamma [ns] in setup); the iteration may pass null between chained iterations
    double *Fc_out;         // iteration: compact [nrows][3] copy of the result for the next chained iteration, may be null
#ifdef EPHC_ROW_TIMING
    unsigned long long *dbg;
#endif
};

inline size_t row_smem_bytes(int Rb, int Ra) { return ((size_t)Rb + (size_t)Ra) * 3 * sizeof(double) + 48; }

// F[3][ns] (API layout) -> Fc[nrows][3]: the rows a tile stages are then one contiguous block
__global__ void __launch_bounds__(256) row_compact_kernel(const double *F, const int32_t *row_state, double *Fc, int nrows,
                                                           int64_t ns) {
    const int r = blockIdx.x * blockDim.x + threadIdx.x;
    if (r < nrows) {
        const int64_t s = row_state[r];
#pragma unroll
        for (int c = 0; c < 3; ++c) Fc[(int64_t)r * 3 + c] = F[(int64_t)c * ns + s];
    }
}

__device__ __forceinline__ void cp_async16(void *smem_dst, const void *gmem_src) {
    const unsigned d = (unsigned)__cvta_generic_to_shared(smem_dst);
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;\n" ::"r"(d), "l"(gmem_src));
}
__device__ __forceinline__ void row_cp_async8(void *smem_dst, const void *gmem_src) {
    const unsigned d = (unsigned)__cvta_generic_to_shared(smem_dst);
    asm volatile("cp.async.ca.shared.global [%0], [%1], 8;\n" ::"r"(d), "l"(gmem_src));
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;\n" ::); }
template <int N>
__device__ __forceinline__ void cp_async_wait() {
    asm volatile("cp.async.wait_group %0;\n" ::"n"(N));
}

// weights of the gather store (written by its transport_setup kernel) -> row-store order
__global__ void __launch_bounds__(256) row_permute_kernel(const double *gW, const uint32_t *perm, double *W, int64_t n) {
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n) W[i] = __ldg(gW + __ldcs(perm + i));
}

// f0[ns] -> f0 of the compact rows (the rows a tile stages are then one contiguous block)
__global__ void __launch_bounds__(256) row_compact1_kernel(const double *f, const int32_t *row_state, double *fc, int nrows) {
    const int r = blockIdx.x * blockDim.x + threadIdx.x;
    if (r < nrows) fc[r] = f[row_state[r]];
}

__device__ __forceinline__ double ld_keep(const double *p, uint64_t policy) {
    double v;
    asm volatile("ld.global.nc.L2::cache_hint.f64 %0, [%1], %2;\n" : "=d"(v) : "l"(p), "l"(policy));
    return v;
}

// transport_setup on the row store (reading R-16): per ordered term a <- b
//     W(a<-b) = w (1 + N - f0_b)  (emission as seen from a)   or   w (N + f0_b)  (absorption),
// written in row-store order for row_iter_kernel, and Gamma_a = sum_b W(a<-b).  Same walk as row_iter_kernel (one CTA per
// strip of destination rows, partner ranges staged in shared memory -- here f0, 8 bytes per row --, 8 lanes per
// destination row); N[iq, nu] comes from the L2-resident table.
__global__ void __launch_bounds__(kRowThreads, 1024 / kRowThreads) row_setup_kernel(const RowParams P) {
    extern __shared__ double smem[];
    double *sF = smem;                   // staged f0 of the partner rows [Rb]
    double *sAcc = smem + (P.Rb + 2);    // [Ra]
    int *sNext = reinterpret_cast<int *>(sAcc + P.Ra);
    const int tid = threadIdx.x, lane = tid & 31;
    const int sub = lane / kRowGroup, gl = lane % kRowGroup;
    constexpr int GPW = 32 / kRowGroup;
    for (int64_t s = (int64_t)blockIdx.x * kRowThreads + tid; s < P.ns; s += (int64_t)gridDim.x * kRowThreads)
        if (P.state_row[s] < 0) P.out[s] = 0.0;  // states outside the window scatter nowhere
    if ((int)blockIdx.x >= P.nstrip) return;
    const RowStrip st = P.strips[blockIdx.x];
    for (int i = tid; i < st.nrows; i += kRowThreads) sAcc[i] = 0.0;
    uint64_t pol_keep;  // the N table is gathered by every strip while 22 bytes per entry stream through the L2
    asm volatile("createpolicy.fractional.L2::evict_last.b64 %0, 1.0;\n" : "=l"(pol_keep));
    const double *wb = P.wst + st.e0;
    const uint32_t *mb = P.meta + st.e0;
    const uint16_t *Ib = P.idx + st.e0;
    double *Wb = P.W + st.e0;
    for (int t = st.t0; t < st.t1; ++t) {
        const RowTile tl = P.tiles[t];
        __syncthreads();
        {
            if (P.cols != nullptr) {  // sparse staging: the partner rows this strip references
                const int32_t *cl = P.cols + tl.col0;
                for (int i = tid; i < tl.ncols; i += kRowThreads) row_cp_async8(sF + i, P.Fc + __ldg(cl + i));
            } else {
                const double *src = P.Fc + tl.col0;  // col0 is even: 16-byte aligned
                const int n16 = (tl.ncols + 1) / 2;
                for (int i = tid; i < n16; i += kRowThreads) cp_async16(sF + 2 * i, src + 2 * i);
            }
            cp_async_commit();
            if (tid == 0) *sNext = 0;
            cp_async_wait<0>();
        }
        __syncthreads();
        for (;;) {
            int g = 0;
            if (lane == 0) g = atomicAdd(sNext, GPW);
            const int sg0 = __shfl_sync(0xffffffffu, g, 0);
            if (sg0 >= tl.nseg) break;
            uint32_t start = 0, len = 0, row = 0;
            if (sg0 + sub < tl.nseg) {
                const uint4 q = __ldg(reinterpret_cast<const uint4 *>(P.segs + tl.seg0 + sg0 + sub));
                start = q.x;
                len = q.y;
                row = q.z;
            }
            uint32_t lmax = len;
            lmax = max(lmax, __shfl_xor_sync(0xffffffffu, lmax, 8));
            lmax = max(lmax, __shfl_xor_sync(0xffffffffu, lmax, 16));
            double acc = 0.0;
            constexpr int U = 4;
            for (uint32_t ib = 0; ib < lmax; ib += U * kRowGroup) {
                double wv[U], Nv[U];
                uint32_t mv[U];
                unsigned jv[U];
#pragma unroll
                for (int u = 0; u < U; ++u) {
                    const uint32_t ii = ib + gl + u * kRowGroup;
                    wv[u] = 0.0;
                    mv[u] = 0;
                    jv[u] = 0;
                    if (ii < len) {
                        wv[u] = __ldcs(wb + start + ii);
                        mv[u] = __ldcs(mb + start + ii);
                        jv[u] = __ldcs(Ib + start + ii);
                    }
                }
#pragma unroll
                for (int u = 0; u < U; ++u) Nv[u] = ld_keep(P.N + (mv[u] & 0x7fffffffu), pol_keep);
#pragma unroll
                for (int u = 0; u < U; ++u) {
                    const uint32_t ii = ib + gl + u * kRowGroup;
                    const double fb = sF[jv[u]];
                    const double W = (mv[u] >> 31) ? wv[u] * (1.0 + Nv[u] - fb) : wv[u] * (Nv[u] + fb);
                    if (ii < len) __stcs(Wb + start + ii, W);
                    acc += W;  // lanes past the end carry w = 0
                }
            }
#pragma unroll
            for (int o = kRowGroup / 2; o > 0; o >>= 1) acc += __shfl_xor_sync(0xffffffffu, acc, o);
            if (gl == 0 && sg0 + sub < tl.nseg) sAcc[row] += acc;  // the only writer of this row in this tile
        }
    }
    __syncthreads();
    for (int i = tid; i < st.nrows; i += kRowThreads) P.out[P.row_state[st.row0 + i]] = sAcc[i];
}

// mode-collapsed specialisation: weight of a (destination, partner) state pair = sum of the weights of its ordered terms
// (adjacent in the row store), in store order
__global__ void __launch_bounds__(256) row_collapse_kernel(const double *__restrict__ W, const uint32_t *__restrict__ first,
                                                           const uint16_t *__restrict__ count, double *__restrict__ Wc, int64_t n) {
    const int64_t c = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (c >= n) return;
    const double *src = W + first[c];
    const int cnt = count[c];
    double s = 0.0;
    for (int j = 0; j < cnt; ++j) s += src[j];
    Wc[c] = s;
}

__global__ void __launch_bounds__(kRowThreads, 1024 / kRowThreads) row_iter_kernel(const RowParams P) {
#ifdef EPHC_ROW_TIMING
    unsigned long long g0, g1, g2, g3;
    asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(g0));
#endif
    extern __shared__ double smem[];
    double *sF = smem;                       // staged partner rows [Rb][3]
    double *sAcc = smem + (P.Rb * 3 + 2);    // [Ra][3]
    int *sNext = reinterpret_cast<int *>(sAcc + P.Ra * 3);
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int sub = lane / kRowGroup, gl = lane % kRowGroup;
    constexpr int GPW = 32 / kRowGroup;  // row groups per warp

    // Chained iterations are launched with programmatic stream serialization: the next launch may take an SM as soon as
    // this CTA leaves it, and waits here until the previous launch has completed and its F is visible (plain launches:
    // both instructions do nothing).
    asm volatile("griddepcontrol.launch_dependents;\n" ::: "memory");
    asm volatile("griddepcontrol.wait;\n" ::: "memory");
    // states outside the window receive no contribution: F' = tau v (grid-stride over all states)
    if (P.out != nullptr)
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

#ifdef EPHC_ROW_TIMING
    asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(g1));
#endif
    for (int t = st.t0; t < st.t1; ++t) {
        const RowTile tl = P.tiles[t];
        __syncthreads();  // previous tile done with sF (and sAcc zeroed)
        {   // stage the tile's partner rows: 16-byte copies global -> shared, no registers in between
            if (P.cols != nullptr) {  // sparse staging: the partner rows this strip references, 24 bytes each
                const int32_t *cl = P.cols + tl.col0;
                for (int i = tid; i < tl.ncols * 3; i += kRowThreads) {
                    const int rr = i / 3, cc = i - 3 * rr;
                    row_cp_async8(sF + i, P.Fc + (int64_t)__ldg(cl + rr) * 3 + cc);
                }
            } else {
                const double *src = P.Fc + (int64_t)tl.col0 * 3;
                const int n16 = (tl.ncols * 3 + 1) / 2;
                for (int i = tid; i < n16; i += kRowThreads) cp_async16(sF + 2 * i, src + 2 * i);
            }
            cp_async_commit();
            if (tid == 0) *sNext = 0;
            cp_async_wait<0>();
        }
        __syncthreads();
        // segments are sorted by descending length; warps take four at a time from a shared counter
        // (order of execution only: every row has one segment per tile, hence one writer).  The header of the next
        // group of segments is fetched while the current one is processed, and its first batch of entries is loaded
        // during the last batch of the current one, so that no load latency is exposed between segments.
        auto fetch = [&](int &sg0, uint32_t &start, uint32_t &len, uint32_t &row) {
            int g = 0;
            if (lane == 0) g = atomicAdd(sNext, GPW);
            sg0 = __shfl_sync(0xffffffffu, g, 0);
            start = len = row = 0;
            if (sg0 + sub < tl.nseg) {
                const uint4 q = __ldg(reinterpret_cast<const uint4 *>(P.segs + tl.seg0 + sg0 + sub));
                start = q.x;
                len = q.y;
                row = q.z;
            }
        };
        double wn[kRowBatch];
        unsigned jn[kRowBatch];
        auto load_batch = [&](uint32_t start, uint32_t len, uint32_t i) {
#pragma unroll
            for (int u = 0; u < kRowBatch; ++u) {
                const uint32_t ii = i + u * kRowGroup;
                wn[u] = 0.0;
                jn[u] = 0;
                if (ii < len) {
                    wn[u] = __ldcs(Wb + start + ii);
                    jn[u] = __ldcs(Ib + start + ii);
                }
            }
        };
        int sg0, sgN;
        uint32_t start, len, row, startN, lenN, rowN;
        fetch(sg0, start, len, row);
        if (sg0 < tl.nseg) load_batch(start, len, gl);
        while (sg0 < tl.nseg) {
            fetch(sgN, startN, lenN, rowN);
            double a0 = 0.0, a1 = 0.0, a2 = 0.0;
            const uint32_t step = kRowBatch * kRowGroup;
            // all lanes of the warp run the same number of trips (the longest segment of the four)
            uint32_t lmax = len;
            lmax = max(lmax, __shfl_xor_sync(0xffffffffu, lmax, 8));
            lmax = max(lmax, __shfl_xor_sync(0xffffffffu, lmax, 16));
            for (uint32_t ib = 0; ib < lmax; ib += step) {
                double wv[kRowBatch];
                unsigned jv[kRowBatch];
#pragma unroll
                for (int u = 0; u < kRowBatch; ++u) {
                    wv[u] = wn[u];
                    jv[u] = jn[u];
                }
                if (ib + step < lmax)
                    load_batch(start, len, ib + step + gl);
                else if (sgN < tl.nseg)
                    load_batch(startN, lenN, gl);
#pragma unroll
                for (int u = 0; u < kRowBatch; ++u) {
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
            if (gl == 0 && sg0 + sub < tl.nseg) {  // the only writer of this row in this tile
                sAcc[row * 3 + 0] += a0;
                sAcc[row * 3 + 1] += a1;
                sAcc[row * 3 + 2] += a2;
            }
            sg0 = sgN;
            start = startN;
            len = lenN;
            row = rowN;
        }
    }
    __syncthreads();
#ifdef EPHC_ROW_TIMING
    asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(g2));
#endif
    for (int i = tid; i < st.nrows; i += kRowThreads) {
        const int64_t s = P.row_state[st.row0 + i];
        const double ta = P.tau[s];
#pragma unroll
        for (int c = 0; c < 3; ++c) {
            const double val = ta * (P.v[(int64_t)c * P.ns + s] + sAcc[i * 3 + c]);
            if (P.out != nullptr) P.out[(int64_t)c * P.ns + s] = val;
            if (P.Fc_out != nullptr) P.Fc_out[(int64_t)(st.row0 + i) * 3 + c] = val;
        }
    }
#ifdef EPHC_ROW_TIMING
    __syncthreads();
    asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(g3));
    if (tid == 0 && P.dbg) {
        P.dbg[4 * blockIdx.x] = g0;
        P.dbg[4 * blockIdx.x + 1] = g1;
        P.dbg[4 * blockIdx.x + 2] = g2;
        P.dbg[4 * blockIdx.x + 3] = g3;
    }
#endif
}

}  // namespace ephc
