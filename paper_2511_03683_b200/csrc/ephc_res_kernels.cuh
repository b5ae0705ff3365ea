// ephc_res_kernels.cuh -- sm_100a kernel of the resident-tile store (variant 3): collision integral with once-stored
// directed entries (step 2 "contribution of every channel" and step 3 "sum over the channels of a
// state" in one kernel; the per-channel terms -- the paper's sc_col -- overwrite the weights in shared memory and
// never reach HBM).
//
// A CTA takes runs (consecutive tiles of one strip of k rows) from a global counter, largest first.  Per tile:
//   load     one elected thread fetches the tile image (codes, gather lists, row tables, weights: one contiguous
//            blob) with bulk copies that complete on an mbarrier (TMA, UBLKCP); meanwhile all threads stage f of the
//            tile's B rows and N[iq,:] of its pairs with cp.async;
//   phase 1  one lane per out-row piece: T = w [(f_out - f_in) N + f_out (1 - f_in)] (Eq. 2, reading R-1, emission
//            form; absorption weights are stored as the reversed entry), T overwrites w, the lane's -sum(T) goes to the
//            X tail;
//   phase 2  one lane per gather task: sums the X values listed for one row (T of its in-entries, sums of its out
//            pieces) and adds them to the row's accumulator (one owner per row and round: no atomics, fixed order,
//            bit-reproducible).
// The accumulators of the strip stay in shared memory for the whole run; B rows go to their partial-sum slot after
// every tile, A rows at the end of the run; finish_kernel (ephc_tile_kernels.cuh) adds the slots per state.
#pragma once
#include <cuda_runtime.h>

#include "ephc_internal.h"
#include "ephc_row_kernels.cuh"  // cp_async helpers

namespace ephc {

struct ResParams {
    const unsigned char *blob;
    const uint32_t *iqn;
    const ResTile *tiles;
    const ResRun *runs;
    const int32_t *order;   // runs by descending work
    int *counter;           // next position in `order` (reset by finish_kernel)
    int32_t nrun;
    const int32_t *row_state;
    const int64_t *slot_off;
    int32_t Rcap, nnu;
    uint32_t gran_magic;    // ceil(2^32 / granules per N row); 0 when there is one granule per row
    int32_t gran;           // granules per N row: nnu/2 pieces of 16 bytes, or nnu pieces of 8 bytes
    int32_t gran16;         // 1: 16-byte granules
    const double *f, *N;
    double *part;
};

inline size_t res_smem_bytes(int Rcap, int64_t smem_tile) { return (size_t)16 * Rcap + (size_t)smem_tile + 256; }

__device__ __forceinline__ void res_cp_async8(void *smem_dst, const void *gmem_src) {
    const unsigned d = (unsigned)__cvta_generic_to_shared(smem_dst);
    asm volatile("cp.async.ca.shared.global [%0], [%1], 8;\n" ::"r"(d), "l"(gmem_src));
}
__device__ __forceinline__ void mbar_init(uint64_t *bar, unsigned count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;\n" ::"r"((unsigned)__cvta_generic_to_shared(bar)), "r"(count));
}
__device__ __forceinline__ void mbar_expect_tx(uint64_t *bar, unsigned bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;\n" ::"r"((unsigned)__cvta_generic_to_shared(bar)),
                 "r"(bytes)
                 : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t *bar, unsigned parity) {
    const unsigned a = (unsigned)__cvta_generic_to_shared(bar);
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "WAIT_%=:\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
        "@p bra DONE_%=;\n"
        "bra WAIT_%=;\n"
        "DONE_%=:\n"
        "}\n" ::"r"(a),
        "r"(parity)
        : "memory");
}
// bulk copy global -> shared, completion counted in bytes on the mbarrier; the stream is read once: evict-first in L2
__device__ __forceinline__ void bulk_g2s(void *smem_dst, const void *gmem_src, unsigned bytes, uint64_t *bar, uint64_t policy) {
    asm volatile(
        "cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes.L2::cache_hint [%0], [%1], %2, [%3], %4;\n" ::"r"(
            (unsigned)__cvta_generic_to_shared(smem_dst)),
        "l"(gmem_src), "r"(bytes), "r"((unsigned)__cvta_generic_to_shared(bar)), "l"(policy)
        : "memory");
}

template <int NT>
__global__ void __launch_bounds__(NT, 2) res_kernel(const ResParams P) {
    constexpr int NW = NT / 32;
    extern __shared__ __align__(128) unsigned char res_smem[];
    double *sF = reinterpret_cast<double *>(res_smem);     // f of the A rows, then of the B rows
    double *sAcc = sF + P.Rcap;                             // accumulators, same indexing
    unsigned char *sBlob = reinterpret_cast<unsigned char *>(sAcc + P.Rcap);
    __shared__ __align__(8) uint64_t sBar;
    __shared__ int sRunNo;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int nnu = P.nnu;
    unsigned parity = 0;
    uint64_t policy;
    asm volatile("createpolicy.fractional.L2::evict_first.b64 %0, 1.0;\n" : "=l"(policy));
    if (tid == 0) {
        mbar_init(&sBar, 1);
        asm volatile("fence.mbarrier_init.release.cluster;\n" ::: "memory");
    }
    __syncthreads();

    while (true) {
        if (tid == 0) sRunNo = atomicAdd(P.counter, 1);  // order of execution only: every run owns its slots
        __syncthreads();
        const int rno = sRunNo;
        if (rno >= P.nrun) break;
        const ResRun run = P.runs[P.order[rno]];
        const int a_rows = run.a_rows;
        for (int r = tid; r < a_rows; r += NT) {
            res_cp_async8(sF + r, P.f + P.row_state[run.a_row0 + r]);
            sAcc[r] = 0.0;
        }
        for (int ti = 0; ti < run.nt; ++ti) {
            const ResTile D = P.tiles[run.t0 + ti];
            const ResLayout L = res_layout(D.ne, D.npiece, D.ntask1, D.ntask2, D.nc1 + D.nc2 + D.nc3, D.ngl1 + D.ngl2);
            double *X = reinterpret_cast<double *>(sBlob + L.w);
            double *sN = reinterpret_cast<double *>(sBlob + ((L.w + 8 * (D.ne + D.npiece + D.npart) + 15) & ~15));
            // ---- load ------------------------------------------------------------------------------------------------
            if (tid == 0) {
                // the previous tile's generic-proxy accesses to this buffer are ordered before the bulk copy
                asm volatile("fence.proxy.async.shared::cta;\n" ::: "memory");
                mbar_expect_tx(&sBar, (unsigned)D.blob_bytes);
                const unsigned char *src = P.blob + D.blob_off;
                for (int o = 0; o < D.blob_bytes; o += 32768)
                    bulk_g2s(sBlob + o, src + o, (unsigned)min(32768, D.blob_bytes - o), &sBar, policy);
            }
            for (int i = tid; i < D.b_rows; i += NT) {
                res_cp_async8(sF + a_rows + i, P.f + P.row_state[D.b_row0 + i]);
                sAcc[a_rows + i] = 0.0;
            }
            {
                const int total = D.nq * P.gran;
                const uint32_t *iqn = P.iqn + D.q0;
                for (int i = tid; i < total; i += NT) {
                    const int pr = P.gran_magic ? (int)__umulhi((unsigned)i, P.gran_magic) : i, part = i - pr * P.gran;
                    if (P.gran16) {
                        cp_async16(sN + pr * nnu + 2 * part, P.N + (size_t)__ldg(iqn + pr) + 2 * part);
                    } else {
                        res_cp_async8(sN + pr * nnu + part, P.N + (size_t)__ldg(iqn + pr) + part);
                    }
                }
            }
            cp_async_commit();
            cp_async_wait<0>();
            mbar_wait(&sBar, parity);
            parity ^= 1u;
            __syncthreads();
            const uint32_t *code = reinterpret_cast<const uint32_t *>(sBlob + L.code);
            const uint16_t *perm = reinterpret_cast<const uint16_t *>(sBlob + L.perm);
            const uint16_t *prow = reinterpret_cast<const uint16_t *>(sBlob + L.prow);
            const uint16_t *d1 = reinterpret_cast<const uint16_t *>(sBlob + L.d1);
            const uint16_t *d2 = reinterpret_cast<const uint16_t *>(sBlob + L.d2);
            const uint32_t *cols = reinterpret_cast<const uint32_t *>(sBlob + L.cols);
            // ---- phase 1: Eq. 2 summand per entry, one lane per out-row piece ------------------------------------------
            for (int s0 = warp * 32; s0 < D.npiece; s0 += NW * 32) {
                const int p = s0 + lane;
                const bool valid = p < D.npiece;
                const double xo = sF[valid ? prow[p] : 0];
                double acc = 0.0;
                for (int j = 0; j < D.nc1; ++j) {
                    const uint32_t c = cols[j];
                    const int cnt = (int)(c & 0xffffu);
                    if (s0 >= cnt) break;  // lists descend in length: nothing left in this group of 32
                    if (p < cnt) {
                        const int e = (int)(c >> 16) + p;
                        const uint32_t cd = code[e];
                        const double wv = X[e];
                        const double xi = *reinterpret_cast<const double *>(reinterpret_cast<const unsigned char *>(sF) + (cd & 0xfff8u));
                        const double Nn = *reinterpret_cast<const double *>(reinterpret_cast<const unsigned char *>(sN) + (cd >> 16));
                        const double T = wv * fma(xo - xi, Nn, fma(-xo, xi, xo));
                        X[e] = T;
                        acc += T;
                    }
                }
                if (valid) X[D.ne + p] = -acc;
            }
            __syncthreads();
            // ---- phase 2, round 1: one lane per gather task -------------------------------------------------------------
            {
                const uint32_t *cols2 = cols + D.nc1;
                for (int s0 = warp * 32; s0 < D.ntask1; s0 += NW * 32) {
                    const int t = s0 + lane;
                    double acc = 0.0;
                    for (int j = 0; j < D.nc2; ++j) {
                        const uint32_t c = cols2[j];
                        const int cnt = (int)(c & 0xffffu);
                        if (s0 >= cnt) break;
                        if (t < cnt) acc += X[perm[(int)(c >> 16) + t]];
                    }
                    if (t < D.ntask1) {
                        const int dst = d1[t];
                        if (dst & 0x8000)
                            X[D.ne + D.npiece + (dst & 0x7fff)] = acc;
                        else
                            sAcc[dst] += acc;
                    }
                }
            }
            if (D.ntask2 > 0) {  // rows with more than Lg inputs: their partial sums are added in a second round
                __syncthreads();
                const uint32_t *cols3 = cols + D.nc1 + D.nc2;
                const uint16_t *perm2 = perm + D.ngl1;
                for (int s0 = warp * 32; s0 < D.ntask2; s0 += NW * 32) {
                    const int t = s0 + lane;
                    double acc = 0.0;
                    for (int j = 0; j < D.nc3; ++j) {
                        const uint32_t c = cols3[j];
                        const int cnt = (int)(c & 0xffffu);
                        if (s0 >= cnt) break;
                        if (t < cnt) acc += X[perm2[(int)(c >> 16) + t]];
                    }
                    if (t < D.ntask2) sAcc[d2[t]] += acc;
                }
            }
            asm volatile("fence.proxy.async.shared::cta;\n" ::: "memory");  // T was written over w: order it before the next bulk copy
            __syncthreads();
            if (D.b_rows > 0) {
                double *dst = P.part + P.slot_off[D.b_slot];
                for (int i = tid; i < D.b_rows; i += NT) dst[i] = sAcc[a_rows + i];
            }
        }
        {
            double *dst = P.part + P.slot_off[run.a_slot];
            for (int i = tid; i < a_rows; i += NT) dst[i] = sAcc[i];
        }
        __syncthreads();  // sRunNo, sF and sAcc are free again
    }
}

}  // namespace ephc
