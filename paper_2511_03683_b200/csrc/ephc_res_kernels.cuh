// ephc_res_kernels.cuh -- sm_100a kernel of the resident-tile store (variant 3): collision integral with once-stored
// directed entries (step 2 "contribution of every channel" and step 3 "sum over the channels of a
// state" in one kernel; the per-channel terms -- the paper's sc_col -- overwrite the weights in shared memory and
// never reach HBM).
//
// One persistent CTA per SM walks its host-assigned sequence of tiles with two tile buffers in shared memory.
// While tile i is computed, tile i+1 is loaded: one elected thread issues bulk copies (TMA, UBLKCP) of the tile
// image (codes, gather lists, row tables, weights: one contiguous blob) and of the compact f values of its A and B
// rows, all completing on the buffer's mbarrier; all threads stage N[iq,:] of its pairs with cp.async, reading the
// pairs' iq from a list that came with the image of tile i.  Per tile:
//   phase 1  one lane per out-row piece: T = w [(f_out - f_in) N + f_out (1 - f_in)] (Eq. 2, reading R-1, emission
//            form; absorption weights are stored as the reversed entry), T overwrites w, the lane's -sum(T) goes to the
//            X tail;
//   phase 2  one lane per gather task: sums the X values listed for one row (T of its in-entries, sums of its out
//            pieces) and adds them to the row's accumulator (one owner per row and round: no atomics, fixed order,
//            bit-reproducible).
// The accumulators of the strip (A rows) stay in shared memory for a run of tiles; B rows go to their partial-sum slot
// after every tile, A rows at the end of the run; finish_kernel (ephc_tile_kernels.cuh) adds the slots per state.
#pragma once
#include <cuda_runtime.h>

#include "ephc_internal.h"
#include "ephc_row_kernels.cuh"  // cp_async helpers

namespace ephc {

struct ResParams {
    const unsigned char *blob;
    const uint32_t *iqn;
    const ResTile *tiles;     // schedule order
    const int32_t *cta_ptr;   // tiles of CTA c: [cta_ptr[c], cta_ptr[c+1])
    const int64_t *slot_off;
    int32_t Ra, Rcap, RbMax, nnu;
    uint32_t buf_bytes, fixed_bytes;
    uint32_t gran_magic;    // ceil(2^32 / granules per N row); 0 when there is one granule per row
    int32_t gran;           // granules per N row: nnu/2 pieces of 16 bytes, or nnu pieces of 8 bytes
    int32_t gran16;         // 1: 16-byte granules
    const double *fc;       // f in compact row order (padded to an even number of rows)
    const double *N;
    double *part;
#ifdef EPHC_RES_TIMING
    long long *dbg;         // per CTA: cycles spent in 8 sections (working builds only)
#endif
};

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
// bulk copy global -> shared, completion counted in bytes on the mbarrier
__device__ __forceinline__ void bulk_g2s(void *smem_dst, const void *gmem_src, unsigned bytes, uint64_t *bar, uint64_t policy) {
    asm volatile(
        "cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes.L2::cache_hint [%0], [%1], %2, [%3], %4;\n" ::"r"(
            (unsigned)__cvta_generic_to_shared(smem_dst)),
        "l"(gmem_src), "r"(bytes), "r"((unsigned)__cvta_generic_to_shared(bar)), "l"(policy)
        : "memory");
}

// f in compact row order: bulk copies need contiguous, 16-byte aligned sources
__global__ void __launch_bounds__(256) res_compact_kernel(const double *__restrict__ f, const int32_t *__restrict__ row_state,
                                                          double *__restrict__ fc, int nrows) {
    const int r = blockIdx.x * blockDim.x + threadIdx.x;
    if (r < nrows) fc[r] = f[row_state[r]];
}

__device__ __forceinline__ void mbar_arrive(uint64_t *bar) {
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];\n" ::"r"((unsigned)__cvta_generic_to_shared(bar)) : "memory");
}
// the mbarrier will also wait for all cp.async copies this thread has issued so far (counted in its expected arrivals)
__device__ __forceinline__ void mbar_arrive_cp_async(uint64_t *bar) {
    asm volatile("cp.async.mbarrier.arrive.noinc.shared::cta.b64 [%0];\n" ::"r"((unsigned)__cvta_generic_to_shared(bar)) : "memory");
}
__device__ __forceinline__ void consumer_sync(int nthreads) { asm volatile("bar.sync 1, %0;\n" ::"r"(nthreads) : "memory"); }

// NL consumer threads (= lanes of a tile image) + one producer warp
template <int NL>
__global__ void __launch_bounds__(NL + 32, kResCtasPerSm) res_kernel(const ResParams P) {
    extern __shared__ __align__(128) unsigned char res_smem[];
    double *sAccA = reinterpret_cast<double *>(res_smem);                  // accumulators of the strip (run)
    ResTile *sD = reinterpret_cast<ResTile *>(res_smem + 8 * P.Ra);        // directory entries of tiles i, i+1, i+2
    __shared__ __align__(8) uint64_t sFull[2], sEmpty[2];
    __shared__ double sDummy;
    const int tid = threadIdx.x, wbase = tid & ~31;
    const int nnu = P.nnu;
    const int i0 = P.cta_ptr[blockIdx.x], n = P.cta_ptr[blockIdx.x + 1] - i0;
    if (n <= 0) return;
    if (tid == 0) {
        mbar_init(&sFull[0], 33);        // the producer's expect_tx arrive + the cp.async arrives of its 32 lanes
        mbar_init(&sFull[1], 33);
        mbar_init(&sEmpty[0], NL / 32);  // one arrive per consumer warp
        mbar_init(&sEmpty[1], NL / 32);
        asm volatile("fence.mbarrier_init.release.cluster;\n" ::: "memory");
    }
    for (int r = tid; r < P.Ra; r += NL + 32) sAccA[r] = 0.0;
    __syncthreads();
    auto buf_of = [&](int b) { return res_smem + P.fixed_bytes + (size_t)b * P.buf_bytes; };

    if (tid >= NL) {
        // ===== producer warp: everything a tile needs, up to two tiles ahead of the consumers ==============================
        const int lane = tid - NL;
        uint64_t pol_stream, pol_keep;
        asm volatile("createpolicy.fractional.L2::evict_first.b64 %0, 1.0;\n" : "=l"(pol_stream));  // the store is read once
        asm volatile("createpolicy.fractional.L2::evict_last.b64 %0, 1.0;\n" : "=l"(pol_keep));     // f is read by every tile
        for (int j = 0; j < n; ++j) {
            const int b = j & 1;
            if (j >= 2) mbar_wait(&sEmpty[b], (unsigned)((j >> 1) - 1) & 1u);  // the consumers are done with tile j - 2
            {   // directory entry of tile j, word by word
                const int32_t *src = reinterpret_cast<const int32_t *>(&P.tiles[i0 + j]);
                int32_t *dst = reinterpret_cast<int32_t *>(&sD[j % 3]);
                dst[lane] = src[lane];
                if (lane + 32 < kResTileWords) dst[lane + 32] = src[lane + 32];
            }
            __syncwarp();
            const ResTile &D = sD[j % 3];
            unsigned char *buf = buf_of(b);
            double *sF = reinterpret_cast<double *>(buf);
            double *sAccB = sF + P.Rcap;
            unsigned char *sBlob = reinterpret_cast<unsigned char *>(sAccB + P.RbMax);
            double *sN = reinterpret_cast<double *>(sBlob + D.o_sn);
            if (lane == 0) {
                const int a_rows = D.a_rows, b_rows = D.b_rows, bytes = D.blob_bytes;
                const unsigned fa = (unsigned)((8 * a_rows + 15) & ~15), fb = (unsigned)((8 * b_rows + 15) & ~15);
                asm volatile("fence.proxy.async.shared::cta;\n" ::: "memory");
                mbar_expect_tx(&sFull[b], (unsigned)bytes + fa + fb);
                const unsigned char *src = P.blob + D.blob_off;
                for (int o = 0; o < bytes; o += 32768) bulk_g2s(sBlob + o, src + o, (unsigned)min(32768, bytes - o), &sFull[b], pol_stream);
                bulk_g2s(sF, P.fc + D.a_row0, fa, &sFull[b], pol_keep);
                if (fb) bulk_g2s(sF + a_rows, P.fc + D.b_row0, fb, &sFull[b], pol_keep);
            }
            for (int k = lane; k < D.b_rows; k += 32) sAccB[k] = 0.0;
            // N[iq, :] of the tile's pairs; their iq * nnu came with the image of the previous tile
            const uint32_t *iq = P.iqn + D.q0;
            if (j > 0) {
                mbar_wait(&sFull[b ^ 1], (unsigned)((j - 1) >> 1) & 1u);
                const unsigned char *prev = buf_of(b ^ 1) + 8 * (size_t)(P.Rcap + P.RbMax);
                iq = reinterpret_cast<const uint32_t *>(prev + sD[(j - 1) % 3].o_nxt);
            }
            const int total = D.nq * P.gran;
            for (int g = lane; g < total; g += 32) {
                const int pr = P.gran_magic ? (int)__umulhi((unsigned)g, P.gran_magic) : g, part = g - pr * P.gran;
                const double *src = P.N + (size_t)iq[pr];
                if (P.gran16)
                    cp_async16(sN + pr * nnu + 2 * part, src + 2 * part);
                else
                    res_cp_async8(sN + pr * nnu + part, src + part);
            }
            mbar_arrive_cp_async(&sFull[b]);
        }
        return;
    }

    // ===== consumers ==========================================================================================================
#ifdef EPHC_RES_TIMING
    long long tacc[8] = {0, 0, 0, 0, 0, 0, 0, 0}, tprev = clock64();
#define EPHC_TICK(k)                         \
    {                                        \
        const long long tn_ = clock64();     \
        tacc[k] += tn_ - tprev;              \
        tprev = tn_;                         \
    }
#else
#define EPHC_TICK(k)
#endif
    for (int i = 0; i < n; ++i) {
        const int b = i & 1;
        unsigned char *buf = buf_of(b);
        double *sF = reinterpret_cast<double *>(buf);
        double *sAccB = sF + P.Rcap;
        unsigned char *sBlob = reinterpret_cast<unsigned char *>(sAccB + P.RbMax);
        EPHC_TICK(0)
        mbar_wait(&sFull[b], (unsigned)(i >> 1) & 1u);
        EPHC_TICK(1)
        const ResTile &D = sD[i % 3];
        const int ne = D.ne, npiece = D.npiece, a_rows = D.a_rows, nc1 = D.nc1, nc2 = D.nc2;
        double *X = reinterpret_cast<double *>(sBlob + D.o_w);
        const uint32_t *code = reinterpret_cast<const uint32_t *>(sBlob);
        const uint16_t *perm = reinterpret_cast<const uint16_t *>(sBlob + D.o_perm);
        const uint16_t *prow = reinterpret_cast<const uint16_t *>(sBlob + D.o_prow);
        const uint32_t *cols = reinterpret_cast<const uint32_t *>(sBlob + D.o_cols);
        const unsigned char *sFb = reinterpret_cast<const unsigned char *>(sF);
        const unsigned char *sNb = sBlob + D.o_sn;
        // ---- phase 1: Eq. 2 summand per entry; a lane walks the pieces packed into it, four columns per step: all loads
        //      of a step are issued before its arithmetic, which is branch-free ------------------------------------------------
        {
            int piece = reinterpret_cast<const uint16_t *>(sBlob + D.o_pf)[tid];
            // f_out of the current piece and of the next two, row of the third: a sliding window that is refilled at every
            // piece end, so that no load sits between a piece end and the next entry
            double xo = sF[prow[piece]], xo1 = sF[prow[piece + 1]], xo2 = sF[prow[piece + 2]];
            int rn = prow[piece + 3];
            double s0 = 0.0, s1 = 0.0;  // sum of w and of w N over the current combo
            double acc = 0.0;
            for (int j = 0; j < nc1; j += 4) {
                const uint4 c4 = *reinterpret_cast<const uint4 *>(cols + j);
                if (wbase >= (int)(c4.x & 0xffffu)) break;  // lanes descend in load: nothing left for this warp
                const bool a0 = tid < (int)(c4.x & 0xffffu), a1 = tid < (int)(c4.y & 0xffffu), a2 = tid < (int)(c4.z & 0xffffu),
                           a3 = tid < (int)(c4.w & 0xffffu);
                const int e0 = a0 ? (int)(c4.x >> 16) + tid : 0, e1 = a1 ? (int)(c4.y >> 16) + tid : 0,
                          e2 = a2 ? (int)(c4.z >> 16) + tid : 0, e3 = a3 ? (int)(c4.w >> 16) + tid : 0;
                // an inactive lane reads entry 0 and treats it as "inside a combo" (no store, no sums)
                const uint32_t cd0 = a0 ? code[e0] : 2u, cd1 = a1 ? code[e1] : 2u, cd2 = a2 ? code[e2] : 2u, cd3 = a3 ? code[e3] : 2u;
                const double w0 = a0 ? X[e0] : 0.0, w1 = a1 ? X[e1] : 0.0, w2 = a2 ? X[e2] : 0.0, w3 = a3 ? X[e3] : 0.0;
                // f_in is needed only where a combo (entries of one lane with the same out and in rows) ends
                const double xi0 = (cd0 & 2u) ? 0.0 : *reinterpret_cast<const double *>(sFb + (cd0 & 0xfff8u));
                const double xi1 = (cd1 & 2u) ? 0.0 : *reinterpret_cast<const double *>(sFb + (cd1 & 0xfff8u));
                const double xi2 = (cd2 & 2u) ? 0.0 : *reinterpret_cast<const double *>(sFb + (cd2 & 0xfff8u));
                const double xi3 = (cd3 & 2u) ? 0.0 : *reinterpret_cast<const double *>(sFb + (cd3 & 0xfff8u));
                const double N0 = *reinterpret_cast<const double *>(sNb + (cd0 >> 16));
                const double N1 = *reinterpret_cast<const double *>(sNb + (cd1 >> 16));
                const double N2 = *reinterpret_cast<const double *>(sNb + (cd2 >> 16));
                const double N3 = *reinterpret_cast<const double *>(sNb + (cd3 >> 16));
                // sum_e w_e [(xo - xi) N_e + xo (1 - xi)] = (xo - xi) sum w_e N_e + xo (1 - xi) sum w_e over a combo
#define EPHC_RES_STEP(E, CD, W, XI, NN)                                                        \
    {                                                                                          \
        s1 = fma(W, NN, s1);                                                                   \
        s0 += W;                                                                               \
        const bool ce = !(CD & 2u), pe = (CD & 1u) != 0; /* last entry of a combo / piece */   \
        const double T = fma(xo - XI, s1, s0 * fma(-xo, XI, xo));                              \
        if (ce) X[E] = T;                                                                      \
        acc += ce ? T : 0.0;                                                                   \
        s1 = ce ? 0.0 : s1;                                                                    \
        s0 = ce ? 0.0 : s0;                                                                    \
        if (pe) X[ne + piece] = -acc;                                                          \
        acc = pe ? 0.0 : acc;                                                                  \
        piece += pe ? 1 : 0;                                                                   \
        xo = pe ? xo1 : xo;                                                                    \
        xo1 = pe ? xo2 : xo1;                                                                  \
        if (pe) xo2 = sF[rn];                                                                  \
        if (pe) rn = prow[piece + 3];                                                          \
    }
                EPHC_RES_STEP(e0, cd0, w0, xi0, N0)
                EPHC_RES_STEP(e1, cd1, w1, xi1, N1)
                EPHC_RES_STEP(e2, cd2, w2, xi2, N2)
                EPHC_RES_STEP(e3, cd3, w3, xi3, N3)
#undef EPHC_RES_STEP
            }
        }
        EPHC_TICK(2)
        consumer_sync(NL);
        EPHC_TICK(3)
        // ---- phase 2, round 1: a lane walks the gather tasks packed into it, four columns per step ----------------------------
        {
            const uint32_t *cols2 = cols + nc1;
            const uint16_t *d1 = reinterpret_cast<const uint16_t *>(sBlob + D.o_d1);
            int task = reinterpret_cast<const uint16_t *>(sBlob + D.o_tf)[tid];
            int dn = d1[task];  // destination of the current task, loaded one task ahead
            // the add of a finished task into its row's accumulator is completed at the next task end (or after the loop),
            // so that the warp never waits for the accumulator's old value
            double *pptr = &sDummy;
            double pold = 0.0, pacc = 0.0, acc = 0.0;
            for (int j = 0; j < nc2; j += 4) {
                const uint4 c4 = *reinterpret_cast<const uint4 *>(cols2 + j);
                if (wbase >= (int)(c4.x & 0xffffu)) break;
                const bool a0 = tid < (int)(c4.x & 0xffffu), a1 = tid < (int)(c4.y & 0xffffu), a2 = tid < (int)(c4.z & 0xffffu),
                           a3 = tid < (int)(c4.w & 0xffffu);
                const uint32_t wd0 = a0 ? perm[(int)(c4.x >> 16) + tid] : 0u, wd1 = a1 ? perm[(int)(c4.y >> 16) + tid] : 0u,
                               wd2 = a2 ? perm[(int)(c4.z >> 16) + tid] : 0u, wd3 = a3 ? perm[(int)(c4.w >> 16) + tid] : 0u;
                const double v0 = a0 ? X[wd0 & 0x7fffu] : 0.0, v1 = a1 ? X[wd1 & 0x7fffu] : 0.0, v2 = a2 ? X[wd2 & 0x7fffu] : 0.0,
                             v3 = a3 ? X[wd3 & 0x7fffu] : 0.0;
#define EPHC_RES_STEP(WD, V)                                                                   \
    {                                                                                          \
        acc += V;                                                                              \
        if (WD & 0x8000u) { /* last input of a task */                                         \
            *pptr = pold + pacc;                                                               \
            const int dst = dn;                                                                \
            dn = d1[++task];                                                                   \
            pptr = (dst & 0x8000) ? X + (ne + npiece + (dst & 0x7fff))                         \
                                  : (dst < a_rows ? sAccA + dst : sAccB + (dst - a_rows));     \
            pold = *pptr;                                                                      \
            if (dst & 0x8000) pold = 0.0;                                                      \
            pacc = acc;                                                                        \
            acc = 0.0;                                                                         \
        }                                                                                      \
    }
                EPHC_RES_STEP(wd0, v0)
                EPHC_RES_STEP(wd1, v1)
                EPHC_RES_STEP(wd2, v2)
                EPHC_RES_STEP(wd3, v3)
#undef EPHC_RES_STEP
            }
            *pptr = pold + pacc;
        }
        EPHC_TICK(4)
        if (D.ntask2 > 0) {  // rows whose inputs were cut: their partial sums are added in a second round
            consumer_sync(NL);
            const uint32_t *cols3 = cols + nc1 + nc2;
            const uint16_t *perm2 = perm + D.ngl1;
            const uint16_t *d2 = reinterpret_cast<const uint16_t *>(sBlob + D.o_d2);
            const int ntask2 = D.ntask2, nc3 = D.nc3;
            for (int t = tid; t < ((ntask2 + 31) & ~31); t += NL) {
                const int s0 = t & ~31;
                double acc = 0.0;
                for (int j = 0; j < nc3; ++j) {
                    const uint32_t c = cols3[j];
                    const int cnt = (int)(c & 0xffffu);
                    if (s0 >= cnt) break;
                    if (t < cnt) acc += X[perm2[(int)(c >> 16) + t]];
                }
                if (t < ntask2) {
                    const int dst = d2[t];
                    if (dst < a_rows)
                        sAccA[dst] += acc;
                    else
                        sAccB[dst - a_rows] += acc;
                }
            }
        }
        EPHC_TICK(5)
        consumer_sync(NL);
        EPHC_TICK(6)
        const int b_rows = D.b_rows;
        if (b_rows > 0) {
            double *dst = P.part + D.b_off;
            for (int k = tid; k < b_rows; k += NL) dst[k] = sAccB[k];
        }
        if (D.flags & 2) {  // last tile of its run: the strip's sums go to their slot
            double *dst = P.part + D.a_off;
            for (int k = tid; k < a_rows; k += NL) {
                dst[k] = sAccA[k];
                sAccA[k] = 0.0;
            }
        }
        // this warp is done with the buffer and with the directory entry: T was written over w, order it before the
        // producer's next bulk copy
        asm volatile("fence.proxy.async.shared::cta;\n" ::: "memory");
        __syncwarp();
        if ((tid & 31) == 0) mbar_arrive(&sEmpty[b]);
        EPHC_TICK(7)
    }
#ifdef EPHC_RES_TIMING
    if (P.dbg && (tid & 31) == 0)
        for (int k = 0; k < 8; ++k) P.dbg[((size_t)blockIdx.x * (NL / 32) + (tid >> 5)) * 8 + k] = tacc[k];
#endif
}

}  // namespace ephc
