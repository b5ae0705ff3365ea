// ephc_res_kernels.cuh -- sm_100a kernel of the resident-tile store (variant 3): collision integral with once-stored
// entries (step 2 "contribution of every channel" and step 3 "sum over the channels of a state" in one
// kernel; the per-channel terms -- the paper's sc_col -- overwrite the weights in shared memory and never reach HBM).
// Layout of a tile image: ephc_internal.h "resident-tile store".
//
// Persistent CTAs (one or two per SM) walk their host-assigned sequence of tiles with two tile buffers in shared memory.
// While the consumer warps compute tile i, four producer warps load tile i+1: one elected thread issues bulk copies (TMA,
// UBLKCP) of the tile image (codes, gather lists, slab tables, weights: one contiguous blob) and of the compact f values
// of its A and B rows, all completing on the buffer's mbarrier; all producer threads stage N[iq,:] of its pairs with
// cp.async (counted on the same mbarrier), reading the pairs' iq from a list that came with the image of tile i.  Per tile:
//   phase 1  a lane owns one piece of an owner row a (32 pieces per slab, column-major): per entry it gathers N and sums
//            |ws| N and the emission / absorption weights over the open combo (the entries with one partner b); at the
//            combo's last entry it gathers f_b and forms T (Eq. 2 with reading R-1, summed over the combo), written over
//            that entry's weight; the lane's sum of T is subtracted from the strip's accumulator of row a;
//   phase 2  a lane owns one piece of a partner row b: it gathers the terms T listed for it and stores their sum to the
//            tile's partial-sum slot (global memory), or adds it to the strip's accumulator on a diagonal tile.
// One owner per row and phase: no atomics, fixed order, bit-reproducible.  The accumulators of the strip
// (A rows) stay in shared memory for a run of tiles and go to their slot at the end of the run; finish_kernel
// (ephc_tile_kernels.cuh) adds the slots per state.
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
    long long *tile_cycles; // calibration (null otherwise): cycles the consumers spent on every tile, in storage order
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

// Segmented sum over the lanes of a slab that own the same row (adjacent lanes): afterwards the first lane of every
// group holds the group's sum (fixed tree order).  `same` = lanes with this lane's row.
__device__ __forceinline__ double res_group_sum(double acc, unsigned same, int lane) {
#pragma unroll
    for (int d = 1; d < 32; d <<= 1) {
        const double v = __shfl_down_sync(0xffffffffu, acc, d);
        if (lane + d < 32 && ((same >> (lane + d)) & 1u)) acc += v;
    }
    return acc;
}

// NL consumer threads + one producer warp
#ifndef EPHC_RES_PRODUCERS
#define EPHC_RES_PRODUCERS 4  // 2: Si 127 us, GaAs 1622 us; 4: 104, 1541; 8: 102, 1620 (collision call)
#endif
constexpr int kResProducerWarps = EPHC_RES_PRODUCERS;  // one of them loads the tile image and f; all of them stage the N rows of the tile's pairs
constexpr int kResProducerThreads = 32 * kResProducerWarps;
__device__ __forceinline__ void producer_sync() { asm volatile("bar.sync 2, %0;\n" ::"n"(kResProducerThreads) : "memory"); }

template <int NL, int CTAS>
__global__ void __launch_bounds__(NL + kResProducerThreads, CTAS) res_kernel(const ResParams P) {
    extern __shared__ __align__(128) unsigned char res_smem[];
    double *sAccA = reinterpret_cast<double *>(res_smem);                  // accumulators of the strip (run)
    ResTile *sD = reinterpret_cast<ResTile *>(res_smem + 8 * P.Ra);        // directory entries of tiles i, i+1, i+2
    __shared__ __align__(8) uint64_t sFull[2], sEmpty[2];
    const int tid = threadIdx.x;
    const int nnu = P.nnu;
    const int i0 = P.cta_ptr[blockIdx.x], n = P.cta_ptr[blockIdx.x + 1] - i0;
    if (n <= 0) return;
    if (tid == 0) {
        mbar_init(&sFull[0], kResProducerThreads + 1);  // the loader's expect_tx arrive + the cp.async arrives of the producer threads (N rows)
        mbar_init(&sFull[1], kResProducerThreads + 1);
        mbar_init(&sEmpty[0], NL / 32);  // one arrive per consumer warp
        mbar_init(&sEmpty[1], NL / 32);
        asm volatile("fence.mbarrier_init.release.cluster;\n" ::: "memory");
    }
    for (int r = tid; r < P.Ra; r += NL + kResProducerThreads) sAccA[r] = 0.0;
    __syncthreads();
    auto buf_of = [&](int b) { return res_smem + P.fixed_bytes + (size_t)b * P.buf_bytes; };

    if (tid >= NL) {
        // ===== producer warps: everything a tile needs, up to two tiles ahead of the consumers; the N rows are staged while
        // the consumers compute (their cp.async wavefronts fill the LSU cycles that the latency-bound phases leave idle) ======
        const int ptid = tid - NL, lane = ptid & 31, pw = ptid >> 5;
        uint64_t pol_stream, pol_keep;
        asm volatile("createpolicy.fractional.L2::evict_first.b64 %0, 1.0;\n" : "=l"(pol_stream));  // the store is read once
        asm volatile("createpolicy.fractional.L2::evict_last.b64 %0, 1.0;\n" : "=l"(pol_keep));     // f is read by every tile
#ifdef EPHC_RES_TIMING
        long long pacc[8] = {0, 0, 0, 0, 0, 0, 0, 0}, pprev = clock64();
#define EPHC_PTICK(k)                        \
    {                                        \
        const long long tn_ = clock64();     \
        pacc[k] += tn_ - pprev;              \
        pprev = tn_;                         \
    }
#else
#define EPHC_PTICK(k)
#endif
        auto load_dir = [&](int j) {  // directory entry of tile j, word by word
            const int32_t *src = reinterpret_cast<const int32_t *>(&P.tiles[i0 + j]);
            int32_t *dst = reinterpret_cast<int32_t *>(&sD[j % 3]);
            if (lane < kResTileWords) dst[lane] = src[lane];
        };
        if (pw == 0) load_dir(0);
        for (int j = 0; j < n; ++j) {
            const int b = j & 1;
            EPHC_PTICK(0)
            if (j >= 2) mbar_wait(&sEmpty[b], (unsigned)((j >> 1) - 1) & 1u);  // the consumers are done with tile j - 2
            EPHC_PTICK(1)
            producer_sync();  // the directory entry of tile j (written by the loader warp one tile ago) is visible to all of them
            const ResTile &D = sD[j % 3];
            unsigned char *buf = buf_of(b);
            double *sF = reinterpret_cast<double *>(buf);
            unsigned char *sBlob = reinterpret_cast<unsigned char *>(sF + P.Rcap);
            if (ptid == 0) {
                const int a_rows = D.a_rows, b_rows = D.b_rows, bytes = D.blob_bytes;
                const unsigned fa = (unsigned)((8 * a_rows + 15) & ~15), fb = (unsigned)((8 * b_rows + 15) & ~15);
                *reinterpret_cast<double *>(sBlob + D.o_w + 8 * (size_t)D.ne_pad) = 0.0;  // the zero that padding reads
                asm volatile("fence.proxy.async.shared::cta;\n" ::: "memory");
                mbar_expect_tx(&sFull[b], (unsigned)bytes + fa + fb);
                const unsigned char *src = P.blob + D.blob_off;
                for (int o = 0; o < bytes; o += 32768) bulk_g2s(sBlob + o, src + o, (unsigned)min(32768, bytes - o), &sFull[b], pol_stream);
                bulk_g2s(sF, P.fc + D.a_row0, fa, &sFull[b], pol_keep);
                if (fb) bulk_g2s(sF + a_rows, P.fc + D.b_row0, fb, &sFull[b], pol_keep);
            }
            EPHC_PTICK(2)
            // the directory entry of the next tile (its slot was last used by tile j - 2), and its image on the way to the L2
            if (pw == 0 && j + 1 < n) {
                load_dir(j + 1);
                __syncwarp();
                if (lane == 0) {
                    const ResTile &Dn = sD[(j + 1) % 3];
                    asm volatile("cp.async.bulk.prefetch.L2.global [%0], %1;\n" ::"l"(P.blob + Dn.blob_off), "r"((unsigned)Dn.blob_bytes) : "memory");
                }
            }
            EPHC_PTICK(3)
            // N[iq, :] of the tile's pairs; their iq * nnu came with the image of the previous tile
            {
                double *sN = reinterpret_cast<double *>(sBlob + ((D.o_w + 8u * (unsigned)(D.ne_pad + 1) + 15u) & ~15u));
                const uint32_t *iq = P.iqn + D.q0;
                if (j > 0) {
                    mbar_wait(&sFull[b ^ 1], (unsigned)((j - 1) >> 1) & 1u);
                    const unsigned char *prev = buf_of(b ^ 1) + 8 * (size_t)P.Rcap;
                    iq = reinterpret_cast<const uint32_t *>(prev + sD[(j - 1) % 3].o_nxt);
                }
                const int total = D.nq * P.gran;
                for (int g = ptid; g < total; g += kResProducerThreads) {
                    const int pr = P.gran_magic ? (int)__umulhi((unsigned)g, P.gran_magic) : g, part = g - pr * P.gran;
                    const double *src = P.N + (size_t)iq[pr];
                    if (P.gran16)
                        cp_async16(sN + pr * nnu + 2 * part, src + 2 * part);
                    else
                        res_cp_async8(sN + pr * nnu + part, src + part);
                }
                mbar_arrive_cp_async(&sFull[b]);
            }
            EPHC_PTICK(4)
#ifdef EPHC_RES_TIMING
            mbar_wait(&sFull[b], (unsigned)(j >> 1) & 1u);  // working build only: how long until the tile is complete
            EPHC_PTICK(5)
#endif
        }
#ifdef EPHC_RES_TIMING
        if (P.dbg && ptid == 0)
            for (int k = 0; k < 8; ++k) P.dbg[((size_t)blockIdx.x * (NL / 32 + 1) + NL / 32) * 8 + k] = pacc[k];
#endif
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
    const int lane = tid & 31, warp = tid >> 5;
    constexpr int NW = NL / 32;
    long long cyc0 = P.tile_cycles != nullptr ? clock64() : 0;
    for (int i = 0; i < n; ++i) {
        const int b = i & 1;
        unsigned char *buf = buf_of(b);
        double *sF = reinterpret_cast<double *>(buf);
        unsigned char *sBlob = reinterpret_cast<unsigned char *>(sF + P.Rcap);
        EPHC_TICK(0)
        mbar_wait(&sFull[b], (unsigned)(i >> 1) & 1u);
        EPHC_TICK(1)
        const ResTile &D = sD[i % 3];
        const int a_rows = D.a_rows;
        double *X = reinterpret_cast<double *>(sBlob + D.o_w);
        const uint32_t *code = reinterpret_cast<const uint32_t *>(sBlob);
        const unsigned char *sFb = reinterpret_cast<const unsigned char *>(sF);
        const unsigned char *sNb = sBlob + ((D.o_w + 8u * (unsigned)(D.ne_pad + 1) + 15u) & ~15u);
        const uint16_t *wptr = reinterpret_cast<const uint16_t *>(sBlob + D.o_wptr);
        // ---- phase 1 (paper step 2): Eq. 2 summand per entry; a lane walks one piece of an a row ---------------------------
        {
            const uint16_t *srow = reinterpret_cast<const uint16_t *>(sBlob + D.o_srow1);
            const uint32_t *shdr = reinterpret_cast<const uint32_t *>(sBlob + D.o_shdr1);
            const int s1 = wptr[warp + 1];
            int s = wptr[warp];
            // header, row and f_a of the next slab are fetched while the current one is computed
            uint32_t hd = 0;
            unsigned u = kResNoRow;
            double xo = 0.0;
            if (s < s1) {
                hd = shdr[s];
                u = srow[32 * s + lane];
                xo = u != kResNoRow ? sF[u] : 0.0;
            }
            for (; s < s1; ++s) {
                const bool more = s + 1 < s1;
                const uint32_t hd_n = more ? shdr[s + 1] : 0u;
                const unsigned u_n = more ? srow[32 * (s + 1) + lane] : (unsigned)kResNoRow;
                const int base = (int)(hd & 1023u) * 32 + lane, H = (int)((hd >> kResHdrHShift) & kResHdrHMask);
                const uint32_t *c = code + base;
                double *x = X + base;
                double acc = 0.0;
                double S1 = 0.0, Se = 0.0, Sa = 0.0;  // over the open combo: sum |ws| N, sum of emission / absorption weights
                // columns in groups of four: the codes and weights of the next group are loaded before the current group's
                // gathers and arithmetic
                uint32_t c0 = c[0], c1 = 1 < H ? c[32] : 0u, c2 = 2 < H ? c[64] : 0u, c3 = 3 < H ? c[96] : 0u;
                double w0 = x[0], w1 = 1 < H ? x[32] : 0.0, w2 = 2 < H ? x[64] : 0.0, w3 = 3 < H ? x[96] : 0.0;
                for (int j = 0; j < H; j += 4) {
                    const bool q0 = j + 4 < H, q1 = j + 5 < H, q2 = j + 6 < H, q3 = j + 7 < H;
                    const uint32_t n0 = q0 ? c[128] : 0u, n1 = q1 ? c[160] : 0u, n2 = q2 ? c[192] : 0u, n3 = q3 ? c[224] : 0u;
                    const double v0 = q0 ? x[128] : 0.0, v1 = q1 ? x[160] : 0.0, v2 = q2 ? x[192] : 0.0, v3 = q3 ? x[224] : 0.0;
                    const double N0 = *reinterpret_cast<const double *>(sNb + (c0 >> 16)), N1 = *reinterpret_cast<const double *>(sNb + (c1 >> 16)),
                                 N2 = *reinterpret_cast<const double *>(sNb + (c2 >> 16)), N3 = *reinterpret_cast<const double *>(sNb + (c3 >> 16));
                    // f_b is needed where a combo ends only (bit 0; padding never ends one)
                    const double b0 = (c0 & 1u) ? *reinterpret_cast<const double *>(sFb + (c0 & 0xfff8u)) : 0.0,
                                 b1 = (c1 & 1u) ? *reinterpret_cast<const double *>(sFb + (c1 & 0xfff8u)) : 0.0,
                                 b2 = (c2 & 1u) ? *reinterpret_cast<const double *>(sFb + (c2 & 0xfff8u)) : 0.0,
                                 b3 = (c3 & 1u) ? *reinterpret_cast<const double *>(sFb + (c3 & 0xfff8u)) : 0.0;
#define EPHC_RES_ENTRY(CD, W, NN, FB, OFF)                                                              \
    {                                                                                                   \
        S1 = fma(fabs(W), NN, S1);                                                                      \
        Se += fmax(W, 0.0);                                                                             \
        Sa += fmin(W, 0.0);                                                                             \
        if ((CD) & 1u) { /* Eq. 2 summed over the combo (reading R-1; the sign of ws carries the kind) */ \
            const double p = xo * (FB);                                                                 \
            const double T = fma(xo - (FB), S1, fma(xo - p, Se, ((FB) - p) * Sa));                      \
            x[OFF] = T;                                                                                 \
            acc += T;                                                                                   \
            S1 = Se = Sa = 0.0;                                                                         \
        }                                                                                               \
    }
                    EPHC_RES_ENTRY(c0, w0, N0, b0, 0)
                    EPHC_RES_ENTRY(c1, w1, N1, b1, 32)
                    EPHC_RES_ENTRY(c2, w2, N2, b2, 64)
                    EPHC_RES_ENTRY(c3, w3, N3, b3, 96)
#undef EPHC_RES_ENTRY
                    c0 = n0, c1 = n1, c2 = n2, c3 = n3;
                    w0 = v0, w1 = v1, w2 = v2, w3 = v3;
                    c += 128;
                    x += 128;
                }
                const double xo_n = u_n != kResNoRow ? sF[u_n] : 0.0;
                bool head = true;
                if (hd & kResHdrMulti) {
                    const unsigned same = __match_any_sync(0xffffffffu, u);
                    acc = res_group_sum(acc, same, lane);
                    head = (same & ((1u << lane) - 1u)) == 0u;
                }
                if (u != kResNoRow && head) sAccA[u] -= acc;  // a rows are rows of the strip
                hd = hd_n;
                u = u_n;
                xo = xo_n;
            }
        }
        EPHC_TICK(2)
        consumer_sync(NL);
        EPHC_TICK(3)
        // ---- phase 2 (paper step 3): a lane sums the T values listed for one piece of a b row -------------------------------
        {
            const uint16_t *srow = reinterpret_cast<const uint16_t *>(sBlob + D.o_srow2);
            const uint32_t *shdr = reinterpret_cast<const uint32_t *>(sBlob + D.o_shdr2);
            const uint16_t *perm = reinterpret_cast<const uint16_t *>(sBlob + D.o_perm);
            double *bdst = P.part + D.b_off - a_rows;  // partial sum of local row u >= a_rows
            const int s1 = wptr[NW + 1 + warp + 1];
            int s = wptr[NW + 1 + warp];
            uint32_t hd = 0;
            unsigned u = kResNoRow;
            if (s < s1) {
                hd = shdr[s];
                u = srow[32 * s + lane];
            }
            for (; s < s1; ++s) {
                const bool more = s + 1 < s1;
                const uint32_t hd_n = more ? shdr[s + 1] : 0u;
                const unsigned u_n = more ? srow[32 * (s + 1) + lane] : (unsigned)kResNoRow;
                const int base = (int)(hd & 1023u) * 32 + lane, H = (int)((hd >> kResHdrHShift) & kResHdrHMask);
                const uint16_t *g = perm + base;
                double acc = 0.0;
                const unsigned zero = (unsigned)D.ne_pad;
                // eight columns per step: all positions, then all T values, then the adds (the lists are short: latency, not
                // bandwidth, bounds this phase)
                for (int j = 0; j < H; j += 8) {
                    unsigned p[8];
#pragma unroll
                    for (int k = 0; k < 8; ++k) p[k] = j + k < H ? g[32 * k] : zero;
                    double v[8];
#pragma unroll
                    for (int k = 0; k < 8; ++k) v[k] = X[p[k]];
#pragma unroll
                    for (int k = 0; k < 8; ++k) acc += v[k];
                    g += 256;
                }
                bool head = true;
                if (hd & kResHdrMulti) {
                    const unsigned same = __match_any_sync(0xffffffffu, u);
                    acc = res_group_sum(acc, same, lane);
                    head = (same & ((1u << lane) - 1u)) == 0u;
                }
                if (u != kResNoRow && head) {
                    if ((int)u < a_rows)
                        sAccA[u] += acc;   // diagonal tile: both ends in the strip
                    else
                        bdst[u] = acc;     // the only contribution of this tile to the row
                }
                hd = hd_n;
                u = u_n;
            }
        }
        EPHC_TICK(4)
        // the strip's accumulators are touched by phase 2 (diagonal tile) or flushed (end of a run): order that against
        // the next tile's phase 1
        const int flags = D.flags, b_rows = D.b_rows;
        if (b_rows == 0 || (flags & 2)) consumer_sync(NL);
        EPHC_TICK(5)
        if (flags & 2) {  // last tile of its run: the strip's sums go to their slot
            double *dst = P.part + D.a_off;
            for (int k = tid; k < a_rows; k += NL) {
                dst[k] = sAccA[k];
                sAccA[k] = 0.0;
            }
            consumer_sync(NL);
        }
        EPHC_TICK(6)
        // this warp is done with the buffer and with the directory entry: T was written over w, order it before the
        // producer's next bulk copy
        asm volatile("fence.proxy.async.shared::cta;\n" ::: "memory");
        __syncwarp();
        if (lane == 0) mbar_arrive(&sEmpty[b]);
        if (P.tile_cycles != nullptr && tid == 0) {  // from the end of the previous tile to the end of this one (waits included)
            const long long cyc1 = clock64();
            P.tile_cycles[i0 + i] = cyc1 - cyc0;
            cyc0 = cyc1;
        }
        EPHC_TICK(7)
    }
#ifdef EPHC_RES_TIMING
    if (P.dbg && lane == 0)
        for (int k = 0; k < 8; ++k) P.dbg[((size_t)blockIdx.x * (NW + 1) + warp) * 8 + k] = tacc[k];
#endif
}

}  // namespace ephc
