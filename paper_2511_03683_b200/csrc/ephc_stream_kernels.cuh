// ephc_stream_kernels.cuh -- sm_100a kernel of the stream store (variant 2): collision integral with once-stored
// channels, one LANE per ENTRY (step 2 "contribution of every channel", step 3 "sum over the
// channels of a state", here both inside one kernel and with the per-channel terms kept in shared memory instead of
// the paper's sc_col array in global memory).
//
// A CTA of 512 threads (two per SM) takes tiles from a global counter, largest first (strip of k rows x range of k' rows; f of both ranges and one
// accumulator per row of both ranges in shared memory).  A tile's entries are sorted by k row and cut into chunks of
// <= 2048.  Per chunk:
//   phase 1  every thread evaluates Eq. 2's summand T of its <= 4 entries (weights and codes stream from HBM fully
//            coalesced, loaded one chunk ahead; N[iq,nu] of the chunk's pairs was copied to shared memory one chunk
//            ahead with cp.async) and stores T to shared memory;
//   phase 2  one thread per k row of the chunk sums that row's contiguous run of T (I[a] -= sum), one thread per
//            k' row sums its T through the chunk-local permutation (I[b] += sum): PAPER.md:94.  Every row has one
//            owner per chunk, chunks are separated by barriers: no atomics, fixed order, bit-reproducible.
// Partial sums of a tile / run go to slots; finish_kernel (ephc_tile_kernels.cuh) adds them per state.
#pragma once
#include <cuda_runtime.h>

#include "ephc_internal.h"
#include "ephc_row_kernels.cuh"  // cp_async helpers

namespace ephc {

constexpr int kStreamThreads = 512;   // two CTAs per SM: the barrier waits of one overlap with the work of the other
constexpr int kStreamEpt = kStreamChunk / kStreamThreads;  // entries per thread and chunk
static_assert(2 * 256 <= kStreamThreads, "two lanes per k row, <= 256 k rows per chunk");

struct StreamParams {
    const double *w;
    const uint32_t *code;
    const uint16_t *perm, *arow_id, *arow_start, *brow_id, *brow_start;
    const uint32_t *iq;
    const StreamChunk *chunks;
    const StreamTile *tiles;
    const int32_t *order;   // tiles by descending work
    int *counter;           // next position in `order` (reset by finish_kernel)
    int32_t ntile;
    const int32_t *row_state;
    const int64_t *slot_off;
    int32_t Ra, Rb, nnu, ncta;
    int64_t ns;
    const double *f, *N;
    double *part;
};

inline size_t stream_smem_bytes(int Ra, int Rb) {
    return ((size_t)2 * Ra + 2 * Rb + 8) * sizeof(double) + (size_t)kStreamChunk * sizeof(double) +
           (size_t)2 * kStreamNSlots * sizeof(double) + (size_t)2 * kStreamChunk * sizeof(uint16_t) + 64;
}

__device__ __forceinline__ void cp_async8(void *smem_dst, const void *gmem_src) {
    const unsigned d = (unsigned)__cvta_generic_to_shared(smem_dst);
    asm volatile("cp.async.ca.shared.global [%0], [%1], 8;\n" ::"r"(d), "l"(gmem_src));
}

__global__ void __launch_bounds__(kStreamThreads, 2) stream_kernel(const StreamParams P) {
    extern __shared__ double smem[];
    double *sIa = smem;                      // f of the k rows
    double *sIb = sIa + P.Ra + 2;            // f of the k' rows
    double *sAa = sIb + P.Rb + 2;            // accumulators of the k rows
    double *sAb = sAa + P.Ra + 2;            // accumulators of the k' rows
    double *sT = sAb + P.Rb + 2;             // per-entry terms of the chunk
    double *sN = sT + kStreamChunk;          // two buffers of N values
    uint16_t *sPerm = reinterpret_cast<uint16_t *>(sN + 2 * kStreamNSlots);  // two buffers
    const int tid = threadIdx.x;
    const int nnu = P.nnu;
    const bool n16 = (nnu % 2 == 0) && ((reinterpret_cast<uintptr_t>(P.N) & 15) == 0);
    __shared__ int sTileNo;

    while (true) {
        __syncthreads();  // previous tile: partial sums written, accumulators and sTileNo free
        if (tid == 0) sTileNo = atomicAdd(P.counter, 1);  // order of execution only: every tile owns its slots
        __syncthreads();
        const int tno = sTileNo;
        if (tno >= P.ntile) break;
        const StreamTile th = P.tiles[P.order[tno]];
        const bool dg = (th.flags & 4) != 0;
        if (th.flags & 1)
            for (int r = tid; r < th.a_rows; r += kStreamThreads) {
                sIa[r] = P.f[P.row_state[th.a_row0 + r]];
                sAa[r] = 0.0;
            }
        if (!dg)
            for (int r = tid; r < th.b_rows; r += kStreamThreads) {
                sIb[r] = P.f[P.row_state[th.b_row0 + r]];
                sAb[r] = 0.0;
            }
        const double *inB = dg ? sIa : sIb;
        double *accB = dg ? sAa : sAb;

        // one chunk ahead: N[iq, nu] of the chunk's pairs and its permutation (cp.async), its entries (registers)
        auto prefetch = [&](const StreamChunk &ch, int buf) {
            double *dN = sN + buf * kStreamNSlots;
            // one thread per pair: its row N[iq, 0..nnu) in 16-byte pieces when rows are 16-byte aligned
            for (int pr = tid; pr < ch.nq; pr += kStreamThreads) {
                const double *src = P.N + (int64_t)__ldg(P.iq + ch.q0 + pr) * nnu;
                double *dst = dN + pr * nnu;
                if (n16) {
                    for (int j = 0; j < nnu; j += 2) cp_async16(dst + j, src + j);
                } else {
                    for (int j = 0; j < nnu; ++j) cp_async8(dst + j, src + j);
                }
            }
            uint16_t *dP = sPerm + buf * kStreamChunk;
            const uint16_t *srcP = P.perm + 4 * (int64_t)ch.pad0;  // 8-byte aligned by construction
            for (int i = tid; i < (ch.ne + 3) / 4; i += kStreamThreads) cp_async8(dP + 4 * i, srcP + 4 * i);
            cp_async_commit();
        };
        double wq[kStreamEpt];
        uint32_t kq[kStreamEpt];
        auto load_entries = [&](const StreamChunk &ch) {
#pragma unroll
            for (int j = 0; j < kStreamEpt; ++j) {
                const int e = j * kStreamThreads + tid;
                wq[j] = 0.0;
                kq[j] = 0;
                if (e < ch.ne) {
                    wq[j] = __ldcs(P.w + ch.e0 + e);
                    kq[j] = __ldcs(P.code + ch.e0 + e);
                }
            }
        };
        StreamChunk ch = P.chunks[th.c0], chn = ch;
        prefetch(ch, 0);
        load_entries(ch);
        for (int ci = 0; ci < th.nc; ++ci) {
            const int buf = ci & 1;
            const double *cN = sN + buf * kStreamNSlots;
            const uint16_t *cP = sPerm + buf * kStreamChunk;
            if (ci + 1 < th.nc) chn = P.chunks[th.c0 + ci + 1];
            // row tasks of this chunk (<= 256 k rows, <= 2048 k' rows): headers to registers before they are needed
            // k rows: two lanes per row from the low warps; k' rows: one thread per row from the high warps downwards
            int ta_row = 0, ta_s0 = 0, ta_s1 = 0, tb_row = 0, tb_s0 = 0, tb_s1 = 0;
            const int arow = tid >> 1, apart = tid & 1;
            if (arow < ch.nar) {
                ta_row = __ldg(P.arow_id + ch.ar0 + arow);
                const int s0 = __ldg(P.arow_start + ch.ar0 + arow), s1 = __ldg(P.arow_start + ch.ar0 + arow + 1);
                const int q = (s1 - s0 + 1) >> 1;
                ta_s0 = min(s0 + apart * q, s1);
                ta_s1 = min(ta_s0 + q, s1);
            }
            const int brow = kStreamThreads - 1 - tid;  // first k' row task of this thread; further ones (rare) below
            if (brow < ch.nbr) {
                tb_row = __ldg(P.brow_id + ch.br0 + brow);
                tb_s0 = __ldg(P.brow_start + ch.br0 + brow);
                tb_s1 = __ldg(P.brow_start + ch.br0 + brow + 1);
            }
            cp_async_wait<0>();
            __syncthreads();  // staged f / N / perm visible; phase 2 of the previous chunk is done with sT
            // ---- phase 1: Eq. 2 summand per entry (reading R-1, rearranged as in tile_kernel) -----------------------
#pragma unroll
            for (int j = 0; j < kStreamEpt; ++j) {
                const int e = j * kStreamThreads + tid;
                const uint32_t k = kq[j];
                const double xa = sIa[ch.a0 + (k & 255u)], xb = inB[(k >> 8) & 2047u], Nn = cN[(k >> 19) & 4095u];
                const double pr = xa * xb;
                const double s = (k >> 31) ? (xa - pr) : (pr - xb);
                if (e < ch.ne) sT[e] = wq[j] * fma(xa - xb, Nn, s);
            }
            if (ci + 1 < th.nc) {
                prefetch(chn, buf ^ 1);
                load_entries(chn);
            }
            __syncthreads();
            // ---- phase 2: one thread per row of the chunk ----------------------------------------------------------------
            if (tid < 2 * ((ch.nar + 15) & ~15)) {  // whole warps: the shuffle below needs all their lanes
                double sum = 0.0;
                for (int i = ta_s0; i < ta_s1; ++i) sum += sT[i];
                sum += __shfl_xor_sync(0xffffffffu, sum, 1);
                if (apart == 0 && arow < ch.nar) sAa[ta_row] -= sum;
            }
            if (dg) __syncthreads();  // the same row can be a k row and a k' row of a diagonal tile
            for (int id = brow; id < ch.nbr; id += kStreamThreads) {
                if (id != brow) {  // more than kStreamThreads k' rows in the chunk: headers were not prefetched
                    tb_row = __ldg(P.brow_id + ch.br0 + id);
                    tb_s0 = __ldg(P.brow_start + ch.br0 + id);
                    tb_s1 = __ldg(P.brow_start + ch.br0 + id + 1);
                }
                double s0 = 0.0, s1 = 0.0;
                int i = tb_s0;
                for (; i + 1 < tb_s1; i += 2) {
                    s0 += sT[cP[i]];
                    s1 += sT[cP[i + 1]];
                }
                if (i < tb_s1) s0 += sT[cP[i]];
                accB[tb_row] += s0 + s1;
            }
            ch = chn;
        }
        __syncthreads();
        if (!dg) {
            double *dst = P.part + P.slot_off[th.b_slot];
            for (int i = tid; i < th.b_rows; i += kStreamThreads) dst[i] = sAb[i];
        }
        if (th.flags & 2) {
            double *dst = P.part + P.slot_off[th.a_slot];
            for (int i = tid; i < th.a_rows; i += kStreamThreads) dst[i] = sAa[i];
        }
    }
}

}  // namespace ephc
