// ephc_tile_kernels.cuh -- sm_100a kernels of the tile path (variant 1): every channel is read ONCE and updates
// both I(n,k) and I(m,k+q); no atomics on global or shared memory.
//
// tile_kernel<MODE, NB>: a CTA walks a contiguous run of (k-block I, k'-block J) tiles.  Per tile it keeps, in
// shared memory, the inputs of both blocks (f, or F for transport) and one accumulator per compact row of both
// blocks.  A warp takes slices of 32 pair records; one LANE = one (k, k') pair:
//   prologue  the pair's f_a[0..nb), f_b[0..nb) (shared memory) and N[iq, 0..nnu) (L2) go to registers
//   loop      the pair's entries stream from HBM, column-major per slice (coalesced, every byte used once);
//             Eq. 2's summand is evaluated from registers and added to per-band register accumulators of both ends
//   epilogue  the lane adds its <= nb partial sums per end into the shared accumulators of k and of k', in the
//             ticket order the host assigned per k point: a plain load-add-store once the k point's counter
//             shows the lane's ticket.  The order is fixed, so results are bit-reproducible.
// At the end of a tile (or of a run of tiles with the same block I) the accumulators go to a partial-sum slot.
// finish_kernel: one thread per state adds the slots of its block in a fixed order and applies the epilogue
// (I, the fused RK4 stage update, Gamma, or tau (v + sum)).
#pragma once
#include <cuda_runtime.h>

#include "ephc_internal.h"

namespace ephc {

enum TileMode : int { kTCollision = 0, kTSetup = 2, kTIter = 3 };
enum FinishMode : int { kFCollision = 0, kFRkStage = 1, kFSetup = 2, kFIter = 3 };

struct TileParams {
    // store
    const double *w;
    const uint16_t *code;
    const uint32_t *prec;  // [3][npiece]
    int64_t npiece;
    const TileSlice *slices;
    const TileHdr *tiles;
    const TileCta *ctas;
    const int32_t *row_state;
    const int64_t *slot_off;
    int32_t Ra, Rb, nnu;
    int32_t cta_group;     // consecutive TileCta shares walked by one CTA (1, or 2 for the 512-thread kernels)
    int32_t ncta;          // number of TileCta shares
    int64_t ns;
    // inputs
    const double *f;  // occupations (collision / RK stage input y_j / f0 of transport_setup)
    const double *N;
    const double *F;  // transport_iter input [3][ns]
    // outputs
    double *part;     // partial-sum slots, [part_rows][C]
    double *Wf, *Wr;  // per entry: W(a<-b), W(b<-a); written by setup, read by iter
};

struct FinishParams {
    const int32_t *state_row, *state_blk, *blk_row0, *blk_ent_ptr;
    const int64_t *blk_ent_off;
    const double *part;
    int64_t ns;
    double *out;  // I, Gamma or Fout
    // rk stage
    int32_t stage;
    double dt;
    double *f0, *ynext, *ksum, *blk_sum;
    double *fc_next;      // compact-row copy of what the next evaluation reads (resident-tile store), may be null
    const double *extra;  // added to k_j per state (drift term of Eq. 1), may be null
    // transport
    const double *v, *tau;
    int *reset;  // tile counter of the stream kernel, set back to 0 for the next evaluation (may be null)
};

template <int NB>
__device__ __forceinline__ double sel_nb(const double (&a)[NB], int j) {
    if (NB == 1) return a[0];
    if (NB == 2) return (j & 1) ? a[1] : a[0];
    const double lo = (j & 1) ? a[1 % NB] : a[0], hi = (j & 1) ? a[3 % NB] : a[2 % NB];
    return (j & 2) ? hi : lo;
}
__device__ __forceinline__ double sel8(const double (&a)[8], int j) {
    const double x0 = (j & 1) ? a[1] : a[0], x1 = (j & 1) ? a[3] : a[2], x2 = (j & 1) ? a[5] : a[4],
                 x3 = (j & 1) ? a[7] : a[6];
    const double y0 = (j & 2) ? x1 : x0, y1 = (j & 2) ? x3 : x2;
    return (j & 4) ? y1 : y0;
}
template <int NB>
__device__ __forceinline__ void put_nb(double (&a)[NB], int j, double x) {
#pragma unroll
    for (int i = 0; i < NB; ++i) a[i] = (j == i) ? x : a[i];
}

__device__ __forceinline__ unsigned ld_cnt(const uint16_t *p) { return *(const volatile uint16_t *)p; }
__device__ __forceinline__ void st_cnt(uint16_t *p, unsigned v) { *(volatile uint16_t *)p = (uint16_t)v; }

constexpr int kTileThreads = 256;      // collision / transport_setup: two CTAs per SM
constexpr int kTileThreadsIter = 512;  // transport_iter: one CTA per SM, accumulators in registers
constexpr int kTileBatch = 4;          // entries per lane whose loads are in flight while the previous batch is evaluated

// Per-thread private rows in shared memory of the collision / setup kernels (row r of thread t at
// [r * kTileThreads + t]: conflict-free):  0..3 f_a[n], 4..7 f_b[m], 8..15 N[nu], 16..19 sums for k, 20..23 sums for k'.
// Dynamic indexing by band / mode costs one LDS here instead of a chain of selects on registers.
constexpr int kRowBytes = kTileThreads * 8;
constexpr int kPrivRows = 24;

inline size_t tile_smem_bytes(int mode, int Ra, int Rb) {
    const int C = (mode == kTIter) ? 3 : 1;
    const size_t rows = (size_t)Ra + (size_t)Rb + 2 * kTileNbMax;
    const size_t cnt = (((size_t)Ra + 7) & ~(size_t)7) + (((size_t)Rb + 7) & ~(size_t)7);
    return 2 * rows * C * sizeof(double) + cnt * sizeof(uint16_t) + 16 +
           (mode == kTIter ? 0 : (size_t)kPrivRows * kRowBytes);
}

__device__ __forceinline__ double &prow(char *tb, unsigned byte_off) { return *reinterpret_cast<double *>(tb + byte_off); }

template <int MODE, int NB>
__global__ void __launch_bounds__((MODE == kTIter) ? kTileThreadsIter : kTileThreads, (MODE == kTIter) ? 1 : 2)
tile_kernel(const TileParams P) {
    constexpr int C = (MODE == kTIter) ? 3 : 1;
    constexpr int U = (MODE == kTIter) ? 2 : kTileBatch;
    constexpr int NT = (MODE == kTIter) ? kTileThreadsIter : kTileThreads;
    extern __shared__ double smem[];
    const int ra_al = P.Ra + kTileNbMax, rb_al = P.Rb + kTileNbMax;
    double *sIa = smem;                  // inputs of the k rows:  f[row] or F[row][3]
    double *sIb = sIa + ra_al * C;       // inputs of the k' rows
    double *sAa = sIb + rb_al * C;       // accumulators of the k rows
    double *sAb = sAa + ra_al * C;       // accumulators of the k' rows
    uint16_t *sCa = reinterpret_cast<uint16_t *>(sAb + rb_al * C);  // ticket counters per k point (first row)
    uint16_t *sCb = sCa + ((P.Ra + 7) & ~7);
    int *sNext = reinterpret_cast<int *>(sCb + ((P.Rb + 7) & ~7));
    double *sPriv = reinterpret_cast<double *>(sNext + 4);

    const int tid = threadIdx.x, lane = tid & 31;
    char *tb = reinterpret_cast<char *>(sPriv + tid);
    const int nnu = P.nnu;
    const int64_t np_all = P.npiece;
    const int share0 = blockIdx.x * P.cta_group, share1 = min(share0 + P.cta_group, P.ncta);
    const int t_begin = P.ctas[share0].t0, t_end = P.ctas[share1 - 1].t1;

    for (int it = t_begin; it < t_end; ++it) {
        const TileHdr th = P.tiles[it];
        const bool dg = (th.flags & 4) != 0;
        // ---- stage the inputs of both row ranges, clear accumulators and ticket counters ------------------------------
        if (th.flags & 1) {
            for (int r = tid; r < th.a_rows + kTileNbMax; r += NT) {
                const int64_t s = (r < th.a_rows) ? P.row_state[th.a_row0 + r] : -1;
#pragma unroll
                for (int c = 0; c < C; ++c) {
                    sIa[r * C + c] = (s < 0) ? 0.0 : (MODE == kTIter ? P.F[(int64_t)c * P.ns + s] : P.f[s]);
                    sAa[r * C + c] = 0.0;
                }
                if (r < th.a_rows) sCa[r] = 0;
            }
        }
        if (!dg) {
            for (int r = tid; r < th.b_rows + kTileNbMax; r += NT) {
                const int64_t s = (r < th.b_rows) ? P.row_state[th.b_row0 + r] : -1;
#pragma unroll
                for (int c = 0; c < C; ++c) {
                    sIb[r * C + c] = (s < 0) ? 0.0 : (MODE == kTIter ? P.F[(int64_t)c * P.ns + s] : P.f[s]);
                    sAb[r * C + c] = 0.0;
                }
                if (r < th.b_rows) sCb[r] = 0;
            }
        }
        __syncthreads();
        const double *inB = dg ? sIa : sIb;
        double *accB = dg ? sAa : sAb;
        uint16_t *cntB = dg ? sCa : sCb;

        // ---- slices: one lane per pair record; warp w takes slices w, w + nwarps, ... in order -----------------------
        // Two slices ahead: header + pair records (stage A).  One slice ahead: N[iq, :] and the first batch of
        // entries (stage B, needs A).  The dependent global loads of a slice are thus in flight while the
        // previous slices are evaluated.
        struct PreA {
            int4 h;
            uint32_t r0, r1, r2;
        };
        struct PreB {
            double Nq[(MODE == kTIter) ? 1 : 8];
            double wq[U], vq[(MODE == kTIter) ? U : 1];
            unsigned kq[U];
            int oq[U];
            int off;
        };
        constexpr int NW = NT / 32;
        const int warp = tid >> 5;
        auto loadA = [&](int g, PreA &A) {
            A.h = __ldg(reinterpret_cast<const int4 *>(P.slices + th.s0 + g));
            const int p0 = th.p0 + 32 * g;
            A.r0 = A.r1 = A.r2 = 0;
            if (lane < th.npc - 32 * g) {
                A.r0 = __ldcs(P.prec + p0 + lane);
                A.r1 = __ldcs(P.prec + np_all + p0 + lane);
                A.r2 = __ldcs(P.prec + 2 * np_all + p0 + lane);
            }
        };
        // columns i0 .. i0+U-1 of a slice (column i holds the lanes with len > i, a prefix of the lanes)
        auto load_batch = [&](int64_t eb, int len, int i0, PreB &B) {
#pragma unroll
            for (int u = 0; u < U; ++u) {
                const bool act = len > i0 + u;
                const int cnt = __popc(__ballot_sync(0xffffffffu, act));
                B.wq[u] = 0.0;
                if (MODE == kTIter) B.vq[u] = 0.0;
                B.kq[u] = 0;
                B.oq[u] = B.off;
                if (act) {
                    B.kq[u] = __ldcs(P.code + eb + B.off);
                    if (MODE == kTIter) {
                        B.wq[u] = __ldcs(P.Wf + eb + B.off);
                        B.vq[u] = __ldcs(P.Wr + eb + B.off);
                    } else {
                        B.wq[u] = __ldcs(P.w + eb + B.off);
                    }
                }
                B.off += cnt;
            }
        };
        auto loadB = [&](const PreA &A, PreB &B) {
            const int64_t eb = (((int64_t)(uint32_t)A.h.x) | ((int64_t)A.h.y << 32)) + lane;
            if (MODE != kTIter) {
                const double *Np = P.N + (int64_t)(A.r1 & 0xffffffu) * nnu;
#pragma unroll
                for (int j = 0; j < 8; ++j) B.Nq[j] = (j < nnu) ? __ldg(Np + j) : 0.0;
            }
            B.off = 0;
            load_batch(eb, (int)(A.r1 >> 24), 0, B);
        };
        PreA A1, A2, A3;
        PreB B1, B2;
        if (warp < th.ns) loadA(warp, A1);
        if (warp + NW < th.ns) loadA(warp + NW, A2);
        if (warp < th.ns) loadB(A1, B1);
        for (int g = warp; g < th.ns; g += NW) {
            if (g + NW < th.ns) loadB(A2, B2);
            if (g + 2 * NW < th.ns) loadA(g + 2 * NW, A3);
            const int64_t e0 = ((int64_t)(uint32_t)A1.h.x) | ((int64_t)A1.h.y << 32);
            const int np = (int)(int16_t)(A1.h.w & 0xffff), maxlen = (int)(int16_t)((uint32_t)A1.h.w >> 16);
            const bool live = lane < np;
            const uint32_t r0 = A1.r0, r1 = A1.r1, r2 = A1.r2;
            const int ra = r0 & 0xffffu, rb = r0 >> 16;
            const int len = (int)(r1 >> 24);
            const int64_t eb = e0 + lane;
            PreB &Bq = B1;

            double acc_a[C][NB], acc_b[C][NB];  // this lane's sums per end and band
            if (MODE == kTIter) {
                // F_a[n][c], F_b[m][c] and the sums in registers (one CTA per SM: 128 registers per thread)
                double Fa[3][NB], Fb[3][NB];
#pragma unroll
                for (int j = 0; j < NB; ++j)
#pragma unroll
                    for (int c = 0; c < 3; ++c) {
                        Fa[c][j] = sIa[(ra + j) * 3 + c];
                        Fb[c][j] = inB[(rb + j) * 3 + c];
                        acc_a[c][j] = 0.0;
                        acc_b[c][j] = 0.0;
                    }
                for (int i = 0; i < maxlen; i += U) {
                    double wc[U], vc[U];
                    unsigned kc[U];
#pragma unroll
                    for (int u = 0; u < U; ++u) {
                        wc[u] = Bq.wq[u];
                        vc[u] = Bq.vq[u];
                        kc[u] = Bq.kq[u];
                    }
                    if (i + U < maxlen) load_batch(eb, len, i + U, Bq);
#pragma unroll
                    for (int u = 0; u < U; ++u) {
                        const int n = kc[u] & 3u, m = (kc[u] >> kTcM) & 3u;
#pragma unroll
                        for (int c = 0; c < 3; ++c) {
                            put_nb<NB>(acc_a[c], n, fma(wc[u], sel_nb<NB>(Fb[c], m), sel_nb<NB>(acc_a[c], n)));
                            put_nb<NB>(acc_b[c], m, fma(vc[u], sel_nb<NB>(Fa[c], n), sel_nb<NB>(acc_b[c], m)));
                        }
                    }
                }
            } else {
                {
#pragma unroll
                    for (int j = 0; j < 4; ++j) {
                        prow(tb, j * kRowBytes) = sIa[ra + j];
                        prow(tb, (4 + j) * kRowBytes) = inB[rb + j];
                    }
#pragma unroll
                    for (int j = 0; j < 8; ++j) {
                        prow(tb, (8 + j) * kRowBytes) = Bq.Nq[j];
                        prow(tb, (16 + j) * kRowBytes) = 0.0;
                    }
                }
                for (int i = 0; i < maxlen; i += U) {
                    double wc[U];
                    unsigned kc[U];
                    int oc[U];
#pragma unroll
                    for (int u = 0; u < U; ++u) {
                        wc[u] = Bq.wq[u];
                        kc[u] = Bq.kq[u];
                        oc[u] = Bq.oq[u];
                    }
                    const int ibase = i;
                    if (i + U < maxlen) load_batch(eb, len, i + U, Bq);
#pragma unroll
                    for (int u = 0; u < U; ++u) {
                        const unsigned k = kc[u];
                        char *pa_ = tb + (k & 3u) * kRowBytes;
                        char *pb_ = tb + (4 + ((k >> kTcM) & 3u)) * kRowBytes;
                        const double Nn = prow(tb, (8 + ((k >> kTcNu) & 7u)) * kRowBytes);
                        const double xa = prow(pa_, 0), xb = prow(pb_, 0);
                        const double sa = prow(pa_, 16 * kRowBytes), sb = prow(pb_, 16 * kRowBytes);
                        const bool em = (k >> kTcKind) & 1u, diag = (k >> kTcDiag) & 1u;
                        if (MODE == kTCollision) {
                            // Eq. 2 summand (reading R-1), rearranged:  F_abs = (fa-fb) N + fa fb - fb,
                            //                                         F_em  = (fa-fb) N + fa - fa fb
                            const double pr = xa * xb;
                            const double s = em ? (xa - pr) : (pr - xb);
                            const double T = (diag ? 0.0 : wc[u]) * fma(xa - xb, Nn, s);
                            prow(pa_, 16 * kRowBytes) = sa + T;
                            prow(pb_, 16 * kRowBytes) = sb + T;
                        } else {
                            // reading R-16: W(a<-b) = w (1 + N - f0_b) [em] or w (N + f0_b) [abs];
                            //               W(b<-a) = w (N + f0_a) [em] or w (1 + N - f0_a) [abs]; diagonal: forward only
                            const double Wf = em ? wc[u] * (1.0 + Nn - xb) : wc[u] * (Nn + xb);
                            const double Wr = diag ? 0.0 : (em ? wc[u] * (Nn + xa) : wc[u] * (1.0 + Nn - xa));
                            if (len > ibase + u) {
                                P.Wf[eb + oc[u]] = Wf;
                                P.Wr[eb + oc[u]] = Wr;
                            }
                            prow(pa_, 16 * kRowBytes) = sa + Wf;
                            prow(pb_, 16 * kRowBytes) = sb + Wr;
                        }
                    }
                }
#pragma unroll
                for (int j = 0; j < NB; ++j) {
                    acc_a[0][j] = prow(tb, (16 + j) * kRowBytes);
                    acc_b[0][j] = prow(tb, (20 + j) * kRowBytes);
                }
            }

            // ---- epilogue: ticket-ordered read-modify-write of the shared accumulators -------------------------------
            // Collision: I[a] -= T, I[b] += T.  Transport: both ends add their own weight sums.
            const unsigned ta = r2 & 0xfffu, tb2 = (r2 >> 16) & 0xfffu;
            const int nia = (int)((r2 >> 12) & 3u) + 1, nib = (int)((r2 >> 28) & 3u) + 1;
            bool pa = live, pb = live;
            while (__any_sync(0xffffffffu, pa || pb)) {
                if (pa && ld_cnt(sCa + ra) == ta) {
                    __threadfence_block();
#pragma unroll
                    for (int j = 0; j < NB; ++j)
                        if (j < nia) {
#pragma unroll
                            for (int c = 0; c < C; ++c) {
                                const double x = acc_a[c][j];
                                sAa[(ra + j) * C + c] += (MODE == kTCollision) ? -x : x;
                            }
                        }
                    __threadfence_block();
                    st_cnt(sCa + ra, ta + 1);
                    pa = false;
                }
                if (pb && !pa && ld_cnt(cntB + rb) == tb2) {
                    __threadfence_block();
#pragma unroll
                    for (int j = 0; j < NB; ++j)
                        if (j < nib) {
#pragma unroll
                            for (int c = 0; c < C; ++c) accB[(rb + j) * C + c] += acc_b[c][j];
                        }
                    __threadfence_block();
                    st_cnt(cntB + rb, tb2 + 1);
                    pb = false;
                }
                __syncwarp();
            }
            A1 = A2;
            B1 = B2;
            A2 = A3;
        }
        __syncthreads();
        // ---- partial sums of this tile / run go to their slots ---------------------------------------------------------
        if (!dg) {
            double *dst = P.part + P.slot_off[th.b_slot] * C;
            for (int i = tid; i < th.b_rows * C; i += NT) dst[i] = sAb[i];
        }
        if (th.flags & 2) {
            double *dst = P.part + P.slot_off[th.a_slot] * C;
            for (int i = tid; i < th.a_rows * C; i += NT) dst[i] = sAa[i];
        }
        __syncthreads();
    }
}

// One thread per state: sum of the block's partial-sum slots in list order, then the epilogue of the call.
template <int FMODE>
__global__ void __launch_bounds__(256) finish_kernel(const FinishParams P) {
    constexpr int C = (FMODE == kFIter) ? 3 : 1;
    const int64_t a = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (a == 0 && P.reset != nullptr) *P.reset = 0;
    double sum[C];
#pragma unroll
    for (int c = 0; c < C; ++c) sum[c] = 0.0;
    double fsum = 0.0;
    if (a < P.ns) {
        const int cr = P.state_row[a];
        double ynew = 0.0;  // rk stage: y_{j+1} (or the new f) of this state
        if (cr >= 0) {
            const int b = P.state_blk[a];
            const int64_t r = cr - P.blk_row0[b];
            // eight slots per step: all offsets, then all values, then the adds in list order (the loads are independent;
            // one at a time this loop is a chain of L2 latencies)
            const int i1 = P.blk_ent_ptr[b + 1];
            int i = P.blk_ent_ptr[b];
            for (; i + 8 <= i1; i += 8) {
                int64_t off[8];
#pragma unroll
                for (int u = 0; u < 8; ++u) off[u] = __ldg(P.blk_ent_off + i + u);
                double val[8][C];
#pragma unroll
                for (int u = 0; u < 8; ++u)
#pragma unroll
                    for (int c = 0; c < C; ++c) val[u][c] = __ldcs(P.part + (off[u] + r) * C + c);
#pragma unroll
                for (int u = 0; u < 8; ++u)
#pragma unroll
                    for (int c = 0; c < C; ++c) sum[c] += val[u][c];
            }
            for (; i < i1; ++i) {
                const double *src = P.part + (P.blk_ent_off[i] + r) * C;
#pragma unroll
                for (int c = 0; c < C; ++c) sum[c] += src[c];
            }
        }
        if (FMODE == kFCollision || FMODE == kFSetup) {
            P.out[a] = sum[0];
        } else if (FMODE == kFIter) {
            const double ta = P.tau[a];
#pragma unroll
            for (int c = 0; c < C; ++c) P.out[(int64_t)c * P.ns + a] = ta * (P.v[(int64_t)c * P.ns + a] + sum[c]);
        } else {  // RK4 stage (reading R-18): k_j = I[y_j]
            const double k = sum[0] + (P.extra ? P.extra[a] : 0.0);
            const double f0 = P.f0[a];
            if (P.stage == 1) {
                P.ksum[a] = k;
                P.ynext[a] = ynew = f0 + 0.5 * P.dt * k;
            } else if (P.stage == 2) {
                P.ksum[a] += 2.0 * k;
                P.ynext[a] = ynew = f0 + 0.5 * P.dt * k;
            } else if (P.stage == 3) {
                P.ksum[a] += 2.0 * k;
                P.ynext[a] = ynew = f0 + P.dt * k;
            } else {
                const double fn = f0 + P.dt / 6.0 * (P.ksum[a] + k);
                P.f0[a] = ynew = fn;
                fsum = fn;
            }
            if (P.fc_next != nullptr && cr >= 0) P.fc_next[cr] = ynew;  // the next stage's gather reads compact rows
        }
    }
    if (FMODE == kFRkStage) {
        if (P.stage == 4 && P.blk_sum != nullptr) {  // uniform over the grid
            __shared__ double sRed[8];
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) fsum += __shfl_xor_sync(0xffffffffu, fsum, o);
            if ((threadIdx.x & 31) == 0) sRed[threadIdx.x >> 5] = fsum;
            __syncthreads();
            if (threadIdx.x == 0) {
                double s = 0.0;
                for (int wi = 0; wi < 8; ++wi) s += sRed[wi];
                P.blk_sum[blockIdx.x] = s;
            }
        }
    }
}

}  // namespace ephc
