// ephc_kernels.cuh -- sm_100a kernels of the gather (destination-sorted, two-sided) path.
//
// One CTA = one work unit = whole destination-k segments, the single owner of their rows of I / Gamma / F'
// ("only one element of I will be updated for each thread" -> no atomics on global memory).
// A work unit is processed in rounds.  Per round:
//   1. stage   the round's pair data in shared memory with coalesced loads: f[k',0..nb) and N[iq,0..nnu)
//              (collision / transport_setup) or F[0..3)[k',0..nb) (transport_iter)        (PAPER.md:96-98 inputs)
//   2. tasks   every warp takes warp tasks (<= 256 consecutive entries that feed ONE destination state):
//              lanes stream (code, weight) with coalesced loads, evaluate the Eq. 2 summand from the staged
//              values, and reduce with warp shuffles (PAPER.md:98 step 2 and 102 step 3 fused: the per-channel
//              scratch sc_col never exists)
//   3. fold    task sums -> per-row accumulators in shared memory, fixed order (bit-reproducible)
// Epilogue (per row, one thread): write I, or the fused RK4 stage update, or Gamma, or tau*(v + sum).
#pragma once
#include <cuda_runtime.h>

#include "ephc_internal.h"

namespace ephc {

enum Mode : int { kCollision = 0, kRkStage = 1, kTransportSetup = 2, kTransportIter = 3 };

struct GatherParams {
    // store
    const uint32_t *code;
    const double *w;
    const int32_t *hp_k, *hp_q;
    const Task *tasks;
    const Round *rounds;
    const WorkUnit *wus;
    int32_t nb, nnu;
    int64_t ns;
    // collision / rk / transport_setup inputs
    const double *f;   // occupations gathered by the kernel (y_j of the RK stage)
    const double *N;
    double *out;       // I (collision), Gamma (setup), Fout (iter)
    // rk stage
    int32_t stage;     // 1..4
    double dt;
    double *f0;        // f at the start of the step (updated in place by stage 4)
    double *ynext;     // y_{j+1} (stages 1..3)
    double *ksum;      // k1 + 2 k2 + 2 k3
    double *wu_sum;    // per work unit: sum of the updated f over its rows (stage 4)
    const double *extra;  // added to k_j per state (drift term of Eq. 1), may be null
    // transport
    double *gW;        // per ordered entry W(a<-b): written by setup, read by iter
    const double *F, *v, *tau;
};

__device__ __forceinline__ double warp_sum(double x) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) x += __shfl_xor_sync(0xffffffffu, x, o);
    return x;
}

// Eq. 2 summand seen from the destination state (reading R-1):
//   F_abs = f_a (1 - f_b) N - f_b (1 - f_a) (N + 1),   F_em = f_a (1 - f_b) (N + 1) - f_b (1 - f_a) N
__device__ __forceinline__ double occ_factor(double fa, double fb, double Nq, bool em) {
    const double out_ = fa * (1.0 - fb), in_ = fb * (1.0 - fa);
    const double N1 = Nq + 1.0;
    return em ? (out_ * N1 - in_ * Nq) : (out_ * Nq - in_ * N1);
}

template <int MODE>
__global__ void __launch_bounds__(kThreads) gather_kernel(const GatherParams P) {
    constexpr int NC = (MODE == kTransportIter) ? 3 : 1;  // accumulators per row
    extern __shared__ double smem[];
    double *sStage = smem;                       // kVMax
    double *sAcc = sStage + kVMax;               // kRowsMax * NC
    double *sPsum = sAcc + kRowsMax * NC;        // kTasksMax * NC
    __shared__ int sNext;
    __shared__ double sRed[kThreads / 32];

    const int tid = threadIdx.x, lane = tid & 31;
    const WorkUnit wu = P.wus[blockIdx.x];
    const int nb = P.nb, nnu = P.nnu;

    for (int i = tid; i < wu.nrows * NC; i += kThreads) sAcc[i] = 0.0;

    for (int r = wu.r0; r < wu.r1; ++r) {
        const Round rd = P.rounds[r];
        // (no barrier needed here: the barrier after staging orders this round's tasks after the previous fold)
        if (tid == 0) sNext = 0;
        // ---- 1. stage ---------------------------------------------------------------------------------------
        if (MODE == kTransportIter) {
            // sStage[(al*nhp + pl)*nb + m] = F[al][k'*nb + m]
            const int per = rd.nhp * nb;
            for (int i = tid; i < per * 3; i += kThreads) {
                const int al = i / per, j = i - al * per;
                const int pl = j / nb, m = j - pl * nb;
                const int kb = __ldg(P.hp_k + rd.hp0 + pl);
                sStage[i] = __ldg(P.F + (int64_t)al * P.ns + (int64_t)kb * nb + m);
            }
        } else {
            // sStage[pl*nb + m] = f[k'*nb + m];  sStage[nhp*nb + pl*nnu + nu] = N[iq*nnu + nu]
            const int nf = rd.nhp * nb, nn = rd.nhp * nnu;
            for (int i = tid; i < nf; i += kThreads) {
                const int pl = i / nb, m = i - pl * nb;
                const int kb = __ldg(P.hp_k + rd.hp0 + pl);
                sStage[i] = __ldg(P.f + (int64_t)kb * nb + m);
            }
            for (int i = tid; i < nn; i += kThreads) {
                const int pl = i / nnu, nu = i - pl * nnu;
                const int q = __ldg(P.hp_q + rd.hp0 + pl);
                sStage[nf + i] = __ldg(P.N + (int64_t)q * nnu + nu);
            }
        }
        __syncthreads();
        // ---- 2. warp tasks --------------------------------------------------------------------------------------
        const double *sF = sStage;
        const double *sN = sStage + rd.nhp * nb;
        const int per = rd.nhp * nb;
        while (true) {
            int t = 0;
            if (lane == 0) t = atomicAdd(&sNext, 1);  // shared-memory work counter: order of execution only
            t = __shfl_sync(0xffffffffu, t, 0);
            if (t >= rd.nt) break;
            const Task tk = P.tasks[rd.t0 + t];
            const uint32_t *code = P.code + tk.e0;
            double a0 = 0.0, a1 = 0.0, a2 = 0.0;
            if (MODE == kCollision || MODE == kRkStage) {
                const double *w = P.w + tk.e0;
                const double fa = __ldg(P.f + tk.row);
#pragma unroll 4
                for (int i = lane; i < tk.len; i += 32) {
                    const uint32_t c = __ldg(code + i);
                    const double wi = __ldg(w + i);
                    const int pl = c & kPairMask, m = (c >> kBandShift) & 15, nu = (c >> kModeShift) & 63;
                    const double fb = sF[pl * nb + m], Nq = sN[pl * nnu + nu];
                    const double t_ = wi * occ_factor(fa, fb, Nq, (c >> kKindBit) & 1u);
                    a0 += (c >> kDiagBit) ? 0.0 : t_;
                }
            } else if (MODE == kTransportSetup) {
                const double *w = P.w + tk.e0;
                double *gW = P.gW + tk.e0;
#pragma unroll 4
                for (int i = lane; i < tk.len; i += 32) {
                    const uint32_t c = __ldg(code + i);
                    const double wi = __ldg(w + i);
                    const int pl = c & kPairMask, m = (c >> kBandShift) & 15, nu = (c >> kModeShift) & 63;
                    const double fb = sF[pl * nb + m], Nq = sN[pl * nnu + nu];
                    // reading R-16: emission term w (1 + N - f0_b), absorption term w (N + f0_b)
                    const double W = ((c >> kKindBit) & 1u) ? wi * (1.0 + Nq - fb) : wi * (Nq + fb);
                    gW[i] = W;
                    a0 += W;
                }
            } else {
                const double *gW = P.gW + tk.e0;
#pragma unroll 4
                for (int i = lane; i < tk.len; i += 32) {
                    const uint32_t c = __ldg(code + i);
                    const double W = __ldg(gW + i);
                    const int j = (c & kPairMask) * nb + ((c >> kBandShift) & 15);
                    a0 += W * sStage[j];
                    a1 += W * sStage[per + j];
                    a2 += W * sStage[2 * per + j];
                }
            }
            a0 = warp_sum(a0);
            if (NC == 3) {
                a1 = warp_sum(a1);
                a2 = warp_sum(a2);
            }
            if (lane == 0) {
                sPsum[t * NC] = a0;
                if (NC == 3) {
                    sPsum[t * NC + 1] = a1;
                    sPsum[t * NC + 2] = a2;
                }
            }
        }
        __syncthreads();
        // ---- 3. fold: the first task of every row adds up that row's tasks of this round, in order ---------------
        for (int t = tid; t < rd.nt; t += kThreads) {
            const int row = P.tasks[rd.t0 + t].row;
            if (t > 0 && P.tasks[rd.t0 + t - 1].row == row) continue;
            double s0 = 0.0, s1 = 0.0, s2 = 0.0;
            for (int u = t; u < rd.nt && P.tasks[rd.t0 + u].row == row; ++u) {
                s0 += sPsum[u * NC];
                if (NC == 3) {
                    s1 += sPsum[u * NC + 1];
                    s2 += sPsum[u * NC + 2];
                }
            }
            const int rl = row - wu.row0;
            sAcc[rl * NC] += s0;
            if (NC == 3) {
                sAcc[rl * NC + 1] += s1;
                sAcc[rl * NC + 2] += s2;
            }
        }
    }
    __syncthreads();
    // ---- epilogue: one thread per destination state ---------------------------------------------------------------
    double fsum = 0.0;
    for (int i = tid; i < wu.nrows; i += kThreads) {
        const int64_t a = wu.row0 + i;
        if (MODE == kCollision) {
            P.out[a] = -sAcc[i];
        } else if (MODE == kTransportSetup) {
            P.out[a] = sAcc[i];
        } else if (MODE == kTransportIter) {
            const double ta = P.tau[a];
#pragma unroll
            for (int al = 0; al < 3; ++al)
                P.out[(int64_t)al * P.ns + a] = ta * (P.v[(int64_t)al * P.ns + a] + sAcc[i * 3 + al]);
        } else {  // RK4 stage (reading R-18): k_j = I[y_j]
            const double k = -sAcc[i] + (P.extra ? P.extra[a] : 0.0);
            const double f0 = P.f0[a];
            if (P.stage == 1) {
                P.ksum[a] = k;
                P.ynext[a] = f0 + 0.5 * P.dt * k;
            } else if (P.stage == 2) {
                P.ksum[a] += 2.0 * k;
                P.ynext[a] = f0 + 0.5 * P.dt * k;
            } else if (P.stage == 3) {
                P.ksum[a] += 2.0 * k;
                P.ynext[a] = f0 + P.dt * k;
            } else {
                const double fn = f0 + P.dt / 6.0 * (P.ksum[a] + k);
                P.f0[a] = fn;
                fsum += fn;
            }
        }
    }
    if (MODE == kRkStage && P.stage == 4 && P.wu_sum != nullptr) {
        // per-work-unit sum of f in a fixed order: warp shuffle tree, then warp 0 over the 8 warp sums
        fsum = warp_sum(fsum);
        if (lane == 0) sRed[tid >> 5] = fsum;
        __syncthreads();
        if (tid == 0) {
            double s = 0.0;
            for (int wi = 0; wi < kThreads / 32; ++wi) s += sRed[wi];
            P.wu_sum[blockIdx.x] = s;
        }
    }
}

// sum of n doubles in a fixed order (one CTA): strided per-thread partial sums, then a shared-memory tree.
__global__ void __launch_bounds__(1024) sum_kernel(const double *x, int64_t n, double *out) {
    __shared__ double s[1024];
    double a = 0.0;
    for (int64_t i = threadIdx.x; i < n; i += 1024) a += x[i];
    s[threadIdx.x] = a;
    __syncthreads();
    for (int o = 512; o > 0; o >>= 1) {
        if ((int)threadIdx.x < o) s[threadIdx.x] += s[threadIdx.x + o];
        __syncthreads();
    }
    if (threadIdx.x == 0) *out = s[0];
}

// Drift term of Eq. 1, reading R-25: out[n,k] = -(1/hbar) sum_i F_i N_i/2 (f[n, k+e_i] - f[n, k-e_i]);
// nbr[d][k] = compact index of k + e_i (d = 2i) / k - e_i (d = 2i+1), or -1 when that grid point is not an active k.
// coef[i] = F_i N_i / (2 hbar).
__global__ void __launch_bounds__(256) drift_kernel(const double *__restrict__ f, const int32_t *__restrict__ nbr, double c0, double c1,
                                                    double c2, double *__restrict__ out, int nk, int nb) {
    const int64_t s = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (s >= (int64_t)nk * nb) return;
    const int k = (int)(s / nb), n = (int)(s - (int64_t)k * nb);
    const double coef[3] = {c0, c1, c2};
    double acc = 0.0;
#pragma unroll
    for (int i = 0; i < 3; ++i) {
        const int kp = nbr[(size_t)(2 * i) * nk + k], km = nbr[(size_t)(2 * i + 1) * nk + k];
        const double fp = kp >= 0 ? f[(int64_t)kp * nb + n] : 0.0, fm = km >= 0 ? f[(int64_t)km * nb + n] : 0.0;
        acc += coef[i] * (fp - fm);
    }
    out[s] = -acc;
}

// Transport post-processing (reading R-26): out[3 al + be] = sum_s f0 (1 - f0) v[al][s] F[be][s], out[9] = sum_s f0;
// one CTA, fixed order (strided per-thread sums, shared-memory tree).
__global__ void __launch_bounds__(1024) moments_kernel(const double *__restrict__ f0, const double *__restrict__ v,
                                                       const double *__restrict__ F, int64_t ns, double *__restrict__ out) {
    __shared__ double s[1024];
    double a[10];
#pragma unroll
    for (int j = 0; j < 10; ++j) a[j] = 0.0;
    for (int64_t i = threadIdx.x; i < ns; i += 1024) {
        const double x = f0[i], wgt = x * (1.0 - x);
#pragma unroll
        for (int al = 0; al < 3; ++al)
#pragma unroll
            for (int be = 0; be < 3; ++be) a[3 * al + be] += wgt * v[(int64_t)al * ns + i] * F[(int64_t)be * ns + i];
        a[9] += x;
    }
    for (int j = 0; j < 10; ++j) {
        s[threadIdx.x] = a[j];
        __syncthreads();
        for (int o = 512; o > 0; o >>= 1) {
            if ((int)threadIdx.x < o) s[threadIdx.x] += s[threadIdx.x + o];
            __syncthreads();
        }
        if (threadIdx.x == 0) out[j] = s[0];
        __syncthreads();
    }
}

// tau = 1/Gamma (0 where Gamma == 0); F0[al] = tau * v[al]
__global__ void tau_f0_kernel(const double *Gamma, const double *v, double *tau, double *F0, int64_t ns) {
    const int64_t a = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (a >= ns) return;
    const double g = Gamma[a];
    const double t = g > 0.0 ? 1.0 / g : 0.0;
    tau[a] = t;
    for (int al = 0; al < 3; ++al) F0[(int64_t)al * ns + a] = t * v[(int64_t)al * ns + a];
}

inline size_t gather_smem_bytes(int mode) {
    const int nc = (mode == kTransportIter) ? 3 : 1;
    return sizeof(double) * (size_t)(kVMax + kRowsMax * nc + kTasksMax * nc);
}

}  // namespace ephc
