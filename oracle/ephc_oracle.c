/*
 * oracle/ephc_oracle.c  --  TEST INFRASTRUCTURE, NOT PRODUCT CODE.
 *
 * Plain, slow, list-based CPU implementation ("oracle B") of the
 * electron-phonon collision integral of arxiv 2511.03683, written from the paper:
 *
 *   PAPER.md:51  (II.B, Eq. 2)   I(n,k) = -(2 pi/hbar)(1/N_q) sum_{m,q,nu} |g|^2
 *                                  [ delta(e_nk - e_mk+q + hw) F_abs + delta(e_nk - e_mk+q - hw) F_em ]
 *   PAPER.md:60  (II.B)          energy window, Gaussian delta, |g| cut-off  -> "active" channels
 *   PAPER.md:74  (II.C.1)        Baseline-CPU loop: (k,q) pairs -> channels -> two updates of I
 *   PAPER.md:94  (II.C.2 step 1) a channel adds equal and opposite amounts to I(n,k) and I(m,k+q)
 *   PAPER.md:110 (II.C.2)        transport: the two sides are no longer +-equal; loop over field directions
 *
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may use
 * this file.  It shares no code, header, table or constant with paper_2511_03683_b200/.
 *
 * Readings of the paper where it is silent:
 *   F_abs = f_a(1-f_b)N - f_b(1-f_a)(N+1),   F_em = f_a(1-f_b)(N+1) - f_b(1-f_a)N          (S-1)
 *   delta_sigma(x) = exp(-x^2/(2 sigma^2)) / (sigma sqrt(2 pi))  if |x| < ncut*sigma, else exactly 0   (S-3, S-4)
 *   a state is in the window iff emin <= E <= emax; a channel needs both end states inside  (S-7)
 *   a channel is active iff g2 >= g2_cut and at least one of the two deltas is non-zero     (S-5, S-6)
 *   prefactor C = 2 pi / (hbar N_q), N_q = number of points of the full grid, hbar in eV fs (S-8, S-9)
 *   N and hw of the emission term are taken at the same q as the absorption term (literal Eq. 2, S-10)
 *   state index s = ik*nb + n; full-grid index i = (i1*N2 + i2)*N3 + i3; k+q component-wise modulo (S-20)
 *   unordered canonical list: (ik<ikq) or (ik==ikq and n<m), order (ik, ikq, nu, m, n)      (S-12)
 *   q=0, n==m terms: zero in the collision integral, kept as forward-only "diagonal" terms for transport
 *   transport (Methods missing; linearised BTE of the paper's ref. 42):
 *        W(a<-b) = C g2 [ delta(x_em)(1 + N - f0_b) + delta(x_abs)(N + f0_b) ]
 *        Gamma_a = sum W(a<-b),  F'[al][a] = tau_a ( v[al][a] + sum W(a<-b) F[al][b] )     (S-16)
 *   rt-BTE: classical RK4 on df/dt = I[f], N fixed, no drift term                           (S-18, S-19)
 *
 * Pins (tests/test_oracle_pins.py): brute force over all (k,q,n,m,nu) (oracle/brute.py, independent
 * numpy code), sum_s I_s = 0, detailed balance, f==c closed form, quadratic structure, Gamma = -dI_a/df_a,
 * dense mat-vec for the transport iteration, two-state logistic closed form for RK4.
 * Parity unpinned: agreement with Perturbo itself on real materials (code and data not available).
 *
 * Build:  gcc -O2 -fPIC -shared -fopenmp -o liboracle.so ephc_oracle.c -lm      (no -ffast-math, no -march)
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define ORC_HBAR 0.6582119569 /* eV fs (S-9) */
#define ORC_PI 3.14159265358979323846

typedef struct {
    int grid[3];
    int nk, nb, nnu;
    double C; /* 2 pi / (hbar N_q) */
    /* canonical unordered channel list */
    int64_t nch;
    int32_t *ik, *ikq, *iq, *n, *m, *nu;
    double *w_abs, *w_em; /* C * g2 * delta_sigma(x_abs / x_em), exactly 0 when that delta fails */
    /* diagonal (q = 0, n == m) terms, transport only */
    int64_t ndiag;
    int32_t *d_s, *d_iq, *d_nu;
    double *d_wabs, *d_wem;
} orc_list;

static double orc_delta(double x, double sigma, double ncut) {
    if (!(fabs(x) < ncut * sigma)) return 0.0;
    return exp(-(x * x) / (2.0 * sigma * sigma)) / (sigma * sqrt(2.0 * ORC_PI));
}

/* index on the full grid of (k' - k) mod grid, from the two full-grid indices */
static int32_t orc_qindex(const int grid[3], int32_t kf, int32_t kqf) {
    int n2 = grid[1], n3 = grid[2];
    int a1 = kf / (n2 * n3), a2 = (kf / n3) % n2, a3 = kf % n3;
    int b1 = kqf / (n2 * n3), b2 = (kqf / n3) % n2, b3 = kqf % n3;
    int q1 = ((b1 - a1) % grid[0] + grid[0]) % grid[0];
    int q2 = ((b2 - a2) % grid[1] + grid[1]) % grid[1];
    int q3 = ((b3 - a3) % grid[2] + grid[2]) % grid[2];
    return (int32_t)((q1 * n2 + q2) * n3 + q3);
}

static int orc_inwin(double e, double emin, double emax) { return e >= emin && e <= emax; }

void orc_free(orc_list *L) {
    if (!L) return;
    free(L->ik); free(L->ikq); free(L->iq); free(L->n); free(L->m); free(L->nu);
    free(L->w_abs); free(L->w_em);
    free(L->d_s); free(L->d_iq); free(L->d_nu); free(L->d_wabs); free(L->d_wem);
    free(L);
}

/*
 * Channel selection and the canonical list.  Two passes over the candidate pairs:
 * pass 0 counts, pass 1 fills.  g2 index: ((p*nnu + nu)*nb + m)*nb + n, n at pair_ik, m at pair_ikq.
 */
orc_list *orc_build(const int *grid, int nk, int nb, int nnu, const int32_t *kfull, const double *E,
                    double emin, double emax, const double *hw, double sigma, double ncut, double g2_cut,
                    int64_t npair, const int32_t *pair_ik, const int32_t *pair_ikq, const double *g2) {
    orc_list *L = (orc_list *)calloc(1, sizeof(orc_list));
    if (!L) return NULL;
    L->grid[0] = grid[0]; L->grid[1] = grid[1]; L->grid[2] = grid[2];
    L->nk = nk; L->nb = nb; L->nnu = nnu;
    double nq = (double)grid[0] * (double)grid[1] * (double)grid[2];
    L->C = 2.0 * ORC_PI / (ORC_HBAR * nq);
    for (int pass = 0; pass < 2; ++pass) {
        int64_t c = 0, d = 0;
        for (int64_t p = 0; p < npair; ++p) {
            int32_t ik = pair_ik[p], ikq = pair_ikq[p];
            int32_t iq = orc_qindex(grid, kfull[ik], kfull[ikq]);
            for (int nu = 0; nu < nnu; ++nu) {
                double w = hw[(int64_t)iq * nnu + nu];
                for (int m = 0; m < nb; ++m) {
                    double eb = E[(int64_t)ikq * nb + m];
                    if (!orc_inwin(eb, emin, emax)) continue;
                    for (int n = 0; n < nb; ++n) {
                        double ea = E[(int64_t)ik * nb + n];
                        if (!orc_inwin(ea, emin, emax)) continue;
                        int self = (ik == ikq);
                        if (self && n > m) continue; /* mirror of the (n<m) entry */
                        double gg = g2[(((int64_t)p * nnu + nu) * nb + m) * nb + n];
                        if (!(gg >= g2_cut)) continue;
                        double dE = ea - eb;
                        double xa = dE + w, xe = dE - w;
                        double da = orc_delta(xa, sigma, ncut), de = orc_delta(xe, sigma, ncut);
                        if (da == 0.0 && de == 0.0) continue;
                        if (self && n == m) {
                            if (pass) {
                                L->d_s[d] = ik * nb + n; L->d_iq[d] = iq; L->d_nu[d] = nu;
                                L->d_wabs[d] = L->C * gg * da; L->d_wem[d] = L->C * gg * de;
                            }
                            ++d;
                        } else {
                            if (pass) {
                                L->ik[c] = ik; L->ikq[c] = ikq; L->iq[c] = iq;
                                L->n[c] = n; L->m[c] = m; L->nu[c] = nu;
                                L->w_abs[c] = L->C * gg * da; L->w_em[c] = L->C * gg * de;
                            }
                            ++c;
                        }
                    }
                }
            }
        }
        if (!pass) {
            L->nch = c; L->ndiag = d;
            size_t cc = (size_t)(c > 0 ? c : 1), dd = (size_t)(d > 0 ? d : 1);
            L->ik = malloc(cc * 4); L->ikq = malloc(cc * 4); L->iq = malloc(cc * 4);
            L->n = malloc(cc * 4); L->m = malloc(cc * 4); L->nu = malloc(cc * 4);
            L->w_abs = malloc(cc * 8); L->w_em = malloc(cc * 8);
            L->d_s = malloc(dd * 4); L->d_iq = malloc(dd * 4); L->d_nu = malloc(dd * 4);
            L->d_wabs = malloc(dd * 8); L->d_wem = malloc(dd * 8);
            if (!L->ik || !L->ikq || !L->iq || !L->n || !L->m || !L->nu || !L->w_abs || !L->w_em ||
                !L->d_s || !L->d_iq || !L->d_nu || !L->d_wabs || !L->d_wem) { orc_free(L); return NULL; }
        }
    }
    return L;
}

int64_t orc_nch(const orc_list *L) { return L->nch; }
int64_t orc_ndiag(const orc_list *L) { return L->ndiag; }
/* number of non-zero delta weights, N_w (N_ch <= N_w <= 2 N_ch) */
int64_t orc_nw(const orc_list *L) {
    int64_t w = 0;
    for (int64_t c = 0; c < L->nch; ++c) w += (L->w_abs[c] != 0.0) + (L->w_em[c] != 0.0);
    return w;
}

void orc_export(const orc_list *L, int32_t *ik, int32_t *ikq, int32_t *iq, int32_t *n, int32_t *m,
                int32_t *nu, double *w_abs, double *w_em) {
    size_t c = (size_t)L->nch;
    memcpy(ik, L->ik, c * 4); memcpy(ikq, L->ikq, c * 4); memcpy(iq, L->iq, c * 4);
    memcpy(n, L->n, c * 4); memcpy(m, L->m, c * 4); memcpy(nu, L->nu, c * 4);
    memcpy(w_abs, L->w_abs, c * 8); memcpy(w_em, L->w_em, c * 8);
}
void orc_export_diag(const orc_list *L, int32_t *s, int32_t *iq, int32_t *nu, double *w_abs, double *w_em) {
    size_t d = (size_t)L->ndiag;
    memcpy(s, L->d_s, d * 4); memcpy(iq, L->d_iq, d * 4); memcpy(nu, L->d_nu, d * 4);
    memcpy(w_abs, L->d_wabs, d * 8); memcpy(w_em, L->d_wem, d * 8);
}

/* occupation factors of Eq. 2 (reading S-1) */
static double orc_Fabs(double fa, double fb, double N) { return fa * (1.0 - fb) * N - fb * (1.0 - fa) * (N + 1.0); }
static double orc_Fem(double fa, double fb, double N) { return fa * (1.0 - fb) * (N + 1.0) - fb * (1.0 - fa) * N; }

/* contribution of channel c (step 2): T = w_abs F_abs + w_em F_em */
static double orc_term(const orc_list *L, int64_t c, const double *f, const double *N) {
    double fa = f[(int64_t)L->ik[c] * L->nb + L->n[c]];
    double fb = f[(int64_t)L->ikq[c] * L->nb + L->m[c]];
    double Nq = N[(int64_t)L->iq[c] * L->nnu + L->nu[c]];
    return L->w_abs[c] * orc_Fabs(fa, fb, Nq) + L->w_em[c] * orc_Fem(fa, fb, Nq);
}

/* Collision integral, serial: I[a] -= T, I[b] += T over the list. */
void orc_collision(const orc_list *L, const double *f, const double *N, double *I) {
    int64_t ns = (int64_t)L->nk * L->nb;
    for (int64_t s = 0; s < ns; ++s) I[s] = 0.0;
    for (int64_t c = 0; c < L->nch; ++c) {
        double T = orc_term(L, c, f, N);
        I[(int64_t)L->ik[c] * L->nb + L->n[c]] -= T;
        I[(int64_t)L->ikq[c] * L->nb + L->m[c]] += T;
    }
}

/* Same sum in the paper's Baseline-CPU shape: OpenMP over the list, atomic updates.
 * Used only to time the oracle on all host cores; summation order is not fixed. */
void orc_collision_omp(const orc_list *L, const double *f, const double *N, double *I) {
    int64_t ns = (int64_t)L->nk * L->nb;
    for (int64_t s = 0; s < ns; ++s) I[s] = 0.0;
#pragma omp parallel for schedule(static)
    for (int64_t c = 0; c < L->nch; ++c) {
        double T = orc_term(L, c, f, N);
        double *pa = &I[(int64_t)L->ik[c] * L->nb + L->n[c]];
        double *pb = &I[(int64_t)L->ikq[c] * L->nb + L->m[c]];
#pragma omp atomic
        *pa -= T;
#pragma omp atomic
        *pb += T;
    }
}
int orc_threads(void) {
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

/* ---------------------------------------------------------------------------------------------
 * Transport (reading S-16; the two sides of a channel are not +-equal).
 * For the stored orientation a=(n,ik), b=(m,ikq):
 *   W(a<-b) = w_em (1 + N - f0_b) + w_abs (N + f0_b)
 *   W(b<-a) = w_abs (1 + N - f0_a) + w_em (N + f0_a)     (mirror term: x_abs' = -x_em, x_em' = -x_abs)
 * ------------------------------------------------------------------------------------------- */
static void orc_W(const orc_list *L, int64_t c, const double *f0, const double *N, double *Wab, double *Wba) {
    double fa = f0[(int64_t)L->ik[c] * L->nb + L->n[c]];
    double fb = f0[(int64_t)L->ikq[c] * L->nb + L->m[c]];
    double Nq = N[(int64_t)L->iq[c] * L->nnu + L->nu[c]];
    *Wab = L->w_em[c] * (1.0 + Nq - fb) + L->w_abs[c] * (Nq + fb);
    *Wba = L->w_abs[c] * (1.0 + Nq - fa) + L->w_em[c] * (Nq + fa);
}
static double orc_Wdiag(const orc_list *L, int64_t d, const double *f0, const double *N) {
    double fa = f0[L->d_s[d]];
    double Nq = N[(int64_t)L->d_iq[d] * L->nnu + L->d_nu[d]];
    return L->d_wem[d] * (1.0 + Nq - fa) + L->d_wabs[d] * (Nq + fa);
}

/* Gamma_a = sum over ordered terms of W(a<-b) */
void orc_transport_setup(const orc_list *L, const double *f0, const double *N, double *Gamma) {
    int64_t ns = (int64_t)L->nk * L->nb;
    for (int64_t s = 0; s < ns; ++s) Gamma[s] = 0.0;
    for (int64_t c = 0; c < L->nch; ++c) {
        double Wab, Wba;
        orc_W(L, c, f0, N, &Wab, &Wba);
        Gamma[(int64_t)L->ik[c] * L->nb + L->n[c]] += Wab;
        Gamma[(int64_t)L->ikq[c] * L->nb + L->m[c]] += Wba;
    }
    for (int64_t d = 0; d < L->ndiag; ++d) Gamma[L->d_s[d]] += orc_Wdiag(L, d, f0, N);
}

/* F'[al][a] = tau_a ( v[al][a] + sum_b W(a<-b) F[al][b] ), al = x,y,z; arrays are [3][ns] */
void orc_transport_iter(const orc_list *L, const double *f0, const double *N, const double *F,
                        const double *v, const double *tau, double *Fout) {
    int64_t ns = (int64_t)L->nk * L->nb;
    for (int64_t i = 0; i < 3 * ns; ++i) Fout[i] = 0.0;
    for (int64_t c = 0; c < L->nch; ++c) {
        double Wab, Wba;
        orc_W(L, c, f0, N, &Wab, &Wba);
        int64_t a = (int64_t)L->ik[c] * L->nb + L->n[c];
        int64_t b = (int64_t)L->ikq[c] * L->nb + L->m[c];
        for (int al = 0; al < 3; ++al) {
            Fout[al * ns + a] += Wab * F[al * ns + b];
            Fout[al * ns + b] += Wba * F[al * ns + a];
        }
    }
    for (int64_t d = 0; d < L->ndiag; ++d) {
        double Wd = orc_Wdiag(L, d, f0, N);
        int64_t a = L->d_s[d];
        for (int al = 0; al < 3; ++al) Fout[al * ns + a] += Wd * F[al * ns + a];
    }
    for (int al = 0; al < 3; ++al)
        for (int64_t s = 0; s < ns; ++s) Fout[al * ns + s] = tau[s] * (v[al * ns + s] + Fout[al * ns + s]);
}

/* ---------------------------------------------------------------------------------------------
 * rt-BTE (reading S-18): classical RK4 on df/dt = I[f]; sumf[0] = sum f before the first step,
 * sumf[i] = sum f after step i (plain left-to-right sum).  f is updated in place.
 * ------------------------------------------------------------------------------------------- */
static double orc_sum(const double *x, int64_t n) {
    double s = 0.0;
    for (int64_t i = 0; i < n; ++i) s += x[i];
    return s;
}
int orc_rt_step(const orc_list *L, double *f, const double *N, double dt, int nsteps, double *sumf) {
    int64_t ns = (int64_t)L->nk * L->nb;
    double *k1 = malloc(8 * (size_t)ns), *k2 = malloc(8 * (size_t)ns), *k3 = malloc(8 * (size_t)ns);
    double *k4 = malloc(8 * (size_t)ns), *y = malloc(8 * (size_t)ns);
    if (!k1 || !k2 || !k3 || !k4 || !y) { free(k1); free(k2); free(k3); free(k4); free(y); return -1; }
    if (sumf) sumf[0] = orc_sum(f, ns);
    for (int it = 0; it < nsteps; ++it) {
        orc_collision(L, f, N, k1);
        for (int64_t s = 0; s < ns; ++s) y[s] = f[s] + 0.5 * dt * k1[s];
        orc_collision(L, y, N, k2);
        for (int64_t s = 0; s < ns; ++s) y[s] = f[s] + 0.5 * dt * k2[s];
        orc_collision(L, y, N, k3);
        for (int64_t s = 0; s < ns; ++s) y[s] = f[s] + dt * k3[s];
        orc_collision(L, y, N, k4);
        for (int64_t s = 0; s < ns; ++s) f[s] += dt / 6.0 * (k1[s] + 2.0 * k2[s] + 2.0 * k3[s] + k4[s]);
        if (sumf) sumf[it + 1] = orc_sum(f, ns);
    }
    free(k1); free(k2); free(k3); free(k4); free(y);
    return 0;
}

/* ---------------------------------------------------------------------------------------------
 * Drift term of Eq. 1: D[f](n,k) = -(1/hbar) F . grad_k f.   The paper gives no discretisation (its
 * Methods section is missing); reading R-25 of DESIGN.md: k in reduced coordinates x_i = c_i / N_i of the grid,
 *     (grad f)_i ~ N_i/2 * [ f(n, k+e_i) - f(n, k-e_i) ]      (central difference, k +- e_i modulo the grid),
 * a neighbour that is not an active k point counts as f = 0, F given by its three components along the reduced axes
 * in eV, so that D is in 1/fs.  Every state slot of an active k point gets a value.
 * ------------------------------------------------------------------------------------------- */
int orc_drift(const int *grid, int nk, int nb, const int32_t *kfull, const double *f, const double *Ffield, double *out) {
    int64_t nq = (int64_t)grid[0] * grid[1] * grid[2];
    int32_t *compact = malloc(sizeof(int32_t) * (size_t)nq);
    if (!compact) return -1;
    for (int64_t i = 0; i < nq; ++i) compact[i] = -1;
    for (int k = 0; k < nk; ++k) compact[kfull[k]] = k;
    for (int k = 0; k < nk; ++k) {
        int c[3] = {kfull[k] / (grid[1] * grid[2]), (kfull[k] / grid[2]) % grid[1], kfull[k] % grid[2]};
        for (int n = 0; n < nb; ++n) {
            double acc = 0.0;
            for (int i = 0; i < 3; ++i) {
                int cp[3] = {c[0], c[1], c[2]}, cm[3] = {c[0], c[1], c[2]};
                cp[i] = (c[i] + 1) % grid[i];
                cm[i] = (c[i] - 1 + grid[i]) % grid[i];
                int32_t kp = compact[((int64_t)cp[0] * grid[1] + cp[1]) * grid[2] + cp[2]];
                int32_t km = compact[((int64_t)cm[0] * grid[1] + cm[1]) * grid[2] + cm[2]];
                double fp = kp >= 0 ? f[(int64_t)kp * nb + n] : 0.0;
                double fm = km >= 0 ? f[(int64_t)km * nb + n] : 0.0;
                acc += Ffield[i] * (0.5 * grid[i]) * (fp - fm);
            }
            out[(int64_t)k * nb + n] = -acc / ORC_HBAR;
        }
    }
    free(compact);
    return 0;
}

/* rt-BTE with the drift term: classical RK4 on df/dt = D[f] + I[f] (Eq. 1 as printed), N fixed. */
int orc_rt_step_field(const orc_list *L, const int32_t *kfull, double *f, const double *N, const double *Ffield,
                      double dt, int nsteps, double *sumf) {
    int64_t ns = (int64_t)L->nk * L->nb;
    double *k[4], *y = malloc(8 * (size_t)ns), *d = malloc(8 * (size_t)ns);
    for (int j = 0; j < 4; ++j) k[j] = malloc(8 * (size_t)ns);
    if (!k[0] || !k[1] || !k[2] || !k[3] || !y || !d) return -1;
    const double a[3] = {0.5, 0.5, 1.0};
    if (sumf) sumf[0] = orc_sum(f, ns);
    for (int it = 0; it < nsteps; ++it) {
        for (int j = 0; j < 4; ++j) {
            const double *src = f;
            if (j > 0) {
                for (int64_t s = 0; s < ns; ++s) y[s] = f[s] + a[j - 1] * dt * k[j - 1][s];
                src = y;
            }
            orc_collision(L, src, N, k[j]);
            if (orc_drift(L->grid, L->nk, L->nb, kfull, src, Ffield, d)) return -1;
            for (int64_t s = 0; s < ns; ++s) k[j][s] += d[s];
        }
        for (int64_t s = 0; s < ns; ++s) f[s] += dt / 6.0 * (k[0][s] + 2.0 * k[1][s] + 2.0 * k[2][s] + k[3][s]);
        if (sumf) sumf[it + 1] = orc_sum(f, ns);
    }
    for (int j = 0; j < 4; ++j) free(k[j]);
    free(y); free(d);
    return 0;
}

/* ---------------------------------------------------------------------------------------------
 * Sampled evaluation straight from the problem definition (no list): I[s] for a few states, as the
 * ordered sum of Eq. 2 over every candidate pair that touches the state's k.  Used by the full-size
 * parity tests, where building the list for 1e8 channels is not wanted.
 * For a state on the ik side the term is (a=(n,ik), b=(m,ikq)) with g2[p][nu][m][n];
 * for a state on the ikq side the ordered term is the mirror: a=(m,ikq), b=(n,ik), q -> -q, same g2
 * (Hermiticity, S-11), hw and N taken at -q (S-10 precondition: they are even in q).
 * ------------------------------------------------------------------------------------------- */
void orc_collision_sampled(const int *grid, int nk, int nb, int nnu, const int32_t *kfull, const double *E,
                           double emin, double emax, const double *hw, double sigma, double ncut, double g2_cut,
                           int64_t npair, const int32_t *pair_ik, const int32_t *pair_ikq, const double *g2,
                           const double *f, const double *N, int nsample, const int32_t *states, double *out) {
    double nq = (double)grid[0] * (double)grid[1] * (double)grid[2];
    double C = 2.0 * ORC_PI / (ORC_HBAR * nq);
    (void)nk;
    for (int j = 0; j < nsample; ++j) {
        int32_t s = states[j];
        int32_t k = s / nb, na = s % nb;
        double ea = E[s], fa = f[s], acc = 0.0;
        if (!orc_inwin(ea, emin, emax)) { out[j] = 0.0; continue; }
        for (int64_t p = 0; p < npair; ++p) {
            int32_t ik = pair_ik[p], ikq = pair_ikq[p];
            for (int side = 0; side < 2; ++side) {
                int32_t kb;
                if (side == 0) { if (ik != k) continue; kb = ikq; }
                else { if (ikq != k || ik == ikq) continue; kb = ik; } /* self pair: side 0 covers all (n,m) */
                int32_t iq = orc_qindex(grid, kfull[k], kfull[kb]);
                for (int nu = 0; nu < nnu; ++nu) {
                    double w = hw[(int64_t)iq * nnu + nu], Nq = N[(int64_t)iq * nnu + nu];
                    for (int mb = 0; mb < nb; ++mb) {
                        double eb = E[(int64_t)kb * nb + mb];
                        if (!orc_inwin(eb, emin, emax)) continue;
                        double gg = (side == 0) ? g2[(((int64_t)p * nnu + nu) * nb + mb) * nb + na]
                                                : g2[(((int64_t)p * nnu + nu) * nb + na) * nb + mb];
                        if (!(gg >= g2_cut)) continue;
                        double dE = ea - eb, fb = f[(int64_t)kb * nb + mb];
                        double da = orc_delta(dE + w, sigma, ncut), de = orc_delta(dE - w, sigma, ncut);
                        acc += gg * (da * orc_Fabs(fa, fb, Nq) + de * orc_Fem(fa, fb, Nq));
                    }
                }
            }
        }
        out[j] = -C * acc;
    }
}
