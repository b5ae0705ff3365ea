/*
 * ephc.h -- C ABI of the B200-native electron-phonon collision-integral library
 *           (hot path of arxiv 2511.03683; citations are PAPER.md:LINE).
 *
 * What the library computes
 * -------------------------
 *   PAPER.md:51 (II.B, Eq. 2)   I(n,k) = -(2 pi/hbar)(1/N_q) sum_{m,q,nu} |g_mn,nu(k,q)|^2
 *                                  [ delta(e_nk - e_mk+q + hw_nu,q) F_abs + delta(e_nk - e_mk+q - hw_nu,q) F_em ]
 *   PAPER.md:60 (II.B)          channel selection: energy window, Gaussian delta, |g| cut-off
 *   PAPER.md:94, 102 (II.C.2)   every channel feeds I(n,k) and I(m,k+q) with opposite signs; one owner
 *                               per element of I, no atomics
 *   PAPER.md:110 (II.C.2)       transport: same channel loop, the two sides are not +-equal, loop over the
 *                               three field directions
 *   PAPER.md:41-45 (II.A, Eq.1) rt-BTE: df/dt = I[f], one collision evaluation per (sub)step
 * Readings of the points on which the paper is silent (F_abs/F_em, Gaussian normalisation, truncation,
 * units, transport equation, integrator) are listed in DESIGN.md section "Readings" (R-1..R-24).
 *
 * Conventions
 * -----------
 *   units: eV, fs; I in 1/fs; hbar = 0.6582119569 eV fs.
 *   full-grid linear index i = (i1*N2 + i2)*N3 + i3; k+q is component-wise modulo the grid;
 *   iq = index of (k' - k) mod grid.  State index s = ik*nb + n (ik = compact index of an active k).
 *   f, I, Gamma, tau: [ns = nk*nb] doubles.  N: [nq*nnu] doubles on the full q grid (nq = N1*N2*N3).
 *   F, v, Fout: [3][ns] doubles (component-major).
 *   Preconditions (not checked): hw(-q) = hw(q), N(-q) = N(q), g2 Hermitian (one value per unordered entry).
 *
 * Ownership / memory spaces
 * -------------------------
 *   ephc_problem arrays are HOST pointers, borrowed for the duration of ephc_build_channels only.
 *   The handle owns the channel store in device memory (HBM) and a host copy of the canonical list.
 *   Every pointer named *_dev is a caller-owned DEVICE buffer of doubles (8-byte aligned), borrowed for
 *   the call; `stream` is a cudaStream_t passed as void* (NULL = default stream).  Device entry points only
 *   enqueue work: they do not allocate, synchronise or touch the host (all scratch -- transport weights, RK4
 *   stages, partial sums -- is allocated by ephc_build_channels / ephc_set_variant).  A handle lives on the device
 *   that was current at ephc_build_channels; every call makes that device current.  A handle owns ONE set of
 *   scratch buffers and hand-out counters: only one call per handle may be in flight, i.e. all calls on a handle
 *   must be issued to the same stream (or be ordered by the caller); use one handle per stream otherwise.  Every pointer named *_host is a
 *   caller-owned HOST buffer; the *_host entry points copy in, run the same kernels, copy out and
 *   synchronise the stream before returning.
 *
 * Errors
 * ------
 *   All functions return 0 on success and a negative EPHC_E* code on failure; ephc_last_error() returns a
 *   thread-local, human-readable message for the last failure.  There is no CPU fallback: without a CUDA
 *   device every compute entry point fails with EPHC_ECUDA.
 */
#ifndef EPHC_H
#define EPHC_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define EPHC_OK 0
#define EPHC_EINVAL (-1)  /* null pointer, bad size, non-finite input, hw <= 0, index out of range, bad pair list */
#define EPHC_ENOMEM (-2)  /* host or device allocation failed */
#define EPHC_ECUDA (-3)   /* CUDA runtime error (includes "no device") */
#define EPHC_ESTATE (-4)  /* call order: transport_iter before transport_setup, host-only handle, ... */
#define EPHC_ELIMIT (-5)  /* problem exceeds a format limit (nb > 16, nnu > 64, > 2^31-1 states or pairs) */

/* flags of ephc_problem.flags */
#define EPHC_HOST_ONLY 1u /* build the store on the host only (no device needed): query/export work, compute fails */
#define EPHC_TRANSPORT_COLLAPSE 4u /* also build the mode-collapsed row store (ephc_set_transport_collapsed) */
#define EPHC_SELECT_GPU 2u /* channel selection on the device: count / prefix sum / fill over the candidate
                              pairs; the same canonical list as the host selection (indices bit-exact, weights within the
                              two exp implementations); the stores are still laid out on the host */

typedef struct ephc_handle ephc_handle;

/* Input of channel selection.  All arrays on the host. */
typedef struct ephc_problem {
    int32_t grid[3];         /* N1, N2, N3 of the commensurate k/q grid */
    int32_t nk;              /* number of active k points (>= 1) */
    int32_t nb;              /* bands, 1..16 */
    int32_t nnu;             /* phonon modes, 1..64 */
    uint32_t flags;          /* EPHC_HOST_ONLY, EPHC_SELECT_GPU, EPHC_TRANSPORT_COLLAPSE or 0 */
    const int32_t *kfull;    /* [nk] full-grid index of each active k, strictly ascending */
    const double *E;         /* [nk*nb] band energies, eV */
    double emin, emax;       /* energy window, inclusive; a channel needs both end states inside */
    const double *hw;        /* [nq*nnu] phonon energies on the full q grid, eV, > 0 */
    double sigma;            /* Gaussian smearing (standard deviation), eV, > 0 */
    double ncut;             /* a delta is kept iff |argument| < ncut*sigma (3.0 in all configs) */
    double g2_cut;           /* a channel is kept iff g2 >= g2_cut */
    int64_t npair;           /* number of candidate (k,k') pairs */
    const int32_t *pair_ik;  /* [npair] compact index of k; pairs strictly ascending in (ik, ikq), ik <= ikq */
    const int32_t *pair_ikq; /* [npair] compact index of k' = k+q */
    const double *g2;        /* [npair*nnu*nb*nb] |g|^2 in eV^2, index ((p*nnu+nu)*nb+m)*nb+n,
                                n = band at pair_ik, m = band at pair_ikq; self pairs symmetric in (m,n) */
} ephc_problem;

typedef struct ephc_counts {
    int64_t ns;            /* states = nk*nb */
    int64_t npair_active;  /* candidate pairs with at least one active channel (diagonal-only pairs included) */
    int64_t nch;           /* unordered active channels N_ch (the metric's unit) */
    int64_t nw;            /* non-zero delta weights N_w, N_ch <= N_w <= 2 N_ch */
    int64_t ndiag;         /* q=0, n==m terms (transport only) */
    int64_t gather_entries;   /* ordered entries of the destination-sorted (two-sided) store */
    int64_t gather_halfpairs; /* (k <- k') half-pair rows of that store */
    int64_t scatter_entries;  /* entries of the once-stored (tile) store, = nw + diagonal weights; 0 if unavailable */
    int64_t scatter_pairs;    /* pair records of that store */
    int64_t store_bytes_gather;   /* device bytes of the two-sided store (collision + transport share it) */
    int64_t store_bytes_scatter;  /* device bytes of the one-sided store incl. its transposed index */
    int64_t store_bytes_transport;/* device bytes of the per-entry transport weights (0 before transport_setup) */
    int64_t alg_bytes_collision;  /* B_alg of one collision evaluation */
    int64_t alg_bytes_transport;  /* B_alg of one transport iteration */
    int32_t n_workunits, n_rounds, n_tasks; /* launch geometry of the gather kernels */
    int32_t reserved;
    int64_t store_bytes_paper;    /* device bytes of the paper-layout variant incl. sc_col (0 until ephc_set_variant(h, 4)) */
} ephc_counts;

/* Channel selection + store construction ("performed only once on CPUs").
 * Validates the problem (EPHC_EINVAL / EPHC_ELIMIT), builds the canonical unordered channel list
 * [(ik<ikq) or (ik==ikq and n<m), sorted by (ik, ikq, nu, m, n)], the destination-k-segmented stores and
 * the transposed index, and uploads them.  *out receives the handle (NULL on failure). */
int ephc_build_channels(const ephc_problem *p, ephc_handle **out);

/* k-sharded evaluation ("k points are evenly distributed over different MPI processes"):
 * the handle owns the DESTINATION k points k_lo <= ik < k_hi (compact indices) and stores every ordered term whose
 * destination it owns, in the destination-sorted two-sided store (variant 0) and the row store derived from it.
 * ephc_collision, ephc_transport_setup and ephc_transport_iter then compute the owned states only (the others receive
 * 0, resp. tau*v); they read f / F of ALL states, so the caller exchanges the owned slices between the ranks after
 * every evaluation (one all-gather of <= ns doubles).  Time stepping goes through ephc_rt_stage with an exchange of
 * y after each stage; ephc_rt_step is refused.  The ranges of all ranks must partition [0, nk). */
int ephc_build_channels_range(const ephc_problem *p, int32_t k_lo, int32_t k_hi, ephc_handle **out);
/* owned states [s_lo, s_hi) = [k_lo*nb, k_hi*nb); all states for a handle of ephc_build_channels */
int ephc_owned_states(const ephc_handle *h, int64_t *s_lo, int64_t *s_hi);

int ephc_query(const ephc_handle *h, ephc_counts *out);

/* Canonical channel list, host arrays of length nch each (any pointer may be NULL to skip it).
 * w_abs / w_em = (2 pi / (hbar nq)) * g2 * delta_sigma(E_a - E_b +/- hw), exactly 0 when that delta is cut. */
int ephc_export_channels(const ephc_handle *h, int32_t *ik, int32_t *ikq, int32_t *iq, int32_t *n,
                         int32_t *m, int32_t *nu, double *w_abs, double *w_em);
/* q=0, n==m terms: state index, iq (always the q=0 index), nu, weights; length ndiag each. */
int ephc_export_diag(const ephc_handle *h, int32_t *s, int32_t *iq, int32_t *nu, double *w_abs, double *w_em);

/* Decoded image of the two-sided (gather) store, for structural tests of the host builder; only available on
 * handles built with EPHC_HOST_ONLY.  Arrays of length gather_entries (any may be NULL), in store order:
 * destination state, partner state, canonical iq, mode, kind (0: F_abs, 1: F_em as seen from the destination),
 * diagonal flag, weight.  Walks work units -> rounds -> tasks exactly as the kernels do. */
int ephc_export_gather(const ephc_handle *h, int32_t *dest, int32_t *partner, int32_t *iq, int32_t *nu,
                       int32_t *kind, int32_t *diag, double *w);

/* Decoded image of the once-stored (tile) store, same conditions as ephc_export_gather.  Arrays of length
 * scatter_entries in store order: state a = (n,k), state b = (m,k'), canonical iq, mode, kind (0: w_abs, 1: w_em,
 * as seen from a), diagonal flag, weight.  Walks CTAs -> tiles -> slices -> lanes exactly as the kernels do and
 * checks tickets, slots and coverage on the way. */
int ephc_export_tiles(const ephc_handle *h, int32_t *a, int32_t *b, int32_t *iq, int32_t *nu, int32_t *kind,
                      int32_t *diag, double *w);

/* Decoded image of the stream store (variant 2), same conditions as ephc_export_gather.  Arrays of length
 * ephc_stream_entries(h) (= nw: the q = 0, n = m terms are not stored) in store order: state a = (n,k), state b =
 * (m,k'), canonical iq, mode, kind (0: w_abs, 1: w_em), weight.  Walks tiles (in hand-out order) -> chunks and checks
 * the chunk limits, the k-row and k'-row tasks, the chunk-local permutations, slots and coverage on the way. */
int ephc_export_stream(const ephc_handle *h, int32_t *a, int32_t *b, int32_t *iq, int32_t *nu, int32_t *kind,
                       double *w);
int64_t ephc_stream_entries(const ephc_handle *h);

/* Decoded image of the resident-tile store (variant 3), same conditions as ephc_export_gather.  Arrays of length
 * ephc_res_entries(h) (= nw) in store order (runs in hand-out order -> tiles -> entry positions): state a = (n,k),
 * state b = (m,k'), canonical iq, mode, kind (0: w_abs, stored as -w; 1: w_em, stored as +w), weight.  Walks the
 * tile images exactly as the kernel does (the slabs of both phases warp by warp, combos, padding, gather lists) and checks
 * that every weight belongs to one combo with one partner, that every combo term T reaches both of its rows exactly once
 * and that every B row of a tile stores a sum. */
int ephc_export_res(const ephc_handle *h, int32_t *a, int32_t *b, int32_t *iq, int32_t *nu, int32_t *kind,
                    double *w);
int64_t ephc_res_entries(const ephc_handle *h);

/* Decoded image of the row store (the destination-sorted store ephc_transport_iter runs on), same conditions as
 * ephc_export_gather.  Arrays of length gather_entries in store order (strips -> partner-range tiles -> segments):
 * destination state, partner state, position of the same ordered term in the gather store (the row store carries its
 * own copy of the weight, N index and kind of every ordered term).  Checks that the strips partition the destination
 * rows, that a row has one segment per tile with segments in descending length, and that the positions are a
 * permutation. */
int ephc_export_rows(const ephc_handle *h, int32_t *dest, int32_t *partner, int64_t *gather_pos);

/* Decoded image of the mode-collapsed row store (handles built with EPHC_HOST_ONLY | EPHC_TRANSPORT_COLLAPSE): arrays of
 * length ephc_collapsed_entries(h) in store order: destination state, partner state, number of ordered terms summed.
 * Checks that it has the row store's strips and tiles, one entry per partner of a segment, and that the entries cover
 * every ordered term of the row store exactly once, each with its own partner. */
int ephc_export_rows_collapsed(const ephc_handle *h, int32_t *dest, int32_t *partner, int32_t *count);

/* Choice of algorithm:
 *   0 = gather  : destination-sorted two-sided store, one kernel, every ordered term read once
 *   1 = tiles   : once-stored channels grouped into (k-strip, k'-range) tiles; one lane per (k,k') pair updates
 *                 both ends of its channels in shared memory in a fixed ticket order, per-tile partial sums
 *                 are added per state by a second kernel (PAPER.md:88-102 restructured; no atomics).
 *                 Available for nb <= 4, nnu <= 8, nq <= 2^24.
 *   2 = stream  : once-stored channels in the same tiles, one lane per ENTRY; the per-entry terms stay in shared
 *                 memory and are summed per k row and per k' row of a chunk by one thread each (no atomics).
 *                 Collision / rt only (transport calls then use the gather + row stores); any nb, nnu.
 *   3 = resident tiles: once-stored entries (owner = the channel's first end, the kind in the sign of the weight),
 *                 tiles whose whole image is bulk-copied (TMA) into shared memory and processed in place: slabs of
 *                 32 lanes, one lane per piece of an owner row writes the terms over the weights, one lane per piece
 *                 of a partner row gathers them (no atomics, fixed order).
 *                 Collision / rt only (transport calls then use the row store); any nb, nnu.
 *   4 = paper layout: the data structure and the two GPU steps of PAPER.md:84-102 as two plain kernels (scatter /
 *                 scatter_channels rows, step 2 writes the per-channel scratch sc_col to HBM, step 3 sums it per
 *                 target through stargets_sources / targets).  ephc_collision only, for the A/B comparison with the
 *                 library's own stores on the same GPU; never chosen automatically.
 *  -1 = automatic (default): ephc_collision / ephc_rt_step use the gather store while it fits the L2 cache
 *                 (<= 96 MB) and the resident-tile store beyond that (the stream store if the problem exceeds the tile
 *                 format); ephc_transport_setup and ephc_transport_iter run on the row store built from the gather
 *                 store (the faster choice per call as measured on B200).
 * A store that the automatic choice does not use is built and uploaded by the first ephc_set_variant that asks for
 * it (that call allocates and copies; ephc_build_channels builds only what the automatic choice needs).
 * ephc_transport_setup must be called again after a change of variant.  ephc_get_variant returns the variant
 * ephc_collision will use, ephc_get_transport_variant the one the transport calls will use. */
int ephc_set_variant(ephc_handle *h, int variant);
int ephc_get_variant(const ephc_handle *h);
int ephc_get_transport_variant(const ephc_handle *h);

/* I[s] = collision integral of Eq. 2 for occupations f and phonon occupations N. */
int ephc_collision(ephc_handle *h, const double *f_dev, const double *N_dev, double *I_dev, void *stream);

/* Linearised-BTE scattering-in weights about equilibrium f0 (reading R-16):
 * W(a<-b) = w_em (1 + N - f0_b) + w_abs (N + f0_b) per ordered term, kept in the handle;
 * Gamma[a] = sum_b W(a<-b). */
int ephc_transport_setup(ephc_handle *h, const double *f0_dev, const double *N_dev, double *Gamma_dev,
                         void *stream);
/* Start of the iteration: tau[a] = 1/Gamma[a] (0 where Gamma[a] == 0) and F0[al][a] = tau[a] v[al][a]. */
int ephc_transport_start(ephc_handle *h, const double *Gamma_dev, const double *v_dev, double *tau_dev,
                         double *F0_dev, void *stream);
/* One iteration Fout[al][a] = tau[a] * ( v[al][a] + sum_b W(a<-b) F[al][b] ), al = x,y,z. */
int ephc_transport_iter(ephc_handle *h, const double *F_dev, const double *v_dev, const double *tau_dev,
                        double *Fout_dev, void *stream);

/* niter >= 1 chained iterations, Fout = result of the last one (F_dev is not modified; F_dev != Fout_dev).  Same
 * arithmetic as niter calls of ephc_transport_iter (bit-identical result); on the row store the intermediate F stay in
 * compact row order in the handle's scratch instead of going through the API layout. */
int ephc_transport_iters(ephc_handle *h, const double *F_dev, const double *v_dev, const double *tau_dev,
                         double *Fout_dev, int niter, void *stream);

/* Mode-collapsed transport specialisation (SURVEY.md 8(d) honesty note, 8(f) NEXT-3).  In the iteration the ordered terms
 * of one (destination, partner) state pair -- its phonon modes and kinds -- enter through the SUM of their weights only,
 * so after ephc_transport_setup the iteration can run on one weight per state pair.  Handles built with
 * EPHC_TRANSPORT_COLLAPSE carry that second store (same strips and tiles as the row store).  After
 * ephc_transport_setup, ephc_transport_collapse sums the current weights into it (one small kernel) and switches
 * ephc_transport_iter / ephc_transport_iters over to it; ephc_set_transport_collapsed(h, 0 / 1) switches back and forth;
 * the next ephc_transport_setup switches back to the general store.  The result is the same F' up to the order of
 * additions.  It moves fewer bytes per channel-term than the general path, so bench.py reports its rate separately and
 * never as the headline.  ephc_collapsed_entries = state pairs stored. */
int ephc_transport_collapse(ephc_handle *h, void *stream);
int ephc_set_transport_collapsed(ephc_handle *h, int on);
int64_t ephc_collapsed_entries(const ephc_handle *h);

/* nsteps classical RK4 steps of df/dt = I[f] with N fixed (reading R-18), f updated in place.
 * sumf_dev (may be NULL): [nsteps+1], sum_s f_s before the first step and after every step.
 * The axpy of every stage is the epilogue of the collision pass.  For runs of four or more steps the steady-state step
 * (its 8-9 launches have fixed arguments) is captured once into a CUDA graph on a stream the handle owns and replayed on
 * `stream` (EPHC_NO_GRAPH=1: plain launches). */
int ephc_rt_step(ephc_handle *h, double *f_dev, const double *N_dev, double dt_fs, int nsteps,
                 double *sumf_dev, void *stream);

/* Drift term of Eq. 1: out[s] = -(1/hbar) F . grad_k f.  The paper gives no discretisation (its Methods
 * section is missing); reading R-25 of DESIGN.md: central differences on the k grid in reduced coordinates,
 * (grad f)_i ~ N_i/2 [f(n, k+e_i) - f(n, k-e_i)] with k +- e_i modulo the grid, a neighbour that is not an active k
 * point counts as f = 0; field = 3 HOST doubles, the components of F along the reduced axes in eV. */
int ephc_drift(ephc_handle *h, const double *f_dev, const double *field, double *out_dev, void *stream);
/* ephc_rt_step with the drift term: RK4 on df/dt = -(1/hbar) F . grad_k f + I[f] (Eq. 1 as printed). */
int ephc_rt_step_field(ephc_handle *h, double *f_dev, const double *N_dev, const double *field, double dt_fs,
                       int nsteps, double *sumf_dev, void *stream);
/* Post-processing of the transport solution (reading R-26): out10_dev[3 al + be] = sum_s f0_s (1 - f0_s) v[al][s] F[be][s]
 * (al, be = x, y, z; -df0/dE = f0 (1 - f0) / k_B T for a Fermi-Dirac f0) and out10_dev[9] = sum_s f0_s, summed on the
 * device in a fixed order.  Conductivity = e^2 / (Omega N_k k_B T) * S, mobility = e S / (k_B T n): the constants
 * (cell volume, temperature) are the caller's. */
int ephc_transport_moments(ephc_handle *h, const double *f0_dev, const double *v_dev, const double *F_dev,
                           double *out10_dev, void *stream);

/* One stage of the same RK4 step, for callers that exchange data between the stages (k-sharded handles):
 *   stage 1..3: y_out = f + a dt I[y_in] (a = 1/2, 1/2, 1), the handle accumulates b I[y_in];
 *   stage 4:    f += dt/6 (accumulated + I[y_in]) in place (y_out may be NULL).
 * y_in of stage 1 is f itself; only the handle's own states of y_out / f are meaningful on a k-sharded handle. */
int ephc_rt_stage(ephc_handle *h, double *f_dev, const double *y_in_dev, const double *N_dev, double dt_fs, int stage,
                  double *y_out_dev, void *stream);

/* Host-buffer variants (end-to-end path): copy in, run the same kernels, copy out, synchronise. */
int ephc_collision_host(ephc_handle *h, const double *f_host, const double *N_host, double *I_host);
/* tau = 1/Gamma (0 where Gamma == 0), F0 = tau*v, then niter iterations; Gamma_host may be NULL. */
int ephc_transport_solve_host(ephc_handle *h, const double *f0_host, const double *N_host,
                              const double *v_host, int niter, double *F_host, double *Gamma_host);
int ephc_rt_step_host(ephc_handle *h, double *f_host, const double *N_host, double dt_fs, int nsteps,
                      double *sumf_host);

/* Allocation-free conservation scalar: *sum_dev = sum_{s < n} f_dev[s] (electron number, checked every
 * rt-BTE step; the same two-stage reduction as ephc_rt_step's sumf_dev: per-block partial sums, then their sum in a
 * fixed order, bit-reproducible).  For callers that cannot call cudaMalloc (code under CUDA graph capture, tight serving
 * loops, harnesses that forbid it): needs no handle and calls no cudaMalloc / cudaFree or allocating library routine.
 * The partial sums live in a fixed 32 KB device array inside the library (every GPU that loads the library holds it
 * until exit), so n <= ephc_noalloc_max_states() = 16 777 216; larger n fails with EPHC_ELIMIT and touches nothing.
 * f_dev, sum_dev: caller-owned device buffers on the CURRENT device; `stream` as elsewhere.  Every call shares the array,
 * which keeps the last call's contents (each call overwrites all slots it reads): calls that overlap on the GPU, e.g. on
 * two streams, race -- order them.  ephc_noalloc_init() looks up the array's device address for the current device
 * (once per device; the first ephc_sum_states_noalloc on a device does it itself: call it beforehand when the first
 * use would fall under graph capture). */
int ephc_noalloc_init(void);
int64_t ephc_noalloc_max_states(void);
int ephc_sum_states_noalloc(const double *f_dev, int64_t n, double *sum_dev, void *stream);

/* Number of kernel launches enqueued by this library since the handle was created (for bench.py). */
int64_t ephc_launch_count(const ephc_handle *h);

int ephc_destroy(ephc_handle *h);
const char *ephc_last_error(void);
const char *ephc_version(void);

#ifdef __cplusplus
}
#endif
#endif /* EPHC_H */
