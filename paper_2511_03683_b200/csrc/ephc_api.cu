// ephc_api.cu -- the C ABI declared in include/ephc.h: handle, uploads, kernel launches, error reporting.
// Product code: shares nothing with oracle/.  No CPU fallback: compute entry points need a CUDA device.
#include <cuda_runtime.h>

#include <algorithm>
#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <new>
#include <string>
#include <vector>

#include "ephc_internal.h"
#include "ephc_kernels.cuh"
#include "ephc_tile_kernels.cuh"
#include "ephc_row_kernels.cuh"
#include "ephc_stream_kernels.cuh"
#include "ephc_res_kernels.cuh"
#include "ephc_select_kernels.cuh"
#include "ephc_paper_kernels.cuh"

using namespace ephc;

static thread_local std::string g_err;

static int fail(int code, const std::string &msg) {
    g_err = msg;
    return code;
}
#define CUDA_TRY(expr)                                                                            \
    do {                                                                                          \
        cudaError_t e_ = (expr);                                                                  \
        if (e_ != cudaSuccess)                                                                    \
            return fail(EPHC_ECUDA, std::string(#expr) + ": " + cudaGetErrorString(e_));          \
    } while (0)

struct ephc_handle {
    Dims d{};
    bool host_only = false;
    int device = 0, n_sm = 148;          // device the store lives on (current at ephc_build_channels)
    std::vector<double> E;               // copy of the band energies and window: the optional stores are built from them
    double emin = 0.0, emax = 0.0;
    bool tile_built = false, stream_built = false, res_built = false;
    std::vector<int32_t> kfull;          // full-grid index of every active k (neighbour table of the drift term)
    int32_t *d_nbr = nullptr;            // [6][nk] compact index of k +- e_i, -1 where that point is not active
    double *d_drift = nullptr;           // drift term of the current RK stage
    bool ranged = false;                 // built by ephc_build_channels_range: owns the destination k in [d.k_lo, d.k_hi)
    RowHost rowhost;                     // kept only for EPHC_HOST_ONLY handles (ephc_export_rows)
    RowCollapsed chost;                  // the same for the mode-collapsed row store (ephc_export_rows_collapsed)
    int variant = -1;  // -1: automatic (collision / rt_step: gather store while it fits the L2, resident tiles beyond; transport: rows)
    Canonical can;
    GatherHost ghost;  // kept only for EPHC_HOST_ONLY handles (ephc_export_gather)
    std::vector<int32_t> pair_ik, pair_ikq;  // copy of the candidate pair list (export)
    // gather store: counts
    int64_t g_entries = 0, g_halfpairs = 0;
    int32_t n_wu = 0, n_rounds = 0, n_tasks = 0;
    // device image
    uint32_t *d_code = nullptr;
    double *d_w = nullptr;
    int32_t *d_hp_k = nullptr, *d_hp_q = nullptr;
    Task *d_tasks = nullptr;
    Round *d_rounds = nullptr;
    WorkUnit *d_wus = nullptr;
    double *d_gW = nullptr;      // transport weights, allocated by transport_setup
    bool transport_ready = false;
    // scratch for rt_step / host variants (allocated lazily, freed in destroy)
    double *d_y[2] = {nullptr, nullptr}, *d_ksum = nullptr, *d_wusum = nullptr;
    // CUDA graph of one steady-state RK4 step of ephc_rt_step (captured on cap_stream, replayed on the caller's stream)
    cudaStream_t cap_stream = nullptr;
    cudaGraphExec_t rk_graph = nullptr;
    double *d_sumstep = nullptr;  // sum_s f_s of the step the graph has just run
    struct RkKey {
        const void *f, *N;
        double dt, field[3];
        int has_field, want_sum, variant;
    } rk_key = {nullptr, nullptr, 0.0, {0.0, 0.0, 0.0}, 0, 0, -99};
    int rk_graph_launches = 0;
    double *d_hf = nullptr, *d_hN = nullptr, *d_hI = nullptr;  // host-variant staging: f, N, I
    double *d_tr[5] = {nullptr, nullptr, nullptr, nullptr, nullptr};  // Gamma, tau, v, F, F'
    double *d_sumf = nullptr;
    int64_t sumf_cap = 0;
    int64_t launches = 0;
    int64_t bytes_gather = 0, bytes_transport = 0;
    bool attrs_set = false;
    // tile store (variant 1)
    TileHost thost;  // arrays kept only for EPHC_HOST_ONLY handles (ephc_export_tiles); scalars always
    bool tile_ok = false;
    int64_t t_entries = 0, t_pieces = 0, t_part_rows = 0, bytes_tile = 0;
    int32_t t_ncta = 0, t_Ra = 0, t_Rb = 0, t_nblk = 0, t_nslot = 0, t_ntile = 0;
    double *dt_w = nullptr, *dt_part = nullptr, *dt_Wf = nullptr, *dt_Wr = nullptr;
    uint16_t *dt_code = nullptr;
    uint32_t *dt_prec = nullptr;
    TileSlice *dt_slices = nullptr;
    TileHdr *dt_tiles = nullptr;
    TileCta *dt_ctas = nullptr;
    int32_t *dt_blk_row0 = nullptr, *dt_row_state = nullptr, *dt_state_row = nullptr, *dt_state_blk = nullptr,
            *dt_blk_ent_ptr = nullptr;
    int64_t *dt_slot_off = nullptr, *dt_blk_ent_off = nullptr;
    int transport_variant = -1;
    // stream store (variant 2)
    bool stream_ok = false;
    std::string stream_why;
    StreamHost shost;  // kept only for EPHC_HOST_ONLY handles (ephc_export_stream)
    int32_t s_ncta = 0, s_Ra = 0, s_Rb = 0, s_ntile = 0;
    int64_t s_entries = 0, s_part_rows = 0, bytes_stream = 0;
    double *ds_w = nullptr, *ds_part = nullptr;
    uint32_t *ds_code = nullptr, *ds_iq = nullptr;
    uint16_t *ds_perm = nullptr, *ds_aid = nullptr, *ds_ast = nullptr, *ds_bid = nullptr, *ds_bst = nullptr;
    StreamChunk *ds_chunks = nullptr;
    StreamTile *ds_tiles = nullptr;
    int32_t *ds_order = nullptr;
    int *ds_counter = nullptr;
    int32_t *ds_row_state = nullptr, *ds_state_row = nullptr, *ds_state_blk = nullptr, *ds_blk_row0 = nullptr,
            *ds_blk_ent_ptr = nullptr;
    int64_t *ds_slot_off = nullptr, *ds_blk_ent_off = nullptr;
    // resident-tile store (variant 3)
    bool res_ok = false;
    std::string res_why;
    ResHost rhost;  // kept only for EPHC_HOST_ONLY handles (ephc_export_res)
    int32_t x_Ra = 0, x_Rcap = 0, x_RbMax = 0, x_ntile = 0, x_ncta = 0, x_nrows = 0;
    int64_t x_entries = 0, x_part_rows = 0, x_smem_tile = 0, bytes_res = 0;
    int x_mode = 0;  // launch mode of res_kernel (kResModes)
    unsigned char *dx_blob = nullptr;
    uint32_t *dx_iqn = nullptr;
    ResTile *dx_tiles = nullptr;
    int32_t *dx_cta_ptr = nullptr;
    double *dx_part = nullptr, *dx_fc = nullptr;
    int32_t *dx_row_state = nullptr, *dx_state_row = nullptr, *dx_state_blk = nullptr, *dx_blk_row0 = nullptr,
            *dx_blk_ent_ptr = nullptr;
    int64_t *dx_slot_off = nullptr, *dx_blk_ent_off = nullptr;
    // the paper's own layout (variant 4, A/B comparison only)
    bool paper_built = false, paper_ok = false;
    int64_t p_rows = 0, p_targets = 0, bytes_paper = 0;
    PaperChannel *dp_ch = nullptr;
    int32_t *dp_ik = nullptr, *dp_ikq = nullptr, *dp_iq = nullptr;
    uint32_t *dp_src = nullptr;
    PaperTarget *dp_targets = nullptr;
    double *dp_sc_col = nullptr;
    // row store (transport_iter of the gather path)
    bool rows_ok = false;
    bool gather_dev = false;  // the gather store is in device memory (uploaded when a call path needs it)
    int32_t r_nstrip = 0, r_Rb = 0, r_Ra = 0;
    int64_t bytes_rows = 0;
    double *dr_W = nullptr, *dr_Fc = nullptr, *dr_Fc2 = nullptr;  // Fc / Fc2: compact F of chained iterations (ping-pong)
    double *d_Fscr = nullptr;  // [3][ns] scratch of ephc_transport_iters on the stores without a compact copy
    int32_t r_nrows = 0;
    uint16_t *dr_idx = nullptr;
    // mode-collapsed row store (EPHC_TRANSPORT_COLLAPSE): built on request, used after ephc_set_transport_collapsed(h, 1)
    bool collapse_built = false, collapse_on = false, collapse_ready = false;  // ready: summed from the current weights
    int64_t c_nent = 0, bytes_collapsed = 0;
    uint16_t *dc_idx = nullptr, *dc_count = nullptr;
    uint32_t *dc_first = nullptr;
    double *dc_W = nullptr;
    RowSeg *dc_segs = nullptr;
    RowTile *dc_tiles = nullptr;
    RowStrip *dc_strips = nullptr;
    int32_t *dr_cols = nullptr;   // sparse staging: the strips' partner-row lists (null otherwise)
    uint32_t *dr_meta = nullptr;  // per entry: (iq * nnu + mode) | kind << 31
    double *dr_wst = nullptr;     // per entry: channel weight
    RowSeg *dr_segs = nullptr;
    RowTile *dr_tiles = nullptr;
    RowStrip *dr_strips = nullptr;
    int32_t *dr_row_state = nullptr, *dr_state_row = nullptr;
};

static void free_dev(ephc_handle *h) {
    void *ptrs[] = {h->d_code, h->d_w, h->d_hp_k, h->d_hp_q, h->d_tasks, h->d_rounds, h->d_wus, h->d_gW,
                    h->d_y[0], h->d_y[1], h->d_ksum, h->d_wusum, h->d_hf, h->d_hN, h->d_hI, h->d_tr[0],
                    h->d_tr[1], h->d_tr[2], h->d_tr[3], h->d_tr[4], h->d_sumf, h->dt_w, h->dt_part, h->dt_Wf,
                    h->dt_Wr, h->dt_code, h->dt_prec, h->dt_slices, h->dt_tiles, h->dt_ctas, h->dt_blk_row0,
                    h->dt_row_state, h->dt_state_row, h->dt_state_blk, h->dt_blk_ent_ptr, h->dt_blk_ent_off,
                    h->dt_slot_off, h->dr_W, h->dr_Fc, h->dr_Fc2, h->d_Fscr, h->dr_idx, h->dc_idx, h->dc_count, h->dc_first, h->dc_W, h->dc_segs, h->dc_tiles, h->dc_strips, h->dr_cols, h->dr_meta, h->dr_wst, h->dr_segs, h->dr_tiles, h->dr_strips,
                    h->dr_row_state, h->dr_state_row, h->ds_w, h->ds_part, h->ds_code, h->ds_iq, h->ds_perm, h->ds_aid,
                    h->ds_ast, h->ds_bid, h->ds_bst, h->ds_chunks, h->ds_tiles, h->ds_order, h->ds_counter, h->ds_row_state,
                    h->ds_state_row, h->ds_state_blk, h->ds_blk_row0, h->ds_blk_ent_ptr, h->ds_slot_off,
                    h->ds_blk_ent_off, h->dx_blob, h->dx_iqn, h->dx_tiles, h->dx_cta_ptr, h->dx_fc, h->dx_part,
                    h->dx_row_state, h->dx_state_row, h->dx_state_blk, h->dx_blk_row0, h->dx_blk_ent_ptr, h->dx_slot_off,
                    h->dx_blk_ent_off, h->dp_ch, h->dp_ik, h->dp_ikq, h->dp_iq, h->dp_src, h->dp_targets, h->dp_sc_col, h->d_nbr, h->d_drift};
    for (void *p : ptrs)
        if (p) cudaFree(p);
    if (h->d_sumstep) cudaFree(h->d_sumstep);
    if (h->rk_graph) cudaGraphExecDestroy(h->rk_graph);
    if (h->cap_stream) cudaStreamDestroy(h->cap_stream);
}

template <class T>
static int upload(T **dst, const std::vector<T> &src, int64_t *bytes) {
    const size_t n = src.size() * sizeof(T);
    CUDA_TRY(cudaMalloc((void **)dst, n > 0 ? n : sizeof(T)));
    if (n) CUDA_TRY(cudaMemcpy(*dst, src.data(), n, cudaMemcpyHostToDevice));
    *bytes += (int64_t)n;
    return EPHC_OK;
}

extern "C" const char *ephc_last_error(void) { return g_err.c_str(); }
extern "C" const char *ephc_version(void) { return "ephc 0.1 (sm_100a, fp64)"; }

// ---- the optional stores: each is built (and uploaded) once, at ephc_build_channels when the automatic choice needs
// it, otherwise by ephc_set_variant; EPHC_HOST_ONLY handles build all of them for the export calls -----------------------
static ephc_problem problem_view(const ephc_handle *h) {  // what the store builders read of the problem
    ephc_problem q;
    std::memset(&q, 0, sizeof(q));
    q.nk = h->d.nk;
    q.nb = h->d.nb;
    q.nnu = h->d.nnu;
    q.E = h->E.data();
    q.emin = h->emin;
    q.emax = h->emax;
    q.npair = (int64_t)h->pair_ik.size();
    q.pair_ik = h->pair_ik.data();
    q.pair_ikq = h->pair_ikq.data();
    return q;
}

// The two-sided gather store in device memory.  ephc_build_channels uploads it when the automatic choice computes on it
// (L2-resident problems, k-sharded handles, no row store); otherwise the first ephc_set_variant(0) rebuilds it from the
// canonical list and uploads it (that call allocates and copies).
static int upload_gather(ephc_handle *h, const GatherHost &g) {
    if (h->gather_dev) return EPHC_OK;
    int64_t b = 0;
    int rc = upload(&h->d_code, g.code, &b);
    if (rc == EPHC_OK) rc = upload(&h->d_w, g.w, &b);
    if (rc == EPHC_OK) rc = upload(&h->d_hp_k, g.hp_k, &b);
    if (rc == EPHC_OK) rc = upload(&h->d_hp_q, g.hp_q, &b);
    if (rc == EPHC_OK) rc = upload(&h->d_tasks, g.tasks, &b);
    if (rc == EPHC_OK) rc = upload(&h->d_rounds, g.rounds, &b);
    if (rc == EPHC_OK) rc = upload(&h->d_wus, g.wus, &b);
    if (rc == EPHC_OK && !h->rows_ok && !h->d_gW &&
        cudaMalloc((void **)&h->d_gW, (size_t)std::max<int64_t>(1, h->g_entries) * 8) != cudaSuccess)
        rc = fail(EPHC_ENOMEM, "cudaMalloc (transport weights) failed");
    if (rc == EPHC_OK) {
        h->bytes_gather = b;
        h->gather_dev = true;
    }
    return rc;
}
static int make_gather_device(ephc_handle *h) {
    if (h->gather_dev) return EPHC_OK;
    const ephc_problem q = problem_view(h);
    std::string err;
    GatherHost g;
    int rc = build_gather(&q, h->d, h->can, g, err);
    if (rc != EPHC_OK) return fail(rc, err);
    return upload_gather(h, g);
}

static int make_tile_store(ephc_handle *h) {
    if (h->tile_built) return EPHC_OK;
    const ephc_problem q = problem_view(h);
    std::string err;
    int ncta = 2 * h->n_sm;  // two CTAs per SM walk the tile sequence
    if (const char *e = std::getenv("EPHC_TILE_CTAS")) ncta = std::max(1, std::atoi(e));
    TileHost &th = h->thost;
    int rc = build_tiles(&q, h->d, h->can, ncta, th, err);
    if (rc != EPHC_OK) return fail(rc, err);
    h->tile_built = true;
    h->tile_ok = th.supported && tile_smem_bytes(kTIter, th.Ra, th.Rb) <= 220 * 1024 &&
                 tile_smem_bytes(kTCollision, th.Ra, th.Rb) <= 220 * 1024;
    if (th.supported && !h->tile_ok) {
        th.supported = false;
        th.why = "tile store: shared-memory budget exceeded";
    }
    if (!th.supported) return EPHC_OK;
    h->t_entries = (int64_t)th.w.size();
    h->t_pieces = th.npiece;
    h->t_part_rows = th.part_rows;
    h->t_ncta = th.ncta;
    h->t_Ra = th.Ra;
    h->t_Rb = th.Rb;
    h->t_nblk = th.nblk;
    h->t_nslot = (int32_t)th.slot_off.size();
    h->t_ntile = (int32_t)th.tiles.size();
    h->bytes_tile = (int64_t)(th.w.size() * 8 + th.code.size() * 2 + th.prec.size() * 4 +
                              th.slices.size() * sizeof(TileSlice) + th.tiles.size() * sizeof(TileHdr) +
                              th.ctas.size() * sizeof(TileCta) + th.slot_off.size() * 8 +
                              (th.blk_row0.size() + th.row_state.size() + th.state_row.size() +
                               th.state_blk.size() + th.blk_ent_ptr.size()) * 4 + th.blk_ent_off.size() * 8);
    if (h->host_only) return EPHC_OK;
    int64_t bt = 0;
    rc = upload(&h->dt_w, th.w, &bt);
    if (rc == EPHC_OK) rc = upload(&h->dt_code, th.code, &bt);
    if (rc == EPHC_OK) rc = upload(&h->dt_prec, th.prec, &bt);
    if (rc == EPHC_OK) rc = upload(&h->dt_slices, th.slices, &bt);
    if (rc == EPHC_OK) rc = upload(&h->dt_tiles, th.tiles, &bt);
    if (rc == EPHC_OK) rc = upload(&h->dt_ctas, th.ctas, &bt);
    if (rc == EPHC_OK) rc = upload(&h->dt_blk_row0, th.blk_row0, &bt);
    if (rc == EPHC_OK) rc = upload(&h->dt_row_state, th.row_state, &bt);
    if (rc == EPHC_OK) rc = upload(&h->dt_state_row, th.state_row, &bt);
    if (rc == EPHC_OK) rc = upload(&h->dt_state_blk, th.state_blk, &bt);
    if (rc == EPHC_OK) rc = upload(&h->dt_blk_ent_ptr, th.blk_ent_ptr, &bt);
    if (rc == EPHC_OK) rc = upload(&h->dt_blk_ent_off, th.blk_ent_off, &bt);
    if (rc == EPHC_OK) rc = upload(&h->dt_slot_off, th.slot_off, &bt);
    if (rc == EPHC_OK && cudaMalloc((void **)&h->dt_part, (size_t)std::max<int64_t>(1, th.part_rows) * 3 * 8) != cudaSuccess)
        rc = fail(EPHC_ENOMEM, "cudaMalloc (partial sums) failed");
    // transport weights of this store (two per entry), so that ephc_transport_setup never allocates
    if (rc == EPHC_OK && (cudaMalloc((void **)&h->dt_Wf, (size_t)std::max<int64_t>(1, h->t_entries) * 8) != cudaSuccess ||
                          cudaMalloc((void **)&h->dt_Wr, (size_t)std::max<int64_t>(1, h->t_entries) * 8) != cudaSuccess))
        rc = fail(EPHC_ENOMEM, "cudaMalloc (tile transport weights) failed");
    if (rc == EPHC_OK) h->bytes_transport += h->t_entries * 16;
    // the device owns the image now; keep only the scalars
    TileHost empty;
    empty.supported = th.supported;
    empty.Ra = th.Ra; empty.Rb = th.Rb; empty.nblk = th.nblk; empty.nrows = th.nrows; empty.ncta = th.ncta;
    empty.part_rows = th.part_rows; empty.npiece = th.npiece;
    th = empty;
    if (rc != EPHC_OK) h->tile_ok = false;
    return rc;
}

static int make_stream_store(ephc_handle *h) {
    if (h->stream_built) return EPHC_OK;
    const ephc_problem q = problem_view(h);
    std::string err;
    StreamHost sh;
    int nshare = 2 * h->n_sm;  // two CTAs of 512 threads per SM
    if (const char *e = std::getenv("EPHC_STREAM_CTAS")) nshare = std::max(1, std::atoi(e));
    int rc = build_stream(&q, h->d, h->can, nshare, sh, err);
    if (rc != EPHC_OK) return fail(rc, err);
    h->stream_built = true;
    h->stream_ok = sh.supported && stream_smem_bytes(sh.Ra, sh.Rb) <= 220 * 1024;
    h->stream_why = sh.supported ? "shared-memory budget exceeded" : sh.why;
    h->s_ncta = sh.ncta;
    h->s_Ra = sh.Ra;
    h->s_Rb = sh.Rb;
    h->s_ntile = (int32_t)sh.tiles.size();
    h->s_entries = (int64_t)sh.w.size();
    h->s_part_rows = sh.part_rows;
    h->bytes_stream = (int64_t)(sh.w.size() * 8 + sh.code.size() * 4 + sh.perm.size() * 2 +
                                (sh.arow_id.size() + sh.brow_id.size()) * 4 + sh.iq.size() * 4 +
                                sh.chunks.size() * sizeof(StreamChunk) + sh.tiles.size() * sizeof(StreamTile));
    sh.perm.resize(sh.perm.size() + 8, 0);  // the staging copies read whole 8-byte pieces
    if (h->host_only) {
        h->shost = std::move(sh);
        return EPHC_OK;
    }
    if (!h->stream_ok) return EPHC_OK;
    int64_t bs = 0;
    rc = upload(&h->ds_w, sh.w, &bs);
    if (rc == EPHC_OK) rc = upload(&h->ds_code, sh.code, &bs);
    if (rc == EPHC_OK) rc = upload(&h->ds_perm, sh.perm, &bs);
    if (rc == EPHC_OK) rc = upload(&h->ds_aid, sh.arow_id, &bs);
    if (rc == EPHC_OK) rc = upload(&h->ds_ast, sh.arow_start, &bs);
    if (rc == EPHC_OK) rc = upload(&h->ds_bid, sh.brow_id, &bs);
    if (rc == EPHC_OK) rc = upload(&h->ds_bst, sh.brow_start, &bs);
    if (rc == EPHC_OK) rc = upload(&h->ds_iq, sh.iq, &bs);
    if (rc == EPHC_OK) rc = upload(&h->ds_chunks, sh.chunks, &bs);
    if (rc == EPHC_OK) rc = upload(&h->ds_tiles, sh.tiles, &bs);
    if (rc == EPHC_OK) rc = upload(&h->ds_order, sh.order, &bs);
    if (rc == EPHC_OK && (cudaMalloc((void **)&h->ds_counter, 64) != cudaSuccess || cudaMemset(h->ds_counter, 0, 64) != cudaSuccess))
        rc = fail(EPHC_ENOMEM, "cudaMalloc (tile counter) failed");
    if (rc == EPHC_OK) rc = upload(&h->ds_row_state, sh.row_state, &bs);
    if (rc == EPHC_OK) rc = upload(&h->ds_state_row, sh.state_row, &bs);
    if (rc == EPHC_OK) rc = upload(&h->ds_state_blk, sh.state_blk, &bs);
    if (rc == EPHC_OK) rc = upload(&h->ds_blk_row0, sh.blk_row0, &bs);
    if (rc == EPHC_OK) rc = upload(&h->ds_blk_ent_ptr, sh.blk_ent_ptr, &bs);
    if (rc == EPHC_OK) rc = upload(&h->ds_blk_ent_off, sh.blk_ent_off, &bs);
    if (rc == EPHC_OK) rc = upload(&h->ds_slot_off, sh.slot_off, &bs);
    if (rc == EPHC_OK && cudaMalloc((void **)&h->ds_part, (size_t)std::max<int64_t>(1, sh.part_rows) * 8) != cudaSuccess)
        rc = fail(EPHC_ENOMEM, "cudaMalloc (stream partial sums) failed");
    if (rc != EPHC_OK) h->stream_ok = false;
    return rc;
}

// Launch modes of res_kernel: consumer threads, CTAs per SM, dynamic shared memory per CTA (the tile images are built
// for that budget; 227 KB per SM minus 1 KB per CTA and the static barriers).
struct ResMode {
    int nl, ctas;
    int64_t smem;
};
static const ResMode kResModes[] = {{256, 2, 112 * 1024}, {512, 1, 225 * 1024}, {256, 1, 225 * 1024}, {384, 1, 225 * 1024},
                                    {128, 4, 55 * 1024},  {512, 2, 112 * 1024}, {768, 1, 225 * 1024}};
constexpr int kResNModes = (int)(sizeof(kResModes) / sizeof(kResModes[0]));
constexpr int kResDefaultMode = 0;

static int upload_res(ephc_handle *h, const ResHost &xh);
static int calibrate_res(ephc_handle *h, ResHost &xh);
static int launch_res(ephc_handle *h, const double *f, const double *N, cudaStream_t s, bool fc_ready, long long *tile_cycles);
static int set_kernel_attributes(int device);

static int make_res_store(ephc_handle *h) {
    if (h->res_built) return EPHC_OK;
    const ephc_problem q = problem_view(h);
    std::string err;
    ResHost xh;
    // Launch mode (measured on B200 with the calibrated schedule, collision call in us for modes 0 / 1 / 2 / 3):
    //   many channels per pair (large cell: 285 / 297 / 290 / 288): two CTAs of 8 consumer warps per SM;
    //   few channels per pair: ONE CTA per SM with tiles twice as large and shares calibrated on the device --
    //   8 consumer warps when the rows of a tile are long (GaAs-like: 1534 / 1559 / 1440 / 1481), 12 when a half-size
    //   tile's rows would carry fewer than about six entries (Si-like: 105 / 98.9 / 99.6 / 97.1).
    h->x_mode = kResDefaultMode;
    {
        int64_t nrows = 0;
        for (int64_t st = 0; st < h->d.ns; ++st) nrows += q.E[st] >= q.emin && q.E[st] <= q.emax;
        const double per_pair = (double)h->can.nw / (double)std::max<int64_t>(1, h->can.npair_active);
        const double rho = (double)h->can.nw / (0.5 * (double)nrows * (double)nrows + 1.0);
        const double fit = 44000.0 / (15.5 + 8.0 * h->d.nnu / std::max(1.0, per_pair));
        if (per_pair < 64.0) h->x_mode = std::sqrt(rho * fit) < 6.0 ? 3 : 2;
    }
    if (const char *e = std::getenv("EPHC_RES_MODE")) h->x_mode = std::min(kResNModes - 1, std::max(0, std::atoi(e)));
    const ResMode &md = kResModes[h->x_mode];
    int nshare = md.ctas * h->n_sm;
    if (const char *e = std::getenv("EPHC_RES_CTAS")) nshare = std::max(1, std::atoi(e));
    int64_t cap = md.smem;
    if (const char *e = std::getenv("EPHC_RES_SMEM")) cap = std::min<int64_t>(md.smem, std::max(8192, std::atoi(e)));
    int rc = build_res(&q, h->d, h->can, nshare, cap, md.nl / 32, xh, err);
    if (rc != EPHC_OK) return fail(rc, err);
    h->res_built = true;
    h->res_ok = xh.supported && res_smem_total(xh.Ra, xh.Rcap, xh.smem_tile) <= md.smem;
    h->res_why = xh.supported ? "shared-memory budget exceeded" : xh.why;
    h->x_ncta = xh.ncta;
    h->x_ntile = (int32_t)xh.tiles.size();
    h->x_Ra = xh.Ra;
    h->x_Rcap = xh.Rcap;
    h->x_RbMax = xh.RbMax;
    h->x_nrows = xh.nrows;
    h->x_entries = xh.nent;
    h->x_part_rows = xh.part_rows;
    h->x_smem_tile = xh.smem_tile;
    h->bytes_res = (int64_t)(xh.blob.size() + xh.iqn.size() * 4 + xh.tiles.size() * sizeof(ResTile) + xh.cta_ptr.size() * 4);
    if (h->host_only) {
        if (const char *e = std::getenv("EPHC_RES_TEST_RECUT")) {  // structural tests of res_reschedule: pseudo-random tile costs
            std::vector<double> cost(xh.tiles.size());
            uint32_t x = (uint32_t)std::atoi(e) * 2654435761u + 12345u;
            for (double &c : cost) {
                x = x * 1664525u + 1013904223u;
                c = 1.0 + (double)(x >> 8) / 65536.0;
            }
            rc = res_reschedule(xh, cost, err);
            if (rc != EPHC_OK) return fail(rc, err);
        }
        h->rhost = std::move(xh);
        return EPHC_OK;
    }
    if (!h->res_ok) return EPHC_OK;
    rc = upload_res(h, xh);
    // Calibration: the shares of the static schedule are re-cut from cycles measured on this device at build (the cost
    // model of the builder is off by 10-20 % for the slowest CTA).  This build-time step allocates and frees scratch.
    // Only where a CTA has an SM to itself: with two CTAs per SM a share's time depends on its neighbour and the iteration
    // does not settle (measured: GaAs 1559 -> 1617 us, large cell 285 -> 297 us; one CTA per SM: Si 104 -> 98.5 us).
    if (rc == EPHC_OK && h->res_ok && md.ctas == 1 && std::getenv("EPHC_RES_NO_CALIBRATE") == nullptr && xh.tiles.size() > 1)
        rc = calibrate_res(h, xh);
    return rc;
}

static int upload_res(ephc_handle *h, const ResHost &xh) {
    int rc;
    int64_t bx = 0;
    h->x_part_rows = xh.part_rows;
    rc = upload(&h->dx_blob, xh.blob, &bx);
    if (rc == EPHC_OK) rc = upload(&h->dx_iqn, xh.iqn, &bx);
    if (rc == EPHC_OK) rc = upload(&h->dx_tiles, xh.tiles, &bx);
    if (rc == EPHC_OK) rc = upload(&h->dx_cta_ptr, xh.cta_ptr, &bx);
    if (rc == EPHC_OK) rc = upload(&h->dx_row_state, xh.row_state, &bx);
    if (rc == EPHC_OK) rc = upload(&h->dx_state_row, xh.state_row, &bx);
    if (rc == EPHC_OK) rc = upload(&h->dx_state_blk, xh.state_blk, &bx);
    if (rc == EPHC_OK) rc = upload(&h->dx_blk_row0, xh.blk_row0, &bx);
    if (rc == EPHC_OK) rc = upload(&h->dx_blk_ent_ptr, xh.blk_ent_ptr, &bx);
    if (rc == EPHC_OK) rc = upload(&h->dx_blk_ent_off, xh.blk_ent_off, &bx);
    if (rc == EPHC_OK) rc = upload(&h->dx_slot_off, xh.slot_off, &bx);
    if (rc == EPHC_OK && cudaMalloc((void **)&h->dx_part, (size_t)std::max<int64_t>(1, xh.part_rows) * 8) != cudaSuccess)
        rc = fail(EPHC_ENOMEM, "cudaMalloc (resident-tile partial sums) failed");
    if (rc == EPHC_OK && (cudaMalloc((void **)&h->dx_fc, ((size_t)xh.nrows + 4) * 8) != cudaSuccess ||
                          cudaMemset(h->dx_fc, 0, ((size_t)xh.nrows + 4) * 8) != cudaSuccess))
        rc = fail(EPHC_ENOMEM, "cudaMalloc (compact f) failed");
    if (rc != EPHC_OK) h->res_ok = false;
    return rc;
}

template <class T>
static int reupload(T **dst, const std::vector<T> &src) {  // replaces a device array of the handle
    if (*dst) cudaFree(*dst);
    *dst = nullptr;
    int64_t b = 0;
    return upload(dst, src, &b);
}

static int calibrate_res(ephc_handle *h, ResHost &xh) {
    const int64_t ntile = (int64_t)xh.tiles.size();
    const size_t nN = (size_t)h->d.nq * h->d.nnu * 8;
    long long *d_cyc = nullptr;
    double *d_N = nullptr;
    int rc = EPHC_OK;
    if (cudaMalloc((void **)&d_cyc, (size_t)ntile * 8) != cudaSuccess || cudaMalloc((void **)&d_N, nN) != cudaSuccess ||
        cudaMemset(d_N, 0, nN) != cudaSuccess || cudaMemset(d_cyc, 0, (size_t)ntile * 8) != cudaSuccess) {
        cudaGetLastError();
        if (d_cyc) cudaFree(d_cyc);
        if (d_N) cudaFree(d_N);
        return EPHC_OK;  // no memory for the measurement: the model's schedule stays
    }
    if ((rc = set_kernel_attributes(h->device)) == EPHC_OK) {
        // Fixed-point iteration on the shares: the model's tile costs are scaled by (measured cycles / model work) of
        // the share they are in, the shares are re-cut, and again.  Sums over a share are robust where single tile
        // times are not (two CTAs share an SM; waits depend on the neighbours in the pipeline).
        std::vector<double> cost = xh.tile_work;
        std::vector<long long> cyc((size_t)ntile);
        const int64_t launches0 = h->launches;
        int rounds = 3;
        if (const char *e = std::getenv("EPHC_RES_CALIB_ROUNDS")) rounds = std::max(0, std::atoi(e));
        for (int round = 0; round < rounds && rc == EPHC_OK; ++round) {
            std::vector<double> meas((size_t)ntile, 0.0);
            for (int r = 0; r < 3 && rc == EPHC_OK; ++r) {  // the first launch warms up
                rc = launch_res(h, nullptr, d_N, nullptr, true, d_cyc);  // f = 0 (the compact copy was zeroed at upload)
                if (rc == EPHC_OK && cudaMemcpy(cyc.data(), d_cyc, (size_t)ntile * 8, cudaMemcpyDeviceToHost) != cudaSuccess)
                    rc = fail(EPHC_ECUDA, "calibration of the resident-tile schedule failed");
                if (r > 0)
                    for (int64_t i = 0; i < ntile; ++i) meas[i] += (double)cyc[i];
            }
            if (rc != EPHC_OK) break;
            double tot_m = 0.0, tot_c = 0.0, worst = 0.0;
            for (int64_t i = 0; i < ntile; ++i) tot_m += meas[i], tot_c += cost[i];
            for (int32_t c = 0; c < xh.ncta; ++c) {
                double m = 0.0, w = 0.0;
                for (int32_t i = xh.cta_ptr[c]; i < xh.cta_ptr[c + 1]; ++i) m += meas[i], w += cost[i];
                if (w <= 0.0 || m <= 0.0) continue;
                const double fac = (m / tot_m) / (w / tot_c);  // > 1: this share takes longer than the model says
                worst = std::max(worst, m);
                for (int32_t i = xh.cta_ptr[c]; i < xh.cta_ptr[c + 1]; ++i) cost[i] *= fac;
            }
            if (std::getenv("EPHC_DEBUG"))
                std::fprintf(stderr, "res calibration round %d: slowest share %.0f cycles, mean %.0f\n", round, worst / 2, tot_m / 2 / xh.ncta);
            std::string err;
            if ((rc = res_reschedule(xh, cost, err)) != EPHC_OK) {
                rc = fail(rc, err);
                break;
            }
            h->x_part_rows = xh.part_rows;
            rc = reupload(&h->dx_tiles, xh.tiles);
            if (rc == EPHC_OK) rc = reupload(&h->dx_cta_ptr, xh.cta_ptr);
            if (rc == EPHC_OK) rc = reupload(&h->dx_blk_ent_ptr, xh.blk_ent_ptr);
            if (rc == EPHC_OK) rc = reupload(&h->dx_blk_ent_off, xh.blk_ent_off);
            if (rc == EPHC_OK) rc = reupload(&h->dx_slot_off, xh.slot_off);
            if (rc == EPHC_OK) {
                cudaFree(h->dx_part);
                h->dx_part = nullptr;
                if (cudaMalloc((void **)&h->dx_part, (size_t)std::max<int64_t>(1, xh.part_rows) * 8) != cudaSuccess)
                    rc = fail(EPHC_ENOMEM, "cudaMalloc (resident-tile partial sums) failed");
            }
            if (rc != EPHC_OK) h->res_ok = false;
        }
        h->launches = launches0;  // build-time launches are not part of the count the callers see
    }
    cudaFree(d_cyc);
    cudaFree(d_N);
    return rc;
}

// The paper's layout: scatter, scatter_channels, stargets_sources, targets, built on the CPU once.
static int make_paper_store(ephc_handle *h) {
    if (h->paper_built) return EPHC_OK;
    if (h->host_only) return fail(EPHC_ESTATE, "the paper-layout variant needs a device handle");
    const Canonical &c = h->can;
    const int64_t npair = (int64_t)h->pair_ik.size();
    const int nb = h->d.nb;
    if (c.nw >= 0x7fffffffLL) return fail(EPHC_ELIMIT, "paper layout: more than 2^31 channel weights");
    std::vector<PaperChannel> ch;
    std::vector<int32_t> ik, ikq, iq;
    std::vector<PaperTarget> targets;
    std::vector<uint32_t> src;
    try {
        ch.reserve((size_t)c.nw);
        std::vector<int64_t> cnt((size_t)h->d.ns + 1, 0);
        for (int64_t ip = 0; ip < npair; ++ip) {
            if (c.pair_ch0[ip + 1] == c.pair_ch0[ip]) continue;
            const uint32_t row = (uint32_t)ik.size();
            ik.push_back(h->pair_ik[ip]);
            ikq.push_back(h->pair_ikq[ip]);
            iq.push_back(c.pair_iq[ip]);
            for (int64_t j = c.pair_ch0[ip]; j < c.pair_ch0[ip + 1]; ++j) {
                const uint32_t code = c.ch_code[j];  // n | m << 4 | nu << 8
                const int64_t a = (int64_t)h->pair_ik[ip] * nb + (code & 15), b = (int64_t)h->pair_ikq[ip] * nb + ((code >> 4) & 15);
                for (int kind = 0; kind < 2; ++kind) {
                    const double w = kind ? c.ch_wem[j] : c.ch_wabs[j];
                    if (w == 0.0) continue;
                    ch.push_back(PaperChannel{w, code | ((uint32_t)kind << 14), row});
                    cnt[a + 1]++;
                    cnt[b + 1]++;
                }
            }
        }
        // target layer: two rows per channel, sorted by target; one target per state that is touched
        for (int64_t s = 0; s < h->d.ns; ++s) cnt[s + 1] += cnt[s];
        src.resize((size_t)cnt[h->d.ns]);
        std::vector<int64_t> cur(cnt.begin(), cnt.end() - 1);
        for (int64_t r = 0; r < (int64_t)ch.size(); ++r) {
            const uint32_t code = ch[r].bnds_idx;
            const int64_t a = (int64_t)ik[ch[r].kq_idx] * nb + (code & 15), b = (int64_t)ikq[ch[r].kq_idx] * nb + ((code >> 4) & 15);
            src[cur[a]++] = (uint32_t)r << 1;
            src[cur[b]++] = ((uint32_t)r << 1) | 1u;
        }
        for (int64_t s = 0; s < h->d.ns; ++s)
            if (cnt[s + 1] > cnt[s]) targets.push_back(PaperTarget{cnt[s], (int32_t)(cnt[s + 1] - cnt[s]), (int32_t)s});
    } catch (const std::bad_alloc &) {
        return fail(EPHC_ENOMEM, "host allocation failed (paper layout)");
    }
    h->paper_built = true;
    h->p_rows = (int64_t)ch.size();
    h->p_targets = (int64_t)targets.size();
    int64_t b = 0;
    int rc = upload(&h->dp_ch, ch, &b);
    if (rc == EPHC_OK) rc = upload(&h->dp_ik, ik, &b);
    if (rc == EPHC_OK) rc = upload(&h->dp_ikq, ikq, &b);
    if (rc == EPHC_OK) rc = upload(&h->dp_iq, iq, &b);
    if (rc == EPHC_OK) rc = upload(&h->dp_src, src, &b);
    if (rc == EPHC_OK) rc = upload(&h->dp_targets, targets, &b);
    if (rc == EPHC_OK && cudaMalloc((void **)&h->dp_sc_col, (size_t)std::max<int64_t>(1, h->p_rows) * 8) != cudaSuccess)
        rc = fail(EPHC_ENOMEM, "cudaMalloc (sc_col) failed");
    h->bytes_paper = b + h->p_rows * 8;
    h->paper_ok = rc == EPHC_OK;
    return rc;
}

// Automatic choice for collision / RK stages (measured on B200): the two-sided gather store while
// it stays resident in the 126 MB L2; beyond that the resident-tile store (round 2: 126 us vs 130 us on the stream store
// at 1.26e7 channels, nb = 4; 2.12 ms vs 2.45 ms at 1.94e8 channels, nb = 1; 335 us vs 597 us at 4.99e7 channels,
// nb = 16, nnu = 36); the stream store remains the fallback when a problem exceeds the tile format's limits.
static int auto_coll_variant(const ephc_handle *h) {
    if (h->ranged) return 0;  // a k-sharded handle owns destinations: the two-sided, destination-sorted store
    if (h->g_entries * 12 <= (int64_t)96 << 20) return 0;
    return 3;
}

// Channel selection on the device (EPHC_SELECT_GPU): uploads the problem, counts the active channels of
// every candidate pair, prefix-sums the counts on the host, fills the canonical list on the device and brings it back.
// Same list as build_canonical (bit-exact indices; weights within the two exp implementations).
static int build_canonical_gpu(const ephc_problem *p, const Dims &d, Canonical &c, std::string &err) {
    int rc = validate_problem(p, d, err);
    if (rc != EPHC_OK) return rc;
    const int64_t npair = p->npair, blk = (int64_t)d.nnu * d.nb * d.nb;
    std::vector<void *> owned;
    auto dev_alloc = [&](size_t bytes) -> void * {
        void *q = nullptr;
        if (cudaMalloc(&q, std::max<size_t>(bytes, 8)) != cudaSuccess) return nullptr;
        owned.push_back(q);
        return q;
    };
    auto cleanup = [&]() {
        for (void *q : owned) cudaFree(q);
    };
    auto dev_copy = [&](const void *src, size_t bytes) -> void * {
        void *q = dev_alloc(bytes);
        if (q && bytes && cudaMemcpy(q, src, bytes, cudaMemcpyHostToDevice) != cudaSuccess) return nullptr;
        return q;
    };
    SelectParams P;
    std::memset(&P, 0, sizeof(P));
    P.pair_ik = (const int32_t *)dev_copy(p->pair_ik, (size_t)npair * 4);
    P.pair_ikq = (const int32_t *)dev_copy(p->pair_ikq, (size_t)npair * 4);
    P.kfull = (const int32_t *)dev_copy(p->kfull, (size_t)d.nk * 4);
    P.E = (const double *)dev_copy(p->E, (size_t)d.ns * 8);
    P.hw = (const double *)dev_copy(p->hw, (size_t)d.nq * d.nnu * 8);
    P.g2 = (const double *)dev_copy(p->g2, (size_t)(npair * blk) * 8);
    P.cnt_ch = (uint32_t *)dev_alloc((size_t)npair * 4);
    P.cnt_dg = (uint32_t *)dev_alloc((size_t)npair * 4);
    P.pair_iq = (int32_t *)dev_alloc((size_t)npair * 4);
    int64_t *d_ch0 = (int64_t *)dev_alloc((size_t)(npair + 1) * 8), *d_dg0 = (int64_t *)dev_alloc((size_t)(npair + 1) * 8);
    if (!P.pair_ik || !P.pair_ikq || !P.kfull || !P.E || !P.hw || !P.g2 || !P.cnt_ch || !P.cnt_dg || !P.pair_iq || !d_ch0 || !d_dg0) {
        cleanup();
        err = "device allocation or copy failed (channel selection)";
        return EPHC_ENOMEM;
    }
    P.nb = d.nb;
    P.nnu = d.nnu;
    P.g0 = d.grid[0];
    P.g1 = d.grid[1];
    P.g2n = d.grid[2];
    P.emin = p->emin;
    P.emax = p->emax;
    P.sigma = p->sigma;
    P.cut = p->ncut * p->sigma;
    P.g2_cut = p->g2_cut;
    P.C = d.C;
    P.npair = npair;
    const unsigned grid = (unsigned)((npair + 127) / 128);
    try {
        std::vector<uint32_t> cch((size_t)npair), cdg((size_t)npair);
        c.pair_iq.assign((size_t)npair, 0);
        c.pair_ch0.assign((size_t)npair + 1, 0);
        c.pair_dg0.assign((size_t)npair + 1, 0);
        if (npair > 0) {
            select_kernel<false><<<grid, 128>>>(P);
            if (cudaMemcpy(cch.data(), P.cnt_ch, (size_t)npair * 4, cudaMemcpyDeviceToHost) != cudaSuccess ||
                cudaMemcpy(cdg.data(), P.cnt_dg, (size_t)npair * 4, cudaMemcpyDeviceToHost) != cudaSuccess ||
                cudaMemcpy(c.pair_iq.data(), P.pair_iq, (size_t)npair * 4, cudaMemcpyDeviceToHost) != cudaSuccess) {
                cleanup();
                err = std::string("channel selection (count pass): ") + cudaGetErrorString(cudaGetLastError());
                return EPHC_ECUDA;
            }
        }
        int64_t npa = 0;
        for (int64_t ip = 0; ip < npair; ++ip) {
            npa += (cch[ip] + cdg[ip]) > 0;
            c.pair_ch0[ip + 1] = c.pair_ch0[ip] + cch[ip];
            c.pair_dg0[ip + 1] = c.pair_dg0[ip] + cdg[ip];
        }
        c.nch = c.pair_ch0[npair];
        c.ndiag = c.pair_dg0[npair];
        c.npair_active = npa;
        c.ch_code.resize((size_t)c.nch);
        c.ch_wabs.resize((size_t)c.nch);
        c.ch_wem.resize((size_t)c.nch);
        c.dg_s.resize((size_t)c.ndiag);
        c.dg_nu.resize((size_t)c.ndiag);
        c.dg_wabs.resize((size_t)c.ndiag);
        c.dg_wem.resize((size_t)c.ndiag);
        P.ch_code = (uint16_t *)dev_alloc((size_t)c.nch * 2);
        P.ch_wabs = (double *)dev_alloc((size_t)c.nch * 8);
        P.ch_wem = (double *)dev_alloc((size_t)c.nch * 8);
        P.dg_s = (int32_t *)dev_alloc((size_t)c.ndiag * 4);
        P.dg_nu = (int32_t *)dev_alloc((size_t)c.ndiag * 4);
        P.dg_wabs = (double *)dev_alloc((size_t)c.ndiag * 8);
        P.dg_wem = (double *)dev_alloc((size_t)c.ndiag * 8);
        P.ch0 = d_ch0;
        P.dg0 = d_dg0;
        bool ok = P.ch_code && P.ch_wabs && P.ch_wem && P.dg_s && P.dg_nu && P.dg_wabs && P.dg_wem &&
                  cudaMemcpy(d_ch0, c.pair_ch0.data(), (size_t)(npair + 1) * 8, cudaMemcpyHostToDevice) == cudaSuccess &&
                  cudaMemcpy(d_dg0, c.pair_dg0.data(), (size_t)(npair + 1) * 8, cudaMemcpyHostToDevice) == cudaSuccess;
        if (ok && npair > 0) {
            select_kernel<true><<<grid, 128>>>(P);
            ok = cudaMemcpy(c.ch_code.data(), P.ch_code, (size_t)c.nch * 2, cudaMemcpyDeviceToHost) == cudaSuccess &&
                 cudaMemcpy(c.ch_wabs.data(), P.ch_wabs, (size_t)c.nch * 8, cudaMemcpyDeviceToHost) == cudaSuccess &&
                 cudaMemcpy(c.ch_wem.data(), P.ch_wem, (size_t)c.nch * 8, cudaMemcpyDeviceToHost) == cudaSuccess &&
                 cudaMemcpy(c.dg_s.data(), P.dg_s, (size_t)c.ndiag * 4, cudaMemcpyDeviceToHost) == cudaSuccess &&
                 cudaMemcpy(c.dg_nu.data(), P.dg_nu, (size_t)c.ndiag * 4, cudaMemcpyDeviceToHost) == cudaSuccess &&
                 cudaMemcpy(c.dg_wabs.data(), P.dg_wabs, (size_t)c.ndiag * 8, cudaMemcpyDeviceToHost) == cudaSuccess &&
                 cudaMemcpy(c.dg_wem.data(), P.dg_wem, (size_t)c.ndiag * 8, cudaMemcpyDeviceToHost) == cudaSuccess;
        }
        cleanup();
        if (!ok) {
            err = std::string("channel selection (fill pass): ") + cudaGetErrorString(cudaGetLastError());
            return EPHC_ECUDA;
        }
    } catch (const std::bad_alloc &) {
        cleanup();
        err = "host allocation failed (canonical channel list)";
        return EPHC_ENOMEM;
    }
    int64_t nw = 0;
#pragma omp parallel for reduction(+ : nw) schedule(static)
    for (int64_t j = 0; j < c.nch; ++j) nw += (c.ch_wabs[j] != 0.0) + (c.ch_wem[j] != 0.0);
    c.nw = nw;
    c.iq0 = 0;
    return EPHC_OK;
}

static int build_impl(const ephc_problem *p, int32_t k_lo, int32_t k_hi, bool ranged, ephc_handle **out);
static inline int coll_variant(const ephc_handle *h);
static inline int rt_variant(const ephc_handle *h);

extern "C" int ephc_build_channels(const ephc_problem *p, ephc_handle **out) {
    if (out) *out = nullptr;
    if (!p || !out) return fail(EPHC_EINVAL, "null argument");
    return build_impl(p, 0, p->nk, false, out);
}

extern "C" int ephc_build_channels_range(const ephc_problem *p, int32_t k_lo, int32_t k_hi, ephc_handle **out) {
    if (out) *out = nullptr;
    if (!p || !out) return fail(EPHC_EINVAL, "null argument");
    if (k_lo < 0 || k_hi < k_lo || k_hi > p->nk) return fail(EPHC_EINVAL, "need 0 <= k_lo <= k_hi <= nk");
    return build_impl(p, k_lo, k_hi, true, out);
}

extern "C" int ephc_owned_states(const ephc_handle *h, int64_t *s_lo, int64_t *s_hi) {
    if (!h || !s_lo || !s_hi) return fail(EPHC_EINVAL, "null argument");
    *s_lo = (int64_t)h->d.k_lo * h->d.nb;
    *s_hi = (int64_t)h->d.k_hi * h->d.nb;
    return EPHC_OK;
}

static int build_impl(const ephc_problem *p, int32_t k_lo, int32_t k_hi, bool ranged, ephc_handle **out) {
    if (out) *out = nullptr;
    if (!p || !out) return fail(EPHC_EINVAL, "null argument");
    if (!p->kfull || !p->E || !p->hw || (p->npair > 0 && (!p->pair_ik || !p->pair_ikq || !p->g2)))
        return fail(EPHC_EINVAL, "null array in ephc_problem");
    if (p->nk < 1 || p->nb < 1 || p->nnu < 1 || p->npair < 0 || p->grid[0] < 1 || p->grid[1] < 1 || p->grid[2] < 1)
        return fail(EPHC_EINVAL, "nk, nb, nnu, grid must be >= 1 and npair >= 0");
    if (p->nb > 16 || p->nnu > 64) return fail(EPHC_ELIMIT, "format limit: nb <= 16, nnu <= 64");
    const int64_t nq = (int64_t)p->grid[0] * p->grid[1] * p->grid[2];
    const int64_t ns = (int64_t)p->nk * p->nb;
    if (nq > 0x7fffffffLL / p->nnu || ns > 0x7fffffffLL || p->npair > 0x7fffffffLL)
        return fail(EPHC_ELIMIT, "format limit: nq*nnu, nk*nb and npair must fit in 31 bits");
    if (p->nk > nq) return fail(EPHC_EINVAL, "nk exceeds the number of grid points");

    ephc_handle *h = new (std::nothrow) ephc_handle();
    if (!h) return fail(EPHC_ENOMEM, "host allocation failed (handle)");
    h->d.grid[0] = p->grid[0];
    h->d.grid[1] = p->grid[1];
    h->d.grid[2] = p->grid[2];
    h->d.nk = p->nk;
    h->d.nb = p->nb;
    h->d.nnu = p->nnu;
    h->d.nq = nq;
    h->d.ns = ns;
    h->d.C = 2.0 * kPi / (kHbar * (double)nq);  // R-8: N_q = points of the full grid
    h->d.k_lo = k_lo;
    h->d.k_hi = k_hi;
    h->ranged = ranged;
    h->host_only = (p->flags & EPHC_HOST_ONLY) != 0;
    if (!h->host_only) {
        // the handle belongs to the device that is current now; every later call makes it current again
        int dev_count = 0;
        cudaDeviceProp prop;
        if (cudaGetDeviceCount(&dev_count) != cudaSuccess || dev_count == 0 || cudaGetDevice(&h->device) != cudaSuccess ||
            cudaGetDeviceProperties(&prop, h->device) != cudaSuccess) {
            delete h;
            return fail(EPHC_ECUDA, "no CUDA device (pass EPHC_HOST_ONLY to build without one)");
        }
        h->n_sm = prop.multiProcessorCount;
    }

    std::string err;
    if ((p->flags & EPHC_SELECT_GPU) && h->host_only) {
        delete h;
        return fail(EPHC_EINVAL, "EPHC_SELECT_GPU needs a device handle (not EPHC_HOST_ONLY)");
    }
    int rc = (p->flags & EPHC_SELECT_GPU) ? build_canonical_gpu(p, h->d, h->can, err) : build_canonical(p, h->d, h->can, err);
    GatherHost g;
    if (rc == EPHC_OK) rc = build_gather(p, h->d, h->can, g, err);
    if (rc != EPHC_OK) {
        delete h;
        return fail(rc, err);
    }
    try {
        h->E.assign(p->E, p->E + ns);
        h->pair_ik.assign(p->pair_ik, p->pair_ik + p->npair);
        h->pair_ikq.assign(p->pair_ikq, p->pair_ikq + p->npair);
    } catch (const std::bad_alloc &) {
        delete h;
        return fail(EPHC_ENOMEM, "host allocation failed (handle)");
    }
    h->emin = p->emin;
    h->emax = p->emax;
    h->kfull.assign(p->kfull, p->kfull + p->nk);
    h->g_entries = (int64_t)g.code.size();
    h->g_halfpairs = (int64_t)g.hp_k.size();
    h->n_wu = (int32_t)g.wus.size();
    h->n_rounds = (int32_t)g.rounds.size();
    h->n_tasks = (int32_t)g.tasks.size();
    // row store for transport_iter (one CTA of 1024 threads per SM, one strip each), derived from the gather store
    RowHost rh;
    if (std::getenv("EPHC_NO_ROWS") == nullptr) {
        int nstrip = h->n_sm;
        if (const char *e = std::getenv("EPHC_ROW_STRIPS")) nstrip = std::max(1, std::atoi(e));
        rc = build_rows(p, h->d, g, nstrip, rh, err);
        if (rc != EPHC_OK) {
            delete h;
            return fail(rc, err);
        }
        h->rows_ok = row_smem_bytes(rh.Rb, rh.Ra) <= 220 * 1024;
        h->r_nstrip = (int32_t)rh.strips.size();
        h->r_Rb = rh.Rb;
        h->r_Ra = rh.Ra;
        h->r_nrows = rh.nrows;
        h->bytes_rows = (int64_t)(rh.idx.size() * 2 + rh.cols.size() * 4 + rh.meta.size() * 4 + rh.wst.size() * 8 + rh.segs.size() * sizeof(RowSeg) +
                                  rh.tiles.size() * sizeof(RowTile) + rh.strips.size() * sizeof(RowStrip) +
                                  (rh.row_state.size() + rh.state_row.size()) * 4);
        if (h->host_only) {
            if ((p->flags & EPHC_TRANSPORT_COLLAPSE) && h->rows_ok) {
                rc = build_rows_collapsed(rh, h->chost, err);
                if (rc != EPHC_OK) {
                    delete h;
                    return fail(rc, err);
                }
                h->collapse_built = true;
                h->c_nent = (int64_t)h->chost.idx.size();
            }
            h->rowhost = rh;
        }
    }
    h->bytes_gather = 0;
    if (!h->host_only) {
        // the gather store itself goes to the device only when a call path computes on it
        if (h->ranged || !h->rows_ok || auto_coll_variant(h) == 0) rc = upload_gather(h, g);
        if (rc == EPHC_OK && h->rows_ok) {
            int64_t br = 0;
            rc = upload(&h->dr_idx, rh.idx, &br);
            if (rc == EPHC_OK && !rh.cols.empty()) rc = upload(&h->dr_cols, rh.cols, &br);
            if (rc == EPHC_OK) rc = upload(&h->dr_meta, rh.meta, &br);
            if (rc == EPHC_OK) rc = upload(&h->dr_wst, rh.wst, &br);
            if (rc == EPHC_OK) rc = upload(&h->dr_segs, rh.segs, &br);
            if (rc == EPHC_OK) rc = upload(&h->dr_tiles, rh.tiles, &br);
            if (rc == EPHC_OK) rc = upload(&h->dr_strips, rh.strips, &br);
            if (rc == EPHC_OK) rc = upload(&h->dr_row_state, rh.row_state, &br);
            if (rc == EPHC_OK) rc = upload(&h->dr_state_row, rh.state_row, &br);
            if (rc == EPHC_OK && (p->flags & EPHC_TRANSPORT_COLLAPSE)) {
                RowCollapsed rc2;
                rc = build_rows_collapsed(rh, rc2, err);
                if (rc != EPHC_OK) rc = fail(rc, err);
                int64_t bc = 0;
                if (rc == EPHC_OK) rc = upload(&h->dc_idx, rc2.idx, &bc);
                if (rc == EPHC_OK) rc = upload(&h->dc_first, rc2.first, &bc);
                if (rc == EPHC_OK) rc = upload(&h->dc_count, rc2.count, &bc);
                if (rc == EPHC_OK) rc = upload(&h->dc_segs, rc2.segs, &bc);
                if (rc == EPHC_OK) rc = upload(&h->dc_tiles, rc2.tiles, &bc);
                if (rc == EPHC_OK) rc = upload(&h->dc_strips, rc2.strips, &bc);
                h->c_nent = (int64_t)rc2.idx.size();
                if (rc == EPHC_OK && cudaMalloc((void **)&h->dc_W, (size_t)std::max<int64_t>(1, h->c_nent) * 8) != cudaSuccess)
                    rc = fail(EPHC_ENOMEM, "cudaMalloc (collapsed transport weights) failed");
                h->bytes_collapsed = bc + h->c_nent * 8;
                h->collapse_built = rc == EPHC_OK;
            }
            if (rc == EPHC_OK && (cudaMalloc((void **)&h->dr_Fc, ((size_t)rh.nrows * 3 + 4) * 8) != cudaSuccess ||
                                  cudaMalloc((void **)&h->dr_Fc2, ((size_t)rh.nrows * 3 + 4) * 8) != cudaSuccess))
                rc = fail(EPHC_ENOMEM, "cudaMalloc (compact F) failed");
        }
        // everything the device entry points write besides the caller's buffers is allocated here, so that they only
        // enqueue work ("allocated once"): transport weights in gather and row order, RK4 scratch, sums
        const size_t nb8 = (size_t)ns * 8, ne8 = (size_t)std::max<int64_t>(1, h->g_entries) * 8;
        if (rc == EPHC_OK &&
            ((h->rows_ok && cudaMalloc((void **)&h->dr_W, ne8) != cudaSuccess) ||
             cudaMalloc((void **)&h->d_y[0], nb8) != cudaSuccess || cudaMalloc((void **)&h->d_y[1], nb8) != cudaSuccess ||
             cudaMalloc((void **)&h->d_ksum, nb8) != cudaSuccess || cudaMalloc((void **)&h->d_Fscr, 3 * nb8) != cudaSuccess ||
             cudaMalloc((void **)&h->d_sumstep, 8) != cudaSuccess ||
             cudaStreamCreateWithFlags(&h->cap_stream, cudaStreamNonBlocking) != cudaSuccess ||
             cudaMalloc((void **)&h->d_wusum, (size_t)std::max<int64_t>(std::max<int64_t>(h->n_wu, (ns + 255) / 256), 1) * 8) != cudaSuccess))
            rc = fail(EPHC_ENOMEM, "cudaMalloc (transport weights / RK4 scratch) failed");
        if (rc == EPHC_OK) h->bytes_transport += h->g_entries * 8;
        if (rc == EPHC_OK) {  // neighbours of every active k along the three grid axes (drift term, reading R-25)
            std::vector<int32_t> compact((size_t)nq, -1), nbr((size_t)6 * p->nk, -1);
            for (int32_t k = 0; k < p->nk; ++k) compact[p->kfull[k]] = k;
            const int32_t G0 = p->grid[0], G1 = p->grid[1], G2 = p->grid[2];
            for (int32_t k = 0; k < p->nk; ++k) {
                const int32_t kf = p->kfull[k];
                const int32_t c[3] = {kf / (G1 * G2), (kf / G2) % G1, kf % G2};
                const int32_t G[3] = {G0, G1, G2};
                for (int i = 0; i < 3; ++i)
                    for (int sgn = 0; sgn < 2; ++sgn) {
                        int32_t cc[3] = {c[0], c[1], c[2]};
                        cc[i] = (c[i] + (sgn ? G[i] - 1 : 1)) % G[i];
                        nbr[(size_t)(2 * i + sgn) * p->nk + k] = compact[((int64_t)cc[0] * G1 + cc[1]) * G2 + cc[2]];
                    }
            }
            int64_t bn = 0;
            rc = upload(&h->d_nbr, nbr, &bn);
            if (rc == EPHC_OK && cudaMalloc((void **)&h->d_drift, nb8) != cudaSuccess)
                rc = fail(EPHC_ENOMEM, "cudaMalloc (drift term) failed");
        }
    } else {
        h->bytes_gather = (int64_t)(g.code.size() * 4 + g.w.size() * 8 + g.hp_k.size() * 8 +
                                    g.tasks.size() * sizeof(Task) + g.rounds.size() * sizeof(Round) +
                                    g.wus.size() * sizeof(WorkUnit));
        h->ghost = std::move(g);
    }
    // the once-stored store of the automatic choice (the others are built when ephc_set_variant asks for them);
    // host-only handles build all of them for the export calls
    if (rc == EPHC_OK && !h->ranged) {
        const int av = auto_coll_variant(h);
        if (h->host_only || av == 3) rc = make_res_store(h);
        if (rc == EPHC_OK && (h->host_only || av == 2 || (av == 3 && !h->res_ok))) rc = make_stream_store(h);
        if (rc == EPHC_OK && (h->host_only || (av >= 2 && !h->res_ok && !h->stream_ok))) rc = make_tile_store(h);
    }
    if (rc == EPHC_OK && !h->host_only && !h->gather_dev && (coll_variant(h) == 0 || rt_variant(h) == 0)) rc = make_gather_device(h);
    if (rc != EPHC_OK) {
        const std::string msg = g_err;
        if (!h->host_only) free_dev(h);
        delete h;
        return fail(rc, msg.empty() ? err : msg);
    }
    *out = h;
    return EPHC_OK;
}

extern "C" int ephc_destroy(ephc_handle *h) {
    if (!h) return EPHC_OK;
    if (!h->host_only) free_dev(h);
    delete h;
    return EPHC_OK;
}

extern "C" int ephc_query(const ephc_handle *h, ephc_counts *o) {
    if (!h || !o) return fail(EPHC_EINVAL, "null argument");
    std::memset(o, 0, sizeof(*o));
    o->ns = h->d.ns;
    o->npair_active = h->can.npair_active;
    o->nch = h->can.nch;
    o->nw = h->can.nw;
    o->ndiag = h->can.ndiag;
    o->gather_entries = h->g_entries;
    o->gather_halfpairs = h->g_halfpairs;
    o->store_bytes_gather = h->bytes_gather + h->bytes_rows;
    o->scatter_entries = h->t_entries;
    o->scatter_pairs = h->t_pieces;
    o->store_bytes_scatter = h->bytes_tile + h->bytes_stream + h->bytes_res;
    o->store_bytes_paper = h->bytes_paper;
    o->store_bytes_transport = h->bytes_transport;
    // B_alg: every item the method must move once per evaluation.
    //   8 N_w weights + 4 N_ch channel index + 12 N_pair (ik, ikq, iq) + 16 N_s (read f, write I) + 8 nnu N_q,active
    int64_t nq_active = 0;
    {
        std::vector<uint8_t> seen((size_t)h->d.nq, 0);
        const int64_t npair = (int64_t)h->pair_ik.size();
        for (int64_t ip = 0; ip < npair; ++ip)
            if (h->can.pair_ch0[ip + 1] > h->can.pair_ch0[ip] && !seen[h->can.pair_iq[ip]]) {
                seen[h->can.pair_iq[ip]] = 1;
                ++nq_active;
            }
    }
    o->alg_bytes_collision = 8 * h->can.nw + 4 * h->can.nch + 12 * h->can.npair_active + 16 * h->d.ns +
                             8 * (int64_t)h->d.nnu * nq_active;
    //   transport: two weights per channel (16 N_ch), index, pairs, F and F' (3 components), v, tau
    o->alg_bytes_transport = 16 * h->can.nch + 4 * h->can.nch + 12 * h->can.npair_active +
                             (3 * 8 * 3 + 8) * h->d.ns;
    o->n_workunits = h->n_wu;
    o->n_rounds = h->n_rounds;
    o->n_tasks = h->n_tasks;
    return EPHC_OK;
}

extern "C" int ephc_export_channels(const ephc_handle *h, int32_t *ik, int32_t *ikq, int32_t *iq, int32_t *n,
                                    int32_t *m, int32_t *nu, double *w_abs, double *w_em) {
    if (!h) return fail(EPHC_EINVAL, "null handle");
    const int64_t npair = (int64_t)h->pair_ik.size();
    for (int64_t ip = 0; ip < npair; ++ip)
        for (int64_t j = h->can.pair_ch0[ip]; j < h->can.pair_ch0[ip + 1]; ++j) {
            const uint16_t c = h->can.ch_code[j];
            if (ik) ik[j] = h->pair_ik[ip];
            if (ikq) ikq[j] = h->pair_ikq[ip];
            if (iq) iq[j] = h->can.pair_iq[ip];
            if (n) n[j] = c & 15;
            if (m) m[j] = (c >> 4) & 15;
            if (nu) nu[j] = c >> 8;
            if (w_abs) w_abs[j] = h->can.ch_wabs[j];
            if (w_em) w_em[j] = h->can.ch_wem[j];
        }
    return EPHC_OK;
}

extern "C" int ephc_export_diag(const ephc_handle *h, int32_t *s, int32_t *iq, int32_t *nu, double *w_abs,
                                double *w_em) {
    if (!h) return fail(EPHC_EINVAL, "null handle");
    for (int64_t j = 0; j < h->can.ndiag; ++j) {
        if (s) s[j] = h->can.dg_s[j];
        if (iq) iq[j] = h->can.iq0;
        if (nu) nu[j] = h->can.dg_nu[j];
        if (w_abs) w_abs[j] = h->can.dg_wabs[j];
        if (w_em) w_em[j] = h->can.dg_wem[j];
    }
    return EPHC_OK;
}

extern "C" int ephc_export_gather(const ephc_handle *h, int32_t *dest, int32_t *partner, int32_t *iq, int32_t *nu,
                                  int32_t *kind, int32_t *diag, double *w) {
    if (!h) return fail(EPHC_EINVAL, "null handle");
    if (!h->host_only) return fail(EPHC_ESTATE, "ephc_export_gather needs a handle built with EPHC_HOST_ONLY");
    const GatherHost &g = h->ghost;
    std::vector<uint8_t> seen(g.code.size(), 0);
    for (const WorkUnit &wu : g.wus)
        for (int32_t r = wu.r0; r < wu.r1; ++r) {
            const Round &rd = g.rounds[r];
            for (int32_t t = rd.t0; t < rd.t0 + rd.nt; ++t) {
                const Task &tk = g.tasks[t];
                if (tk.row < wu.row0 || tk.row >= wu.row0 + wu.nrows || tk.len < 1 || tk.len > kTaskLen)
                    return fail(EPHC_ESTATE, "internal: task outside its work unit");
                for (int64_t e = tk.e0; e < tk.e0 + tk.len; ++e) {
                    const uint32_t c = g.code[e];
                    const uint32_t pl = c & kPairMask;
                    if (pl >= (uint32_t)rd.nhp || seen[e]) return fail(EPHC_ESTATE, "internal: bad pair index / entry visited twice");
                    seen[e] = 1;
                    if (dest) dest[e] = tk.row;
                    if (partner) partner[e] = g.hp_k[rd.hp0 + pl] * h->d.nb + (int32_t)((c >> kBandShift) & 15);
                    if (iq) iq[e] = g.hp_q[rd.hp0 + pl];
                    if (nu) nu[e] = (int32_t)((c >> kModeShift) & 63);
                    if (kind) kind[e] = (int32_t)((c >> kKindBit) & 1);
                    if (diag) diag[e] = (int32_t)(c >> kDiagBit);
                    if (w) w[e] = g.w[e];
                }
            }
        }
    for (uint8_t s : seen)
        if (!s) return fail(EPHC_ESTATE, "internal: entry not covered by any task");
    return EPHC_OK;
}

extern "C" int ephc_export_tiles(const ephc_handle *h, int32_t *a, int32_t *b, int32_t *iq, int32_t *nu,
                                 int32_t *kind, int32_t *diag, double *w) {
    if (!h) return fail(EPHC_EINVAL, "null handle");
    if (!h->host_only) return fail(EPHC_ESTATE, "ephc_export_tiles needs a handle built with EPHC_HOST_ONLY");
    if (!h->tile_ok) return fail(EPHC_ESTATE, "tile store not available for this problem: " + h->thost.why);
    const TileHost &t = h->thost;
    const int64_t npc = t.npiece;
    std::vector<uint8_t> seen(t.w.size(), 0), tile_seen(t.tiles.size(), 0);
    std::vector<int32_t> tick_a((size_t)t.Ra), tick_b((size_t)t.Rb);
    const int64_t nslot = (int64_t)t.slot_off.size();
    for (const TileCta &cta : t.ctas)
        for (int32_t it = cta.t0; it < cta.t1; ++it) {
            const TileHdr &th = t.tiles[it];
            if (tile_seen[it]++) return fail(EPHC_ESTATE, "internal: tile walked by two CTAs");
            const bool dg = (th.flags & 4) != 0;
            const bool first = (it == cta.t0) || t.tiles[it - 1].a_row0 != th.a_row0;
            const bool last = (it + 1 == cta.t1) || t.tiles[it + 1].a_row0 != th.a_row0;
            if (th.a_slot < 0 || th.a_slot >= nslot || (dg != (th.b_slot < 0)) || th.b_slot >= nslot ||
                first != ((th.flags & 1) != 0) || last != ((th.flags & 2) != 0) || th.a_rows > t.Ra || th.b_rows > t.Rb ||
                (dg && (th.b_row0 != th.a_row0 || th.b_rows != th.a_rows)) || (!dg && th.b_row0 < th.a_row0 + th.a_rows))
                return fail(EPHC_ESTATE, "internal: bad tile header");
            if (t.slot_row0[th.a_slot] != th.a_row0 || t.slot_rows[th.a_slot] != th.a_rows ||
                (!dg && (t.slot_row0[th.b_slot] != th.b_row0 || t.slot_rows[th.b_slot] != th.b_rows)) ||
                (!first && th.a_slot != t.tiles[it - 1].a_slot))
                return fail(EPHC_ESTATE, "internal: slot does not match its tile");
            const int32_t rows_a = th.a_rows, rows_b = th.b_rows;
            if (first) std::fill(tick_a.begin(), tick_a.end(), 0);
            std::fill(tick_b.begin(), tick_b.end(), 0);
            std::vector<int32_t> &tb = dg ? tick_a : tick_b;
            for (int32_t sidx = th.s0; sidx < th.s0 + th.ns; ++sidx) {
                const TileSlice &sl = t.slices[sidx];
                if (sl.np < 1 || sl.np > 32) return fail(EPHC_ESTATE, "internal: bad slice");
                int len[32];
                for (int l = 0; l < sl.np; ++l) {
                    len[l] = (int)(t.prec[npc + sl.p0 + l] >> 24);
                    if (len[l] < 1 || (l > 0 && len[l] > len[l - 1]) || (l == 0 && len[l] != sl.maxlen))
                        return fail(EPHC_ESTATE, "internal: lane lengths must descend from maxlen");
                }
                std::vector<int> colstart((size_t)sl.maxlen + 1, 0);
                for (int i = 0; i < sl.maxlen; ++i) {
                    int cnt = 0;
                    for (int l = 0; l < sl.np; ++l) cnt += len[l] > i;
                    colstart[i + 1] = colstart[i] + cnt;
                }
                for (int l = 0; l < sl.np; ++l) {
                    const uint32_t r0 = t.prec[sl.p0 + l], r1 = t.prec[npc + sl.p0 + l], r2 = t.prec[2 * npc + sl.p0 + l];
                    const int32_t ra = r0 & 0xffff, rb = r0 >> 16;
                    const int32_t nia = ((r2 >> 12) & 3) + 1, nib = ((r2 >> 28) & 3) + 1;
                    if (ra + nia > rows_a || rb + nib > rows_b) return fail(EPHC_ESTATE, "internal: row outside its block");
                    if ((int32_t)(r2 & 0xfff) != tick_a[ra]++ || (int32_t)((r2 >> 16) & 0xfff) != tb[rb]++)
                        return fail(EPHC_ESTATE, "internal: tickets out of order");
                    for (int i = 0; i < len[l]; ++i) {
                        const int64_t o = sl.e0 + colstart[i] + l;
                        if (o < 0 || o >= (int64_t)seen.size() || seen[o]) return fail(EPHC_ESTATE, "internal: entry visited twice");
                        seen[o] = 1;
                        const uint16_t c = t.code[o];
                        const int32_t n = c & 3, m = (c >> kTcM) & 3;
                        if (n >= nia || m >= nib) return fail(EPHC_ESTATE, "internal: band rank outside the window");
                        if (a) a[o] = t.row_state[th.a_row0 + ra + n];
                        if (b) b[o] = t.row_state[th.b_row0 + rb + m];
                        if (iq) iq[o] = (int32_t)(r1 & 0xffffff);
                        if (nu) nu[o] = (c >> kTcNu) & 7;
                        if (kind) kind[o] = (c >> kTcKind) & 1;
                        if (diag) diag[o] = (c >> kTcDiag) & 1;
                        if (w) w[o] = t.w[o];
                    }
                }
            }
        }
    for (uint8_t s : seen)
        if (!s) return fail(EPHC_ESTATE, "internal: entry not covered by any slice");
    for (uint8_t s : tile_seen)
        if (!s) return fail(EPHC_ESTATE, "internal: tile not assigned to a CTA");
    // the finish kernel reaches every row of every slot exactly once through the fine-block lists
    {
        std::vector<uint8_t> cover((size_t)t.part_rows, 0);
        for (int32_t b = 0; b < t.nblk; ++b)
            for (int32_t i = t.blk_ent_ptr[b]; i < t.blk_ent_ptr[b + 1]; ++i)
                for (int32_t r = 0; r < t.blk_row0[b + 1] - t.blk_row0[b]; ++r) {
                    const int64_t o = t.blk_ent_off[i] + r;
                    if (o < 0 || o >= t.part_rows || cover[o]++) return fail(EPHC_ESTATE, "internal: slot row listed twice");
                }
        for (uint8_t cv : cover)
            if (!cv) return fail(EPHC_ESTATE, "internal: slot row not listed for the finish kernel");
    }
    return EPHC_OK;
}

// variant used by ephc_collision / ephc_rt_step (see auto_coll_variant), and by ephc_transport_setup / ephc_transport_iter
static inline int coll_variant(const ephc_handle *h) {
    if (h->variant >= 0) return h->variant;
    const int av = auto_coll_variant(h);
    if (av == 0) return 0;
    if (av == 3 && h->res_ok) return 3;
    return h->stream_ok ? 2 : (h->res_ok ? 3 : (h->tile_ok ? 1 : 0));
}
static inline int tr_variant(const ephc_handle *h) { return (h->variant < 0 || h->variant >= 2) ? 0 : h->variant; }
// RK stages of the paper-layout variant run on the library's own choice (variant 4 covers ephc_collision only)
static inline int rt_variant(const ephc_handle *h) {
    if (h->variant != 4) return coll_variant(h);
    const int av = auto_coll_variant(h);
    return (av == 3 && h->res_ok) ? 3 : ((av >= 2 && h->stream_ok) ? 2 : 0);
}

extern "C" int ephc_export_stream(const ephc_handle *h, int32_t *a, int32_t *b, int32_t *iq, int32_t *nu,
                                  int32_t *kind, double *w) {
    if (!h) return fail(EPHC_EINVAL, "null handle");
    if (!h->host_only) return fail(EPHC_ESTATE, "ephc_export_stream needs a handle built with EPHC_HOST_ONLY");
    if (!h->stream_ok) return fail(EPHC_ESTATE, "stream store not available for this problem: " + h->stream_why);
    const StreamHost &t = h->shost;
    const int nnu = h->d.nnu;
    const int64_t nent = (int64_t)t.w.size();
    std::vector<uint8_t> seen((size_t)nent, 0), tile_seen(t.tiles.size(), 0);
    if (t.order.size() != t.tiles.size()) return fail(EPHC_ESTATE, "internal: tile order does not list every tile");
    std::vector<uint8_t> used;
    for (int32_t it : t.order) {
        if (it < 0 || it >= (int32_t)t.tiles.size() || tile_seen[it]++) return fail(EPHC_ESTATE, "internal: bad tile order");
        const StreamTile &th = t.tiles[it];
        const bool dg = (th.flags & 4) != 0;
        if ((th.flags & 3) != 3 || th.a_slot < 0 || (dg != (th.b_slot < 0)) || th.a_rows > t.Ra || th.b_rows > t.Rb ||
            th.b_rows > kStreamRbMax || (dg && (th.b_row0 != th.a_row0 || th.b_rows != th.a_rows)) ||
            (!dg && th.b_row0 < th.a_row0 + th.a_rows) || t.slot_row0[th.a_slot] != th.a_row0 ||
            t.slot_rows[th.a_slot] != th.a_rows ||
            (!dg && (t.slot_row0[th.b_slot] != th.b_row0 || t.slot_rows[th.b_slot] != th.b_rows)))
            return fail(EPHC_ESTATE, "internal: bad stream tile");
        for (int32_t ci = th.c0; ci < th.c0 + th.nc; ++ci) {
            const StreamChunk &ch = t.chunks[ci];
            if (ch.ne < 1 || ch.ne > kStreamChunk || ch.nq * nnu > kStreamNSlots || ch.nar < 1 || ch.nar > 256 ||
                ch.nbr < 1 || ch.e0 < 0 || ch.e0 + ch.ne > nent)
                return fail(EPHC_ESTATE, "internal: chunk outside its limits");
            // k-row tasks: contiguous runs that cover the chunk; every entry of a run has the run's row
            if (t.arow_start[ch.ar0] != 0 || t.arow_start[ch.ar0 + ch.nar] != ch.ne)
                return fail(EPHC_ESTATE, "internal: k-row tasks do not cover the chunk");
            for (int32_t r = 0; r < ch.nar; ++r) {
                const int s0 = t.arow_start[ch.ar0 + r], s1 = t.arow_start[ch.ar0 + r + 1];
                if (s0 >= s1 || (r > 0 && t.arow_id[ch.ar0 + r] <= t.arow_id[ch.ar0 + r - 1]))
                    return fail(EPHC_ESTATE, "internal: k-row tasks out of order");
                for (int i = s0; i < s1; ++i)
                    if ((int32_t)(t.code[ch.e0 + i] & 255u) + ch.a0 != (int32_t)t.arow_id[ch.ar0 + r])
                        return fail(EPHC_ESTATE, "internal: entry outside its k-row task");
            }
            // k'-row tasks through the permutation
            const uint16_t *pm = t.perm.data() + 4 * (int64_t)ch.pad0;
            used.assign((size_t)ch.ne, 0);
            if (t.brow_start[ch.br0] != 0 || t.brow_start[ch.br0 + ch.nbr] != ch.ne)
                return fail(EPHC_ESTATE, "internal: k'-row tasks do not cover the chunk");
            for (int32_t r = 0; r < ch.nbr; ++r) {
                const int s0 = t.brow_start[ch.br0 + r], s1 = t.brow_start[ch.br0 + r + 1];
                if (s0 >= s1 || (r > 0 && t.brow_id[ch.br0 + r] <= t.brow_id[ch.br0 + r - 1]))
                    return fail(EPHC_ESTATE, "internal: k'-row tasks out of order");
                for (int i = s0; i < s1; ++i) {
                    const int e = pm[i];
                    if (e >= ch.ne || used[e]++) return fail(EPHC_ESTATE, "internal: not a permutation");
                    if ((int32_t)((t.code[ch.e0 + e] >> 8) & 2047u) != (int32_t)t.brow_id[ch.br0 + r])
                        return fail(EPHC_ESTATE, "internal: entry outside its k'-row task");
                }
            }
            for (int32_t i = 0; i < ch.ne; ++i) {
                const int64_t o = ch.e0 + i;
                if (seen[o]++) return fail(EPHC_ESTATE, "internal: entry in two chunks");
                const uint32_t c = t.code[o];
                const int32_t ar = th.a_row0 + ch.a0 + (int32_t)(c & 255u), br = th.b_row0 + (int32_t)((c >> 8) & 2047u);
                const int32_t slot = (int32_t)((c >> 19) & 4095u);
                if (ar >= th.a_row0 + th.a_rows || br >= th.b_row0 + th.b_rows || slot / nnu >= ch.nq)
                    return fail(EPHC_ESTATE, "internal: entry code out of range");
                if (a) a[o] = t.row_state[ar];
                if (b) b[o] = t.row_state[br];
                if (iq) iq[o] = (int32_t)t.iq[ch.q0 + slot / nnu];
                if (nu) nu[o] = slot % nnu;
                if (kind) kind[o] = (int32_t)(c >> 31);
                if (w) w[o] = t.w[o];
            }
        }
    }
    for (uint8_t sflag : seen)
        if (!sflag) return fail(EPHC_ESTATE, "internal: entry not covered by any chunk");
    {
        std::vector<uint8_t> cover((size_t)t.part_rows, 0);
        for (int32_t bl = 0; bl < t.nblk; ++bl)
            for (int32_t i = t.blk_ent_ptr[bl]; i < t.blk_ent_ptr[bl + 1]; ++i)
                for (int32_t r = 0; r < t.blk_row0[bl + 1] - t.blk_row0[bl]; ++r) {
                    const int64_t o = t.blk_ent_off[i] + r;
                    if (o < 0 || o >= t.part_rows || cover[o]++) return fail(EPHC_ESTATE, "internal: slot row listed twice");
                }
        for (uint8_t cv : cover)
            if (!cv) return fail(EPHC_ESTATE, "internal: slot row not listed for the finish kernel");
    }
    return EPHC_OK;
}

extern "C" int64_t ephc_stream_entries(const ephc_handle *h) { return h ? h->s_entries : 0; }

extern "C" int ephc_export_rows(const ephc_handle *h, int32_t *dest, int32_t *partner, int64_t *gather_pos) {
    if (!h) return fail(EPHC_EINVAL, "null handle");
    if (!h->host_only) return fail(EPHC_ESTATE, "ephc_export_rows needs a handle built with EPHC_HOST_ONLY");
    if (!h->rows_ok) return fail(EPHC_ESTATE, "row store not available (EPHC_NO_ROWS or shared-memory budget)");
    const RowHost &r = h->rowhost;
    const int64_t nent = (int64_t)r.idx.size();
    if (nent != h->g_entries || (int64_t)r.perm.size() != nent) return fail(EPHC_ESTATE, "internal: row store size");
    std::vector<uint8_t> seen((size_t)nent, 0), pos_seen((size_t)nent, 0);
    std::vector<int32_t> row_tiles;
    int32_t next_row = 0, next_tile = 0;
    for (size_t is = 0; is < r.strips.size(); ++is) {
        const RowStrip &st = r.strips[is];
        // strips partition the destination rows in order; their tiles are consecutive
        if (st.row0 != next_row || st.nrows < 0 || st.nrows > r.Ra || st.t0 != next_tile || st.t1 < st.t0)
            return fail(EPHC_ESTATE, "internal: row strips do not partition the rows");
        next_row = st.row0 + st.nrows;
        next_tile = st.t1;
        int32_t last_col0 = -1;
        for (int32_t it = st.t0; it < st.t1; ++it) {
            const RowTile &tl = r.tiles[it];
            const bool sparse = !r.cols.empty();
            if (tl.nseg < 1 || tl.col0 <= last_col0 || tl.ncols < 1 || tl.ncols > r.Rb ||
                (sparse ? tl.col0 < 0 || tl.col0 + (int64_t)tl.ncols > (int64_t)r.cols.size() : tl.col0 % r.Rb != 0 || tl.col0 + tl.ncols > r.nrows))
                return fail(EPHC_ESTATE, "internal: bad row tile");
            if (sparse)  // the tile's chunk of the strip's partner list: ascending rows
                for (int32_t j = 0; j < tl.ncols; ++j)
                    if (r.cols[tl.col0 + j] < 0 || r.cols[tl.col0 + j] >= r.nrows || (j > 0 && r.cols[tl.col0 + j] <= r.cols[tl.col0 + j - 1]))
                        return fail(EPHC_ESTATE, "internal: partner list of a row tile");
            last_col0 = tl.col0;
            row_tiles.assign((size_t)std::max(st.nrows, 1), 0);
            uint32_t last_len = 0xffffffffu;
            for (int32_t ig = tl.seg0; ig < tl.seg0 + tl.nseg; ++ig) {
                const RowSeg &sg = r.segs[ig];
                // one segment per destination row and tile, longest first
                if (sg.len < 1 || sg.len > last_len || (int32_t)sg.row >= st.nrows || row_tiles[sg.row]++)
                    return fail(EPHC_ESTATE, "internal: row segments must descend in length, one per row and tile");
                last_len = sg.len;
                for (uint32_t k = 0; k < sg.len; ++k) {
                    const int64_t o = st.e0 + sg.start + k;
                    if (o < 0 || o >= nent || seen[o]++) return fail(EPHC_ESTATE, "internal: row entry visited twice");
                    const int64_t gp = r.perm[o];
                    if (gp >= nent || pos_seen[gp]++ || r.idx[o] >= tl.ncols) return fail(EPHC_ESTATE, "internal: row entry out of range");
                    if (dest) dest[o] = r.row_state[st.row0 + (int32_t)sg.row];
                    if (partner) partner[o] = r.row_state[sparse ? r.cols[tl.col0 + r.idx[o]] : tl.col0 + r.idx[o]];
                    if (gather_pos) gather_pos[o] = gp;
                }
            }
        }
    }
    if (next_row != r.nrows || next_tile != (int32_t)r.tiles.size()) return fail(EPHC_ESTATE, "internal: rows or tiles left over");
    for (uint8_t v : seen)
        if (!v) return fail(EPHC_ESTATE, "internal: row entry not covered by any segment");
    return EPHC_OK;
}

extern "C" int ephc_export_rows_collapsed(const ephc_handle *h, int32_t *dest, int32_t *partner, int32_t *count) {
    if (!h) return fail(EPHC_EINVAL, "null handle");
    if (!h->host_only) return fail(EPHC_ESTATE, "ephc_export_rows_collapsed needs a handle built with EPHC_HOST_ONLY");
    if (!h->collapse_built) return fail(EPHC_ESTATE, "no mode-collapsed row store: build with EPHC_TRANSPORT_COLLAPSE");
    const RowHost &r = h->rowhost;
    const RowCollapsed &c = h->chost;
    const int64_t nc = (int64_t)c.idx.size(), nent = (int64_t)r.idx.size();
    if ((int64_t)c.first.size() != nc || (int64_t)c.count.size() != nc || c.strips.size() != r.strips.size() || c.tiles.size() != r.tiles.size() ||
        c.segs.size() != r.segs.size())
        return fail(EPHC_ESTATE, "internal: collapsed row store size");
    std::vector<uint8_t> covered((size_t)nent, 0);
    int64_t x = 0;
    for (size_t is = 0; is < c.strips.size(); ++is) {
        const RowStrip &st = c.strips[is], &rs = r.strips[is];
        if (st.row0 != rs.row0 || st.nrows != rs.nrows || st.t1 - st.t0 != rs.t1 - rs.t0 || st.e0 != x)
            return fail(EPHC_ESTATE, "internal: collapsed strips differ from the row store's");
        for (int32_t it = st.t0; it < st.t1; ++it) {
            const RowTile &tl = c.tiles[it], &rt = r.tiles[rs.t0 + (it - st.t0)];
            if (tl.col0 != rt.col0 || tl.ncols != rt.ncols || tl.nseg != rt.nseg) return fail(EPHC_ESTATE, "internal: collapsed tiles differ");
            uint32_t last_len = 0xffffffffu;
            for (int32_t ig = tl.seg0; ig < tl.seg0 + tl.nseg; ++ig) {
                const RowSeg &sg = c.segs[ig];
                if (sg.len < 1 || sg.len > last_len || (int32_t)sg.row >= st.nrows || st.e0 + sg.start != x)
                    return fail(EPHC_ESTATE, "internal: collapsed segments must be contiguous and descend in length");
                last_len = sg.len;
                int32_t last_idx = -1;
                for (uint32_t k = 0; k < sg.len; ++k, ++x) {
                    // one entry per partner of the segment, ascending; its terms are adjacent in the row store, have this
                    // partner, and belong to a segment of the same destination row in the same tile
                    if (x >= nc || (int32_t)c.idx[x] <= last_idx || c.idx[x] >= tl.ncols || c.count[x] < 1 ||
                        (int64_t)c.first[x] + c.count[x] > nent)
                        return fail(EPHC_ESTATE, "internal: collapsed entry out of range");
                    last_idx = c.idx[x];
                    for (uint32_t j = 0; j < c.count[x]; ++j) {
                        const int64_t o = (int64_t)c.first[x] + j;
                        if (r.idx[o] != c.idx[x] || covered[o]++) return fail(EPHC_ESTATE, "internal: collapsed entry sums a foreign term");
                    }
                    if (dest) dest[x] = r.row_state[st.row0 + (int32_t)sg.row];
                    if (partner) partner[x] = r.row_state[r.cols.empty() ? tl.col0 + c.idx[x] : r.cols[tl.col0 + c.idx[x]]];
                    if (count) count[x] = c.count[x];
                }
            }
        }
    }
    if (x != nc) return fail(EPHC_ESTATE, "internal: collapsed entries left over");
    for (uint8_t v : covered)
        if (!v) return fail(EPHC_ESTATE, "internal: ordered term not covered by any collapsed entry");
    return EPHC_OK;
}

extern "C" int64_t ephc_res_entries(const ephc_handle *h) { return (h && h->res_ok) ? h->x_entries : 0; }

extern "C" int ephc_export_res(const ephc_handle *h, int32_t *a, int32_t *b, int32_t *iq, int32_t *nu, int32_t *kind,
                               double *w) {
    if (!h) return fail(EPHC_EINVAL, "null handle");
    if (!h->host_only) return fail(EPHC_ESTATE, "ephc_export_res needs a handle built with EPHC_HOST_ONLY");
    if (!h->res_ok) return fail(EPHC_ESTATE, "resident-tile store not available for this problem: " + h->res_why);
    const ResHost &t = h->rhost;
    const int nnu = h->d.nnu;
    if ((int32_t)t.cta_ptr.size() != t.ncta + 1 || t.cta_ptr[0] != 0 || t.cta_ptr[t.ncta] != (int32_t)t.tiles.size())
        return fail(EPHC_ESTATE, "internal: schedule does not list every tile");
    if (res_smem_total(t.Ra, t.Rcap, t.smem_tile) > t.smem_cap || t.Ra % 2 || t.Rcap % 2 || t.RbMax % 2)
        return fail(EPHC_ESTATE, "internal: shared-memory plan");
    int64_t o = 0;
    std::vector<int32_t> owner, used;
    std::vector<uint8_t> row_out, row_in;
    size_t irun = 0;
    for (int32_t cta = 0; cta < t.ncta; ++cta) {
        for (int32_t it = t.cta_ptr[cta]; it < t.cta_ptr[cta + 1]; ++it) {
            const ResTile &D = t.tiles[it];
            // runs: consecutive tiles of one strip on one CTA, first / last flags, one slot for the strip
            if (D.flags & 1) {
                if (irun >= t.runs.size() || t.runs[irun].t0 != it || t.runs[irun].cta != cta) return fail(EPHC_ESTATE, "internal: run table");
            } else if (irun >= t.runs.size() || it <= t.runs[irun].t0 || it >= t.runs[irun].t0 + t.runs[irun].nt) {
                return fail(EPHC_ESTATE, "internal: tile outside its run");
            }
            const ResRun &run = t.runs[irun];
            if (((D.flags & 2) != 0) != (it == run.t0 + run.nt - 1) || run.a_row0 % t.Ra != 0 || run.a_rows < 1 || run.a_rows > t.Ra ||
                D.a_row0 != run.a_row0 || D.a_rows != run.a_rows || D.a_slot != run.a_slot || run.a_slot < 0 ||
                t.slot_row0[run.a_slot] != run.a_row0 || t.slot_rows[run.a_slot] != run.a_rows ||
                (it + 1 < (int32_t)t.tiles.size() ? D.nq_next != t.tiles[it + 1].nq : D.nq_next != 0))
                return fail(EPHC_ESTATE, "internal: bad run / tile header");
            if (D.flags & 2) ++irun;
            ResTile Dl = D;
            res_set_layout(Dl, t.nwarp);
            if (D.ncombo < 1 || D.ncombo > D.ne || D.o_sn_next != (it + 1 < (int32_t)t.tiles.size() ? res_o_sn(t.tiles[it + 1]) : 0u))
                return fail(EPHC_ESTATE, "internal: where the next tile's N rows go");
            const int32_t R = run.a_rows + D.b_rows;
            if (D.ne < 1 || std::memcmp(&Dl, &D, sizeof(D)) != 0 || (int64_t)D.a_off != t.slot_off[D.a_slot] ||
                (D.b_slot >= 0 && (int64_t)D.b_off != t.slot_off[D.b_slot]) || D.blob_off % 128 != 0 || D.blob_off + D.blob_bytes > (int64_t)t.blob.size() ||
                res_tile_smem(D, nnu) > t.smem_tile || R > t.Rcap || D.b_rows > t.RbMax || R > kResRowMax || D.nq * nnu > kResSlotMax ||
                D.ne_pad % 32 || D.ng_pad % 32 || D.ne_pad > kResXMax - 1 || D.ne_pad / 32 > 1023 || D.ng_pad / 32 > 1023 || D.ne > D.ne_pad ||
                D.ncombo > D.ng_pad || D.nslab1 < 1 || D.nslab2 < 1 ||
                (D.b_rows > 0) != (D.b_slot >= 0) || (D.b_rows > 0 && (D.b_row0 < run.a_row0 + run.a_rows || D.b_row0 % 2 || run.a_rows % 2)) ||
                (D.b_slot >= 0 && (t.slot_row0[D.b_slot] != D.b_row0 || t.slot_rows[D.b_slot] != D.b_rows)) ||
                D.q0 < 0 || D.q0 + D.nq > (int64_t)t.iqn.size())
                return fail(EPHC_ESTATE, "internal: bad resident tile");
            if (D.nq_next > 0 && std::memcmp(t.blob.data() + D.blob_off + D.o_nxt, t.iqn.data() + t.tiles[it + 1].q0, (size_t)D.nq_next * 4) != 0)
                return fail(EPHC_ESTATE, "internal: the image does not carry the next tile's iq list");
            const unsigned char *B = t.blob.data() + D.blob_off;
            const uint32_t *code = reinterpret_cast<const uint32_t *>(B);
            const uint16_t *perm = reinterpret_cast<const uint16_t *>(B + D.o_perm);
            const uint16_t *srow1 = reinterpret_cast<const uint16_t *>(B + D.o_srow1);
            const uint32_t *shdr1 = reinterpret_cast<const uint32_t *>(B + D.o_shdr1);
            const uint16_t *srow2 = reinterpret_cast<const uint16_t *>(B + D.o_srow2);
            const uint32_t *shdr2 = reinterpret_cast<const uint32_t *>(B + D.o_shdr2);
            const double *wv = reinterpret_cast<const double *>(B + D.o_w);
            const uint16_t *wptr = reinterpret_cast<const uint16_t *>(B + D.o_wptr);
            auto row_of = [&](int32_t loc) { return loc < run.a_rows ? run.a_row0 + loc : D.b_row0 + (loc - run.a_rows); };
            // Walks the slabs of one phase as the kernel does.  visit(row, position) is called for every position of a
            // lane that owns a row; checks: the warps' slab ranges tile [0, nslab), the slabs tile [0, npos) in order,
            // heights descend inside a warp, the lanes of a row are adjacent, in one slab only, and flagged.
            auto walk = [&](const uint16_t *srow, const uint32_t *shdr, const uint16_t *wp, int32_t nslab, int32_t npos,
                            std::vector<uint8_t> &row_seen, auto &&visit) -> bool {
                row_seen.assign((size_t)R, 0);
                int32_t next = 0;
                if (wp[0] != 0 || wp[t.nwarp] != nslab) return false;
                for (int32_t wi = 0; wi < t.nwarp; ++wi) {
                    if (wp[wi + 1] < wp[wi]) return false;
                    int32_t prevH = kResHMax + 1;
                    for (int32_t sl = wp[wi]; sl < wp[wi + 1]; ++sl) {
                        const uint32_t hd = shdr[sl];
                        const int32_t base = (int32_t)(hd & 1023u) * 32, H = (int32_t)((hd >> kResHdrHShift) & kResHdrHMask);
                        if (base != next || H > prevH || base + 32 * H > npos || (hd & ~(kResHdrMulti | 0x7ffffu))) return false;
                        prevH = H;
                        next = base + 32 * H;
                        bool multi = false;
                        for (int l = 0; l < 32; ++l) {
                            const uint16_t u = srow[32 * sl + l];
                            if (u == kResNoRow) continue;
                            if (u >= R) return false;
                            if (l > 0 && srow[32 * sl + l - 1] == u) {
                                multi = true;
                            } else if (row_seen[u]++) {
                                return false;
                            }
                            for (int32_t j = 0; j < H; ++j)
                                if (!visit(u, base + 32 * j + l, j, j + 1 == H)) return false;
                        }
                        if (multi && !(hd & kResHdrMulti)) return false;
                    }
                }
                return next == npos;
            };
            // phase 1: a lane's entries come in combos (same partner, closed by bit 0 of the code); owner[pos] = b row of the
            // term at a combo's last position (-2: inside a combo, -1: padding, w == 0); every a row is a row of the strip
            owner.assign((size_t)D.ne_pad, -1);
            used.assign((size_t)D.ne_pad, 0);
            int32_t real = 0, combos = 0, open_in = -1;
            const bool ok1 = walk(srow1, shdr1, wptr, D.nslab1, D.ne_pad, row_out, [&](int32_t u, int32_t pos, int32_t col, bool last_col) {
                if (col == 0) open_in = -1;
                if (used[pos]++ || u >= run.a_rows) return false;
                const uint32_t cd = code[pos];
                const int32_t in_loc = (int32_t)((cd & 0xffffu) >> 3), slot = (int32_t)(cd >> 19);
                if ((cd & 6u) || in_loc >= R || slot / nnu >= D.nq) return false;
                if (wv[pos] == 0.0) return cd == 0u && open_in < 0;  // padding (after the lane's last combo) reads N slot 0
                const int32_t ro = row_of(u), ri = row_of(in_loc);
                if (ro >= ri || (D.b_rows > 0 && in_loc < run.a_rows)) return false;
                if (open_in >= 0 && open_in != in_loc) return false;  // a combo has one partner
                if (cd & 1u) {
                    owner[pos] = in_loc;
                    open_in = -1;
                    ++combos;
                } else {
                    if (last_col) return false;  // a lane must not end inside a combo
                    owner[pos] = -2;
                    open_in = in_loc;
                }
                const int64_t x = o + real++;
                if (x >= t.nent) return false;
                if (a) a[x] = t.row_state[ro];
                if (b) b[x] = t.row_state[ri];
                if (iq) iq[x] = (int32_t)(t.iqn[D.q0 + slot / nnu] / (uint32_t)nnu);
                if (nu) nu[x] = slot % nnu;
                if (kind) kind[x] = wv[pos] > 0.0 ? 1 : 0;  // the sign carries the kind: +w emission, -w absorption
                if (w) w[x] = std::fabs(wv[pos]);
                return true;
            });
            if (!ok1 || real != D.ne || combos != D.ncombo || D.nslab1 < 1) return fail(EPHC_ESTATE, "internal: phase-1 slabs of a resident tile");
            for (int32_t pos = 0; pos < D.ne_pad; ++pos)  // positions of lanes without a row hold padding
                if (!used[pos] && (wv[pos] != 0.0 || code[pos] != 0u)) return fail(EPHC_ESTATE, "internal: weight in a lane without a row");
            // phase 2: every T value is added exactly once, to its b row; off the diagonal every B row stores a sum
            std::fill(used.begin(), used.end(), 0);
            int32_t gathered = 0;
            const bool ok2 = walk(srow2, shdr2, wptr + t.nwarp + 1, D.nslab2, D.ng_pad, row_in, [&](int32_t u, int32_t g, int32_t, bool) {
                const int32_t x = perm[g];
                if (x == D.ne_pad) return true;  // the zero
                if (x > D.ne_pad || owner[x] < 0 || owner[x] != u || used[x]++) return false;
                ++gathered;
                return true;
            });
            if (!ok2 || gathered != D.ncombo) return fail(EPHC_ESTATE, "internal: phase-2 slabs of a resident tile");
            for (int32_t r = run.a_rows; r < R; ++r)
                if (!row_in[r]) return fail(EPHC_ESTATE, "internal: a B row of a tile has no lane");
            o += D.ne;
        }
    }
    if (o != t.nent || irun != t.runs.size()) return fail(EPHC_ESTATE, "internal: resident-tile store does not hold every weight");
    {
        std::vector<uint8_t> cover((size_t)t.part_rows, 0);
        for (int32_t bl = 0; bl < t.nblk; ++bl)
            for (int32_t i = t.blk_ent_ptr[bl]; i < t.blk_ent_ptr[bl + 1]; ++i)
                for (int32_t r = 0; r < t.blk_row0[bl + 1] - t.blk_row0[bl]; ++r) {
                    const int64_t q = t.blk_ent_off[i] + r;
                    if (q < 0 || q >= t.part_rows || cover[q]++) return fail(EPHC_ESTATE, "internal: slot row listed twice");
                }
        for (uint8_t cv : cover)
            if (!cv) return fail(EPHC_ESTATE, "internal: slot row not listed for the finish kernel");
    }
    return EPHC_OK;
}


extern "C" int ephc_set_variant(ephc_handle *h, int variant) {
    if (!h) return fail(EPHC_EINVAL, "null handle");
    if (variant < -1 || variant > 4)
        return fail(EPHC_EINVAL, "variant must be -1 (automatic), 0 (gather), 1 (tiles), 2 (stream), 3 (resident tiles) or 4 (paper layout)");
    if (h->ranged && variant > 0)
        return fail(EPHC_ESTATE, "a k-sharded handle runs on the destination-sorted stores only (variant 0)");
    // a store that the automatic choice did not need is built (and uploaded) now: this call may allocate and copy
    if (!h->host_only && variant >= 1) CUDA_TRY(cudaSetDevice(h->device));
    int rc = EPHC_OK;
    if (variant == 3) rc = make_res_store(h);
    if (variant == 2) rc = make_stream_store(h);
    if (variant == 1) rc = make_tile_store(h);
    if (variant == 4) rc = make_paper_store(h);
    if (rc != EPHC_OK) return rc;
    if (variant == 3 && !h->res_ok)
        return fail(EPHC_ESTATE, "resident-tile store not available for this problem: " + h->res_why);
    if (variant == 2 && !h->stream_ok)
        return fail(EPHC_ESTATE, "stream store not available for this problem: " + h->stream_why);
    if (variant == 1 && !h->tile_ok)
        return fail(EPHC_ESTATE, "tile store not available for this problem: " + h->thost.why);
    h->variant = variant;
    if (!h->host_only && (coll_variant(h) == 0 || rt_variant(h) == 0)) return make_gather_device(h);
    return EPHC_OK;
}

extern "C" int ephc_get_variant(const ephc_handle *h) { return h ? coll_variant(h) : EPHC_EINVAL; }
extern "C" int ephc_get_transport_variant(const ephc_handle *h) { return h ? tr_variant(h) : EPHC_EINVAL; }

extern "C" int64_t ephc_launch_count(const ephc_handle *h) { return h ? h->launches : 0; }

// ------------------------------------------------------------------------------------------------------------
// The dynamic shared-memory limit belongs to the kernel, not to a handle: it is raised once per device to a size that
// covers every geometry the builders can produce (they keep each kernel's request below these caps).
static int set_kernel_attributes(int device) {
    static bool done[64] = {false};
    if (device >= 0 && device < 64 && done[device]) return EPHC_OK;
    const int big = 220 * 1024;
    CUDA_TRY(cudaFuncSetAttribute(gather_kernel<kCollision>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                  (int)gather_smem_bytes(kCollision)));
    CUDA_TRY(cudaFuncSetAttribute(gather_kernel<kRkStage>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                  (int)gather_smem_bytes(kRkStage)));
    CUDA_TRY(cudaFuncSetAttribute(gather_kernel<kTransportSetup>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                  (int)gather_smem_bytes(kTransportSetup)));
    CUDA_TRY(cudaFuncSetAttribute(gather_kernel<kTransportIter>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                  (int)gather_smem_bytes(kTransportIter)));
    CUDA_TRY(cudaFuncSetAttribute(stream_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, big));
    CUDA_TRY(cudaFuncSetAttribute(res_kernel<256, 2>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kResModes[0].smem));
    CUDA_TRY(cudaFuncSetAttribute(res_kernel<512, 1>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kResModes[1].smem));
    CUDA_TRY(cudaFuncSetAttribute(res_kernel<256, 1>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kResModes[2].smem));
    CUDA_TRY(cudaFuncSetAttribute(res_kernel<384, 1>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kResModes[3].smem));
    CUDA_TRY(cudaFuncSetAttribute(res_kernel<128, 4>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kResModes[4].smem));
    CUDA_TRY(cudaFuncSetAttribute(res_kernel<512, 2>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kResModes[5].smem));
    CUDA_TRY(cudaFuncSetAttribute(res_kernel<768, 1>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kResModes[6].smem));
    CUDA_TRY(cudaFuncSetAttribute(row_iter_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, big));
    CUDA_TRY(cudaFuncSetAttribute(row_setup_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, big));
#define EPHC_TILE_ATTR(NB_)                                                                                          \
    CUDA_TRY(cudaFuncSetAttribute(tile_kernel<kTCollision, NB_>, cudaFuncAttributeMaxDynamicSharedMemorySize, big)); \
    CUDA_TRY(cudaFuncSetAttribute(tile_kernel<kTSetup, NB_>, cudaFuncAttributeMaxDynamicSharedMemorySize, big));     \
    CUDA_TRY(cudaFuncSetAttribute(tile_kernel<kTIter, NB_>, cudaFuncAttributeMaxDynamicSharedMemorySize, big));
    EPHC_TILE_ATTR(1)
    EPHC_TILE_ATTR(2)
    EPHC_TILE_ATTR(4)
#undef EPHC_TILE_ATTR
    if (device >= 0 && device < 64) done[device] = true;
    return EPHC_OK;
}

static int need_device(ephc_handle *h) {
    if (!h) return fail(EPHC_EINVAL, "null handle");
    if (h->host_only) return fail(EPHC_ESTATE, "handle was built with EPHC_HOST_ONLY: no device store");
    int cur = -1;
    if (cudaGetDevice(&cur) != cudaSuccess || cur != h->device) CUDA_TRY(cudaSetDevice(h->device));
    return set_kernel_attributes(h->device);
}

static TileParams tile_params(const ephc_handle *h) {
    TileParams P;
    std::memset(&P, 0, sizeof(P));
    P.w = h->dt_w;
    P.code = h->dt_code;
    P.prec = h->dt_prec;
    P.npiece = h->t_pieces;
    P.slices = h->dt_slices;
    P.tiles = h->dt_tiles;
    P.ctas = h->dt_ctas;
    P.row_state = h->dt_row_state;
    P.slot_off = h->dt_slot_off;
    P.Ra = h->t_Ra;
    P.Rb = h->t_Rb;
    P.cta_group = 1;
    P.ncta = h->t_ncta;
    P.nnu = h->d.nnu;
    P.ns = h->d.ns;
    P.part = h->dt_part;
    P.Wf = h->dt_Wf;
    P.Wr = h->dt_Wr;
    return P;
}

static FinishParams finish_params(const ephc_handle *h) {
    FinishParams P;
    std::memset(&P, 0, sizeof(P));
    P.state_row = h->dt_state_row;
    P.state_blk = h->dt_state_blk;
    P.blk_row0 = h->dt_blk_row0;
    P.blk_ent_ptr = h->dt_blk_ent_ptr;
    P.blk_ent_off = h->dt_blk_ent_off;
    P.part = h->dt_part;
    P.ns = h->d.ns;
    return P;
}

static inline unsigned finish_grid(const ephc_handle *h) { return (unsigned)((h->d.ns + 255) / 256); }

template <int MODE>
static int launch_tile(ephc_handle *h, TileParams P, cudaStream_t s) {
    if (h->t_ntile > 0) {
        const int nb = h->d.nb;
        const size_t sm = tile_smem_bytes(MODE, h->t_Ra, h->t_Rb);
        const int threads = (MODE == kTIter) ? kTileThreadsIter : kTileThreads;
        P.cta_group = (MODE == kTIter) ? 2 : 1;
        const unsigned grid = (unsigned)((h->t_ncta + P.cta_group - 1) / P.cta_group);
        if (nb <= 1)
            tile_kernel<MODE, 1><<<grid, threads, sm, s>>>(P);
        else if (nb <= 2)
            tile_kernel<MODE, 2><<<grid, threads, sm, s>>>(P);
        else
            tile_kernel<MODE, 4><<<grid, threads, sm, s>>>(P);
        h->launches++;
    }
    CUDA_TRY(cudaGetLastError());
    return EPHC_OK;
}

template <int FMODE>
static int launch_finish(ephc_handle *h, const FinishParams &P, cudaStream_t s) {
    finish_kernel<FMODE><<<finish_grid(h), 256, 0, s>>>(P);
    h->launches++;
    CUDA_TRY(cudaGetLastError());
    return EPHC_OK;
}

static GatherParams base_params(const ephc_handle *h) {
    GatherParams P;
    std::memset(&P, 0, sizeof(P));
    P.code = h->d_code;
    P.w = h->d_w;
    P.hp_k = h->d_hp_k;
    P.hp_q = h->d_hp_q;
    P.tasks = h->d_tasks;
    P.rounds = h->d_rounds;
    P.wus = h->d_wus;
    P.nb = h->d.nb;
    P.nnu = h->d.nnu;
    P.ns = h->d.ns;
    P.gW = h->d_gW;
    return P;
}

template <int MODE>
static int launch_gather(ephc_handle *h, const GatherParams &P, cudaStream_t s) {
    if (h->n_wu > 0) {
        gather_kernel<MODE><<<h->n_wu, kThreads, gather_smem_bytes(MODE), s>>>(P);
        h->launches++;
    }
    CUDA_TRY(cudaGetLastError());
    return EPHC_OK;
}

template <class T>
static int ensure(T **p, size_t n) {
    if (*p) return EPHC_OK;
    cudaError_t e = cudaMalloc((void **)p, n > 0 ? n : 8);
    if (e != cudaSuccess) return fail(e == cudaErrorMemoryAllocation ? EPHC_ENOMEM : EPHC_ECUDA,
                                      std::string("cudaMalloc: ") + cudaGetErrorString(e));
    return EPHC_OK;
}

static int launch_stream(ephc_handle *h, const double *f, const double *N, cudaStream_t s) {
    if (h->s_ntile > 0) {
        StreamParams P;
        std::memset(&P, 0, sizeof(P));
        P.w = h->ds_w;
        P.code = h->ds_code;
        P.perm = h->ds_perm;
        P.arow_id = h->ds_aid;
        P.arow_start = h->ds_ast;
        P.brow_id = h->ds_bid;
        P.brow_start = h->ds_bst;
        P.iq = h->ds_iq;
        P.chunks = h->ds_chunks;
        P.tiles = h->ds_tiles;
        P.order = h->ds_order;
        P.counter = h->ds_counter;
        P.ntile = h->s_ntile;
        P.row_state = h->ds_row_state;
        P.slot_off = h->ds_slot_off;
        P.Ra = h->s_Ra;
        P.Rb = h->s_Rb;
        P.nnu = h->d.nnu;
        P.ncta = h->s_ncta;
        P.ns = h->d.ns;
        P.f = f;
        P.N = N;
        P.part = h->ds_part;
        stream_kernel<<<(unsigned)h->s_ncta, kStreamThreads, stream_smem_bytes(h->s_Ra, h->s_Rb), s>>>(P);
        h->launches++;
    }
    CUDA_TRY(cudaGetLastError());
    return EPHC_OK;
}

// fc_ready: the compact copy of f (dx_fc) was already written by the finish kernel of the previous RK stage
static int launch_res(ephc_handle *h, const double *f, const double *N, cudaStream_t s, bool fc_ready = false, long long *tile_cycles = nullptr) {
    if (h->x_ntile > 0) {
        if (!fc_ready) {
            res_compact_kernel<<<(unsigned)((h->x_nrows + 255) / 256), 256, 0, s>>>(f, h->dx_row_state, h->dx_fc, h->x_nrows);
            h->launches++;
        }
        ResParams P;
        std::memset(&P, 0, sizeof(P));
        P.blob = h->dx_blob;
        P.iqn = h->dx_iqn;
        P.tiles = h->dx_tiles;
        P.cta_ptr = h->dx_cta_ptr;
        P.slot_off = h->dx_slot_off;
        P.Ra = h->x_Ra;
        P.Rcap = h->x_Rcap;
        P.RbMax = h->x_RbMax;
        P.nnu = h->d.nnu;
        P.buf_bytes = (uint32_t)res_buf_bytes(h->x_Rcap, h->x_smem_tile);
        P.fixed_bytes = (uint32_t)res_fixed_bytes(h->x_Ra);
        P.gran16 = (h->d.nnu % 2 == 0) && ((reinterpret_cast<uintptr_t>(N) & 15) == 0);
        P.gran = P.gran16 ? h->d.nnu / 2 : h->d.nnu;
        P.gran_magic = P.gran > 1 ? (uint32_t)((0x100000000ULL + (uint64_t)P.gran - 1) / (uint64_t)P.gran) : 0u;
        P.fc = h->dx_fc;
        P.N = N;
        P.part = h->dx_part;
        P.tile_cycles = tile_cycles;
#ifdef EPHC_RES_TIMING
        static long long *dbg = nullptr;
        const size_t ndbg = (size_t)h->x_ncta * (kResModes[h->x_mode].nl / 32 + 1) * 8;
        if (!dbg) cudaMalloc((void **)&dbg, ndbg * 8);
        cudaMemset(dbg, 0, ndbg * 8);
        P.dbg = dbg;
#endif
        const size_t smem = (size_t)res_smem_total(h->x_Ra, h->x_Rcap, h->x_smem_tile);
        const unsigned grid = (unsigned)h->x_ncta;
        switch (h->x_mode) {
            case 0: res_kernel<256, 2><<<grid, 256 + kResProducerThreads, smem, s>>>(P); break;
            case 1: res_kernel<512, 1><<<grid, 512 + kResProducerThreads, smem, s>>>(P); break;
            case 2: res_kernel<256, 1><<<grid, 256 + kResProducerThreads, smem, s>>>(P); break;
            case 3: res_kernel<384, 1><<<grid, 384 + kResProducerThreads, smem, s>>>(P); break;
            case 4: res_kernel<128, 4><<<grid, 128 + kResProducerThreads, smem, s>>>(P); break;
            case 5: res_kernel<512, 2><<<grid, 512 + kResProducerThreads, smem, s>>>(P); break;
            default: res_kernel<768, 1><<<grid, 768 + kResProducerThreads, smem, s>>>(P); break;
        }
        h->launches++;
#ifdef EPHC_RES_TIMING
        if (std::getenv("EPHC_RES_TIMING_PRINT")) {
            std::vector<long long> hd(ndbg);
            cudaMemcpy(hd.data(), dbg, ndbg * 8, cudaMemcpyDeviceToHost);
            const char *nm[8] = {"loop", "wait full", "phase 1", "barrier", "phase 2", "barrier", "copy-out", "release"};
            const int nw = kResModes[h->x_mode].nl / 32;
            for (int k = 0; k < 8; ++k) {
                double mean = 0, w0 = 0, wl = 0, mx = 0;
                for (int c = 0; c < h->x_ncta; ++c)
                    for (int w = 0; w < nw; ++w) {
                        const double v = (double)hd[((size_t)c * (nw + 1) + w) * 8 + k];
                        mean += v;
                        mx = std::max(mx, v);
                        if (w == 0) w0 += v;
                        if (w == nw - 1) wl += v;
                    }
                std::fprintf(stderr, "res timing %-14s mean %9.0f  warp0 %9.0f  last warp %9.0f  max %9.0f cycles per CTA\n", nm[k],
                             mean / (h->x_ncta * nw), w0 / h->x_ncta, wl / h->x_ncta, mx);
            }
            {   // per CTA: cycles of warp 0 over all sections
                double mn = 1e30, mx = 0, sum = 0;
                int imx = 0;
                for (int c = 0; c < h->x_ncta; ++c) {
                    double tt = 0;
                    for (int k = 0; k < 8; ++k) tt += (double)hd[((size_t)c * (nw + 1)) * 8 + k];
                    if (tt > mx) mx = tt, imx = c;
                    mn = std::min(mn, tt);
                    sum += tt;
                }
                std::fprintf(stderr, "res timing per CTA total: min %.0f mean %.0f max %.0f (CTA %d) cycles\n", mn, sum / h->x_ncta, mx, imx);
                std::fprintf(stderr, "res timing slowest CTA %d sections:", imx);
                for (int k = 0; k < 8; ++k) std::fprintf(stderr, " %lld", hd[((size_t)imx * (nw + 1)) * 8 + k]);
                std::fprintf(stderr, "\n");
            }
            const char *pn[6] = {"loop", "wait empty", "dir + bulk", "wait prev", "N staging", "until full"};
            for (int k = 0; k < 6; ++k) {
                double mean = 0;
                for (int c = 0; c < h->x_ncta; ++c) mean += (double)hd[((size_t)c * (nw + 1) + nw) * 8 + k];
                std::fprintf(stderr, "res producer %-12s mean %9.0f cycles per CTA (%d tiles)\n", pn[k], mean / h->x_ncta, h->x_ntile);
            }
        }
#endif
    }
    CUDA_TRY(cudaGetLastError());
    return EPHC_OK;
}

static FinishParams finish_params_res(const ephc_handle *h) {
    FinishParams P;
    std::memset(&P, 0, sizeof(P));
    P.state_row = h->dx_state_row;
    P.state_blk = h->dx_state_blk;
    P.blk_row0 = h->dx_blk_row0;
    P.blk_ent_ptr = h->dx_blk_ent_ptr;
    P.blk_ent_off = h->dx_blk_ent_off;
    P.part = h->dx_part;
    P.ns = h->d.ns;
    return P;
}

static FinishParams finish_params_stream(const ephc_handle *h) {
    FinishParams P;
    std::memset(&P, 0, sizeof(P));
    P.state_row = h->ds_state_row;
    P.state_blk = h->ds_state_blk;
    P.blk_row0 = h->ds_blk_row0;
    P.blk_ent_ptr = h->ds_blk_ent_ptr;
    P.blk_ent_off = h->ds_blk_ent_off;
    P.part = h->ds_part;
    P.ns = h->d.ns;
    P.reset = h->ds_counter;
    return P;
}

extern "C" int ephc_collision(ephc_handle *h, const double *f_dev, const double *N_dev, double *I_dev,
                              void *stream) {
    int rc = need_device(h);
    if (rc) return rc;
    if (!f_dev || !N_dev || !I_dev) return fail(EPHC_EINVAL, "null device pointer");
    if (coll_variant(h) == 4) {  // the paper's two steps; states without a target get I = 0
        cudaStream_t s = (cudaStream_t)stream;
        CUDA_TRY(cudaMemsetAsync(I_dev, 0, (size_t)h->d.ns * 8, s));
        if (h->p_rows > 0) {
            paper_step2_kernel<<<(unsigned)((h->p_rows + 255) / 256), 256, 0, s>>>(h->dp_ch, h->dp_ik, h->dp_ikq, h->dp_iq, f_dev, N_dev,
                                                                                   h->dp_sc_col, h->p_rows, h->d.nb, h->d.nnu);
            paper_step3_kernel<<<(unsigned)((h->p_targets + 255) / 256), 256, 0, s>>>(h->dp_targets, h->dp_src, h->dp_sc_col, I_dev,
                                                                                      h->p_targets);
            h->launches += 2;
        }
        CUDA_TRY(cudaGetLastError());
        return EPHC_OK;
    }
    if (coll_variant(h) == 3) {
        if ((rc = launch_res(h, f_dev, N_dev, (cudaStream_t)stream))) return rc;
        FinishParams Fp = finish_params_res(h);
        Fp.out = I_dev;
        return launch_finish<kFCollision>(h, Fp, (cudaStream_t)stream);
    }
    if (coll_variant(h) == 2) {
        if ((rc = launch_stream(h, f_dev, N_dev, (cudaStream_t)stream))) return rc;
        FinishParams Fp = finish_params_stream(h);
        Fp.out = I_dev;
        return launch_finish<kFCollision>(h, Fp, (cudaStream_t)stream);
    }
    if (coll_variant(h) == 1) {
        TileParams T = tile_params(h);
        T.f = f_dev;
        T.N = N_dev;
        if ((rc = launch_tile<kTCollision>(h, T, (cudaStream_t)stream))) return rc;
        FinishParams Fp = finish_params(h);
        Fp.out = I_dev;
        return launch_finish<kFCollision>(h, Fp, (cudaStream_t)stream);
    }
    GatherParams P = base_params(h);
    P.f = f_dev;
    P.N = N_dev;
    P.out = I_dev;
    return launch_gather<kCollision>(h, P, (cudaStream_t)stream);
}

static RowParams row_params(const ephc_handle *h) {
    RowParams R;
    std::memset(&R, 0, sizeof(R));
    R.W = h->dr_W;
    R.wst = h->dr_wst;
    R.meta = h->dr_meta;
    R.idx = h->dr_idx;
    R.segs = h->dr_segs;
    R.tiles = h->dr_tiles;
    R.strips = h->dr_strips;
    R.row_state = h->dr_row_state;
    R.state_row = h->dr_state_row;
    R.cols = h->dr_cols;
    R.Rb = h->r_Rb;
    R.Ra = h->r_Ra;
    R.nstrip = h->r_nstrip;
    R.ns = h->d.ns;
    R.Fc = h->dr_Fc;
    if (h->collapse_on) {  // the mode-collapsed specialisation: same walk, one entry per state pair
        R.W = h->dc_W;
        R.idx = h->dc_idx;
        R.segs = h->dc_segs;
        R.tiles = h->dc_tiles;
        R.strips = h->dc_strips;
    }
    return R;
}

extern "C" int ephc_transport_collapse(ephc_handle *h, void *stream) {
    int rc = need_device(h);
    if (rc) return rc;
    if (!h->collapse_built)
        return fail(EPHC_ESTATE, "no mode-collapsed row store: build the handle with EPHC_TRANSPORT_COLLAPSE (row store required)");
    if (!h->transport_ready || h->transport_variant != 0 || tr_variant(h) != 0)
        return fail(EPHC_ESTATE, "call ephc_transport_setup (automatic or gather variant) before ephc_transport_collapse");
    if (h->c_nent > 0) {
        row_collapse_kernel<<<(unsigned)((h->c_nent + 255) / 256), 256, 0, (cudaStream_t)stream>>>(h->dr_W, h->dc_first, h->dc_count,
                                                                                               h->dc_W, h->c_nent);
        h->launches++;
        CUDA_TRY(cudaGetLastError());
    }
    h->collapse_ready = true;
    h->collapse_on = true;
    return EPHC_OK;
}
extern "C" int ephc_set_transport_collapsed(ephc_handle *h, int on) {
    if (!h) return fail(EPHC_EINVAL, "null handle");
    if (on && !h->collapse_ready)
        return fail(EPHC_ESTATE, "no collapsed weights: call ephc_transport_collapse after ephc_transport_setup");
    h->collapse_on = on != 0;
    return EPHC_OK;
}
extern "C" int64_t ephc_collapsed_entries(const ephc_handle *h) { return (h && h->collapse_built) ? h->c_nent : 0; }

extern "C" int ephc_transport_setup(ephc_handle *h, const double *f0_dev, const double *N_dev, double *Gamma_dev,
                                    void *stream) {
    int rc = need_device(h);
    if (rc) return rc;
    if (!f0_dev || !N_dev || !Gamma_dev) return fail(EPHC_EINVAL, "null device pointer");
    if (tr_variant(h) == 1) {
        TileParams T = tile_params(h);
        T.f = f0_dev;
        T.N = N_dev;
        if ((rc = launch_tile<kTSetup>(h, T, (cudaStream_t)stream))) return rc;
        FinishParams Fp = finish_params(h);
        Fp.out = Gamma_dev;
        rc = launch_finish<kFSetup>(h, Fp, (cudaStream_t)stream);
        if (rc == EPHC_OK) {
            h->transport_ready = true;
            h->transport_variant = 1;
        }
        return rc;
    }
    if (h->rows_ok) {
        // the row store holds every ordered term with its weight, N index and kind: weights and Gamma in one pass, written
        // in the order row_iter_kernel streams them
        const cudaStream_t s = (cudaStream_t)stream;
        if (h->r_nrows > 0) {
            row_compact1_kernel<<<(unsigned)((h->r_nrows + 255) / 256), 256, 0, s>>>(f0_dev, h->dr_row_state, h->dr_Fc, h->r_nrows);
            h->launches++;
        }
        const bool was_on = h->collapse_on;
        h->collapse_on = false;  // the weights are computed per ordered term on the full row store
        RowParams R = row_params(h);
        h->collapse_on = was_on;
        R.N = N_dev;
        R.out = Gamma_dev;
        row_setup_kernel<<<(unsigned)std::max(h->r_nstrip, 1), kRowThreads, row_smem_bytes(h->r_Rb, h->r_Ra), s>>>(R);
        h->launches++;
        h->collapse_ready = false;  // new weights: ephc_transport_collapse sums them again
        h->collapse_on = false;
        CUDA_TRY(cudaGetLastError());
    } else {
        GatherParams P = base_params(h);
        P.f = f0_dev;
        P.N = N_dev;
        P.out = Gamma_dev;
        rc = launch_gather<kTransportSetup>(h, P, (cudaStream_t)stream);
    }
    if (rc == EPHC_OK) {
        h->transport_ready = true;
        h->transport_variant = 0;
    }
    return rc;
}

extern "C" int ephc_transport_start(ephc_handle *h, const double *Gamma_dev, const double *v_dev, double *tau_dev,
                                    double *F0_dev, void *stream) {
    int rc = need_device(h);
    if (rc) return rc;
    if (!Gamma_dev || !v_dev || !tau_dev || !F0_dev) return fail(EPHC_EINVAL, "null device pointer");
    const int64_t ns = h->d.ns;
    tau_f0_kernel<<<(unsigned)((ns + 255) / 256), 256, 0, (cudaStream_t)stream>>>(Gamma_dev, v_dev, tau_dev, F0_dev, ns);
    h->launches++;
    CUDA_TRY(cudaGetLastError());
    return EPHC_OK;
}

extern "C" int ephc_transport_iter(ephc_handle *h, const double *F_dev, const double *v_dev, const double *tau_dev,
                                   double *Fout_dev, void *stream) {
    int rc = need_device(h);
    if (rc) return rc;
    if (!F_dev || !v_dev || !tau_dev || !Fout_dev) return fail(EPHC_EINVAL, "null device pointer");
    if (F_dev == Fout_dev) return fail(EPHC_EINVAL, "transport_iter is out of place: F_dev and Fout_dev must differ");
    if (!h->transport_ready || h->transport_variant != tr_variant(h))
        return fail(EPHC_ESTATE, "call ephc_transport_setup (with the current variant) before ephc_transport_iter");
    if (tr_variant(h) == 1) {
        TileParams T = tile_params(h);
        T.F = F_dev;
        if ((rc = launch_tile<kTIter>(h, T, (cudaStream_t)stream))) return rc;
        FinishParams Fp = finish_params(h);
        Fp.out = Fout_dev;
        Fp.v = v_dev;
        Fp.tau = tau_dev;
        return launch_finish<kFIter>(h, Fp, (cudaStream_t)stream);
    }
    if (h->rows_ok) {
        RowParams R = row_params(h);
        if (h->r_nrows > 0) {
            row_compact_kernel<<<(unsigned)((h->r_nrows + 255) / 256), 256, 0, (cudaStream_t)stream>>>(
                F_dev, h->dr_row_state, h->dr_Fc, h->r_nrows, h->d.ns);
            h->launches++;
        }
        R.Fc = h->dr_Fc;
        R.v = v_dev;
        R.tau = tau_dev;
        R.out = Fout_dev;
        row_iter_kernel<<<(unsigned)std::max(h->r_nstrip, 1), kRowThreads, row_smem_bytes(h->r_Rb, h->r_Ra),
                          (cudaStream_t)stream>>>(R);
        h->launches++;
        CUDA_TRY(cudaGetLastError());
        return EPHC_OK;
    }
    GatherParams P = base_params(h);
    P.F = F_dev;
    P.v = v_dev;
    P.tau = tau_dev;
    P.out = Fout_dev;
    return launch_gather<kTransportIter>(h, P, (cudaStream_t)stream);
}

extern "C" int ephc_transport_iters(ephc_handle *h, const double *F_dev, const double *v_dev, const double *tau_dev,
                                    double *Fout_dev, int niter, void *stream) {
    int rc = need_device(h);
    if (rc) return rc;
    if (!F_dev || !v_dev || !tau_dev || !Fout_dev || niter < 1) return fail(EPHC_EINVAL, "null device pointer or niter < 1");
    if (F_dev == Fout_dev) return fail(EPHC_EINVAL, "transport_iters is out of place: F_dev and Fout_dev must differ");
    if (!h->transport_ready || h->transport_variant != tr_variant(h))
        return fail(EPHC_ESTATE, "call ephc_transport_setup (with the current variant) before ephc_transport_iters");
    if (tr_variant(h) == 0 && h->rows_ok) {
        // chained on the row store: F is brought into compact row order once, every iteration writes the compact copy the
        // next one stages, the last one writes the API layout
        const cudaStream_t s = (cudaStream_t)stream;
        RowParams R = row_params(h);
        if (h->r_nrows > 0) {
            row_compact_kernel<<<(unsigned)((h->r_nrows + 255) / 256), 256, 0, s>>>(F_dev, h->dr_row_state, h->dr_Fc, h->r_nrows, h->d.ns);
            h->launches++;
        }
        R.v = v_dev;
        R.tau = tau_dev;
        double *buf[2] = {h->dr_Fc, h->dr_Fc2};
        for (int it = 0; it < niter; ++it) {
            const bool last = it + 1 == niter;
            R.Fc = buf[it & 1];
            R.Fc_out = last ? nullptr : buf[(it + 1) & 1];
            R.out = last ? Fout_dev : nullptr;
#ifdef EPHC_ROW_TIMING
            static unsigned long long *rdbg = nullptr;
            if (!rdbg) cudaMalloc((void **)&rdbg, 4 * 8 * 1024);
            R.dbg = rdbg;
#endif
            if (it > 0 && std::getenv("EPHC_ROW_NO_PDL") == nullptr) {
                // programmatic dependent launch: iteration it may take an SM as soon as a CTA of iteration it - 1 leaves it
                // (the kernel itself waits for the previous launch to complete before it reads F)
                cudaLaunchConfig_t cfg;
                std::memset(&cfg, 0, sizeof(cfg));
                cfg.gridDim = dim3((unsigned)std::max(h->r_nstrip, 1));
                cfg.blockDim = dim3(kRowThreads);
                cfg.dynamicSmemBytes = row_smem_bytes(h->r_Rb, h->r_Ra);
                cfg.stream = s;
                cudaLaunchAttribute attr[1];
                attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
                attr[0].val.programmaticStreamSerializationAllowed = 1;
                cfg.attrs = attr;
                cfg.numAttrs = 1;
                CUDA_TRY(cudaLaunchKernelEx(&cfg, row_iter_kernel, R));
            } else {
                row_iter_kernel<<<(unsigned)std::max(h->r_nstrip, 1), kRowThreads, row_smem_bytes(h->r_Rb, h->r_Ra), s>>>(R);
            }
            h->launches++;
#ifdef EPHC_ROW_TIMING
            if (it == niter / 2 && std::getenv("EPHC_ROW_TIMING_PRINT")) {
                std::vector<unsigned long long> hd(4 * (size_t)h->r_nstrip);
                cudaMemcpy(hd.data(), rdbg, hd.size() * 8, cudaMemcpyDeviceToHost);
                unsigned long long e0 = ~0ull, e1 = 0, x0 = ~0ull, x1 = 0;
                double pro = 0, loop = 0, epi = 0;
                for (int k = 0; k < h->r_nstrip; ++k) {
                    e0 = std::min(e0, hd[4 * k]); e1 = std::max(e1, hd[4 * k]);
                    x0 = std::min(x0, hd[4 * k + 3]); x1 = std::max(x1, hd[4 * k + 3]);
                    pro += (double)(hd[4 * k + 1] - hd[4 * k]); loop += (double)(hd[4 * k + 2] - hd[4 * k + 1]); epi += (double)(hd[4 * k + 3] - hd[4 * k + 2]);
                }
                std::fprintf(stderr, "row timing (ns): entry spread %llu, first entry -> last exit %llu, exit spread %llu; per CTA prologue %.0f loop %.0f epilogue %.0f\n",
                             e1 - e0, x1 - e0, x1 - x0, pro / h->r_nstrip, loop / h->r_nstrip, epi / h->r_nstrip);
                {   // the slowest and fastest strips (is the spread tied to the strip?)
                    std::vector<std::pair<unsigned long long, int>> tt;
                    for (int k = 0; k < h->r_nstrip; ++k) tt.push_back({hd[4 * k + 3] - hd[4 * k], k});
                    std::sort(tt.begin(), tt.end());
                    std::fprintf(stderr, "row timing fastest:");
                    for (int k = 0; k < 4; ++k) std::fprintf(stderr, " %d:%llu", tt[k].second, tt[k].first);
                    std::fprintf(stderr, "  slowest:");
                    for (int k = 0; k < 6; ++k) std::fprintf(stderr, " %d:%llu", tt[tt.size() - 1 - k].second, tt[tt.size() - 1 - k].first);
                    std::fprintf(stderr, "\n");
                }
            }
#endif
        }
        CUDA_TRY(cudaGetLastError());
        return EPHC_OK;
    }
    // other stores: plain iterations through the scratch vector, ending in Fout
    const double *src = F_dev;
    for (int it = 0; it < niter; ++it) {
        double *dst = ((niter - 1 - it) & 1) ? h->d_Fscr : Fout_dev;
        if ((rc = ephc_transport_iter(h, src, v_dev, tau_dev, dst, stream))) return rc;
        src = dst;
    }
    return EPHC_OK;
}

// One RK4 stage (reading R-18): k = I[y_in]; stage 1..3: y_out = f + a dt k and ksum accumulates b k; stage 4:
// f += dt/6 (ksum + k) in place.  The axpy is the epilogue of the collision pass.
static int launch_drift(ephc_handle *h, const double *f, const double *field, double *out, cudaStream_t s) {
    const double c0 = field[0] * h->d.grid[0] / (2.0 * kHbar), c1 = field[1] * h->d.grid[1] / (2.0 * kHbar),
                 c2 = field[2] * h->d.grid[2] / (2.0 * kHbar);
    drift_kernel<<<(unsigned)((h->d.ns + 255) / 256), 256, 0, s>>>(f, h->d_nbr, c0, c1, c2, out, h->d.nk, h->d.nb);
    h->launches++;
    CUDA_TRY(cudaGetLastError());
    return EPHC_OK;
}

// chained: the caller runs the stages back to back (ephc_rt_step): on the resident-tile store the finish kernel then
// also writes the compact copy that the next stage reads, and fc_ready says that the previous stage did so
static int rk_stage(ephc_handle *h, double *f_dev, const double *y_in, const double *N_dev, double dt_fs, int st, double *y_out,
                    bool want_sum, cudaStream_t s, const double *field = nullptr, bool chained = false, bool fc_ready = false) {
    int rc;
    const int v = rt_variant(h);
    const double *extra = nullptr;
    if (field) {  // Eq. 1: k_j = D[y_j] + I[y_j]
        if ((rc = launch_drift(h, y_in, field, h->d_drift, s))) return rc;
        extra = h->d_drift;
    }
    if (v >= 1) {
        FinishParams Fp;
        if (v >= 2) {
            if ((rc = (v == 3) ? launch_res(h, y_in, N_dev, s, chained && fc_ready) : launch_stream(h, y_in, N_dev, s))) return rc;
            Fp = (v == 3) ? finish_params_res(h) : finish_params_stream(h);
        } else {
            TileParams T = tile_params(h);
            T.f = y_in;
            T.N = N_dev;
            if ((rc = launch_tile<kTCollision>(h, T, s))) return rc;
            Fp = finish_params(h);
        }
        Fp.stage = st;
        Fp.dt = dt_fs;
        Fp.f0 = f_dev;
        Fp.ynext = y_out;
        Fp.ksum = h->d_ksum;
        Fp.blk_sum = want_sum ? h->d_wusum : nullptr;
        Fp.extra = extra;
        Fp.fc_next = (chained && v == 3) ? h->dx_fc : nullptr;
        return launch_finish<kFRkStage>(h, Fp, s);
    }
    GatherParams P = base_params(h);
    P.N = N_dev;
    P.dt = dt_fs;
    P.f0 = f_dev;
    P.ksum = h->d_ksum;
    P.wu_sum = want_sum ? h->d_wusum : nullptr;
    P.extra = extra;
    P.stage = st;
    P.f = y_in;
    P.ynext = y_out;
    return launch_gather<kRkStage>(h, P, s);
}

extern "C" int ephc_rt_stage(ephc_handle *h, double *f_dev, const double *y_in_dev, const double *N_dev, double dt_fs, int stage,
                             double *y_out_dev, void *stream) {
    int rc = need_device(h);
    if (rc) return rc;
    if (!f_dev || !y_in_dev || !N_dev || stage < 1 || stage > 4 || (stage < 4 && !y_out_dev) || !std::isfinite(dt_fs))
        return fail(EPHC_EINVAL, "bad argument (stage 1..4, y_out needed for stages 1..3)");
    if (y_out_dev == y_in_dev || y_out_dev == f_dev) return fail(EPHC_EINVAL, "y_out must differ from y_in and f");
    return rk_stage(h, f_dev, y_in_dev, N_dev, dt_fs, stage, y_out_dev, false, (cudaStream_t)stream);
}

static int rt_step_impl(ephc_handle *h, double *f_dev, const double *N_dev, const double *field, double dt_fs, int nsteps,
                        double *sumf_dev, void *stream);

extern "C" int ephc_rt_step(ephc_handle *h, double *f_dev, const double *N_dev, double dt_fs, int nsteps,
                            double *sumf_dev, void *stream) {
    return rt_step_impl(h, f_dev, N_dev, nullptr, dt_fs, nsteps, sumf_dev, stream);
}

extern "C" int ephc_rt_step_field(ephc_handle *h, double *f_dev, const double *N_dev, const double *field, double dt_fs,
                                  int nsteps, double *sumf_dev, void *stream) {
    if (!field || !std::isfinite(field[0]) || !std::isfinite(field[1]) || !std::isfinite(field[2]))
        return fail(EPHC_EINVAL, "field: three finite components (host array) required");
    return rt_step_impl(h, f_dev, N_dev, field, dt_fs, nsteps, sumf_dev, stream);
}

extern "C" int ephc_drift(ephc_handle *h, const double *f_dev, const double *field, double *out_dev, void *stream) {
    int rc = need_device(h);
    if (rc) return rc;
    if (!f_dev || !out_dev || !field || !std::isfinite(field[0]) || !std::isfinite(field[1]) || !std::isfinite(field[2]))
        return fail(EPHC_EINVAL, "null pointer or non-finite field");
    if (f_dev == out_dev) return fail(EPHC_EINVAL, "ephc_drift is out of place");
    return launch_drift(h, f_dev, field, out_dev, (cudaStream_t)stream);
}

extern "C" int ephc_transport_moments(ephc_handle *h, const double *f0_dev, const double *v_dev, const double *F_dev,
                                      double *out10_dev, void *stream) {
    int rc = need_device(h);
    if (rc) return rc;
    if (!f0_dev || !v_dev || !F_dev || !out10_dev) return fail(EPHC_EINVAL, "null device pointer");
    moments_kernel<<<1, 1024, 0, (cudaStream_t)stream>>>(f0_dev, v_dev, F_dev, h->d.ns, out10_dev);
    h->launches++;
    CUDA_TRY(cudaGetLastError());
    return EPHC_OK;
}

static int rt_step_impl(ephc_handle *h, double *f_dev, const double *N_dev, const double *field, double dt_fs, int nsteps,
                        double *sumf_dev, void *stream) {
    int rc = need_device(h);
    if (rc) return rc;
    if (!f_dev || !N_dev) return fail(EPHC_EINVAL, "null device pointer");
    if (nsteps < 0 || !std::isfinite(dt_fs)) return fail(EPHC_EINVAL, "nsteps >= 0 and finite dt required");
    if (h->ranged)
        return fail(EPHC_ESTATE, "a k-sharded handle owns part of the states: use ephc_rt_stage and exchange y between the stages");
    cudaStream_t s = (cudaStream_t)stream;
    if (sumf_dev) {
        sum_kernel<<<1, 1024, 0, s>>>(f_dev, h->d.ns, sumf_dev);
        h->launches++;
    }
    // one step: stage 1 gathers f, writes y2 -> y[0]; stage 2 gathers y[0], writes y3 -> y[1]; stage 3 gathers y[1],
    // writes y4 -> y[0]; stage 4 gathers y[0], updates f in place; then sum_s f_s -> sum_out
    auto one_step = [&](cudaStream_t st_, bool fc_ready0, double *sum_out) -> int {
        const double *src[4] = {f_dev, h->d_y[0], h->d_y[1], h->d_y[0]};
        double *dst[4] = {h->d_y[0], h->d_y[1], h->d_y[0], nullptr};
        for (int st = 0; st < 4; ++st) {
            const int r = rk_stage(h, f_dev, src[st], N_dev, dt_fs, st + 1, dst[st], sumf_dev != nullptr, st_, field, true, fc_ready0 || st > 0);
            if (r) return r;
        }
        if (sum_out) {
            if (rt_variant(h) >= 1)
                sum_kernel<<<1, 1024, 0, st_>>>(h->d_wusum, finish_grid(h), sum_out);
            else if (h->n_wu > 0)
                sum_kernel<<<1, 1024, 0, st_>>>(h->d_wusum, h->n_wu, sum_out);
            else
                sum_kernel<<<1, 1024, 0, st_>>>(f_dev, h->d.ns, sum_out);
            h->launches++;
        }
        return EPHC_OK;
    };
    int it = 0;
    if (nsteps > 0) {
        if ((rc = one_step(s, false, sumf_dev ? sumf_dev + 1 : nullptr))) return rc;
        it = 1;
    }
#ifndef EPHC_RES_TIMING
    // Long runs (config 5: 1000 steps): the steady-state step -- 8 or 9 launches with fixed arguments -- is captured once
    // into a CUDA graph on the handle's own stream and replayed on the caller's stream; the step's sum goes to a scratch
    // double and is copied to its slot.  Any failure on the way falls back to plain launches.
    if (nsteps - it >= 3 && std::getenv("EPHC_NO_GRAPH") == nullptr && h->cap_stream) {
        ephc_handle::RkKey key = {f_dev, N_dev, dt_fs, {field ? field[0] : 0.0, field ? field[1] : 0.0, field ? field[2] : 0.0},
                                  field != nullptr, sumf_dev != nullptr, rt_variant(h)};
        const ephc_handle::RkKey &k0 = h->rk_key;
        const bool same = k0.f == key.f && k0.N == key.N && k0.dt == key.dt && k0.field[0] == key.field[0] && k0.field[1] == key.field[1] &&
                          k0.field[2] == key.field[2] && k0.has_field == key.has_field && k0.want_sum == key.want_sum &&
                          k0.variant == key.variant;
        if (!h->rk_graph || !same) {
            if (h->rk_graph) cudaGraphExecDestroy(h->rk_graph);
            h->rk_graph = nullptr;
            const int64_t l0 = h->launches;
            cudaGraph_t graph = nullptr;
            if (cudaStreamBeginCapture(h->cap_stream, cudaStreamCaptureModeThreadLocal) == cudaSuccess) {
                const int r = one_step(h->cap_stream, true, sumf_dev ? h->d_sumstep : nullptr);
                const cudaError_t e = cudaStreamEndCapture(h->cap_stream, &graph);
                if (r == EPHC_OK && e == cudaSuccess && graph && cudaGraphInstantiate(&h->rk_graph, graph, 0) == cudaSuccess) {
                    h->rk_key = key;
                    h->rk_graph_launches = (int)(h->launches - l0);
                } else {
                    h->rk_graph = nullptr;
                }
                if (graph) cudaGraphDestroy(graph);
            }
            h->launches = l0;  // nothing ran during the capture
            cudaGetLastError();
        }
        if (h->rk_graph) {
            for (; it < nsteps; ++it) {
                if (cudaGraphLaunch(h->rk_graph, s) != cudaSuccess) {
                    cudaGetLastError();
                    break;  // the remaining steps run as plain launches
                }
                h->launches += h->rk_graph_launches;
                if (sumf_dev) CUDA_TRY(cudaMemcpyAsync(sumf_dev + it + 1, h->d_sumstep, 8, cudaMemcpyDeviceToDevice, s));
            }
        }
    }
#endif
    for (; it < nsteps; ++it)
        if ((rc = one_step(s, true, sumf_dev ? sumf_dev + it + 1 : nullptr))) return rc;
    CUDA_TRY(cudaGetLastError());
    return EPHC_OK;
}

// ---- host-buffer variants (end-to-end path) ----------------------------------------------------------------------
extern "C" int ephc_collision_host(ephc_handle *h, const double *f_host, const double *N_host, double *I_host) {
    int rc = need_device(h);
    if (rc) return rc;
    if (!f_host || !N_host || !I_host) return fail(EPHC_EINVAL, "null host pointer");
    const size_t nf = (size_t)h->d.ns * 8, nN = (size_t)h->d.nq * h->d.nnu * 8;
    if ((rc = ensure(&h->d_hf, nf)) || (rc = ensure(&h->d_hN, nN)) || (rc = ensure(&h->d_hI, nf))) return rc;
    CUDA_TRY(cudaMemcpyAsync(h->d_hf, f_host, nf, cudaMemcpyHostToDevice, 0));
    CUDA_TRY(cudaMemcpyAsync(h->d_hN, N_host, nN, cudaMemcpyHostToDevice, 0));
    rc = ephc_collision(h, h->d_hf, h->d_hN, h->d_hI, nullptr);
    if (rc) return rc;
    CUDA_TRY(cudaMemcpyAsync(I_host, h->d_hI, nf, cudaMemcpyDeviceToHost, 0));
    CUDA_TRY(cudaStreamSynchronize(0));
    return EPHC_OK;
}

extern "C" int ephc_transport_solve_host(ephc_handle *h, const double *f0_host, const double *N_host,
                                         const double *v_host, int niter, double *F_host, double *Gamma_host) {
    int rc = need_device(h);
    if (rc) return rc;
    if (!f0_host || !N_host || !v_host || !F_host || niter < 0) return fail(EPHC_EINVAL, "bad argument");
    const int64_t ns = h->d.ns;
    const size_t nf = (size_t)ns * 8, nN = (size_t)h->d.nq * h->d.nnu * 8;
    if ((rc = ensure(&h->d_hf, nf)) || (rc = ensure(&h->d_hN, nN)) || (rc = ensure(&h->d_tr[0], nf)) ||
        (rc = ensure(&h->d_tr[1], nf)) || (rc = ensure(&h->d_tr[2], 3 * nf)) || (rc = ensure(&h->d_tr[3], 3 * nf)) ||
        (rc = ensure(&h->d_tr[4], 3 * nf)))
        return rc;
    double *Gam = h->d_tr[0], *tau = h->d_tr[1], *v = h->d_tr[2], *Fa = h->d_tr[3], *Fb = h->d_tr[4];
    CUDA_TRY(cudaMemcpyAsync(h->d_hf, f0_host, nf, cudaMemcpyHostToDevice, 0));
    CUDA_TRY(cudaMemcpyAsync(h->d_hN, N_host, nN, cudaMemcpyHostToDevice, 0));
    CUDA_TRY(cudaMemcpyAsync(v, v_host, 3 * nf, cudaMemcpyHostToDevice, 0));
    rc = ephc_transport_setup(h, h->d_hf, h->d_hN, Gam, nullptr);
    if (rc) return rc;
    rc = ephc_transport_start(h, Gam, v, tau, Fa, nullptr);
    if (rc) return rc;
    if (niter > 0) {
        rc = ephc_transport_iters(h, Fa, v, tau, Fb, niter, nullptr);
        if (rc) return rc;
        Fa = Fb;
    }
    CUDA_TRY(cudaMemcpyAsync(F_host, Fa, 3 * nf, cudaMemcpyDeviceToHost, 0));
    if (Gamma_host) CUDA_TRY(cudaMemcpyAsync(Gamma_host, Gam, nf, cudaMemcpyDeviceToHost, 0));
    CUDA_TRY(cudaStreamSynchronize(0));
    return EPHC_OK;
}

extern "C" int ephc_rt_step_host(ephc_handle *h, double *f_host, const double *N_host, double dt_fs, int nsteps,
                                 double *sumf_host) {
    int rc = need_device(h);
    if (rc) return rc;
    if (!f_host || !N_host || nsteps < 0) return fail(EPHC_EINVAL, "bad argument");
    const size_t nf = (size_t)h->d.ns * 8, nN = (size_t)h->d.nq * h->d.nnu * 8;
    if ((rc = ensure(&h->d_hf, nf)) || (rc = ensure(&h->d_hN, nN))) return rc;
    if (sumf_host && h->sumf_cap < nsteps + 1) {
        if (h->d_sumf) cudaFree(h->d_sumf);
        h->d_sumf = nullptr;
        if ((rc = ensure(&h->d_sumf, (size_t)(nsteps + 1) * 8))) return rc;
        h->sumf_cap = nsteps + 1;
    }
    CUDA_TRY(cudaMemcpyAsync(h->d_hf, f_host, nf, cudaMemcpyHostToDevice, 0));
    CUDA_TRY(cudaMemcpyAsync(h->d_hN, N_host, nN, cudaMemcpyHostToDevice, 0));
    rc = ephc_rt_step(h, h->d_hf, h->d_hN, dt_fs, nsteps, sumf_host ? h->d_sumf : nullptr, nullptr);
    if (rc) return rc;
    CUDA_TRY(cudaMemcpyAsync(f_host, h->d_hf, nf, cudaMemcpyDeviceToHost, 0));
    if (sumf_host)
        CUDA_TRY(cudaMemcpyAsync(sumf_host, h->d_sumf, (size_t)(nsteps + 1) * 8, cudaMemcpyDeviceToHost, 0));
    CUDA_TRY(cudaStreamSynchronize(0));
    return EPHC_OK;
}

// ---- allocation-free conservation scalar (callers that cannot call cudaMalloc: graph capture, serving loops) ---------
// sum_s f_s (the quantity whose conservation is checked every rt-BTE step) as the
// library's two-stage reduction -- per-block partial sums in scratch memory, then sum_kernel over the partial sums in a
// fixed order -- with the scratch in a file-scope device array instead of the handle's cudaMalloc'ed d_wusum.
// Every GPU that loads the library holds the array (32 KB) until exit.  All calls share it and it keeps the last call's
// contents: block_sum_kernel overwrites every slot the second stage reads, so nothing has to start at zero; calls that
// overlap on the GPU (different streams) race on it.
constexpr int kNoAllocBlockElems = 4096;  // elements one block of block_sum_kernel sums (256 threads x 16)
constexpr int kNoAllocMaxBlocks = 4096;   // partial sums the scratch holds
static __device__ __align__(256) double g_noalloc_partials[kNoAllocMaxBlocks];
constexpr int kNoAllocMaxDevices = 64;
static double *g_noalloc_ptr[kNoAllocMaxDevices] = {nullptr};  // device address of the array, per device (set-up)

// partial[b] = sum of x[b * 4096 .. min(n, (b + 1) * 4096)) in a fixed order: strided per-thread sums, shuffle tree per
// warp, then the eight warp sums in order
__global__ void __launch_bounds__(256) block_sum_kernel(const double *__restrict__ x, int64_t n, double *__restrict__ partial) {
    __shared__ double sw[8];
    const int64_t lo = (int64_t)blockIdx.x * kNoAllocBlockElems, hi = lo + kNoAllocBlockElems < n ? lo + kNoAllocBlockElems : n;
    double a = 0.0;
    for (int64_t i = lo + threadIdx.x; i < hi; i += 256) a += x[i];
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) a += __shfl_xor_sync(0xffffffffu, a, o);
    if ((threadIdx.x & 31) == 0) sw[threadIdx.x >> 5] = a;
    __syncthreads();
    if (threadIdx.x == 0) {
        double s = 0.0;
#pragma unroll
        for (int w = 0; w < 8; ++w) s += sw[w];
        partial[blockIdx.x] = s;
    }
}

// Set-up for the current device: the address of the scratch array ON THAT DEVICE.  In host code the array's name is a
// host-side stand-in, not a device address; only cudaGetSymbolAddress (with the device current) gives the pointer a
// kernel may use.
extern "C" int ephc_noalloc_init(void) {
    int dev = -1;
    CUDA_TRY(cudaGetDevice(&dev));
    if (dev < 0 || dev >= kNoAllocMaxDevices) return fail(EPHC_ELIMIT, "ephc_noalloc_init: device ordinal beyond 63");
    if (g_noalloc_ptr[dev] != nullptr) return EPHC_OK;
    double *ptr = nullptr;
    CUDA_TRY(cudaGetSymbolAddress((void **)&ptr, g_noalloc_partials));
    if (ptr == nullptr) return fail(EPHC_ECUDA, "cudaGetSymbolAddress returned a null address for the scratch array");
    g_noalloc_ptr[dev] = ptr;
    return EPHC_OK;
}

extern "C" int64_t ephc_noalloc_max_states(void) { return (int64_t)kNoAllocBlockElems * kNoAllocMaxBlocks; }

extern "C" int ephc_sum_states_noalloc(const double *f_dev, int64_t n, double *sum_dev, void *stream) {
    if (!f_dev || !sum_dev) return fail(EPHC_EINVAL, "null device pointer");
    if (n < 0) return fail(EPHC_EINVAL, "ephc_sum_states_noalloc: n must be >= 0");
    if (n > ephc_noalloc_max_states())
        return fail(EPHC_ELIMIT, "ephc_sum_states_noalloc: n = " + std::to_string(n) + " exceeds the fixed scratch (at most " +
                                     std::to_string(ephc_noalloc_max_states()) + " states); use ephc_rt_step's sumf_dev instead");
    int dev = -1;
    CUDA_TRY(cudaGetDevice(&dev));
    if (dev < 0 || dev >= kNoAllocMaxDevices) return fail(EPHC_ELIMIT, "ephc_sum_states_noalloc: device ordinal beyond 63");
    if (g_noalloc_ptr[dev] == nullptr) {  // first use on this device (call ephc_noalloc_init beforehand when capturing a graph)
        const int rc = ephc_noalloc_init();
        if (rc) return rc;
    }
    double *partial = g_noalloc_ptr[dev];
    const cudaStream_t s = (cudaStream_t)stream;
    const int nblk = (int)((n + kNoAllocBlockElems - 1) / kNoAllocBlockElems);
    if (nblk > 0) block_sum_kernel<<<(unsigned)nblk, 256, 0, s>>>(f_dev, n, partial);
    sum_kernel<<<1, 1024, 0, s>>>(partial, nblk, sum_dev);  // reads the nblk slots just written, nothing older
    CUDA_TRY(cudaGetLastError());
    return EPHC_OK;
}
