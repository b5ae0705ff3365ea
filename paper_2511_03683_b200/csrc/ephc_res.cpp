// ephc_res.cpp -- host side of the resident-tile store (variant 3): once-stored directed entries, tile images that
// a CTA fetches with bulk copies and processes in place (see ephc_internal.h "resident-tile store" and DESIGN.md).
// Performed once on the CPU.  The diagonal (q = 0, n == m) terms are left out: they contribute
// exactly 0 to the collision integral; this store serves ephc_collision / ephc_rt_step.
//
// Product code: shares nothing with oracle/.
#include <algorithm>
#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <cstring>

#include "ephc_internal.h"

namespace ephc {

namespace {

struct DEnt {          // directed entry: T = w F_em(f_out, f_in, N[iq, nu]); I[out] -= T; I[in] += T
    int32_t out, in;   // compact rows
    int32_t ip;        // candidate pair (-> iq)
    int32_t nu;
    double w;
};

struct Image {
    ResTile dir;
    std::vector<unsigned char> blob;
    std::vector<uint32_t> iqn;
    int64_t smem = 0;   // blob + X tail + N rows
    int64_t work = 0;
};

struct ImgParams {
    int32_t a_row0, a_rows, b_row0, b_rows;
    int nnu, Lp, Lg;
    int64_t budget;     // bytes available for blob + X tail + N rows
    const int32_t *pair_iq;
};

struct Scratch {
    std::vector<int32_t> cnt, start, idx, pos_of, in_cnt, in_start, in_list;
    std::vector<uint32_t> pair_local;
};

struct Piece {
    int32_t row, start, len;
};
struct GTask {
    int32_t dest, start, len;   // start into a flat list
};

// Column tables of a set of lists sorted by descending length: col[j] = (number of lists longer than j) | (first
// element of column j) << 16.
static void make_cols(const std::vector<int32_t> &lens_desc, std::vector<uint32_t> &cols, int32_t &ncol) {
    ncol = lens_desc.empty() ? 0 : lens_desc[0];
    cols.assign((size_t)ncol, 0);
    size_t n = lens_desc.size();
    int32_t base = 0;
    for (int32_t j = 0; j < ncol; ++j) {
        while (n > 0 && lens_desc[n - 1] <= j) --n;
        cols[j] = (uint32_t)n | ((uint32_t)base << 16);
        base += (int32_t)n;
    }
}

// Builds the image of one tile from entries e[0..n) (sorted by pair).  Returns false when a format limit or the
// shared-memory budget is exceeded (the caller then splits the entry range).
static bool build_image(const DEnt *e, int64_t n, const ImgParams &P, Scratch &S, Image &out) {
    const int32_t R = P.a_rows + P.b_rows;
    if (n > kResXMax || R > kResRowMax) return false;
    auto loc = [&](int32_t row) {
        return (row >= P.a_row0 && row < P.a_row0 + P.a_rows) ? row - P.a_row0 : P.a_rows + (row - P.b_row0);
    };
    // pairs
    S.pair_local.resize((size_t)n);
    out.iqn.clear();
    for (int64_t i = 0; i < n; ++i) {
        if (i == 0 || e[i].ip != e[i - 1].ip) out.iqn.push_back((uint32_t)P.pair_iq[e[i].ip] * (uint32_t)P.nnu);
        S.pair_local[i] = (uint32_t)out.iqn.size() - 1u;
    }
    const int32_t nq = (int32_t)out.iqn.size();
    if ((int64_t)nq * P.nnu > kResSlotMax) return false;
    // out rows -> pieces
    S.cnt.assign((size_t)R + 1, 0);
    for (int64_t i = 0; i < n; ++i) S.cnt[loc(e[i].out) + 1]++;
    S.start.assign((size_t)R + 1, 0);
    for (int32_t r = 0; r < R; ++r) S.start[r + 1] = S.start[r] + S.cnt[r + 1];
    S.idx.resize((size_t)n);
    {
        std::vector<int32_t> &cur = S.cnt;  // reuse as cursor
        for (int32_t r = 0; r < R; ++r) cur[r] = S.start[r];
        for (int64_t i = 0; i < n; ++i) S.idx[cur[loc(e[i].out)]++] = (int32_t)i;
    }
    std::vector<Piece> pieces;
    for (int32_t r = 0; r < R; ++r) {
        const int32_t c = S.start[r + 1] - S.start[r];
        if (c == 0) continue;
        const int32_t npc = (c + P.Lp - 1) / P.Lp, base = c / npc, rem = c % npc;
        int32_t s = S.start[r];
        for (int32_t k = 0; k < npc; ++k) {
            const int32_t len = base + (k < rem ? 1 : 0);
            pieces.push_back(Piece{r, s, len});
            s += len;
        }
    }
    std::stable_sort(pieces.begin(), pieces.end(), [](const Piece &x, const Piece &y) { return x.len > y.len; });
    const int32_t npiece = (int32_t)pieces.size();
    std::vector<int32_t> lens((size_t)npiece);
    for (int32_t p = 0; p < npiece; ++p) lens[p] = pieces[p].len;
    std::vector<uint32_t> cols1, cols2, cols3;
    int32_t nc1 = 0, nc2 = 0, nc3 = 0;
    make_cols(lens, cols1, nc1);
    // entry positions
    S.pos_of.resize((size_t)n);
    for (int32_t p = 0; p < npiece; ++p)
        for (int32_t j = 0; j < pieces[p].len; ++j)
            S.pos_of[S.idx[pieces[p].start + j]] = (int32_t)(cols1[j] >> 16) + p;
    // inputs of every row: positions of its in-entries (ascending), then of its out pieces (ascending)
    S.in_cnt.assign((size_t)R + 1, 0);
    for (int64_t i = 0; i < n; ++i) S.in_cnt[loc(e[i].in) + 1]++;
    for (int32_t p = 0; p < npiece; ++p) S.in_cnt[pieces[p].row + 1]++;
    S.in_start.assign((size_t)R + 1, 0);
    for (int32_t r = 0; r < R; ++r) S.in_start[r + 1] = S.in_start[r] + S.in_cnt[r + 1];
    S.in_list.resize((size_t)n + npiece);
    {
        std::vector<int32_t> &cur = S.in_cnt;
        for (int32_t r = 0; r < R; ++r) cur[r] = S.in_start[r];
        for (int64_t i = 0; i < n; ++i) S.in_list[cur[loc(e[i].in)]++] = S.pos_of[i];
        for (int32_t r = 0; r < R; ++r) std::sort(S.in_list.begin() + S.in_start[r], S.in_list.begin() + cur[r]);
        for (int32_t p = 0; p < npiece; ++p) S.in_list[cur[pieces[p].row]++] = (int32_t)n + p;
    }
    // gather tasks: round 1 (final tasks of rows with <= Lg inputs, partial tasks of the others), round 2 (final tasks
    // of the split rows over their partial sums)
    std::vector<GTask> t1, t2;
    std::vector<int32_t> list2;
    int32_t npart = 0;
    for (int32_t r = 0; r < R; ++r) {
        const int32_t L = S.in_start[r + 1] - S.in_start[r];
        if (L == 0) continue;
        if (L <= P.Lg) {
            t1.push_back(GTask{r, S.in_start[r], L});
            continue;
        }
        const int32_t nchunk = (L + P.Lg - 1) / P.Lg, base = L / nchunk, rem = L % nchunk;
        int32_t s = S.in_start[r];
        t2.push_back(GTask{r, (int32_t)list2.size(), nchunk});
        for (int32_t k = 0; k < nchunk; ++k) {
            const int32_t len = base + (k < rem ? 1 : 0);
            t1.push_back(GTask{0x8000 | npart, s, len});
            list2.push_back((int32_t)n + npiece + npart);
            ++npart;
            s += len;
        }
    }
    if (npart > 0x7fff || n + npiece + npart > kResXMax) return false;
    std::stable_sort(t1.begin(), t1.end(), [](const GTask &x, const GTask &y) { return x.len > y.len; });
    std::stable_sort(t2.begin(), t2.end(), [](const GTask &x, const GTask &y) { return x.len > y.len; });
    const int32_t ntask1 = (int32_t)t1.size(), ntask2 = (int32_t)t2.size();
    lens.resize((size_t)ntask1);
    for (int32_t t = 0; t < ntask1; ++t) lens[t] = t1[t].len;
    make_cols(lens, cols2, nc2);
    lens.resize((size_t)ntask2);
    for (int32_t t = 0; t < ntask2; ++t) lens[t] = t2[t].len;
    make_cols(lens, cols3, nc3);
    const int32_t ngl1 = (int32_t)n + npiece, ngl2 = (int32_t)list2.size();
    const ResLayout L = res_layout((int32_t)n, npiece, ntask1, ntask2, nc1 + nc2 + nc3, ngl1 + ngl2);
    out.smem = (int64_t)L.bytes + 8 * (int64_t)(npiece + npart) + 16 + 8 * (int64_t)nq * P.nnu;
    if (out.smem > P.budget) return false;
    // ---- fill the blob ---------------------------------------------------------------------------------------------
    out.blob.assign((size_t)L.bytes, 0);
    uint32_t *code = reinterpret_cast<uint32_t *>(out.blob.data() + L.code);
    uint16_t *perm = reinterpret_cast<uint16_t *>(out.blob.data() + L.perm);
    uint16_t *prow = reinterpret_cast<uint16_t *>(out.blob.data() + L.prow);
    uint16_t *d1 = reinterpret_cast<uint16_t *>(out.blob.data() + L.d1);
    uint16_t *d2 = reinterpret_cast<uint16_t *>(out.blob.data() + L.d2);
    uint32_t *cols = reinterpret_cast<uint32_t *>(out.blob.data() + L.cols);
    double *w = reinterpret_cast<double *>(out.blob.data() + L.w);
    for (int64_t i = 0; i < n; ++i) {
        const int32_t pos = S.pos_of[i];
        code[pos] = ((uint32_t)loc(e[i].in) << 3) | ((S.pair_local[i] * (uint32_t)P.nnu + (uint32_t)e[i].nu) << 19);
        w[pos] = e[i].w;
    }
    for (int32_t p = 0; p < npiece; ++p) prow[p] = (uint16_t)pieces[p].row;
    for (int32_t t = 0; t < ntask1; ++t) {
        d1[t] = (uint16_t)t1[t].dest;
        for (int32_t j = 0; j < t1[t].len; ++j) perm[(cols2[j] >> 16) + t] = (uint16_t)S.in_list[t1[t].start + j];
    }
    for (int32_t t = 0; t < ntask2; ++t) {
        d2[t] = (uint16_t)t2[t].dest;
        for (int32_t j = 0; j < t2[t].len; ++j) perm[ngl1 + (cols3[j] >> 16) + t] = (uint16_t)list2[t2[t].start + j];
    }
    std::copy(cols1.begin(), cols1.end(), cols);
    std::copy(cols2.begin(), cols2.end(), cols + nc1);
    std::copy(cols3.begin(), cols3.end(), cols + nc1 + nc2);
    ResTile &D = out.dir;
    std::memset(&D, 0, sizeof(D));
    D.blob_bytes = L.bytes;
    D.ne = (int32_t)n;
    D.npiece = npiece;
    D.npart = npart;
    D.ntask1 = ntask1;
    D.ntask2 = ntask2;
    D.nc1 = nc1;
    D.nc2 = nc2;
    D.nc3 = nc3;
    D.ngl1 = ngl1;
    D.ngl2 = ngl2;
    D.nq = nq;
    D.b_row0 = P.b_row0;
    D.b_rows = P.b_rows;
    D.b_slot = -1;
    // cost model of a tile for the run cut and the hand-out order (entries, row pieces / tasks, staged N rows, fixed)
    out.work = n + 4 * (int64_t)(npiece + ntask1 + ntask2) + 3 * (int64_t)nq + 400;
    return true;
}

static int build_images(const DEnt *e, int64_t n, const ImgParams &P, Scratch &S, std::vector<Image> &outs) {
    if (n <= 0) return EPHC_OK;
    Image img;
    if (build_image(e, n, P, S, img)) {
        outs.push_back(std::move(img));
        return EPHC_OK;
    }
    if (n == 1) return EPHC_ELIMIT;
    int64_t mid = n / 2, lo = mid, hi = mid;  // prefer a pair boundary near the middle
    while (lo > n / 4 && e[lo].ip == e[lo - 1].ip) --lo;
    while (hi < n - n / 4 && e[hi].ip == e[hi - 1].ip) ++hi;
    if (lo > 0 && e[lo].ip != e[lo - 1].ip)
        mid = lo;
    else if (hi < n && e[hi].ip != e[hi - 1].ip)
        mid = hi;
    int rc = build_images(e, mid, P, S, outs);
    if (rc == EPHC_OK) rc = build_images(e + mid, n - mid, P, S, outs);
    return rc;
}

static int env_int(const char *name, int dflt) {
    const char *e = std::getenv(name);
    return e ? std::atoi(e) : dflt;
}

}  // namespace

int build_res(const ephc_problem *p, const Dims &d, const Canonical &c, int ncta, int64_t smem_cap, ResHost &t,
              std::string &err) {
    const int nb = d.nb, nnu = d.nnu;
    const int64_t npair = p->npair;
    t = ResHost();
    t.nnu = nnu;
    if (ncta < 1) ncta = 1;
    try {
        t.state_row.assign((size_t)d.ns, -1);
        for (int64_t s = 0; s < d.ns; ++s)
            if (p->E[s] >= p->emin && p->E[s] <= p->emax) {
                t.state_row[s] = (int32_t)t.row_state.size();
                t.row_state.push_back((int32_t)s);
            }
        t.nrows = (int32_t)t.row_state.size();
        const int64_t nent = c.nw;
        t.nent = nent;
        // ---- geometry: strips of Ra rows, B ranges of <= RbMax rows in units of fine blocks of Rf rows --------------
        int Ra = env_int("EPHC_RES_ROWS", 1024), RbMax = env_int("EPHC_RES_ROWS_B", 512);
        const int Lp = std::max(1, env_int("EPHC_RES_LP", 16)), Lg = std::max(2, env_int("EPHC_RES_LG", 16));
        Ra = std::max(1, std::min(Ra, kResRowMax / 2));
        RbMax = std::max(1, std::min(RbMax, kResRowMax / 2));
        if (!std::getenv("EPHC_RES_ROWS")) {
            // small problems: enough strips that every CTA gets a few runs
            while (Ra > 16 && (int64_t)(t.nrows / Ra) * (t.nrows / Ra) < 8 * (int64_t)ncta) Ra /= 2;
        }
        const int64_t budget = smem_cap - 16 * (int64_t)(Ra + RbMax) - 512;
        if (budget < 4096) {
            t.why = "resident-tile store: shared-memory budget too small";
            return EPHC_OK;
        }
        int Rf = env_int("EPHC_RES_FINE", 0);
        if (Rf <= 0) {
            // an atom (strip x fine block) should hold about a sixth of what fits in a tile
            const double rho = (double)std::max<int64_t>(nent, 1) / (0.5 * (double)t.nrows * (double)t.nrows + 1.0);
            const double per_row = std::max(1e-9, rho * Ra) * (14.5 + 8.0 * nnu / std::max(1.0, (double)nent / std::max<int64_t>(1, c.npair_active)));
            Rf = 128;
            while (Rf > 4 && Rf * per_row > (double)budget / 6.0) Rf /= 2;
        }
        Rf = std::max(1, std::min(Rf, Ra));
        Ra = std::max(Rf, Ra / Rf * Rf);
        RbMax = std::max(Rf, RbMax / Rf * Rf);
        t.Ra = Ra;
        t.rf = Rf;
        t.nblk = std::max(1, (t.nrows + Rf - 1) / Rf);
        t.blk_row0.resize((size_t)t.nblk + 1);
        for (int32_t b = 0; b <= t.nblk; ++b) t.blk_row0[b] = std::min(t.nrows, b * Rf);
        t.state_blk.assign((size_t)d.ns, -1);
        for (int64_t s = 0; s < d.ns; ++s)
            if (t.state_row[s] >= 0) t.state_blk[s] = t.state_row[s] / Rf;
        const int32_t bps = Ra / Rf;
        const int32_t nstrip = (t.nblk + bps - 1) / bps;
        std::vector<int64_t> atom0((size_t)nstrip + 1, 0);  // atoms of strip I: diagonal, then the fine blocks after it
        for (int32_t I = 0; I < nstrip; ++I) atom0[I + 1] = atom0[I] + 1 + std::max(0, t.nblk - (I + 1) * bps);
        const int64_t natom = atom0[nstrip];
        auto atom_of = [&](int32_t a, int32_t b) {  // a < b compact rows
            const int32_t I = a / Ra, j = b / Rf;
            return (j < (I + 1) * bps) ? atom0[I] : atom0[I] + 1 + (j - (I + 1) * bps);
        };
        // entries and pairs per atom
        std::vector<int64_t> atom_ne((size_t)natom + 1, 0);
        std::vector<int32_t> atom_np((size_t)natom + 1, 0);
        for (int64_t ip = 0; ip < npair; ++ip) {
            const int64_t sa = (int64_t)p->pair_ik[ip] * nb, sb = (int64_t)p->pair_ikq[ip] * nb;
            int64_t last = -1;
            for (int64_t j = c.pair_ch0[ip]; j < c.pair_ch0[ip + 1]; ++j) {
                const int n = c.ch_code[j] & 15, m = (c.ch_code[j] >> 4) & 15;
                const int64_t at = atom_of(t.state_row[sa + n], t.state_row[sb + m]);
                atom_ne[at + 1] += (c.ch_wabs[j] != 0.0) + (c.ch_wem[j] != 0.0);
                if (at != last) atom_np[at + 1]++;  // upper bound (a pair can come back to an atom)
                last = at;
            }
        }
        // initial tiles: consecutive atoms of a strip while the estimated image fits
        struct Init {
            int64_t at0, at1;
            int32_t strip;
        };
        std::vector<Init> inits;
        for (int32_t I = 0; I < nstrip; ++I) {
            const int32_t a_rows = std::min(t.nrows, (I + 1) * Ra) - std::min(t.nrows, I * Ra);
            if (atom_ne[atom0[I] + 1] > 0) inits.push_back(Init{atom0[I], atom0[I] + 1, I});
            int64_t a0 = atom0[I] + 1;
            while (a0 < atom0[I + 1]) {
                if (atom_ne[a0 + 1] == 0) {
                    ++a0;
                    continue;
                }
                int64_t a1 = a0, E = 0, Pq = 0;
                while (a1 < atom0[I + 1] && (a1 + 1 - a0) * Rf <= RbMax) {
                    const int64_t E2 = E + atom_ne[a1 + 1], P2 = Pq + atom_np[a1 + 1];
                    const int64_t rows = a_rows + (a1 + 1 - a0) * Rf;
                    const int64_t est = 15 * E2 + 8 * (int64_t)nnu * P2 + 14 * std::min<int64_t>(rows, 2 * E2) + 12 * E2 / Lp + 512;
                    if (a1 > a0 && (est > budget || E2 > kResXMax * 3 / 4 || P2 * nnu > kResSlotMax)) break;
                    E = E2;
                    Pq = P2;
                    ++a1;
                }
                while (a1 - 1 > a0 && atom_ne[a1] == 0) --a1;
                inits.push_back(Init{a0, a1, I});
                a0 = a1;
            }
        }
        for (int64_t i = 0; i < natom; ++i) atom_ne[i + 1] += atom_ne[i];
        const int64_t ninit = (int64_t)inits.size();
        std::vector<int64_t> init_e0((size_t)ninit + 1, 0);
        std::vector<int32_t> atom_init((size_t)natom, -1);
        for (int64_t it = 0; it < ninit; ++it) {
            for (int64_t at = inits[it].at0; at < inits[it].at1; ++at) atom_init[at] = (int32_t)it;
            init_e0[it + 1] = init_e0[it] + (atom_ne[inits[it].at1] - atom_ne[inits[it].at0]);
        }
        if (init_e0[ninit] != nent) {
            err = "internal: resident-tile store lost entries";
            return EPHC_ESTATE;
        }
        // bucket the directed entries by initial tile (canonical order inside a tile = sorted by pair)
        std::vector<DEnt> ents((size_t)nent);
        {
            std::vector<int64_t> cur(init_e0.begin(), init_e0.end() - 1);
            for (int64_t ip = 0; ip < npair; ++ip) {
                const int64_t sa = (int64_t)p->pair_ik[ip] * nb, sb = (int64_t)p->pair_ikq[ip] * nb;
                for (int64_t j = c.pair_ch0[ip]; j < c.pair_ch0[ip + 1]; ++j) {
                    const int n = c.ch_code[j] & 15, m = (c.ch_code[j] >> 4) & 15, nu = c.ch_code[j] >> 8;
                    const int32_t a = t.state_row[sa + n], b = t.state_row[sb + m];
                    const int64_t it = atom_init[atom_of(a, b)];
                    // emission weight: out = a, in = b; absorption weight: out = b, in = a (F_abs(a,b) = -F_em(b,a))
                    if (c.ch_wem[j] != 0.0) ents[cur[it]++] = DEnt{a, b, (int32_t)ip, nu, c.ch_wem[j]};
                    if (c.ch_wabs[j] != 0.0) ents[cur[it]++] = DEnt{b, a, (int32_t)ip, nu, c.ch_wabs[j]};
                }
            }
        }
        // images (parallel over initial tiles)
        std::vector<std::vector<Image>> imgs((size_t)ninit);
        int rc_all = EPHC_OK;
#pragma omp parallel
        {
            Scratch S;
#pragma omp for schedule(dynamic, 4)
            for (int64_t it = 0; it < ninit; ++it) {
                const Init &in = inits[it];
                ImgParams P;
                P.a_row0 = std::min(t.nrows, in.strip * Ra);
                P.a_rows = std::min(t.nrows, (in.strip + 1) * Ra) - P.a_row0;
                if (in.at0 == atom0[in.strip]) {
                    P.b_row0 = P.a_row0;
                    P.b_rows = 0;
                } else {
                    const int32_t j0 = (in.strip + 1) * bps + (int32_t)(in.at0 - atom0[in.strip] - 1);
                    const int32_t j1 = (in.strip + 1) * bps + (int32_t)(in.at1 - 1 - atom0[in.strip] - 1);
                    P.b_row0 = t.blk_row0[j0];
                    P.b_rows = t.blk_row0[j1 + 1] - P.b_row0;
                }
                P.nnu = nnu;
                P.Lp = Lp;
                P.Lg = Lg;
                P.budget = budget;
                P.pair_iq = c.pair_iq.data();
                const int rc = build_images(ents.data() + init_e0[it], init_e0[it + 1] - init_e0[it], P, S, imgs[it]);
                if (rc != EPHC_OK) {
#pragma omp critical
                    rc_all = rc;
                }
            }
        }
        if (rc_all != EPHC_OK) {
            err = "resident-tile store: a single entry does not fit the shared-memory budget";
            return rc_all;
        }
        std::vector<DEnt>().swap(ents);
        // ---- concatenate: tiles, runs, slots ------------------------------------------------------------------------
        int64_t total_work = 0, blob_bytes = 0;
        for (auto &v : imgs)
            for (Image &im : v) {
                total_work += im.work;
                blob_bytes += (im.dir.blob_bytes + 127) & ~127;
            }
        const int runs_per_cta = std::max(1, env_int("EPHC_RES_RUNS_PER_CTA", 6));
        const int64_t run_goal = std::max<int64_t>(1, total_work / ((int64_t)ncta * runs_per_cta));
        t.blob.assign((size_t)blob_bytes + 128, 0);
        int64_t rows = 0, boff = 0;
        auto new_slot = [&](int32_t row0, int32_t nrows_) {
            const int32_t sl = (int32_t)t.slot_off.size();
            t.slot_off.push_back(rows);
            t.slot_row0.push_back(row0);
            t.slot_rows.push_back(nrows_);
            rows += nrows_;
            return sl;
        };
        std::vector<int64_t> run_work;
        int32_t cur_strip = -1;
        int64_t cur_work = 0;
        t.Rcap = 2;
        for (int64_t it = 0; it < ninit; ++it) {
            const int32_t I = inits[it].strip;
            const int32_t a_row0 = std::min(t.nrows, I * Ra), a_rows = std::min(t.nrows, (I + 1) * Ra) - a_row0;
            for (Image &im : imgs[it]) {
                if (I != cur_strip || cur_work + im.work / 2 > run_goal) {
                    ResRun r;
                    std::memset(&r, 0, sizeof(r));
                    r.t0 = (int32_t)t.tiles.size();
                    r.nt = 0;
                    r.a_row0 = a_row0;
                    r.a_rows = a_rows;
                    r.a_slot = new_slot(a_row0, a_rows);
                    t.runs.push_back(r);
                    run_work.push_back(0);
                    cur_strip = I;
                    cur_work = 0;
                }
                ResTile D = im.dir;
                D.blob_off = boff;
                D.q0 = (int32_t)t.iqn.size();
                if (D.b_rows > 0) D.b_slot = new_slot(D.b_row0, D.b_rows);
                if ((int64_t)t.iqn.size() + D.nq > 0x7fffffffLL) {
                    err = "resident-tile store: more than 2^31 tile pairs";
                    return EPHC_ELIMIT;
                }
                std::memcpy(t.blob.data() + boff, im.blob.data(), im.blob.size());
                boff += (D.blob_bytes + 127) & ~127;
                t.iqn.insert(t.iqn.end(), im.iqn.begin(), im.iqn.end());
                t.smem_tile = std::max(t.smem_tile, im.smem);
                t.Rcap = std::max(t.Rcap, a_rows + D.b_rows);
                t.tiles.push_back(D);
                t.runs.back().nt++;
                run_work.back() += im.work;
                cur_work += im.work;
                im = Image();
            }
        }
        t.Rcap = (t.Rcap + 1) & ~1;
        t.order.resize(t.runs.size());
        for (size_t i = 0; i < t.runs.size(); ++i) t.order[i] = (int32_t)i;
        std::stable_sort(t.order.begin(), t.order.end(), [&](int32_t x, int32_t y) { return run_work[x] > run_work[y]; });
        t.part_rows = rows;
        t.blk_ent_ptr.assign((size_t)t.nblk + 1, 0);
        const int64_t nslot = (int64_t)t.slot_off.size();
        for (int64_t sl = 0; sl < nslot; ++sl)
            for (int32_t b = t.slot_row0[sl] / Rf; b * Rf < t.slot_row0[sl] + t.slot_rows[sl]; ++b) t.blk_ent_ptr[b + 1]++;
        for (int32_t b = 0; b < t.nblk; ++b) t.blk_ent_ptr[b + 1] += t.blk_ent_ptr[b];
        t.blk_ent_off.assign((size_t)t.blk_ent_ptr[t.nblk], 0);
        {
            std::vector<int32_t> cur(t.blk_ent_ptr.begin(), t.blk_ent_ptr.end() - 1);
            for (int64_t sl = 0; sl < nslot; ++sl)
                for (int32_t b = t.slot_row0[sl] / Rf; b * Rf < t.slot_row0[sl] + t.slot_rows[sl]; ++b)
                    t.blk_ent_off[cur[b]++] = t.slot_off[sl] + (t.blk_row0[b] - t.slot_row0[sl]);
        }
        if (std::getenv("EPHC_DEBUG")) {
            double ne = 0, np = 0, nt1 = 0, nt2 = 0, nq = 0, bb = 0, br = 0;
            for (const ResTile &D : t.tiles) {
                ne += D.ne;
                np += D.npiece;
                nt1 += D.ntask1;
                nt2 += D.ntask2;
                nq += D.nq;
                bb += D.blob_bytes;
                br += D.b_rows;
            }
            const double n = (double)std::max<size_t>(t.tiles.size(), 1);
            std::fprintf(stderr,
                         "res store: Ra %d Rf %d RbMax %d budget %lld | %zu tiles in %zu runs, per tile: %.0f entries, %.0f pieces, "
                         "%.0f + %.0f tasks, %.0f pairs, %.0f B rows, %.0f blob bytes (%.2f B/entry), smem max %lld, part rows %lld\n",
                         Ra, Rf, RbMax, (long long)budget, t.tiles.size(), t.runs.size(), ne / n, np / n, nt1 / n, nt2 / n,
                         nq / n, br / n, bb / n, bb / std::max(ne, 1.0), (long long)t.smem_tile, (long long)t.part_rows);
        }
    } catch (const std::bad_alloc &) {
        err = "host allocation failed (resident-tile store)";
        return EPHC_ENOMEM;
    }
    t.supported = true;
    return EPHC_OK;
}

}  // namespace ephc
