// ephc_internal.h -- private declarations shared by the host builder, the kernels and the C ABI.
// Product code: shares nothing with oracle/.
#pragma once
#include <cstdint>
#include <string>
#include <vector>

#include "../../include/ephc.h"

namespace ephc {

constexpr double kHbar = 0.6582119569;  // eV fs (R-9)
constexpr double kPi = 3.14159265358979323846;

// ---- launch geometry of the gather kernels ------------------------------
constexpr int kThreads = 256;       // threads per CTA (8 warps)
constexpr int kVMax = 5120;         // doubles of staged pair data per round (40 KB)
constexpr int kRowsMax = 256;       // destination rows (states) per work unit
constexpr int kTasksMax = 384;      // warp tasks per round
constexpr int kTaskLen = 256;       // max entries per warp task
constexpr int kEntriesTarget = 8192;  // entries per work unit (soft)

// ---- entry code of the gather store ------------------------------------------------------------------
//  bits  0..19  half-pair index relative to the round's first half-pair
//  bits 20..23  band of the partner state
//  bits 24..29  phonon mode
//  bit  30      kind: 0 = absorption factor F_abs, 1 = emission factor F_em (as seen from the destination)
//  bit  31      diagonal (q = 0, n == m) term: transport only
constexpr uint32_t kPairBits = 20, kPairMask = (1u << kPairBits) - 1u;
constexpr uint32_t kBandShift = 20, kModeShift = 24, kKindBit = 30, kDiagBit = 31;

struct Task {      // one warp task: a run of entries that all feed the same destination state
    int64_t e0;    // first entry
    int32_t len;   // 1..kTaskLen
    int32_t row;   // destination state index s = ik*nb + n
};
struct Round {     // pair data staged together in shared memory
    int32_t hp0, nhp;  // half-pair range
    int32_t t0, nt;    // task range
};
struct WorkUnit {  // one CTA: whole k segments, the single owner of their rows
    int32_t r0, r1;      // round range
    int32_t row0, nrows; // state range
};

// canonical unordered channel list + diagonal terms (host)
struct Canonical {
    std::vector<int64_t> pair_ch0;   // [npair+1] first channel of each candidate pair
    std::vector<int64_t> pair_dg0;   // [npair+1] first diagonal term of each candidate pair
    std::vector<int32_t> pair_iq;    // [npair]
    std::vector<uint16_t> ch_code;   // n | m << 4 | nu << 8
    std::vector<double> ch_wabs, ch_wem;
    std::vector<int32_t> dg_s, dg_nu;
    std::vector<double> dg_wabs, dg_wem;
    int64_t nch = 0, nw = 0, ndiag = 0, npair_active = 0;
    int32_t iq0 = 0;                 // q = 0 index (always 0 on this grid convention)
};

// destination-sorted two-sided store (host image)
struct GatherHost {
    std::vector<uint32_t> code;
    std::vector<double> w;
    std::vector<int32_t> hp_k, hp_q;   // partner k (compact), canonical iq
    std::vector<Task> tasks;
    std::vector<Round> rounds;
    std::vector<WorkUnit> wus;
};

struct Dims {
    int32_t grid[3];
    int32_t nk, nb, nnu;
    int64_t nq, ns;
    double C;
    int32_t k_lo = 0, k_hi = 0;  // destination k points this handle owns (k-sharded evaluation); [0, nk) = all
};

// host builder (ephc_build.cu)
int validate_problem(const ephc_problem *p, const Dims &d, std::string &err);
int build_canonical(const ephc_problem *p, const Dims &d, Canonical &c, std::string &err);
int build_gather(const ephc_problem *p, const Dims &d, const Canonical &c, GatherHost &g, std::string &err);

// ---- tile store (variant 1): every channel stored once, both of its ends updated by the same thread ----------
// (DESIGN.md "Tile store").  States inside the energy window get a compact row index; compact rows are cut into
// fine blocks (whole k points), fine blocks into strips.  A tile holds every active pair with k in strip I and
// k' in a range of fine blocks (or in strip I itself: diagonal tile); tile boundaries are chosen so that every
// CTA gets the same work in one to three tiles.  Per tile the CTA keeps f (or F) and the accumulators of both
// row ranges in shared memory, processes the tile's pairs one lane per pair (slices of 32 pairs, sorted by length,
// entries stored column-major per slice), and adds every pair's partial sums into the shared accumulators in a
// fixed, host-assigned ticket order per k point (plain read-modify-write, no atomics, bit-reproducible).
constexpr int kTileNbMax = 4;        // bands handled in registers (compact band rank < 4)
constexpr int kTileNnuMax = 8;       // modes handled in registers
constexpr int kTilePieceMax = 255;   // entries per pair record (longer pairs are split into pieces)
constexpr int kTileTicketMax = 4095; // pair records per k point and tile
// entry code (uint16): compact band rank at k | rank at k' << 2 | mode << 4 | kind << 7 | diagonal << 8
constexpr uint32_t kTcM = 2, kTcNu = 4, kTcKind = 7, kTcDiag = 8;
// pair record: 3 x uint32, stored as three arrays [3][npiece]
//   [0] first compact row of k, local to block I | first compact row of k', local to block J << 16
//   [1] canonical iq (24 bits) | number of entries (8 bits) << 24
//   [2] ticket at k (12 bits) | (in-window bands at k) - 1 << 12 | ticket at k' << 16 | (bands at k') - 1 << 28
struct TileSlice {   // 32 pair records, lanes sorted by descending length
    int64_t e0;      // first entry
    int32_t p0;      // first pair record
    int16_t np;      // pair records (1..32)
    int16_t maxlen;  // entries of lane 0
};
struct TileHdr {
    int32_t s0, ns;          // slice range
    int32_t a_row0, a_rows;  // compact rows of the k side (a strip of fine blocks)
    int32_t b_row0, b_rows;  // compact rows of the k' side (a range of fine blocks; the strip itself on a diagonal tile)
    int32_t a_slot, b_slot;  // partial-sum slots (b_slot = -1 on a diagonal tile)
    int32_t flags;           // bit 0: first tile of an a-run (stage the strip, zero its accumulators); bit 1: last;
                             // bit 2: diagonal tile (k and k' in the same strip: one set of arrays)
    int32_t p0, npc;         // first pair record and number of pair records (slice g holds records p0 + 32 g ...)
    int32_t pad;
};
struct TileCta {
    int32_t t0, t1;          // tile range
};
struct TileHost {
    int32_t Ra = 0, Rb = 0;           // largest a_rows / b_rows of any tile (shared-memory sizing)
    int32_t nblk = 0, nrows = 0, ncta = 0;
    std::vector<int32_t> blk_row0;    // [nblk+1] compact row range of a FINE block (unit of tile boundaries)
    std::vector<int32_t> row_state;   // [nrows] state index of a compact row
    std::vector<int32_t> state_row;   // [ns] compact row of a state, -1 outside the window
    std::vector<int32_t> state_blk;   // [ns] fine block of a state's row, -1 outside the window
    std::vector<double> w;            // entries
    std::vector<uint16_t> code;
    std::vector<uint32_t> prec;       // [3][npiece]
    std::vector<TileSlice> slices;
    std::vector<TileHdr> tiles;
    std::vector<TileCta> ctas;
    std::vector<int64_t> slot_off;    // [nslot] offset of a slot in rows (x components in the kernels)
    std::vector<int32_t> slot_row0, slot_rows;  // [nslot] compact row range a slot covers
    std::vector<int32_t> blk_ent_ptr; // [nblk+1] CSR over fine blocks: the slots that hold partial sums of the block
    std::vector<int64_t> blk_ent_off; // per entry: row offset in the partial-sum buffer of the block's first row
    int64_t part_rows = 0;            // total rows of all slots
    int64_t npiece = 0;               // pair records
    bool supported = false;           // false: shape outside the register path (nb > 4, nnu > 8, ...)
    std::string why;                  // reason when unsupported
};
int build_tiles(const ephc_problem *p, const Dims &d, const Canonical &c, int ncta, TileHost &t, std::string &err);

// ---- row store (transport_iter): destination-sorted, two-sided, tiled over the partner rows ---------------------
// In the transport iteration the two directions of a channel carry DIFFERENT weights W(a<-b), W(b<-a)
// (PAPER.md:110), so storing every ordered term with its destination costs no extra weight bytes.  Compact rows
// (states inside the window) are cut into strips of equal ordered-entry count, one per CTA, which is the single
// owner of its rows of F'.  The partner rows are cut into ranges of <= Rb rows whose F values
// are staged in shared memory; inside a (strip, range) tile every destination row has one contiguous segment
// of entries (weight fp64 + partner row relative to the range, uint16), segments sorted by descending length.
struct RowSeg {        // 16 bytes: one destination row inside one tile
    uint32_t start;    // first entry, relative to the strip's first entry
    uint32_t len;
    uint32_t row;      // destination row, local to the strip
    uint32_t pad;
};
struct RowTile {
    int32_t seg0, nseg;      // segment range
    int32_t col0, ncols;     // partner rows staged for this tile: compact rows [col0, col0 + ncols), or -- sparse staging --
                             // the rows cols[col0 .. col0 + ncols) of the strip's list of referenced partner rows
};
struct RowStrip {
    int64_t e0;              // first entry of the strip
    int32_t row0, nrows;     // destination rows (compact)
    int32_t t0, t1;          // tile range
};
struct RowHost {
    int32_t Rb = 0, Ra = 0, nrows = 0;
    std::vector<int32_t> row_state, state_row;
    std::vector<int32_t> cols;        // sparse staging (empty otherwise): per strip the sorted partner rows its entries reference
    std::vector<uint16_t> idx;        // per entry: partner row - col0 of its tile (sparse staging: position in the tile's chunk of cols)
    std::vector<uint32_t> perm;       // per entry: index of the same ordered term in the gather store (host only: export / tests)
    std::vector<double> wst;          // per entry: the channel weight |g|^2 delta of this ordered term (transport_setup reads it)
    std::vector<uint32_t> meta;       // per entry: (iq * nnu + mode) | kind << 31 (kind as seen from the destination)
    std::vector<RowSeg> segs;
    std::vector<RowTile> tiles;
    std::vector<RowStrip> strips;
};
int build_rows(const ephc_problem *p, const Dims &d, const GatherHost &g, int nstrip, RowHost &r, std::string &err);
// Mode-collapsed row store (transport specialisation, SURVEY.md 8(d) honesty note / 8(f) NEXT-3): in
// F'_a = tau_a (v_a + sum_b W(a<-b) F_b) the ordered terms of one (a, b) state pair -- its modes and kinds -- enter
// through the SUM of their weights only, so the iteration can run on one weight per state pair.  Same strips, ranges and
// tiles as the row store; one entry per (destination, partner) pair of a segment (the row store keeps them adjacent);
// first[] / count[] locate the terms whose weights transport_setup sums into it.  Fewer bytes per channel-term than the
// general path: reported separately, never chosen by default.
struct RowCollapsed {
    std::vector<uint16_t> idx;        // per collapsed entry: partner row - col0 of its tile
    std::vector<uint32_t> first;      // per collapsed entry: first ordered term in the row store (absolute position)
    std::vector<uint16_t> count;      // per collapsed entry: ordered terms summed
    std::vector<RowSeg> segs;
    std::vector<RowTile> tiles;
    std::vector<RowStrip> strips;
};
int build_rows_collapsed(const RowHost &r, RowCollapsed &c, std::string &err);

// ---- stream store (variant 2, collision / RK stages): one LANE per ENTRY ------------------------------------------
// Same tiles and partial-sum slots as the tile store (strip of k rows x range of k' rows, both staged in shared
// memory), but inside a tile the entries are sorted by their k-side row and cut into chunks of <= 2048 entries.
// A chunk is evaluated by all threads of the CTA, one entry per lane and step, fully coalesced; the per-entry terms
// T stay in shared memory and are then summed per k row (contiguous runs) and per k' row (through a chunk-local
// permutation) by one thread per row: one owner per row and chunk, no atomics, fixed order.
//   entry: w fp64 + code uint32 = k row - chunk.a0 (8 bit) | k' row - tile.b_row0 (11 bit) << 8 |
//                                 N slot = pair_in_chunk * nnu + mode (12 bit) << 19 | kind << 31
constexpr int kStreamChunk = 2048;     // entries per chunk
constexpr int kStreamNSlots = 2048;    // N values staged per chunk
constexpr int kStreamRbMax = 2048;    // 11-bit k' row in the entry code
struct StreamChunk {          // 48 bytes
    int64_t e0;               // first entry (also first perm element)
    int32_t ne;               // entries
    int32_t a0;               // k row (local to the tile) that a_loc counts from
    int32_t ar0, nar;         // k-row tasks:  arow_id / arow_start [ar0 .. ar0+nar], start relative to the chunk
    int32_t br0, nbr;         // k'-row tasks
    int32_t q0, nq;           // pairs: iq[q0 .. q0+nq)
    int32_t pad0, pad1;       // pad0: first element of the chunk's permutation / 4 (starts are multiples of 4)
};
struct StreamTile {
    int32_t c0, nc;           // chunk range
    int32_t a_row0, a_rows, b_row0, b_rows;
    int32_t a_slot, b_slot;
    int32_t flags;            // as TileHdr
    int32_t pad;
};
struct StreamHost {
    int32_t Ra = 0, Rb = 0, nblk = 0, nrows = 0, ncta = 0, rf = 0;
    std::vector<int32_t> blk_row0, row_state, state_row, state_blk;
    std::vector<double> w;
    std::vector<uint32_t> code;
    std::vector<uint16_t> perm;                 // per chunk (padded to a multiple of 4): chunk-local entry index, sorted by k' row
    std::vector<uint16_t> arow_id, arow_start;  // per k-row task (+1 sentinel per chunk in arow_start)
    std::vector<uint16_t> brow_id, brow_start;
    std::vector<uint32_t> iq;                   // per (chunk, pair)
    std::vector<StreamChunk> chunks;
    std::vector<StreamTile> tiles;
    std::vector<int32_t> order;                 // tiles by descending work: the order in which CTAs take them
    std::vector<TileCta> ctas;                  // shares used to cut the tiles (host only)
    std::vector<int64_t> slot_off;
    std::vector<int32_t> slot_row0, slot_rows, blk_ent_ptr;
    std::vector<int64_t> blk_ent_off;
    int64_t part_rows = 0;
    bool supported = false;
    std::string why;
};
int build_stream(const ephc_problem *p, const Dims &d, const Canonical &c, int ncta, StreamHost &t, std::string &err);

// ---- resident-tile store (variant 3, collision / RK stages) -----------------------------------------------------
// Every weight is stored ONCE, with the channel's first end a = (n,k) as its owner and the second end b = (m,k+q) as
// its partner; the kind rides in the sign of the stored weight (emission +w, absorption -w; weights are positive):
//     T = |ws| (f_a - f_b) N + ws (x - f_a f_b),  x = f_a (ws > 0) or f_b (ws < 0);   I[a] -= T,   I[b] += T
// which is w F_em resp. w F_abs of Eq. 2 (reading R-1).
// Compact rows are cut into strips of Ra rows; a tile holds the entries between one strip (A rows, the a ends) and a
// range of rows after it (B rows, the b ends), or inside the strip (diagonal tile), sized so that TWO tile images fit
// in shared memory: an image is one contiguous, 16-byte aligned blob that the CTA fetches with bulk copies (TMA) one
// tile ahead and then works on in place.  Consecutive tiles of a strip form a run: the strip's accumulators stay in
// shared memory for the whole run.  The tiles in strip-major order are cut into one contiguous share of equal work
// per CTA and are stored in that order.  Inside an image the work is laid out in SLABS of 32 lanes x H columns,
// column-major (element j of lane l at base + 32 j + l: every warp access is one coalesced shared-memory wavefront):
//   phase 1 (paper step 2): the entries of an a row are cut into pieces of at most Hcap entries, the pieces are
//            sorted by descending length (pieces of one row adjacent) and dealt 32 per slab; a lane walks its piece with
//            f_a in a register.  The entries of one (a, b) state pair inside a piece -- a COMBO: its modes and kinds --
//            are adjacent; the lane sums |ws| N, the emission and the absorption weights over the combo and forms ONE
//            term T at its last entry (bit 0 of the code), written over that entry's weight:
//                T = (f_a - f_b) sum|ws|N + (f_a - f_a f_b) sum_em ws + (f_b - f_a f_b) sum_abs ws.
//            Shorter lanes are padded with w = 0 entries.  Lanes of a slab that share a row (flag "multi") are combined
//            with a segmented warp-shuffle reduction before the first of them subtracts the sum from the row's
//            accumulator in shared memory.
//   phase 2 (paper step 3): the same slab layout over the b rows: perm[] holds, per (slab, column, lane), the position
//            of a term T of that row (padding points at a zero behind the entries); the sum of a B row goes straight
//            to the tile's partial-sum slot in global memory (every B row of the tile has a lane, rows without
//            entries store 0), on a diagonal tile it is added to the strip's accumulator.
// One owner per row and phase, fixed order, no atomics.  The slabs of a phase are dealt to the warps of the CTA by the
// host (longest first, to the least loaded warp) and stored warp by warp: warp w takes slabs wptr[w] .. wptr[w+1].
struct ResTile {           // 120 bytes (device directory)
    int64_t blob_off;      // byte offset of the image in the blob array (multiple of 128)
    int32_t blob_bytes;    // multiple of 16
    int32_t ne;            // weights (real entries)
    int32_t ne_pad;        // phase-1 positions = 32 * sum of the slab heights; X[ne_pad] is the zero that padding reads
    int32_t ng_pad;        // phase-2 positions
    int32_t nslab1, nslab2;
    int32_t q0, nq;        // pairs: iqn[q0 .. q0+nq) = iq * nnu of the tile's pairs
    int32_t nq_next;       // pairs of the next tile of the same CTA: their iq * nnu ride in this image (section nxt)
    int32_t b_row0, b_rows;// B rows (b_rows = 0 on a diagonal tile)
    int32_t b_slot;        // partial-sum slot of the B rows (-1 on a diagonal tile)
    int32_t a_row0, a_rows, a_slot;  // the run's strip and its partial-sum slot
    int32_t flags;         // bit 0: first tile of its run, bit 1: last tile of its run
    // byte offsets of the sections inside the image (= inside the tile buffer), each 16-byte aligned; the code section
    // is at offset 0 and w comes last so that the zero and then the N rows can follow it in shared memory
    uint32_t o_perm, o_srow1, o_shdr1, o_srow2, o_shdr2, o_wptr, o_nxt, o_w;
    uint32_t a_off, b_off; // first element of the A / B slot in the partial-sum buffer
    uint32_t o_sn_next;    // where the N rows of the next tile of the same CTA go in ITS buffer (res_o_sn of that tile)
    int32_t ncombo;        // terms T (one per combo = run of a lane's entries with the same partner): what phase 2 gathers
};
static_assert(sizeof(ResTile) == 120 && sizeof(ResTile) / 4 <= 32, "ResTile is copied word by word by one warp");
constexpr int kResTileWords = sizeof(ResTile) / 4;
// slab header (uint32): first position / 32 (10 bits) | height H << 10 (9 bits) | multi << 31
constexpr uint32_t kResHdrHShift = 10, kResHdrHMask = 0x1ff, kResHdrMulti = 0x80000000u;
constexpr int kResHMax = 511;
constexpr uint16_t kResNoRow = 0xffff;  // lane without a piece
constexpr int kResWarpMax = 32;         // consumer warps per CTA
struct ResRun {            // host only: consecutive tiles of one strip (indices into the scheduled tile sequence)
    int32_t t0, nt;
    int32_t a_row0, a_rows, a_slot;
    int32_t cta;
};
inline int32_t res_al16(int32_t x) { return (x + 15) & ~15; }
// fills the section offsets and blob_bytes of D from its counts (code section first, at offset 0)
inline void res_set_layout(ResTile &D, int nwarp) {
    D.o_perm = (uint32_t)res_al16(4 * D.ne_pad);
    D.o_srow1 = D.o_perm + (uint32_t)res_al16(2 * D.ng_pad);
    D.o_shdr1 = D.o_srow1 + (uint32_t)res_al16(2 * 32 * D.nslab1);
    D.o_srow2 = D.o_shdr1 + (uint32_t)res_al16(4 * D.nslab1);
    D.o_shdr2 = D.o_srow2 + (uint32_t)res_al16(2 * 32 * D.nslab2);
    D.o_wptr = D.o_shdr2 + (uint32_t)res_al16(4 * D.nslab2);
    D.o_nxt = D.o_wptr + (uint32_t)res_al16(2 * 2 * (nwarp + 1));
    D.o_w = D.o_nxt + (uint32_t)res_al16(4 * D.nq_next);
    D.blob_bytes = (int32_t)D.o_w + res_al16(8 * D.ne_pad);
}
// the N rows of the tile's pairs follow the zero in shared memory
inline uint32_t res_o_sn(const ResTile &D) { return (uint32_t)res_al16((int32_t)D.o_w + 8 * (D.ne_pad + 1)); }
// shared memory a tile needs behind the f / accumulator arrays: image, the zero, N rows of its pairs
inline int64_t res_tile_smem(const ResTile &D, int nnu) { return (int64_t)res_o_sn(D) + 8 * (int64_t)D.nq * nnu; }
constexpr int kResSlotMax = 8192;     // N slots (pair * nnu + mode) per tile: slot * 8 fits the 16-bit field of the code
constexpr int kResRowMax = 8192;      // rows (A + B) per tile: row * 8 fits the 16-bit field of the code
constexpr int kResXMax = 32767;       // positions per tile (10-bit slab base in units of 32; uint16 perm)
struct ResHost {
    int32_t Ra = 0, RbMax = 0, Rcap = 0, rf = 0, nblk = 0, nrows = 0, nnu = 0, ncta = 0, nwarp = 0;
    int64_t smem_tile = 0;            // largest res_tile_smem of any tile
    int64_t smem_cap = 0;             // shared-memory budget per CTA the store was built for
    std::vector<int32_t> blk_row0, row_state, state_row, state_blk;
    std::vector<unsigned char> blob;  // all tile images, in schedule order
    std::vector<uint32_t> iqn;        // per (tile, pair): iq * nnu
    std::vector<ResTile> tiles;       // in schedule order: the tiles of CTA c are tiles[cta_ptr[c] .. cta_ptr[c+1])
    std::vector<int32_t> cta_ptr;
    std::vector<double> tile_work;    // cost-model work of every tile (storage order)
    std::vector<ResRun> runs;
    std::vector<int64_t> slot_off;
    std::vector<int32_t> slot_row0, slot_rows, blk_ent_ptr;
    std::vector<int64_t> blk_ent_off;
    int64_t part_rows = 0, nent = 0, nent_pad = 0, ngather_pad = 0, nslab = 0;
    bool supported = false;
    std::string why;
};
// bytes of res_kernel's dynamic shared memory: strip accumulators, three directory entries, two tile buffers
// (f of the A and B rows, image + zero + N rows)
inline int64_t res_buf_bytes(int Rcap, int64_t smem_tile) { return ((int64_t)8 * Rcap + smem_tile + 127) & ~(int64_t)127; }
inline int64_t res_fixed_bytes(int Ra) { return ((int64_t)8 * Ra + 3 * (int64_t)sizeof(ResTile) + 127) & ~(int64_t)127; }
inline int64_t res_smem_total(int Ra, int Rcap, int64_t smem_tile) { return res_fixed_bytes(Ra) + 2 * res_buf_bytes(Rcap, smem_tile); }
int build_res(const ephc_problem *p, const Dims &d, const Canonical &c, int ncta, int64_t smem_cap, int nwarp, ResHost &t,
              std::string &err);
int res_reschedule(ResHost &t, const std::vector<double> &cost, std::string &err);

}  // namespace ephc
