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
};

// host builder (ephc_build.cu)
int build_canonical(const ephc_problem *p, const Dims &d, Canonical &c, std::string &err);
int build_gather(const ephc_problem *p, const Dims &d, const Canonical &c, GatherHost &g, std::string &err);

}  // namespace ephc
