// cc_schedule.hpp -- host-built schedule of the COLUMN-CACHE tendency kernel (kernels_cc.cu;
// internal header).
//
// The kernel keeps whole vn / w columns in shared memory ("slots") and fills them with bulk
// asynchronous copies (cp.async.bulk, the 1-D TMA path) issued by a warpgroup of producer warps; eight
// consumer warps in two groups each finish one self-contained patch (sc_tables.hpp) per STEP (= four
// patches) from those slots. Which column sits in which slot at which step is decided HERE, on the host,
// once per grid: the work order of every CTA is fixed (tiles of consecutive patches of the generation
// order dealt round-robin to the CTAs), so the whole future of the reference stream is known and the
// replacement is Belady's (evict the column whose next use is farthest). The device never searches or
// hashes anything: a step is a list of (first column id, first slot, bytes) copies plus, per patch, the
// slot of each of its 43 columns.
//
// Pipeline rule the schedule guarantees (kernels_cc.cu relies on it, cc_schedule_check.cpp replays it):
// the loads of step s only overwrite slots whose last reader ran in a step <= s - depth(s), with
// depth(s) = kCcDepth normally (the copies of step s are in flight while the steps s-1 .. s-depth+1
// compute) and smaller (stored per step) only when the steps in flight together need more columns
// than there are slots; the producers issue the copies of step s once step s - depth(s) has drained.
// A patch that reads a column loaded by one of the steps s-1 .. s-kCcDepth+1 names that step in its
// wait mask (copies of different steps complete in any order).
#pragma once
#include <cstdint>
#include <string>
#include <vector>

#include "sc_tables.hpp"

namespace icon {

#ifdef __CUDACC__
#define CC_HD __host__ __device__
#else
#define CC_HD
#endif

// Pipeline shape of the kernel (kernels_cc.cu): kCcWarps consumer warps in groups of kCcGroup (= patches per
// step), ring of kCcDepth steps. Measured against 8/2/6 (two patches per step, ring of six) on B200: config 3
// 5.11 -> 4.91 ms, config 4 4.01 -> 3.38 ms, config 5 12.25 -> 9.84 ms.
constexpr int kCcWarps = 8, kCcGroup = 4, kCcDepth = 3;
// Level mappings (template parameter L of the kernel = values a lane holds per column):
//   L = 3 (33 <= nlev+1 <= 96): one patch per warp, a lane owns levels 2*lane, 2*lane+1 and 64+lane;
//   L = 2 (nlev+1 <= 32): TWO patches per warp, one per half-warp, a lane owns levels 2*(lane%16), 2*(lane%16)+1 --
//         a step is then 8 patches, and every per-patch cost of a warp (coefficient and slot lookups, waits, address
//         arithmetic) is paid once per two patches;
//   L = 6 (4-byte columns, 33 <= nlev+1 <= 96, div / vort mode only): two patches per warp as well, a lane owns the
//         three pairs 32*p + 2*(lane%16), +1 (p = 0, 1, 2). Measured at config 4: div_vort 2.08 -> 1.69 ms and the
//         tendency alone 2.86 -> 2.37 ms, but the fused step 3.39 -> 3.61 ms (the consumers hold per-half ids and
//         pointers besides six values per column and spill 100 bytes at 216 registers; with four producer warps and 232
//         registers everything was slower). The tendency shares its schedule with the fused step, so both keep L = 3.
CC_HD constexpr int cc_patches_per_warp(int L) { return L == 2 || L == 6 ? 2 : 1; }
// Consumer warps of a CTA as a function of the column type and the level mapping: kCcWarps everywhere. The shape is a
// parameter because 4-byte columns were tried with SIXTEEN consumer warps (two groups of eight, eight patches per step,
// 104 registers each, four producer warps; launch 640 x 96): the consumers then spill 96-288 bytes and config 4 measured
// 3.29 ms against 3.37 ms for the fused step and 2.76 against 2.72 ms for the tendency -- the 8-warp kernel is not bound
// by the number of warps a scheduler can pick from (profiles/r02_experiments.md).
CC_HD constexpr int cc_consumer_warps(int elem_bytes, int L) { return (void)elem_bytes, (void)L, kCcWarps; }
CC_HD constexpr int cc_group(int elem_bytes, int L) { return cc_consumer_warps(elem_bytes, L) / 2; }
CC_HD constexpr int cc_patches_per_step(int elem_bytes, int L) { return cc_group(elem_bytes, L) * cc_patches_per_warp(L); }
// Producer warps are added to the consumers; the CTA is launched with the registers of the average warp and
// re-balances them with setmaxnreg: producers keep CcWarps::producer_regs, consumers grow to CcWarps::consumer_regs
// (the pool is what the LAUNCH allocated: 384 * 168 = (4 * 56 + 8 * 224) * 32 = 64512 registers).
// 8-byte columns: 4 producer warps with 56 registers, 8 consumer warps with 224 (launch: 384 threads x 168).
// 4-byte columns: the consumers need fewer registers and the columns are half as long, i.e. twice the copies per byte,
// so a second producer warpgroup issues them: 8 producer warps with 40 registers, consumers 216 (launch: 512 x 128).
// Shallow columns (L = 2, nlev <= 31) are the same case: short columns, light consumers.
// (`wide`: the 16-consumer shape that was tried for 4-byte columns, see cc_consumer_warps; never true now.)
template <class T, int L>
struct CcWarps {
    static constexpr bool light = sizeof(T) == 4 || L == 2;
    static constexpr bool wide = cc_consumer_warps((int)sizeof(T), L) > kCcWarps;
    static constexpr int consumers = cc_consumer_warps((int)sizeof(T), L);
    static constexpr int group = cc_group((int)sizeof(T), L);
    static constexpr int producers = wide ? 4 : light ? 8 : 4;
    static constexpr int producer_regs = light ? 40 : 56;
    static constexpr int consumer_regs = wide ? 104 : light ? 216 : 224;
};
constexpr int kCcMaxProducers = 8;
constexpr int kCcAhead = 3;              // steps the producers read the schedule ahead; `loads` is padded for it
constexpr int kCcBarrierBytes = 512;    // the mbarriers
// What a launch of the kernel produces; each mode has a schedule of its own (DevCcTables::mode).
enum { kCcTend = 0 /* ddt_vn */, kCcStep = 1 /* ddt_vn + div + vort */, kCcDivVort = 2 /* div + vort only */,
       kCcStepW = 3 /* ddt_vn + div + vort + ddt_w (P-19): three more w columns and twelve more coefficients per patch */,
       kCcTendM = 4 /* ddt_vn in its metric form (P-20): 24 more coefficients per patch; the four metric columns of an owned
                       edge are read straight from global memory */,
       kCcWTend = 5 /* ddt_w alone (dycore_w_tendency, P-19): the nine in-patch vn columns and the ten w columns of a patch,
                       compact records of twelve coefficients */ };
// kCcDivVort reads 27 of the 36 vn columns of a patch and no w column, and its records carry only the 52 coefficients it
// needs: geofac_div [4][3], rot of the midpoints [3][6] (+2 pad), rot of the corners [3][6] (+2 pad)
enum { DVF_DIV = 0, DVF_ROT = 12, DVF_XROT = 32, kCcDvCoefWords = 52 };
// kCcWTend: the records carry only SCF_ADV [4][3]
enum { WF_ADV = 0, kCcWCoefWords = 12 };
CC_HD constexpr int cc_coef_words(int mode) {
    return mode == kCcDivVort ? (int)kCcDvCoefWords : mode == kCcWTend ? (int)kCcWCoefWords : mode == kCcTendM ? (int)kScCoefWords : mode == kCcStepW ? (int)SCF_CGRAD : (int)SCF_ADV;
}
// id slots (sc_tables.hpp) a mode reads: bit i of the mask = column i of the patch is needed
constexpr uint64_t cc_use_mask(int mode) {
    if (mode == kCcStepW) return (1ull << SID_PAD) - 1;                  // every column
    if (mode == kCcWTend) return ((1ull << SID_OM0) - 1) | (((1ull << SID_PAD) - 1) & ~((1ull << SID_T0) - 1));      // i0..i2 b0..b5 | all ten cells
    if (mode != kCcDivVort) return (1ull << SID_XW0) - 1;                // 36 vn + 7 w: all but X1 X3 X5
    uint64_t m = (1ull << SID_X0) - 1;                                   // i0..i2, b0..b5, om0..om5, oc0..oc5
    for (int x = 0; x < 3; ++x) m |= 3ull << (SID_X0 + 5 * x + 3);       // n1, n2 of the three corners
    return m;
}
// a patch record on the device = kScCoefWords coefficients (T), then kCcRecordIds int32 (user ids of
// the outputs), then kCcSlotWords uint32 byte offsets of the slots; c_lin is
// stored halved there (the kernel forms w(k) + w(k+1) = 2 w_f(k))
constexpr int kCcSlotWords = 48;     // per patch: 46 slots (order of sc_tables.hpp id slots), mask, pad
constexpr int kCcMaskWord = 46;      // bit r set: one of the patch's columns was loaded by step s-r (0 < r < depth)
constexpr int kCcRecordIds = 16;     // int32: owned edges i0 i1 i2 b0 b2 b4, cells T0..T3, owned vertices ab bc ca a b c (-1 = not ours)
constexpr int kCcRecordTail = 4 * kCcRecordIds + 4 * kCcSlotWords;
// lanes past the end of a column read up to 3 * 32 levels * 8 bytes beyond their slot: readable pad after the last slot
constexpr int kCcSlotTailPad = 768;

struct CcStep {                      // 16 bytes
    uint32_t load_begin;             // first entry of this step in `loads`
    uint16_t n_loads;                // bulk copies of this step (a copy moves a run of 1..kCcMaxRun columns)
    uint8_t n_patches;               // 1..group
    uint8_t depth;                   // the loads may be issued once step s-depth has drained (1..schedule depth)
    uint32_t tx16;                   // bytes / 16 those copies deliver (patch records not included); for the checker
    uint32_t ahead_begin;            // load_begin of step s + kCcAhead of the same CTA (the producers' prefetch)
};

struct CcLoad {                      // 8 bytes: one bulk copy
    uint32_t id;                     // user id of the first edge (vn) or cell (w) column of the run
    uint16_t slot;                   // first slot; the run fills consecutive slots
    uint16_t bytes16_kind;           // bit 15: 0 = vn, 1 = w; bits 0..14: bytes / 16 of the copy
};

// Byte geometry of the columns the schedule is built for. A run of n columns with consecutive ids
// is one copy of (n-1)*stride + col bytes into n consecutive slots; that needs slot_bytes == stride,
// so runs longer than 1 are only formed for a kind whose stride equals slot_bytes.
struct CcGeometry {
    int slot_bytes;                  // multiple of 16
    int col_bytes[2];                // bytes copied for one vn / w column (multiple of 16)
    int stride_bytes[2];             // distance of consecutive vn / w columns in the caller's field
};
constexpr int kCcMaxRun = 8;

struct CcSchedule {
    int n_ctas = 0, n_slots = 0;
    int group = 0;                           // patches per step
    int depth = 0;                           // steps a load may run ahead of its readers (pipeline depth)
    CcGeometry geom = {0, {0, 0}, {0, 0}};
    int tile = 0;                            // patches per round-robin tile (0 = contiguous ranges)
    uint64_t use = 0;                        // cc_use_mask the schedule was built for
    std::vector<int64_t> patch_order;        // [n_patches] work position -> patch of the ScTables
    std::vector<int64_t> cta_patch_begin;    // [n_ctas + 1], work positions
    std::vector<int64_t> cta_step_begin;     // [n_ctas + 1]
    std::vector<CcStep> steps;
    std::vector<CcLoad> loads;
    std::vector<uint16_t> patch_slots;       // [work position][kCcSlotWords], slot index
    // statistics (icon_grid_cc_schedule_check, tests)
    int64_t n_sync_steps = 0, n_vn_loads = 0, n_w_loads = 0;   // columns loaded
    int64_t n_copies = 0;                                      // bulk copies (runs)
};

// Returns an empty string on success, else an error message (e.g. too few slots for one step).
// `tile`: 0 = every CTA walks a contiguous range of the generation order; > 0 = tiles of that many
// patches are dealt round-robin to the CTAs (CcSchedule::patch_order).
// `use` = cc_use_mask(mode): the columns of a patch the kernel reads in that mode (slots of unused columns stay 0).
std::string build_cc_schedule(const ScTables& sc, int n_ctas, int n_slots, const CcGeometry& geom, int group, int depth,
                              int tile, uint64_t use, CcSchedule& out);

// cc_schedule_check.cpp: replays `cs` as the kernel would and checks the guarantees it relies on
// (independent of the builder). Empty string = valid.
std::string check_cc_schedule(const ScTables& sc, const CcSchedule& cs, int64_t n_edges, int64_t n_cells);

}  // namespace icon
