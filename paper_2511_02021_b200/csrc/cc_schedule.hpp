// cc_schedule.hpp -- host-built schedule of the COLUMN-CACHE tendency kernel (kernels_cc.cu;
// internal header).
//
// The kernel keeps whole vn / w columns in shared memory ("slots") and fills them with bulk
// asynchronous copies (cp.async.bulk, the 1-D TMA path) issued by a producer warp; eight consumer
// warps each finish one self-contained patch (sc_tables.hpp) per STEP from those slots. Which
// column sits in which slot at which step is decided HERE, on the host, once per grid: the work
// order of every CTA is fixed (a contiguous range of the generation order), so the whole future
// of the reference stream is known and the replacement is Belady's (evict the column whose next
// use is farthest). The device never searches or hashes anything: a step is a list of
// (column id, slot) loads plus, per patch, the slot of each of its 43 columns.
//
// Pipeline rule the schedule guarantees (kernels_cc.cu relies on it): the loads of step s only
// overwrite slots whose last reader ran in a step <= s-2, so they can be in flight while step
// s-1 computes; a step flagged `sync` may also overwrite slots last read in step s-1 and the
// producer waits for that step to drain first (rare: only when two consecutive steps together
// need more columns than there are slots).
#pragma once
#include <cstdint>
#include <string>
#include <vector>

#include "sc_tables.hpp"

namespace icon {

// pipeline shapes of the kernel (kernels_cc.cu): consumer warps, patches per step, ring depth.
// kCcProducers producer warps (one warpgroup) are added to `warps`; the CTA is launched with
// 168 registers per thread and re-balances them with setmaxnreg: producers keep
// CcWarps<T>::producer_regs, consumers grow to CcWarps<T>::consumer_regs
// (the pool is what the launch allocated: 384 * 168 = (4 * 56 + 8 * 224) * 32 = 64512 registers).
// 8-byte columns: 4 producer warps with 56 registers, 8 consumer warps with 224 (launch: 384 threads x 168).
// 4-byte columns: the consumers need fewer registers and the columns are half as long, i.e. twice the copies per byte,
// so a second producer warpgroup issues them: 8 producer warps with 40 registers, consumers 216 (launch: 512 x 128).
// One level per lane (L = 1, nlev <= 31) is the same case: short columns, light consumers.
template <class T, int L>
struct CcWarps {
    static constexpr bool light = sizeof(T) == 4 || L == 1;
    static constexpr int producers = light ? 8 : 4;
    static constexpr int producer_regs = light ? 40 : 56;
    static constexpr int consumer_regs = light ? 216 : 224;
};
constexpr int kCcMaxProducers = 8;
constexpr int kCcAhead = 3;              // steps the producers read the schedule ahead; `loads` is padded for it
struct CcShape {
    int warps, group, depth;
};
constexpr int kCcNumShapes = 2;
#ifndef CC_S1_G          // shape 1 can be re-defined at build time for pipeline-shape experiments (ICON_NVCC_EXTRA)
#define CC_S1_G 4
#define CC_S1_D 3
#endif
constexpr CcShape kCcShapes[kCcNumShapes] = {{8, 2, 6}, {8, CC_S1_G, CC_S1_D}};
inline const CcShape& cc_shape(int i) { return kCcShapes[i >= 0 && i < kCcNumShapes ? i : 0]; }
constexpr int kCcBarrierBytes = 512;    // the mbarriers
constexpr int kCcOutCols = 3;            // ddt_vn staging columns per consumer warp (one store batch)
// a patch record on the device = kScCoefWords coefficients (T), then kCcRecordIds int32 (user ids of
// the outputs), then kCcSlotWords uint32 byte offsets of the slots; c_lin is
// stored halved there (the kernel forms w(k) + w(k+1) = 2 w_f(k))
constexpr int kCcSlotWords = 48;     // per patch: 43 slots (order of sc_tables.hpp id slots), mask, pad
constexpr int kCcMaskWord = 43;      // bit r set: one of the 43 columns was loaded by step s-r (0 < r < depth)
constexpr int kCcRecordIds = 16;     // int32: owned edges i0 i1 i2 b0 b2 b4, cells T0..T3, owned vertices ab bc ca a b c (-1 = not ours)
constexpr int kCcRecordTail = 4 * kCcRecordIds + 4 * kCcSlotWords;
// lanes past the end of a column read up to 3 * 32 levels * 8 bytes beyond their slot: readable pad after the last slot
constexpr int kCcSlotTailPad = 768;

struct CcStep {                      // 16 bytes
    uint32_t load_begin;             // first entry of this step in `loads`
    uint16_t n_loads;                // bulk copies of this step (a copy moves a run of 1..kCcMaxRun columns)
    uint8_t n_patches;               // 1..group
    uint8_t depth;                   // the loads may be issued once step s-depth has drained (1..schedule depth)
    uint32_t tx16;                   // bytes / 16 those copies deliver (patch records not included)
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
    std::vector<int64_t> patch_order;        // [n_patches] work position -> patch of the ScTables
    std::vector<int64_t> cta_patch_begin;    // [n_ctas + 1], work positions
    std::vector<int64_t> cta_step_begin;     // [n_ctas + 1]
    std::vector<CcStep> steps;
    std::vector<CcLoad> loads;
    std::vector<uint16_t> patch_slots;       // [work position][kCcSlotWords], slot index
    // statistics (icon_grid_worklist_stats, tests)
    int64_t n_sync_steps = 0, n_vn_loads = 0, n_w_loads = 0;   // columns loaded
    int64_t n_copies = 0;                                      // bulk copies (runs)
};

// Returns an empty string on success, else an error message (e.g. too few slots for one step).
// `tile`: 0 = every CTA walks a contiguous range of the generation order; > 0 = tiles of that many
// patches are dealt round-robin to the CTAs (CcSchedule::patch_order).
std::string build_cc_schedule(const ScTables& sc, int n_ctas, int n_slots, const CcGeometry& geom, int group, int depth,
                              int tile, CcSchedule& out);

// cc_schedule_check.cpp: replays `cs` as the kernel would and checks the guarantees it relies on
// (independent of the builder). Empty string = valid.
std::string check_cc_schedule(const ScTables& sc, const CcSchedule& cs, int64_t n_edges, int64_t n_cells);

}  // namespace icon
