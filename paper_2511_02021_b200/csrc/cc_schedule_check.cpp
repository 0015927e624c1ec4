// cc_schedule_check.cpp -- replays a column-cache schedule (cc_schedule.hpp) the way the kernel
// executes it and checks the guarantees kernels_cc.cu relies on. Shares nothing with the builder
// but the data structures: it only knows what the DEVICE does with a schedule.
//
//   1. every bulk copy of a step lands in slots [slot, slot + n) inside the pool, n = columns of the run;
//   2. it never overwrites a slot that a patch of the steps s-depth+1 .. s reads (those may still be
//      running, or are this step's own hits), nor a slot that one of those steps filled (its copy may still be in
//      flight);
//   3. after the copies of step s, each of the 43 slots a patch of step s names holds exactly the
//      column (kind, id) its record names;
//   4. the byte count the step header announces (tx16) is the sum of its copies, every copy is a
//      multiple of 16 bytes and stays inside the caller's field rows it was cut from;
//   6. a patch that reads a column filled by one of the last depth-1 steps names that step in its
//      wait mask (bulk copies of different steps complete in any order);
//   5. steps and patches tile the CTA's range without gaps, depth is in 1..schedule depth, and
//      ahead_begin names the list of step s + kCcAhead.
#include "cc_schedule.hpp"

#include <algorithm>
#include <atomic>

namespace icon {

std::string check_cc_schedule(const ScTables& sc, const CcSchedule& cs, int64_t n_edges, int64_t n_cells) {
    const CcGeometry& gm = cs.geom;
    if (cs.n_ctas <= 0 || cs.group <= 0 || cs.depth <= 0) return "check: empty schedule";
    if (cs.cta_patch_begin.front() != 0 || cs.cta_patch_begin.back() != sc.n_patches) return "check: patches not covered";
    if (cs.cta_step_begin.front() != 0 || cs.cta_step_begin.back() != (int64_t)cs.steps.size()) return "check: steps not covered";
    {   // the work order visits every patch exactly once
        if ((int64_t)cs.patch_order.size() != sc.n_patches) return "check: work order has the wrong length";
        std::vector<char> seen((size_t)sc.n_patches, 0);
        for (int64_t p : cs.patch_order) {
            if (p < 0 || p >= sc.n_patches || seen[(size_t)p]) return "check: work order is not a permutation";
            seen[(size_t)p] = 1;
        }
    }
    std::atomic<int> err(0);
#pragma omp parallel for schedule(dynamic, 1)
    for (int b = 0; b < cs.n_ctas; ++b) {
        auto fail = [&](int code) { int z = 0; err.compare_exchange_strong(z, code); };
        const int64_t pb = cs.cta_patch_begin[(size_t)b], pe = cs.cta_patch_begin[(size_t)b + 1];
        const int64_t s0 = cs.cta_step_begin[(size_t)b], s1 = cs.cta_step_begin[(size_t)b + 1];
        if (s1 - s0 != (pe - pb + cs.group - 1) / cs.group) { fail(1); continue; }
        std::vector<int64_t> content((size_t)cs.n_slots, -1);      // key = id * 2 + kind, -1 = nothing
        std::vector<int64_t> last_read((size_t)cs.n_slots, -1000000);
        std::vector<int64_t> loaded_at((size_t)cs.n_slots, -1000000);
        uint32_t expect_begin = s0 < s1 ? cs.steps[(size_t)s0].load_begin : 0;
        for (int64_t s = 0; s < s1 - s0; ++s) {
            const CcStep& st = cs.steps[(size_t)(s0 + s)];
            const int64_t p0 = pb + s * cs.group, p1 = std::min(pe, p0 + cs.group);
            if (st.n_patches != p1 - p0 || st.depth < 1 || st.depth > cs.depth) { fail(2); break; }
            if (st.load_begin != expect_begin) { fail(3); break; }
            expect_begin += st.n_loads;
            const int64_t sa = std::min(s + kCcAhead, s1 - s0 - 1);
            if (st.ahead_begin != cs.steps[(size_t)(s0 + sa)].load_begin) { fail(4); break; }
            // what this step's patches will read (rule 2 also protects this step's own hits)
            for (int64_t p = p0; p < p1; ++p)
                for (int i = 0; i < SID_PAD; ++i) {
                    const int q = cs.patch_slots[(size_t)p * kCcSlotWords + i];
                    if (q >= cs.n_slots) { fail(5); break; }
                }
            if (err) break;
            uint64_t tx = 0;
            for (uint32_t j = 0; j < st.n_loads; ++j) {
                const CcLoad& ld = cs.loads[(size_t)st.load_begin + j];
                const int kind = ld.bytes16_kind >> 15;
                const int64_t bytes = (int64_t)(ld.bytes16_kind & 0x7fff) * 16;
                tx += (uint64_t)bytes;
                if (bytes < gm.col_bytes[kind]) { fail(6); break; }
                const int64_t extra = bytes - gm.col_bytes[kind];
                int64_t n = 1;
                if (extra) {
                    if (gm.stride_bytes[kind] != gm.slot_bytes || extra % gm.stride_bytes[kind]) { fail(7); break; }
                    n += extra / gm.stride_bytes[kind];
                }
                if (n > kCcMaxRun || ld.slot + n > cs.n_slots) { fail(8); break; }
                if ((int64_t)ld.id + n > (kind ? n_cells : n_edges)) { fail(9); break; }
                for (int64_t t = 0; t < n; ++t) {
                    const size_t q = (size_t)ld.slot + (size_t)t;
                    if (last_read[q] > s - st.depth) { fail(10); break; }          // a reader may still be running
                    if (loaded_at[q] > s - st.depth) { fail(15); break; }          // an earlier copy into it may still be in flight
                    content[q] = ((int64_t)ld.id + t) * 2 + kind;
                    loaded_at[q] = s;
                    last_read[q] = -1000000;
                }
                if (err) break;
            }
            if (err) break;
            if (tx != (uint64_t)st.tx16 * 16) { fail(11); break; }
            for (int64_t p = p0; p < p1 && !err; ++p) {
                const unsigned mask = cs.patch_slots[(size_t)p * kCcSlotWords + kCcMaskWord];
                for (int i = 0; i < SID_PAD; ++i) {
                    if (!((cs.use >> i) & 1)) continue;              // a column this mode never reads
                    const size_t q = cs.patch_slots[(size_t)p * kCcSlotWords + i];
                    const int64_t want = (int64_t)sc.ids[(size_t)cs.patch_order[(size_t)p] * kScIdWords + i] * 2 + (i >= SID_T0 ? 1 : 0);
                    if (content[q] != want) { fail(12); break; }
                    last_read[q] = s;
                    // rule 6: a column filled by a step that has not necessarily drained (s-depth < s' < s)
                    // must be named in the patch's wait mask; the kernel waits for that step's barrier too
                    const int64_t age = s - loaded_at[q];
                    if (age > 0 && age < cs.depth && !((mask >> age) & 1u)) { fail(13); break; }
                }
                if (mask & 1u) fail(14);
            }
            if (err) break;
        }
    }
    if (err) return "check: schedule violates rule code " + std::to_string((int)err);
    return std::string();
}

}  // namespace icon
