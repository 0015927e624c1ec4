// cc_schedule.cpp -- builds the column-cache schedule (cc_schedule.hpp) by simulating, per CTA,
// the reference stream of its patches against a pool of n_slots shared-memory slots.
#include "cc_schedule.hpp"

#include <algorithm>
#include <atomic>
#include <unordered_map>

namespace icon {
namespace {

constexpr int kRefs = SID_PAD;            // 46 column slots per patch: 36 vn, then 10 w (the use mask says which a mode reads)
constexpr int kFirstCell = SID_T0;        // id slots >= this are cell (w) columns
constexpr int32_t kNever = 0x7fffffff;

struct CtaResult {
    std::vector<CcStep> steps;
    std::vector<CcLoad> loads;
    int64_t n_sync = 0, n_vn = 0, n_w = 0, n_copies = 0;
    bool ok = true;
};

inline uint64_t key_of(int slot_in_patch, int32_t id) {
    return ((uint64_t)(uint32_t)id << 1) | (slot_in_patch >= kFirstCell ? 1u : 0u);
}

void simulate_cta(const ScTables& sc, const int64_t* order, int64_t pb, int64_t pe, int n_slots, const CcGeometry& geom, int kCcGroup,
                  int max_depth, uint64_t use, uint16_t* patch_slots, CtaResult& r) {
    const int64_t n_steps = (pe - pb + kCcGroup - 1) / kCcGroup;
    // pass 1: the distinct columns of every step
    std::vector<std::vector<uint64_t>> keys((size_t)n_steps);
    for (int64_t s = 0; s < n_steps; ++s) {
        auto& ks = keys[(size_t)s];
        const int64_t p0 = pb + s * kCcGroup, p1 = std::min(pe, p0 + kCcGroup);
        for (int64_t p = p0; p < p1; ++p)
            for (int i = 0; i < kRefs; ++i)
                if ((use >> i) & 1) ks.push_back(key_of(i, sc.ids[(size_t)order[p] * kScIdWords + i]));
        std::sort(ks.begin(), ks.end());
        ks.erase(std::unique(ks.begin(), ks.end()), ks.end());
    }
    // pass 2 (backward): the next step that uses each of them
    std::vector<std::vector<int32_t>> next_use((size_t)n_steps);
    {
        std::unordered_map<uint64_t, int32_t> seen;
        seen.reserve(4096);
        for (int64_t s = n_steps - 1; s >= 0; --s) {
            const auto& ks = keys[(size_t)s];
            auto& nu = next_use[(size_t)s];
            nu.resize(ks.size());
            for (size_t i = 0; i < ks.size(); ++i) {
                auto it = seen.find(ks[i]);
                nu[i] = it == seen.end() ? kNever : it->second;
                seen[ks[i]] = (int32_t)s;
            }
        }
    }
    // pass 3 (forward): residency
    std::unordered_map<uint64_t, int32_t> resident;      // key -> slot
    resident.reserve((size_t)n_slots * 2);
    std::vector<uint64_t> slot_key((size_t)n_slots, ~0ull);
    std::vector<int32_t> slot_last((size_t)n_slots, -1000), slot_next((size_t)n_slots, kNever);
    std::vector<int32_t> slot_loaded((size_t)n_slots, -1000);      // the step whose copies filled the slot
    std::vector<int32_t> cand;
    std::vector<size_t> miss;
    std::unordered_map<uint64_t, int32_t> step_slot;     // key -> slot, for this step's patches
    r.steps.reserve((size_t)n_steps);
    for (int64_t s = 0; s < n_steps; ++s) {
        const auto& ks = keys[(size_t)s];
        const auto& nu = next_use[(size_t)s];
        step_slot.clear();
        miss.clear();
        for (size_t i = 0; i < ks.size(); ++i) {
            auto it = resident.find(ks[i]);
            if (it == resident.end()) {
                miss.push_back(i);
            } else {
                slot_last[(size_t)it->second] = (int32_t)s;
                slot_next[(size_t)it->second] = nu[i];
                step_slot[ks[i]] = it->second;
            }
        }
        int depth = max_depth;
        for (; depth >= 1; --depth) {
            cand.clear();
            for (int32_t q = 0; q < n_slots; ++q)
                if (slot_last[(size_t)q] <= (int32_t)s - depth) cand.push_back(q);
            if (cand.size() >= miss.size()) break;
        }
        const int sync = depth < max_depth;
        if (cand.size() < miss.size()) {
            r.ok = false;
            return;
        }
        // What this step loads: its misses (key, next use after this step)
        struct Item { uint64_t key; int32_t next; };
        std::vector<Item> items;
        items.reserve(miss.size());
        for (size_t mi : miss) items.push_back(Item{ks[mi], nu[mi]});
        std::sort(items.begin(), items.end(), [](const Item& a, const Item& b2) {
            if ((a.key & 1) != (b2.key & 1)) return (a.key & 1) < (b2.key & 1);
            return (a.key >> 1) < (b2.key >> 1);
        });
        // grouped into runs of consecutive column ids of one kind
        struct Run { int kind; uint32_t id; int len; size_t first; };   // first = index into `items`
        std::vector<Run> runs;
        for (size_t m = 0; m < items.size(); ++m) {
            const int kind = (int)(items[m].key & 1);
            const uint32_t id = (uint32_t)(items[m].key >> 1);
            const bool mergeable = geom.stride_bytes[kind] == geom.slot_bytes;
            if (!runs.empty() && mergeable && runs.back().kind == kind && runs.back().len < kCcMaxRun &&
                runs.back().id + (uint32_t)runs.back().len == id) {
                ++runs.back().len;
            } else {
                runs.push_back(Run{kind, id, 1, m});
            }
        }
        // Place the runs, longest first: a window of `len` consecutive evictable slots whose
        // earliest next use is farthest (Belady on the window; empty slots count as never used
        // again). A run that finds no window is split in two.
        std::vector<char> evictable((size_t)n_slots, 0);
        for (int32_t q : cand) evictable[(size_t)q] = 1;
        auto worth = [&](int32_t q) { return slot_key[(size_t)q] == ~0ull ? kNever : slot_next[(size_t)q]; };
        CcStep st;
        st.load_begin = (uint32_t)r.loads.size();
        st.n_loads = 0;
        st.n_patches = (uint8_t)(std::min(pe, pb + (s + 1) * kCcGroup) - (pb + s * kCcGroup));
        st.depth = (uint8_t)depth;
        st.tx16 = 0;
        st.ahead_begin = 0;
        std::vector<Run> work(runs);
        std::stable_sort(work.begin(), work.end(), [](const Run& a, const Run& b2) { return a.len > b2.len; });
        for (size_t w = 0; w < work.size(); ++w) {
            const Run run = work[w];
            int32_t best = -1, best_worth = -1;
            int32_t streak = 0;
            for (int32_t q = 0; q < n_slots; ++q) {
                streak = evictable[(size_t)q] ? streak + 1 : 0;
                if (streak >= run.len) {
                    int32_t wmin = kNever;
                    for (int32_t t = q - run.len + 1; t <= q; ++t) wmin = std::min(wmin, worth(t));
                    if (wmin > best_worth) {
                        best_worth = wmin;
                        best = q - run.len + 1;
                    }
                }
            }
            if (best < 0) {
                if (run.len == 1) {          // cannot happen: |cand| >= |miss|
                    r.ok = false;
                    return;
                }
                const int h = run.len / 2;
                work.push_back(Run{run.kind, run.id, h, run.first});
                work.push_back(Run{run.kind, run.id + (uint32_t)h, run.len - h, run.first + (size_t)h});
                continue;
            }
            for (int t = 0; t < run.len; ++t) {
                const int32_t q = best + t;
                const Item& it = items[run.first + (size_t)t];
                const uint64_t k = it.key;
                if (slot_key[(size_t)q] != ~0ull) resident.erase(slot_key[(size_t)q]);
                slot_key[(size_t)q] = k;
                slot_last[(size_t)q] = (int32_t)s;
                slot_next[(size_t)q] = it.next;
                slot_loaded[(size_t)q] = (int32_t)s;
                evictable[(size_t)q] = 0;
                resident[k] = q;
                step_slot[k] = q;
            }
            const int bytes = (run.len - 1) * geom.stride_bytes[run.kind] + geom.col_bytes[run.kind];
            CcLoad ld;
            ld.id = run.id;
            ld.slot = (uint16_t)best;
            ld.bytes16_kind = (uint16_t)((bytes / 16) | (run.kind << 15));
            r.loads.push_back(ld);
            ++st.n_loads;
            st.tx16 += (uint32_t)(bytes / 16);
            if (run.kind) r.n_w += run.len; else r.n_vn += run.len;
            ++r.n_copies;
        }
        r.n_sync += sync;
        r.steps.push_back(st);
        const int64_t p0 = pb + s * kCcGroup, p1 = std::min(pe, p0 + kCcGroup);
        for (int64_t p = p0; p < p1; ++p) {
            uint16_t* o = patch_slots + (size_t)p * kCcSlotWords;
            // bit r of the mask: a column of this patch was loaded by step s-r, whose copies may still
            // be in flight when step s starts (copies of different steps complete in any order)
            uint16_t mask = 0;
            for (int i = 0; i < kRefs; ++i) {
                if (!((use >> i) & 1)) {          // a column this mode never reads
                    o[i] = 0;
                    continue;
                }
                const int32_t q = step_slot[key_of(i, sc.ids[(size_t)order[p] * kScIdWords + i])];
                o[i] = (uint16_t)q;
                const int64_t age = s - slot_loaded[(size_t)q];
                if (age > 0 && age < max_depth) mask |= (uint16_t)(1u << age);
            }
            for (int i = kRefs; i < kCcSlotWords; ++i) o[i] = 0;
            o[kCcMaskWord] = mask;
        }
    }
}

}  // namespace

std::string build_cc_schedule(const ScTables& sc, int n_ctas, int n_slots, const CcGeometry& geom, int group, int depth,
                              int tile, uint64_t use, CcSchedule& out) {
    const int kCcGroup = group;
    const int64_t np = sc.n_patches;
    if (np <= 0 || n_ctas <= 0) return "cc schedule: empty grid";
    if (n_slots < kRefs) return "cc schedule: fewer shared-memory slots than one patch needs";
    if (n_slots > 65535) return "cc schedule: slot indices do not fit 16 bits";
    if (geom.slot_bytes % 16 || geom.col_bytes[0] % 16 || geom.col_bytes[1] % 16 || geom.col_bytes[0] > geom.slot_bytes ||
        geom.col_bytes[1] > geom.slot_bytes || (kCcMaxRun - 1) * (int64_t)geom.slot_bytes + geom.slot_bytes > 16 * 32767)
        return "cc schedule: bad column geometry";
    const int64_t max_ctas = (np + kCcGroup - 1) / kCcGroup;
    if (n_ctas > max_ctas) n_ctas = (int)max_ctas;
    out = CcSchedule();
    out.n_ctas = n_ctas;
    out.n_slots = n_slots;
    out.geom = geom;
    out.group = group;
    out.depth = depth;
    out.tile = tile;
    out.use = use;
    out.cta_patch_begin.resize((size_t)n_ctas + 1);
    // whole steps per CTA, spread evenly
    const int64_t total_steps = max_ctas;
    for (int b = 0; b <= n_ctas; ++b)
        out.cta_patch_begin[(size_t)b] = std::min(np, (total_steps * b / n_ctas) * kCcGroup);
    // Work order: position -> patch of sc. tile == 0: generation order, each CTA a contiguous range.
    // tile > 0: tiles of `tile` consecutive patches dealt round-robin, CTA b walks the tiles b, b+n_ctas,
    // ...: at any time the CTAs work on neighbouring tiles, so a halo column that two tiles share is
    // fetched twice within microseconds and the second fetch hits the L2 instead of HBM.
    out.patch_order.resize((size_t)np);
    if (tile > 0) {
        if (tile % group) return "cc schedule: tile must be a multiple of the group";
        const int64_t nt = (np + tile - 1) / tile;
        if (n_ctas > nt) n_ctas = (int)nt;
        out.n_ctas = n_ctas;
        out.cta_patch_begin.assign((size_t)n_ctas + 1, 0);
        int64_t pos = 0;
        for (int b = 0; b < n_ctas; ++b) {
            for (int64_t t = b; t < nt; t += n_ctas)
                for (int64_t p = t * tile; p < std::min(np, (t + 1) * tile); ++p) out.patch_order[(size_t)pos++] = p;
            out.cta_patch_begin[(size_t)b + 1] = pos;
        }
    } else {
        for (int64_t p = 0; p < np; ++p) out.patch_order[(size_t)p] = p;
    }
    out.patch_slots.assign((size_t)np * kCcSlotWords, 0);
    std::vector<CtaResult> res((size_t)n_ctas);
#pragma omp parallel for schedule(dynamic, 1)
    for (int b = 0; b < n_ctas; ++b)
        simulate_cta(sc, out.patch_order.data(), out.cta_patch_begin[(size_t)b], out.cta_patch_begin[(size_t)b + 1], n_slots, geom, group,
                     depth, use, out.patch_slots.data(), res[(size_t)b]);
    out.cta_step_begin.assign((size_t)n_ctas + 1, 0);
    size_t n_loads = 0;
    for (int b = 0; b < n_ctas; ++b) {
        if (!res[(size_t)b].ok) return "cc schedule: one step needs more columns than there are shared-memory slots";
        out.cta_step_begin[(size_t)b + 1] = out.cta_step_begin[(size_t)b] + (int64_t)res[(size_t)b].steps.size();
        n_loads += res[(size_t)b].loads.size();
    }
    if (n_loads > 0xffffffffull) return "cc schedule: load list too long";
    out.steps.reserve((size_t)out.cta_step_begin[(size_t)n_ctas]);
    out.loads.reserve(n_loads);
    for (int b = 0; b < n_ctas; ++b) {
        const uint32_t base = (uint32_t)out.loads.size();
        for (CcStep st : res[(size_t)b].steps) {
            st.load_begin += base;
            out.steps.push_back(st);
        }
        out.loads.insert(out.loads.end(), res[(size_t)b].loads.begin(), res[(size_t)b].loads.end());
        out.n_sync_steps += res[(size_t)b].n_sync;
        out.n_vn_loads += res[(size_t)b].n_vn;
        out.n_w_loads += res[(size_t)b].n_w;
        out.n_copies += res[(size_t)b].n_copies;
        res[(size_t)b] = CtaResult();
    }
    for (int b = 0; b < n_ctas; ++b) {
        const int64_t s0 = out.cta_step_begin[(size_t)b], s1 = out.cta_step_begin[(size_t)b + 1];
        for (int64_t i = s0; i < s1; ++i)
            out.steps[(size_t)i].ahead_begin = out.steps[(size_t)std::min(i + kCcAhead, s1 - 1)].load_begin;
    }
    // every producer lane may read one entry of a step's first round without a bounds check
    CcLoad zero;
    zero.id = 0; zero.slot = 0; zero.bytes16_kind = 0;
    out.loads.insert(out.loads.end(), (size_t)32 * kCcMaxProducers, zero);
    return std::string();
}

}  // namespace icon
