// kernels_cc.cu -- column-cache kernel for the velocity tendency and, fused
// into the same pass on request, divergence and vorticity (S1, S2: dycore_step), sm_100a. Six modes (template
// parameter MODE, cc_schedule.hpp): kCcTend = ddt_vn (dycore_velocity_tendencies), kCcStep = ddt_vn + div + vort
// (dycore_step), kCcDivVort = div + vort alone from the 27 vn columns they need (dycore_div_vort), kCcStepW = kCcStep
// plus the vertical-wind tendency ddt_w (dycore_step_w, reading P-19), kCcWTend = ddt_w alone (dycore_w_tendency) from the
// nine in-patch vn columns and the ten w columns of a patch, kCcTendM = ddt_vn in its metric form
// (dycore_velocity_tendencies_metric, reading P-20).
//
// One warp finishes one self-contained patch (sc_tables.hpp: four sibling cells, six owned edges,
// 36 vn + 7 w columns, no exchange between warps), lanes = levels. The vn / w columns do not come
// through the L1: PRODUCER warps (one warpgroup, setmaxnreg down) move whole columns from HBM into
// shared-memory slots with bulk asynchronous copies (cp.async.bulk = the 1-D TMA path, completion on
// an mbarrier), following a schedule the host computed once per grid (cc_schedule.hpp: which columns
// into which slots at which step, Belady replacement, consecutive ids merged into one copy). Eight
// CONSUMER warps (setmaxnreg up) read the slots:
//
//   * every column crosses L2 -> SM once per residency instead of once per patch that touches it
//     (~15 instead of 43 column fetches per patch), and the fetches are in flight one or more steps
//     ahead of their readers without holding a single register;
//   * a lane owns L = 3 levels of a column, the PAIR 2*lane, 2*lane+1 and the single level 64+lane
//     (nlev <= 31: two patches per warp, see cc_schedule.hpp): a coefficient / slot lookup, which is warp-uniform, is paid once
//     per 96 levels; a column is read with one 16-byte and one 8-byte conflict-free shared-memory load
//     per lane, and an output column leaves STRAIGHT FROM REGISTERS with one 16-byte and one 8-byte
//     coalesced streaming store -- no transposition through shared memory (the previous mapping, three
//     consecutive levels per lane, paid 12 L1 wavefronts per output column for it, 144 of ~740 per
//     patch); the vertical stencil (S6) costs two shuffles up and two down per column (inside the pair
//     the neighbour level is in the lane's own registers);
//   * kCcStep: div of the patch's four cells comes from the nine in-patch columns, and the sums zm, zc
//     the tendency needs ARE half the vorticity at the patch's three midpoint and three corner
//     vertices; every vertex of the grid is one of those for some patch, the lowest patch stores it.
//
// Why a warpgroup of producers: issuing one bulk copy is a ~100-cycle serial chain on the uniform datapath
// (R2UR / ELECT / UBLKCP), and an SM accepts one copy per ~31 cycles at best
// (profiles/r01_bulk_copy_microbench.md), so the issue is spread over four (eight) warps and runs of
// columns are merged. Why the warp index goes through a shuffle: it makes the role / range branches
// uniform for the compiler, which removed a third of the instructions (divergence handling around
// every shuffle) -- the kernel had outgrown the instruction cache.
//
// Synchronisation: ring of NB barrier pairs, full[s % NB] (one arrival per producer warp, each
// announcing the bytes of its share of step s before issuing them; the copies complete it) and done[s % NB] (one arrival per
// consumer warp of the step's group). The schedule guarantees that the loads of step s only overwrite
// slots last read in a step <= s-depth (depth <= D stored per step), and the producers issue them once
// those steps have drained. Copies of different steps complete in any order, so a patch that reads a
// column filled by one of the steps s-1 .. s-D+1 (a "hit" on a column still in flight) also waits on
// that step's full barrier; the record carries the mask.
// A parity wait is only right while the barrier is in the awaited phase or the one after it. NB is a
// multiple of the number of consumer groups NGRP (steps s and s-NB belong to the same group, which
// has consumed s-NB), NB >= NGRP + D (when a group is at step s every step <= s-NGRP-D has drained,
// so the previous phase of any barrier it waits on is closed) and NB >= 2D-1 (the next phase of a
// barrier awaited for step s-r cannot open before step s itself has drained). Every producer warp
// arrives on every step, so none of them can fall a whole ring behind either.
#include <cstdio>
#include <mutex>

#include "../../include/icon_dycore.h"
#include "kernels.cuh"
#include "cc_schedule.hpp"

namespace icon {
namespace {

constexpr unsigned kFull = 0xffffffffu;

// ---- PTX wrappers (mbarrier + bulk copies) ------------------------------------------------------
__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void mbar_init(uint32_t bar, uint32_t count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_arrive_expect_tx(uint32_t bar, uint32_t bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint32_t bar) {
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(bar) : "memory");
}
#ifdef CC_DEBUG
// debug build (python -m paper_2511_02021_b200.build --force with ICON_NVCC_EXTRA=-DCC_DEBUG): a wait that does
// not end reports where it hangs and traps
__device__ __forceinline__ void mbar_wait(uint32_t bar, uint32_t parity, int what = 0, int step = 0) {
    for (long it = 0;; ++it) {
        uint32_t ok;
        asm volatile(
            "{\n.reg .pred p;\nmbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\nselp.u32 %0, 1, 0, p;\n}\n"
            : "=r"(ok) : "r"(bar), "r"(parity) : "memory");
        if (ok) return;
        if (it > (1l << 22)) {
            if ((threadIdx.x & 31) == 0)
                printf("cc hang: block %d warp %d what %d step %d bar %u parity %u\n", blockIdx.x, threadIdx.x >> 5, what, step, bar, parity);
            __trap();
        }
    }
}
#else
// Plain polling loop on purpose: a try_wait with a suspend-time hint (500 ns, 2 us and 10 ms measured) made the fused
// step 6 % slower whatever the value (4.69 ms against 4.41 ms), although the polling instructions are a quarter of all
// instructions the kernel issues.
__device__ __forceinline__ void mbar_wait(uint32_t bar, uint32_t parity, int = 0, int = 0) {
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "WAIT_%=:\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
        "@p bra DONE_%=;\n"
        "bra WAIT_%=;\n"
        "DONE_%=:\n"
        "}\n" ::"r"(bar), "r"(parity) : "memory");
}
#endif
// global -> shared, completion counted in bytes on `bar`
__device__ __forceinline__ void bulk_g2s(uint32_t dst, const void* src, uint32_t bytes, uint32_t bar) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(dst),
                 "l"(src), "r"(bytes), "r"(bar) : "memory");
}
// the same with an L2 eviction-priority hint
__device__ __forceinline__ void bulk_g2s_hint(uint32_t dst, const void* src, uint32_t bytes, uint32_t bar, uint64_t pol) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes.L2::cache_hint [%0], [%1], %2, [%3], %4;" ::"r"(dst),
                 "l"(src), "r"(bytes), "r"(bar), "l"(pol) : "memory");
}
__device__ __forceinline__ uint64_t l2_policy_evict_first() {
    uint64_t p;
    asm volatile("createpolicy.fractional.L2::evict_first.b64 %0, 1.0;" : "=l"(p));
    return p;
}

// ---- device view of the schedule ------------------------------------------------------------------
template <class T>
struct CcDev {
    const CcStep* steps;
    const CcLoad* loads;
    const unsigned char* records;     // [n_patches][record_bytes<T>()]
    const int64_t* cta_patch_begin;   // [n_ctas + 1]
    const int64_t* cta_step_begin;    // [n_ctas + 1]
    int n_slots;
    int slot_bytes;
    int64_t ne, nc, nv;               // rows of the caller's fields (bounds asserts of the CC_DEBUG build)
};

#ifdef CC_DEBUG
// the pool's own bounds checks (compute-sanitizer is closed on the B200 pool): every slot read stays inside the slot
// pool + its readable pad, every output column id is a row of its field
#define CC_ASSERT(cond, what, a, b) \
    do { if (!(cond)) { printf("cc assert %s: block %d thread %d: %lld %lld\n", what, blockIdx.x, threadIdx.x, (long long)(a), (long long)(b)); __trap(); } } while (0)
#else
#define CC_ASSERT(cond, what, a, b) do { } while (0)
#endif

// ---- the L levels of one column a lane owns ---------------------------------------------------------
// L == 3: v[0], v[1] = levels 2*lane, 2*lane+1 (one 16-byte access), v[2] = level 64+lane.
// L == 2: v[0], v[1] = levels 2*(lane%16), 2*(lane%16)+1 of the half-warp's own patch.
// L == 6: v[2p], v[2p+1] = levels 32*p + 2*(lane%16), +1 of the half-warp's own patch (p = 0, 1, 2).
template <class T, int L>
struct Col {
    T v[L];
};
#define FORL _Pragma("unroll") for (int l = 0; l < L; ++l)

template <int L>
__device__ __forceinline__ int level_of(int lane, int l) {
    return L == 2 ? 2 * (lane & 15) + l : L == 6 ? 32 * (l >> 1) + 2 * (lane & 15) + (l & 1) : (l < 2 ? 2 * lane + l : 64 + lane);
}

template <class T> struct Pair;
template <> struct Pair<double> { using type = double2; };
template <> struct Pair<float> { using type = float2; };

// value one level up (k-1) / down (k+1). Inside the pair the neighbour is the lane's own register; across lanes one
// shuffle per segment. The seam between the segments (levels 63 | 64) rides on the same shuffles: lane 31 feeds its
// level 63 to lane 0's level 64 (up), lane 0 feeds its level 64 to lane 31's level 63 (down). Lanes whose neighbour
// level does not exist get a value the caller masks.
template <class T, int L>
__device__ __forceinline__ Col<T, L> level_up(const Col<T, L>& a, int lane) {
    Col<T, L> r;
    if constexpr (L == 2) {
        r.v[0] = __shfl_up_sync(kFull, a.v[1], 1, 16);        // inside the half-warp
        r.v[1] = a.v[0];
    } else if constexpr (L == 6) {
        // rotate right by one inside the half-warp; its last lane hands the end of the PREVIOUS pair segment to lane 0
        const int src = ((lane + 15) & 15) | (lane & 16);
        const bool last = (lane & 15) == 15;
#pragma unroll
        for (int p = 0; p < 3; ++p) {
            r.v[2 * p] = __shfl_sync(kFull, last && p > 0 ? a.v[2 * p - 1] : a.v[2 * p + 1], src);
            r.v[2 * p + 1] = a.v[2 * p];
        }
    } else {
        r.v[0] = __shfl_up_sync(kFull, a.v[1], 1);
        r.v[1] = a.v[0];
        r.v[2] = __shfl_sync(kFull, lane == 31 ? a.v[1] : a.v[2], (lane + 31) & 31);
    }
    return r;
}
template <class T, int L>
__device__ __forceinline__ Col<T, L> level_down(const Col<T, L>& a, int lane) {
    Col<T, L> r;
    if constexpr (L == 2) {
        r.v[0] = a.v[1];
        r.v[1] = __shfl_down_sync(kFull, a.v[0], 1, 16);
    } else if constexpr (L == 6) {
        // rotate left by one inside the half-warp; its first lane hands the start of the NEXT pair segment to lane 15
        const int src = ((lane + 1) & 15) | (lane & 16);
        const bool first = (lane & 15) == 0;
#pragma unroll
        for (int p = 0; p < 3; ++p) {
            r.v[2 * p] = a.v[2 * p + 1];
            r.v[2 * p + 1] = __shfl_sync(kFull, first && p < 2 ? a.v[2 * p + 2] : a.v[2 * p], src);
        }
    } else {
        r.v[0] = a.v[1];
        r.v[1] = __shfl_sync(kFull, lane == 0 ? a.v[2] : a.v[0], (lane + 1) & 31);
        r.v[2] = __shfl_down_sync(kFull, a.v[2], 1);
    }
    return r;
}
template <class T, int L>
__device__ __forceinline__ Col<T, L> dot4(const T* r, const Col<T, L>& a, const Col<T, L>& b, const Col<T, L>& c,
                                          const Col<T, L>& d) {
    Col<T, L> o;
    FORL o.v[l] = r[0] * a.v[l] + r[1] * b.v[l] + r[2] * c.v[l] + r[3] * d.v[l];
    return o;
}
template <class T, int L>
__device__ __forceinline__ Col<T, L> ke2(const Col<T, L>& n, const Col<T, L>& t) {   // n^2 + t^2 = 2 KE_e (S4)
    Col<T, L> o;
    FORL o.v[l] = n.v[l] * n.v[l] + t.v[l] * t.v[l];
    return o;
}
template <class T, int L>
__device__ __forceinline__ void axpy(Col<T, L>& acc, T a, const Col<T, L>& x) {
    FORL acc.v[l] += a * x.v[l];
}
template <class T, int L>
__device__ __forceinline__ Col<T, L> scale(T a, const Col<T, L>& x) {
    Col<T, L> o;
    FORL o.v[l] = a * x.v[l];
    return o;
}

// N warp-uniform coefficients from shared memory (16-byte broadcasts)
template <int N, class T>
__device__ __forceinline__ void ld_coef(const T* __restrict__ p, T (&out)[N]) {
    constexpr int per = 16 / sizeof(T);
    static_assert(N % per == 0, "coefficient group must be a multiple of 16 bytes");
    const int4* q = reinterpret_cast<const int4*>(p);
#pragma unroll
    for (int i = 0; i < N / per; ++i) {
        int4 v = q[i];
        T tmp[per];
        *reinterpret_cast<int4*>(tmp) = v;
#pragma unroll
        for (int j = 0; j < per; ++j) out[i * per + j] = tmp[j];
    }
}
// N slot byte offsets (uint32) from the record
template <int N>
__device__ __forceinline__ void ld_slots(const uint32_t* __restrict__ p, uint32_t (&out)[N]) {
    static_assert(N % 4 == 0, "slot group must be a multiple of 16 bytes");
    const int4* q = reinterpret_cast<const int4*>(p);
#pragma unroll
    for (int i = 0; i < N / 4; ++i) {
        int4 v = q[i];
        out[4 * i] = (uint32_t)v.x; out[4 * i + 1] = (uint32_t)v.y; out[4 * i + 2] = (uint32_t)v.z; out[4 * i + 3] = (uint32_t)v.w;
    }
}

template <class T>
__host__ __device__ constexpr int cc_record_bytes(int mode) { return cc_coef_words(mode) * (int)sizeof(T) + kCcRecordTail; }

// kCcWarps consumer warps in two groups of kCcGroup; group g runs the steps s = g (mod 2); ring depth kCcDepth.
// MODE kCcTend: ddt_vn only (dycore_velocity_tendencies). MODE kCcStep: the same pass also stores div of the patch's four
// cells and the vorticity of the vertices the patch owns (dycore_step): both are by-products of columns and sums the
// tendency needs anyway. MODE kCcDivVort: ONLY div and vorticity (dycore_div_vort) from the 27 vn columns they need, with
// compact records (52 coefficients) and a schedule of its own.
template <class T, int L, int MODE>
__global__ void __launch_bounds__((CcWarps<T, L>::consumers + CcWarps<T, L>::producers) * 32, 1)
k_tend_cc(CcDev<T> d, int nlev, int ldk, int ldk_w, const T* __restrict__ abc, const T* __restrict__ vn,
          const T* __restrict__ w, T* __restrict__ ddt_vn, T* __restrict__ div, T* __restrict__ vort,
          unsigned long long* pace_counter, unsigned long long pace_per_launch, int pace_mask, int pace_last,
          const T* __restrict__ wk, T* __restrict__ ddt_w, CcMetric<T> met) {
    extern __shared__ __align__(128) unsigned char smem[];
    using C = Col<T, L>;
    constexpr int W = CcWarps<T, L>::consumers, G = CcWarps<T, L>::group, D = kCcDepth;
    constexpr int PPW = cc_patches_per_warp(L), PPS = G * PPW;      // patches per warp, per step
    constexpr bool METRIC = MODE == kCcTendM;
    constexpr bool WONLY = MODE == kCcWTend;
    constexpr bool FUSED = MODE != kCcTend && !METRIC && !WONLY, DVONLY = MODE == kCcDivVort, WTEND = MODE == kCcStepW || WONLY;
    constexpr int kCcProducers = CcWarps<T, L>::producers;
    constexpr int REC = cc_record_bytes<T>(MODE), COEF = cc_coef_words(MODE);
    constexpr int NGRP = W / G;
    static_assert(W % G == 0 && W % 4 == 0 && D > NGRP && D <= 16, "bad pipeline shape");
    // the shuffle tells the compiler that the warp index is warp-uniform: branches on it (role, patch in range)
    // become uniform branches and the shuffles below need no divergence handling
    const int warp = __shfl_sync(kFull, (int)(threadIdx.x >> 5), 0), lane = threadIdx.x & 31;
    uint64_t* bars = reinterpret_cast<uint64_t*>(smem);                       // full[NB], done[NB]
    unsigned char* rec_base = smem + kCcBarrierBytes;
    unsigned char* slot_base = rec_base + D * PPS * REC;
    const uint32_t bar0 = smem_u32(bars);
    auto full_bar = [&](int i) { return bar0 + 8u * (uint32_t)i; };
    // NB >= 2D-1 and >= NGRP+D: see the parity argument in the header comment
    constexpr int NBmin = (2 * D - 1 > NGRP + D) ? 2 * D - 1 : NGRP + D;
    constexpr int NB = NGRP * ((NBmin + NGRP - 1) / NGRP);
    static_assert(2 * NB * 8 <= kCcBarrierBytes, "barrier area too small");
    auto done_bar = [&](int i) { return bar0 + 8u * (uint32_t)(NB + i); };

    const int64_t pb = d.cta_patch_begin[blockIdx.x], pe = d.cta_patch_begin[blockIdx.x + 1];
    const int64_t sb = d.cta_step_begin[blockIdx.x];
    const int n_steps = (int)(d.cta_step_begin[blockIdx.x + 1] - sb);

    if (threadIdx.x == 0) {
        for (int i = 0; i < NB; ++i) {
            mbar_init(full_bar(i), kCcProducers);
            mbar_init(done_bar(i), G);
        }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();

    if (warp >= W) {
        // ================= producers (one or two warpgroups) =================
        // Issuing a bulk copy costs a ~100-cycle chain on the uniform datapath, so the list of a
        // step is dealt round-robin to kCcProducers warps. Registers go to the consumers.
        asm volatile("setmaxnreg.dec.sync.aligned.u32 %0;" ::"n"(CcWarps<T, L>::producer_regs));
        const int pw = warp - W;
        const uint64_t cs = (uint64_t)ldk * sizeof(T), cs_w = (uint64_t)ldk_w * sizeof(T);
        const uint32_t slot0 = smem_u32(slot_base), rec0 = smem_u32(rec_base);
        const uint64_t pol_first = l2_policy_evict_first();
        const uint2* lraw = reinterpret_cast<const uint2*>(d.loads);
        const int mine = kCcProducers * lane + pw;          // this lane's entry of each round of 32 * kCcProducers
        int drained = 0;
        // Pacing epoch: the counter is never reset and every launch adds exactly pace_per_launch events, so the
        // events of all earlier launches are the multiple of pace_per_launch at or below the value this CTA reads
        // before it adds its own first event (launches of one handle are stream-ordered; the counter cannot reach
        // the next multiple before every CTA, this one included, has added all of its events). Kept on the device so
        // that a captured CUDA graph replays correctly.
        unsigned long long pace_base = 0;
        if ((MODE == kCcStep || MODE == kCcStepW) && !CcWarps<T, L>::light && pace_mask && lane == 0) {
            unsigned long long have;
            asm volatile("ld.relaxed.gpu.global.u64 %0, [%1];" : "=l"(have) : "l"(pace_counter) : "memory");
            pace_base = have - have % pace_per_launch;
        }
        // The schedule is read kCcAhead steps ahead through a register ring (the step loop is unrolled
        // by kCcAhead so that the ring is statically indexed): header s+kCcAhead, and this lane's first
        // list entry of step s+kCcAhead, whose position header s already names (CcStep::ahead_begin).
        // Raw 16-/8-byte loads: no field is touched before its step, so nothing waits on them early.
        const uint4* hraw = reinterpret_cast<const uint4*>(d.steps + sb);
        uint4 h[kCcAhead];
        uint2 e[kCcAhead];
#pragma unroll
        for (int u = 0; u < kCcAhead; ++u) {
            h[u] = u < n_steps ? __ldg(hraw + u) : make_uint4(0u, 0u, 0u, 0u);
            e[u] = make_uint2(0u, 0u);
        }
#pragma unroll
        for (int u = 0; u < kCcAhead; ++u) e[u] = __ldg(lraw + h[u].x + mine);      // the list is padded: always readable
        for (int s0 = 0; s0 < n_steps; s0 += kCcAhead) {
#pragma unroll
            for (int u = 0; u < kCcAhead; ++u) {
                const int s = s0 + u;
                if (s < n_steps) {
                    // CcStep: load_begin | n_loads n_patches depth | tx16 | ahead_begin
                    const uint32_t load_begin = h[u].x, n_loads_u = h[u].y & 0xffffu, n_pat = (h[u].y >> 16) & 0xffu;
                    const uint32_t depth = h[u].y >> 24, ahead_begin = h[u].w;       // h[u].z = tx16, for the checker
                    const uint2 e0 = e[u];
                    if (s + kCcAhead < n_steps) {
                        h[u] = __ldg(hraw + s + kCcAhead);
                        e[u] = __ldg(lraw + ahead_begin + mine);
                    }
                    const int n_loads = (int)n_loads_u;
                    // compiled into the fused fp64 three-levels-per-lane kernel only: the tendency-only kernel lost 3 %
                    // to the mere presence of this block, and the light instantiations (fp32, one level per lane)
                    // slowed down by 40-50 % with the barrier active
                    if ((MODE == kCcStep || MODE == kCcStepW) && !CcWarps<T, L>::light && pace_mask && s && (s & pace_mask) == 0 && s <= pace_last) {
                        // every pace_mask + 1 steps the producers of all CTAs meet (bounded wait: pacing is an
                        // optimisation, never a condition for progress): SMs run at slightly different rates, and once
                        // the CTAs are rounds apart neighbouring tiles no longer share their halo columns through the L2
                        if (lane == 0) {
                            if (pw == 0) asm volatile("red.relaxed.gpu.global.add.u64 [%0], 1;" ::"l"(pace_counter) : "memory");
                            const unsigned long long need = pace_base + (unsigned long long)(s / (pace_mask + 1)) * gridDim.x;
                            for (int spin = 0; spin < (1 << 15); ++spin) {
                                unsigned long long have;
                                asm volatile("ld.relaxed.gpu.global.u64 %0, [%1];" : "=l"(have) : "l"(pace_counter) : "memory");
                                if (have >= need) break;
                                __nanosleep(200);
                            }
                        }
                        __syncwarp();
                    }
                    // The producers run ahead of the consumers and spend most of their time right here, waiting for step
                    // s - depth to drain. ONE warp polls the mbarrier, the others sleep in a hardware barrier: four
                    // polling warps were 450 of the 2500 instructions the kernel issued per patch (profiles/r02_*),
                    // pure heat in a kernel that runs into the board's power cap.
                    if (drained < s - (int)depth + 1) {            // the same decision in every producer warp
                        if (pw == 0)
                            for (int t = drained; t < s - (int)depth + 1; ++t) mbar_wait(done_bar(t % NB), (uint32_t)((t / NB) & 1), 1, s);
                        drained = s - (int)depth + 1;
                        asm volatile("bar.sync 1, %0;" ::"n"(kCcProducers * 32) : "memory");
                    }
                    const uint32_t fb = full_bar(s % NB);
                    // Every producer warp announces the bytes of its own share before it issues them
                    // (the transaction count of the barrier never runs negative), then copies.
                    uint32_t my16 = 0;
                    for (int base = 0; base + mine < n_loads; base += 32 * kCcProducers) {
                        const uint2 q = base == 0 ? e0 : __ldg(lraw + load_begin + base + mine);
                        my16 += (q.y >> 16) & 0x7fffu;
                    }
                    my16 = __reduce_add_sync(kFull, my16);
                    const bool rec_warp = pw == kCcProducers - 1;
                    if (lane == 0) mbar_arrive_expect_tx(fb, my16 * 16u + (rec_warp ? n_pat * (uint32_t)REC : 0u));
                    __syncwarp();
                    if (rec_warp && lane == 0) {
                        // the records of a step's patches are consecutive in memory and in the ring: one copy
                        // (evict-first: a record is read once)
                        const int64_t p = pb + (int64_t)s * PPS;
                        const uint32_t dst = rec0 + (uint32_t)(((s % D) * PPS) * REC);
                        bulk_g2s_hint(dst, d.records + p * REC, n_pat * (uint32_t)REC, fb, pol_first);
                    }
                    for (int base = 0; base + mine < n_loads; base += 32 * kCcProducers) {
                        const uint2 q = base == 0 ? e0 : __ldg(lraw + load_begin + base + mine);
                        // CcLoad: id | slot (bits 0..15) bytes/16 (bits 16..30) kind (bit 31)
                        const uint32_t slot = q.y & 0xffffu, kind = q.y >> 31, bytes = ((q.y >> 16) & 0x7fffu) << 4;
                        CC_ASSERT(slot * (uint32_t)d.slot_bytes + bytes <= (uint32_t)d.n_slots * (uint32_t)d.slot_bytes && bytes > 0, "copy destination", slot, bytes);
                        CC_ASSERT((uint64_t)q.x * (kind ? cs_w : cs) + bytes <= (uint64_t)(kind ? d.nc : d.ne) * (kind ? cs_w : cs), "copy source", q.x, kind);
                        const unsigned char* src = kind ? reinterpret_cast<const unsigned char*>(w) + (uint64_t)q.x * cs_w
                                                        : reinterpret_cast<const unsigned char*>(vn) + (uint64_t)q.x * cs;
                        bulk_g2s(slot0 + slot * (uint32_t)d.slot_bytes, src, bytes, fb);
                    }
                }
            }
        }
        return;
    }
    asm volatile("setmaxnreg.inc.sync.aligned.u32 %0;" ::"n"(CcWarps<T, L>::consumer_regs));

    // ================= consumers =================
    const int grp = warp / G, wi = warp % G;
    // per-lane level coefficients of the vertical term (reading P-14)
    T cA[L], cB[L], cC[L];
    bool po[L];              // this lane's levels that exist in a vn / ddt_vn column
    bool below_missing[L];   // level k+1 does not exist (k = nlev-1) or lies past the column end
    FORL {
        const int k = level_of<L>(lane, l);
        po[l] = k < nlev;
        below_missing[l] = k + 1 >= nlev;
        cA[l] = !DVONLY && !METRIC && po[l] ? __ldg(abc + k) : (T)0;
        cB[l] = !DVONLY && !METRIC && po[l] ? __ldg(abc + nlev + k) : (T)0;
        cC[l] = !DVONLY && !METRIC && po[l] ? __ldg(abc + 2 * nlev + k) : (T)0;
    }
    // vertical-wind tendency (mode kCcStepW, P-19): weight of vn(k) in vn_ie(k), 1 / (z_half[k-1] - z_half[k+1]) (both 0
    // outside the interior half levels 1 .. nlev-1, so that ddt_w comes out 0 at the top and the surface) and the half
    // levels that exist in a w / ddt_w column
    bool pow_[L], w_int[L];
    FORL {
        const int k = level_of<L>(lane, l);
        pow_[l] = (WTEND || METRIC) && k <= nlev;
        w_int[l] = WTEND && k >= 1 && k <= nlev - 1;
    }
    const uint64_t cs = (uint64_t)ldk * sizeof(T), cs_wout = (uint64_t)ldk_w * sizeof(T);
    const int hl = PPW == 2 ? lane & 15 : lane, half = PPW == 2 ? lane >> 4 : 0;      // lane inside its patch, patch of the warp
    // this lane's two read positions inside every slot
    const unsigned char* my_pair = slot_base + 2 * hl * (int)sizeof(T);
    const unsigned char* my_single = slot_base + (64 + lane) * (int)sizeof(T);
    // and its two byte offsets inside every output column
    const uint32_t st_pair = (uint32_t)(2 * hl * (int)sizeof(T)), st_single = (uint32_t)((64 + lane) * (int)sizeof(T));

    for (int s = grp; s < n_steps; s += NGRP) {
        const int64_t p_first = pb + (int64_t)s * PPS + wi * PPW;       // the warp's first patch of this step
        mbar_wait(full_bar(s % NB), (uint32_t)((s / NB) & 1), 2, s);
        if (p_first < pe) {
            // L == 2: the second half-warp's patch may lie past the end of the CTA's range (odd patch count): it then
            // repeats the first one's reads and arithmetic and stores nothing
            const bool live = p_first + half < pe;
            const int my_patch = wi * PPW + (live ? half : 0);
            if constexpr (PPW == 2) {
                if (!live) { FORL { po[l] = false; pow_[l] = false; } }
            }
            const unsigned char* rec = rec_base + ((s % D) * PPS + my_patch) * REC;
            const T* cf = reinterpret_cast<const T*>(rec);
            const int32_t* oid = reinterpret_cast<const int32_t*>(rec + COEF * sizeof(T));
            const uint32_t* sl = reinterpret_cast<const uint32_t*>(rec + COEF * sizeof(T) + kCcRecordIds * 4);

            // Every lane reads its levels whether they exist or not: lanes past the column end pick up stale bytes of
            // the slot (or of the next one; the pool ends with a readable pad) that only ever reach outputs through
            // the level-below neighbour of the last level, which VD masks.
            auto LD = [&](uint32_t off) {
                CC_ASSERT(off % 16 == 0 && off + 96 * sizeof(T) <= (uint32_t)d.n_slots * (uint32_t)d.slot_bytes + kCcSlotTailPad, "slot offset", off, d.n_slots);
                C c;
                using P2 = typename Pair<T>::type;
                const P2 pr = *reinterpret_cast<const P2*>(my_pair + off);
                c.v[0] = pr.x; c.v[1] = pr.y;
                if constexpr (L == 3) c.v[2] = *reinterpret_cast<const T*>(my_single + off);
                if constexpr (L == 6) {
                    const P2 p1 = *reinterpret_cast<const P2*>(my_pair + off + 32 * sizeof(T));
                    const P2 p2 = *reinterpret_cast<const P2*>(my_pair + off + 64 * sizeof(T));
                    c.v[2] = p1.x; c.v[3] = p1.y; c.v[4] = p2.x; c.v[5] = p2.y;
                }
                return c;
            };
            auto WS = [&](uint32_t off) {       // w(k) + w(k+1) = 2 w_f(k) (S6); the 1/2 is folded into c_lin
                const C c = LD(off);
                const C dn = level_down(c, lane);
                C o;
                FORL o.v[l] = c.v[l] + dn.v[l];
                return o;
            };
            auto VD = [&](const C& x) {         // (vn_ie(k) - vn_ie(k+1)) / dz_k, reading P-14 folded into A, B, C
                C up = level_up(x, lane), dn = level_down(x, lane), o;
                FORL if (below_missing[l]) dn.v[l] = (T)0;      // C_k = 0 there, but the stale value may be NaN
                FORL o.v[l] = cA[l] * up.v[l] + cB[l] * x.v[l] + cC[l] * dn.v[l];
                return o;
            };
            // one finished output column, straight from the registers: coalesced streaming stores (outputs should
            // not push halo columns out of the L2); id < 0 = not ours
            auto ST = [&](T* base, int32_t id, const C& x) {
                if (id < 0) return;
                CC_ASSERT(id < (base == ddt_vn ? d.ne : base == div ? d.nc : d.nv), "output id", id, base == ddt_vn ? 0 : base == div ? 1 : 2);
                // one 64-bit column base (warp-uniform) plus the lane's two 32-bit byte offsets
                unsigned char* col = reinterpret_cast<unsigned char*>(base) + (uint64_t)(uint32_t)id * cs;
                using P2 = typename Pair<T>::type;
                P2 pr;
                pr.x = x.v[0]; pr.y = x.v[1];
                if (po[1]) __stcs(reinterpret_cast<P2*>(col + st_pair), pr);
                else if (po[0]) __stcs(reinterpret_cast<T*>(col + st_pair), x.v[0]);
                if constexpr (L == 3) {
                    if (po[2]) __stcs(reinterpret_cast<T*>(col + st_single), x.v[2]);
                }
                if constexpr (L == 6) {
#pragma unroll
                    for (int q = 1; q < 3; ++q) {
                        pr.x = x.v[2 * q]; pr.y = x.v[2 * q + 1];
                        if (po[2 * q + 1]) __stcs(reinterpret_cast<P2*>(col + st_pair + 32 * q * sizeof(T)), pr);
                        else if (po[2 * q]) __stcs(reinterpret_cast<T*>(col + st_pair + 32 * q * sizeof(T)), x.v[2 * q]);
                    }
                }
            };

            // one column of a caller's field straight from global memory, in the lane's level mapping (metric columns of
            // an owned edge: used by this patch only, so they bypass the column cache); levels that do not exist read as 0
            auto GL = [&](const T* base, int32_t id, uint64_t stride, const bool (&valid)[L]) {
                using P2 = typename Pair<T>::type;
                const unsigned char* col = reinterpret_cast<const unsigned char*>(base) + (uint64_t)(uint32_t)id * stride;
                C c;
                FORL c.v[l] = (T)0;
                constexpr int NP = L == 6 ? 3 : 1;
#pragma unroll
                for (int q = 0; q < NP; ++q) {
                    const unsigned char* a = col + st_pair + 32 * q * sizeof(T);
                    if (valid[2 * q + 1]) {
                        const P2 pr = __ldcs(reinterpret_cast<const P2*>(a));
                        c.v[2 * q] = pr.x; c.v[2 * q + 1] = pr.y;
                    } else if (valid[2 * q]) {
                        c.v[2 * q] = __ldcs(reinterpret_cast<const T*>(a));
                    }
                }
                if constexpr (L == 3) {
                    if (valid[2]) c.v[2] = __ldcs(reinterpret_cast<const T*>(col + st_single));
                }
                return c;
            };
            // (vn_ie(k) - vn_ie(k+1)) inv_ddqz with the per-edge weights of reading P-20 (wg on half levels, two-point
            // extrapolation at both ends); neighbours that do not exist are never selected
            auto VDM = [&](const C& x, const C& wg, const C& inv) {
                const C up = level_up(x, lane), dn = level_down(x, lane), wgd = level_down(wg, lane);
                C o;
                FORL {
                    const int k = level_of<L>(lane, l);
                    const bool top = k == 0, bot = k == nlev - 1;
                    const T vk = (top ? x.v[l] : up.v[l]) + wg.v[l] * (x.v[l] - (top ? dn.v[l] : up.v[l]));
                    const T vk1 = x.v[l] + wgd.v[l] * (bot ? x.v[l] - up.v[l] : dn.v[l] - x.v[l]);
                    o.v[l] = po[l] ? (vk - vk1) * inv.v[l] : (T)0;
                }
                return o;
            };

            // columns this patch shares with the steps s-1 .. s-D+1 were copied on THEIR barriers, and
            // copies of different steps land in any order: wait for the steps the record names
            {
                uint32_t mask = sl[kCcMaskWord];
                if constexpr (PPW == 2) mask |= __shfl_xor_sync(kFull, mask, 16);      // the warp waits for both patches' steps
#pragma unroll
                for (int r = 1; r < D; ++r)
                    if ((mask >> r) & 1u) mbar_wait(full_bar((s - r) % NB), (uint32_t)(((s - r) / NB) & 1), 3, s);
            }
            uint32_t sE[24];                    // i0 i1 i2 b0..b5 om0..om5 oc0..oc5 x0[0..2]
            ld_slots(sl + SID_I0, sE);
            C vI[3], vB[6];
#pragma unroll
            for (int j = 0; j < 3; ++j) vI[j] = LD(sE[j]);
#pragma unroll
            for (int j = 0; j < 6; ++j) vB[j] = LD(sE[3 + j]);

            int32_t ido[16];                    // owned edges i0 i1 i2 b0 b2 b4 | cells T0..T3 | vertices ab bc ca a b c (-1 = not ours)
#pragma unroll
            for (int i = 0; i < (FUSED ? 4 : WONLY ? 3 : 2); ++i) {
                const int4 a = reinterpret_cast<const int4*>(oid)[i];
                ido[4 * i] = a.x; ido[4 * i + 1] = a.y; ido[4 * i + 2] = a.z; ido[4 * i + 3] = a.w;
            }
            if constexpr (METRIC) {
                // Request the 24 metric columns of this patch (4 fields x 6 owned edges, 6 lines of 128 bytes each for 90 fp64
                // levels) into the L2 now: they are needed ~2 us from now, straight from global memory, and a DRAM round trip
                // per batch was what bounded this mode (12.8 ms at config 3 before). One line per lane and request.
                for (int i = hl; i < 24 * 8; i += 32 / PPW) {          // two patches per warp: every half-warp covers its own patch
                    const int colm = i >> 3, line = i & 7, field = colm / 6, edge = colm - 6 * field;
                    const unsigned char* base = reinterpret_cast<const unsigned char*>(field == 0 ? met.wgt : field == 1 ? met.inv : field == 2 ? met.zn : met.zt);
                    const uint64_t first = (uint64_t)(uint32_t)oid[edge] * (field == 0 ? cs_wout : cs);
                    const uint64_t last = first + (uint64_t)(nlev + (field == 0 ? 1 : 0)) * sizeof(T) - 1;
                    const uint64_t at = (first & ~(uint64_t)127) + ((uint64_t)line << 7);       // only lines that hold bytes of the column
                    if (at <= last && live) asm volatile("prefetch.global.L2 [%0];" ::"l"(base + at));
                }
            }
            if constexpr (FUSED) {
                // ---- S1: div of the four cells from their edges (slot order of SCF_BLN) ------------
                T gd[12];
                ld_coef(cf + (DVONLY ? (int)DVF_DIV : (int)SCF_DIV), gd);
                C dv;
                FORL dv.v[l] = gd[0] * vB[0].v[l] + gd[1] * vI[0].v[l] + gd[2] * vB[5].v[l];
                ST(div, ido[6], dv);
                FORL dv.v[l] = gd[3] * vB[1].v[l] + gd[4] * vB[2].v[l] + gd[5] * vI[1].v[l];
                ST(div, ido[7], dv);
                FORL dv.v[l] = gd[6] * vI[2].v[l] + gd[7] * vB[3].v[l] + gd[8] * vB[4].v[l];
                ST(div, ido[8], dv);
                FORL dv.v[l] = gd[9] * vI[1].v[l] + gd[10] * vI[2].v[l] + gd[11] * vI[0].v[l];
                ST(div, ido[9], dv);
            }
            if constexpr (WTEND) {
                // ---- vertical-wind tendency of the four cells (P-19), while only the nine in-patch columns are live ----
                // ddt_w(c,k) = -[ sum_j a(c,j) vn_ie(e_j,k) (w(cell across e_j,k) - w(c,k)) + w(c,k) (w(c,k-1) - w(c,k+1)) rdz2(k) ]
                // the two per-level constants are fetched here (L1-resident after the first patch) instead of living in
                // registers for the whole kernel: the fused instantiation sits at its register limit
                T wg[L], wrdz[L];
                FORL {
                    const int k = level_of<L>(lane, l);
                    wg[l] = w_int[l] ? __ldg(wk + k) : (T)0;
                    wrdz[l] = w_int[l] ? __ldg(wk + nlev + 1 + k) : (T)0;
                }
                T av[12];
                ld_coef(cf + (WONLY ? (int)WF_ADV : (int)SCF_ADV), av);
                uint32_t sW[12];                    // T0..T3 X0 X2 X4 X1 X3 X5 + mask + pad
                ld_slots(sl + SID_T0, sW);
                C wT[4];
#pragma unroll
                for (int j = 0; j < 4; ++j) wT[j] = LD(sW[j]);
                auto VIE = [&](const C& x) {        // vn at the half level k: g_k vn(k) + (1 - g_k) vn(k-1); 0 outside 1 .. nlev-1
                    const C up = level_up(x, lane);
                    C o;
                    FORL o.v[l] = w_int[l] ? wg[l] * x.v[l] + ((T)1 - wg[l]) * up.v[l] : (T)0;
                    return o;
                };
                C acc[4];
                {
                    const C v0 = VIE(vI[0]), v1 = VIE(vI[1]), v2 = VIE(vI[2]);
                    FORL {
                        acc[3].v[l] = av[9] * v1.v[l] * (wT[1].v[l] - wT[3].v[l]) + av[10] * v2.v[l] * (wT[2].v[l] - wT[3].v[l]) +
                                      av[11] * v0.v[l] * (wT[0].v[l] - wT[3].v[l]);
                        acc[0].v[l] = av[1] * v0.v[l] * (wT[3].v[l] - wT[0].v[l]);
                        acc[1].v[l] = av[5] * v1.v[l] * (wT[3].v[l] - wT[1].v[l]);
                        acc[2].v[l] = av[6] * v2.v[l] * (wT[3].v[l] - wT[2].v[l]);
                    }
                }
#pragma unroll
                for (int j = 0; j < 6; ++j) {
                    constexpr int cell_of[6] = {0, 1, 1, 2, 2, 0};
                    constexpr int bslot[6] = {0, 3, 4, 7, 8, 2};
                    constexpr int xslot[6] = {4, 7, 5, 8, 6, 9};      // X0 X1 X2 X3 X4 X5 inside sW
                    const C wx = LD(sW[xslot[j]]);
                    const C v = VIE(vB[j]);
                    FORL acc[cell_of[j]].v[l] += av[bslot[j]] * v.v[l] * (wx.v[l] - wT[cell_of[j]].v[l]);
                }
                if constexpr (WONLY) {              // ddt_w alone: that was the last slot read of the patch
                    __syncwarp();
                    if (lane == 0) mbar_arrive(done_bar(s % NB));
                }
#pragma unroll
                for (int c4 = 0; c4 < 4; ++c4) {
                    const C up = level_up(wT[c4], lane), dn = level_down(wT[c4], lane);
                    C o;
                    // the neighbours of the first and last half level do not exist (stale values): rdz2 is 0 there, select
                    FORL o.v[l] = w_int[l] ? -(acc[c4].v[l] + wT[c4].v[l] * (up.v[l] - dn.v[l]) * wrdz[l]) : (T)0;
                    const int32_t id = ido[6 + c4];
                    unsigned char* col = reinterpret_cast<unsigned char*>(ddt_w) + (uint64_t)(uint32_t)id * cs_wout;
                    using P2 = typename Pair<T>::type;
                    P2 pr;
                    pr.x = o.v[0]; pr.y = o.v[1];
                    if (pow_[1]) __stcs(reinterpret_cast<P2*>(col + st_pair), pr);
                    else if (pow_[0]) __stcs(reinterpret_cast<T*>(col + st_pair), o.v[0]);
                    if constexpr (L == 3) {
                        if (pow_[2]) __stcs(reinterpret_cast<T*>(col + st_single), o.v[2]);
                    }
                }
            }
            if constexpr (DVONLY) {
                // ---- S2 alone: the six vorticities from the patch's own columns, the om / oc columns and n1, n2 -------
                T g18[20], gx[20];
                ld_coef(cf + DVF_ROT, g18);
                ld_coef(cf + DVF_XROT, gx);
                uint32_t sX[12];                    // x0[3..4] x1[0..4] x2[0..4]
                ld_slots(sl + SID_X0 + 3, sX);
                C zm[3], zc[3];
                FORL {
                    zm[0].v[l] = g18[0] * vB[0].v[l] + g18[1] * vB[1].v[l] + g18[2] * vI[0].v[l] + g18[3] * vI[1].v[l];
                    zm[1].v[l] = g18[6] * vB[2].v[l] + g18[7] * vB[3].v[l] + g18[8] * vI[1].v[l] + g18[9] * vI[2].v[l];
                    zm[2].v[l] = g18[12] * vB[4].v[l] + g18[13] * vB[5].v[l] + g18[14] * vI[2].v[l] + g18[15] * vI[0].v[l];
                    zc[0].v[l] = gx[0] * vB[0].v[l] + gx[5] * vB[5].v[l];
                    zc[1].v[l] = gx[6] * vB[2].v[l] + gx[11] * vB[1].v[l];
                    zc[2].v[l] = gx[12] * vB[4].v[l] + gx[17] * vB[3].v[l];
                }
#pragma unroll
                for (int j = 0; j < 6; ++j) {
                    const C vM = LD(sE[9 + j]), vO = LD(sE[15 + j]);
                    axpy(zm[j / 2], g18[6 * (j / 2) + 4 + (j & 1)], vM);
                    if (j & 1) {
                        const int xn = ((j + 1) % 6) / 2;
                        axpy(zc[xn], gx[6 * xn + 4], vO);
                    } else {
                        const int x = j / 2;
                        const C n1 = LD(sX[5 * x]), n2 = LD(sX[5 * x + 1]);
                        FORL zc[x].v[l] += gx[6 * x + 1] * vO.v[l] + gx[6 * x + 2] * n1.v[l] + gx[6 * x + 3] * n2.v[l];
                    }
                }
                __syncwarp();
                if (lane == 0) mbar_arrive(done_bar(s % NB));
#pragma unroll
                for (int m = 0; m < 3; ++m) {
                    C z2;
                    FORL z2.v[l] = (T)2 * zm[m].v[l];
                    ST(vort, ido[10 + m], z2);
                    FORL z2.v[l] = (T)2 * zc[m].v[l];
                    ST(vort, ido[13 + m], z2);
                }
            } else if constexpr (!WONLY) {
            // ---- interior edges: vt, KE_e; start the cell sums -------------------------------
            T r12[12];
            ld_coef(cf + SCF_RBF, r12);
            C tI[3];
            tI[0] = dot4(r12 + 0, vB[0], vB[5], vI[1], vI[2]);
            tI[1] = dot4(r12 + 4, vB[1], vB[2], vI[2], vI[0]);
            tI[2] = dot4(r12 + 8, vB[3], vB[4], vI[0], vI[1]);
            T bl[12];
            ld_coef(cf + SCF_BLN, bl);
            C ke[4];
            {
                C kI0 = ke2(vI[0], tI[0]), kI1 = ke2(vI[1], tI[1]), kI2 = ke2(vI[2], tI[2]);
                ke[0] = scale(bl[1], kI0);
                ke[1] = scale(bl[5], kI1);
                ke[2] = scale(bl[6], kI2);
                FORL ke[3].v[l] = bl[9] * kI1.v[l] + bl[10] * kI2.v[l] + bl[11] * kI0.v[l];
            }
            // ---- midpoint vorticities (x 1/2): interior + boundary part ----------------------
            T g18[20];
            ld_coef(cf + SCF_ROT, g18);
            C zm[3];
            FORL {
                zm[0].v[l] = g18[0] * vB[0].v[l] + g18[1] * vB[1].v[l] + g18[2] * vI[0].v[l] + g18[3] * vI[1].v[l];
                zm[1].v[l] = g18[6] * vB[2].v[l] + g18[7] * vB[3].v[l] + g18[8] * vI[1].v[l] + g18[9] * vI[2].v[l];
                zm[2].v[l] = g18[12] * vB[4].v[l] + g18[13] * vB[5].v[l] + g18[14] * vI[2].v[l] + g18[15] * vI[0].v[l];
            }
            // ---- corner vorticities (x 1/2): the part from the patch's own boundary edges ------
            T gx[20];
            ld_coef(cf + SCF_XROT, gx);
            C zc[3];
            FORL {
                zc[0].v[l] = gx[0] * vB[0].v[l] + gx[5] * vB[5].v[l];
                zc[1].v[l] = gx[6] * vB[2].v[l] + gx[11] * vB[1].v[l];
                zc[2].v[l] = gx[12] * vB[4].v[l] + gx[17] * vB[3].v[l];
            }
            // ---- boundary edges b0..b5 with their outer columns ------------------------------
            uint32_t sX[24];                    // x0[3..4] x1[0..4] x2[0..4] T0..T3 X0 X2 X4 + pad
            ld_slots(sl + SID_X0 + 3, sX);
            T rB[24];
            ld_coef(cf + SCF_RBF + 12, rB);
            T xrm[12], xro[12], xbl[12];
            ld_coef(cf + SCF_XRM, xrm);
            ld_coef(cf + SCF_XRO, xro);
            ld_coef(cf + SCF_XBL, xbl);
            C tBo[3], keX[3];
#pragma unroll
            for (int j = 0; j < 6; ++j) {
                const C vM = LD(sE[9 + j]), vO = LD(sE[15 + j]);
                // neighbour pairs (a, b) of the stencil of b_j inside the patch
                const C& na = j == 0 ? vI[0] : j == 1 ? vB[2] : j == 2 ? vB[1] : j == 3 ? vI[2] : j == 4 ? vI[2] : vB[0];
                const C& nb = j == 0 ? vB[5] : j == 1 ? vI[1] : j == 2 ? vI[1] : j == 3 ? vB[4] : j == 4 ? vB[3] : vI[0];
                const C tB = dot4(rB + 4 * j, na, nb, vM, vO);
                const C kB = ke2(vB[j], tB);
                // KE_c of the patch cell that holds b_j (bln slot order of sc_tables.cpp)
                constexpr int cell_of[6] = {0, 1, 1, 2, 2, 0};
                constexpr int bslot[6] = {0, 3, 4, 7, 8, 2};
                axpy(ke[cell_of[j]], bl[bslot[j]], kB);
                // midpoint vorticity: om_j is fan slot 4 + (j & 1) of midpoint j / 2
                axpy(zm[j / 2], g18[6 * (j / 2) + 4 + (j & 1)], vM);
                if (j & 1) {
                    // oc_j is slot 4 (oc_jp) of the corner of the next owned boundary edge
                    const int xn = ((j + 1) % 6) / 2;
                    axpy(zc[xn], gx[6 * xn + 4], vO);
                } else {
                    const int x = j / 2;
                    // ring columns pm0 pm1 pcf n1 n2 of x: id slots SID_X0 + 5x ..; sE holds x0[0..2], sX the rest
                    const uint32_t s_pm0 = x == 0 ? sE[21] : sX[5 * x - 3], s_pm1 = x == 0 ? sE[22] : sX[5 * x - 2];
                    const uint32_t s_pcf = x == 0 ? sE[23] : sX[5 * x - 1];
                    const uint32_t s_n1 = sX[5 * x], s_n2 = sX[5 * x + 1];
                    const C pm0 = LD(s_pm0), pm1 = LD(s_pm1), pcf = LD(s_pcf), n1 = LD(s_n1), n2 = LD(s_n2);
                    const C tM = dot4(xrm + 4 * x, vB[j], vO, pm0, pm1);
                    const C tO = dot4(xro + 4 * x, vB[j], vM, n1, pcf);
                    const C kM = ke2(vM, tM), kO = ke2(vO, tO);
                    FORL keX[x].v[l] = xbl[3 * x] * kB.v[l] + xbl[3 * x + 1] * kM.v[l] + xbl[3 * x + 2] * kO.v[l];
                    FORL zc[x].v[l] += gx[6 * x + 1] * vO.v[l] + gx[6 * x + 2] * n1.v[l] + gx[6 * x + 3] * n2.v[l];
                    tBo[x] = tB;
                }
            }
            if constexpr (FUSED) {
                // ---- S2: zm, zc hold zeta / 2 at the three midpoints and the three corners ------------
#pragma unroll
                for (int m = 0; m < 3; ++m) {
                    C z2;
                    FORL z2.v[l] = (T)2 * zm[m].v[l];
                    ST(vort, ido[10 + m], z2);
                }
#pragma unroll
                for (int m = 0; m < 3; ++m) {
                    C z2;
                    FORL z2.v[l] = (T)2 * zc[m].v[l];
                    ST(vort, ido[13 + m], z2);
                }
            }
            // ---- horizontal part H of the six owned edges (S5); frees the KE / vorticity columns ----
            if constexpr (METRIC) {
                // ---- metric form (reading P-20), in three phases. (1) The part of H that needs no metric column,
                // A0 = -(gH KE_c(H) - gL KE_c(L) + gE (vn^2 + vt^2) + vt (f + zeta_e)), frees the KE / vorticity columns.
                // (2) w at the owned edges: the last slot reads, the step is released. (3) One pass over the owned edges with
                // the four metric columns of an edge fetched in ONE batch straight from global memory (requested into the L2
                // when the patch started), the batch of the NEXT edge in flight while this one is used; each output column
                // leaves as soon as it is complete.
                C A0[6];
#pragma unroll
                for (int x = 0; x < 6; ++x) {
                    const C& v = x < 3 ? vI[x] : vB[2 * (x - 3)];
                    const C& t = x < 3 ? tI[x] : tBo[x - 3];
                    const C& kL = ke[x % 3];
                    const C& kH = x < 3 ? ke[3] : keX[x - 3];
                    const C& za = x < 3 ? (x == 2 ? zm[1] : zm[0]) : zm[x - 3];
                    const C& zb = x < 3 ? (x == 1 ? zm[1] : zm[2]) : zc[x - 3];      // i0: (ab, ca), i1: (ab, bc), i2: (bc, ca)
                    T e4[4], m4[4];                     // f_e | gL, gH, gE: read where they are used
                    ld_coef(cf + SCF_EDGE + 4 * x, e4);
                    ld_coef(cf + SCF_CGRAD + 4 * x, m4);
                    // gradK = gH KE_c(H) - gL KE_c(L) + gE (vn^2 + vt^2): second order at the edge midpoint
                    FORL A0[x].v[l] = -(m4[1] * kH.v[l] - m4[0] * kL.v[l] + m4[2] * (v.v[l] * v.v[l] + t.v[l] * t.v[l]) +
                                        t.v[l] * (e4[1] + (za.v[l] + zb.v[l])));
                }
                C we[6];
                {
                    C wf[4];
#pragma unroll
                    for (int j = 0; j < 4; ++j) wf[j] = WS(sX[12 + j]);
#pragma unroll
                    for (int x = 0; x < 3; ++x)
                        FORL we[x].v[l] = cf[SCF_EDGE + 4 * x + 2] * wf[x].v[l] + cf[SCF_EDGE + 4 * x + 3] * wf[3].v[l];
#pragma unroll
                    for (int x = 0; x < 3; ++x) {
                        const C wx = WS(sX[16 + x]);
                        FORL we[3 + x].v[l] = cf[SCF_EDGE + 4 * (3 + x) + 2] * wf[x].v[l] + cf[SCF_EDGE + 4 * (3 + x) + 3] * wx.v[l];
                    }
                }
                __syncwarp();
                if (lane == 0) mbar_arrive(done_bar(s % NB));
                C zn = GL(met.zn, ido[0], cs, po), zt = GL(met.zt, ido[0], cs, po);
                C wg = GL(met.wgt, ido[0], cs_wout, pow_), inv = GL(met.inv, ido[0], cs, po);
#pragma unroll
                for (int x = 0; x < 6; ++x) {
                    const C& v = x < 3 ? vI[x] : vB[2 * (x - 3)];
                    const C& t = x < 3 ? tI[x] : tBo[x - 3];
                    C zn1, zt1, wg1, inv1;
                    if (x < 5) {                        // the next edge's batch goes out before this one is used
                        zn1 = GL(met.zn, ido[x + 1], cs, po); zt1 = GL(met.zt, ido[x + 1], cs, po);
                        wg1 = GL(met.wgt, ido[x + 1], cs_wout, pow_); inv1 = GL(met.inv, ido[x + 1], cs, po);
                    }
                    const C Dv = VDM(v, wg, inv);
                    C o;
                    // V = (w_e - w_cc) Dv with the contravariant correction w_cc = vn ddxn_z + vt ddxt_z
                    FORL o.v[l] = A0[x].v[l] - (we[x].v[l] - (v.v[l] * zn.v[l] + t.v[l] * zt.v[l])) * Dv.v[l];
                    ST(ddt_vn, ido[x], o);
                    if (x < 5) { zn = zn1; zt = zt1; wg = wg1; inv = inv1; }
                }
            } else {
            // ---- horizontal part H of the six owned edges (S5); frees the KE / vorticity columns ----
            T ec[24];
            ld_coef(cf + SCF_EDGE, ec);
            C H[6];
#pragma unroll
            for (int x = 0; x < 3; ++x) {       // interior: i0 (ab, ca), i1 (ab, bc), i2 (bc, ca); cells (T_x, T3)
                const C& za = x == 2 ? zm[1] : zm[0];
                const C& zb = x == 0 ? zm[2] : x == 1 ? zm[1] : zm[2];
                const T* e4 = ec + 4 * x;
                FORL H[x].v[l] = (ke[3].v[l] - ke[x].v[l]) * e4[0] + tI[x].v[l] * (e4[1] + (za.v[l] + zb.v[l]));
            }
#pragma unroll
            for (int x = 0; x < 3; ++x) {       // boundary: b0 (a, ab), b2 (b, bc), b4 (c, ca); cells (T_x, X_2x)
                const T* e4 = ec + 4 * (3 + x);
                FORL H[3 + x].v[l] = (keX[x].v[l] - ke[x].v[l]) * e4[0] + tBo[x].v[l] * (e4[1] + (zm[x].v[l] + zc[x].v[l]));
            }
            // ---- cell-centre w at the six owned edges (S6): w_e = c_lin(L) w_f(L) + c_lin(H) w_f(H); these are the
            // last reads of the slots
            C we[6];
            {
                C wf[4];
#pragma unroll
                for (int j = 0; j < 4; ++j) wf[j] = WS(sX[12 + j]);
#pragma unroll
                for (int x = 0; x < 3; ++x) FORL we[x].v[l] = ec[4 * x + 2] * wf[x].v[l] + ec[4 * x + 3] * wf[3].v[l];
#pragma unroll
                for (int x = 0; x < 3; ++x) {
                    const C wx = WS(sX[16 + x]);
                    FORL we[3 + x].v[l] = ec[4 * (3 + x) + 2] * wf[x].v[l] + ec[4 * (3 + x) + 3] * wx.v[l];
                }
            }
            // everything this patch needs from the slots and its record is in registers: release the stage
            __syncwarp();
            if (lane == 0) mbar_arrive(done_bar(s % NB));

            // ---- vertical part and the tendency (S6, S7) -----------------------------------------
#pragma unroll
            for (int x = 0; x < 6; ++x) {
                const C Dv = VD(x < 3 ? vI[x] : vB[2 * (x - 3)]);
                C o;
                FORL o.v[l] = -H[x].v[l] - we[x].v[l] * Dv.v[l];
                ST(ddt_vn, ido[x], o);
            }
            }   // !METRIC
            }   // !DVONLY && !WONLY
        } else {
            __syncwarp();
            if (lane == 0) mbar_arrive(done_bar(s % NB));
        }
    }
}

}  // namespace

template <class T>
int cc_slot_bytes(int nlev) { return (((nlev + 1) * (int)sizeof(T) + 15) & ~15); }

template <class T>
static size_t cc_fixed_smem(int mode, int L) {
    return kCcBarrierBytes + (size_t)kCcDepth * cc_patches_per_step((int)sizeof(T), L) * cc_record_bytes<T>(mode);
}

template <class T>
int cc_max_slots(int slot_bytes, int smem_optin, int mode, int nlev) {
    const long avail = (long)smem_optin - (long)cc_fixed_smem<T>(mode, cc_level_mapping(nlev, (int)sizeof(T), mode)) - kCcSlotTailPad;
    if (avail <= 0) return 0;
    return (int)(avail / slot_bytes);
}
template int cc_max_slots<double>(int, int, int, int);
template int cc_max_slots<float>(int, int, int, int);
template int cc_slot_bytes<double>(int);
template int cc_slot_bytes<float>(int);

int cc_levels_per_lane(int nlev) { return nlev + 1 <= 32 ? 2 : nlev + 1 <= 96 ? 3 : 0; }
int cc_level_mapping(int nlev, int elem_bytes, int mode) {
    const int l = cc_levels_per_lane(nlev);
    return l == 3 && elem_bytes == 4 && mode == kCcDivVort ? 6 : l;
}
int cc_patches_per_step_for(int nlev, int elem_bytes, int mode) { return cc_patches_per_step(elem_bytes, cc_level_mapping(nlev, elem_bytes, mode)); }

namespace {
template <class T, int L, int MODE>
cudaError_t cc_launch_one(const CcDev<T>& d, int device, int n_ctas, size_t smem, int nlev, int ldk, int ldk_w, const T* abc,
                          const T* vn, const T* w, T* ddt_vn, T* div, T* vort, unsigned long long* pc, unsigned long long ppl,
                          int pm, int pl, const T* wk, T* ddt_w, const CcMetric<T>& met, cudaStream_t s) {
    auto k = k_tend_cc<T, L, MODE>;
    // the opt-in for > 48 KB of dynamic shared memory is a per-DEVICE attribute of the function: remembered per device
    static std::mutex mu;
    static size_t configured[64] = {0};       // largest size this instantiation was opted in for, per device ordinal
    {
        std::lock_guard<std::mutex> lock(mu);
        const bool known = device >= 0 && device < 64;
        if (!known || smem > configured[device]) {
            cudaError_t err = cudaFuncSetAttribute(k, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
            if (err != cudaSuccess) return err;
            if (known) configured[device] = smem;
        }
    }
    k<<<(unsigned)n_ctas, (CcWarps<T, L>::consumers + CcWarps<T, L>::producers) * 32, smem, s>>>(d, nlev, ldk, ldk_w, abc, vn, w, ddt_vn, div, vort, pc, ppl, pm, pl, wk, ddt_w, met);
    return cudaGetLastError();
}
}  // namespace

template <class T>
int launch_tendencies_cc(const icon_grid& g, DevCcTables<T>& p, int mode, int nlev, int64_t ldk, int64_t ldk_w,
                         const T* abc, const T* vn, const T* w, T* ddt_vn, T* div, T* vort, cudaStream_t s, const T* wk, T* ddt_w,
                         const CcMetric<T>* met) {
    CcDev<T> d;
    d.steps = p.steps; d.loads = p.loads; d.records = p.records;
    d.cta_patch_begin = p.cta_patch_begin; d.cta_step_begin = p.cta_step_begin;
    d.n_slots = p.n_slots; d.slot_bytes = p.slot_bytes;
    d.ne = g.host.ne; d.nc = g.host.nc; d.nv = g.host.nv;
    // pacing: a barrier of the producers every `period` steps (power of two), counted in p.progress (never reset)
    const int period = g.options[ICON_OPT_CC_PACE];
    const int L = cc_level_mapping(nlev, (int)sizeof(T), mode);
    const bool heavy = sizeof(T) == 8 && L == 3;
    int pace_mask = period > 0 && p.progress && (mode == kCcStep || mode == kCcStepW) && heavy ? period - 1 : 0;      // fused fp64 step only
    const int n_barriers = pace_mask ? (int)((p.min_steps - 1) / period) : 0;      // barriers every CTA reaches
    if (n_barriers == 0) pace_mask = 0;
    const int pace_last = n_barriers * period;
    const unsigned long long per_launch = (unsigned long long)n_barriers * (unsigned long long)p.n_ctas;
    // the tables must have been built for this mode (kCcTend runs on the tables of kCcStep: same columns, same records)
    const bool wants_div = mode == kCcStep || mode == kCcStepW || mode == kCcDivVort;
    const bool no_ddt_vn = mode == kCcDivVort || mode == kCcWTend;
    if ((mode == kCcTend ? (int)kCcStep : mode) != p.built_for || no_ddt_vn != (ddt_vn == nullptr) || wants_div != (div != nullptr) ||
        (mode == kCcStepW || mode == kCcWTend) != (ddt_w != nullptr) || (mode == kCcTendM) != (met != nullptr))
        return -(int)cudaErrorInvalidValue;
    const CcMetric<T> metric = met ? *met : CcMetric<T>{nullptr, nullptr, nullptr, nullptr};
    const size_t smem = cc_fixed_smem<T>(mode, L) + (size_t)p.n_slots * p.slot_bytes + kCcSlotTailPad;
    cudaError_t err = cudaErrorInvalidValue;
#define CC_ONE(LL, MM) \
    if (L == LL && mode == MM) \
        err = cc_launch_one<T, LL, MM>(d, g.device, p.n_ctas, smem, nlev, (int)ldk, (int)ldk_w, abc, vn, w, ddt_vn, div, vort, p.progress, per_launch, pace_mask, pace_last, wk, ddt_w, metric, s);
    CC_ONE(2, kCcTend) CC_ONE(2, kCcStep) CC_ONE(2, kCcDivVort) CC_ONE(3, kCcTend) CC_ONE(3, kCcStep)
    CC_ONE(2, kCcStepW) CC_ONE(3, kCcStepW) CC_ONE(2, kCcTendM) CC_ONE(3, kCcTendM) CC_ONE(2, kCcWTend) CC_ONE(3, kCcWTend)
    constexpr int LDV = sizeof(T) == 4 ? 6 : 3;          // deep columns in the div / vort mode
    CC_ONE(LDV, kCcDivVort)
#undef CC_ONE
    return err == cudaSuccess ? 1 : -(int)err;
}

template int launch_tendencies_cc<double>(const icon_grid&, DevCcTables<double>&, int, int, int64_t, int64_t,
                                          const double*, const double*, const double*, double*, double*, double*, cudaStream_t, const double*, double*, const CcMetric<double>*);
template int launch_tendencies_cc<float>(const icon_grid&, DevCcTables<float>&, int, int, int64_t, int64_t,
                                         const float*, const float*, const float*, float*, float*, float*, cudaStream_t, const float*, float*, const CcMetric<float>*);

}  // namespace icon
