// device_grid.hpp -- the opaque icon_grid handle: host tables + device tables + workspaces.
// Internal header of libicon_dycore.
#pragma once
#include <cuda_runtime.h>

#include <cstdint>
#include <map>
#include <vector>

#include "host_grid.hpp"
#include "sc_tables.hpp"
#include "cc_schedule.hpp"
#include "partition.hpp"

namespace icon {

// Device tables the kernels read. Rows are in WORK ORDER (generation order = spatially local,
// identical to user order unless the grid is permuted); entries are USER ids, so they address
// the caller's fields directly.
template <class T>
struct DevCoeffs {
    T* rbf = nullptr;         // [ne][4]
    T* bln = nullptr;         // [nc][3]
    T* geofac_div = nullptr;  // [nc][3]
    T* geofac_rot = nullptr;  // [nv][6]
    T* inv_d_e = nullptr;     // [ne]
    T* f_e = nullptr;         // [ne]
    T* c_lin = nullptr;       // [ne][2]
    T* adv_c = nullptr;       // [nc][3]
    T* cgrad = nullptr;       // [ne][2]
    bool ready = false;
};

struct DevTables {
    int32_t* c2e = nullptr;   // [nc][3]
    int32_t* e2c = nullptr;   // [ne][2]
    int32_t* e2v = nullptr;   // [ne][2]
    int32_t* e2e4 = nullptr;  // [ne][4]
    int32_t* v2e = nullptr;   // [nv][6]
    // user id of work position p; nullptr = identity
    int32_t* user_c = nullptr;
    int32_t* user_e = nullptr;
    int32_t* user_v = nullptr;
    // work position of user id (inverse of the above); nullptr = identity
    int32_t* pos_c = nullptr;
    int32_t* pos_e = nullptr;
    int32_t* pos_v = nullptr;
};

// Device copy of the self-contained patch records (sc_tables.hpp), coefficient words in T.
template <class T>
struct DevScTables {
    int32_t* ids = nullptr;
    T* coef = nullptr;
    int64_t n_patches = 0;
    bool ready = false;
};

// Device copy of the column-cache schedule (cc_schedule.hpp) for one (T, nlev): records are the
// patch records of kernels_cc.cu (coefficients in T + owned edge ids + slot offsets).
template <class T>
struct DevCcTables {
    CcStep* steps = nullptr;
    CcLoad* loads = nullptr;
    unsigned char* records = nullptr;
    int64_t* cta_patch_begin = nullptr;
    int64_t* cta_step_begin = nullptr;
    int n_ctas = 0, n_slots = 0, slot_bytes = 0;
    int nlev = -1;                 // the level count the slot size was derived from
    int64_t ldk = -1, ldk_w = -1;  // column strides the runs were merged for
    int tile = -1;                 // ICON_OPT_CC_TILE it was built with
    int built_for = 1;             // kCcStep (serves kCcTend too), kCcDivVort (27 vn columns, compact records) or kCcStepW (+3 w columns)
    unsigned long long* progress = nullptr;   // device counter of the producers' pacing barriers, never reset
    int64_t min_steps = 0;         // steps of the CTA with the fewest (pacing barriers every CTA reaches)
    bool ready = false;
    bool unsupported = false;      // this (T, nlev) cannot use the kernel: callers fall back
    int64_t stats[5] = {0, 0, 0, 0, 0};   // steps, steps with reduced depth, vn columns, w columns, bulk copies
};

// per-level coefficients of the vertical term (reading P-14), device copy for one z_half
struct LevelCoeffs {
    std::vector<double> z_half;   // host key
    int dtype = 0;
    void* abc = nullptr;          // device [3][nlev] of T: A_k, B_k, C_k
    void* wk = nullptr;           // device [2][nlev+1] of T: g_k of vn_ie(k), 1 / (z_half[k-1] - z_half[k+1]) (P-19)
};

struct Workspace {                // unfused pipeline intermediates, [n][ldk] of T
    int dtype = -1;
    int64_t ldk = 0;
    void *vt = nullptr, *ke_e = nullptr, *ke_c = nullptr, *vort = nullptr;
};

struct HostStage {                // device staging for dycore_step_host
    int dtype = -1;
    int64_t ldk = 0, ldk_w = 0;
    void *vn = nullptr, *w = nullptr, *ddt = nullptr, *div = nullptr, *vort = nullptr;
    cudaStream_t stream = nullptr;                      // kernels
    cudaStream_t stream_in = nullptr, stream_out = nullptr;      // host -> device, device -> host copies
    cudaEvent_t ev_vn = nullptr, ev_w = nullptr, ev_dv = nullptr, ev_t = nullptr;
};

}  // namespace icon

struct icon_grid {
    icon::HostGrid host;
    unsigned flags = 0;
    uint64_t seed = 0;
    bool host_only = false;
    bool worklist = false;        // work order differs from user order
    int device = -1;
    int num_sms = 0;
    icon::DevTables tab;
    icon::DevCoeffs<double> c64;
    icon::DevCoeffs<float> c32;
    icon::ScTables sc_host;                            // built on first use of the self-contained kernel
    bool sc_host_ready = false;
    icon::DevScTables<double> s64;
    icon::DevScTables<float> s32;
    icon::DevCcTables<double> cc64;                    // built on first use of the column-cache kernel
    icon::DevCcTables<float> cc32;
    icon::DevCcTables<double> dv64;                    // the same for dycore_div_vort (mode kCcDivVort)
    icon::DevCcTables<float> dv32;
    icon::DevCcTables<double> sw64;                    // the same for dycore_step_w (mode kCcStepW)
    icon::DevCcTables<float> sw32;
    icon::DevCcTables<double> wt64;                    // the same for dycore_w_tendency (mode kCcWTend)
    icon::DevCcTables<float> wt32;
    icon::DevCcTables<double> m64;                     // the same for dycore_velocity_tendencies_metric (mode kCcTendM)
    icon::DevCcTables<float> m32;
    int smem_optin = 0;                                // cudaDevAttrMaxSharedMemoryPerBlockOptin
    std::vector<icon::LevelCoeffs> level_coeffs;
    icon::Workspace ws;
    icon::HostStage stage;
    std::map<std::pair<int, int>, void*> public_dev;   // (which, dtype) -> device copy in user order
    std::vector<void*> owned;                          // every device allocation, freed on destroy
    int options[8] = {0};
    int64_t launches = 0;
    icon::PartTables part;                             // part.n_parts > 0: the local grid of one rank (icon_grid_create_part)
    int32_t* d_send_ids[2] = {nullptr, nullptr};       // device copies of part.send_ids (dycore_halo_pack)
};
