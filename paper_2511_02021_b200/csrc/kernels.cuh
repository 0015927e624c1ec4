// kernels.cuh -- launcher declarations of the sm_100a kernels (internal).
#pragma once
#include <cuda_runtime.h>

#include <cstdint>

#include "device_grid.hpp"

namespace icon {

// S1 + S2 in one launch. Returns the number of kernels launched (>0) or a negative cudaError.
template <class T>
int launch_div_vort(const icon_grid& g, const DevCoeffs<T>& c, int nlev, int64_t ldk, const T* vn, T* div, T* vort,
                    cudaStream_t s);

// S3-S7, unfused: vt/KE_e -> KE_c, zeta -> ddt_vn, intermediates in HBM (workspace or the
// caller's optional outputs).
template <class T>
int launch_tendencies_unfused(const icon_grid& g, const DevCoeffs<T>& c, int nlev, int64_t ldk, int64_t ldk_w,
                              const T* abc, const T* vn, const T* w, T* ddt_vn, T* vt, T* ke_e, T* ke_c, T* vort,
                              cudaStream_t s);

// Vertical-wind tendency (reading P-19): wk = device [2][nlev+1], g_k and 1 / (z_half[k-1] - z_half[k+1]).
template <class T>
int launch_w_tendency(const icon_grid& g, const DevCoeffs<T>& c, int nlev, int64_t ldk, int64_t ldk_w, const T* wk,
                      const T* vn, const T* w, T* ddt_w, cudaStream_t s);

// Metric variant (reading P-20): set-up of the per-edge vertical metrics, and the unfused pipeline with its metric last stage.
// dycore_halo_pack: out[i] = rows[ids[i]], rows of row_bytes (a multiple of 16) bytes
int launch_halo_pack(const int32_t* ids, int64_t n_rows, int64_t row_bytes, const void* field, void* out, cudaStream_t s);

template <class T>
int launch_metric_from_zhalf(const icon_grid& g, int nlev, int64_t ldk, int64_t ldk_w, const T* zh, T* wgt, T* inv, cudaStream_t s);
template <class T>
int launch_tendencies_unfused_metric(const icon_grid& g, const DevCoeffs<T>& c, int nlev, int64_t ldk, int64_t ldk_w, const T* wgt,
                                     const T* inv, const T* zn, const T* zt, const T* vn, const T* w, T* ddt_vn, T* vt, T* ke_e,
                                     T* ke_c, T* vort, cudaStream_t s);

// S2-S7, self-contained patch kernel (kernels_sc.cu): one warp per patch, all level chunks of a
// column in flight at once, no exchange between warps; reads vn, w and the records, writes ddt_vn.
template <class T>
int launch_tendencies_sc(const icon_grid& g, const DevScTables<T>& p, int nlev, int64_t ldk, int64_t ldk_w,
                         const T* abc, const T* vn, const T* w, T* ddt_vn, cudaStream_t s);

// S2-S7, column-cache kernel (kernels_cc.cu): a producer warp streams whole vn / w columns into
// shared-memory slots with bulk asynchronous copies following the host-built schedule
// (cc_schedule.hpp); consumer warps finish one self-contained patch each from the slots. mode = kCcTend (ddt_vn),
// kCcStep (ddt_vn + div + vort in one pass: dycore_step) or kCcDivVort (div + vort only, tables built for that mode).
// device pointers of the metric columns of reading P-20 (mode kCcTendM)
template <class T>
struct CcMetric {
    const T *wgt, *inv, *zn, *zt;      // wgt_e [ne][ldk_w]; inv_ddqz_e, ddxn_z, ddxt_z [ne][ldk]
};
template <class T>
int launch_tendencies_cc(const icon_grid& g, DevCcTables<T>& p, int mode, int nlev, int64_t ldk, int64_t ldk_w,
                         const T* abc, const T* vn, const T* w, T* ddt_vn, T* div, T* vort, cudaStream_t s,
                         const T* wk = nullptr, T* ddt_w = nullptr, const CcMetric<T>* met = nullptr);
// shape helpers of that kernel: level mapping (values a lane holds per column; 0 = nlev not supported), bytes of one w column
// (the smallest possible slot), and how many slots of `slot_bytes` fit beside the fixed buffers in `smem_optin` bytes of shared memory
int cc_levels_per_lane(int nlev);
template <class T>
int cc_slot_bytes(int nlev);
template <class T>
int cc_max_slots(int slot_bytes, int smem_optin, int mode, int nlev);
int cc_patches_per_step_for(int nlev, int elem_bytes, int mode);
int cc_level_mapping(int nlev, int elem_bytes, int mode);     // template parameter L of the kernel for this level count, element size and mode

}  // namespace icon
