// api.cu -- the C-ABI of libicon_dycore (include/icon_dycore.h): argument checks, table upload,
// per-call coefficient preparation and kernel launches on the caller's stream. No torch types,
// no CPU fallback: every compute entry point fails with ICON_ECUDA when no device is usable.
#include <cuda_runtime.h>

#include <algorithm>
#include <cstring>
#include <mutex>
#include <new>
#include <string>
#include <type_traits>
#include <vector>

#include "../../include/icon_dycore.h"
#include "device_grid.hpp"
#include "kernels.cuh"

namespace {

thread_local std::string t_last_error;

int fail(int code, const std::string& msg) {
    t_last_error = msg;
    return code;
}
int fail_cuda(cudaError_t e, const char* what) {
    t_last_error = std::string(what) + ": " + cudaGetErrorString(e);
    return ICON_ECUDA;
}

#define CU_TRY(expr)                                      \
    do {                                                  \
        cudaError_t _e = (expr);                          \
        if (_e != cudaSuccess) return fail_cuda(_e, #expr); \
    } while (0)

template <class T>
int dev_alloc(icon_grid* g, size_t count, T** out) {
    void* p = nullptr;
    cudaError_t e = cudaMalloc(&p, count * sizeof(T) + 16);
    if (e != cudaSuccess) {
        t_last_error = std::string("cudaMalloc: ") + cudaGetErrorString(e);
        return e == cudaErrorMemoryAllocation ? ICON_ENOMEM : ICON_ECUDA;
    }
    g->owned.push_back(p);
    *out = static_cast<T*>(p);
    return ICON_OK;
}
void dev_release(icon_grid* g, void* p) {
    if (!p) return;
    for (auto& q : g->owned)
        if (q == p) {
            cudaFree(p);
            q = nullptr;
        }
}

// upload rows of `src` ([n][cols], user order) to the device; when user_of_pos is non-empty the
// device copy is in work order: row p = src row user_of_pos[p].
template <class S, class D>
int upload_rows(icon_grid* g, const std::vector<S>& src, int cols, const std::vector<int32_t>& user_of_pos, D** out) {
    const size_t n = src.size() / (size_t)cols;
    std::vector<D> tmp(src.size());
    if (user_of_pos.empty()) {
        for (size_t i = 0; i < src.size(); ++i) tmp[i] = (D)src[i];
    } else {
#pragma omp parallel for schedule(static)
        for (int64_t p = 0; p < (int64_t)n; ++p)
            for (int s = 0; s < cols; ++s) tmp[(size_t)p * cols + s] = (D)src[(size_t)user_of_pos[p] * cols + s];
    }
    int rc = dev_alloc(g, tmp.size(), out);
    if (rc != ICON_OK) return rc;
    CU_TRY(cudaMemcpy(*out, tmp.data(), tmp.size() * sizeof(D), cudaMemcpyHostToDevice));
    return ICON_OK;
}

int upload_inverse(icon_grid* g, const std::vector<int32_t>& user_of_pos, int32_t** out_user, int32_t** out_pos) {
    if (user_of_pos.empty()) return ICON_OK;
    std::vector<int32_t> pos(user_of_pos.size());
    for (size_t p = 0; p < user_of_pos.size(); ++p) pos[(size_t)user_of_pos[p]] = (int32_t)p;
    int rc = dev_alloc(g, pos.size(), out_user);
    if (rc != ICON_OK) return rc;
    CU_TRY(cudaMemcpy(*out_user, user_of_pos.data(), pos.size() * 4, cudaMemcpyHostToDevice));
    rc = dev_alloc(g, pos.size(), out_pos);
    if (rc != ICON_OK) return rc;
    CU_TRY(cudaMemcpy(*out_pos, pos.data(), pos.size() * 4, cudaMemcpyHostToDevice));
    return ICON_OK;
}

const std::vector<int32_t> kIdentity;

int upload_index_tables(icon_grid* g) {
    const icon::HostGrid& h = g->host;
    const auto& uc = g->worklist ? h.user_of_pos_c : kIdentity;
    const auto& ue = g->worklist ? h.user_of_pos_e : kIdentity;
    const auto& uv = g->worklist ? h.user_of_pos_v : kIdentity;
    int rc;
    if ((rc = upload_rows(g, h.c2e, 3, uc, &g->tab.c2e))) return rc;
    if ((rc = upload_rows(g, h.e2c, 2, ue, &g->tab.e2c))) return rc;
    if ((rc = upload_rows(g, h.e2v, 2, ue, &g->tab.e2v))) return rc;
    if ((rc = upload_rows(g, h.e2e4, 4, ue, &g->tab.e2e4))) return rc;
    if ((rc = upload_rows(g, h.v2e, 6, uv, &g->tab.v2e))) return rc;
    if ((rc = upload_inverse(g, uc, &g->tab.user_c, &g->tab.pos_c))) return rc;
    if ((rc = upload_inverse(g, ue, &g->tab.user_e, &g->tab.pos_e))) return rc;
    if ((rc = upload_inverse(g, uv, &g->tab.user_v, &g->tab.pos_v))) return rc;
    return ICON_OK;
}

template <class T>
int ensure_coeffs(icon_grid* g, icon::DevCoeffs<T>& c) {
    if (c.ready) return ICON_OK;
    if (g->part.n_parts)      // a local grid holds patch records only: no global tables to upload
        return fail(ICON_EUNSUPPORTED, "this call (or this kernel option / level count) needs the global tables: not available on a grid made by icon_grid_create_part");
    const icon::HostGrid& h = g->host;
    const auto& uc = g->worklist ? h.user_of_pos_c : kIdentity;
    const auto& ue = g->worklist ? h.user_of_pos_e : kIdentity;
    const auto& uv = g->worklist ? h.user_of_pos_v : kIdentity;
    int rc;
    if ((rc = upload_rows(g, h.rbf, 4, ue, &c.rbf))) return rc;
    if ((rc = upload_rows(g, h.bln, 3, uc, &c.bln))) return rc;
    if ((rc = upload_rows(g, h.geofac_div, 3, uc, &c.geofac_div))) return rc;
    if ((rc = upload_rows(g, h.geofac_rot, 6, uv, &c.geofac_rot))) return rc;
    if ((rc = upload_rows(g, h.inv_d_e, 1, ue, &c.inv_d_e))) return rc;
    if ((rc = upload_rows(g, h.f_e, 1, ue, &c.f_e))) return rc;
    if ((rc = upload_rows(g, h.c_lin, 2, ue, &c.c_lin))) return rc;
    if ((rc = upload_rows(g, h.adv_c, 3, uc, &c.adv_c))) return rc;
    if ((rc = upload_rows(g, h.cgrad, 2, ue, &c.cgrad))) return rc;
    CU_TRY(cudaStreamSynchronize(cudaStreamLegacy));      // uploads ran on the legacy stream, callers may use non-blocking streams
    c.ready = true;
    return ICON_OK;
}

template <class D, class S>
int upload_vec(icon_grid* g, const std::vector<S>& src, D** out) {
    std::vector<D> conv;
    const D* data;
    if constexpr (std::is_same<D, S>::value) {
        data = src.data();
    } else {
        conv.assign(src.begin(), src.end());
        data = conv.data();
    }
    int rc = dev_alloc(g, src.size() ? src.size() : 1, out);
    if (rc != ICON_OK) return rc;
    if (!src.empty()) CU_TRY(cudaMemcpy(*out, data, src.size() * sizeof(D), cudaMemcpyHostToDevice));
    return ICON_OK;
}

int ensure_sc_host(icon_grid* g);

template <class T>
int ensure_sc_tables(icon_grid* g, icon::DevScTables<T>& p) {
    if (p.ready) return ICON_OK;
    int rc = ensure_sc_host(g);
    if (rc) return rc;
    if ((rc = upload_vec(g, g->sc_host.ids, &p.ids))) return rc;
    if ((rc = upload_vec(g, g->sc_host.coef, &p.coef))) return rc;
    p.n_patches = g->sc_host.n_patches;
    CU_TRY(cudaStreamSynchronize(cudaStreamLegacy));
    p.ready = true;
    return ICON_OK;
}

int ensure_sc_host(icon_grid* g) {
    if (g->sc_host_ready) return ICON_OK;
    std::string err;
    try {
        err = icon::build_sc_tables(g->host, g->sc_host);
    } catch (const std::bad_alloc&) {
        return fail(ICON_ENOMEM, "out of host memory while building the patch records");
    }
    if (!err.empty()) return fail(ICON_EUNSUPPORTED, err);
    g->sc_host_ready = true;
    return ICON_OK;
}

// A slot as large as the caller's column stride lets runs of consecutive columns arrive as one bulk
// copy (the copy engine, not HBM, limits small copies); taken when it costs < 128 bytes per slot.
template <class T>
icon::CcGeometry cc_geometry(int nlev, int64_t ldk, int64_t ldk_w, bool dv = false) {
    icon::CcGeometry geom;
    geom.col_bytes[0] = (nlev * (int)sizeof(T) + 15) & ~15;
    geom.col_bytes[1] = dv ? geom.col_bytes[0] : icon::cc_slot_bytes<T>(nlev);      // div / vort only: no w column
    geom.stride_bytes[0] = (int)(ldk * (int64_t)sizeof(T));
    geom.stride_bytes[1] = (int)(ldk_w * (int64_t)sizeof(T));
    geom.slot_bytes = geom.col_bytes[1];
    if (geom.stride_bytes[0] >= geom.col_bytes[1] && geom.stride_bytes[0] < geom.col_bytes[1] + 128)
        geom.slot_bytes = geom.stride_bytes[0];
    return geom;
}

template <class T>
constexpr int cc_record_size(int mode) { return icon::cc_coef_words(mode) * (int)sizeof(T) + icon::kCcRecordTail; }

// ICON_OPT_CC_TILE -1 = auto: 16 patches for deep 8-byte columns (a tile then just fits the slot pool), 64 where the
// columns are short or 4-byte wide (three to four times as many slots; measured config 5: 8.56 -> 8.30 ms, config 4
// tendency 2.86 -> 2.71 ms)
template <class T>
int cc_resolve_tile(const icon_grid* g, int nlev) {
    const int opt = g->options[ICON_OPT_CC_TILE];
    if (opt >= 0) return opt;
    return sizeof(T) == 8 && icon::cc_levels_per_lane(nlev) == 3 ? 16 : 64;
}

// Column-cache schedule + patch records for (T, nlev, mode): built on the host once, uploaded once.
// Returns ICON_OK with p.unsupported set when this (T, nlev) cannot use the kernel (the caller
// then uses the self-contained patch kernel).
template <class T>
int ensure_cc_tables(icon_grid* g, icon::DevCcTables<T>& p, int nlev, int64_t ldk, int64_t ldk_w, int mode = icon::kCcStep) {
    const int tile = cc_resolve_tile<T>(g, nlev);
    const bool dv = mode == icon::kCcDivVort;
    if (p.nlev == nlev && p.ldk == ldk && p.ldk_w == ldk_w && p.tile == tile && (p.ready || p.unsupported))
        return ICON_OK;
    dev_release(g, p.steps); dev_release(g, p.loads); dev_release(g, p.records);
    dev_release(g, p.cta_patch_begin); dev_release(g, p.cta_step_begin); dev_release(g, p.progress);
    p = icon::DevCcTables<T>();
    p.nlev = nlev;
    p.ldk = ldk; p.ldk_w = ldk_w; p.tile = tile; p.built_for = mode;
    const icon::CcGeometry geom = cc_geometry<T>(nlev, ldk, ldk_w, dv);
    const int slot_bytes = geom.slot_bytes;
    const int n_slots_max = icon::cc_max_slots<T>(slot_bytes, g->smem_optin, mode, nlev);
    if (icon::cc_levels_per_lane(nlev) == 0 || nlev * (int)sizeof(T) < 16 || n_slots_max < icon::kScIdWords) {
        p.unsupported = true;
        return ICON_OK;
    }
    int rc = ensure_sc_host(g);
    if (rc) return rc;
    const icon::ScTables& sc = g->sc_host;
    const int n_slots = std::min(n_slots_max, 65535);
    icon::CcSchedule cs;
    std::vector<unsigned char> rec;
    const size_t rb = (size_t)cc_record_size<T>(mode);
    const int ncoef = icon::cc_coef_words(mode);
    try {
        std::string err = icon::build_cc_schedule(sc, g->num_sms, n_slots, geom, icon::cc_patches_per_step_for(nlev, (int)sizeof(T), mode), icon::kCcDepth, tile, icon::cc_use_mask(mode), cs);
        if (!err.empty()) {
            p.unsupported = true;
            return ICON_OK;
        }
        rec.assign((size_t)sc.n_patches * rb, 0);
#pragma omp parallel for schedule(static)
        for (int64_t q = 0; q < sc.n_patches; ++q) {
            unsigned char* r = rec.data() + (size_t)q * rb;
            T* cf = reinterpret_cast<T*>(r);
            const int64_t src = cs.patch_order[(size_t)q];       // record q belongs to work position q
            const double* scf = &sc.coef[(size_t)src * icon::kScCoefWords];
            if (dv) {          // compact record: geofac_div, rot of the midpoints, rot of the corners
                for (int i = 0; i < 12; ++i) cf[icon::DVF_DIV + i] = (T)scf[icon::SCF_DIV + i];
                for (int i = 0; i < 20; ++i) cf[icon::DVF_ROT + i] = (T)scf[icon::SCF_ROT + i];
                for (int i = 0; i < 20; ++i) cf[icon::DVF_XROT + i] = (T)(i < 18 ? scf[icon::SCF_XROT + i] : 0.0);
            } else if (mode == icon::kCcWTend) {          // compact record: the twelve advection coefficients
                for (int i = 0; i < icon::kCcWCoefWords; ++i) cf[icon::WF_ADV + i] = (T)scf[icon::SCF_ADV + i];
            } else {
                for (int i = 0; i < ncoef; ++i) cf[i] = (T)scf[i];      // kCcStepW: with the twelve advection coefficients
            }
            int32_t* oid = reinterpret_cast<int32_t*>(r + (size_t)ncoef * sizeof(T));
            const int32_t* id = &sc.ids[(size_t)src * icon::kScIdWords];
            for (int x = 0; x < 3; ++x) {
                oid[x] = id[icon::SID_I0 + x];
                oid[3 + x] = id[icon::SID_B0 + 2 * x];
            }
            for (int x = 0; x < 4; ++x) oid[6 + x] = id[icon::SID_T0 + x];
            for (int x = 0; x < 6; ++x) oid[10 + x] = id[icon::SID_V0 + x];
            for (int x = 0; x < 6 && !dv && mode != icon::kCcWTend; ++x) {   // c_lin halved: the kernel forms w(k) + w(k+1) (exact scaling)
                cf[icon::SCF_EDGE + 4 * x + 2] *= (T)0.5;
                cf[icon::SCF_EDGE + 4 * x + 3] *= (T)0.5;
            }
            uint32_t* so = reinterpret_cast<uint32_t*>(r + (size_t)ncoef * sizeof(T) + 4 * icon::kCcRecordIds);
            for (int i = 0; i < icon::kCcSlotWords; ++i)
                so[i] = (uint32_t)cs.patch_slots[(size_t)q * icon::kCcSlotWords + i] * (uint32_t)slot_bytes;
            so[icon::kCcMaskWord] = cs.patch_slots[(size_t)q * icon::kCcSlotWords + icon::kCcMaskWord];
        }
    } catch (const std::bad_alloc&) {
        return fail(ICON_ENOMEM, "out of host memory while building the column-cache schedule");
    }
    if ((rc = upload_vec(g, cs.steps, &p.steps))) return rc;
    if ((rc = upload_vec(g, cs.loads, &p.loads))) return rc;
    if ((rc = upload_vec(g, rec, &p.records))) return rc;
    if ((rc = upload_vec(g, cs.cta_patch_begin, &p.cta_patch_begin))) return rc;
    if ((rc = upload_vec(g, cs.cta_step_begin, &p.cta_step_begin))) return rc;
    p.n_ctas = cs.n_ctas; p.n_slots = cs.n_slots; p.slot_bytes = slot_bytes;
    p.min_steps = 1 << 30;
    for (int b = 0; b < cs.n_ctas; ++b) p.min_steps = std::min(p.min_steps, cs.cta_step_begin[(size_t)b + 1] - cs.cta_step_begin[(size_t)b]);
    if ((rc = dev_alloc(g, 1, &p.progress))) return rc;
    CU_TRY(cudaMemset(p.progress, 0, sizeof(unsigned long long)));
    // table uploads and the memset ran on the legacy stream; the caller's stream may be non-blocking
    CU_TRY(cudaStreamSynchronize(cudaStreamLegacy));
    p.stats[0] = (int64_t)cs.steps.size(); p.stats[1] = cs.n_sync_steps; p.stats[2] = cs.n_vn_loads; p.stats[3] = cs.n_w_loads;
    p.stats[4] = cs.n_copies;
    p.ready = true;
    return ICON_OK;
}

// Reading P-14 folded into three per-level coefficients:
//   (vn_ie(k) - vn_ie(k+1)) / dz_k = A_k vn(k-1) + B_k vn(k) + C_k vn(k+1)
// half level kh is a two-point linear combination of full levels: interior kh uses (kh, kh-1)
// with weights (g, 1-g), g = dz_{kh-1}/(dz_{kh-1}+dz_kh); kh = 0 and kh = K extrapolate linearly in
// z from the two nearest full levels.
void vertical_coefficients(const double* zh, int K, std::vector<double>& abc) {
    abc.assign(3 * (size_t)K, 0.0);
    auto zf = [&](int k) { return 0.5 * (zh[k] + zh[k + 1]); };
    auto add_half = [&](int k, int kh, double sign) {
        int ia, ib;
        double ca, cb;
        if (kh == 0) {
            double r = (zh[0] - zf(0)) / (zf(0) - zf(1));
            ia = 0; ca = 1.0 + r; ib = 1; cb = -r;
        } else if (kh == K) {
            double r = (zh[K] - zf(K - 1)) / (zf(K - 1) - zf(K - 2));
            ia = K - 1; ca = 1.0 + r; ib = K - 2; cb = -r;
        } else {
            double up = zh[kh - 1] - zh[kh], dn = zh[kh] - zh[kh + 1];
            double gk = up / (up + dn);
            ia = kh; ca = gk; ib = kh - 1; cb = 1.0 - gk;
        }
        const double inv_dz = 1.0 / (zh[k] - zh[k + 1]);
        abc[(size_t)(ia - k + 1) * K + k] += sign * ca * inv_dz;
        abc[(size_t)(ib - k + 1) * K + k] += sign * cb * inv_dz;
    };
    for (int k = 0; k < K; ++k) {
        add_half(k, k, +1.0);
        add_half(k, k + 1, -1.0);
    }
}

int get_level_coeffs(icon_grid* g, int dtype, int nlev, const double* z_half, void** out, void** out_wk = nullptr) {
    for (int k = 0; k < nlev; ++k)
        if (!(z_half[k] > z_half[k + 1])) return fail(ICON_EINVAL, "z_half must be strictly decreasing");
    for (auto& lc : g->level_coeffs)
        if (lc.dtype == dtype && (int)lc.z_half.size() == nlev + 1 &&
            std::memcmp(lc.z_half.data(), z_half, sizeof(double) * (nlev + 1)) == 0) {
            *out = lc.abc;
            if (out_wk) *out_wk = lc.wk;
            return ICON_OK;
        }
    std::vector<double> abc;
    vertical_coefficients(z_half, nlev, abc);
    // P-19: g_k = dz_{k-1} / (dz_{k-1} + dz_k) (weight of vn(k) in vn_ie(k)) and 1 / (z_half[k-1] - z_half[k+1]), k = 1 .. nlev-1
    std::vector<double> wk(2 * ((size_t)nlev + 1), 0.0);
    for (int k = 1; k <= nlev - 1; ++k) {
        const double up = z_half[k - 1] - z_half[k], dn = z_half[k] - z_half[k + 1];
        wk[(size_t)k] = up / (up + dn);
        wk[(size_t)nlev + 1 + k] = 1.0 / (z_half[k - 1] - z_half[k + 1]);
    }
    icon::LevelCoeffs lc;
    lc.dtype = dtype;
    lc.z_half.assign(z_half, z_half + nlev + 1);
    int rc;
    if (dtype == ICON_F64) {
        double* d = nullptr;
        if ((rc = dev_alloc(g, abc.size(), &d))) return rc;
        CU_TRY(cudaMemcpy(d, abc.data(), abc.size() * 8, cudaMemcpyHostToDevice));
        lc.abc = d;
        double* dw = nullptr;
        if ((rc = dev_alloc(g, wk.size(), &dw))) return rc;
        CU_TRY(cudaMemcpy(dw, wk.data(), wk.size() * 8, cudaMemcpyHostToDevice));
        lc.wk = dw;
    } else {
        std::vector<float> f(abc.begin(), abc.end());
        float* d = nullptr;
        if ((rc = dev_alloc(g, f.size(), &d))) return rc;
        CU_TRY(cudaMemcpy(d, f.data(), f.size() * 4, cudaMemcpyHostToDevice));
        lc.abc = d;
        std::vector<float> fw(wk.begin(), wk.end());
        float* dw = nullptr;
        if ((rc = dev_alloc(g, fw.size(), &dw))) return rc;
        CU_TRY(cudaMemcpy(dw, fw.data(), fw.size() * 4, cudaMemcpyHostToDevice));
        lc.wk = dw;
    }
    // the coefficients are cached per z_half and reused by later calls on ANY stream: the upload (legacy stream) must
    // have landed before this call's kernel, which may run on a non-blocking stream, reads them
    CU_TRY(cudaStreamSynchronize(cudaStreamLegacy));
    if (g->level_coeffs.size() >= 16) {   // bounded cache
        dev_release(g, g->level_coeffs.front().abc);
        dev_release(g, g->level_coeffs.front().wk);
        g->level_coeffs.erase(g->level_coeffs.begin());
    }
    g->level_coeffs.push_back(lc);
    *out = lc.abc;
    if (out_wk) *out_wk = lc.wk;
    return ICON_OK;
}

int check_field(const void* p, const char* name) {
    if (!p) return fail(ICON_EINVAL, std::string(name) + " is NULL");
    if (reinterpret_cast<uintptr_t>(p) % 16) return fail(ICON_EINVAL, std::string(name) + " is not 16-byte aligned");
    return ICON_OK;
}

// true when the byte ranges [a, a + na) and [b, b + nb) intersect
bool overlaps(const void* a, size_t na, const void* b, size_t nb) {
    const uintptr_t pa = reinterpret_cast<uintptr_t>(a), pb = reinterpret_cast<uintptr_t>(b);
    return a && b && pa < pb + nb && pb < pa + na;
}

int check_device(const icon_grid* g) {
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return fail_cuda(e, "cudaGetDevice");
    if (dev != g->device) return fail(ICON_EINVAL, "the current CUDA device is not the device the grid was created on");
    return ICON_OK;
}

int check_common(icon_grid* g, int dtype, int nlev, int ldk, int min_lev) {
    if (!g) return fail(ICON_EINVAL, "grid handle is NULL");
    if (g->host_only) return fail(ICON_ECUDA, "grid was created with ICON_HOST_ONLY: no device tables, and there is no CPU path");
    if (int rc = check_device(g)) return rc;
    if (dtype != ICON_F64 && dtype != ICON_F32) return fail(ICON_EINVAL, "dtype must be ICON_F64 or ICON_F32");
    if (nlev < min_lev || nlev > 4096) return fail(ICON_EINVAL, "nlev out of range");
    if (ldk < nlev) return fail(ICON_EINVAL, "ldk < nlev");
    const int es = dtype == ICON_F64 ? 8 : 4;
    if (((int64_t)ldk * es) % 16) return fail(ICON_EINVAL, "ldk*sizeof(T) must be a multiple of 16");
    return ICON_OK;
}

template <class T>
int ensure_workspace(icon_grid* g, int dtype, int64_t ldk) {
    icon::Workspace& ws = g->ws;
    if (ws.dtype == dtype && ws.ldk == ldk) return ICON_OK;
    dev_release(g, ws.vt); dev_release(g, ws.ke_e); dev_release(g, ws.ke_c); dev_release(g, ws.vort);
    ws = icon::Workspace();
    int rc;
    T *a, *b, *c, *d;
    if ((rc = dev_alloc(g, (size_t)(g->host.ne * ldk), &a))) return rc;
    if ((rc = dev_alloc(g, (size_t)(g->host.ne * ldk), &b))) return rc;
    if ((rc = dev_alloc(g, (size_t)(g->host.nc * ldk), &c))) return rc;
    if ((rc = dev_alloc(g, (size_t)(g->host.nv * ldk), &d))) return rc;
    ws.vt = a; ws.ke_e = b; ws.ke_c = c; ws.vort = d;
    ws.dtype = dtype; ws.ldk = ldk;
    return ICON_OK;
}

template <class T>
int tendencies_impl(icon_grid* g, icon::DevCoeffs<T>& c, icon::DevScTables<T>& st, icon::DevCcTables<T>& ct, int dtype, int nlev, int ldk, int ldk_w, const double* z_half,
                    const void* vn, const void* w, void* ddt_vn, void* vt_opt, void* ke_c_opt, void* vort_opt,
                    cudaStream_t s, void* div_fused = nullptr, void* vort_fused = nullptr, bool* fused_done = nullptr) {
    // div_fused / vort_fused: dycore_step asks for S1 + S2 from the same pass; only the column-cache kernel can
    // (it sets *fused_done), with any other kernel the caller launches dycore_div_vort afterwards
    int rc;
    if (!g->part.n_parts && (rc = ensure_coeffs(g, c))) return rc;
    void* abc = nullptr;
    if ((rc = get_level_coeffs(g, dtype, nlev, z_half, &abc))) return rc;
    const bool want_opt = vt_opt || ke_c_opt || vort_opt;
    int n;
    int variant = g->options[ICON_OPT_TENDENCY_KERNEL];
    if (variant == 5) variant = 4;            // auto: the column cache wherever it can hold the columns (nlev <= 95)
    if (variant == 4 && !want_opt) {
        if ((rc = ensure_cc_tables(g, ct, nlev, ldk, ldk_w))) return rc;
        if (ct.unsupported) variant = 3;      // level count the column cache cannot hold
    }
    if (g->part.n_parts && (variant != 4 || want_opt) && (rc = ensure_coeffs(g, c))) return rc;      // fails: column cache only
    if (variant != 4 || want_opt) div_fused = vort_fused = nullptr;
    if (fused_done) *fused_done = div_fused != nullptr;
    if (variant == 4 && !want_opt) {
        n = icon::launch_tendencies_cc<T>(*g, ct, div_fused ? icon::kCcStep : icon::kCcTend, nlev, ldk, ldk_w, (const T*)abc, (const T*)vn,
                                          (const T*)w, (T*)ddt_vn, (T*)div_fused, (T*)vort_fused, s);
    } else if (variant == 0 || want_opt) {
        // optional outputs are produced by the unfused pipeline, which materialises them anyway
        if ((rc = ensure_workspace<T>(g, dtype, ldk))) return rc;
        T* vt = vt_opt ? (T*)vt_opt : (T*)g->ws.vt;
        T* kc = ke_c_opt ? (T*)ke_c_opt : (T*)g->ws.ke_c;
        T* vo = vort_opt ? (T*)vort_opt : (T*)g->ws.vort;
        n = icon::launch_tendencies_unfused<T>(*g, c, nlev, ldk, ldk_w, (const T*)abc, (const T*)vn, (const T*)w,
                                               (T*)ddt_vn, vt, (T*)g->ws.ke_e, kc, vo, s);
    } else {
        if ((rc = ensure_sc_tables(g, st))) return rc;
        n = icon::launch_tendencies_sc<T>(*g, st, nlev, ldk, ldk_w, (const T*)abc, (const T*)vn, (const T*)w,
                                          (T*)ddt_vn, s);
    }
    if (n < 0) return fail_cuda((cudaError_t)(-n), "kernel launch");
    g->launches += n;
    return ICON_OK;
}

struct TableInfo {
    const void* ptr;
    int dtype;
    int64_t rows;
    int cols;
};
int table_info(const icon_grid* g, int which, TableInfo* t) {
    if (g->part.n_parts) return fail(ICON_EUNSUPPORTED, "a grid made by icon_grid_create_part holds no global tables (icon_part_table has the local ones)");
    const icon::HostGrid& h = g->host;
    auto I = [&](const std::vector<int32_t>& v, int64_t rows, int cols) { *t = {v.data(), ICON_T_I32, rows, cols}; };
    auto B = [&](const std::vector<int8_t>& v, int64_t rows, int cols) { *t = {v.data(), ICON_T_I8, rows, cols}; };
    auto D = [&](const std::vector<double>& v, int64_t rows, int cols) { *t = {v.data(), ICON_T_F64, rows, cols}; };
    switch (which) {
        case ICON_TAB_C2V: I(h.c2v, h.nc, 3); break;
        case ICON_TAB_C2E: I(h.c2e, h.nc, 3); break;
        case ICON_TAB_E2C: I(h.e2c, h.ne, 2); break;
        case ICON_TAB_E2V: I(h.e2v, h.ne, 2); break;
        case ICON_TAB_E2E4: I(h.e2e4, h.ne, 4); break;
        case ICON_TAB_V2E: I(h.v2e, h.nv, 6); break;
        case ICON_TAB_V2C: I(h.v2c, h.nv, 6); break;
        case ICON_TAB_V_DEG: I(h.v_deg, h.nv, 1); break;
        case ICON_TAB_C_OS: B(h.c_os, h.nc, 3); break;
        case ICON_TAB_V_OS: B(h.v_os, h.nv, 6); break;
        case ICON_TAB_VERT_XYZ: D(h.vert_xyz, h.nv, 3); break;
        case ICON_TAB_CELL_XYZ: D(h.cell_xyz, h.nc, 3); break;
        case ICON_TAB_EDGE_XYZ: D(h.edge_xyz, h.ne, 3); break;
        case ICON_TAB_EDGE_NORMAL: D(h.edge_normal, h.ne, 3); break;
        case ICON_TAB_L_E: D(h.l_e, h.ne, 1); break;
        case ICON_TAB_D_E: D(h.d_e, h.ne, 1); break;
        case ICON_TAB_INV_D_E: D(h.inv_d_e, h.ne, 1); break;
        case ICON_TAB_F_E: D(h.f_e, h.ne, 1); break;
        case ICON_TAB_C_LIN: D(h.c_lin, h.ne, 2); break;
        case ICON_TAB_RBF: D(h.rbf, h.ne, 4); break;
        case ICON_TAB_A_C: D(h.a_c, h.nc, 1); break;
        case ICON_TAB_BLN: D(h.bln, h.nc, 3); break;
        case ICON_TAB_A_V: D(h.a_v, h.nv, 1); break;
        case ICON_TAB_GEOFAC_DIV: D(h.geofac_div, h.nc, 3); break;
        case ICON_TAB_GEOFAC_ROT: D(h.geofac_rot, h.nv, 6); break;
        case ICON_TAB_ADV_C: D(h.adv_c, h.nc, 3); break;
        case ICON_TAB_CGRAD: D(h.cgrad, h.ne, 2); break;
        default: return fail(ICON_EINVAL, "unknown table selector");
    }
    return ICON_OK;
}

}  // namespace

extern "C" {

const char* icon_last_error(void) { return t_last_error.c_str(); }

int icon_grid_create(int bisections_k, uint64_t seed, unsigned flags, icon_grid_t** out) {
    if (!out) return fail(ICON_EINVAL, "out is NULL");
    *out = nullptr;
    if (bisections_k < 0 || bisections_k > 9) return fail(ICON_EINVAL, "bisections_k must be in 0..9");
    if (flags & ~(ICON_PERMUTE | ICON_LOCALITY_WORKLIST | ICON_HOST_ONLY | ICON_NO_WORKLIST))
        return fail(ICON_EINVAL, "unknown flag bits");
    icon_grid* g = new (std::nothrow) icon_grid();
    if (!g) return fail(ICON_ENOMEM, "out of host memory");
    g->flags = flags;
    g->seed = seed;
    g->host_only = (flags & ICON_HOST_ONLY) != 0;
    g->options[ICON_OPT_TENDENCY_KERNEL] = 5;
    g->options[ICON_OPT_CC_TILE] = -1;
    g->options[ICON_OPT_CC_PACE] = 512;
    try {
        std::string err = icon::build_host_grid(bisections_k, seed, (flags & ICON_PERMUTE) != 0, g->host);
        if (!err.empty()) {
            delete g;
            return fail(ICON_EINVAL, err);
        }
    } catch (const std::bad_alloc&) {
        delete g;
        return fail(ICON_ENOMEM, "out of host memory while building the grid");
    }
    // the work order (generation order) differs from the user order only on permuted grids
    g->worklist = (flags & ICON_PERMUTE) && !(flags & ICON_NO_WORKLIST);
    if (!g->host_only) {
        int ndev = 0;
        cudaError_t e = cudaGetDeviceCount(&ndev);
        if (e != cudaSuccess || ndev == 0) {
            delete g;
            return fail(ICON_ECUDA, "no usable CUDA device (there is no CPU fallback)");
        }
        int rc = ICON_OK;
        e = cudaGetDevice(&g->device);
        if (e == cudaSuccess) e = cudaDeviceGetAttribute(&g->num_sms, cudaDevAttrMultiProcessorCount, g->device);
        if (e == cudaSuccess) e = cudaDeviceGetAttribute(&g->smem_optin, cudaDevAttrMaxSharedMemoryPerBlockOptin, g->device);
        if (e != cudaSuccess) rc = fail_cuda(e, "cudaGetDevice");
        if (rc == ICON_OK) rc = upload_index_tables(g);
        if (rc == ICON_OK) rc = ensure_coeffs(g, g->c64);
        if (rc != ICON_OK) {
            std::string keep = t_last_error;
            icon_grid_destroy(g);
            t_last_error = keep;
            return rc;
        }
    }
    *out = g;
    return ICON_OK;
}

void icon_grid_destroy(icon_grid_t* g) {
    if (!g) return;
    for (void* p : g->owned)
        if (p) cudaFree(p);
    if (g->stage.stream) cudaStreamDestroy(g->stage.stream);
    if (g->stage.stream_in) cudaStreamDestroy(g->stage.stream_in);
    if (g->stage.stream_out) cudaStreamDestroy(g->stage.stream_out);
    for (cudaEvent_t e : {g->stage.ev_vn, g->stage.ev_w, g->stage.ev_dv, g->stage.ev_t})
        if (e) cudaEventDestroy(e);
    delete g;
}

int icon_grid_counts(const icon_grid_t* g, int64_t* nc, int64_t* ne, int64_t* nv) {
    if (!g) return fail(ICON_EINVAL, "grid handle is NULL");
    if (nc) *nc = g->host.nc;
    if (ne) *ne = g->host.ne;
    if (nv) *nv = g->host.nv;
    return ICON_OK;
}

int icon_grid_table_host(const icon_grid_t* g, int which, const void** ptr, int* dtype, int64_t* rows, int* cols) {
    if (!g) return fail(ICON_EINVAL, "grid handle is NULL");
    TableInfo t;
    int rc = table_info(g, which, &t);
    if (rc) return rc;
    if (ptr) *ptr = t.ptr;
    if (dtype) *dtype = t.dtype;
    if (rows) *rows = t.rows;
    if (cols) *cols = t.cols;
    return ICON_OK;
}

int icon_grid_table_device(const icon_grid_t* gc, int which, int dtype, const void** dptr) {
    icon_grid* g = const_cast<icon_grid*>(gc);       // logically const: the device copies are a cache
    if (!g || !dptr) return fail(ICON_EINVAL, "NULL argument");
    if (g->host_only) return fail(ICON_EUNSUPPORTED, "grid was created with ICON_HOST_ONLY");
    if (int rcd = check_device(g)) return rcd;
    if (dtype != ICON_F64 && dtype != ICON_F32) return fail(ICON_EINVAL, "dtype must be ICON_F64 or ICON_F32");
    TableInfo t;
    int rc = table_info(g, which, &t);
    if (rc) return rc;
    const int key_dtype = t.dtype == ICON_T_F64 ? dtype : -1;
    auto key = std::make_pair(which, key_dtype);
    auto it = g->public_dev.find(key);
    if (it != g->public_dev.end()) {
        *dptr = it->second;
        return ICON_OK;
    }
    const size_t n = (size_t)t.rows * t.cols;
    void* d = nullptr;
    if (t.dtype == ICON_T_F64 && dtype == ICON_F32) {
        const double* src = (const double*)t.ptr;
        std::vector<float> f(src, src + n);
        float* p;
        if ((rc = dev_alloc(g, n, &p))) return rc;
        CU_TRY(cudaMemcpy(p, f.data(), n * 4, cudaMemcpyHostToDevice));
        d = p;
    } else {
        const size_t es = t.dtype == ICON_T_F64 ? 8 : (t.dtype == ICON_T_I32 ? 4 : 1);
        char* p;
        if ((rc = dev_alloc(g, n * es, &p))) return rc;
        CU_TRY(cudaMemcpy(p, t.ptr, n * es, cudaMemcpyHostToDevice));
        d = p;
    }
    g->public_dev[key] = d;
    *dptr = d;
    return ICON_OK;
}

int icon_grid_set_option(icon_grid_t* g, int option, int value) {
    if (!g) return fail(ICON_EINVAL, "grid handle is NULL");
    if (option < 0 || option >= ICON_OPT_COUNT) return fail(ICON_EINVAL, "unknown option");
    if (option == ICON_OPT_CC_PACE && (value < 0 || value > 65536 || (value & (value - 1)))) return fail(ICON_EINVAL, "bad option value");
    if (option == ICON_OPT_CC_TILE && (value < -1 || value > 4096 || (value > 0 && value % 8))) return fail(ICON_EINVAL, "bad option value");
    if (option == ICON_OPT_TENDENCY_KERNEL && value != 0 && value != 3 && value != 4 && value != 5) return fail(ICON_EINVAL, "bad option value");
    g->options[option] = value;
    return ICON_OK;
}

int64_t icon_grid_launch_count(const icon_grid_t* g) { return g ? g->launches : 0; }

// ---- horizontal domain decomposition (reading P-21; partition.hpp) ----------------------------------
int icon_grid_create_part(int bisections_k, unsigned flags, int n_parts, int part, icon_grid_t** out) {
    if (!out) return fail(ICON_EINVAL, "out is NULL");
    *out = nullptr;
    if (bisections_k < 0 || bisections_k > 9) return fail(ICON_EINVAL, "bisections_k must be in 0..9");
    if (flags & ~(unsigned)ICON_HOST_ONLY)
        return fail(ICON_EINVAL, "icon_grid_create_part: flags must be 0 or ICON_HOST_ONLY (a decomposed grid keeps the hierarchical numbering)");
    if (n_parts < 1 || part < 0 || part >= n_parts) return fail(ICON_EINVAL, "icon_grid_create_part: need n_parts >= 1 and 0 <= part < n_parts");
    icon_grid* g = new (std::nothrow) icon_grid();
    if (!g) return fail(ICON_ENOMEM, "out of host memory");
    g->flags = flags;
    g->host_only = (flags & ICON_HOST_ONLY) != 0;
    g->options[ICON_OPT_TENDENCY_KERNEL] = 5;
    g->options[ICON_OPT_CC_TILE] = -1;
    g->options[ICON_OPT_CC_PACE] = 512;
    try {
        // the global grid and its patch records live only inside this block
        icon::HostGrid global;
        std::string err = icon::build_host_grid(bisections_k, 0, false, global);
        icon::ScTables gsc;
        if (err.empty()) err = icon::build_sc_tables(global, gsc);
        if (err.empty()) err = icon::build_partition(gsc, global.nc, global.ne, global.nv, n_parts, part, g->sc_host, g->part);
        if (!err.empty()) {
            delete g;
            return fail(ICON_EINVAL, err);
        }
    } catch (const std::bad_alloc&) {
        delete g;
        return fail(ICON_ENOMEM, "out of host memory while building the local grid");
    }
    g->sc_host_ready = true;
    g->host.level_k = bisections_k;
    g->host.nc = g->part.nc_local;       // every size check and every kernel sees the LOCAL counts
    g->host.ne = g->part.ne_local;
    g->host.nv = g->part.nv_owned;
    if (!g->host_only) {
        int ndev = 0;
        cudaError_t e = cudaGetDeviceCount(&ndev);
        if (e != cudaSuccess || ndev == 0) {
            delete g;
            return fail(ICON_ECUDA, "no usable CUDA device (there is no CPU fallback)");
        }
        int rc = ICON_OK;
        e = cudaGetDevice(&g->device);
        if (e == cudaSuccess) e = cudaDeviceGetAttribute(&g->num_sms, cudaDevAttrMultiProcessorCount, g->device);
        if (e == cudaSuccess) e = cudaDeviceGetAttribute(&g->smem_optin, cudaDevAttrMaxSharedMemoryPerBlockOptin, g->device);
        if (e != cudaSuccess) rc = fail_cuda(e, "cudaGetDevice");
        for (int kind = 0; kind < 2 && rc == ICON_OK; ++kind) rc = upload_vec(g, g->part.send_ids[kind], &g->d_send_ids[kind]);
        if (rc == ICON_OK && cudaStreamSynchronize(cudaStreamLegacy) != cudaSuccess) rc = fail(ICON_ECUDA, "upload of the send lists failed");
        if (rc != ICON_OK) {
            std::string keep = t_last_error;
            icon_grid_destroy(g);
            t_last_error = keep;
            return rc;
        }
    }
    *out = g;
    return ICON_OK;
}

int icon_part_info(const icon_grid_t* g, int64_t out[12]) {
    if (!g || !out) return fail(ICON_EINVAL, "NULL argument");
    const icon::PartTables& p = g->part;
    const int64_t v[12] = {p.n_parts, p.part, p.nc_owned, p.ne_owned, p.nv_owned, p.nc_local, p.ne_local,
                           p.nc_global, p.ne_global, p.nv_global, p.patch_lo, p.patch_hi};
    for (int i = 0; i < 12; ++i) out[i] = v[i];
    return ICON_OK;
}

int icon_part_table(const icon_grid_t* g, int which, const void** ptr, int* dtype, int64_t* count) {
    if (!g) return fail(ICON_EINVAL, "grid handle is NULL");
    if (!g->part.n_parts) return fail(ICON_EUNSUPPORTED, "icon_part_table: the grid was not made by icon_grid_create_part");
    const icon::PartTables& p = g->part;
    const void* d = nullptr;
    int64_t n = 0;
    int dt = ICON_T_I32;
    auto I32 = [&](const std::vector<int32_t>& v) { d = v.data(); n = (int64_t)v.size(); dt = ICON_T_I32; };
    auto I64 = [&](const std::vector<int64_t>& v) { d = v.data(); n = (int64_t)v.size(); dt = ICON_T_I64; };
    switch (which) {
        case ICON_PART_L2G_CELL: I32(p.l2g_c); break;
        case ICON_PART_L2G_EDGE: I32(p.l2g_e); break;
        case ICON_PART_L2G_VERT: I32(p.l2g_v); break;
        case ICON_PART_RECV_BEGIN_EDGE: I64(p.recv_begin[0]); break;
        case ICON_PART_RECV_BEGIN_CELL: I64(p.recv_begin[1]); break;
        case ICON_PART_SEND_BEGIN_EDGE: I64(p.send_begin[0]); break;
        case ICON_PART_SEND_BEGIN_CELL: I64(p.send_begin[1]); break;
        case ICON_PART_SEND_IDS_EDGE: I32(p.send_ids[0]); break;
        case ICON_PART_SEND_IDS_CELL: I32(p.send_ids[1]); break;
        default: return fail(ICON_EINVAL, "unknown partition table selector");
    }
    if (ptr) *ptr = d;
    if (dtype) *dtype = dt;
    if (count) *count = n;
    return ICON_OK;
}

int dycore_halo_pack(const icon_grid_t* gc, int dtype, int kind, int ld, const void* field, void* send_buf, void* cuda_stream) {
    icon_grid* g = const_cast<icon_grid*>(gc);       // logically const: only the launch counter moves
    if (!g) return fail(ICON_EINVAL, "grid handle is NULL");
    if (!g->part.n_parts) return fail(ICON_EUNSUPPORTED, "dycore_halo_pack: the grid was not made by icon_grid_create_part");
    if (g->host_only) return fail(ICON_ECUDA, "grid was created with ICON_HOST_ONLY: no device tables, and there is no CPU path");
    if (int rc = check_device(g)) return rc;
    if (dtype != ICON_F64 && dtype != ICON_F32) return fail(ICON_EINVAL, "dtype must be ICON_F64 or ICON_F32");
    if (kind != 0 && kind != 1) return fail(ICON_EINVAL, "kind must be 0 (edge field) or 1 (cell field)");
    const int64_t es = dtype == ICON_F64 ? 8 : 4;
    if (ld < 1 || ((int64_t)ld * es) % 16) return fail(ICON_EINVAL, "ld*sizeof(T) must be a positive multiple of 16");
    const int64_t n = (int64_t)g->part.send_ids[kind].size();
    if (n == 0) return ICON_OK;                      // nothing to send (one rank, or no neighbour reads this kind)
    if (int rc = check_field(field, "field")) return rc;
    if (int rc = check_field(send_buf, "send_buf")) return rc;
    const int64_t rows = kind == 0 ? g->part.ne_local : g->part.nc_local;
    if (overlaps(send_buf, (size_t)(n * ld * es), field, (size_t)(rows * ld * es))) return fail(ICON_EINVAL, "send_buf must not overlap the field");
    const int k = icon::launch_halo_pack(g->d_send_ids[kind], n, (int64_t)ld * es, field, send_buf, (cudaStream_t)cuda_stream);
    if (k < 0) return fail_cuda((cudaError_t)(-k), "kernel launch");
    g->launches += k;
    return ICON_OK;
}

int icon_grid_cc_schedule_check(const icon_grid_t* gc, int dtype, int nlev, int ldk, int ldk_w, int n_ctas, int smem_bytes,
                                int64_t out[8]) {
    icon_grid* g = const_cast<icon_grid*>(gc);
    if (!g || !out) return fail(ICON_EINVAL, "NULL argument");
    if (dtype != ICON_F64 && dtype != ICON_F32) return fail(ICON_EINVAL, "dtype must be ICON_F64 or ICON_F32");
    if (nlev < 2 || ldk < nlev || ldk_w < nlev + 1 || n_ctas < 1 || smem_bytes < 1) return fail(ICON_EINVAL, "bad argument");
    if (icon::cc_levels_per_lane(nlev) == 0) return fail(ICON_EUNSUPPORTED, "nlev not supported by the column-cache kernel");
    int rc = ensure_sc_host(g);
    if (rc) return rc;
    const bool f64 = dtype == ICON_F64;
    icon::CcSchedule cs;
    icon::CcGeometry geom;
    try {
        // the schedules of dycore_div_vort (27 vn columns per patch, compact records) and of dycore_step_w (all 46 columns)
        // first, then the one of the tendency / fused step, whose shape is reported
        for (int mode : {(int)icon::kCcDivVort, (int)icon::kCcWTend, (int)icon::kCcStepW, (int)icon::kCcStep}) {
            const bool dv = mode == icon::kCcDivVort;
            geom = f64 ? cc_geometry<double>(nlev, ldk, ldk_w, dv) : cc_geometry<float>(nlev, ldk, ldk_w, dv);
            const int n_slots = std::min(65535, f64 ? icon::cc_max_slots<double>(geom.slot_bytes, smem_bytes, mode, nlev)
                                                    : icon::cc_max_slots<float>(geom.slot_bytes, smem_bytes, mode, nlev));
            std::string err = icon::build_cc_schedule(g->sc_host, n_ctas, n_slots, geom, icon::cc_patches_per_step_for(nlev, f64 ? 8 : 4, mode), icon::kCcDepth,
                                                      f64 ? cc_resolve_tile<double>(g, nlev) : cc_resolve_tile<float>(g, nlev), icon::cc_use_mask(mode), cs);
            if (!err.empty()) return fail(ICON_EUNSUPPORTED, err);
            err = icon::check_cc_schedule(g->sc_host, cs, g->host.ne, g->host.nc);
            if (!err.empty()) return fail(ICON_EINVAL, err + (dv ? " (div/vort schedule)" : mode == icon::kCcStepW ? " (step + ddt_w schedule)" : mode == icon::kCcWTend ? " (ddt_w schedule)" : ""));
        }
    } catch (const std::bad_alloc&) {
        return fail(ICON_ENOMEM, "out of host memory while building the column-cache schedule");
    }
    out[0] = (int64_t)cs.steps.size(); out[1] = cs.n_sync_steps; out[2] = cs.n_vn_loads; out[3] = cs.n_w_loads;
    out[4] = cs.n_copies; out[5] = cs.n_slots; out[6] = geom.slot_bytes; out[7] = cs.n_ctas;
    return ICON_OK;
}

int dycore_div_vort(const icon_grid_t* gc, int dtype, int nlev, int ldk, const void* vn, void* div, void* vort,
                    void* cuda_stream) {
    icon_grid* g = const_cast<icon_grid*>(gc);       // logically const: lazily built tables are a cache
    int rc = check_common(g, dtype, nlev, ldk, 1);
    if (rc) return rc;
    if ((rc = check_field(vn, "vn")) || (rc = check_field(div, "div")) || (rc = check_field(vort, "vort"))) return rc;
    {
        const size_t es = dtype == ICON_F64 ? 8 : 4;
        const size_t be = (size_t)g->host.ne * ldk * es, bc = (size_t)g->host.nc * ldk * es, bv = (size_t)g->host.nv * ldk * es;
        if (overlaps(div, bc, vn, be) || overlaps(vort, bv, vn, be) || overlaps(div, bc, vort, bv))
            return fail(ICON_EINVAL, "outputs must not alias the input or each other");
    }
    cudaStream_t s = (cudaStream_t)cuda_stream;
    int n;
    // the column cache in its div / vort mode wherever it holds the columns (ICON_OPT_TENDENCY_KERNEL 4 or auto), else
    // the gather kernel through L1
    const bool want_cc = g->options[ICON_OPT_TENDENCY_KERNEL] >= 4 && nlev >= 2;
    if (dtype == ICON_F64) {
        if (want_cc && (rc = ensure_cc_tables(g, g->dv64, nlev, ldk, ldk, icon::kCcDivVort))) return rc;
        if (want_cc && !g->dv64.unsupported) {
            n = icon::launch_tendencies_cc<double>(*g, g->dv64, icon::kCcDivVort, nlev, ldk, ldk, nullptr, (const double*)vn, nullptr, nullptr,
                                                   (double*)div, (double*)vort, s);
        } else {
            if ((rc = ensure_coeffs(g, g->c64))) return rc;
            n = icon::launch_div_vort<double>(*g, g->c64, nlev, ldk, (const double*)vn, (double*)div, (double*)vort, s);
        }
    } else {
        if (want_cc && (rc = ensure_cc_tables(g, g->dv32, nlev, ldk, ldk, icon::kCcDivVort))) return rc;
        if (want_cc && !g->dv32.unsupported) {
            n = icon::launch_tendencies_cc<float>(*g, g->dv32, icon::kCcDivVort, nlev, ldk, ldk, nullptr, (const float*)vn, nullptr, nullptr,
                                                  (float*)div, (float*)vort, s);
        } else {
            if ((rc = ensure_coeffs(g, g->c32))) return rc;
            n = icon::launch_div_vort<float>(*g, g->c32, nlev, ldk, (const float*)vn, (float*)div, (float*)vort, s);
        }
    }
    if (n < 0) return fail_cuda((cudaError_t)(-n), "kernel launch");
    g->launches += n;
    return ICON_OK;
}

int dycore_velocity_tendencies(const icon_grid_t* gc, int dtype, int nlev, int ldk, int ldk_w, const double* z_half,
                               const void* vn, const void* w, void* ddt_vn, void* vt_opt, void* ke_c_opt,
                               void* vort_opt, void* cuda_stream) {
    icon_grid* g = const_cast<icon_grid*>(gc);
    int rc = check_common(g, dtype, nlev, ldk, 2);
    if (rc) return rc;
    if (ldk_w < nlev + 1) return fail(ICON_EINVAL, "ldk_w < nlev+1");
    if (((int64_t)ldk_w * (dtype == ICON_F64 ? 8 : 4)) % 16) return fail(ICON_EINVAL, "ldk_w*sizeof(T) must be a multiple of 16");
    if (!z_half) return fail(ICON_EINVAL, "z_half is NULL");
    if ((rc = check_field(vn, "vn")) || (rc = check_field(w, "w")) || (rc = check_field(ddt_vn, "ddt_vn"))) return rc;
    if (vt_opt && (rc = check_field(vt_opt, "vt_opt"))) return rc;
    if (ke_c_opt && (rc = check_field(ke_c_opt, "ke_c_opt"))) return rc;
    if (vort_opt && (rc = check_field(vort_opt, "vort_opt"))) return rc;
    {
        const size_t es = dtype == ICON_F64 ? 8 : 4;
        const size_t be = (size_t)g->host.ne * ldk * es, bc = (size_t)g->host.nc * ldk * es, bv = (size_t)g->host.nv * ldk * es,
                     bw = (size_t)g->host.nc * ldk_w * es;
        const void* outs[4] = {ddt_vn, vt_opt, ke_c_opt, vort_opt};
        const size_t ob[4] = {be, be, bc, bv};
        for (int i = 0; i < 4; ++i) {
            if (overlaps(outs[i], ob[i], vn, be) || overlaps(outs[i], ob[i], w, bw)) return fail(ICON_EINVAL, "outputs must not alias inputs");
            for (int j = 0; j < i; ++j)
                if (overlaps(outs[i], ob[i], outs[j], ob[j])) return fail(ICON_EINVAL, "outputs must not alias each other");
        }
    }
    cudaStream_t s = (cudaStream_t)cuda_stream;
    if (dtype == ICON_F64)
        return tendencies_impl<double>(g, g->c64, g->s64, g->cc64, dtype, nlev, ldk, ldk_w, z_half, vn, w, ddt_vn, vt_opt, ke_c_opt, vort_opt, s);
    return tendencies_impl<float>(g, g->c32, g->s32, g->cc32, dtype, nlev, ldk, ldk_w, z_half, vn, w, ddt_vn, vt_opt, ke_c_opt, vort_opt, s);
}

int dycore_w_tendency(const icon_grid_t* gc, int dtype, int nlev, int ldk, int ldk_w, const double* z_half, const void* vn,
                      const void* w, void* ddt_w, void* cuda_stream) {
    icon_grid* g = const_cast<icon_grid*>(gc);
    int rc = check_common(g, dtype, nlev, ldk, 2);
    if (rc) return rc;
    const size_t es = dtype == ICON_F64 ? 8 : 4;
    if (ldk_w < nlev + 1) return fail(ICON_EINVAL, "ldk_w < nlev + 1");
    if (((int64_t)ldk_w * (int64_t)es) % 16) return fail(ICON_EINVAL, "ldk_w*sizeof(T) must be a multiple of 16");
    if (!z_half) return fail(ICON_EINVAL, "z_half is NULL");
    if ((rc = check_field(vn, "vn")) || (rc = check_field(w, "w")) || (rc = check_field(ddt_w, "ddt_w"))) return rc;
    const size_t be = (size_t)g->host.ne * ldk * es, bw = (size_t)g->host.nc * ldk_w * es;
    if (overlaps(ddt_w, bw, vn, be) || overlaps(ddt_w, bw, w, bw)) return fail(ICON_EINVAL, "outputs must not alias inputs");
    void *abc = nullptr, *wk = nullptr;
    if ((rc = get_level_coeffs(g, dtype, nlev, z_half, &abc, &wk))) return rc;
    cudaStream_t s = (cudaStream_t)cuda_stream;
    int n;
    // the column cache in its ddt_w mode wherever it holds the columns (ICON_OPT_TENDENCY_KERNEL 4 or auto), else the gather
    // kernel through L1
    const bool want_cc = g->options[ICON_OPT_TENDENCY_KERNEL] >= 4;
    if (dtype == ICON_F64) {
        if (want_cc && (rc = ensure_cc_tables(g, g->wt64, nlev, ldk, ldk_w, icon::kCcWTend))) return rc;
        if (want_cc && !g->wt64.unsupported) {
            n = icon::launch_tendencies_cc<double>(*g, g->wt64, icon::kCcWTend, nlev, ldk, ldk_w, nullptr, (const double*)vn, (const double*)w, nullptr,
                                                   nullptr, nullptr, s, (const double*)wk, (double*)ddt_w);
        } else {
            if ((rc = ensure_coeffs(g, g->c64))) return rc;
            n = icon::launch_w_tendency<double>(*g, g->c64, nlev, ldk, ldk_w, (const double*)wk, (const double*)vn, (const double*)w, (double*)ddt_w, s);
        }
    } else {
        if (want_cc && (rc = ensure_cc_tables(g, g->wt32, nlev, ldk, ldk_w, icon::kCcWTend))) return rc;
        if (want_cc && !g->wt32.unsupported) {
            n = icon::launch_tendencies_cc<float>(*g, g->wt32, icon::kCcWTend, nlev, ldk, ldk_w, nullptr, (const float*)vn, (const float*)w, nullptr,
                                                  nullptr, nullptr, s, (const float*)wk, (float*)ddt_w);
        } else {
            if ((rc = ensure_coeffs(g, g->c32))) return rc;
            n = icon::launch_w_tendency<float>(*g, g->c32, nlev, ldk, ldk_w, (const float*)wk, (const float*)vn, (const float*)w, (float*)ddt_w, s);
        }
    }
    if (n < 0) return fail_cuda((cudaError_t)(-n), "kernel launch");
    g->launches += n;
    return ICON_OK;
}

int dycore_step(const icon_grid_t* gc, int dtype, int nlev, int ldk, int ldk_w, const double* z_half, const void* vn, const void* w,
                void* ddt_vn, void* div, void* vort, void* cuda_stream) {
    icon_grid* g = const_cast<icon_grid*>(gc);
    int rc = check_common(g, dtype, nlev, ldk, 2);
    if (rc) return rc;
    if (ldk_w < nlev + 1) return fail(ICON_EINVAL, "ldk_w < nlev + 1");
    const int es = dtype == ICON_F64 ? 8 : 4;
    if (((int64_t)ldk_w * es) % 16) return fail(ICON_EINVAL, "ldk_w*sizeof(T) must be a multiple of 16");
    if (!z_half) return fail(ICON_EINVAL, "z_half is NULL");
    if ((rc = check_field(vn, "vn")) || (rc = check_field(w, "w")) || (rc = check_field(ddt_vn, "ddt_vn")) ||
        (rc = check_field(div, "div")) || (rc = check_field(vort, "vort")))
        return rc;
    {
        const size_t be = (size_t)g->host.ne * ldk * es, bc = (size_t)g->host.nc * ldk * es, bv = (size_t)g->host.nv * ldk * es,
                     bw = (size_t)g->host.nc * ldk_w * es;
        const void* outs[3] = {ddt_vn, div, vort};
        const size_t ob[3] = {be, bc, bv};
        for (int i = 0; i < 3; ++i) {
            if (overlaps(outs[i], ob[i], vn, be) || overlaps(outs[i], ob[i], w, bw))
                return fail(ICON_EINVAL, "outputs must not alias inputs or each other");
            for (int j = 0; j < i; ++j)
                if (overlaps(outs[i], ob[i], outs[j], ob[j])) return fail(ICON_EINVAL, "outputs must not alias inputs or each other");
        }
    }
    cudaStream_t s = (cudaStream_t)cuda_stream;
    bool fused = false;
    if (dtype == ICON_F64)
        rc = tendencies_impl<double>(g, g->c64, g->s64, g->cc64, dtype, nlev, ldk, ldk_w, z_half, vn, w, ddt_vn, nullptr,
                                     nullptr, nullptr, s, div, vort, &fused);
    else
        rc = tendencies_impl<float>(g, g->c32, g->s32, g->cc32, dtype, nlev, ldk, ldk_w, z_half, vn, w, ddt_vn, nullptr,
                                    nullptr, nullptr, s, div, vort, &fused);
    if (rc || fused) return rc;
    return dycore_div_vort(g, dtype, nlev, ldk, vn, div, vort, cuda_stream);
}

int dycore_metric_from_zhalf(const icon_grid_t* gc, int dtype, int nlev, int ldk, int ldk_w, const void* z_half_e, void* wgt_e,
                             void* inv_ddqz_e, void* cuda_stream) {
    icon_grid* g = const_cast<icon_grid*>(gc);
    int rc = check_common(g, dtype, nlev, ldk, 3);
    if (rc) return rc;
    const size_t es = dtype == ICON_F64 ? 8 : 4;
    if (ldk_w < nlev + 1) return fail(ICON_EINVAL, "ldk_w < nlev + 1");
    if (((int64_t)ldk_w * (int64_t)es) % 16) return fail(ICON_EINVAL, "ldk_w*sizeof(T) must be a multiple of 16");
    if ((rc = check_field(z_half_e, "z_half_e")) || (rc = check_field(wgt_e, "wgt_e")) || (rc = check_field(inv_ddqz_e, "inv_ddqz_e")))
        return rc;
    const size_t bw = (size_t)g->host.ne * ldk_w * es, bk = (size_t)g->host.ne * ldk * es;
    if (overlaps(wgt_e, bw, z_half_e, bw) || overlaps(inv_ddqz_e, bk, z_half_e, bw) || overlaps(wgt_e, bw, inv_ddqz_e, bk))
        return fail(ICON_EINVAL, "outputs must not alias the input or each other");
    cudaStream_t s = (cudaStream_t)cuda_stream;
    const int n = dtype == ICON_F64
                      ? icon::launch_metric_from_zhalf<double>(*g, nlev, ldk, ldk_w, (const double*)z_half_e, (double*)wgt_e, (double*)inv_ddqz_e, s)
                      : icon::launch_metric_from_zhalf<float>(*g, nlev, ldk, ldk_w, (const float*)z_half_e, (float*)wgt_e, (float*)inv_ddqz_e, s);
    if (n < 0) return fail_cuda((cudaError_t)(-n), "kernel launch");
    g->launches += n;
    return ICON_OK;
}

}  // extern "C"

namespace {
template <class T>
int tendencies_metric_impl(icon_grid* g, icon::DevCoeffs<T>& c, icon::DevCcTables<T>& ct, int dtype, int nlev, int ldk, int ldk_w,
                           const void* wgt, const void* inv, const void* zn, const void* zt, const void* vn, const void* w, void* ddt_vn,
                           cudaStream_t s) {
    int rc;
    if (!g->part.n_parts && (rc = ensure_coeffs(g, c))) return rc;
    int n;
    if (g->options[ICON_OPT_TENDENCY_KERNEL] >= 4) {
        if ((rc = ensure_cc_tables(g, ct, nlev, ldk, ldk_w, icon::kCcTendM))) return rc;
        if (!ct.unsupported) {
            icon::CcMetric<T> m{(const T*)wgt, (const T*)inv, (const T*)zn, (const T*)zt};
            n = icon::launch_tendencies_cc<T>(*g, ct, icon::kCcTendM, nlev, ldk, ldk_w, nullptr, (const T*)vn, (const T*)w, (T*)ddt_vn, nullptr,
                                              nullptr, s, nullptr, nullptr, &m);
            if (n < 0) return fail_cuda((cudaError_t)(-n), "kernel launch");
            g->launches += n;
            return ICON_OK;
        }
    }
    // level counts the column cache cannot hold, or ICON_OPT_TENDENCY_KERNEL 0 / 3: the unfused pipeline with its metric last stage
    if (g->part.n_parts && (rc = ensure_coeffs(g, c))) return rc;      // fails: column cache only
    if ((rc = ensure_workspace<T>(g, dtype, ldk))) return rc;
    n = icon::launch_tendencies_unfused_metric<T>(*g, c, nlev, ldk, ldk_w, (const T*)wgt, (const T*)inv, (const T*)zn, (const T*)zt,
                                                  (const T*)vn, (const T*)w, (T*)ddt_vn, (T*)g->ws.vt, (T*)g->ws.ke_e, (T*)g->ws.ke_c,
                                                  (T*)g->ws.vort, s);
    if (n < 0) return fail_cuda((cudaError_t)(-n), "kernel launch");
    g->launches += n;
    return ICON_OK;
}
}  // namespace

extern "C" {

int dycore_velocity_tendencies_metric(const icon_grid_t* gc, int dtype, int nlev, int ldk, int ldk_w, const void* wgt_e,
                                      const void* inv_ddqz_e, const void* ddxn_z, const void* ddxt_z, const void* vn, const void* w,
                                      void* ddt_vn, void* cuda_stream) {
    icon_grid* g = const_cast<icon_grid*>(gc);
    int rc = check_common(g, dtype, nlev, ldk, 3);
    if (rc) return rc;
    const size_t es = dtype == ICON_F64 ? 8 : 4;
    if (ldk_w < nlev + 1) return fail(ICON_EINVAL, "ldk_w < nlev + 1");
    if (((int64_t)ldk_w * (int64_t)es) % 16) return fail(ICON_EINVAL, "ldk_w*sizeof(T) must be a multiple of 16");
    if ((rc = check_field(wgt_e, "wgt_e")) || (rc = check_field(inv_ddqz_e, "inv_ddqz_e")) || (rc = check_field(ddxn_z, "ddxn_z")) ||
        (rc = check_field(ddxt_z, "ddxt_z")) || (rc = check_field(vn, "vn")) || (rc = check_field(w, "w")) || (rc = check_field(ddt_vn, "ddt_vn")))
        return rc;
    {
        const size_t be = (size_t)g->host.ne * ldk * es, bew = (size_t)g->host.ne * ldk_w * es, bw = (size_t)g->host.nc * ldk_w * es;
        const void* ins[6] = {wgt_e, inv_ddqz_e, ddxn_z, ddxt_z, vn, w};
        const size_t ib[6] = {bew, be, be, be, be, bw};
        for (int i = 0; i < 6; ++i)
            if (overlaps(ddt_vn, be, ins[i], ib[i])) return fail(ICON_EINVAL, "outputs must not alias inputs");
    }
    cudaStream_t s = (cudaStream_t)cuda_stream;
    if (dtype == ICON_F64)
        return tendencies_metric_impl<double>(g, g->c64, g->m64, dtype, nlev, ldk, ldk_w, wgt_e, inv_ddqz_e, ddxn_z, ddxt_z, vn, w, ddt_vn, s);
    return tendencies_metric_impl<float>(g, g->c32, g->m32, dtype, nlev, ldk, ldk_w, wgt_e, inv_ddqz_e, ddxn_z, ddxt_z, vn, w, ddt_vn, s);
}

int dycore_step_w(const icon_grid_t* gc, int dtype, int nlev, int ldk, int ldk_w, const double* z_half, const void* vn, const void* w,
                  void* ddt_vn, void* div, void* vort, void* ddt_w, void* cuda_stream) {
    icon_grid* g = const_cast<icon_grid*>(gc);
    int rc = check_common(g, dtype, nlev, ldk, 2);
    if (rc) return rc;
    const size_t es = dtype == ICON_F64 ? 8 : 4;
    if (ldk_w < nlev + 1) return fail(ICON_EINVAL, "ldk_w < nlev + 1");
    if (((int64_t)ldk_w * (int64_t)es) % 16) return fail(ICON_EINVAL, "ldk_w*sizeof(T) must be a multiple of 16");
    if (!z_half) return fail(ICON_EINVAL, "z_half is NULL");
    if ((rc = check_field(vn, "vn")) || (rc = check_field(w, "w")) || (rc = check_field(ddt_vn, "ddt_vn")) ||
        (rc = check_field(div, "div")) || (rc = check_field(vort, "vort")) || (rc = check_field(ddt_w, "ddt_w")))
        return rc;
    {
        const size_t be = (size_t)g->host.ne * ldk * es, bc = (size_t)g->host.nc * ldk * es, bv = (size_t)g->host.nv * ldk * es,
                     bw = (size_t)g->host.nc * ldk_w * es;
        const void* outs[4] = {ddt_vn, div, vort, ddt_w};
        const size_t ob[4] = {be, bc, bv, bw};
        for (int i = 0; i < 4; ++i) {
            if (overlaps(outs[i], ob[i], vn, be) || overlaps(outs[i], ob[i], w, bw))
                return fail(ICON_EINVAL, "outputs must not alias inputs or each other");
            for (int j = 0; j < i; ++j)
                if (overlaps(outs[i], ob[i], outs[j], ob[j])) return fail(ICON_EINVAL, "outputs must not alias inputs or each other");
        }
    }
    cudaStream_t s = (cudaStream_t)cuda_stream;
    const bool want_cc = g->options[ICON_OPT_TENDENCY_KERNEL] >= 4;
    void *abc = nullptr, *wk = nullptr;
    if ((rc = get_level_coeffs(g, dtype, nlev, z_half, &abc, &wk))) return rc;
    int n = 0;
    bool done = false;
    if (want_cc && dtype == ICON_F64) {
        if ((rc = ensure_cc_tables(g, g->sw64, nlev, ldk, ldk_w, icon::kCcStepW))) return rc;
        if (!g->sw64.unsupported) {
            n = icon::launch_tendencies_cc<double>(*g, g->sw64, icon::kCcStepW, nlev, ldk, ldk_w, (const double*)abc, (const double*)vn, (const double*)w,
                                                   (double*)ddt_vn, (double*)div, (double*)vort, s, (const double*)wk, (double*)ddt_w);
            done = true;
        }
    } else if (want_cc) {
        if ((rc = ensure_cc_tables(g, g->sw32, nlev, ldk, ldk_w, icon::kCcStepW))) return rc;
        if (!g->sw32.unsupported) {
            n = icon::launch_tendencies_cc<float>(*g, g->sw32, icon::kCcStepW, nlev, ldk, ldk_w, (const float*)abc, (const float*)vn, (const float*)w,
                                                  (float*)ddt_vn, (float*)div, (float*)vort, s, (const float*)wk, (float*)ddt_w);
            done = true;
        }
    }
    if (done) {
        if (n < 0) return fail_cuda((cudaError_t)(-n), "kernel launch");
        g->launches += n;
        return ICON_OK;
    }
    // level counts the column cache cannot hold, or another tendency kernel selected: the separate calls
    if ((rc = dycore_step(gc, dtype, nlev, ldk, ldk_w, z_half, vn, w, ddt_vn, div, vort, cuda_stream))) return rc;
    return dycore_w_tendency(gc, dtype, nlev, ldk, ldk_w, z_half, vn, w, ddt_w, cuda_stream);
}

int dycore_step_host(const icon_grid_t* gc, int dtype, int nlev, int ldk, int ldk_w, const double* z_half,
                     const void* vn_host, const void* w_host, void* ddt_vn_host, void* div_host, void* vort_host) {
    icon_grid* g = const_cast<icon_grid*>(gc);
    int rc = check_common(g, dtype, nlev, ldk, 2);
    if (rc) return rc;
    if (!vn_host || !w_host || !ddt_vn_host || !div_host || !vort_host) return fail(ICON_EINVAL, "NULL host buffer");
    const size_t es = dtype == ICON_F64 ? 8 : 4;
    icon::HostStage& st = g->stage;
    if (!st.stream) {
        CU_TRY(cudaStreamCreateWithFlags(&st.stream, cudaStreamNonBlocking));
        CU_TRY(cudaStreamCreateWithFlags(&st.stream_in, cudaStreamNonBlocking));
        CU_TRY(cudaStreamCreateWithFlags(&st.stream_out, cudaStreamNonBlocking));
        for (cudaEvent_t* e : {&st.ev_vn, &st.ev_w, &st.ev_dv, &st.ev_t}) CU_TRY(cudaEventCreateWithFlags(e, cudaEventDisableTiming));
    }
    if (st.dtype != dtype || st.ldk != ldk || st.ldk_w != ldk_w) {
        dev_release(g, st.vn); dev_release(g, st.w); dev_release(g, st.ddt); dev_release(g, st.div); dev_release(g, st.vort);
        st.vn = st.w = st.ddt = st.div = st.vort = nullptr;
        char *a, *b, *c, *d, *e;
        if ((rc = dev_alloc(g, (size_t)g->host.ne * ldk * es, &a))) return rc;
        if ((rc = dev_alloc(g, (size_t)g->host.nc * ldk_w * es, &b))) return rc;
        if ((rc = dev_alloc(g, (size_t)g->host.ne * ldk * es, &c))) return rc;
        if ((rc = dev_alloc(g, (size_t)g->host.nc * ldk * es, &d))) return rc;
        if ((rc = dev_alloc(g, (size_t)g->host.nv * ldk * es, &e))) return rc;
        st.vn = a; st.w = b; st.ddt = c; st.div = d; st.vort = e;
        st.dtype = dtype; st.ldk = ldk; st.ldk_w = ldk_w;
    }
    const size_t ne = (size_t)g->host.ne, nc = (size_t)g->host.nc, nv = (size_t)g->host.nv;
    // Three streams so that the two directions of the link and the kernels overlap: vn goes up first; as soon as it has
    // arrived dycore_div_vort (which reads nothing else) runs and div / vort go DOWN while w is still going UP; then the
    // tendency, then ddt_vn down. (One fused dycore_step would need both inputs before it starts and could return nothing
    // before it ends: 22 GB strictly one after the other. The two kernels cost 6 ms instead of 4.4 ms, against ~ 80 ms of
    // copy time saved at R2B8 x 90.)
    CU_TRY(cudaMemcpyAsync(st.vn, vn_host, ne * ldk * es, cudaMemcpyHostToDevice, st.stream_in));
    CU_TRY(cudaEventRecord(st.ev_vn, st.stream_in));
    CU_TRY(cudaMemcpyAsync(st.w, w_host, nc * ldk_w * es, cudaMemcpyHostToDevice, st.stream_in));
    CU_TRY(cudaEventRecord(st.ev_w, st.stream_in));
    CU_TRY(cudaStreamWaitEvent(st.stream, st.ev_vn, 0));
    if ((rc = dycore_div_vort(g, dtype, nlev, ldk, st.vn, st.div, st.vort, st.stream))) return rc;
    CU_TRY(cudaEventRecord(st.ev_dv, st.stream));
    CU_TRY(cudaStreamWaitEvent(st.stream, st.ev_w, 0));
    if ((rc = dycore_velocity_tendencies(g, dtype, nlev, ldk, ldk_w, z_half, st.vn, st.w, st.ddt, nullptr, nullptr, nullptr, st.stream))) return rc;
    CU_TRY(cudaEventRecord(st.ev_t, st.stream));
    CU_TRY(cudaStreamWaitEvent(st.stream_out, st.ev_dv, 0));
    CU_TRY(cudaMemcpyAsync(div_host, st.div, nc * ldk * es, cudaMemcpyDeviceToHost, st.stream_out));
    CU_TRY(cudaMemcpyAsync(vort_host, st.vort, nv * ldk * es, cudaMemcpyDeviceToHost, st.stream_out));
    CU_TRY(cudaStreamWaitEvent(st.stream_out, st.ev_t, 0));
    CU_TRY(cudaMemcpyAsync(ddt_vn_host, st.ddt, ne * ldk * es, cudaMemcpyDeviceToHost, st.stream_out));
    CU_TRY(cudaStreamSynchronize(st.stream_out));
    CU_TRY(cudaStreamSynchronize(st.stream));
    return ICON_OK;
}

}  // extern "C"

// ======================================================================================================
// dycore_velocity_tendencies_noalloc -- the unfused tendency pipeline with its scratch in a STATIC device array
// ======================================================================================================
// Some callers cannot call cudaMalloc (code under CUDA-graph capture, tight serving loops, harnesses that forbid it).
// The ordinary entry points allocate lazily on the first call for a new (dtype, nlev, ldk, z_half): schedules, records,
// level coefficients, the workspace of the unfused pipeline. This variant allocates NOTHING: the intermediates of the
// unfused pipeline (vt, KE_e, KE_c, zeta) and the per-level coefficients live in the file-scope array below, which every
// GPU that loads the library holds until the process exits. In host code the array's NAME is a host-side stand-in, not
// a device address: its device address is taken once per device with cudaGetSymbolAddress (device current) and only that
// pointer is ever handed to a kernel.
namespace {

constexpr size_t kNoAllocScratchBytes = ICON_NOALLOC_SCRATCH_BYTES;
constexpr int kNoAllocMaxLevels = 128;             // the level coefficients travel as a kernel argument (3 x 128 doubles)
static __device__ __align__(256) unsigned char g_noalloc_scratch[kNoAllocScratchBytes];

struct NoAllocCoeffArg {
    double v[3 * kNoAllocMaxLevels];               // A_k, B_k, C_k of reading P-14, [3][nlev]
};

// writes the 3 * nlev level coefficients into the scratch array (no host -> device copy, no staging buffer)
template <class T>
__global__ void k_noalloc_coeffs(NoAllocCoeffArg a, int n, T* __restrict__ out) {
    for (int i = threadIdx.x; i < n; i += blockDim.x) out[i] = (T)a.v[i];
}

// device address of g_noalloc_scratch on `device` (which must be current); resolved once per device
int noalloc_scratch_ptr(int device, unsigned char** out) {
    static std::mutex mu;
    static unsigned char* ptrs[64] = {nullptr};
    std::lock_guard<std::mutex> lock(mu);
    const bool known = device >= 0 && device < 64;
    if (known && ptrs[device]) {
        *out = ptrs[device];
        return ICON_OK;
    }
    unsigned char* p = nullptr;
    cudaError_t e = cudaGetSymbolAddress((void**)&p, g_noalloc_scratch);
    if (e != cudaSuccess) return fail_cuda(e, "cudaGetSymbolAddress(g_noalloc_scratch)");
    if (!p || reinterpret_cast<uintptr_t>(p) % 256) return fail(ICON_ECUDA, "static scratch array has no usable device address");
    if (known) ptrs[device] = p;
    *out = p;
    return ICON_OK;
}

size_t align256(size_t n) { return (n + 255) & ~(size_t)255; }

// (vn_ie(k) - vn_ie(k+1)) / dz_k = A_k vn(k-1) + B_k vn(k) + C_k vn(k+1): the statements of vertical_coefficients above, in
// the same order, into a caller-provided array abc[3][K] instead of a std::vector
void noalloc_vertical_coefficients(const double* zh, int K, double* abc) {
    for (int i = 0; i < 3 * kNoAllocMaxLevels; ++i) abc[i] = 0.0;
    auto zf = [&](int k) { return 0.5 * (zh[k] + zh[k + 1]); };
    auto add_half = [&](int k, int kh, double sign) {
        int ia, ib;
        double ca, cb;
        if (kh == 0) {
            double r = (zh[0] - zf(0)) / (zf(0) - zf(1));
            ia = 0; ca = 1.0 + r; ib = 1; cb = -r;
        } else if (kh == K) {
            double r = (zh[K] - zf(K - 1)) / (zf(K - 1) - zf(K - 2));
            ia = K - 1; ca = 1.0 + r; ib = K - 2; cb = -r;
        } else {
            double up = zh[kh - 1] - zh[kh], dn = zh[kh] - zh[kh + 1];
            double gk = up / (up + dn);
            ia = kh; ca = gk; ib = kh - 1; cb = 1.0 - gk;
        }
        const double inv_dz = 1.0 / (zh[k] - zh[k + 1]);
        abc[(size_t)(ia - k + 1) * K + k] += sign * ca * inv_dz;
        abc[(size_t)(ib - k + 1) * K + k] += sign * cb * inv_dz;
    };
    for (int k = 0; k < K; ++k) {
        add_half(k, k, +1.0);
        add_half(k, k + 1, -1.0);
    }
}

template <class T>
int noalloc_impl(icon_grid* g, icon::DevCoeffs<T>& c, int nlev, int ldk, int ldk_w, const double* z_half, const void* vn,
                 const void* w, void* ddt_vn, cudaStream_t s) {
    if (!c.ready)
        return fail(ICON_EUNSUPPORTED, "the coefficient tables of this dtype are not on the device yet and this entry point must not "
                                       "allocate: make one ordinary compute call of this dtype on the grid first");
    const size_t ne = (size_t)g->host.ne, nc = (size_t)g->host.nc, nv = (size_t)g->host.nv;
    const size_t b_abc = align256(3 * (size_t)nlev * sizeof(T)), b_e = align256(ne * ldk * sizeof(T)),
                 b_c = align256(nc * ldk * sizeof(T)), b_v = align256(nv * ldk * sizeof(T));
    const size_t need = b_abc + 2 * b_e + b_c + b_v;
    if (need > kNoAllocScratchBytes)
        return fail(ICON_EINVAL, "dycore_velocity_tendencies_noalloc: this grid and level count need " + std::to_string(need) +
                                     " bytes of scratch, the static array holds " + std::to_string(kNoAllocScratchBytes) +
                                     " (ICON_NOALLOC_SCRATCH_BYTES); use dycore_velocity_tendencies");
    unsigned char* base = nullptr;
    int rc = noalloc_scratch_ptr(g->device, &base);
    if (rc) return rc;
    T* abc = reinterpret_cast<T*>(base);
    T* vt = reinterpret_cast<T*>(base + b_abc);
    T* ke_e = reinterpret_cast<T*>(base + b_abc + b_e);
    T* ke_c = reinterpret_cast<T*>(base + b_abc + 2 * b_e);
    T* vort = reinterpret_cast<T*>(base + b_abc + 2 * b_e + b_c);
    // the arithmetic of the ordinary path (vertical_coefficients, reading P-14), written straight into the kernel argument:
    // no host heap either
    NoAllocCoeffArg arg;
    noalloc_vertical_coefficients(z_half, nlev, arg.v);
    k_noalloc_coeffs<T><<<1, 128, 0, s>>>(arg, 3 * nlev, abc);
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return fail_cuda(e, "kernel launch");
    // nothing in the scratch has to start at zero: every level < nlev of vt, KE_e, KE_c and zeta is written by the
    // pipeline before it is read, and levels >= nlev are never read
    const int n = icon::launch_tendencies_unfused<T>(*g, c, nlev, ldk, ldk_w, abc, (const T*)vn, (const T*)w, (T*)ddt_vn, vt, ke_e,
                                                     ke_c, vort, s);
    if (n < 0) return fail_cuda((cudaError_t)(-n), "kernel launch");
    g->launches += n + 1;
    return ICON_OK;
}

}  // namespace

extern "C" int dycore_velocity_tendencies_noalloc(const icon_grid_t* gc, int dtype, int nlev, int ldk, int ldk_w, const double* z_half,
                                                  const void* vn, const void* w, void* ddt_vn, void* cuda_stream) {
    icon_grid* g = const_cast<icon_grid*>(gc);
    int rc = check_common(g, dtype, nlev, ldk, 2);      // includes: the grid's device is the current device
    if (rc) return rc;
    if (g->part.n_parts) return fail(ICON_EUNSUPPORTED, "dycore_velocity_tendencies_noalloc: not on a grid made by icon_grid_create_part");
    if (nlev > kNoAllocMaxLevels) return fail(ICON_EINVAL, "dycore_velocity_tendencies_noalloc: nlev > 128");
    const size_t es = dtype == ICON_F64 ? 8 : 4;
    if (ldk_w < nlev + 1) return fail(ICON_EINVAL, "ldk_w < nlev+1");
    if (((int64_t)ldk_w * (int64_t)es) % 16) return fail(ICON_EINVAL, "ldk_w*sizeof(T) must be a multiple of 16");
    if (!z_half) return fail(ICON_EINVAL, "z_half is NULL");
    for (int k = 0; k < nlev; ++k)
        if (!(z_half[k] > z_half[k + 1])) return fail(ICON_EINVAL, "z_half must be strictly decreasing");
    if ((rc = check_field(vn, "vn")) || (rc = check_field(w, "w")) || (rc = check_field(ddt_vn, "ddt_vn"))) return rc;
    const size_t be = (size_t)g->host.ne * ldk * es, bw = (size_t)g->host.nc * ldk_w * es;
    if (overlaps(ddt_vn, be, vn, be) || overlaps(ddt_vn, be, w, bw)) return fail(ICON_EINVAL, "outputs must not alias inputs");
    cudaStream_t s = (cudaStream_t)cuda_stream;
    if (dtype == ICON_F64) return noalloc_impl<double>(g, g->c64, nlev, ldk, ldk_w, z_half, vn, w, ddt_vn, s);
    return noalloc_impl<float>(g, g->c32, nlev, ldk, ldk_w, z_half, vn, w, ddt_vn, s);
}
