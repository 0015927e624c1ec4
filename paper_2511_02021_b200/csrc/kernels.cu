// kernels.cu -- sm_100a kernels for the dycore sweep.
//
// Layout facts every kernel here relies on (include/icon_dycore.h):
//   fields are level-contiguous x[i*ldk + k]; a warp owns ONE entity column and its 32 lanes walk
//   consecutive levels, so every gather of a neighbour column is a fully coalesced 256-byte
//   (fp64) / 128-byte (fp32) read, whatever the horizontal numbering is; neighbour indices and
//   coefficients are warp-uniform and are read once per column, not once per point (the
//   index-lookup amortisation of PAPER.md:186).
#include "kernels.cuh"

namespace icon {
namespace {

constexpr int kWarp = 32;

__device__ __forceinline__ int lane_id() { return threadIdx.x & 31; }
// through a shuffle so that the compiler knows the value is warp-uniform (uniform branches, no divergence handling)
__device__ __forceinline__ int warp_in_block() { return __shfl_sync(0xffffffffu, (int)(threadIdx.x >> 5), 0); }

template <class T>
__device__ __forceinline__ T ldg(const T* p) {
    return __ldg(p);
}

// ------------------------------------------------------------------------------------------
// S1 + S2: div(c,k) = sum_j geofac_div(c,j) vn(c2e[c][j],k); vort(v,k) = sum_j geofac_rot(v,j) vn(v2e[v][j],k)
// block = 12 warps: warps 0..7 take 8 consecutive cells, warps 8..11 take the 4 vertices of the
// same stretch of the generation order, so both read the same vn columns while they are in L1/L2.
// ------------------------------------------------------------------------------------------
// All 6 * L column loads of a warp are issued before the first use (L = level chunks per lane is a
// template parameter so that the loop over chunks unrolls): the kernel is a pure stream with one
// dependent lookup (ids -> columns), and what limits it is the number of bytes in flight per SM.
// volatile asm: the loads keep their program order, i.e. all of them are issued before the first FMA
__device__ __forceinline__ double ld_stream(const double* p) {
    double v;
    asm volatile("ld.global.nc.f64 %0, [%1];" : "=d"(v) : "l"(p));
    return v;
}
__device__ __forceinline__ float ld_stream(const float* p) {
    float v;
    asm volatile("ld.global.nc.f32 %0, [%1];" : "=f"(v) : "l"(p));
    return v;
}

// Persistent version: 8 warps per block, warps 0..3 take two cells each, warps 4..7 one vertex each
// of chunk t (8 cells + the 4 vertices of the same stretch of the generation order, so both hit the
// same vn columns while they are in L1/L2) -- 6 neighbour columns and 18 loads in flight per warp
// either way. The ids and coefficients of the NEXT chunk are fetched before the columns of the
// current one are, which takes the dependent lookup (ids -> columns) off the critical path; with
// one short-lived block per 8 cells the kernel spent its time in waves of two latencies each.
template <class T, int L>
__global__ void __launch_bounds__(256, 2) k_div_vort(int64_t nc, int64_t nv, int nlev, int64_t ldk,
                                                     const int32_t* __restrict__ c2e, const T* __restrict__ geofac_div,
                                                     const int32_t* __restrict__ v2e, const T* __restrict__ geofac_rot,
                                                     const int32_t* __restrict__ user_c, const int32_t* __restrict__ user_v,
                                                     const T* __restrict__ vn, T* __restrict__ div, T* __restrict__ vort) {
    const int w = warp_in_block(), lane = lane_id();
    const bool cells = w < 4;
    const int wi = w & 3;
    const int64_t n_ent = cells ? nc : nv;
    const int32_t* ids = cells ? c2e : v2e;
    const T* coef = cells ? geofac_div : geofac_rot;
    const int32_t* user = cells ? user_c : user_v;
    T* out = cells ? div : vort;
    const int64_t n_chunks = (nc + 7) / 8 > (nv + 3) / 4 ? (nc + 7) / 8 : (nv + 3) / 4;
    // six (id, coefficient) pairs: two cells (3 + 3) or one vertex (6); row = first entity of the warp
    struct Meta {
        int32_t id[6];
        T g[6];
        int64_t o0, o1;       // output columns (user ids), -1 = none
    };
    auto load_meta = [&](int64_t t) {
        Meta m;
        const int64_t p = cells ? t * 8 + wi * 2 : t * 4 + wi;
        const bool v0 = t < n_chunks && p < n_ent, v1 = cells && t < n_chunks && p + 1 < n_ent;
#pragma unroll
        for (int j = 0; j < 6; ++j) {
            const bool ok = cells ? (j < 3 ? v0 : v1) : v0;
            m.id[j] = ok ? ldg(ids + 6 * (cells ? p / 2 : p) + j) : 0;       // cells: rows p, p+1 = 6 consecutive entries (p even)
            m.g[j] = ok ? ldg(coef + 6 * (cells ? p / 2 : p) + j) : (T)0;
        }
        m.o0 = v0 ? (user ? (int64_t)ldg(user + p) : p) : -1;
        m.o1 = v1 ? (user ? (int64_t)ldg(user + p + 1) : p + 1) : -1;
        return m;
    };
    // a block takes kRun consecutive chunks (64 cells + their 32 vertices) before it jumps on, so that the
    // columns neighbouring chunks share are still in its L1 when the next one asks for them
    constexpr int kRun = 8;
    auto chunk_of = [&](int64_t q) { return ((int64_t)blockIdx.x + (q / kRun) * (int64_t)gridDim.x) * kRun + q % kRun; };
    Meta nxt = load_meta(chunk_of(0));
    for (int64_t q = 0; chunk_of(q) - q % kRun < n_chunks; ++q) {
        const Meta cur = nxt;
        nxt = load_meta(chunk_of(q + 1));
        for (int k0 = 0; k0 < nlev; k0 += kWarp * L) {
            T x[6][L];
#pragma unroll
            for (int j = 0; j < 6; ++j) {
                const T* col = vn + (int64_t)cur.id[j] * ldk + k0;
#pragma unroll
                for (int l = 0; l < L; ++l) {
                    const int k = lane + kWarp * l;
                    x[j][l] = ld_stream(col + (k0 + k < nlev ? k : nlev - 1 - k0));   // past the end: re-read the last level, unused
                }
            }
#pragma unroll
            for (int l = 0; l < L; ++l) {
                const int k = k0 + lane + kWarp * l;
                const T a = cur.g[0] * x[0][l] + cur.g[1] * x[1][l] + cur.g[2] * x[2][l];
                const T b = cur.g[3] * x[3][l] + cur.g[4] * x[4][l] + cur.g[5] * x[5][l];
                if (k < nlev) {
                    if (cells) {
                        if (cur.o0 >= 0) out[cur.o0 * ldk + k] = a;
                        if (cur.o1 >= 0) out[cur.o1 * ldk + k] = b;
                    } else if (cur.o0 >= 0) {
                        // S2 in slot order: ((((g0 x0 + g1 x1) + g2 x2) + g3 x3) + g4 x4) + g5 x5 up to rounding order
                        out[cur.o0 * ldk + k] = a + b;
                    }
                }
            }
        }
    }
}

// ------------------------------------------------------------------------------------------
// unfused pipeline (validation baseline; intermediates through HBM)
// ------------------------------------------------------------------------------------------
// S3 + S4a: vt = sum_j rbf(e,j) vn(e2e4[e][j]); KE_e = 1/2 (vn^2 + vt^2)
template <class T>
__global__ void __launch_bounds__(256) k_vt_kee(int64_t ne, int nlev, int64_t ldk, const int32_t* __restrict__ e2e4,
                                                const T* __restrict__ rbf, const int32_t* __restrict__ user_e,
                                                const T* __restrict__ vn, T* __restrict__ vt, T* __restrict__ ke_e) {
    const int64_t p = (int64_t)blockIdx.x * 8 + warp_in_block();
    if (p >= ne) return;
    const int lane = lane_id();
    const int64_t e = user_e ? user_e[p] : p;
    const T* col[4];
    T r[4];
#pragma unroll
    for (int j = 0; j < 4; ++j) {
        col[j] = vn + (int64_t)ldg(e2e4 + 4 * p + j) * ldk;
        r[j] = ldg(rbf + 4 * p + j);
    }
    const T* own = vn + e * ldk;
    for (int k = lane; k < nlev; k += kWarp) {
        T t = r[0] * col[0][k] + r[1] * col[1][k] + r[2] * col[2][k] + r[3] * col[3][k];
        T n = own[k];
        vt[e * ldk + k] = t;
        ke_e[e * ldk + k] = (T)0.5 * (n * n + t * t);
    }
}

// S4b + S2: KE_c = sum_j bln(c,j) KE_e(c2e[c][j]); zeta
template <class T>
__global__ void __launch_bounds__(384) k_kec_vort(int64_t nc, int64_t nv, int nlev, int64_t ldk,
                                                  const int32_t* __restrict__ c2e, const T* __restrict__ bln,
                                                  const int32_t* __restrict__ v2e, const T* __restrict__ geofac_rot,
                                                  const int32_t* __restrict__ user_c, const int32_t* __restrict__ user_v,
                                                  const T* __restrict__ ke_e, const T* __restrict__ vn,
                                                  T* __restrict__ ke_c, T* __restrict__ vort) {
    const int w = warp_in_block(), lane = lane_id();
    if (w < 8) {
        const int64_t p = (int64_t)blockIdx.x * 8 + w;
        if (p >= nc) return;
        const int64_t c = user_c ? user_c[p] : p;
        const T* col0 = ke_e + (int64_t)ldg(c2e + 3 * p) * ldk;
        const T* col1 = ke_e + (int64_t)ldg(c2e + 3 * p + 1) * ldk;
        const T* col2 = ke_e + (int64_t)ldg(c2e + 3 * p + 2) * ldk;
        const T b0 = ldg(bln + 3 * p), b1 = ldg(bln + 3 * p + 1), b2 = ldg(bln + 3 * p + 2);
        T* out = ke_c + c * ldk;
        for (int k = lane; k < nlev; k += kWarp) out[k] = b0 * col0[k] + b1 * col1[k] + b2 * col2[k];
    } else {
        const int64_t p = (int64_t)blockIdx.x * 4 + (w - 8);
        if (p >= nv) return;
        const int64_t v = user_v ? user_v[p] : p;
        const T* col[6];
        T g[6];
#pragma unroll
        for (int j = 0; j < 6; ++j) {
            col[j] = vn + (int64_t)ldg(v2e + 6 * p + j) * ldk;
            g[j] = ldg(geofac_rot + 6 * p + j);
        }
        T* out = vort + v * ldk;
        for (int k = lane; k < nlev; k += kWarp) {
            T s = g[0] * col[0][k];
#pragma unroll
            for (int j = 1; j < 6; ++j) s += g[j] * col[j][k];
            out[k] = s;
        }
    }
}

// vertical difference (vn_ie(k) - vn_ie(k+1))/dz_k = A_k vn(k-1) + B_k vn(k) + C_k vn(k+1)
// with A_0 = C_{K-1} = 0 (reading P-14 folded into per-level coefficients on the host)
template <class T>
__device__ __forceinline__ T vertical_diff(const T* __restrict__ col, const T* __restrict__ abc, int nlev, int k) {
    const int km = k > 0 ? k - 1 : 0, kp = k < nlev - 1 ? k + 1 : nlev - 1;
    return ldg(abc + k) * col[km] + ldg(abc + nlev + k) * col[k] + ldg(abc + 2 * nlev + k) * col[kp];
}

// S5 + S6 + S7
template <class T>
__global__ void __launch_bounds__(256) k_ddt_vn(int64_t ne, int nlev, int64_t ldk, int64_t ldk_w,
                                                const int32_t* __restrict__ e2c, const int32_t* __restrict__ e2v,
                                                const T* __restrict__ inv_d_e, const T* __restrict__ f_e,
                                                const T* __restrict__ c_lin, const int32_t* __restrict__ user_e,
                                                const T* __restrict__ abc, const T* __restrict__ vn,
                                                const T* __restrict__ w, const T* __restrict__ vt,
                                                const T* __restrict__ ke_c, const T* __restrict__ vort,
                                                T* __restrict__ ddt_vn) {
    const int64_t p = (int64_t)blockIdx.x * 8 + warp_in_block();
    if (p >= ne) return;
    const int lane = lane_id();
    const int64_t e = user_e ? user_e[p] : p;
    const int64_t c0 = ldg(e2c + 2 * p), c1 = ldg(e2c + 2 * p + 1), v0 = ldg(e2v + 2 * p), v1 = ldg(e2v + 2 * p + 1);
    const T inv_d = ldg(inv_d_e + p), f = ldg(f_e + p), cl0 = ldg(c_lin + 2 * p), cl1 = ldg(c_lin + 2 * p + 1);
    const T* col = vn + e * ldk;
    for (int k = lane; k < nlev; k += kWarp) {
        T gradk = (ke_c[c1 * ldk + k] - ke_c[c0 * ldk + k]) * inv_d;
        T zeta_e = (T)0.5 * (vort[v0 * ldk + k] + vort[v1 * ldk + k]);
        T H = gradk + vt[e * ldk + k] * (f + zeta_e);
        T wf0 = (T)0.5 * (w[c0 * ldk_w + k] + w[c0 * ldk_w + k + 1]);
        T wf1 = (T)0.5 * (w[c1 * ldk_w + k] + w[c1 * ldk_w + k + 1]);
        T w_e = cl0 * wf0 + cl1 * wf1;
        ddt_vn[e * ldk + k] = -(H + w_e * vertical_diff(col, abc, nlev, k));
    }
}

// ------------------------------------------------------------------------------------------
// Vertical-wind tendency (reading P-19): one warp per cell column, lanes = half levels.
//   ddt_w(c,k) = -[ sum_j adv_c(c,j) vn_ie(e_j,k) (w(c1_j,k) - w(c0_j,k)) inv_d_e(e_j) + w(c,k) (w(c,k-1) - w(c,k+1)) rdz2(k) ]
// for k = 1 .. nlev-1, 0 at k = 0 and k = nlev. wk = [2][nlev+1]: g_k (weight of vn(k) in vn_ie(k), P-14) and
// rdz2(k) = 1 / (z_half[k-1] - z_half[k+1]). Ids, cells and the folded coefficient adv_c * inv_d_e are warp-uniform.
// ------------------------------------------------------------------------------------------
template <class T>
__global__ void __launch_bounds__(256) k_w_tend(int64_t nc, int nlev, int64_t ldk, int64_t ldk_w,
                                                const int32_t* __restrict__ c2e, const int32_t* __restrict__ e2c,
                                                const T* __restrict__ inv_d_e, const T* __restrict__ adv_c,
                                                const int32_t* __restrict__ user_c, const int32_t* __restrict__ pos_e,
                                                const T* __restrict__ wk, const T* __restrict__ vn, const T* __restrict__ w,
                                                T* __restrict__ ddt_w) {
    const int64_t p = (int64_t)blockIdx.x * 8 + warp_in_block();
    if (p >= nc) return;
    const int lane = lane_id();
    const int64_t c = user_c ? user_c[p] : p;
    const T *vcol[3], *w0[3], *w1[3];
    T a[3];
#pragma unroll
    for (int j = 0; j < 3; ++j) {
        const int64_t e = ldg(c2e + 3 * p + j);
        const int64_t pe = pos_e ? pos_e[e] : e;                 // row of the edge tables (work order)
        vcol[j] = vn + e * ldk;
        w0[j] = w + (int64_t)ldg(e2c + 2 * pe) * ldk_w;
        w1[j] = w + (int64_t)ldg(e2c + 2 * pe + 1) * ldk_w;
        a[j] = ldg(adv_c + 3 * p + j) * ldg(inv_d_e + pe);
    }
    const T* wc = w + c * ldk_w;
    T* out = ddt_w + c * ldk_w;
    for (int k = lane; k <= nlev; k += kWarp) {
        T val = (T)0;
        if (k >= 1 && k <= nlev - 1) {
            const T g = ldg(wk + k), rdz2 = ldg(wk + nlev + 1 + k);
            T hadv = (T)0;
#pragma unroll
            for (int j = 0; j < 3; ++j) {
                const T vie = g * vcol[j][k] + ((T)1 - g) * vcol[j][k - 1];
                hadv += a[j] * vie * (w1[j][k] - w0[j][k]);
            }
            val = -(hadv + wc[k] * (wc[k - 1] - wc[k + 1]) * rdz2);
        }
        out[k] = val;
    }
}

// ------------------------------------------------------------------------------------------
// Metric variant (reading P-20), plain kernels: set-up of the per-edge vertical metrics and the
// last stage of the unfused pipeline. One warp per edge column, lanes = levels.
// ------------------------------------------------------------------------------------------
template <class T>
__global__ void __launch_bounds__(256) k_metric_from_zhalf(int64_t ne, int nlev, int64_t ldk, int64_t ldk_w,
                                                           const T* __restrict__ zh, T* __restrict__ wgt, T* __restrict__ inv) {
    const int64_t e = (int64_t)blockIdx.x * 8 + warp_in_block();
    if (e >= ne) return;
    const T* z = zh + e * ldk_w;
    for (int k = lane_id(); k <= nlev; k += kWarp) {
        if (k < nlev) inv[e * ldk + k] = (T)1 / (z[k] - z[k + 1]);
        T up, dn;
        if (k == 0) { up = z[0] - z[1]; dn = z[1] - z[2]; }                                   // dz0 / (dz0 + dz1)
        else if (k == nlev) { up = z[nlev - 1] - z[nlev]; dn = z[nlev - 2] - z[nlev - 1]; }   // dz(K-1) / (dz(K-1) + dz(K-2))
        else { up = z[k - 1] - z[k]; dn = z[k] - z[k + 1]; }
        wgt[e * ldk_w + k] = up / (up + dn);
    }
}

template <class T>
__global__ void __launch_bounds__(256) k_ddt_vn_metric(int64_t ne, int nlev, int64_t ldk, int64_t ldk_w,
                                                       const int32_t* __restrict__ e2c, const int32_t* __restrict__ e2v,
                                                       const T* __restrict__ cgrad, const T* __restrict__ f_e,
                                                       const T* __restrict__ c_lin, const int32_t* __restrict__ user_e,
                                                       const T* __restrict__ wgt, const T* __restrict__ inv,
                                                       const T* __restrict__ zn, const T* __restrict__ zt,
                                                       const T* __restrict__ vn, const T* __restrict__ w,
                                                       const T* __restrict__ vt, const T* __restrict__ ke_e,
                                                       const T* __restrict__ ke_c, const T* __restrict__ vort,
                                                       T* __restrict__ ddt_vn) {
    const int64_t p = (int64_t)blockIdx.x * 8 + warp_in_block();
    if (p >= ne) return;
    const int lane = lane_id();
    const int64_t e = user_e ? user_e[p] : p;
    const int64_t c0 = ldg(e2c + 2 * p), c1 = ldg(e2c + 2 * p + 1), v0 = ldg(e2v + 2 * p), v1 = ldg(e2v + 2 * p + 1);
    const T g0 = ldg(cgrad + 2 * p), g1 = ldg(cgrad + 2 * p + 1), f = ldg(f_e + p), cl0 = ldg(c_lin + 2 * p), cl1 = ldg(c_lin + 2 * p + 1);
    const T* col = vn + e * ldk;
    const T* wg = wgt + e * ldk_w;
    auto half = [&](int k) {
        if (k == 0) return col[0] + wg[0] * (col[0] - col[1]);
        if (k == nlev) return col[nlev - 1] + wg[nlev] * (col[nlev - 1] - col[nlev - 2]);
        return wg[k] * col[k] + ((T)1 - wg[k]) * col[k - 1];
    };
    for (int k = lane; k < nlev; k += kWarp) {
        const int64_t i = e * ldk + k;
        const T t = vt[i];
        const T gradk = g1 * ke_c[c1 * ldk + k] - g0 * ke_c[c0 * ldk + k] + ke_e[i] * (g0 - g1);
        const T zeta_e = (T)0.5 * (vort[v0 * ldk + k] + vort[v1 * ldk + k]);
        const T H = gradk + t * (f + zeta_e);
        const T wf0 = (T)0.5 * (w[c0 * ldk_w + k] + w[c0 * ldk_w + k + 1]);
        const T wf1 = (T)0.5 * (w[c1 * ldk_w + k] + w[c1 * ldk_w + k + 1]);
        const T w_e = cl0 * wf0 + cl1 * wf1;
        const T w_cc = col[k] * zn[i] + t * zt[i];
        ddt_vn[i] = -(H + (w_e - w_cc) * (half(k) - half(k + 1)) * inv[i]);
    }
}

inline unsigned blocks_for(int64_t n, int per_block) { return (unsigned)((n + per_block - 1) / per_block); }

}  // namespace

template <class T>
int launch_div_vort(const icon_grid& g, const DevCoeffs<T>& c, int nlev, int64_t ldk, const T* vn, T* div, T* vort,
                    cudaStream_t s) {
    const int64_t nc = g.host.nc, nv = g.host.nv;
    unsigned nb = blocks_for(nc, 8);
    unsigned nbv = blocks_for(nv, 4);
    if (nbv > nb) nb = nbv;
    nb = (nb + 7) / 8;                                                                 // a block walks runs of 8 chunks
    const unsigned persistent = (unsigned)(g.num_sms > 0 ? g.num_sms : 148) * 2u;      // two blocks per SM
    if (nb > persistent) nb = persistent;
    if (nlev <= 32)
        k_div_vort<T, 1><<<nb, 256, 0, s>>>(nc, nv, nlev, ldk, g.tab.c2e, c.geofac_div, g.tab.v2e, c.geofac_rot, g.tab.user_c,
                                            g.tab.user_v, vn, div, vort);
    else if (nlev <= 64)
        k_div_vort<T, 2><<<nb, 256, 0, s>>>(nc, nv, nlev, ldk, g.tab.c2e, c.geofac_div, g.tab.v2e, c.geofac_rot, g.tab.user_c,
                                            g.tab.user_v, vn, div, vort);
    else
        k_div_vort<T, 3><<<nb, 256, 0, s>>>(nc, nv, nlev, ldk, g.tab.c2e, c.geofac_div, g.tab.v2e, c.geofac_rot, g.tab.user_c,
                                            g.tab.user_v, vn, div, vort);
    cudaError_t err = cudaGetLastError();
    return err == cudaSuccess ? 1 : -(int)err;
}

template <class T>
int launch_tendencies_unfused(const icon_grid& g, const DevCoeffs<T>& c, int nlev, int64_t ldk, int64_t ldk_w,
                              const T* abc, const T* vn, const T* w, T* ddt_vn, T* vt, T* ke_e, T* ke_c, T* vort,
                              cudaStream_t s) {
    const int64_t nc = g.host.nc, ne = g.host.ne, nv = g.host.nv;
    k_vt_kee<T><<<blocks_for(ne, 8), 256, 0, s>>>(ne, nlev, ldk, g.tab.e2e4, c.rbf, g.tab.user_e, vn, vt, ke_e);
    unsigned nb = blocks_for(nc, 8), nbv = blocks_for(nv, 4);
    if (nbv > nb) nb = nbv;
    k_kec_vort<T><<<nb, 384, 0, s>>>(nc, nv, nlev, ldk, g.tab.c2e, c.bln, g.tab.v2e, c.geofac_rot, g.tab.user_c,
                                     g.tab.user_v, ke_e, vn, ke_c, vort);
    k_ddt_vn<T><<<blocks_for(ne, 8), 256, 0, s>>>(ne, nlev, ldk, ldk_w, g.tab.e2c, g.tab.e2v, c.inv_d_e, c.f_e, c.c_lin,
                                                  g.tab.user_e, abc, vn, w, vt, ke_c, vort, ddt_vn);
    cudaError_t err = cudaGetLastError();
    return err == cudaSuccess ? 3 : -(int)err;
}

// ------------------------------------------------------------------------------------------
// dycore_halo_pack: the send side of the halo exchange. Whole rows (columns of the field with their
// padding) are gathered by 16-byte chunks: consecutive threads take consecutive chunks of a row, so the reads of a row
// and all writes are contiguous. Bytes moved = 2 x n_rows x row_bytes, a few MB per rank at R2B8 / 8 ranks.
// ------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256) k_halo_pack(const int32_t* __restrict__ ids, int64_t n_rows, int chunks_per_row,
                                                   const int4* __restrict__ field, int4* __restrict__ out) {
    const int64_t total = n_rows * chunks_per_row;
    for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < total; i += (int64_t)gridDim.x * blockDim.x) {
        const int64_t r = i / chunks_per_row;
        const int c = (int)(i - r * chunks_per_row);
        out[i] = __ldg(field + (int64_t)__ldg(ids + r) * chunks_per_row + c);
    }
}

int launch_halo_pack(const int32_t* ids, int64_t n_rows, int64_t row_bytes, const void* field, void* out, cudaStream_t s) {
    if (n_rows == 0) return 0;
    const int cpr = (int)(row_bytes / 16);
    const int64_t total = n_rows * cpr;
    int64_t nb = (total + 255) / 256;
    if (nb > 148 * 8) nb = 148 * 8;
    k_halo_pack<<<(unsigned)nb, 256, 0, s>>>(ids, n_rows, cpr, (const int4*)field, (int4*)out);
    cudaError_t err = cudaGetLastError();
    return err == cudaSuccess ? 1 : -(int)err;
}

template <class T>
int launch_metric_from_zhalf(const icon_grid& g, int nlev, int64_t ldk, int64_t ldk_w, const T* zh, T* wgt, T* inv, cudaStream_t s) {
    const int64_t ne = g.host.ne;
    k_metric_from_zhalf<T><<<blocks_for(ne, 8), 256, 0, s>>>(ne, nlev, ldk, ldk_w, zh, wgt, inv);
    cudaError_t err = cudaGetLastError();
    return err == cudaSuccess ? 1 : -(int)err;
}

template <class T>
int launch_tendencies_unfused_metric(const icon_grid& g, const DevCoeffs<T>& c, int nlev, int64_t ldk, int64_t ldk_w, const T* wgt,
                                     const T* inv, const T* zn, const T* zt, const T* vn, const T* w, T* ddt_vn, T* vt, T* ke_e,
                                     T* ke_c, T* vort, cudaStream_t s) {
    const int64_t nc = g.host.nc, ne = g.host.ne, nv = g.host.nv;
    k_vt_kee<T><<<blocks_for(ne, 8), 256, 0, s>>>(ne, nlev, ldk, g.tab.e2e4, c.rbf, g.tab.user_e, vn, vt, ke_e);
    unsigned nb = blocks_for(nc, 8), nbv = blocks_for(nv, 4);
    if (nbv > nb) nb = nbv;
    k_kec_vort<T><<<nb, 384, 0, s>>>(nc, nv, nlev, ldk, g.tab.c2e, c.bln, g.tab.v2e, c.geofac_rot, g.tab.user_c,
                                     g.tab.user_v, ke_e, vn, ke_c, vort);
    k_ddt_vn_metric<T><<<blocks_for(ne, 8), 256, 0, s>>>(ne, nlev, ldk, ldk_w, g.tab.e2c, g.tab.e2v, c.cgrad, c.f_e, c.c_lin,
                                                         g.tab.user_e, wgt, inv, zn, zt, vn, w, vt, ke_e, ke_c, vort, ddt_vn);
    cudaError_t err = cudaGetLastError();
    return err == cudaSuccess ? 3 : -(int)err;
}

template <class T>
int launch_w_tendency(const icon_grid& g, const DevCoeffs<T>& c, int nlev, int64_t ldk, int64_t ldk_w, const T* wk,
                      const T* vn, const T* w, T* ddt_w, cudaStream_t s) {
    const int64_t nc = g.host.nc;
    k_w_tend<T><<<blocks_for(nc, 8), 256, 0, s>>>(nc, nlev, ldk, ldk_w, g.tab.c2e, g.tab.e2c, c.inv_d_e, c.adv_c, g.tab.user_c,
                                                  g.tab.pos_e, wk, vn, w, ddt_w);
    cudaError_t err = cudaGetLastError();
    return err == cudaSuccess ? 1 : -(int)err;
}

#define ICON_INSTANTIATE(T)                                                                                             \
    template int launch_div_vort<T>(const icon_grid&, const DevCoeffs<T>&, int, int64_t, const T*, T*, T*, cudaStream_t); \
    template int launch_tendencies_unfused<T>(const icon_grid&, const DevCoeffs<T>&, int, int64_t, int64_t, const T*,     \
                                              const T*, const T*, T*, T*, T*, T*, T*, cudaStream_t);                      \
    template int launch_w_tendency<T>(const icon_grid&, const DevCoeffs<T>&, int, int64_t, int64_t, const T*, const T*,   \
                                      const T*, T*, cudaStream_t);                                                        \
    template int launch_metric_from_zhalf<T>(const icon_grid&, int, int64_t, int64_t, const T*, T*, T*, cudaStream_t);    \
    template int launch_tendencies_unfused_metric<T>(const icon_grid&, const DevCoeffs<T>&, int, int64_t, int64_t,        \
                                                     const T*, const T*, const T*, const T*, const T*, const T*, T*, T*,  \
                                                     T*, T*, T*, cudaStream_t);
ICON_INSTANTIATE(double)
ICON_INSTANTIATE(float)

}  // namespace icon
