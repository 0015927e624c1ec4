// kernels_sc.cu -- self-contained patch kernel for the velocity tendency,
// sm_100a.
//
// One warp = one patch (four sibling cells, six owned edges; sc_tables.hpp), no exchange between
// warps, no block barrier. The lanes of the warp are consecutive LEVELS, and every lane carries
// L level chunks at once, so that a neighbour id or a coefficient, which is warp-uniform, is
// fetched from shared memory once per patch and used for L*30 levels (the index-lookup
// amortisation of PAPER.md:186 taken to the whole column): with lanes = levels a coefficient
// costs one shared-memory broadcast per 32 points, which is what bounded the previous kernel
// (profiles/r01_lsu_microbench.md); with L = 3 it is one per 90.
//
// Level chunks overlap by one level on each side: chunk c covers levels 30c-1 .. 30c+30, lanes
// 1..30 produce output, lanes 0 and 31 only feed vn(k-1), vn(k+1) and w(k+1) to their neighbours
// through warp shuffles (S6), so the vertical stencil costs no extra memory access. 90 levels are
// exactly three chunks.
//
// Per patch and chunk the warp reads 36 vn columns and 7 w columns straight from global memory
// (each a contiguous 256-byte run, reuse between neighbouring patches through L1/L2), evaluates 15
// tangential winds, 15 edge and 7 cell kinetic energies and 6 vorticities in registers and stores 6
// ddt_vn columns. The patch record (ids + coefficients in local slot order) is staged per warp
// with cp.async one patch ahead. No intermediate reaches HBM.
#include <cuda_pipeline.h>

#include "kernels.cuh"
#include "sc_tables.hpp"

namespace icon {
namespace {

constexpr int kScWarps = 8;
constexpr int kScThreads = kScWarps * 32;
constexpr int kChunk = 30;                      // output levels per chunk
constexpr unsigned kFull = 0xffffffffu;

template <class T>
struct ScDev {
    const int32_t* ids;
    const T* coef;
    int64_t n_patches;
};

template <class T>
__host__ __device__ constexpr int sc_record_bytes() { return kScCoefWords * (int)sizeof(T) + kScIdWords * 4; }

template <class T, int L>
struct Col {
    T v[L];
};

#define FORL _Pragma("unroll") for (int l = 0; l < L; ++l)

template <class T, int L>
__device__ __forceinline__ Col<T, L> shfl_up1(const Col<T, L>& a) {
    Col<T, L> r;
    FORL r.v[l] = __shfl_up_sync(kFull, a.v[l], 1);
    return r;
}
template <class T, int L>
__device__ __forceinline__ Col<T, L> shfl_down1(const Col<T, L>& a) {
    Col<T, L> r;
    FORL r.v[l] = __shfl_down_sync(kFull, a.v[l], 1);
    return r;
}

// r0*a + r1*b + r2*c + r3*d
template <class T, int L>
__device__ __forceinline__ Col<T, L> dot4(const T* r, const Col<T, L>& a, const Col<T, L>& b, const Col<T, L>& c,
                                          const Col<T, L>& d) {
    Col<T, L> o;
    FORL o.v[l] = r[0] * a.v[l] + r[1] * b.v[l] + r[2] * c.v[l] + r[3] * d.v[l];
    return o;
}
// n^2 + t^2 (twice the edge kinetic energy, S4)
template <class T, int L>
__device__ __forceinline__ Col<T, L> ke2(const Col<T, L>& n, const Col<T, L>& t) {
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

// N coefficients (N * sizeof(T) a multiple of 16, p 16-byte aligned) from shared memory
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
template <int N>
__device__ __forceinline__ void ld_ids(const int32_t* __restrict__ p, int32_t (&out)[N]) {
    static_assert(N % 4 == 0, "id group must be a multiple of 16 bytes");
    const int4* q = reinterpret_cast<const int4*>(p);
#pragma unroll
    for (int i = 0; i < N / 4; ++i) {
        int4 v = q[i];
        out[4 * i] = v.x; out[4 * i + 1] = v.y; out[4 * i + 2] = v.z; out[4 * i + 3] = v.w;
    }
}

// one warp stages the record of patch p into its private buffer
template <class T>
__device__ __forceinline__ void stage_record(const ScDev<T>& d, unsigned char* buf, int64_t p, int lane) {
    const unsigned char* sc = reinterpret_cast<const unsigned char*>(d.coef + p * kScCoefWords);
    const unsigned char* si = reinterpret_cast<const unsigned char*>(d.ids + p * kScIdWords);
    constexpr int cb = kScCoefWords * (int)sizeof(T), ib = kScIdWords * 4;
    for (int o = lane * 16; o < cb; o += 512) __pipeline_memcpy_async(buf + o, sc + o, 16);
    for (int o = lane * 16; o < ib; o += 512) __pipeline_memcpy_async(buf + cb + o, si + o, 16);
    __pipeline_commit();
}

template <class T, int L>
__global__ void __launch_bounds__(kScThreads, 1)
k_tend_sc(ScDev<T> d, int nlev, int ldk, int ldk_w, const T* __restrict__ abc, const T* __restrict__ vn,
          const T* __restrict__ w, T* __restrict__ ddt_vn) {
    extern __shared__ __align__(16) unsigned char smem[];
    using C = Col<T, L>;
    constexpr int rec = sc_record_bytes<T>();
    const int warp = __shfl_sync(0xffffffffu, (int)(threadIdx.x >> 5), 0), lane = threadIdx.x & 31;      // warp-uniform for the compiler
    unsigned char* mybuf = smem + warp * 2 * rec;
    const int n_chunks = (nlev + kChunk - 1) / kChunk;
    const uint64_t cs = (uint64_t)ldk * sizeof(T), cs_w = (uint64_t)ldk_w * sizeof(T);
    const int64_t stride = (int64_t)gridDim.x * kScWarps;

    int64_t p = (int64_t)blockIdx.x * kScWarps + warp;
    if (p >= d.n_patches) return;
    stage_record(d, mybuf, p, lane);
    int rb = 0;
    for (; p < d.n_patches; p += stride, rb ^= 1) {
        const int64_t pn = p + stride;
        if (pn < d.n_patches) {
            stage_record(d, mybuf + (rb ^ 1) * rec, pn, lane);
            __pipeline_wait_prior(1);
        } else {
            __pipeline_wait_prior(0);
        }
        __syncwarp();
        const T* cf = reinterpret_cast<const T*>(mybuf + rb * rec);
        const int32_t* sid = reinterpret_cast<const int32_t*>(mybuf + rb * rec + kScCoefWords * sizeof(T));

        for (int c0 = 0; c0 < n_chunks; c0 += L) {
            const int k0 = kChunk * c0 - 1 + lane;
            bool pv[L], pw[L], po[L];
            T cA[L], cB[L], cC[L];
            FORL {
                const int k = k0 + kChunk * l;
                pv[l] = k >= 0 && k < nlev;
                pw[l] = k >= 0 && k <= nlev;
                po[l] = pv[l] && lane >= 1 && lane <= kChunk;
                cA[l] = pv[l] ? __ldg(abc + k) : (T)0;
                cB[l] = pv[l] ? __ldg(abc + nlev + k) : (T)0;
                cC[l] = pv[l] ? __ldg(abc + 2 * nlev + k) : (T)0;
            }
            const uint64_t vn_lane = reinterpret_cast<uint64_t>(vn) + (int64_t)k0 * (int64_t)sizeof(T);
            const uint64_t w_lane = reinterpret_cast<uint64_t>(w) + (int64_t)k0 * (int64_t)sizeof(T);
            const uint64_t out_lane = reinterpret_cast<uint64_t>(ddt_vn) + (int64_t)k0 * (int64_t)sizeof(T);
            auto LD = [&](int32_t id) {
                const T* q = reinterpret_cast<const T*>(vn_lane + (uint64_t)(uint32_t)id * cs);
                C c;
                FORL c.v[l] = pv[l] ? q[kChunk * l] : (T)0;
                return c;
            };
            auto WF = [&](int32_t id) {       // w_f(k) = (w(k) + w(k+1)) / 2 (S6)
                const T* q = reinterpret_cast<const T*>(w_lane + (uint64_t)(uint32_t)id * cs_w);
                C c;
                FORL c.v[l] = pw[l] ? q[kChunk * l] : (T)0;
                C dn = shfl_down1(c);
                FORL c.v[l] = (T)0.5 * (c.v[l] + dn.v[l]);
                return c;
            };
            auto VD = [&](const C& x) {       // (vn_ie(k) - vn_ie(k+1)) / dz_k, reading P-14 folded into A, B, C
                C up = shfl_up1(x), dn = shfl_down1(x), o;
                FORL o.v[l] = cA[l] * up.v[l] + cB[l] * x.v[l] + cC[l] * dn.v[l];
                return o;
            };
            auto ST = [&](int32_t id, const C& x) {
                T* q = reinterpret_cast<T*>(out_lane + (uint64_t)(uint32_t)id * cs);
                FORL if (po[l]) q[kChunk * l] = x.v[l];
            };

            int32_t idE[12];                    // i0 i1 i2 b0..b5 om0 om1 om2
            ld_ids(sid + SID_I0, idE);
            C vI[3], vB[6];
#pragma unroll
            for (int j = 0; j < 3; ++j) vI[j] = LD(idE[j]);
#pragma unroll
            for (int j = 0; j < 6; ++j) vB[j] = LD(idE[3 + j]);
            int32_t idT[8];                     // T0..T3 X0 X2 X4 pad
            ld_ids(sid + SID_T0, idT);

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
            int32_t idO[12];                    // om3 om4 om5 oc0..oc5 x0[0..2]
            ld_ids(sid + SID_OM0 + 3, idO);
            int32_t idX[12];                    // x0[3..4] x1[0..4] x2[0..4]
            ld_ids(sid + SID_X0 + 3, idX);
            T rB[24];
            ld_coef(cf + SCF_RBF + 12, rB);
            T xrm[12], xro[12], xbl[12];
            ld_coef(cf + SCF_XRM, xrm);
            ld_coef(cf + SCF_XRO, xro);
            ld_coef(cf + SCF_XBL, xbl);
            C tBo[3], keX[3];
#pragma unroll
            for (int j = 0; j < 6; ++j) {
                const int32_t id_om = j < 3 ? idE[9 + j] : idO[j - 3];
                const int32_t id_oc = idO[3 + j];
                const C vM = LD(id_om), vO = LD(id_oc);
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
                    const int32_t* ex = x == 0 ? nullptr : idX + 2 + 5 * (x - 1);
                    const int32_t e_pm0 = x == 0 ? idO[9] : ex[0], e_pm1 = x == 0 ? idO[10] : ex[1];
                    const int32_t e_pcf = x == 0 ? idO[11] : ex[2];
                    const int32_t e_n1 = x == 0 ? idX[0] : ex[3], e_n2 = x == 0 ? idX[1] : ex[4];
                    const C pm0 = LD(e_pm0), pm1 = LD(e_pm1), pcf = LD(e_pcf), n1 = LD(e_n1), n2 = LD(e_n2);
                    const C tM = dot4(xrm + 4 * x, vB[j], vO, pm0, pm1);
                    const C tO = dot4(xro + 4 * x, vB[j], vM, n1, pcf);
                    const C kM = ke2(vM, tM), kO = ke2(vO, tO);
                    FORL keX[x].v[l] = xbl[3 * x] * kB.v[l] + xbl[3 * x + 1] * kM.v[l] + xbl[3 * x + 2] * kO.v[l];
                    FORL zc[x].v[l] += gx[6 * x + 1] * vO.v[l] + gx[6 * x + 2] * n1.v[l] + gx[6 * x + 3] * n2.v[l];
                    tBo[x] = tB;
                }
            }
            // ---- owned edges (S5-S7) -----------------------------------------------------------
            T ec[24];
            ld_coef(cf + SCF_EDGE, ec);
            C wf[4];
#pragma unroll
            for (int j = 0; j < 4; ++j) wf[j] = WF(idT[j]);
#pragma unroll
            for (int x = 0; x < 3; ++x) {       // interior: i0 (ab, ca), i1 (ab, bc), i2 (bc, ca); cells (T_x, T3)
                const C D = VD(vI[x]);
                const C& za = x == 2 ? zm[1] : zm[0];
                const C& zb = x == 0 ? zm[2] : x == 1 ? zm[1] : zm[2];
                const T* e4 = ec + 4 * x;
                C o;
                FORL {
                    const T H = (ke[3].v[l] - ke[x].v[l]) * e4[0] + tI[x].v[l] * (e4[1] + (za.v[l] + zb.v[l]));
                    const T V = (e4[2] * wf[x].v[l] + e4[3] * wf[3].v[l]) * D.v[l];
                    o.v[l] = -(H + V);
                }
                ST(idE[x], o);
            }
#pragma unroll
            for (int x = 0; x < 3; ++x) {       // boundary: b0 (a, ab), b2 (b, bc), b4 (c, ca); cells (T_x, X_2x)
                const C D = VD(vB[2 * x]);
                const C wx = WF(idT[4 + x]);
                const T* e4 = ec + 4 * (3 + x);
                C o;
                FORL {
                    const T H = (keX[x].v[l] - ke[x].v[l]) * e4[0] + tBo[x].v[l] * (e4[1] + (zm[x].v[l] + zc[x].v[l]));
                    const T V = (e4[2] * wf[x].v[l] + e4[3] * wx.v[l]) * D.v[l];
                    o.v[l] = -(H + V);
                }
                ST(idE[3 + 2 * x], o);
            }
        }
        __syncwarp();
    }
}

}  // namespace

template <class T>
int launch_tendencies_sc(const icon_grid& g, const DevScTables<T>& p, int nlev, int64_t ldk, int64_t ldk_w,
                         const T* abc, const T* vn, const T* w, T* ddt_vn, cudaStream_t s) {
    ScDev<T> d;
    d.ids = p.ids; d.coef = p.coef; d.n_patches = p.n_patches;
    const size_t smem = (size_t)kScWarps * 2 * sc_record_bytes<T>();
    const int64_t ctas = (p.n_patches + kScWarps - 1) / kScWarps;
    const int64_t grid = ctas < g.num_sms ? ctas : g.num_sms;
    const int n_chunks = (nlev + kChunk - 1) / kChunk;
    const int L = n_chunks == 1 ? 1 : (n_chunks == 2 || n_chunks == 4) ? 2 : 3;
    if (L == 1)
        k_tend_sc<T, 1><<<(unsigned)grid, kScThreads, smem, s>>>(d, nlev, (int)ldk, (int)ldk_w, abc, vn, w, ddt_vn);
    else if (L == 2)
        k_tend_sc<T, 2><<<(unsigned)grid, kScThreads, smem, s>>>(d, nlev, (int)ldk, (int)ldk_w, abc, vn, w, ddt_vn);
    else
        k_tend_sc<T, 3><<<(unsigned)grid, kScThreads, smem, s>>>(d, nlev, (int)ldk, (int)ldk_w, abc, vn, w, ddt_vn);
    cudaError_t err = cudaGetLastError();
    return err == cudaSuccess ? 1 : -(int)err;
}

template int launch_tendencies_sc<double>(const icon_grid&, const DevScTables<double>&, int, int64_t, int64_t,
                                          const double*, const double*, const double*, double*, cudaStream_t);
template int launch_tendencies_sc<float>(const icon_grid&, const DevScTables<float>&, int, int64_t, int64_t,
                                         const float*, const float*, const float*, float*, cudaStream_t);

}  // namespace icon
