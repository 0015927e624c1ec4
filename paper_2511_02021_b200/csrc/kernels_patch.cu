// kernels_patch.cu -- fused, register-resident tendency kernel for sm_100a.
//
// Work decomposition (patch_tables.hpp): TILE = 16 consecutive patches of the generation order =
// one CTA of 16 warps; PATCH = 4 sibling cells = one warp; the 32 lanes of the warp are 32
// consecutive levels of every column the patch touches, so every global access is one contiguous
// 256-byte (fp64) / 128-byte (fp32) line pair whatever the horizontal numbering is.
//
// Per level chunk a warp loads the 21 vn columns of its patch ONCE into registers and evaluates
// 9 tangential winds, 9 edge and 4 cell kinetic energies and 3 midpoint vorticities from them
// (3.5 column loads per owned edge instead of the ~50 of a per-edge gather). What a patch cannot
// know by itself -- KE and w of the cell across an owned boundary edge, vorticity at the three
// corner vertices -- is exchanged through shared memory: patches of the tile publish their cells,
// cells outside the tile and the corner vertices are evaluated by small halo tasks spread over the
// warps. One __syncthreads per level chunk (exchange buffers are double buffered). The CTA is
// persistent: it walks tiles blockIdx.x, +gridDim.x, ... and prefetches the next tile's tables with
// cp.async while it computes.
//
// No intermediate (vt, KE_e, KE_c, zeta) is written to HBM: the kernel reads vn, w and the tables
// and writes ddt_vn, which is the algorithmic traffic of SURVEY.md 8(d).
#include <cuda_pipeline.h>

#include "kernels.cuh"
#include "patch_tables.hpp"

namespace icon {
namespace {

constexpr int kNW = kPatchesPerTile;          // warps per CTA
constexpr int kThreads = kNW * 32;
constexpr int kCellSlots0 = 3 * kNW;          // exchange slots of the tile's own cells (T0..T2 of each patch)

template <class T>
struct SmemLayout {
    // per table buffer (two of them): patch coefficients, patch ids, halo + vertex task tables
    int max_halo, max_vert;
    __host__ __device__ size_t coef_bytes() const { return (size_t)kNW * kPatchCoefWords * sizeof(T); }
    __host__ __device__ size_t ids_bytes() const { return (size_t)kNW * kPatchIdWords * 4; }
    __host__ __device__ size_t hcoef_bytes() const { return (size_t)max_halo * kHaloCoefWords * sizeof(T); }
    __host__ __device__ size_t hids_bytes() const { return (size_t)max_halo * kHaloIdWords * 4; }
    __host__ __device__ size_t vcoef_bytes() const { return (size_t)max_vert * kVertCoefWords * sizeof(T); }
    __host__ __device__ size_t vids_bytes() const { return (size_t)max_vert * kVertIdWords * 4; }
    __host__ __device__ size_t table_bytes() const {
        return coef_bytes() + ids_bytes() + hcoef_bytes() + hids_bytes() + vcoef_bytes() + vids_bytes();
    }
    __host__ __device__ int cell_slots() const { return kCellSlots0 + max_halo; }
    __host__ __device__ size_t cell_bytes() const { return (size_t)cell_slots() * 2 * 32 * sizeof(T); }   // per buffer
    __host__ __device__ size_t vert_bytes() const { return (size_t)max_vert * 32 * sizeof(T); }           // per buffer
    __host__ __device__ size_t total() const { return 2 * table_bytes() + 2 * cell_bytes() + 2 * vert_bytes(); }
};

// 16-byte vector load of N coefficients (N * sizeof(T) a multiple of 16) from shared memory
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

__device__ __forceinline__ void cp_async16(void* smem, const void* gmem) {
    __pipeline_memcpy_async(smem, gmem, 16);
}

// cooperative asynchronous copy of `bytes` (multiple of 16, both sides 16-byte aligned)
__device__ __forceinline__ void stage_async(unsigned char* dst, const void* src, size_t bytes) {
    const unsigned char* s = static_cast<const unsigned char*>(src);
    for (size_t o = (size_t)threadIdx.x * 16; o < bytes; o += (size_t)kThreads * 16) cp_async16(dst + o, s + o);
}

template <class T>
struct PatchDev {
    const int32_t* patch_ids;
    const T* patch_coef;
    const int32_t* tile_hdr;
    const int32_t* halo_ids;
    const T* halo_coef;
    const int32_t* vert_ids;
    const T* vert_coef;
    int64_t n_patches, n_tiles;
    int max_halo, max_vert;
};

template <class T>
__device__ __forceinline__ void stage_tile_tables(const PatchDev<T>& d, const SmemLayout<T>& L, unsigned char* buf, int64_t tile) {
    const int64_t p0 = tile * kNW;
    const int np = (int)min((int64_t)kNW, d.n_patches - p0);
    const int32_t* h = d.tile_hdr + 4 * tile;
    const int halo_off = h[0], n_halo = h[1], vert_off = h[2], n_vert = h[3];
    unsigned char* o = buf;
    stage_async(o, d.patch_coef + p0 * kPatchCoefWords, (size_t)np * kPatchCoefWords * sizeof(T));
    o += L.coef_bytes();
    stage_async(o, d.patch_ids + p0 * kPatchIdWords, (size_t)np * kPatchIdWords * 4);
    o += L.ids_bytes();
    stage_async(o, d.halo_coef + (int64_t)halo_off * kHaloCoefWords, (size_t)n_halo * kHaloCoefWords * sizeof(T));
    o += L.hcoef_bytes();
    stage_async(o, d.halo_ids + (int64_t)halo_off * kHaloIdWords, (size_t)n_halo * kHaloIdWords * 4);
    o += L.hids_bytes();
    stage_async(o, d.vert_coef + (int64_t)vert_off * kVertCoefWords, (size_t)n_vert * kVertCoefWords * sizeof(T));
    o += L.vcoef_bytes();
    stage_async(o, d.vert_ids + (int64_t)vert_off * kVertIdWords, (size_t)n_vert * kVertIdWords * 4);
    __pipeline_commit();
}

// tangential wind of one edge from its four neighbours (S3)
template <class T>
__device__ __forceinline__ T vt4(const T* r, T a, T b, T c, T d) {
    return r[0] * a + r[1] * b + r[2] * c + r[3] * d;
}

template <class T>
__global__ void __launch_bounds__(kThreads, 1)
k_tend_patch(PatchDev<T> d, int nlev, int ldk, int ldk_w, const T* __restrict__ abc, const T* __restrict__ vn,
             const T* __restrict__ w, T* __restrict__ ddt_vn) {
    extern __shared__ __align__(16) unsigned char smem[];
    SmemLayout<T> L{d.max_halo, d.max_vert};
    const size_t tab_bytes = L.table_bytes();
    T* s_cell = reinterpret_cast<T*>(smem + 2 * L.table_bytes());
    T* s_vert = reinterpret_cast<T*>(smem + 2 * L.table_bytes() + 2 * L.cell_bytes());
    const int cell_stride = L.cell_slots() * 64;      // elements per exchange buffer
    const int vert_stride = d.max_vert * 32;

    const int warp = __shfl_sync(0xffffffffu, (int)(threadIdx.x >> 5), 0), lane = threadIdx.x & 31;      // warp-uniform for the compiler
    const int n_chunks = (nlev + 31) >> 5;
    const uint32_t cs = (uint32_t)ldk * (uint32_t)sizeof(T), cs_w = (uint32_t)ldk_w * (uint32_t)sizeof(T);   // column strides in bytes

    int64_t tile = blockIdx.x;
    if (tile >= d.n_tiles) return;
    stage_tile_tables(d, L, smem, tile);
    __pipeline_wait_prior(0);
    __syncthreads();

    int tb = 0;          // table buffer of the current tile
    unsigned xb = 0;     // exchange buffer parity, advances with every chunk
    for (; tile < d.n_tiles; tile += gridDim.x, tb ^= 1) {
        const int64_t next = tile + gridDim.x;
        const int np = (int)min((int64_t)kNW, d.n_patches - tile * kNW);
        const int32_t* hdr = d.tile_hdr + 4 * tile;
        const int n_halo = hdr[1], n_vert = hdr[3];
        const unsigned char* tbuf = smem + tb * tab_bytes;
        const T* s_coef = reinterpret_cast<const T*>(tbuf) + warp * kPatchCoefWords;
        const int32_t* s_ids = reinterpret_cast<const int32_t*>(tbuf + L.coef_bytes()) + warp * kPatchIdWords;
        const T* s_hcoef = reinterpret_cast<const T*>(tbuf + L.coef_bytes() + L.ids_bytes());
        const int32_t* s_hids = reinterpret_cast<const int32_t*>(tbuf + L.coef_bytes() + L.ids_bytes() + L.hcoef_bytes());
        const T* s_vcoef = reinterpret_cast<const T*>(tbuf + L.coef_bytes() + L.ids_bytes() + L.hcoef_bytes() + L.hids_bytes());
        const int32_t* s_vids = reinterpret_cast<const int32_t*>(tbuf + L.coef_bytes() + L.ids_bytes() + L.hcoef_bytes() +
                                                                 L.hids_bytes() + L.vcoef_bytes());

        // every thread is past the last barrier of the previous tile, and nothing after that barrier
        // reads the tables, so the other table buffer is free: prefetch the next tile's tables
        if (next < d.n_tiles) stage_tile_tables(d, L, smem + (tb ^ 1) * tab_bytes, next);

        for (int ch = 0; ch < n_chunks; ++ch, xb ^= 1) {
            const int k = (ch << 5) + lane;
            const bool active = k < nlev;
            const int kk = active ? k : nlev - 1;                 // clamped: padding lanes are never read
            const int km = kk > 0 ? kk - 1 : 0, kp = kk < nlev - 1 ? kk + 1 : nlev - 1;
            const unsigned char* vn_k = reinterpret_cast<const unsigned char*>(vn + kk);
            const unsigned char* w_k = reinterpret_cast<const unsigned char*>(w + kk);
            T* xc = s_cell + xb * cell_stride + lane;
            T* xv = s_vert + xb * vert_stride + lane;
            auto VN = [&](int32_t id) { return *reinterpret_cast<const T*>(vn_k + (uint64_t)(uint32_t)id * cs); };
            auto WF = [&](int32_t id) {
                const T* p = reinterpret_cast<const T*>(w_k + (uint64_t)(uint32_t)id * cs_w);
                return (T)0.5 * (p[0] + p[1]);
            };

            // ---- halo tasks: cells outside the tile, corner vertices -------------------------
            for (int task = warp; task < n_halo + n_vert; task += kNW) {
                if (task < n_halo) {
                    int32_t id[kHaloIdWords];
                    T cf[kHaloCoefWords];
                    ld_ids(s_hids + task * kHaloIdWords, id);
                    ld_coef(s_hcoef + task * kHaloCoefWords, cf);
                    const T e0 = VN(id[0]), e1 = VN(id[1]), e2 = VN(id[2]);
                    const T t0 = cf[0] * e1 + cf[1] * e2 + cf[2] * VN(id[3]) + cf[3] * VN(id[4]);
                    const T t1 = cf[4] * e2 + cf[5] * e0 + cf[6] * VN(id[5]) + cf[7] * VN(id[6]);
                    const T t2 = cf[8] * e0 + cf[9] * e1 + cf[10] * VN(id[7]) + cf[11] * VN(id[8]);
                    const T ke = (T)0.5 * (cf[12] * (e0 * e0 + t0 * t0) + cf[13] * (e1 * e1 + t1 * t1) + cf[14] * (e2 * e2 + t2 * t2));
                    xc[(kCellSlots0 + task) * 64] = ke;
                    xc[(kCellSlots0 + task) * 64 + 32] = WF(id[9]);
                } else {
                    const int v = task - n_halo;
                    int32_t id[kVertIdWords];
                    T cf[kVertCoefWords];
                    ld_ids(s_vids + v * kVertIdWords, id);
                    ld_coef(s_vcoef + v * kVertCoefWords, cf);
                    T z = cf[0] * VN(id[0]);
#pragma unroll
                    for (int q = 1; q < 6; ++q) z += cf[q] * VN(id[q]);
                    xv[v * 32] = z;
                }
            }

            // ---- phase A: the patch ----------------------------------------------------------
            T keL[3], q_part[3], hv[3], dH[3], sS[3];     // state of the owned boundary edges b0, b2, b4 carried over the barrier
            int32_t xslot[3], vslot[3], bid[3];
            if (warp < np) {
                int32_t id[kPatchIdWords];
                ld_ids(s_ids, id);
                T vI[3], vB[6], vM[6], vO[6];
#pragma unroll
                for (int j = 0; j < 3; ++j) vI[j] = VN(id[PID_I0 + j]);
#pragma unroll
                for (int j = 0; j < 6; ++j) {
                    vB[j] = VN(id[PID_B0 + j]);
                    vM[j] = VN(id[PID_OM0 + j]);
                    vO[j] = VN(id[PID_OC0 + j]);
                }
                T wf[4];
#pragma unroll
                for (int j = 0; j < 4; ++j) wf[j] = WF(id[PID_T0 + j]);

                T r[36];
                ld_coef(s_coef + PCF_RBF, r);
                T tI[3], tB[6];
                tI[0] = vt4(r + 0, vB[0], vB[5], vI[1], vI[2]);
                tI[1] = vt4(r + 4, vB[1], vB[2], vI[2], vI[0]);
                tI[2] = vt4(r + 8, vB[3], vB[4], vI[0], vI[1]);
                tB[0] = vt4(r + 12, vI[0], vB[5], vM[0], vO[0]);
                tB[1] = vt4(r + 16, vB[2], vI[1], vM[1], vO[1]);
                tB[2] = vt4(r + 20, vB[1], vI[1], vM[2], vO[2]);
                tB[3] = vt4(r + 24, vI[2], vB[4], vM[3], vO[3]);
                tB[4] = vt4(r + 28, vI[2], vB[3], vM[4], vO[4]);
                tB[5] = vt4(r + 32, vB[0], vI[0], vM[5], vO[5]);
                // 2*KE_e = vn^2 + vt^2 (S4); the factor 1/2 is applied once per cell (exact in binary)
                T kI[3], kB[6];
#pragma unroll
                for (int j = 0; j < 3; ++j) kI[j] = vI[j] * vI[j] + tI[j] * tI[j];
#pragma unroll
                for (int j = 0; j < 6; ++j) kB[j] = vB[j] * vB[j] + tB[j] * tB[j];
                T bl[12];
                ld_coef(s_coef + PCF_BLN, bl);
                T ke[4];
                ke[0] = (T)0.5 * (bl[0] * kB[0] + bl[1] * kI[0] + bl[2] * kB[5]);
                ke[1] = (T)0.5 * (bl[3] * kB[1] + bl[4] * kB[2] + bl[5] * kI[1]);
                ke[2] = (T)0.5 * (bl[6] * kI[2] + bl[7] * kB[3] + bl[8] * kB[4]);
                ke[3] = (T)0.5 * (bl[9] * kI[1] + bl[10] * kI[2] + bl[11] * kI[0]);
                // publish T0..T2 for the neighbouring patches
#pragma unroll
                for (int j = 0; j < 3; ++j) {
                    xc[(3 * warp + j) * 64] = ke[j];
                    xc[(3 * warp + j) * 64 + 32] = wf[j];
                }
                // midpoint vorticities (S2) and per-edge coefficients
                T g[44];
                ld_coef(s_coef + PCF_ROT, g);
                const T zab = g[0] * vB[0] + g[1] * vB[1] + g[2] * vI[0] + g[3] * vI[1] + g[4] * vM[0] + g[5] * vM[1];
                const T zbc = g[6] * vB[2] + g[7] * vB[3] + g[8] * vI[1] + g[9] * vI[2] + g[10] * vM[2] + g[11] * vM[3];
                const T zca = g[12] * vB[4] + g[13] * vB[5] + g[14] * vI[2] + g[15] * vI[0] + g[16] * vM[4] + g[17] * vM[5];
                const T* ec = g + (PCF_EDGE - PCF_ROT);      // [6][4]: s_inv_d, f, c_lin(L), c_lin(H)
                const T A = __ldg(abc + kk), B = __ldg(abc + nlev + kk), C = __ldg(abc + 2 * nlev + kk);
                auto VD = [&](int32_t e, T mid) {   // (vn_ie(k) - vn_ie(k+1)) / dz_k, reading P-14 folded into A, B, C
                    const T* col = reinterpret_cast<const T*>(reinterpret_cast<const unsigned char*>(vn) + (uint64_t)(uint32_t)e * cs);
                    return A * col[km] + B * mid + C * col[kp];
                };
                // interior edges: complete here (S5-S7)
                const T zm[3] = {(T)0.5 * (zab + zca), (T)0.5 * (zab + zbc), (T)0.5 * (zbc + zca)};
#pragma unroll
                for (int x = 0; x < 3; ++x) {
                    const int32_t e = id[PID_I0 + x];
                    const T D = VD(e, vI[x]);
                    const T H = (ke[3] - ke[x]) * ec[4 * x] + tI[x] * (ec[4 * x + 1] + zm[x]);
                    const T V = (ec[4 * x + 2] * wf[x] + ec[4 * x + 3] * wf[3]) * D;
                    if (active) ddt_vn[(uint64_t)(uint32_t)e * (uint32_t)ldk + k] = -(H + V);
                }
                // owned boundary edges b0 (T0, ab), b2 (T1, bc), b4 (T2, ca): everything local now, the rest after the barrier
                const T zmid[3] = {zab, zbc, zca};
#pragma unroll
                for (int x = 0; x < 3; ++x) {
                    const int32_t e = id[PID_B0 + 2 * x];
                    const T D = VD(e, vB[2 * x]);
                    const T* c4 = ec + 4 * (3 + x);
                    keL[x] = ke[x];
                    q_part[x] = tB[2 * x] * (c4[1] + (T)0.5 * zmid[x]) + (c4[2] * wf[x]) * D;
                    hv[x] = (T)0.5 * tB[2 * x];
                    dH[x] = c4[3] * D;
                    sS[x] = c4[0];
                    xslot[x] = id[PID_XSLOT + x];
                    vslot[x] = id[PID_VSLOT + x];
                    bid[x] = e;
                }
            }
            if (ch == n_chunks - 1 && next < d.n_tiles) __pipeline_wait_prior(0);   // next tile's tables have landed
            __syncthreads();

            // ---- phase B: owned boundary edges ------------------------------------------------
            if (warp < np) {
#pragma unroll
                for (int x = 0; x < 3; ++x) {
                    const T keX = xc[xslot[x] * 64], wfX = xc[xslot[x] * 64 + 32], zc = xv[vslot[x] * 32];
                    const T r = (keX - keL[x]) * sS[x] + q_part[x] + hv[x] * zc + dH[x] * wfX;
                    if (active) ddt_vn[(uint64_t)(uint32_t)bid[x] * (uint32_t)ldk + k] = -r;
                }
            }
        }
    }
}

}  // namespace

template <class T>
int launch_tendencies_patch(const icon_grid& g, const DevPatchTables<T>& p, int nlev, int64_t ldk, int64_t ldk_w,
                            const T* abc, const T* vn, const T* w, T* ddt_vn, cudaStream_t s) {
    PatchDev<T> d;
    d.patch_ids = p.patch_ids; d.patch_coef = p.patch_coef; d.tile_hdr = p.tile_hdr;
    d.halo_ids = p.halo_ids; d.halo_coef = p.halo_coef; d.vert_ids = p.vert_ids; d.vert_coef = p.vert_coef;
    d.n_patches = p.n_patches; d.n_tiles = p.n_tiles; d.max_halo = p.max_halo; d.max_vert = p.max_vert;
    SmemLayout<T> L{p.max_halo, p.max_vert};
    const size_t smem = L.total();
    if (smem > 227 * 1024) return -(int)cudaErrorInvalidValue;
    static thread_local size_t configured = 0;
    if (smem > configured) {
        cudaError_t e = cudaFuncSetAttribute(k_tend_patch<T>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (e != cudaSuccess) return -(int)e;
        configured = smem;
    }
    const int64_t grid = p.n_tiles < g.num_sms ? p.n_tiles : g.num_sms;
    k_tend_patch<T><<<(unsigned)grid, kThreads, smem, s>>>(d, nlev, (int)ldk, (int)ldk_w, abc, vn, w, ddt_vn);
    cudaError_t err = cudaGetLastError();
    return err == cudaSuccess ? 1 : -(int)err;
}

template int launch_tendencies_patch<double>(const icon_grid&, const DevPatchTables<double>&, int, int64_t, int64_t,
                                             const double*, const double*, const double*, double*, cudaStream_t);
template int launch_tendencies_patch<float>(const icon_grid&, const DevPatchTables<float>&, int, int64_t, int64_t,
                                            const float*, const float*, const float*, float*, cudaStream_t);

}  // namespace icon
