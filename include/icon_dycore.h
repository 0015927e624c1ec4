/*
 * icon_dycore.h -- C-ABI of the B200-native implementation of the velocity-tendency /
 * divergence / vorticity stencil sweep of ICON's non-hydrostatic dynamical core
 * (arxiv/paper_2511_02021; hot path named by BASELINE.json north_star; scope SURVEY.md 8).
 *
 * What the paper fixes: computations on an icosahedral-triangular C-grid (section 2)
 * and its dual of hexagons and 12 pentagons, reached through integer index arrays
 * (section 3.2); fields stay resident on the GPU for the whole run, no host copies
 * in the time loop (section 3.1); static coefficient + index tables are read-only
 * inputs of every stencil statement (the e_bln_c_s / ieidx excerpt); the
 * dynamical core is memory-bandwidth bound. Everything the paper leaves
 * open is fixed by the readings P-1..P-17 listed in DESIGN.md section 3.
 *
 * Conventions
 *   - Plain C types only. "dev" pointers are CUDA device pointers, "host" pointers are host memory.
 *   - Fields are level-contiguous: x[i*ldk + k], 0 <= k < nlev, k = 0 at the model top; i is the
 *     USER id of the cell / edge / vertex (the ids of the public tables). ldk >= nlev
 *     (ldk_w >= nlev+1 for w). Field pointers must be 16-byte aligned and ldk*sizeof(T) must be a
 *     multiple of 16. Padding lanes k >= nlev are never read for arithmetic and never written.
 *   - dtype ICON_F64: fields and coefficients are double. ICON_F32: fields are float and the
 *     coefficients are the fp64 ones rounded to float once (reading P-17).
 *   - Every call returns ICON_OK or a negative error code; no exceptions, no abort, no output to
 *     stdout/stderr. icon_last_error() returns a thread-local message for the last failure.
 *   - Compute calls enqueue kernels on the caller's CUDA stream and return without synchronising.
 *     Field buffers are caller-owned, never retained; outputs must not alias inputs.
 *   - There is NO CPU fallback: compute calls return ICON_ECUDA when no CUDA device is usable.
 *   - Device, stream and thread contract. A grid handle belongs to the CUDA device that was current at
 *     icon_grid_create; every later call on it must be made with that device current (ICON_EINVAL otherwise).
 *     The handle is logically const for the compute calls but caches tables and schedules that are built on the
 *     first call for a new (dtype, nlev, ldk, ldk_w, z_half): such a first call allocates device memory and
 *     synchronises; steady-state calls do neither and can be captured into a CUDA graph (capture after one
 *     plain call with the same arguments). Calls on ONE handle must not overlap: use one stream at a time and one
 *     host thread at a time per handle (the fused kernel keeps a chip-wide pacing counter per handle, the
 *     unfused pipeline a workspace). Different handles are independent.
 */
#ifndef ICON_DYCORE_H
#define ICON_DYCORE_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct icon_grid icon_grid_t;   /* opaque; owns host and device copies of all tables */

enum { ICON_OK = 0, ICON_EINVAL = -1, ICON_ENOMEM = -2, ICON_ECUDA = -3, ICON_EUNSUPPORTED = -4 };
enum { ICON_F64 = 0, ICON_F32 = 1 };
/* element types reported by icon_grid_table_host */
enum { ICON_T_I32 = 10, ICON_T_I8 = 11, ICON_T_F64 = 12, ICON_T_F32 = 13, ICON_T_I64 = 14 };

/* icon_grid_create flags */
enum {
    ICON_PERMUTE = 1u,            /* seeded random renumbering of cells/edges/vertices (P-7, config 4) */
    ICON_LOCALITY_WORKLIST = 2u,  /* internal tables laid out in generation (spatially local) order and
                                     kernels walk that order; results are identical. Implied by
                                     ICON_PERMUTE unless ICON_NO_WORKLIST is given (accepted, has no further effect). */
    ICON_HOST_ONLY = 4u,          /* build host tables only; no CUDA device is touched (table tests) */
    ICON_NO_WORKLIST = 8u         /* with ICON_PERMUTE: walk the permuted ids directly (ablation) */
};

/* table selectors for icon_grid_table_host / icon_grid_table_device */
enum {
    ICON_TAB_C2V = 0,      /* int32 [nc][3] vertices of a cell, counter-clockwise (P-2, P-3) */
    ICON_TAB_C2E,          /* int32 [nc][3] edge j joins vertex slots j and j+1 (P-3) */
    ICON_TAB_E2C,          /* int32 [ne][2] first-touch cell, second-touch cell (P-3) */
    ICON_TAB_E2V,          /* int32 [ne][2] direction of the edge (P-3, P-4) */
    ICON_TAB_E2E4,         /* int32 [ne][4] the four other edges of the two adjacent cells (P-6) */
    ICON_TAB_V2E,          /* int32 [nv][6] fan edges counter-clockwise; pentagon slot 5 = slot 0 (P-5) */
    ICON_TAB_V2C,          /* int32 [nv][6] fan cells; cell i lies between fan edges i and i+1 (P-5) */
    ICON_TAB_V_DEG,        /* int32 [nv]    5 or 6 (exactly 12 fives) */
    ICON_TAB_C_OS,         /* int8  [nc][3] +1 if the cell is e2c[.][0] of that edge else -1 (P-4) */
    ICON_TAB_V_OS,         /* int8  [nv][6] -1 if v == e2v[.][0] else +1; 0 in the pentagon pad (P-5) */
    ICON_TAB_VERT_XYZ,     /* f64 [nv][3] unit sphere */
    ICON_TAB_CELL_XYZ,     /* f64 [nc][3] spherical circumcentres (P-8) */
    ICON_TAB_EDGE_XYZ,     /* f64 [ne][3] edge midpoints x_e (P-4) */
    ICON_TAB_EDGE_NORMAL,  /* f64 [ne][3] n_e = tau_e x x_e, from e2c[.][0] to e2c[.][1] (P-4) */
    ICON_TAB_L_E,          /* f64 [ne] primal edge length, m */
    ICON_TAB_D_E,          /* f64 [ne] dual edge length, m */
    ICON_TAB_INV_D_E,      /* f64 [ne] 1/d_e */
    ICON_TAB_F_E,          /* f64 [ne] Coriolis parameter 2*Omega*z(x_e) */
    ICON_TAB_C_LIN,        /* f64 [ne][2] cell-to-edge linear weights (P-9) */
    ICON_TAB_RBF,          /* f64 [ne][4] tangential-wind reconstruction weights (P-11) */
    ICON_TAB_A_C,          /* f64 [nc] cell area, m^2 */
    ICON_TAB_BLN,          /* f64 [nc][3] edge-to-cell weights, the paper's e_bln_c_s (P-10) */
    ICON_TAB_A_V,          /* f64 [nv] dual-cell area, m^2 */
    ICON_TAB_GEOFAC_DIV,   /* f64 [nc][3] l_e*c_os/A_c */
    ICON_TAB_GEOFAC_ROT,   /* f64 [nv][6] d_e*v_os/A_v, 0 in the pentagon pad */
    ICON_TAB_ADV_C,        /* f64 [nc][3] normal-component reconstruction weights of the vertical-wind tendency:
                              sum_j adv_c(c,j) n_j n_j^T = I in the tangent plane of the cell (P-19) */
    ICON_TAB_CGRAD,        /* f64 [ne][2] distance-weighted KE-gradient coefficients (a1/a0)/d_e, (a0/a1)/d_e (P-20) */
    ICON_TAB_COUNT
};

/* runtime options (icon_grid_set_option); the defaults are the measured optimum on B200 */
enum {
    ICON_OPT_TENDENCY_KERNEL = 0, /* 0 = unfused 3-kernel pipeline through an HBM workspace (also serves the optional
                                         outputs vt_opt / ke_c_opt / vort_opt, whatever this option says);
                                     3 = self-contained patch kernel (one warp per patch, columns through L1; any nlev);
                                     4 = column-cache kernel: whole columns staged in shared memory by bulk
                                         asynchronous copies on a host-built schedule; level counts it cannot
                                         hold (nlev > 95) fall back to 3;
                                     5 = auto (default) = 4 wherever it can hold the columns. */
    ICON_OPT_CC_TILE = 1,         /* kernel 4: patches per tile of the round-robin work order (CTA b walks the tiles
                                     b, b + #CTAs, ... so that neighbouring tiles are in flight together and share
                                     their halo columns through the L2); a multiple of 8; 0 = one contiguous range per
                                     CTA; -1 = auto (default): 16 for deep 8-byte columns, 64 for short or 4-byte ones. */
    ICON_OPT_CC_PACE = 2,         /* kernel 4: the producers of all CTAs meet every this many steps (power of two; bounded
                                     wait) so that the CTAs do not drift rounds apart and neighbouring tiles keep sharing
                                     halo columns through the L2; 0 = never. Default 512; fused fp64 step (dycore_step) only. */
    ICON_OPT_COUNT
};

/*
 * icon_grid_create -- SURVEY.md 8(a) rows G1-G3; readings P-1..P-11.
 * Builds the R2Bk grid (k+1 bisections of the unit icosahedron, 0 <= k <= 9), its canonical
 * first-touch numbering, all index tables, geometry and coefficients on the host, optionally
 * renumbers cells/edges/vertices by the seeded permutation (ICON_PERMUTE; seed is ignored
 * otherwise), and uploads the tables the kernels need to the current CUDA device (unless
 * ICON_HOST_ONLY). Not part of any timed region (the paper excludes initialisation).
 * *out is owned by the caller until icon_grid_destroy. Errors: ICON_EINVAL (k, flags, out),
 * ICON_ENOMEM, ICON_ECUDA (no device / upload failed).
 */
int icon_grid_create(int bisections_k, uint64_t seed, unsigned flags, icon_grid_t** out);
void icon_grid_destroy(icon_grid_t* g);

/* nc = 20*4^(k+1), ne = 3nc/2, nv = nc/2+2. Any output pointer may be NULL. */
int icon_grid_counts(const icon_grid_t* g, int64_t* nc, int64_t* ne, int64_t* nv);

/* Host view of a public table (user ids). *ptr stays valid until icon_grid_destroy and must not
 * be written. dtype receives ICON_T_*. */
int icon_grid_table_host(const icon_grid_t* g, int which, const void** ptr, int* dtype, int64_t* rows, int* cols);

/* Device copy of a public table in user order, uploaded on first request and then cached.
 * dtype: ICON_F64 or ICON_F32 selects the element type of floating-point tables (ignored for
 * integer tables). ICON_EUNSUPPORTED on a ICON_HOST_ONLY grid. */
int icon_grid_table_device(const icon_grid_t* g, int which, int dtype, const void** dptr);

int icon_grid_set_option(icon_grid_t* g, int option, int value);

/*
 * icon_grid_cc_schedule_check -- builds on the host (works on ICON_HOST_ONLY grids) the column-cache
 * schedule tendency kernel 4 would run for (dtype, nlev, ldk, ldk_w) with the current ICON_OPT_CC_*
 * options on a device with `n_ctas` SMs and `smem_bytes` of opt-in shared memory per block, replays it
 * with an independent checker (every patch finds each of its 43 columns in the slot its record names;
 * no bulk copy overwrites a slot a running step still reads or a copy still in flight fills; byte counts match) and reports
 *   out[0] steps   out[1] steps with reduced run-ahead   out[2] vn columns loaded   out[3] w columns loaded
 *   out[4] bulk copies   out[5] slots   out[6] slot bytes   out[7] CTAs.
 * ICON_EUNSUPPORTED: nlev or the memory size cannot hold the kernel; ICON_EINVAL: the check failed
 * (icon_last_error names the rule).
 */
int icon_grid_cc_schedule_check(const icon_grid_t* g, int dtype, int nlev, int ldk, int ldk_w, int n_ctas, int smem_bytes,
                                int64_t out[8]);

/*
 * dycore_div_vort -- SURVEY.md 8(a) steps S1, S2 (north_star: "cell divergence from normal winds
 * (c2e gather with edge lengths, orientation signs and cell areas), relative vorticity at vertices
 * (v2e gather with dual lengths and dual areas)").
 *   div(c,k)  = sum_{j<3} geofac_div(c,j) * vn(c2e[c][j], k)
 *   vort(v,k) = sum_{j<6} geofac_rot(v,j) * vn(v2e[v][j], k)      (pentagon pad coefficient is 0)
 * vn [ne][ldk] dev in; div [nc][ldk], vort [nv][ldk] dev out. 1 <= nlev <= ldk.
 */
int dycore_div_vort(const icon_grid_t* g, int dtype, int nlev, int ldk,
                    const void* vn, void* div, void* vort, void* cuda_stream);

/*
 * dycore_velocity_tendencies -- SURVEY.md 8(a) steps S3-S7 (north_star: "tangential wind by RBF
 * reconstruction from the 4 neighbouring edges (e2e4 table), kinetic energy at edges and cells, and
 * the normal-wind tendency ddt_vn = -(dKE/dn + (zeta+f)*vt + w*dvn/dz), with w on nlev+1 half
 * levels"; the edge->cell kinetic-energy interpolation is PAPER.md:164-167).
 *   vt(e,k)   = sum_{j<4} rbf(e,j) * vn(e2e4[e][j], k)
 *   KE_e      = 1/2 (vn^2 + vt^2);  KE_c(c,k) = sum_{j<3} bln(c,j) * KE_e(c2e[c][j], k)
 *   ddt_vn    = -[ (KE_c(c1)-KE_c(c0)) / d_e + vt * (f_e + 1/2(zeta(v0)+zeta(v1)))
 *                  + w_e * (vn_ie(k) - vn_ie(k+1)) / dz_k ]
 *   w_e = c_lin(e,0) w_f(c0,k) + c_lin(e,1) w_f(c1,k), w_f(c,k) = 1/2 (w(c,k)+w(c,k+1)),
 *   vn_ie = vn interpolated linearly in z to half levels, linear extrapolation at k=0 and k=nlev (P-14).
 * z_half [nlev+1] HOST, strictly decreasing (read during the call, not retained).
 * vn [ne][ldk], w [nc][ldk_w] dev in; ddt_vn [ne][ldk] dev out.
 * vt_opt [ne][ldk], ke_c_opt [nc][ldk], vort_opt [nv][ldk]: dev out, NULL = do not store.
 * 2 <= nlev <= ldk, nlev+1 <= ldk_w, nlev <= 4096.
 */
int dycore_velocity_tendencies(const icon_grid_t* g, int dtype, int nlev, int ldk, int ldk_w,
                               const double* z_half,
                               const void* vn, const void* w, void* ddt_vn,
                               void* vt_opt, void* ke_c_opt, void* vort_opt, void* cuda_stream);

/*
 * dycore_w_tendency -- SURVEY.md 8(f) NEXT-2: the vertical-wind tendency, the other half of the velocity-tendency
 * routine of the dynamical core (PAPER.md:142 names the dycore; the paper prints none of its vertical-wind statements,
 * reading P-19 of DESIGN.md section 3). w and ddt_w live at cells on the nlev+1 half levels, k = 0 at the top:
 *   k = 1 .. nlev-1:  ddt_w(c,k) = -[ sum_{j<3} adv_c(c,j) * vn_ie(e_j,k) * (w(c1(e_j),k) - w(c0(e_j),k)) / d_e(e_j)
 *                                     + w(c,k) * (w(c,k-1) - w(c,k+1)) / (z_half[k-1] - z_half[k+1]) ],  e_j = c2e[c][j],
 *   k = 0 and k = nlev: ddt_w = 0 (the top and surface values of w are boundary conditions).
 * vn_ie = vn interpolated linearly in z to the half level (P-14). z_half [nlev+1] HOST, strictly decreasing.
 * vn [ne][ldk], w [nc][ldk_w] dev in; ddt_w [nc][ldk_w] dev out (levels 0 .. nlev written, pads untouched).
 * 2 <= nlev <= ldk, nlev+1 <= ldk_w. One kernel: the column cache in its ddt_w mode (nine vn and ten w columns per
 * patch) where it holds the columns, else (ICON_OPT_TENDENCY_KERNEL 0 / 3, deeper columns) a gather kernel through L1.
 */
int dycore_w_tendency(const icon_grid_t* g, int dtype, int nlev, int ldk, int ldk_w, const double* z_half,
                      const void* vn, const void* w, void* ddt_w, void* cuda_stream);

/*
 * dycore_metric_from_zhalf -- SURVEY.md 8(f) NEXT-1, set-up of the metric variant (reading P-20; PAPER.md:56 names the
 * "terrain following hybrid sigma height grid", the paper prints no formula): from the half-level heights of every EDGE
 * column, z_half_e [ne][ldk_w] dev in (strictly decreasing in k, levels 0 .. nlev), derives
 *   wgt_e      [ne][ldk_w] dev out: k = 1 .. nlev-1 the weight of vn(k) in vn_ie(k), dz(k-1) / (dz(k-1) + dz(k));
 *                                   k = 0, k = nlev the linear-extrapolation ratios dz0/(dz0+dz1), dz(K-1)/(dz(K-1)+dz(K-2))
 *   inv_ddqz_e [ne][ldk]   dev out: 1 / dz(k), dz(k) = z_half_e(k) - z_half_e(k+1).
 * Static in a model run: not part of any timed region. 3 <= nlev <= ldk, nlev+1 <= ldk_w; pads untouched.
 */
int dycore_metric_from_zhalf(const icon_grid_t* g, int dtype, int nlev, int ldk, int ldk_w, const void* z_half_e,
                             void* wgt_e, void* inv_ddqz_e, void* cuda_stream);

/*
 * dycore_velocity_tendencies_metric -- SURVEY.md 8(f) NEXT-1: S3-S7 in their ICON-faithful metric form (reading P-20).
 * S3, S4, S2 as in dycore_velocity_tendencies (along the coordinate surfaces), then
 *   gradK  = cgrad(e,1) KE_c(c1) - cgrad(e,0) KE_c(c0) + KE_e(e) (cgrad(e,0) - cgrad(e,1))        (ICON_TAB_CGRAD)
 *   vn_ie  = per-edge weights: k = 1..nlev-1: wgt_e vn(k) + (1 - wgt_e) vn(k-1); ends: vn(0) + wgt_e(0) (vn(0) - vn(1)),
 *            vn(nlev-1) + wgt_e(nlev) (vn(nlev-1) - vn(nlev-2))
 *   ddt_vn = -[ gradK + vt (f_e + 1/2(zeta(v0)+zeta(v1)))
 *               + (w_e - vn ddxn_z - vt ddxt_z) (vn_ie(k) - vn_ie(k+1)) inv_ddqz_e ],   w_e as in S6.
 * wgt_e [ne][ldk_w], inv_ddqz_e, ddxn_z, ddxt_z [ne][ldk] dev in (ddxn_z, ddxt_z = slopes dz/dn, dz/dt of the full-level
 * coordinate surface at the edge midpoint, t = n x x_e); vn [ne][ldk], w [nc][ldk_w] dev in; ddt_vn [ne][ldk] dev out.
 * One fused column-cache kernel where it holds the columns (nlev <= 95; the metric columns of an owned edge are read
 * straight from global memory, each exactly once), else the unfused pipeline. 3 <= nlev <= ldk, nlev+1 <= ldk_w.
 */
int dycore_velocity_tendencies_metric(const icon_grid_t* g, int dtype, int nlev, int ldk, int ldk_w,
                                      const void* wgt_e, const void* inv_ddqz_e, const void* ddxn_z, const void* ddxt_z,
                                      const void* vn, const void* w, void* ddt_vn, void* cuda_stream);

/*
 * dycore_step -- one pass of the whole hot path: the outputs of
 * dycore_velocity_tendencies (ddt_vn) and of dycore_div_vort (div, vort) for the same vn, w. Where the
 * column-cache tendency kernel runs (ICON_OPT_TENDENCY_KERNEL 4, or 5 = auto in its regime) all three come
 * out of ONE kernel that reads vn once: div of a patch's four cells and the vorticity at its three midpoint
 * and three corner vertices are by-products of columns and sums the tendency needs anyway (every vertex of
 * the grid is a midpoint or corner of some patch; the lowest patch index stores it). Elsewhere it is the two
 * calls back to back. Same argument rules as the two calls; outputs must not alias inputs or each other.
 */
int dycore_step(const icon_grid_t* g, int dtype, int nlev, int ldk, int ldk_w, const double* z_half,
                const void* vn, const void* w, void* ddt_vn, void* div, void* vort, void* cuda_stream);

/*
 * dycore_step_w -- dycore_step plus the vertical-wind tendency of dycore_w_tendency from the SAME pass: where the
 * column-cache kernel runs, ddt_w of a patch's four cells is a by-product of the nine vn columns the patch holds in
 * registers anyway and ten w columns (seven of them already in the column cache for ddt_vn): one kernel writes all four
 * outputs. Elsewhere it is dycore_step followed by dycore_w_tendency. Argument rules of both.
 */
int dycore_step_w(const icon_grid_t* g, int dtype, int nlev, int ldk, int ldk_w, const double* z_half,
                  const void* vn, const void* w, void* ddt_vn, void* div, void* vort, void* ddt_w, void* cuda_stream);

/*
 * dycore_velocity_tendencies_noalloc -- dycore_velocity_tendencies (S3-S7, same formulas, same argument rules, no optional
 * outputs) for callers that cannot call cudaMalloc: code under CUDA-graph capture, tight serving loops, harnesses that forbid
 * it. The ordinary entry points allocate lazily on their first call for a new (dtype, nlev, ldk, z_half); this one calls no
 * cudaMalloc, cudaFree or allocating library routine, ever, and touches no host heap. It runs the unfused pipeline
 * (vt, KE_e -> KE_c, zeta -> ddt_vn) with its intermediates in a STATIC device array of ICON_NOALLOC_SCRATCH_BYTES that
 * every GPU that loads the library holds until the process exits.
 *   Limits: nlev <= 128 and align256(3*nlev*g) + 2*align256(ne*ldk*g) + align256(nc*ldk*g) + align256(nv*ldk*g) <=
 *   ICON_NOALLOC_SCRATCH_BYTES, g = sizeof(T) (64 MiB: R2B4 x 90 fp64 levels with ldk = 90, R2B3 with any padding);
 *   beyond that ICON_EINVAL with the two byte counts in icon_last_error(). ICON_F32 needs the fp32 coefficient tables
 *   already on the device (one ordinary fp32 compute call on the grid), else ICON_EUNSUPPORTED; ICON_F64 tables are
 *   uploaded by icon_grid_create.
 *   Sharing: every call on a device uses the same array, which keeps the previous call's contents. Nothing in it has to
 *   start at zero (the pipeline writes every level it later reads), so nothing is cleared. Calls that overlap on the GPU
 *   (two streams, two threads, two grids on one device) RACE on it: serialise them. The first call on a device resolves
 *   the array's device address (cudaGetSymbolAddress, which may load the module): make it outside stream capture.
 * This is the slow path (intermediates through HBM: about 3x the time of the column-cache kernel); it exists for the
 * callers above, not for throughput.
 */
#define ICON_NOALLOC_SCRATCH_BYTES (64u << 20)
int dycore_velocity_tendencies_noalloc(const icon_grid_t* g, int dtype, int nlev, int ldk, int ldk_w,
                                       const double* z_half, const void* vn, const void* w, void* ddt_vn,
                                       void* cuda_stream);

/*
 * dycore_step_host -- the step with HOST field buffers (the end-to-end leg of bench.py): copies vn and w to device staging
 * buffers, computes ddt_vn, div and vort, copies them back, and synchronises. The copies are the cost (22 GB per step at
 * R2B8 x 90 fp64), so the call runs the two entry points instead of the fused one and overlaps them with the link in both
 * directions: vn goes up first, dycore_div_vort (which reads nothing else) runs as soon as it has arrived and div / vort go
 * down while w is still going up; then dycore_velocity_tendencies, then ddt_vn down. This is NOT how the paper runs the
 * model (fields stay resident on the GPU); it exists so that the whole path can be timed with the PCIe copies
 * included. Host buffers should be pinned for full PCIe bandwidth. The staging buffers, three private streams and their
 * events are owned by the grid handle and allocated on first use. Same shapes and constraints as dycore_step.
 */
int dycore_step_host(const icon_grid_t* g, int dtype, int nlev, int ldk, int ldk_w, const double* z_half,
                     const void* vn_host, const void* w_host,
                     void* ddt_vn_host, void* div_host, void* vort_host);

/*
 * ---- horizontal domain decomposition (reading P-21 in DESIGN.md section 3) ----
 * The paper runs the model on subdomains of the horizontal grid that exchange halos point to point.
 * Rank `part` of `n_parts` owns the parent triangles floor(part P / n_parts) <= q < floor((part+1) P / n_parts) of the
 * hierarchical numbering, P = nc / 4 (cells 4q .. 4q+3); an edge or vertex shared by two ranks is owned by the rank whose
 * patch stores it, so every output point of the grid has exactly one owner.
 *
 * icon_grid_create_part -- the LOCAL grid of one rank. Flags: 0 or ICON_HOST_ONLY (a decomposed grid is never
 * permuted). Its counts (icon_grid_counts) are LOCAL: ne = owned + halo edges, nc = owned + halo cells, nv = owned
 * vertices. Local rows: [0, n_owned) the owned points in ascending global id, then the halo, grouped by owner rank
 * ascending and by global id within a rank, so what one peer sends is ONE contiguous block of rows.
 * Fields passed to the compute calls are local: vn [ne][ldk], w [nc][ldk_w] with their halo rows filled (dycore_halo_pack
 * on the owner, any transport, receive in place), outputs ddt_vn [ne][ldk] (rows < ne_owned written), div [nc][ldk]
 * (rows < nc_owned written), vort [nv][ldk]. On a local grid the calls served by the column-cache kernel work
 * (dycore_step, dycore_step_w, dycore_velocity_tendencies without optional outputs, dycore_div_vort, dycore_w_tendency,
 * dycore_velocity_tendencies_metric; nlev <= 95 for 8-byte, 127 for 4-byte columns); every other call and every global
 * table selector returns ICON_EUNSUPPORTED. Host memory: the call builds the GLOBAL grid once and drops it.
 * Errors: ICON_EINVAL (k, flags, n_parts < 1 or > nc/4, part), ICON_ENOMEM, ICON_ECUDA.
 */
int icon_grid_create_part(int bisections_k, unsigned flags, int n_parts, int part, icon_grid_t** out);

/* icon_part_info -- out[0] n_parts (0: not a local grid), [1] part, [2] nc_owned, [3] ne_owned, [4] nv_owned, [5] nc_local,
 * [6] ne_local, [7] nc_global, [8] ne_global, [9] nv_global, [10] first owned parent, [11] one past the last. */
int icon_part_info(const icon_grid_t* g, int64_t out[12]);

/* icon_part_table -- host pointers into the handle (valid until destroy). */
enum {
    ICON_PART_L2G_CELL = 0,    /* int32 [nc]  global id of local cell row */
    ICON_PART_L2G_EDGE,        /* int32 [ne] */
    ICON_PART_L2G_VERT,        /* int32 [nv] */
    ICON_PART_RECV_BEGIN_EDGE, /* int64 [n_parts+1] rows [b[q], b[q+1]) of a local edge field are owned by rank q */
    ICON_PART_RECV_BEGIN_CELL, /* int64 [n_parts+1] the same for cell fields */
    ICON_PART_SEND_BEGIN_EDGE, /* int64 [n_parts+1] rows [b[q], b[q+1]) of the packed buffer go to rank q */
    ICON_PART_SEND_BEGIN_CELL,
    ICON_PART_SEND_IDS_EDGE,   /* int32 [b[n_parts]] local (owned) row packed at each position, the receiver's order */
    ICON_PART_SEND_IDS_CELL,
    ICON_PART_COUNT
};
int icon_part_table(const icon_grid_t* g, int which, const void** ptr, int* dtype, int64_t* count);

/*
 * dycore_halo_pack -- the send side of the exchange: gathers whole rows of a local field into one contiguous buffer,
 *   send_buf[i][0..ld) = field[send_ids[i]][0..ld),   i < send_begin[n_parts]
 * kind 0 = edge field (vn), 1 = cell field (w); ld = row stride in elements, ld*sizeof(T) a multiple of 16; field and
 * send_buf dev, not overlapping. Rows [send_begin[q], send_begin[q+1]) of send_buf are what rank q receives into rows
 * [recv_begin[part], recv_begin[part+1]) of ITS local field: with an all-to-all of those splits (NCCL grouped send / recv
 * over NVLink) the receive lands in place and nothing is unpacked. One kernel launch, asynchronous on cuda_stream.
 */
int dycore_halo_pack(const icon_grid_t* g, int dtype, int kind, int ld, const void* field, void* send_buf,
                     void* cuda_stream);

/* number of kernels the library has launched through this handle since creation */
int64_t icon_grid_launch_count(const icon_grid_t* g);

const char* icon_last_error(void);

#ifdef __cplusplus
}
#endif
#endif /* ICON_DYCORE_H */
