"""Seeded synthetic inputs shared by the tests, bench.py and smoke().

This module holds NONE of the method's arithmetic: it only draws the prognostic fields
(vn, w) and the level heights that both the oracle and the CUDA library receive as inputs.
It imports neither ``oracle`` nor ``paper_2511_02021_b200``; the geometry it needs (edge
midpoints and normals on the unit sphere) is passed in as plain arrays by the caller.

The fields stand in for the paper's global km-scale atmosphere state (a reanalysis
interpolated to the grid), which is not available; shapes follow Table 2
(90 levels, R2B8 = the 10 km grid). Recipe: DESIGN.md section 4 /
SURVEY.md section 8(d).
"""
import numpy as np

U0 = 20.0            # m/s, solid-body rotation about the z axis
H_TOP = 30.0e3       # m
CONFIGS = {
    # id: (R2Bk, nlev, dtype, permuted, jet)
    1: dict(k=4, nlev=90, dtype="f64", permute=False, jet=False),
    2: dict(k=6, nlev=90, dtype="f64", permute=False, jet=False),
    3: dict(k=8, nlev=90, dtype="f64", permute=False, jet=False),
    4: dict(k=8, nlev=90, dtype="f32", permute=True, jet=False),
    5: dict(k=9, nlev=30, dtype="f64", permute=False, jet=True),
}
PERMUTE_SEED = 4     # config 4: ICON_PERMUTE with seed 4


def z_half_levels(nlev, h_top=H_TOP):
    """Flat stretched half-level heights, strictly decreasing, k=0 at the top:
    z_half[k] = H (0.06 eta + 0.94 eta^3), eta = (K-k)/K."""
    eta = (nlev - np.arange(nlev + 1, dtype=np.float64)) / nlev
    return h_top * (0.06 * eta + 0.94 * eta ** 3)


def _fill_normal(rng, out, scale, chunk_rows=1 << 16):
    """out[:, :] = scale * N(0,1), drawn row-chunk by row-chunk (bounded temporaries)."""
    n, m = out.shape
    for r0 in range(0, n, chunk_rows):
        r1 = min(n, r0 + chunk_rows)
        blk = rng.standard_normal((r1 - r0, m))
        if scale != 1.0:
            blk *= scale
        out[r0:r1, :] = blk


def solid_body_vn(edge_xyz, edge_normal, u0=U0):
    """(u0 * z_hat x x_e) . n_e  == u0 cos(lat) (east . n_e)"""
    vx = -edge_xyz[:, 1]
    vy = edge_xyz[:, 0]
    return u0 * (vx * edge_normal[:, 0] + vy * edge_normal[:, 1])


def galewsky_jet_vn(edge_xyz, edge_normal, u_max=80.0):
    """Compactly supported mid-latitude zonal jet (Galewsky form) with a localised
    multiplicative perturbation, projected on n_e. Constants are the harness's own."""
    lat = np.arcsin(np.clip(edge_xyz[:, 2], -1.0, 1.0))
    lon = np.arctan2(edge_xyz[:, 1], edge_xyz[:, 0])
    phi0, phi1 = np.pi / 7.0, np.pi / 2.0 - np.pi / 7.0
    e_n = np.exp(-4.0 / (phi1 - phi0) ** 2)
    inside = (lat > phi0) & (lat < phi1)
    u = np.zeros_like(lat)
    li = lat[inside]
    u[inside] = (u_max / e_n) * np.exp(1.0 / ((li - phi0) * (li - phi1)))
    alpha, beta, phi2 = 1.0 / 3.0, 1.0 / 15.0, np.pi / 4.0
    u *= 1.0 + 0.01 * np.cos(lat) * np.exp(-(lon / alpha) ** 2) * np.exp(-((phi2 - lat) / beta) ** 2)
    coslat = np.maximum(np.cos(lat), 1e-300)
    east_dot_n = (-edge_xyz[:, 1] * edge_normal[:, 0] + edge_xyz[:, 0] * edge_normal[:, 1]) / coslat
    return u * east_dot_n


def make_fields(config, edge_xyz, edge_normal, nc, nlev=None, ldk=None, ldk_w=None, dtype=None, jet=None,
                pad_value=np.nan):
    """Draw (vn [ne][ldk], w [nc][ldk_w], z_half [nlev+1]) for a BASELINE.json config id.

    vn(e,k) = solid body (u0 = 20 m/s) + N(0, 1 m/s), seed 1000+config;
    w(c,k)  = N(0, 0.1 m/s) on nlev+1 half levels, seed 2000+config.
    dtype 'f32' rounds the values to fp32 (arrays are returned as float32).
    Padding lanes k >= nlev (k >= nlev+1 for w) hold ``pad_value``.
    """
    cfg = CONFIGS[config]
    nlev = cfg["nlev"] if nlev is None else nlev
    dtype = cfg["dtype"] if dtype is None else dtype
    jet = cfg["jet"] if jet is None else jet
    ldk = nlev if ldk is None else ldk
    ldk_w = nlev + 1 if ldk_w is None else ldk_w
    ne = edge_xyz.shape[0]
    vn = np.empty((ne, ldk), dtype=np.float64)
    _fill_normal(np.random.Generator(np.random.PCG64(1000 + config)), vn[:, :nlev], 1.0)
    base = solid_body_vn(edge_xyz, edge_normal)
    if jet:
        base = base + galewsky_jet_vn(edge_xyz, edge_normal)
    vn[:, :nlev] += base[:, None]
    w = np.empty((nc, ldk_w), dtype=np.float64)
    _fill_normal(np.random.Generator(np.random.PCG64(2000 + config)), w[:, :nlev + 1], 0.1)
    if ldk > nlev:
        vn[:, nlev:] = pad_value
    if ldk_w > nlev + 1:
        w[:, nlev + 1:] = pad_value
    z_half = z_half_levels(nlev)
    if dtype == "f32":
        vn = vn.astype(np.float32)
        w = w.astype(np.float32)
    return vn, w, z_half


def sample_points(seed, n_entities, nlev, n):
    """n seeded (entity, level) pairs, always including the corners of the index space."""
    rng = np.random.Generator(np.random.PCG64(seed))
    idx = rng.integers(0, n_entities, size=n, dtype=np.int64)
    lev = rng.integers(0, nlev, size=n, dtype=np.int64).astype(np.int32)
    idx[:4] = [0, 0, n_entities - 1, n_entities - 1]
    lev[:4] = [0, nlev - 1, 0, nlev - 1]
    return idx, lev


def make_metric_heights(config, edge_xyz, edge_normal, nlev, ldk, ldk_w, dtype="f64", h_top=H_TOP, pad_value=np.nan):
    """Seeded synthetic terrain-following level heights for the metric variant (reading P-20 of DESIGN.md): inputs only.

    Terrain h(x) = a few seeded Gaussian mountains (up to ~3 km) on the unit sphere; hybrid levels
    z_half_e(e,k) = z_flat(k) + h(x_e) * (1 - z_flat(k) / h_top)  (terrain following at the ground, flat at the top);
    slopes of the full-level surfaces at the edge midpoint along n_e and along n_e x x_e. Stand-in for the model's own
    orography and SLEVE levels, which are not available. Returns z_half_e [ne][ldk_w], ddxn_z, ddxt_z [ne][ldk].
    """
    rng = np.random.Generator(np.random.PCG64(3000 + config))
    n_mtn = 6
    centres = rng.standard_normal((n_mtn, 3))
    centres /= np.linalg.norm(centres, axis=1)[:, None]
    heights = 1000.0 + 2000.0 * rng.random(n_mtn)
    widths = 0.15 + 0.25 * rng.random(n_mtn)                 # radians
    ne = edge_xyz.shape[0]
    h = np.zeros(ne)
    grad = np.zeros((ne, 3))                                 # tangential gradient on the sphere of radius 6.371e6 m
    for c, hh, wd in zip(centres, heights, widths):
        d2 = ((edge_xyz - c[None, :]) ** 2).sum(1)           # squared chord distance
        gm = hh * np.exp(-d2 / wd ** 2)
        h += gm
        g3 = gm[:, None] * (-2.0 / wd ** 2) * (edge_xyz - c[None, :])
        g3 -= (g3 * edge_xyz).sum(1)[:, None] * edge_xyz
        grad += g3 / 6.371e6
    zflat = z_half_levels(nlev, h_top)
    zf = 0.5 * (zflat[:-1] + zflat[1:])
    tang = np.cross(edge_normal, edge_xyz)
    zh = np.full((ne, ldk_w), pad_value)
    zh[:, :nlev + 1] = zflat[None, :] + h[:, None] * (1.0 - zflat[None, :] / h_top)
    zn = np.full((ne, ldk), pad_value)
    zt = np.full((ne, ldk), pad_value)
    decay = (1.0 - zf / h_top)[None, :]
    zn[:, :nlev] = (grad * edge_normal).sum(1)[:, None] * decay
    zt[:, :nlev] = (grad * tang).sum(1)[:, None] * decay
    if dtype == "f32":
        zh, zn, zt = zh.astype(np.float32), zn.astype(np.float32), zt.astype(np.float32)
    return zh, zn, zt
