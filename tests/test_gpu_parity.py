"""GPU parity tests (run on the B200 box with -m gpu): the CUDA path, called through the C-ABI,
against the oracle element by element on the same seeded inputs.

Tolerance (BASELINE.json north_star "relative 1e-12 per point in fp64, 1e-5 in the fp32 variant",
reading P-16 of DESIGN.md section 3): |gpu - oracle| <= tol * M(p), M(p) = sum of the absolute
values of the terms entering point p, computed by the oracle next to each output.
"""
import numpy as np
import pytest

import seeded_inputs as si

pytestmark = pytest.mark.gpu

TOL = {"f64": 1e-12, "f32": 1e-5}


@pytest.fixture(scope="module")
def torch_cuda():
    import torch
    if not torch.cuda.is_available():
        pytest.fail("-m gpu tests need a CUDA device")
    return torch


@pytest.fixture(scope="module")
def lib():
    import paper_2511_02021_b200 as lib
    lib.load_library()          # raises if the CUDA extension has not been built: no fallback
    return lib


_libgrids = {}


# ICON_OPT_TENDENCY_KERNEL values (4 = column cache, the default wherever it holds the columns)
VARIANTS = [0, 3, 4]


def lib_grid(lib, k, seed=0, flags=0):
    key = (k, seed, flags)
    if key not in _libgrids:
        _libgrids[key] = lib.IconGrid(k, seed, flags)
    return _libgrids[key]


def run_gpu(torch, lib, g, vn, w, zh, nlev, variant, want_opt=False, sentinel=None):
    """returns dict of numpy outputs from dycore_velocity_tendencies + dycore_div_vort"""
    dev = torch.device("cuda:0")
    tdt = torch.float64 if vn.dtype == np.float64 else torch.float32
    d_vn = torch.from_numpy(vn).to(dev)
    d_w = torch.from_numpy(w).to(dev)
    ldk = vn.shape[1]

    def out(n):
        t = torch.empty((n, ldk), dtype=tdt, device=dev)
        t.fill_(float("nan") if sentinel is None else sentinel)
        return t
    ddt, div, vort = out(g.ne), out(g.nc), out(g.nv)
    opt = dict(vt=out(g.ne), ke_c=out(g.nc), vort=out(g.nv)) if want_opt else {}
    g.set_option(lib.ICON_OPT_TENDENCY_KERNEL, variant)
    n0 = g.launch_count
    lib.dycore_velocity_tendencies(g, zh, d_vn, d_w, ddt, nlev, **opt)
    lib.dycore_div_vort(g, d_vn, div, vort, nlev)
    torch.cuda.synchronize()
    assert g.launch_count > n0
    res = dict(ddt_vn=ddt.cpu().numpy(), div=div.cpu().numpy(), vort=vort.cpu().numpy())
    for k_, t in opt.items():
        res[k_ + "_opt"] = t.cpu().numpy()
    return res


def oracle_reference(og, vn, w, zh, nlev, f32):
    """oracle outputs + tolerance scales; fp32 variant: fp64 arithmetic on fp32-rounded inputs (P-17)"""
    o = og.rounded_f32() if f32 else og
    vn64, w64 = vn.astype(np.float64), w.astype(np.float64)
    vn64 = np.where(np.isnan(vn64), 0.0, vn64)       # padding lanes: never enter the compared levels
    w64 = np.where(np.isnan(w64), 0.0, w64)
    t = o.velocity_tendencies(vn64, w64, zh, nlev, with_scale=True)
    div, vort, md, mv = o.div_vort(vn64, nlev, with_scale=True)
    t.update(div=div, m_div=md, vort_dv=vort, m_vort=mv)
    return t


def assert_close(name, got, want, scale, tol, nlev):
    got = got[:, :nlev].astype(np.float64)
    err = np.abs(got - want[:, :nlev])
    bound = tol * scale[:, :nlev]
    bad = ~(err <= bound)
    assert not bad.any(), "%s: %d points outside tol*M, worst err/M = %.3e" % (
        name, bad.sum(), (err / np.maximum(scale[:, :nlev], 1e-300)).max())


def check_all(res, ref, nlev, tol, opt=False):
    assert_close("ddt_vn", res["ddt_vn"], ref["ddt_vn"], ref["m_ddt"], tol, nlev)
    assert_close("div", res["div"], ref["div"], ref["m_div"], tol, nlev)
    assert_close("vort", res["vort"], ref["vort_dv"], ref["m_vort"], tol, nlev)
    if opt:
        assert_close("vort_opt", res["vort_opt"], ref["vort"], ref["m_vort"], tol, nlev)
        # vt: sum of 4 products, scale = |vn| level of the stencil (<= max |vn| * sum|rbf| ~ 1.3 max|vn|)
        s_vt = np.full_like(ref["vt"], 1.3 * np.abs(ref["vt"]).max() + 1.0)
        assert_close("vt_opt", res["vt_opt"], ref["vt"], s_vt, tol, nlev)
        assert_close("ke_c_opt", res["ke_c_opt"], ref["ke_c"], np.abs(ref["ke_c"]) + np.abs(ref["ke_c"]).mean(), tol, nlev)


# ----------------------------------------------------------------------------------------------
# configs[0]: R2B4 x 90 fp64, element by element, every kernel variant, optional outputs
# ----------------------------------------------------------------------------------------------
@pytest.mark.parametrize("variant", VARIANTS)
def test_config1_r2b4_fp64_elementwise(torch_cuda, lib, oracle_grid, variant):
    og = oracle_grid(4)
    g = lib_grid(lib, 4)
    vn, w, zh = si.make_fields(1, og.edge_xyz, og.edge_normal, og.nc, ldk_w=92)   # ldk_w*8 must be a multiple of 16
    ref = oracle_reference(og, vn, w, zh, 90, False)
    res = run_gpu(torch_cuda, lib, g, vn, w, zh, 90, variant, want_opt=(variant == 0))
    check_all(res, ref, 90, TOL["f64"], opt=(variant == 0))
    res = run_gpu(torch_cuda, lib, g, vn, w, zh, 90, variant, want_opt=True)
    check_all(res, ref, 90, TOL["f64"], opt=True)


def test_library_geometry_fed_to_oracle(torch_cuda, lib, oracle_mod, oracle_grid):
    """P-18: operator parity with the oracle evaluating on the LIBRARY's exported tables"""
    g = lib_grid(lib, 3)
    t = {n: g.table_host(n) for n in ("c2e", "e2c", "e2v", "e2e4", "v2e", "rbf", "bln", "geofac_rot", "geofac_div",
                                      "inv_d_e", "f_e", "c_lin")}
    nlev = 17
    vn, w, zh = si.make_fields(1, g.table_host("edge_xyz"), g.table_host("edge_normal"), g.nc, nlev=nlev, ldk=18, ldk_w=18)
    vn64, w64 = np.nan_to_num(vn), np.nan_to_num(w)
    ref = oracle_mod.velocity_tendencies_from_arrays(t, vn64, w64, zh, nlev)
    div, md = oracle_mod.divergence(t["c2e"], t["geofac_div"], vn64, nlev)
    vort, mv = oracle_mod.vorticity(t["v2e"], t["geofac_rot"], vn64, nlev)
    ref.update(div=div, m_div=md, vort_dv=vort, m_vort=mv)
    for variant in VARIANTS:
        res = run_gpu(torch_cuda, lib, g, vn, w, zh, nlev, variant)
        check_all(res, ref, nlev, TOL["f64"])


# ----------------------------------------------------------------------------------------------
# edge cases: tiny grids, ragged level counts, minimum nlev, padded leading dimension
# ----------------------------------------------------------------------------------------------
@pytest.mark.parametrize("k,nlev,ldk,ldk_w", [(0, 2, 2, 4), (0, 3, 4, 4), (1, 31, 32, 32), (1, 33, 34, 34),
                                               (2, 64, 64, 66), (2, 65, 66, 66), (3, 90, 96, 92), (2, 130, 130, 132)])
@pytest.mark.parametrize("variant", VARIANTS)
def test_ragged_levels_and_padding(torch_cuda, lib, oracle_grid, k, nlev, ldk, ldk_w, variant):
    og = oracle_grid(k)
    g = lib_grid(lib, k)
    vn, w, zh = si.make_fields(1, og.edge_xyz, og.edge_normal, og.nc, nlev=nlev, ldk=ldk, ldk_w=ldk_w)
    ref = oracle_reference(og, vn, w, zh, nlev, False)
    sentinel = -12345.5
    res = run_gpu(torch_cuda, lib, g, vn, w, zh, nlev, variant, sentinel=sentinel)
    check_all(res, ref, nlev, TOL["f64"])
    for name in ("ddt_vn", "div", "vort"):            # padding lanes of outputs are left untouched
        assert (res[name][:, nlev:] == sentinel).all(), name


@pytest.mark.parametrize("flags_extra", [0, 8])
@pytest.mark.parametrize("variant", VARIANTS)
def test_permuted_grid_fp64(torch_cuda, lib, oracle_grid, flags_extra, variant):
    """seeded renumbering, with the locality work-list (default) and without (ICON_NO_WORKLIST)"""
    og = oracle_grid(3, si.PERMUTE_SEED, 1)
    g = lib_grid(lib, 3, si.PERMUTE_SEED, 1 | flags_extra)
    nlev = 40
    vn, w, zh = si.make_fields(4, og.edge_xyz, og.edge_normal, og.nc, nlev=nlev, ldk=40, ldk_w=42, dtype="f64")
    ref = oracle_reference(og, vn, w, zh, nlev, False)
    res = run_gpu(torch_cuda, lib, g, vn, w, zh, nlev, variant, want_opt=True)
    check_all(res, ref, nlev, TOL["f64"], opt=True)
    res = run_gpu(torch_cuda, lib, g, vn, w, zh, nlev, variant)
    check_all(res, ref, nlev, TOL["f64"])


@pytest.mark.parametrize("variant", VARIANTS)
def test_fp32_variant_permuted_r2b4(torch_cuda, lib, oracle_grid, variant):
    """config 4 at a size the oracle finishes in seconds: fp32 fields, permuted ids, tol 1e-5"""
    og = oracle_grid(4, si.PERMUTE_SEED, 1)
    g = lib_grid(lib, 4, si.PERMUTE_SEED, 1)
    vn, w, zh = si.make_fields(4, og.edge_xyz, og.edge_normal, og.nc, ldk=92, ldk_w=92)
    assert vn.dtype == np.float32
    ref = oracle_reference(og, vn, w, zh, 90, True)
    res = run_gpu(torch_cuda, lib, g, vn, w, zh, 90, variant, want_opt=True)
    check_all(res, ref, 90, TOL["f32"], opt=True)
    res = run_gpu(torch_cuda, lib, g, vn, w, zh, 90, variant)
    check_all(res, ref, 90, TOL["f32"])


def test_column_cache_never_reads_a_stale_slot(torch_cuda, lib, oracle_grid):
    """Kernel 4 keeps columns in shared memory across steps. Repeating ONE input hides a read that comes too
    early (the slot still holds the same column from the previous launch), so two different inputs alternate
    and every launch is compared with the oracle. This is the test that caught bulk copies of an earlier step
    still in flight when a later step read their slot."""
    torch = torch_cuda
    og = oracle_grid(4)
    g = lib_grid(lib, 4)
    dev = torch.device("cuda:0")
    nlev = 90
    sets = []
    for cfg, fv, fw in ((1, 1.0, 1.0), (2, -3.0, 5.0)):
        vn, w, zh = si.make_fields(cfg, og.edge_xyz, og.edge_normal, og.nc, nlev=nlev, ldk=90, ldk_w=92)
        vn, w = np.nan_to_num(vn) * fv, np.nan_to_num(w) * fw
        ref = og.velocity_tendencies(vn, w, zh, nlev, with_scale=True)
        sets.append((torch.from_numpy(vn).to(dev), torch.from_numpy(w).to(dev), zh, ref))
    g.set_option(lib.ICON_OPT_TENDENCY_KERNEL, 4)
    for it in range(300):
        d_vn, d_w, zh, ref = sets[it % 2]
        ddt = torch.full((g.ne, 90), float("nan"), dtype=torch.float64, device=dev)
        lib.dycore_velocity_tendencies(g, zh, d_vn, d_w, ddt, nlev)
        torch.cuda.synchronize()
        err = np.abs(ddt.cpu().numpy() - ref["ddt_vn"])
        assert (err <= TOL["f64"] * ref["m_ddt"]).all(), "launch %d" % it


@pytest.mark.parametrize("variant", [5, 4, 3])
@pytest.mark.parametrize("k,seed,flags,nlev,ldk,ldk_w,cfg", [(4, 0, 0, 90, 96, 96, 1), (4, 0, 0, 90, 90, 92, 1), (2, 0, 0, 33, 34, 34, 1),
                                                         (1, 0, 0, 30, 30, 32, 1), (0, 0, 0, 3, 4, 4, 1),
                                                         (3, si.PERMUTE_SEED, 1, 40, 40, 42, 4)])
def test_dycore_step_matches_the_two_calls_and_the_oracle(torch_cuda, lib, oracle_grid, variant, k, seed, flags, nlev, ldk,
                                                          ldk_w, cfg):
    """dycore_step: ddt_vn, div and vort from one pass (one fused kernel where kernel 4 runs). Every level of every
    column of all three outputs is written exactly once (NaN sentinel), pads stay untouched, values match the oracle."""
    torch = torch_cuda
    og = oracle_grid(k, seed, flags)
    g = lib_grid(lib, k, seed, flags)
    vn, w, zh = si.make_fields(cfg, og.edge_xyz, og.edge_normal, og.nc, nlev=nlev, ldk=ldk, ldk_w=ldk_w, dtype="f64")
    ref = oracle_reference(og, vn, w, zh, nlev, False)
    dev = torch.device("cuda:0")
    d_vn, d_w = torch.from_numpy(vn).to(dev), torch.from_numpy(w).to(dev)
    sentinel = -4321.25
    outs = [torch.full((n, ldk), sentinel, dtype=torch.float64, device=dev) for n in (g.ne, g.nc, g.nv)]
    g.set_option(lib.ICON_OPT_TENDENCY_KERNEL, variant)
    n0 = g.launch_count
    lib.dycore_step(g, zh, d_vn, d_w, outs[0], outs[1], outs[2], nlev)
    torch.cuda.synchronize()
    launches = g.launch_count - n0
    fused_regime = variant in (4, 5)            # every nlev of this test fits the column cache
    assert launches == (1 if fused_regime else 2)
    res = dict(ddt_vn=outs[0].cpu().numpy(), div=outs[1].cpu().numpy(), vort=outs[2].cpu().numpy())
    check_all(res, ref, nlev, TOL["f64"])
    for name in ("ddt_vn", "div", "vort"):
        assert (res[name][:, nlev:] == sentinel).all(), name
        assert not (res[name][:, :nlev] == sentinel).any(), name
    g.set_option(lib.ICON_OPT_TENDENCY_KERNEL, 5)


@pytest.mark.parametrize("period", [0, 4, 16, 512])
def test_fused_step_pacing_barrier_periods(torch_cuda, lib, oracle_grid, period):
    """The fused fp64 kernel's producers meet at a chip-wide counter every `period` steps (ICON_OPT_CC_PACE; DESIGN.md
    section 6.1). The counter's base advances from launch to launch, so several launches run back to back on alternating
    inputs; every one is compared with the oracle. R2B5 gives each CTA ~70 steps: periods 4 and 16 arm many barriers,
    512 arms none, 0 switches pacing off."""
    torch = torch_cuda
    og = oracle_grid(5)
    g = lib_grid(lib, 5)
    dev = torch.device("cuda:0")
    nlev = 90
    sets = []
    for cfg, fv in ((1, 1.0), (2, -2.0)):
        vn, w, zh = si.make_fields(cfg, og.edge_xyz, og.edge_normal, og.nc, nlev=nlev, ldk=96, ldk_w=96)
        vn, w = np.nan_to_num(vn) * fv, np.nan_to_num(w)
        ref = oracle_reference(og, vn, w, zh, nlev, False)
        sets.append((torch.from_numpy(vn).to(dev), torch.from_numpy(w).to(dev), zh, ref))
    g.set_option(lib.ICON_OPT_TENDENCY_KERNEL, 5)
    g.set_option(lib.ICON_OPT_CC_PACE, period)
    try:
        for it in range(6):
            d_vn, d_w, zh, ref = sets[it % 2]
            outs = [torch.full((n, 96), float("nan"), dtype=torch.float64, device=dev) for n in (g.ne, g.nc, g.nv)]
            n0 = g.launch_count
            lib.dycore_step(g, zh, d_vn, d_w, outs[0], outs[1], outs[2], nlev)
            torch.cuda.synchronize()
            assert g.launch_count - n0 == 1
            res = dict(ddt_vn=outs[0].cpu().numpy(), div=outs[1].cpu().numpy(), vort=outs[2].cpu().numpy())
            check_all(res, ref, nlev, TOL["f64"])
    finally:
        g.set_option(lib.ICON_OPT_CC_PACE, 512)


@pytest.mark.parametrize("tile", [16, 64, 0])
@pytest.mark.parametrize("dtype,nlev,ldk,ldk_w", [("f64", 90, 96, 96), ("f64", 90, 90, 92), ("f64", 33, 34, 34), ("f32", 90, 96, 96),
                                                   ("f32", 90, 92, 92), ("f64", 30, 32, 32), ("f64", 3, 4, 4), ("f64", 64, 64, 66),
                                                   ("f64", 95, 96, 96), ("f32", 30, 32, 32), ("f32", 31, 32, 32)])
def test_column_cache_level_mappings_and_tiles(torch_cuda, lib, oracle_grid, tile, dtype, nlev, ldk, ldk_w):
    """kernel 4 with the default tiles, larger tiles and contiguous ranges; every level
    mapping (one level per lane; pair + single with the single segment empty, partly and completely filled, odd and even
    level counts so that the last pair is half valid); tendency-only and fused step"""
    torch = torch_cuda
    og = oracle_grid(4)
    g = lib_grid(lib, 4)
    vn, w, zh = si.make_fields(1 if dtype == "f64" else 4, og.edge_xyz, og.edge_normal, og.nc, nlev=nlev, ldk=ldk, ldk_w=ldk_w,
                               dtype=dtype)
    ref = oracle_reference(og, vn, w, zh, nlev, dtype == "f32")
    g.set_option(lib.ICON_OPT_CC_TILE, tile)
    try:
        res = run_gpu(torch, lib, g, vn, w, zh, nlev, 4, sentinel=-77.5)
        check_all(res, ref, nlev, TOL[dtype])
        assert (res["ddt_vn"][:, nlev:] == -77.5).all()
        dev = torch.device("cuda:0")
        outs = [torch.full((n, ldk), -77.5, dtype=torch.from_numpy(vn).dtype, device=dev) for n in (g.ne, g.nc, g.nv)]
        n0 = g.launch_count
        lib.dycore_step(g, zh, torch.from_numpy(vn).to(dev), torch.from_numpy(w).to(dev), outs[0], outs[1], outs[2], nlev)
        torch.cuda.synchronize()
        assert g.launch_count - n0 == 1
        res = dict(ddt_vn=outs[0].cpu().numpy(), div=outs[1].cpu().numpy(), vort=outs[2].cpu().numpy())
        check_all(res, ref, nlev, TOL[dtype])
        for name in res:
            assert (res[name][:, nlev:] == -77.5).all(), name
            assert not (res[name][:, :nlev] == -77.5).any(), name
    finally:
        g.set_option(lib.ICON_OPT_CC_TILE, -1)
        g.set_option(lib.ICON_OPT_TENDENCY_KERNEL, 5)


@pytest.mark.parametrize("k,period", [(5, 4), (5, 512), (3, 16)])
def test_dycore_step_replays_in_a_cuda_graph(torch_cuda, lib, oracle_grid, k, period):
    """SURVEY.md 8(f) NEXT-4 (the paper's remedy for launch-bound small kernels): dycore_step captured once
    into a CUDA graph and replayed 12 times on alternating inputs written into the captured buffers; every replay is
    compared with the oracle. The pacing epoch lives on the device (a captured kernel argument would go stale): periods 4
    and 16 arm many barriers per launch."""
    torch = torch_cuda
    og = oracle_grid(k)
    g = lib_grid(lib, k)
    dev = torch.device("cuda:0")
    nlev = 90
    sets = []
    for cfg, fv in ((1, 1.0), (2, -2.0)):
        vn, w, zh = si.make_fields(cfg, og.edge_xyz, og.edge_normal, og.nc, nlev=nlev, ldk=96, ldk_w=96)
        vn, w = np.nan_to_num(vn) * fv, np.nan_to_num(w)
        sets.append((torch.from_numpy(vn).to(dev), torch.from_numpy(w).to(dev), zh, oracle_reference(og, vn, w, zh, nlev, False)))
    g.set_option(lib.ICON_OPT_TENDENCY_KERNEL, 5)
    g.set_option(lib.ICON_OPT_CC_PACE, period)
    try:
        s_vn, s_w = sets[0][0].clone(), sets[0][1].clone()                       # the buffers the graph reads
        outs = [torch.full((n, 96), float("nan"), dtype=torch.float64, device=dev) for n in (g.ne, g.nc, g.nv)]
        zh = sets[0][2]
        side = torch.cuda.Stream()
        side.wait_stream(torch.cuda.current_stream())
        with torch.cuda.stream(side):                                            # first call: builds and uploads the tables
            lib.dycore_step(g, zh, s_vn, s_w, outs[0], outs[1], outs[2], nlev)
        torch.cuda.current_stream().wait_stream(side)
        torch.cuda.synchronize()
        graph = torch.cuda.CUDAGraph()
        with torch.cuda.graph(graph):
            lib.dycore_step(g, zh, s_vn, s_w, outs[0], outs[1], outs[2], nlev)
        for it in range(12):
            d_vn, d_w, _, ref = sets[it % 2]
            s_vn.copy_(d_vn)
            s_w.copy_(d_w)
            for o in outs:
                o.fill_(float("nan"))
            graph.replay()
            torch.cuda.synchronize()
            res = dict(ddt_vn=outs[0].cpu().numpy(), div=outs[1].cpu().numpy(), vort=outs[2].cpu().numpy())
            check_all(res, ref, nlev, TOL["f64"])
        # plain launches still work after the replays (the device-side epoch stays consistent)
        for o in outs:
            o.fill_(float("nan"))
        lib.dycore_step(g, zh, sets[1][0], sets[1][1], outs[0], outs[1], outs[2], nlev)
        torch.cuda.synchronize()
        check_all(dict(ddt_vn=outs[0].cpu().numpy(), div=outs[1].cpu().numpy(), vort=outs[2].cpu().numpy()), sets[1][3], nlev, TOL["f64"])
    finally:
        g.set_option(lib.ICON_OPT_CC_PACE, 512)


# ----------------------------------------------------------------------------------------------
# vertical-wind tendency (reading P-19)
# ----------------------------------------------------------------------------------------------
@pytest.mark.parametrize("variant", [5, 0])
@pytest.mark.parametrize("k,seed,flags,nlev,ldk,ldk_w,dtype", [
    (4, 0, 0, 90, 90, 92, "f64"), (4, 0, 0, 90, 96, 96, "f64"), (3, si.PERMUTE_SEED, 1, 40, 40, 42, "f64"),
    (3, si.PERMUTE_SEED, 1 | 8, 40, 40, 42, "f64"), (4, si.PERMUTE_SEED, 1, 90, 92, 92, "f32"), (0, 0, 0, 2, 2, 4, "f64"),
    (0, 0, 0, 3, 4, 4, "f64"), (1, 0, 0, 31, 32, 32, "f64"), (1, 0, 0, 33, 34, 34, "f64"), (2, 0, 0, 130, 130, 132, "f64"),
    (2, 0, 0, 30, 32, 32, "f64"), (2, 0, 0, 64, 64, 66, "f64"), (2, 0, 0, 65, 66, 66, "f64"), (2, 0, 0, 95, 96, 96, "f64"),
    (3, 0, 0, 30, 32, 32, "f32"), (3, 0, 0, 63, 64, 64, "f32")])
def test_w_tendency_elementwise(torch_cuda, lib, oracle_mod, oracle_grid, variant, k, seed, flags, nlev, ldk, ldk_w, dtype):
    """dycore_w_tendency against og_w_tendency, every half level of every cell; pads stay untouched; also with the
    oracle evaluating on the LIBRARY's exported tables (P-18). variant 5 (auto): the column cache in its ddt_w mode
    (nlev = 130 falls back to the gather kernel); variant 0: the gather kernel. Two launches on different inputs (a stale
    slot of the cache would carry the other input)."""
    torch = torch_cuda
    og = oracle_grid(k, seed, flags & 1)
    g = lib_grid(lib, k, seed, flags)
    f32 = dtype == "f32"
    o = og.rounded_f32() if f32 else og
    dev = torch.device("cuda:0")
    sentinel = -9.25
    g.set_option(lib.ICON_OPT_TENDENCY_KERNEL, variant)
    try:
        for cfg, fv in ((4 if flags & 1 else 1, 1.0), (2, -2.5)):
            vn, w, zh = si.make_fields(cfg, og.edge_xyz, og.edge_normal, og.nc, nlev=nlev, ldk=ldk, ldk_w=ldk_w, dtype=dtype)
            vn = (vn * fv).astype(vn.dtype)
            vn64, w64 = np.nan_to_num(vn.astype(np.float64)), np.nan_to_num(w.astype(np.float64))
            want, m = o.w_tendency(vn64, w64, zh, nlev, with_scale=True)
            out = torch.full((g.nc, ldk_w), sentinel, dtype=torch.from_numpy(w).dtype, device=dev)
            n0 = g.launch_count
            lib.dycore_w_tendency(g, zh, torch.from_numpy(vn).to(dev), torch.from_numpy(w).to(dev), out, nlev)
            torch.cuda.synchronize()
            assert g.launch_count - n0 == 1
            got = out.cpu().numpy().astype(np.float64)
            err = np.abs(got[:, :nlev + 1] - want[:, :nlev + 1])
            assert (err <= TOL[dtype] * m[:, :nlev + 1]).all(), "worst err/M %.3e" % (err / np.maximum(m[:, :nlev + 1], 1e-300)).max()
            assert (got[:, 0] == 0).all() and (got[:, nlev] == 0).all()
            assert (got[:, nlev + 1:] == sentinel).all()
            if not f32:
                t = {n: g.table_host(n) for n in ("c2e", "e2c", "inv_d_e", "adv_c")}
                want2, m2 = oracle_mod.w_tendency_from_arrays(t, vn64, w64, zh, nlev)
                assert (np.abs(got[:, :nlev + 1] - want2[:, :nlev + 1]) <= TOL[dtype] * m2[:, :nlev + 1]).all()
    finally:
        g.set_option(lib.ICON_OPT_TENDENCY_KERNEL, 5)


@pytest.mark.parametrize("k,seed,flags,nlev,ldk,ldk_w,dtype", [
    (4, 0, 0, 90, 96, 96, "f64"), (4, 0, 0, 90, 90, 92, "f64"), (3, si.PERMUTE_SEED, 1, 40, 40, 42, "f64"),
    (4, si.PERMUTE_SEED, 1, 90, 96, 96, "f32"), (2, 0, 0, 30, 32, 32, "f64"), (1, 0, 0, 31, 32, 32, "f64"), (2, 0, 0, 33, 34, 34, "f64"),
    (2, 0, 0, 65, 66, 66, "f64"), (2, 0, 0, 95, 96, 96, "f64"), (0, 0, 0, 3, 4, 4, "f64"), (2, 0, 0, 130, 130, 132, "f64"),
    (3, 0, 0, 30, 32, 32, "f32")])
def test_dycore_step_w_all_four_outputs(torch_cuda, lib, oracle_grid, k, seed, flags, nlev, ldk, ldk_w, dtype):
    """dycore_step_w: ddt_vn, div, vort AND ddt_w from one pass (one fused kernel where the column cache runs; nlev = 130
    takes the separate calls). Two launches on different inputs; every level of every column written once, pads untouched."""
    torch = torch_cuda
    og = oracle_grid(k, seed, flags & 1)
    g = lib_grid(lib, k, seed, flags)
    f32 = dtype == "f32"
    dev = torch.device("cuda:0")
    o = og.rounded_f32() if f32 else og
    g.set_option(lib.ICON_OPT_TENDENCY_KERNEL, 5)
    for cfg, fv in ((1, 1.0), (2, -2.5)):
        vn, w, zh = si.make_fields(cfg, og.edge_xyz, og.edge_normal, og.nc, nlev=nlev, ldk=ldk, ldk_w=ldk_w, dtype=dtype)
        vn = (vn * fv).astype(vn.dtype)
        ref = oracle_reference(og, vn, w, zh, nlev, f32)
        vn64, w64 = np.nan_to_num(vn.astype(np.float64)), np.nan_to_num(w.astype(np.float64))
        want_w, m_w = o.w_tendency(vn64, w64, zh, nlev, with_scale=True)
        tdt = torch.from_numpy(vn).dtype
        sentinel = -4321.25
        outs = [torch.full((n, ldk), sentinel, dtype=tdt, device=dev) for n in (g.ne, g.nc, g.nv)]
        dw = torch.full((g.nc, ldk_w), sentinel, dtype=tdt, device=dev)
        n0 = g.launch_count
        lib.dycore_step_w(g, zh, torch.from_numpy(vn).to(dev), torch.from_numpy(w).to(dev), outs[0], outs[1], outs[2], dw, nlev)
        torch.cuda.synchronize()
        assert g.launch_count - n0 == (1 if nlev + 1 <= 96 else 3)
        res = dict(ddt_vn=outs[0].cpu().numpy(), div=outs[1].cpu().numpy(), vort=outs[2].cpu().numpy())
        check_all(res, ref, nlev, TOL[dtype])
        for name in res:
            assert (res[name][:, nlev:] == sentinel).all(), name
            assert not (res[name][:, :nlev] == sentinel).any(), name
        got = dw.cpu().numpy().astype(np.float64)
        err = np.abs(got[:, :nlev + 1] - want_w[:, :nlev + 1])
        assert (err <= TOL[dtype] * m_w[:, :nlev + 1]).all(), "ddt_w worst err/M %.3e" % (err / np.maximum(m_w[:, :nlev + 1], 1e-300)).max()
        assert (got[:, 0] == 0).all() and (got[:, nlev] == 0).all() and (got[:, nlev + 1:] == sentinel).all()


# ----------------------------------------------------------------------------------------------
# metric variant (reading P-20)
# ----------------------------------------------------------------------------------------------
@pytest.mark.parametrize("variant", [5, 0])
@pytest.mark.parametrize("k,seed,flags,nlev,ldk,ldk_w,dtype", [
    (4, 0, 0, 90, 96, 96, "f64"), (4, 0, 0, 90, 90, 92, "f64"), (3, si.PERMUTE_SEED, 1, 40, 40, 42, "f64"),
    (4, si.PERMUTE_SEED, 1, 90, 96, 96, "f32"), (2, 0, 0, 30, 32, 32, "f64"), (1, 0, 0, 31, 32, 32, "f64"), (2, 0, 0, 33, 34, 34, "f64"),
    (2, 0, 0, 64, 64, 66, "f64"), (2, 0, 0, 65, 66, 66, "f64"), (2, 0, 0, 95, 96, 96, "f64"), (0, 0, 0, 3, 4, 4, "f64"),
    (2, 0, 0, 130, 130, 132, "f64"), (3, 0, 0, 30, 32, 32, "f32")])
def test_metric_variant_elementwise(torch_cuda, lib, oracle_mod, oracle_grid, variant, k, seed, flags, nlev, ldk, ldk_w, dtype):
    """dycore_metric_from_zhalf and dycore_velocity_tendencies_metric against the oracle on a seeded terrain-following grid:
    the fused column-cache mode (variant 5 = auto; nlev = 130 falls back) and the unfused pipeline (variant 0); two launches
    on different inputs; every level written once, pads untouched"""
    torch = torch_cuda
    og = oracle_grid(k, seed, flags & 1)
    g = lib_grid(lib, k, seed, flags)
    f32 = dtype == "f32"
    dev = torch.device("cuda:0")
    o = og.rounded_f32() if f32 else og
    zh_e, zn, zt = si.make_metric_heights(1, og.edge_xyz, og.edge_normal, nlev, ldk, ldk_w, dtype=dtype)
    tdt = torch.float32 if f32 else torch.float64
    d_zh = torch.from_numpy(zh_e).to(dev)
    sentinel = -6.75
    d_wgt = torch.full((g.ne, ldk_w), sentinel, dtype=tdt, device=dev)
    d_inv = torch.full((g.ne, ldk), sentinel, dtype=tdt, device=dev)
    lib.dycore_metric_from_zhalf(g, d_zh, d_wgt, d_inv, nlev)
    torch.cuda.synchronize()
    wgt_o, inv_o = oracle_mod.metric_from_zhalf(np.nan_to_num(zh_e.astype(np.float64)), nlev, ldk)
    rel = 1e-5 if f32 else 1e-12          # the thicknesses of fp32 heights of 30 km carry ~1e-4 relative rounding themselves:
    wgt_g, inv_g = d_wgt.cpu().numpy().astype(np.float64), d_inv.cpu().numpy().astype(np.float64)
    if not f32:                           # compared in fp64 only; fp32 goes on with the device's own metrics below
        assert np.abs(wgt_g[:, :nlev + 1] - wgt_o[:, :nlev + 1]).max() <= rel
        assert np.abs(inv_g[:, :nlev] / inv_o[:, :nlev] - 1).max() <= rel
    assert (wgt_g[:, nlev + 1:] == sentinel).all() and (inv_g[:, nlev:] == sentinel).all()
    # the operator is compared on the metrics the DEVICE derived (inputs of the operator; fp32: rounded to fp32 there)
    wgt_in, inv_in = np.nan_to_num(np.where(wgt_g == sentinel, 0, wgt_g)), np.nan_to_num(np.where(inv_g == sentinel, 0, inv_g))
    zn64, zt64 = np.nan_to_num(zn.astype(np.float64)), np.nan_to_num(zt.astype(np.float64))
    d_zn, d_zt = torch.from_numpy(zn).to(dev), torch.from_numpy(zt).to(dev)
    g.set_option(lib.ICON_OPT_TENDENCY_KERNEL, variant)
    try:
        for cfg, fv in ((1, 1.0), (2, -2.5)):
            vn, w, _ = si.make_fields(cfg, og.edge_xyz, og.edge_normal, og.nc, nlev=nlev, ldk=ldk, ldk_w=ldk_w, dtype=dtype)
            vn = (vn * fv).astype(vn.dtype)
            vn64, w64 = np.nan_to_num(vn.astype(np.float64)), np.nan_to_num(w.astype(np.float64))
            ref = o.velocity_tendencies_metric(vn64, w64, wgt_in, inv_in, zn64, zt64, nlev, with_scale=True)
            out = torch.full((g.ne, ldk), sentinel, dtype=tdt, device=dev)
            n0 = g.launch_count
            lib.dycore_velocity_tendencies_metric(g, d_wgt, d_inv, d_zn, d_zt, torch.from_numpy(vn).to(dev), torch.from_numpy(w).to(dev), out, nlev)
            torch.cuda.synchronize()
            assert g.launch_count - n0 == (1 if (variant == 5 and nlev + 1 <= 96) else 3)
            got = out.cpu().numpy().astype(np.float64)
            assert_close("ddt_vn (metric)", got, ref["ddt_vn"], ref["m_ddt"], TOL[dtype], nlev)
            assert (got[:, nlev:] == sentinel).all() and not (got[:, :nlev] == sentinel).any()
    finally:
        g.set_option(lib.ICON_OPT_TENDENCY_KERNEL, 5)


def test_argument_errors_on_device(torch_cuda, lib):
    torch = torch_cuda
    g = lib_grid(lib, 1)
    dev = torch.device("cuda:0")
    vn = torch.zeros((g.ne, 6), dtype=torch.float64, device=dev)
    w = torch.zeros((g.nc, 8), dtype=torch.float64, device=dev)
    out = torch.zeros_like(vn)
    zh = si.z_half_levels(6)
    with pytest.raises(lib.IconError):                 # z_half not strictly decreasing
        lib.dycore_velocity_tendencies(g, zh[::-1].copy(), vn, w, out, 6)
    with pytest.raises(lib.IconError):                 # output aliases input
        lib.dycore_velocity_tendencies(g, zh, vn, w, vn, 6)
    with pytest.raises(lib.IconError):                 # nlev > ldk
        lib.dycore_div_vort(g, vn, torch.zeros((g.nc, 6), dtype=torch.float64, device=dev),
                            torch.zeros((g.nv, 6), dtype=torch.float64, device=dev), 7)
    with pytest.raises(lib.IconError):                 # outputs overlap each other (views of one buffer)
        buf = torch.zeros((g.ne + g.nc, 6), dtype=torch.float64, device=dev)
        lib.dycore_step(g, zh, vn, w, buf[:g.ne], buf[g.nc:g.nc + g.nc], torch.zeros((g.nv, 6), dtype=torch.float64, device=dev), 6)
    with pytest.raises(ValueError):                    # wrong row count
        lib.dycore_div_vort(g, vn, torch.zeros((g.nc + 1, 6), dtype=torch.float64, device=dev),
                            torch.zeros((g.nv, 6), dtype=torch.float64, device=dev), 6)
    with pytest.raises(ValueError):                    # non-contiguous view
        lib.dycore_div_vort(g, torch.zeros((g.ne, 12), dtype=torch.float64, device=dev)[:, ::2],
                            torch.zeros((g.nc, 6), dtype=torch.float64, device=dev), torch.zeros((g.nv, 6), dtype=torch.float64, device=dev), 6)
    with pytest.raises(TypeError):                     # mixed dtypes
        lib.dycore_div_vort(g, vn, torch.zeros((g.nc, 6), dtype=torch.float32, device=dev),
                            torch.zeros((g.nv, 6), dtype=torch.float64, device=dev), 6)
    vn3 = torch.zeros((g.ne, 3), dtype=torch.float64, device=dev)   # ldk*8 not a multiple of 16
    with pytest.raises(lib.IconError):
        lib.dycore_div_vort(g, vn3, torch.zeros((g.nc, 3), dtype=torch.float64, device=dev),
                            torch.zeros((g.nv, 3), dtype=torch.float64, device=dev), 3)


def test_step_host_end_to_end(torch_cuda, lib, oracle_grid):
    """dycore_step_host: host buffers in, host buffers out, same numbers as the device calls"""
    torch = torch_cuda
    og = oracle_grid(3)
    g = lib_grid(lib, 3)
    vn, w, zh = si.make_fields(1, og.edge_xyz, og.edge_normal, og.nc, nlev=30, ldk=30, ldk_w=32)
    ref = oracle_reference(og, vn, w, zh, 30, False)
    h_vn, h_w = torch.from_numpy(vn).pin_memory(), torch.from_numpy(w).pin_memory()
    ddt = torch.zeros((g.ne, 30), dtype=torch.float64).pin_memory()
    div = torch.zeros((g.nc, 30), dtype=torch.float64).pin_memory()
    vort = torch.zeros((g.nv, 30), dtype=torch.float64).pin_memory()
    g.set_option(lib.ICON_OPT_TENDENCY_KERNEL, 5)
    lib.dycore_step_host(g, zh, h_vn, h_w, ddt, div, vort, 30)
    check_all(dict(ddt_vn=ddt.numpy(), div=div.numpy(), vort=vort.numpy()), ref, 30, TOL["f64"])


# ----------------------------------------------------------------------------------------------
# full-size configs (BASELINE.json configs[1..4]): sampled outputs the oracle computes one by one.
# Leg A is the call and the launch configuration bench.py times: dycore_step (one fused kernel) with bench.py's
# column padding (whole 128-byte lines: ldk = ldk_w = 96 for 90 fp64 or fp32 levels, 32 for 30 fp64 levels), default
# options (the pacing barrier armed at its default period), two alternating inputs. Leg B is the two separate
# entry points of SURVEY.md 8(b) with unpadded columns.
# ----------------------------------------------------------------------------------------------
def _need_host_gb(gb):
    import psutil
    avail = psutil.virtual_memory().available / 2 ** 30
    if avail < gb:
        pytest.skip("needs %.0f GB of host memory, %.0f GB available" % (gb, avail))


def bench_padding(nlev, f32):
    """the leading dimensions bench.py uses (columns padded to whole 128-byte lines)"""
    line = 32 if f32 else 16
    return (nlev + line - 1) // line * line, (nlev + 1 + line - 1) // line * line


def _sampled_check(torch, o, tag, config, outs, sizes, nlev, vn64, w64, zh, tol, nsamp, seed):
    dev = outs[0].device
    for what, arr, n in zip(("ddt_vn", "div", "vort"), outs, sizes):
        idx, lev = si.sample_points(seed, n, nlev, nsamp)
        got = arr[torch.from_numpy(idx).to(dev), torch.from_numpy(lev.astype(np.int64)).to(dev)].cpu().numpy().astype(np.float64)
        want, m = o.sample(what, idx, lev, vn64, nlev, w=w64, z_half=zh)
        err = np.abs(got - want)
        assert (err <= tol * m).all(), "%s %s config %d: worst err/M %.3e" % (tag, what, config, (err / m).max())
        # properties that hold at any size: every level of every column was written, no pad was touched
        assert not torch.isnan(arr[:, :nlev]).any(), (tag, what)
        if arr.shape[1] > nlev:
            assert torch.isnan(arr[:, nlev:]).all(), (tag, what)


@pytest.mark.slow
@pytest.mark.parametrize("config,host_gb", [(2, 6), (3, 60), (4, 40), (5, 90)])
def test_full_size_sampled(torch_cuda, lib, oracle_mod, config, host_gb):
    torch = torch_cuda
    _need_host_gb(host_gb)
    cfg = si.CONFIGS[config]
    flags = 1 if cfg["permute"] else 0
    seed = si.PERMUTE_SEED if cfg["permute"] else 0
    nlev = cfg["nlev"]
    f32 = cfg["dtype"] == "f32"
    tol = TOL[cfg["dtype"]]
    g = lib.IconGrid(cfg["k"], seed, flags)
    og = oracle_mod.Grid(cfg["k"], seed, flags)
    o = og.rounded_f32() if f32 else og
    for name in ("c2e", "e2c", "e2v", "e2e4", "v2e"):          # bit-exact tables at full size
        assert np.array_equal(g.table_host(name), og.table(name)), name
    dev = torch.device("cuda:0")
    sizes = (g.ne, g.nc, g.nv)
    nsamp = 20000

    # ---- leg A: dycore_step as bench.py launches it -------------------------------------------------------
    ldk, ldk_w = bench_padding(nlev, f32)
    vn, w, zh = si.make_fields(config, og.edge_xyz, og.edge_normal, og.nc, ldk=ldk, ldk_w=ldk_w)      # NaN pads
    d_vn, d_w = torch.from_numpy(vn).to(dev), torch.from_numpy(w).to(dev)
    fv, fw = -3.0, 5.0                                            # the second input: a rescaled copy (kept on the device)
    d_vn2, d_w2 = d_vn * fv, d_w * fw

    def fresh():
        return [torch.full((n, ldk), float("nan"), dtype=d_vn.dtype, device=dev) for n in sizes]

    def as64(a):
        return np.nan_to_num(a.astype(np.float64)) if f32 else np.nan_to_num(a)
    vn64, w64 = as64(vn), as64(w)
    first = None
    for it in range(4):                                           # A B A B: a stale slot would carry the OTHER input
        second = it % 2 == 1
        outs = fresh()
        n0 = g.launch_count
        lib.dycore_step(g, zh, d_vn2 if second else d_vn, d_w2 if second else d_w, outs[0], outs[1], outs[2], nlev)
        torch.cuda.synchronize()
        assert g.launch_count - n0 == 1, "dycore_step must be ONE fused kernel at every BASELINE config"
        if second:
            # the rescaled fields in the precision the device holds them (fp32: rounded products)
            v2 = as64(d_vn2.cpu().numpy()) if it == 1 else v2
            w2 = as64(d_w2.cpu().numpy()) if it == 1 else w2
            _sampled_check(torch, o, "step B%d" % it, config, outs, sizes, nlev, v2, w2, zh, tol, nsamp, 400 + config)
        else:
            _sampled_check(torch, o, "step A%d" % it, config, outs, sizes, nlev, vn64, w64, zh, tol, nsamp, 300 + config)
            if first is None:
                first = [t.clone() for t in outs]
            else:                                                 # the kernel is deterministic: bit-identical re-run
                for a, b in zip(first, outs):
                    assert torch.equal(torch.nan_to_num(a), torch.nan_to_num(b))
    if second:
        del v2, w2
    # discrete Gauss on the GPU result (launch A): area-weighted divergence sums to ~0 per level
    a_c = torch.from_numpy(og.a_c).to(dev).to(torch.float64)
    l_e = torch.from_numpy(og.l_e).to(dev).to(torch.float64)
    num = (a_c[:, None] * first[1][:, :nlev].to(torch.float64)).sum(0).abs()
    den = (l_e[:, None] * d_vn[:, :nlev].to(torch.float64).abs()).sum(0)
    assert (num / den).max().item() < (1e-6 if f32 else 1e-13)
    del first, outs, d_vn, d_w, d_vn2, d_w2, vn, w, vn64, w64
    torch.cuda.empty_cache()

    # ---- leg B: the two entry points of SURVEY.md 8(b), unpadded columns ----------------------------------
    ldk = 92 if f32 else nlev            # fp32: ldk*4 must be a multiple of 16
    ldk_w = 92 if f32 else nlev + 1 + (nlev + 1) % 2
    vn, w, zh = si.make_fields(config, og.edge_xyz, og.edge_normal, og.nc, ldk=ldk, ldk_w=ldk_w)
    d_vn, d_w = torch.from_numpy(vn).to(dev), torch.from_numpy(w).to(dev)
    outs = fresh()
    lib.dycore_velocity_tendencies(g, zh, d_vn, d_w, outs[0], nlev)
    lib.dycore_div_vort(g, d_vn, outs[1], outs[2], nlev)
    torch.cuda.synchronize()
    _sampled_check(torch, o, "two calls", config, outs, sizes, nlev, as64(vn), as64(w), zh, tol, nsamp, 300 + config)
    # ---- leg C: the vertical-wind tendency on the same fields ----------------------------
    ddt_w = torch.full((g.nc, ldk_w), float("nan"), dtype=d_vn.dtype, device=dev)
    lib.dycore_w_tendency(g, zh, d_vn, d_w, ddt_w, nlev)
    torch.cuda.synchronize()
    idx, lev = si.sample_points(500 + config, g.nc, nlev + 1, nsamp)
    got = ddt_w[torch.from_numpy(idx).to(dev), torch.from_numpy(lev.astype(np.int64)).to(dev)].cpu().numpy().astype(np.float64)
    want, m = o.sample("ddt_w", idx, lev, as64(vn), nlev, w=as64(w), z_half=zh)
    err = np.abs(got - want)
    assert (err <= tol * m).all(), "ddt_w config %d: worst err/M %.3e" % (config, (err / np.maximum(m, 1e-300)).max())
    assert not torch.isnan(ddt_w[:, :nlev + 1]).any()
    if ldk_w > nlev + 1:
        assert torch.isnan(ddt_w[:, nlev + 1:]).all()
    # the same from the fused pass (dycore_step_w: one kernel, four outputs)
    outs = fresh()
    ddt_w2 = torch.full((g.nc, ldk_w), float("nan"), dtype=d_vn.dtype, device=dev)
    n0 = g.launch_count
    lib.dycore_step_w(g, zh, d_vn, d_w, outs[0], outs[1], outs[2], ddt_w2, nlev)
    torch.cuda.synchronize()
    assert g.launch_count - n0 == 1
    _sampled_check(torch, o, "step_w", config, outs, sizes, nlev, as64(vn), as64(w), zh, tol, nsamp, 300 + config)
    got2 = ddt_w2[torch.from_numpy(idx).to(dev), torch.from_numpy(lev.astype(np.int64)).to(dev)].cpu().numpy().astype(np.float64)
    assert (np.abs(got2 - want) <= tol * m).all(), "fused ddt_w config %d" % config
    assert not torch.isnan(ddt_w2[:, :nlev + 1]).any()
    del outs, ddt_w, ddt_w2
    torch.cuda.empty_cache()
    # ---- leg D: the metric variant on the same fields, seeded terrain-following levels ----------
    zh_e, zn, zt = si.make_metric_heights(config, og.edge_xyz, og.edge_normal, nlev, ldk, ldk_w, dtype=cfg["dtype"])
    d_zh = torch.from_numpy(zh_e).to(dev)
    del zh_e
    d_wgt = torch.full((g.ne, ldk_w), float("nan"), dtype=d_vn.dtype, device=dev)
    d_inv = torch.full((g.ne, ldk), float("nan"), dtype=d_vn.dtype, device=dev)
    lib.dycore_metric_from_zhalf(g, d_zh, d_wgt, d_inv, nlev)
    del d_zh
    d_zn, d_zt = torch.from_numpy(zn).to(dev), torch.from_numpy(zt).to(dev)
    out = torch.full((g.ne, ldk), float("nan"), dtype=d_vn.dtype, device=dev)
    n0 = g.launch_count
    lib.dycore_velocity_tendencies_metric(g, d_wgt, d_inv, d_zn, d_zt, d_vn, d_w, out, nlev)
    torch.cuda.synchronize()
    assert g.launch_count - n0 == 1
    idx, lev = si.sample_points(600 + config, g.ne, nlev, nsamp)
    got = out[torch.from_numpy(idx).to(dev), torch.from_numpy(lev.astype(np.int64)).to(dev)].cpu().numpy().astype(np.float64)
    # the oracle evaluates on the metrics the device derived (inputs of the operator), pads read as 0
    wgt_h, inv_h = as64(d_wgt.cpu().numpy()), as64(d_inv.cpu().numpy())
    want, m = o.sample_metric(idx, lev, as64(vn), as64(w), wgt_h, inv_h, as64(zn), as64(zt), nlev)
    err = np.abs(got - want)
    assert (err <= tol * m).all(), "metric ddt_vn config %d: worst err/M %.3e" % (config, (err / np.maximum(m, 1e-300)).max())
    assert not torch.isnan(out[:, :nlev]).any()
    if ldk > nlev:
        assert torch.isnan(out[:, nlev:]).all()
    g.close()
