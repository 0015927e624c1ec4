"""GPU test of dycore_velocity_tendencies_noalloc (include/icon_dycore.h): the tendency pipeline with its scratch in a
static device array, for callers that cannot call cudaMalloc. Its output is compared with the EXISTING path
(dycore_velocity_tendencies, default kernel) on the same inputs within the tolerance the parity tests use
(|a - b| <= tol * M(p), M(p) from the oracle, reading P-16), on two calls in a row.

The file is named so that pytest collects it last (the suite runs with pytest -x). It depends on nothing another test
file sets up: it passes alone in a fresh process and after the other tests."""
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
    lib.load_library()
    return lib


def _fields(og, cfg, nlev, ldk, ldk_w, dtype, factor):
    vn, w, zh = si.make_fields(cfg, og.edge_xyz, og.edge_normal, og.nc, nlev=nlev, ldk=ldk, ldk_w=ldk_w, dtype=dtype)
    vn = (np.nan_to_num(vn) * factor).astype(vn.dtype)
    return vn, np.nan_to_num(w), zh


def _scale(og, vn, w, zh, nlev, f32):
    o = og.rounded_f32() if f32 else og
    ref = o.velocity_tendencies(vn.astype(np.float64), w.astype(np.float64), zh, nlev, with_scale=True)
    return ref["ddt_vn"], ref["m_ddt"]


def _both_paths(torch, lib, g, vn, w, zh, nlev, sentinel=-31.5):
    dev = torch.device("cuda:0")
    d_vn, d_w = torch.from_numpy(vn).to(dev), torch.from_numpy(w).to(dev)
    new = torch.full(d_vn.shape, sentinel, dtype=d_vn.dtype, device=dev)
    old = torch.full(d_vn.shape, sentinel, dtype=d_vn.dtype, device=dev)
    lib.dycore_velocity_tendencies_noalloc(g, zh, d_vn, d_w, new, nlev)
    lib.dycore_velocity_tendencies(g, zh, d_vn, d_w, old, nlev)
    torch.cuda.synchronize()
    return new.cpu().numpy().astype(np.float64), old.cpu().numpy().astype(np.float64)


@pytest.mark.parametrize("k,nlev,ldk,ldk_w", [(4, 90, 90, 92), (3, 40, 48, 48)])
def test_noalloc_matches_the_existing_path_on_two_calls_in_a_row(torch_cuda, lib, oracle_mod, k, nlev, ldk, ldk_w):
    """R2B4 x 90 fp64 with ldk = 90 needs 66.36 MB of the 64 MiB (67.1 MB) array: the largest BASELINE config that fits.
    Two calls in a row on DIFFERENT inputs (the array keeps the first call's intermediates: none of them may leak into the
    second result); each against the existing path and against the oracle; pads of the output stay untouched."""
    torch = torch_cuda
    og = oracle_mod.Grid(k)
    g = lib.IconGrid(k)
    try:
        for cfg, factor in ((1, 1.0), (2, -2.5)):
            vn, w, zh = _fields(og, cfg, nlev, ldk, ldk_w, "f64", factor)
            want, m = _scale(og, vn, w, zh, nlev, False)
            new, old = _both_paths(torch, lib, g, vn, w, zh, nlev)
            err = np.abs(new[:, :nlev] - old[:, :nlev])
            assert (err <= TOL["f64"] * m[:, :nlev]).all(), "vs existing path: worst err/M %.3e" % (err / m[:, :nlev]).max()
            err = np.abs(new[:, :nlev] - want[:, :nlev])
            assert (err <= TOL["f64"] * m[:, :nlev]).all(), "vs oracle: worst err/M %.3e" % (err / m[:, :nlev]).max()
            assert (new[:, nlev:] == -31.5).all()
    finally:
        g.close()


def test_noalloc_stale_scratch_of_another_shape_does_not_leak(torch_cuda, lib, oracle_mod):
    """the second call uses fewer levels and another padding than the first: the scratch layout moves, stale bytes of the
    first call sit where the second call's intermediates go"""
    torch = torch_cuda
    og = oracle_mod.Grid(3)
    g = lib.IconGrid(3)
    try:
        for nlev, ldk, ldk_w, cfg in ((64, 64, 66, 1), (30, 32, 32, 2), (64, 64, 66, 2)):
            vn, w, zh = _fields(og, cfg, nlev, ldk, ldk_w, "f64", 1.0)
            _, m = _scale(og, vn, w, zh, nlev, False)
            new, old = _both_paths(torch, lib, g, vn, w, zh, nlev)
            assert (np.abs(new[:, :nlev] - old[:, :nlev]) <= TOL["f64"] * m[:, :nlev]).all(), nlev
    finally:
        g.close()


def test_noalloc_allocates_no_device_memory(torch_cuda, lib, oracle_mod):
    """free device memory (cudaMemGetInfo) is the same before and after two calls, once the first call on the device has
    resolved the array's address; a fresh grid is used so that no lazily built table exists for these arguments"""
    torch = torch_cuda
    og = oracle_mod.Grid(3)
    g = lib.IconGrid(3)
    try:
        dev = torch.device("cuda:0")
        nlev = 40
        vn, w, zh = _fields(og, 1, nlev, 40, 42, "f64", 1.0)
        d_vn, d_w = torch.from_numpy(vn).to(dev), torch.from_numpy(w).to(dev)
        out = torch.zeros_like(d_vn)
        lib.dycore_velocity_tendencies_noalloc(g, zh, d_vn, d_w, out, nlev)      # address resolution, module load
        torch.cuda.synchronize()
        free0, _ = torch.cuda.mem_get_info()
        n0 = g.launch_count
        zh2 = si.z_half_levels(nlev, h_top=25.0e3)                                # new level heights: still no allocation
        lib.dycore_velocity_tendencies_noalloc(g, zh2, d_vn, d_w, out, nlev)
        lib.dycore_velocity_tendencies_noalloc(g, zh, d_vn, d_w, out, nlev)
        torch.cuda.synchronize()
        free1, _ = torch.cuda.mem_get_info()
        assert free1 == free0, (free0, free1)
        assert g.launch_count - n0 == 8                                           # 2 x (coefficients + three pipeline kernels)
        _, m = _scale(og, vn, w, zh, nlev, False)
        ref = torch.zeros_like(d_vn)
        lib.dycore_velocity_tendencies(g, zh, d_vn, d_w, ref, nlev)
        torch.cuda.synchronize()
        assert (np.abs(out.cpu().numpy() - ref.cpu().numpy())[:, :nlev] <= TOL["f64"] * m[:, :nlev]).all()
    finally:
        g.close()


def test_noalloc_fp32_needs_resident_tables_then_matches(torch_cuda, lib, oracle_mod):
    torch = torch_cuda
    og = oracle_mod.Grid(3, si.PERMUTE_SEED, 1)
    g = lib.IconGrid(3, si.PERMUTE_SEED, lib.ICON_PERMUTE)
    try:
        dev = torch.device("cuda:0")
        nlev = 90
        vn, w, zh = _fields(og, 4, nlev, 92, 92, "f32", 1.0)
        assert vn.dtype == np.float32
        d_vn, d_w = torch.from_numpy(vn).to(dev), torch.from_numpy(w).to(dev)
        out = torch.zeros_like(d_vn)
        with pytest.raises(lib.IconError) as ei:                                  # fp32 tables not uploaded yet: it must not allocate
            lib.dycore_velocity_tendencies_noalloc(g, zh, d_vn, d_w, out, nlev)
        assert ei.value.code == -4 and "must not" in str(ei.value)
        _, m = _scale(og, vn, w, zh, nlev, True)
        new, old = _both_paths_after_ordinary_call(torch, lib, g, d_vn, d_w, zh, nlev)
        assert (np.abs(new[:, :nlev] - old[:, :nlev]) <= TOL["f32"] * m[:, :nlev]).all()
    finally:
        g.close()


def _both_paths_after_ordinary_call(torch, lib, g, d_vn, d_w, zh, nlev):
    old = torch.zeros_like(d_vn)
    lib.dycore_velocity_tendencies(g, zh, d_vn, d_w, old, nlev)                   # uploads the fp32 coefficient tables
    new = torch.zeros_like(d_vn)
    lib.dycore_velocity_tendencies_noalloc(g, zh, d_vn, d_w, new, nlev)
    torch.cuda.synchronize()
    return new.cpu().numpy().astype(np.float64), old.cpu().numpy().astype(np.float64)


def test_noalloc_rejects_what_does_not_fit(torch_cuda, lib):
    torch = torch_cuda
    dev = torch.device("cuda:0")
    g = lib.IconGrid(5)                     # R2B5 x 90 fp64 needs ~265 MB of scratch
    try:
        vn = torch.zeros((g.ne, 90), dtype=torch.float64, device=dev)
        w = torch.zeros((g.nc, 92), dtype=torch.float64, device=dev)
        out = torch.zeros_like(vn)
        with pytest.raises(lib.IconError) as ei:
            lib.dycore_velocity_tendencies_noalloc(g, si.z_half_levels(90), vn, w, out, 90)
        assert ei.value.code == -1 and "ICON_NOALLOC_SCRATCH_BYTES" in str(ei.value) and str(lib.binding.NOALLOC_SCRATCH_BYTES) in str(ei.value)
    finally:
        g.close()
    g = lib.IconGrid(1)
    try:
        vn = torch.zeros((g.ne, 130), dtype=torch.float64, device=dev)
        w = torch.zeros((g.nc, 132), dtype=torch.float64, device=dev)
        with pytest.raises(lib.IconError):          # nlev > 128: the level coefficients no longer fit the kernel argument
            lib.dycore_velocity_tendencies_noalloc(g, si.z_half_levels(130), vn, w, torch.zeros_like(vn), 130)
        vn = torch.zeros((g.ne, 6), dtype=torch.float64, device=dev)
        w = torch.zeros((g.nc, 8), dtype=torch.float64, device=dev)
        with pytest.raises(lib.IconError):          # output aliases an input
            lib.dycore_velocity_tendencies_noalloc(g, si.z_half_levels(6), vn, w, vn, 6)
    finally:
        g.close()
