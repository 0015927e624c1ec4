"""CPU-only tests of the C-ABI library: it loads, exports every symbol include/icon_dycore.h declares,
its host-side grid generator reproduces the oracle's tables bit-for-bit (two different algorithms,
SURVEY.md section 8(c) P-18 / test tier T2), and compute calls fail loudly without a GPU."""
import ctypes
import os
import re

import numpy as np
import pytest

import paper_2511_02021_b200 as lib
from paper_2511_02021_b200 import binding

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def L():
    from paper_2511_02021_b200 import build
    build.build()
    return lib.load_library()


def test_exports_every_declared_symbol(L):
    header = open(os.path.join(ROOT, "include", "icon_dycore.h")).read()
    header = re.sub(r"/\*.*?\*/", "", header, flags=re.S)
    declared = set(re.findall(r"\b((?:icon|dycore)_[a-z_0-9]+)\s*\(", header))
    assert declared == set(binding.EXPORTS)
    for name in declared:
        assert getattr(L, name) is not None
    # table selectors in the header and in the binding agree
    tabs = re.findall(r"ICON_TAB_([A-Z0-9_]+)", header)
    tabs = [t.lower() for t in tabs if t != "COUNT"]
    assert tuple(tabs) == binding.TABLES


@pytest.mark.parametrize("k,seed,flags", [(0, 0, 0), (1, 0, 0), (2, 0, 0), (3, 0, 0), (4, 0, 0), (5, 0, 0),
                                          (2, 4, 1), (4, 4, 1), (3, 99, 1)])
def test_tables_bit_exact_and_geometry_close(L, oracle_mod, k, seed, flags):
    g = lib.IconGrid(k, seed, flags | lib.ICON_HOST_ONLY)
    o = oracle_mod.Grid(k, seed, flags)
    assert (g.nc, g.ne, g.nv) == (o.nc, o.ne, o.nv)
    for name in lib.TABLES:
        a, b = g.table_host(name), o.table(name)
        assert a.shape == b.shape and a.dtype == b.dtype, name
        if a.dtype.kind == "i":
            assert (a == b).all(), name                       # bit-exact index / sign tables
        else:
            scale = np.abs(b).max()
            assert np.abs(a - b).max() <= 1e-12 * scale, name  # P-18: geometry at 1e-12 relative
    g.close()


def test_no_cpu_fallback_and_argument_errors(L):
    g = lib.IconGrid(1, 0, lib.ICON_HOST_ONLY)
    dummy = np.zeros(64)
    p = ctypes.c_void_p(dummy.ctypes.data)
    rc = L.dycore_div_vort(g._h, 0, 4, 4, p, p, p, None)
    assert rc == binding.ICON_ECUDA                           # host-only grid: no device tables, no CPU path
    assert b"no CPU path" in L.icon_last_error()
    z = np.linspace(1.0, 0.0, 5)
    rc = L.dycore_velocity_tendencies(g._h, 0, 4, 4, 5, ctypes.c_void_p(z.ctypes.data), p, p, p, None, None, None, None)
    assert rc == binding.ICON_ECUDA
    rc = L.icon_grid_table_device(g._h, 0, 0, ctypes.byref(ctypes.c_void_p()))
    assert rc == binding.ICON_EUNSUPPORTED
    h = ctypes.c_void_p()
    assert L.icon_grid_create(10, 0, 4, ctypes.byref(h)) == binding.ICON_EINVAL
    assert L.icon_grid_create(-1, 0, 4, ctypes.byref(h)) == binding.ICON_EINVAL
    assert L.icon_grid_create(1, 0, 1 << 10, ctypes.byref(h)) == binding.ICON_EINVAL
    assert L.icon_grid_create(1, 0, 4, None) == binding.ICON_EINVAL
    assert L.dycore_div_vort(None, 0, 4, 4, p, p, p, None) == binding.ICON_EINVAL
    assert L.icon_grid_set_option(g._h, 99, 0) == binding.ICON_EINVAL
    with pytest.raises(lib.IconError):
        g.table_device("c2e")
    g.close()


def test_create_without_device_fails_loudly(L):
    import torch
    if torch.cuda.is_available():
        pytest.skip("a CUDA device is present")
    h = ctypes.c_void_p()
    rc = L.icon_grid_create(0, 0, 0, ctypes.byref(h))
    assert rc == binding.ICON_ECUDA and not h.value
    assert b"no CPU fallback" in L.icon_last_error()


@pytest.mark.parametrize("k,seed,flags", [(0, 0, 0), (1, 0, 0), (2, 0, 0), (3, 0, 0), (5, 0, 0), (6, 0, 0),
                                          (2, 4, 1), (4, 4, 1)])
def test_patch_records_cover_the_grid(L, k, seed, flags):
    """host logic of the fused kernel (the internal work-list): every group of four sibling cells
    passes the local-topology checks of csrc/sc_tables.cpp (canonical and permuted ids; a grid that is not a 4-child
    bisection hierarchy, or a vertex no patch owns, is an error there), and the schedule built on the records replays"""
    g = lib.IconGrid(k, seed, flags | lib.ICON_HOST_ONLY)
    st = g.cc_schedule_check(0, 90, 96, 96)
    assert st["steps"] >= -(-(g.nc // 4) // 4) and st["ctas"] >= 1
    g.close()


# ----------------------------------------------------------------------------------------------
# column-cache schedule of tendency kernel 4 (host logic): built for a B200-sized device and
# replayed by the independent checker of cc_schedule_check.cpp
# ----------------------------------------------------------------------------------------------
@pytest.mark.parametrize("k,seed,flags", [(0, 0, 0), (2, 0, 0), (4, 0, 0), (3, 4, 1)])
def test_cc_schedule_replays_correctly(k, seed, flags):
    g = lib.IconGrid(k, seed, flags | binding.ICON_HOST_ONLY)
    for dtype, nlev, ldk, ldk_w in ((0, 90, 96, 96), (0, 90, 90, 92), (1, 90, 92, 92), (1, 90, 96, 96), (0, 30, 30, 32), (0, 30, 32, 32),
                                    (0, 2, 2, 4), (0, 65, 66, 66)):
        for tile in (16, 0, 64, -1):
            g.set_option(lib.ICON_OPT_CC_TILE, tile)
            st = g.cc_schedule_check(dtype, nlev, ldk, ldk_w, n_ctas=148, smem_bytes=232448)
            np_ = g.nc // 4
            group = 8 if nlev + 1 <= 32 else 4      # shallow columns: two patches per warp, eight per step (reported: the tendency schedule)
            eff = tile if tile >= 0 else (16 if (dtype == 0 and nlev + 1 > 32) else 64)
            assert st["ctas"] == min(148, -(-np_ // (eff or group)))
            assert st["steps"] >= -(-np_ // group)
            # every patch needs its 36 + 7 columns at least once per CTA range, never more than 43 per patch
            assert 6 * np_ <= st["vn_columns"] <= 36 * np_ and 4 * np_ <= st["w_columns"] <= 7 * np_
            assert st["copies"] <= st["vn_columns"] + st["w_columns"]
    g.close()


def test_cc_schedule_merges_runs_on_the_canonical_grid():
    """generation-order numbering: consecutive column ids arrive as one bulk copy when the column stride allows
    (stride == slot size, i.e. columns padded to whole 128-byte lines as bench.py pads them)"""
    g = lib.IconGrid(4, 0, binding.ICON_HOST_ONLY)
    merged = g.cc_schedule_check(0, 90, 96, 96)
    single = g.cc_schedule_check(0, 90, 90, 92)
    assert merged["slot_bytes"] == 768 and single["slot_bytes"] == 736
    assert merged["copies"] < 0.7 * single["copies"]
    assert single["copies"] >= single["vn_columns"]      # vn stride 720 != slot 736: one copy per vn column (w, stride 736, still merges)
    # a small device: fewer CTAs, fewer slots -> still a valid schedule, or a clean refusal
    small = g.cc_schedule_check(0, 90, 96, 96, n_ctas=4, smem_bytes=120000)
    assert small["ctas"] == 4 and small["slots"] < merged["slots"]
    with pytest.raises(lib.IconError):
        g.cc_schedule_check(0, 90, 96, 96, n_ctas=4, smem_bytes=40000)
    with pytest.raises(lib.IconError):
        g.cc_schedule_check(0, 200, 200, 202)        # nlev the kernel does not hold
    g.close()


def test_binding_rejects_malformed_fields_before_the_library_sees_them():
    """the ctypes binding only marshals, but it refuses what would become an illegal address or an out-of-bounds write:
    host tensors, non-contiguous views, wrong row counts, mismatched leading dimensions or dtypes"""
    import torch
    g = lib.IconGrid(1, 0, binding.ICON_HOST_ONLY)
    zh = np.linspace(3.0, 0.0, 5)
    vn, w = torch.zeros((g.ne, 4), dtype=torch.float64), torch.zeros((g.nc, 6), dtype=torch.float64)
    out = torch.zeros((g.ne, 4), dtype=torch.float64)
    with pytest.raises(TypeError):                      # host tensors: there is no CPU path
        lib.dycore_velocity_tendencies(g, zh, vn, w, out, 4)
    with pytest.raises(TypeError):
        lib.dycore_div_vort(g, vn, torch.zeros((g.nc, 4), dtype=torch.float64), torch.zeros((g.nv, 4), dtype=torch.float64), 4)
    with pytest.raises(ValueError):                     # z_half of the wrong length
        lib.dycore_step(g, zh[:-1], vn, w, out, out, out, 4)
    g.close()
