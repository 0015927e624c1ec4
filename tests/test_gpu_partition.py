"""GPU parity of the DECOMPOSED sweep (reading P-21): every rank's local grid runs the
library's kernels on ONE GPU, rank after rank (no kernel waits on another), with the halo rows filled by the library's
pack kernel and a device copy standing in for the transport (the transport itself, all_to_all_single, is covered on
gloo ranks in tests/test_partition_host.py). The union of the owned outputs must equal the GLOBAL oracle's result within
the parity tolerance: a missing halo column, a wrong local id or a wrong send list all show up as a wrong number."""
import numpy as np
import pytest

import seeded_inputs as si
from test_gpu_parity import TOL, oracle_reference

pytestmark = pytest.mark.gpu


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


class Rank:
    """one rank's local grid, fields (owned rows from the global field, halo rows NaN) and tables"""

    def __init__(self, torch, lib, k, R, r, vn, w, dev):
        self.g = lib.IconGrid(k, n_parts=R, part=r)
        self.info = self.g.part_info()
        self.l2g = {n: self.g.part_table("l2g_" + n).astype(np.int64) for n in ("edge", "cell", "vert")}
        self.fields = []
        for kind, (name, glob) in enumerate((("edge", vn), ("cell", w))):
            n_owned = self.info["ne_owned" if kind == 0 else "nc_owned"]
            loc = np.full((len(self.l2g[name]), glob.shape[1]), np.nan, dtype=glob.dtype)
            loc[:n_owned] = glob[self.l2g[name][:n_owned]]
            self.fields.append(torch.from_numpy(loc).to(dev))
        self.tab = {n: self.g.part_table(n) for n in ("recv_begin_edge", "recv_begin_cell", "send_begin_edge", "send_begin_cell")}


def exchange_on_one_gpu(torch, lib, ranks):
    """pack on every rank with the library's kernel, then move block (p -> q) of p's buffer into q's halo rows"""
    for kind, name in enumerate(("edge", "cell")):
        bufs = []
        for rk in ranks:
            f = rk.fields[kind]
            n_send = int(rk.tab["send_begin_" + name][-1])
            b = torch.full((n_send, f.shape[1]), -777.0, dtype=f.dtype, device=f.device)
            n0 = rk.g.launch_count
            lib.dycore_halo_pack(rk.g, kind, f, b)
            assert rk.g.launch_count - n0 == (1 if n_send else 0)
            bufs.append(b)
        torch.cuda.synchronize()
        for p, rp in enumerate(ranks):
            sb = rp.tab["send_begin_" + name]
            for q, rq in enumerate(ranks):
                rb = rq.tab["recv_begin_" + name]
                assert sb[q + 1] - sb[q] == rb[p + 1] - rb[p]
                rq.fields[kind][rb[p]:rb[p + 1]] = bufs[p][sb[q]:sb[q + 1]]
    torch.cuda.synchronize()


def gather_owned(ranks, name, n_owned_key, outs, n_glob):
    """global array assembled from the owned rows of every rank; every global row must be written exactly once"""
    ld = outs[0].shape[1]
    glob = np.full((n_glob, ld), np.nan)
    seen = np.zeros(n_glob, dtype=np.int64)
    for rk, o in zip(ranks, outs):
        n = rk.info[n_owned_key]
        rows = rk.l2g[name][:n]
        glob[rows] = o[:n]
        seen[rows] += 1
    assert (seen == 1).all()
    return glob


@pytest.mark.parametrize("k,R,nlev,ldk,ldk_w,dtype,cfg", [
    (4, 8, 90, 96, 96, "f64", 1), (4, 3, 90, 90, 92, "f64", 1), (3, 5, 30, 32, 32, "f64", 2), (3, 2, 64, 64, 66, "f64", 1),
    (4, 8, 90, 96, 96, "f32", 1), (2, 80, 33, 34, 34, "f64", 1), (3, 1, 40, 40, 42, "f64", 1), (5, 148, 90, 96, 96, "f64", 1)])
def test_decomposed_step_equals_the_global_oracle(torch_cuda, lib, oracle_grid, k, R, nlev, ldk, ldk_w, dtype, cfg):
    """dycore_step on every local grid after the exchange; R = 80 at R2B2 gives ranks of four parent triangles (fewer
    patches than SMs, halo larger than the interior) -- here ONE parent per rank; R = 148 at R2B5 is 34 or 35 parents per
    rank; R = 1 has no halo"""
    torch = torch_cuda
    dev = torch.device("cuda:0")
    og = oracle_grid(k)
    f32 = dtype == "f32"
    vn, w, zh = si.make_fields(cfg, og.edge_xyz, og.edge_normal, og.nc, nlev=nlev, ldk=ldk, ldk_w=ldk_w, dtype=dtype)
    vn, w = np.nan_to_num(vn), np.nan_to_num(w)          # pads 0: whole rows travel, NaN pads would be equal anyway
    ref = oracle_reference(og, vn, w, zh, nlev, f32)
    ranks = [Rank(torch, lib, k, R, r, vn, w, dev) for r in range(R)]
    try:
        exchange_on_one_gpu(torch, lib, ranks)
        tdt = ranks[0].fields[0].dtype
        sentinel = -1234.5
        res = {"ddt_vn": [], "div": [], "vort": []}
        for rk in ranks:
            g = rk.g
            # after the exchange every local row holds its global row: the halo is complete
            assert torch.equal(rk.fields[0], torch.from_numpy(vn[rk.l2g["edge"]]).to(dev))
            assert torch.equal(rk.fields[1], torch.from_numpy(w[rk.l2g["cell"]]).to(dev))
            outs = [torch.full((n, ldk), sentinel, dtype=tdt, device=dev) for n in (g.ne, g.nc, g.nv)]
            n0 = g.launch_count
            lib.dycore_step(g, zh, rk.fields[0], rk.fields[1], outs[0], outs[1], outs[2], nlev)
            torch.cuda.synchronize()
            assert g.launch_count - n0 == 1                                   # the fused column-cache kernel
            for name, o, n_owned in zip(("ddt_vn", "div", "vort"), outs, (rk.info["ne_owned"], rk.info["nc_owned"], rk.info["nv_owned"])):
                a = o.cpu().numpy()
                assert (a[n_owned:] == sentinel).all(), name + ": a halo row of an output was written"
                assert (a[:n_owned, nlev:] == sentinel).all() and not (a[:n_owned, :nlev] == sentinel).any(), name
                res[name].append(a.astype(np.float64))
        tol = TOL[dtype]
        for name, key, n_owned_key, n_glob, want, scale in (
                ("ddt_vn", "edge", "ne_owned", og.ne, ref["ddt_vn"], ref["m_ddt"]),
                ("div", "cell", "nc_owned", og.nc, ref["div"], ref["m_div"]),
                ("vort", "vert", "nv_owned", og.nv, ref["vort_dv"], ref["m_vort"])):
            got = gather_owned(ranks, key, n_owned_key, res[name], n_glob)
            err = np.abs(got[:, :nlev] - want[:, :nlev])
            assert (err <= tol * scale[:, :nlev]).all(), "%s: worst err/M %.3e" % (name, (err / np.maximum(scale[:, :nlev], 1e-300)).max())
    finally:
        for rk in ranks:
            rk.g.close()


def test_decomposed_other_calls_and_rejections(torch_cuda, lib, oracle_grid):
    """on one rank of three: the separate calls (tendency, div / vort), the fused step with ddt_w and the metric variant
    against the global oracle on the owned rows; calls that need the global tables are refused"""
    torch = torch_cuda
    dev = torch.device("cuda:0")
    k, R, r, nlev, ldk, ldk_w = 3, 3, 1, 60, 64, 64
    og = oracle_grid(k)
    vn, w, zh = si.make_fields(2, og.edge_xyz, og.edge_normal, og.nc, nlev=nlev, ldk=ldk, ldk_w=ldk_w, dtype="f64")
    vn, w = np.nan_to_num(vn), np.nan_to_num(w)
    ref = oracle_reference(og, vn, w, zh, nlev, False)
    want_w, m_w = og.w_tendency(vn, w, zh, nlev, with_scale=True)
    g = lib.IconGrid(k, n_parts=R, part=r)
    try:
        i = g.part_info()
        le, lc, lv = (g.part_table("l2g_" + n).astype(np.int64) for n in ("edge", "cell", "vert"))
        d_vn, d_w = torch.from_numpy(vn[le]).to(dev), torch.from_numpy(w[lc]).to(dev)      # halo filled from the global field
        ne_o, nc_o = i["ne_owned"], i["nc_owned"]

        def close(name, got, want, scale, rows, n, nl):
            err = np.abs(got[:n, :nl] - want[rows[:n], :nl])
            assert (err <= 1e-12 * scale[rows[:n], :nl]).all(), name

        ddt, div, vort = (torch.zeros((n, ldk), dtype=torch.float64, device=dev) for n in (g.ne, g.nc, g.nv))
        lib.dycore_velocity_tendencies(g, zh, d_vn, d_w, ddt, nlev)
        lib.dycore_div_vort(g, d_vn, div, vort, nlev)
        torch.cuda.synchronize()
        close("ddt_vn", ddt.cpu().numpy(), ref["ddt_vn"], ref["m_ddt"], le, ne_o, nlev)
        close("div", div.cpu().numpy(), ref["div"], ref["m_div"], lc, nc_o, nlev)
        close("vort", vort.cpu().numpy(), ref["vort_dv"], ref["m_vort"], lv, g.nv, nlev)
        ddt2, div2, vort2 = torch.zeros_like(ddt), torch.zeros_like(div), torch.zeros_like(vort)
        ddw = torch.zeros((g.nc, ldk_w), dtype=torch.float64, device=dev)
        lib.dycore_step_w(g, zh, d_vn, d_w, ddt2, div2, vort2, ddw, nlev)
        torch.cuda.synchronize()
        close("step_w ddt_vn", ddt2.cpu().numpy(), ref["ddt_vn"], ref["m_ddt"], le, ne_o, nlev)
        close("ddt_w", ddw.cpu().numpy(), want_w, m_w, lc, nc_o, nlev + 1)
        # metric variant: per-edge metric fields are local rows like every edge field
        zh_e, zn, zt = si.make_metric_heights(2, og.edge_xyz, og.edge_normal, nlev, ldk, ldk_w, dtype="f64", pad_value=0.0)
        from oracle import metric_from_zhalf
        wgt, inv = metric_from_zhalf(zh_e, nlev, ldk)
        wantm = og.velocity_tendencies_metric(vn, w, wgt, inv, zn, zt, nlev, with_scale=True)
        d_wgt, d_inv = torch.zeros((g.ne, ldk_w), dtype=torch.float64, device=dev), torch.zeros((g.ne, ldk), dtype=torch.float64, device=dev)
        lib.dycore_metric_from_zhalf(g, torch.from_numpy(zh_e[le]).to(dev), d_wgt, d_inv, nlev)
        ddt3 = torch.zeros_like(ddt)
        lib.dycore_velocity_tendencies_metric(g, d_wgt, d_inv, torch.from_numpy(zn[le]).to(dev), torch.from_numpy(zt[le]).to(dev), d_vn, d_w, ddt3, nlev)
        torch.cuda.synchronize()
        close("metric ddt_vn", ddt3.cpu().numpy(), wantm["ddt_vn"], wantm["m_ddt"], le, ne_o, nlev)
        # refused: everything that needs the global tables
        ddw2 = torch.zeros_like(ddw)
        lib.dycore_w_tendency(g, zh, d_vn, d_w, ddw2, nlev)                 # the column cache's ddt_w mode: runs on a local grid
        torch.cuda.synchronize()
        close("w_tendency", ddw2.cpu().numpy(), want_w, m_w, lc, nc_o, nlev + 1)
        for call in (lambda: lib.dycore_velocity_tendencies(g, zh, d_vn, d_w, ddt, nlev, vt=torch.zeros_like(ddt)),
                     lambda: lib.dycore_velocity_tendencies_noalloc(g, zh, d_vn, d_w, ddt, nlev),
                     lambda: g.table_device("c2e")):
            with pytest.raises(lib.IconError) as ei:
                call()
            assert ei.value.code == -4
        g.set_option(lib.ICON_OPT_TENDENCY_KERNEL, 0)
        with pytest.raises(lib.IconError):
            lib.dycore_step(g, zh, d_vn, d_w, ddt, div, vort, nlev)
        g.set_option(lib.ICON_OPT_TENDENCY_KERNEL, 5)
        big = 130                       # a level count the column cache cannot hold: no fallback on a local grid
        v2 = torch.zeros((g.ne, big), dtype=torch.float64, device=dev)
        w2 = torch.zeros((g.nc, big + 2), dtype=torch.float64, device=dev)
        with pytest.raises(lib.IconError) as ei:
            lib.dycore_step(g, si.z_half_levels(big), v2, w2, torch.zeros_like(v2), torch.zeros((g.nc, big), dtype=torch.float64, device=dev),
                            torch.zeros((g.nv, big), dtype=torch.float64, device=dev), big)
        assert ei.value.code == -4
    finally:
        g.close()


@pytest.mark.slow
@pytest.mark.parametrize("config,R,parts,host_gb", [(2, 8, tuple(range(8)), 6), (3, 8, (5,), 60), (3, 64, (0, 63), 60)])
def test_full_size_decomposed_sampled(torch_cuda, lib, oracle_mod, config, R, parts, host_gb):
    """ranks of eight (all eight at config 2, one at config 3) and the first and last rank of sixty-four at config 3, at
    BASELINE.json's sizes in the launch configuration `bench.py --parts R` times (padded leading dimensions, halo rows
    holding the owners' values): the owned outputs on sampled points the oracle computes one by one, the properties that
    hold at any size (every owned level written once, no halo row and no pad written), and, where every rank ran, that
    each output row of the global grid was produced by exactly one rank"""
    import psutil
    torch = torch_cuda
    if psutil.virtual_memory().available / 2 ** 30 < host_gb:
        pytest.skip("needs %d GB of host memory" % host_gb)
    from test_gpu_parity import bench_padding
    cfg = si.CONFIGS[config]
    nlev = cfg["nlev"]
    dev = torch.device("cuda:0")
    og = oracle_mod.Grid(cfg["k"])
    ldk, ldk_w = bench_padding(nlev, False)
    vn, w, zh = si.make_fields(config, og.edge_xyz, og.edge_normal, og.nc, ldk=ldk, ldk_w=ldk_w, pad_value=0.0)
    seen = [np.zeros(n, dtype=np.int64) for n in (og.ne, og.nc, og.nv)]
    for part in parts:
        g = lib.IconGrid(cfg["k"], n_parts=R, part=part)
        try:
            i = g.part_info()
            assert (i["nc_global"], i["ne_global"]) == (og.nc, og.ne) and i["nc_owned"] == og.nc // R
            l2g = [g.part_table("l2g_" + n).astype(np.int64) for n in ("edge", "cell", "vert")]
            d_vn, d_w = torch.from_numpy(vn[l2g[0]]).to(dev), torch.from_numpy(w[l2g[1]]).to(dev)
            sent = float("nan")
            outs = [torch.full((n, ldk), sent, dtype=torch.float64, device=dev) for n in (g.ne, g.nc, g.nv)]
            n0 = g.launch_count
            lib.dycore_step(g, zh, d_vn, d_w, outs[0], outs[1], outs[2], nlev)
            torch.cuda.synchronize()
            assert g.launch_count - n0 == 1
            for k_, (what, arr, rows, n_owned) in enumerate(zip(("ddt_vn", "div", "vort"), outs, l2g, (i["ne_owned"], i["nc_owned"], i["nv_owned"]))):
                idx, lev = si.sample_points(900 + config + part, n_owned, nlev, 20000 if len(parts) < 4 else 4000)
                got = arr[torch.from_numpy(idx).to(dev), torch.from_numpy(lev.astype(np.int64)).to(dev)].cpu().numpy()
                want, m = og.sample(what, rows[idx], lev, vn, nlev, w=w, z_half=zh)
                err = np.abs(got - want)
                assert (err <= 1e-12 * m).all(), "%s config %d part %d: worst err/M %.3e" % (what, config, part, (err / m).max())
                assert not torch.isnan(arr[:n_owned, :nlev]).any(), what
                assert torch.isnan(arr[n_owned:]).all() and torch.isnan(arr[:, nlev:]).all(), what
                seen[k_][rows[:n_owned]] += 1
            del outs, d_vn, d_w
        finally:
            g.close()
    if len(parts) == R:         # every rank ran: each output row of the global grid was produced by exactly one of them
        for sarr in seen:
            assert (sarr == 1).all()
    else:
        for sarr in seen:
            assert sarr.max() == 1
