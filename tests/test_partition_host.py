"""Host logic of the horizontal decomposition (reading P-21), on CPU: the local grids the
library builds (ICON_HOST_ONLY) against the oracle's statement of the decomposition (oracle/decomposition.py), and the
exchange plumbing on two gloo ranks. The GPU parity of the local sweep is tests/test_gpu_parity.py."""
import os
import subprocess
import sys

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    import paper_2511_02021_b200 as lib
    lib.load_library()
    return lib


def _parts(lib, k, R):
    return [lib.IconGrid(k, flags=lib.ICON_HOST_ONLY, n_parts=R, part=r) for r in range(R)]


@pytest.mark.parametrize("k,R", [(1, 1), (1, 2), (2, 3), (2, 8), (3, 5), (3, 8), (4, 16)])
def test_local_grids_against_the_oracle_decomposition(lib, oracle_grid, k, R):
    from oracle import decomposition as dd
    og = oracle_grid(k)
    gs = _parts(lib, k, R)
    try:
        info = [g.part_info() for g in gs]
        l2g = [{n: g.part_table("l2g_" + n) for n in ("cell", "edge", "vert")} for g in gs]
        # ---- ownership: every point of the global grid is owned exactly once; cells as P-21 says -----------------------
        edge_owner = np.full(og.ne, -1)
        vert_owner = np.full(og.nv, -1)
        cell_owner = np.full(og.nc, -1)
        for r, (g, i, t) in enumerate(zip(gs, info, l2g)):
            assert (i["n_parts"], i["part"]) == (R, r)
            assert (i["nc_global"], i["ne_global"], i["nv_global"]) == (og.nc, og.ne, og.nv)
            assert (g.nc, g.ne, g.nv) == (i["nc_local"], i["ne_local"], i["nv_owned"])
            assert (len(t["cell"]), len(t["edge"]), len(t["vert"])) == (g.nc, g.ne, g.nv)
            for name, owner, n_owned in (("edge", edge_owner, i["ne_owned"]), ("vert", vert_owner, i["nv_owned"]),
                                         ("cell", cell_owner, i["nc_owned"])):
                mine = t[name][:n_owned]
                assert (np.diff(mine) > 0).all()                       # owned rows in ascending global id
                assert (owner[mine] == -1).all()
                owner[mine] = r
            lo, hi = dd.part_range(og.nc // 4, R, r)
            assert (i["parent_lo"], i["parent_hi"]) == (lo, hi)
        assert (edge_owner >= 0).all() and (vert_owner >= 0).all()
        assert (cell_owner == dd.cell_owner(og.nc, R)).all()
        assert dd.check_ownership(og, R, edge_owner, vert_owner) == []
        # ---- halo: holds every column the owned outputs read (S1-S7), grouped by owner rank, ascending ids --------------
        for r, (g, i, t) in enumerate(zip(gs, info, l2g)):
            need_e, need_c = dd.required_columns(og, t["edge"][:i["ne_owned"]], t["cell"][:i["nc_owned"]], t["vert"])
            assert set(need_e.tolist()) <= set(t["edge"].tolist()), "a vn column the owned outputs read is missing"
            assert set(need_c.tolist()) <= set(t["cell"].tolist()), "a w column the owned outputs read is missing"
            assert len(np.unique(t["edge"])) == g.ne and len(np.unique(t["cell"])) == g.nc
            for name, owner, n_owned in (("edge", edge_owner, i["ne_owned"]), ("cell", cell_owner, i["nc_owned"])):
                rb = g.part_table("recv_begin_" + name)
                assert len(rb) == R + 1 and rb[0] == n_owned and rb[-1] == len(t[name]) and (np.diff(rb) >= 0).all()
                assert rb[r] == rb[r + 1]                               # nothing from myself
                for q in range(R):
                    blk = t[name][rb[q]:rb[q + 1]]
                    assert (owner[blk] == q).all() and (np.diff(blk) > 0).all()
        # ---- exchange lists: what p packs for q is, row by row, what q expects from p ----------------------------------
        for name in ("edge", "cell"):
            for p in range(R):
                sb = gs[p].part_table("send_begin_" + name)
                ids = gs[p].part_table("send_ids_" + name)
                n_owned = info[p]["ne_owned" if name == "edge" else "nc_owned"]
                assert len(sb) == R + 1 and sb[0] == 0 and sb[-1] == len(ids)
                assert (ids >= 0).all() and (ids < n_owned).all()     # only owned rows are sent
                for q in range(R):
                    rb = gs[q].part_table("recv_begin_" + name)
                    sent = l2g[p][name][ids[sb[q]:sb[q + 1]]]
                    want = l2g[q][name][rb[p]:rb[p + 1]]
                    assert (sent == want).all(), (name, p, q)
    finally:
        for g in gs:
            g.close()


def test_local_schedule_replays_and_unsupported_calls_are_rejected(lib):
    """the column-cache schedule built from LOCAL records passes the independent checker; the global tables are gone"""
    g = lib.IconGrid(3, flags=lib.ICON_HOST_ONLY, n_parts=3, part=1)
    try:
        st = g.cc_schedule_check(lib.ICON_F64, 90, 96, 96)
        assert st["steps"] > 0 and st["vn_columns"] >= g.part_info()["ne_owned"]
        st = g.cc_schedule_check(lib.ICON_F32, 30, 32, 32)
        assert st["steps"] > 0
        with pytest.raises(lib.IconError) as ei:
            g.table_host("c2e")
        assert ei.value.code == -4
    finally:
        g.close()
    g = lib.IconGrid(2, flags=lib.ICON_HOST_ONLY)
    try:
        with pytest.raises(lib.IconError):
            g.part_table("l2g_edge")                 # not a local grid
        assert g.part_info()["n_parts"] == 0
    finally:
        g.close()
    for bad in (dict(n_parts=4, part=4), dict(n_parts=4, part=-1), dict(n_parts=81, part=0)):      # R2B1: 80 parents
        with pytest.raises(lib.IconError):
            lib.IconGrid(1, flags=lib.ICON_HOST_ONLY, **bad)
    with pytest.raises(lib.IconError):
        lib.IconGrid(1, flags=lib.ICON_HOST_ONLY | lib.ICON_PERMUTE, n_parts=2, part=0)


def test_halo_fraction_matches_the_two_ring_estimate(lib):
    """a halo two cell rings deep. At R2B5 on 8 ranks the halo is a small fraction of the owned columns"""
    g = lib.IconGrid(5, flags=lib.ICON_HOST_ONLY, n_parts=8, part=3)
    try:
        i = g.part_info()
        assert i["nc_owned"] == 20 * 4 ** 6 // 8
        frac_e = (i["ne_local"] - i["ne_owned"]) / i["ne_owned"]
        frac_c = (i["nc_local"] - i["nc_owned"]) / i["nc_owned"]
        assert 0.0 < frac_e < 0.35 and 0.0 < frac_c < 0.35
    finally:
        g.close()


_WORKER = r"""
import os, sys
sys.path.insert(0, %r)
import numpy as np
import torch
import torch.distributed as dist
import paper_2511_02021_b200 as lib
from paper_2511_02021_b200.halo import HaloExchange
dist.init_process_group("gloo")
rank, world = dist.get_rank(), dist.get_world_size()
g = lib.IconGrid(3, flags=lib.ICON_HOST_ONLY, n_parts=world, part=rank)
hx = HaloExchange(g)
info = g.part_info()
def host_pack(grid, kind, field, send):          # stands in for the CUDA gather kernel: this test is about the plumbing
    ids = grid.part_table("send_ids_edge" if kind == 0 else "send_ids_cell")
    send.copy_(field[torch.from_numpy(ids.astype(np.int64))])
ok = True
for kind, name, n_glob, ld in ((0, "edge", info["ne_global"], 6), (1, "cell", info["nc_global"], 8)):
    l2g = g.part_table("l2g_" + name).astype(np.int64)
    n_owned = hx.n_owned[kind]
    glob = (np.arange(n_glob, dtype=np.float64)[:, None] * 100.0 + np.arange(ld)[None, :])      # value names (row, level)
    field = torch.full((len(l2g), ld), float("nan"), dtype=torch.float64)
    field[:n_owned] = torch.from_numpy(glob[l2g[:n_owned]])
    hx.exchange(field, kind, pack=host_pack)
    ok = ok and bool((field.numpy() == glob[l2g]).all()) and len(l2g) > n_owned
flag = torch.tensor([1.0 if ok else 0.0])
dist.all_reduce(flag, op=dist.ReduceOp.MIN)
if rank == 0:
    print("RESULT %%d %%d" %% (world, int(flag.item())))
g.close()
dist.destroy_process_group()
"""


@pytest.mark.parametrize("world", [2, 3])
def test_exchange_fills_every_halo_row_gloo(tmp_path, world):
    script = tmp_path / "worker.py"
    script.write_text(_WORKER % ROOT)
    env = dict(os.environ, MASTER_ADDR="127.0.0.1", OMP_NUM_THREADS="2")
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", str(world), "--master-addr", "127.0.0.1",
           "--master-port", str(29740 + world), str(script)]
    res = subprocess.run(cmd, cwd=ROOT, env=env, stdout=subprocess.PIPE, stderr=subprocess.PIPE, text=True, timeout=600)
    assert res.returncode == 0, res.stderr[-2000:]
    out = [ln for ln in res.stdout.splitlines() if ln.startswith("RESULT")]
    assert out == ["RESULT %d 1" % world], res.stdout + res.stderr[-1000:]
