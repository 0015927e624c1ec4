#!/usr/bin/env python
"""bench.py -- the headline measurement (BASELINE.json metric): ddt_vn edge-level points/s and
achieved HBM GB/s of the dycore sweep on one B200.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config 3] [--impl ours|reference]

One "step" = one pass of the whole hot path = one dycore_step call (ddt_vn, div and
vort; a single fused kernel where the column-cache kernel runs, else dycore_velocity_tendencies + dycore_div_vort
back to back; the two entry points are also timed on their own) on seeded synthetic fields (DESIGN.md
section 4) of BASELINE.json configs[2] (R2B8 x 90 levels fp64, the headline roofline config) unless
--config says otherwise. Prints ONE JSON line (rank 0). The path does not shard ("replicas only",
DESIGN.md section 9): with N > 1 every rank runs an independent replica on its own GPU.

--impl reference times the oracle (oracle/, plain C loops) on the host cores on a bounded sample
of the same workload; it is a deliberately slow program, not a target.
"""
import argparse
import json
import os
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

import seeded_inputs as si  # noqa: E402

METRIC = "ddt_vn edge-level points/s"
UNIT = "Gpts/s"
FALLBACK_HBM_GBS = 6650.0     # /opt/skills/guides/B200_PROFILING.md fallback, used only if MEASURED_PEAKS.json is absent


def workload_name(config):
    c = si.CONFIGS[config]
    return "config%d: R2B%d x %d levels %s%s" % (config, c["k"], c["nlev"], c["dtype"], " permuted" if c["permute"] else "")


def algorithmic_bytes(nc, ne, nv, nlev, g):
    """compulsory traffic: every input read once, every output written once,
    one pass over the static tables; g = bytes per floating-point element"""
    tend = (ne * nlev + nc * (nlev + 1) + ne * nlev) * g \
        + ne * (16 + 4 * g + 8 + 8 + g + g + 2 * g) + nc * (12 + 3 * g) + nv * (24 + 6 * g)
    dv = (ne * nlev + nc * nlev + nv * nlev) * g + nc * (12 + 3 * g) + nv * (24 + 6 * g)
    return tend, dv


KERNEL_SOURCES = ("kernels_cc.cu", "cc_schedule.cpp", "cc_schedule.hpp", "sc_tables.cpp", "sc_tables.hpp", "kernels.cu", "api.cu")


def kernel_source_hash():
    """sha256 (16 hex digits) of the sources that decide the kernels' DRAM traffic: profiles/traffic.csv is stamped with
    it, and a capture made from other sources is not reported as this run's traffic"""
    import hashlib
    h = hashlib.sha256()
    for name in KERNEL_SOURCES:
        with open(os.path.join(ROOT, "paper_2511_02021_b200", "csrc", name), "rb") as f:
            h.update(f.read())
    return h.hexdigest()[:16]


def committed_traffic(config, call):
    """ncu dram__bytes_read.sum + dram__bytes_write.sum per launch from profiles/traffic.csv (columns: config, call,
    bytes, capture file, kernel source hash), or (None, why) when the capture was made from other kernel sources"""
    tp = os.path.join(ROOT, "profiles", "traffic.csv")
    if not os.path.exists(tp):
        return None, "profiles/traffic.csv missing"
    try:
        have = kernel_source_hash()
        for ln in open(tp).read().splitlines()[1:]:
            f = [x.strip() for x in ln.split(",")]
            if len(f) >= 5 and f[0] == str(config) and f[1] == call:
                if f[4] != have:
                    return None, "stale: captured from kernel sources %s, this tree is %s" % (f[4], have)
                return int(f[2]), "profiles/%s (ncu --set full, kernel sources %s)" % (f[3], f[4])
    except Exception as e:          # noqa: BLE001
        return None, "unreadable: %s" % e
    return None, "no capture for this config / call"


def peak_hbm_gbs():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        try:
            return float(json.load(open(p))["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
        except Exception:
            pass
    return FALLBACK_HBM_GBS, "fallback (B200_PROFILING.md)"


class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled DURING the timed region"""
    Q = "clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown," \
        "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap,clocks.mem"

    def __init__(self, index):
        self.index, self.proc, self.lines = index, None, []

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.index), "--query-gpu=" + self.Q,
                                          "--format=csv,noheader,nounits", "-lms", "20"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.t = threading.Thread(target=self._read, daemon=True)
            self.t.start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.lines.append(line.strip())

    def wait_first_sample(self, timeout=8.0):
        """nvidia-smi needs up to a second to start on a fresh box: wait for its first line BEFORE the warm-up, so that
        the short timed region is not over before the first sample"""
        t0 = time.perf_counter()
        while self.proc and not self.lines and time.perf_counter() - t0 < timeout:
            time.sleep(0.01)

    def mark_begin(self):
        self.n0 = len(self.lines)

    def mark_end(self):
        time.sleep(0.03)              # a line printed just after the region was sampled inside it
        self.n1 = len(self.lines)

    def stop(self):
        if not self.proc:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except Exception:
            self.proc.kill()
        sm, mx, pw, mem, reasons, capped = [], [], [], [], set(), 0
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        n0, n1 = getattr(self, "n0", 0), getattr(self, "n1", len(self.lines))
        window, note = self.lines[n0:n1], []
        if not window:                # region shorter than one sampling period: the last samples of the warm-up (same load)
            window, note = self.lines[max(0, n0 - 3):n1], ["no sample inside the timed region: last warm-up samples"]
        for ln in window:
            f = [x.strip() for x in ln.split(",")]
            if len(f) < 7:
                continue
            try:
                sm.append(float(f[0])); mx.append(float(f[1])); pw.append(float(f[2]))
            except ValueError:
                continue
            try:
                mem.append(float(f[7]))
            except (IndexError, ValueError):
                pass
            for n, v in zip(names, f[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(n)
                    capped += n == "sw_power_cap"
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "sm_mhz_min": min(sm) if sm else None, "mem_mhz": float(np.median(mem)) if mem else None,
                "power_w_max": max(pw) if pw else None, "power_w_median": float(np.median(pw)) if pw else None,
                "samples": len(sm), "samples_sw_power_cap": capped, "reasons": sorted(reasons) + note}


def max_over_ranks(seconds, device=None):
    """the slowest rank's time: every multi-GPU number is the max over ranks (replicas only: no data-path collective,
    just this one scalar all-reduce after the timed region). Works on any initialised backend (nccl on the GPUs, gloo in
    the CPU test)."""
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return float(seconds)
    tt = torch.tensor([seconds], dtype=torch.float64, device=device)
    dist.all_reduce(tt, op=dist.ReduceOp.MAX)
    return float(tt.item())


def aggregate_value(points_per_rank, seconds_max, world):
    """whole-job throughput in Gpts/s: `world` independent replicas each finish points_per_rank in seconds_max"""
    return world * points_per_rank / seconds_max / 1e9


def oracle_step_seconds(og, vn, w, zh, nlev, reps):
    ts = []
    for _ in range(reps):
        t0 = time.perf_counter()
        og.velocity_tendencies(vn, w, zh, nlev)
        og.div_vort(vn, nlev)
        ts.append(time.perf_counter() - t0)
    return ts


def set_oracle_threads(n):
    """the oracle's loops are OpenMP loops inside oracle/libicon_oracle.so: set the team size of the libgomp it links"""
    import ctypes
    try:
        ctypes.CDLL("libgomp.so.1").omp_set_num_threads(int(n))
        return True
    except OSError:
        return False


def cpu_threads():
    try:
        n = len(os.sched_getaffinity(0))
    except AttributeError:
        n = os.cpu_count() or 1
    env = os.environ.get("OMP_NUM_THREADS")
    return min(n, int(env)) if env and env.isdigit() else n


def oracle_sample(config, k_sample):
    """the oracle on a bounded sample: the same field recipe and level count on a coarser R2Bk grid"""
    import oracle
    cfg = si.CONFIGS[config]
    og = oracle.Grid(k_sample, si.PERMUTE_SEED if cfg["permute"] else 0, 1 if cfg["permute"] else 0)
    vn, w, zh = si.make_fields(config, og.edge_xyz, og.edge_normal, og.nc)
    vn, w = vn.astype(np.float64), w.astype(np.float64)
    if cfg["dtype"] == "f32":
        og = og.rounded_f32()
    return og, vn, w, zh, cfg["nlev"]


def run_reference(args):
    """--impl reference: the oracle, as it stands, on the host cores"""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return 0
    k_sample = min(si.CONFIGS[args.config]["k"], 6)
    og, vn, w, zh, nlev = oracle_sample(args.config, k_sample)
    oracle_step_seconds(og, vn, w, zh, nlev, args.warmup)
    ts = oracle_step_seconds(og, vn, w, zh, nlev, args.steps)
    t = float(np.mean(ts))
    val = og.ne * nlev / t / 1e9
    sample = "R2B%d x %d levels (%d edge-level points per step), same field recipe as %s" % (
        k_sample, nlev, og.ne * nlev, workload_name(args.config))
    line = {"impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": t * 1e3, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": workload_name(args.config), "sample": sample},
            "cpu_baseline": {"value": val, "unit": UNIT, "cores": cpu_threads(), "kind": "oracle", "sample": sample},
            "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line))
    return 0


def run_ours(args):
    import torch
    import torch.distributed as dist
    import paper_2511_02021_b200 as lib

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the product has no CPU path")
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    if world > 1:
        dist.init_process_group("nccl", device_id=dev)
    lib.load_library()

    cfg = si.CONFIGS[args.config]
    nlev = cfg["nlev"]
    f32 = cfg["dtype"] == "f32"
    gsize = 4 if f32 else 8
    # columns padded to whole 128-byte lines so that every 32-level chunk of a column is line aligned
    # (DESIGN.md section 5); the roofline counts the nlev levels only, never the padding
    line = 32 if f32 else 16
    ldk = args.ldk or (nlev + line - 1) // line * line
    ldk_w = args.ldk_w or (nlev + 1 + line - 1) // line * line
    flags = lib.ICON_PERMUTE if cfg["permute"] else 0
    t0 = time.perf_counter()
    g = lib.IconGrid(cfg["k"], si.PERMUTE_SEED if cfg["permute"] else 0, flags)
    if args.variant is not None:
        g.set_option(lib.ICON_OPT_TENDENCY_KERNEL, args.variant)
    if args.cc_tile is not None:
        g.set_option(lib.ICON_OPT_CC_TILE, args.cc_tile)
    if args.cc_pace is not None:
        g.set_option(lib.ICON_OPT_CC_PACE, args.cc_pace)
    t_grid = time.perf_counter() - t0
    vn_h, w_h, zh = si.make_fields(args.config, g.table_host("edge_xyz"), g.table_host("edge_normal"), g.nc,
                                   ldk=ldk, ldk_w=ldk_w, pad_value=0.0)
    tdt = torch.float32 if f32 else torch.float64
    vn = torch.from_numpy(vn_h).to(dev)
    w = torch.from_numpy(w_h).to(dev)
    ddt = torch.zeros((g.ne, ldk), dtype=tdt, device=dev)
    div = torch.zeros((g.nc, ldk), dtype=tdt, device=dev)
    vort = torch.zeros((g.nv, ldk), dtype=tdt, device=dev)
    bytes_tend, bytes_dv = algorithmic_bytes(g.nc, g.ne, g.nv, nlev, gsize)
    l2_flush = None
    if bytes_tend < 512 * 2 ** 20:      # small configs are L2 resident: flush between iterations
        l2_flush = torch.empty(256 * 2 ** 20, dtype=torch.uint8, device=dev)

    def step(ev=None):
        """one pass of the whole hot path: dycore_step (one fused kernel where the column-cache kernel runs)"""
        if l2_flush is not None:
            l2_flush.fill_(1)
        if ev:
            ev[0].record()
        lib.dycore_step(g, zh, vn, w, ddt, div, vort, nlev)
        if ev:
            ev[1].record()

    def step_two_calls(ev):
        """the same outputs through the two separate entry points (reported beside the step)"""
        if l2_flush is not None:
            l2_flush.fill_(1)
        ev[0].record()
        lib.dycore_velocity_tendencies(g, zh, vn, w, ddt, nlev)
        ev[1].record()
        lib.dycore_div_vort(g, vn, div, vort, nlev)
        ev[2].record()

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    sampler = ClockSampler(local)
    if rank == 0:
        sampler.start()
        sampler.wait_first_sample()
    for _ in range(args.warmup):
        step()
    barrier()
    evs = [[torch.cuda.Event(enable_timing=True) for _ in range(2)] for _ in range(args.steps)]
    launches0 = g.launch_count
    barrier()
    sampler.mark_begin()
    for i in range(args.steps):
        step(evs[i])
    barrier()
    sampler.mark_end()
    launches = g.launch_count - launches0
    clocks = sampler.stop() if rank == 0 else None
    fused = launches == args.steps            # one kernel per step
    t_steps = np.array([e[0].elapsed_time(e[1]) for e in evs]) * 1e-3
    t_step = float(t_steps.mean())
    # sampled values of the TIMED output buffers (the last timed launch wrote them), checked against the oracle below
    picks = {}
    if rank == 0 and not args.no_parity_spot:
        for what, arr, n in (("ddt_vn", ddt, g.ne), ("div", div, g.nc), ("vort", vort, g.nv)):
            idx, lev = si.sample_points(700 + args.config, n, nlev, args.spot_points)
            got = arr[torch.from_numpy(idx).to(dev), torch.from_numpy(lev.astype(np.int64)).to(dev)]
            picks[what] = (idx, lev, got.cpu().numpy().astype(np.float64))
    # the two entry points on their own (not part of the headline)
    n2 = max(3, args.steps // 2)
    evs2 = [[torch.cuda.Event(enable_timing=True) for _ in range(3)] for _ in range(n2)]
    for i in range(min(3, n2)):
        step_two_calls(evs2[i])
    barrier()
    for i in range(n2):
        step_two_calls(evs2[i])
    barrier()
    t_tend = np.array([e[0].elapsed_time(e[1]) for e in evs2]) * 1e-3
    t_dv = np.array([e[1].elapsed_time(e[2]) for e in evs2]) * 1e-3
    # the vertical-wind tendency (its own call, not part of the step's value)
    ddt_w = torch.zeros((g.nc, ldk_w), dtype=tdt, device=dev)
    evs3 = [[torch.cuda.Event(enable_timing=True) for _ in range(2)] for _ in range(n2)]
    for i in range(n2 + 2):
        if l2_flush is not None:
            l2_flush.fill_(1)
        ev = evs3[min(i, n2 - 1)]
        ev[0].record()
        lib.dycore_w_tendency(g, zh, vn, w, ddt_w, nlev)
        ev[1].record()
    barrier()
    t_w = np.array([e[0].elapsed_time(e[1]) for e in evs3[:-1] or evs3]) * 1e-3
    bytes_w = (g.ne * nlev + 2 * g.nc * (nlev + 1)) * gsize + g.nc * (12 + 3 * gsize) + g.ne * (8 + gsize)
    # ... and as a by-product of the fused pass (dycore_step_w: one kernel, four outputs)
    evs4 = [[torch.cuda.Event(enable_timing=True) for _ in range(2)] for _ in range(n2)]
    for i in range(n2 + 2):
        if l2_flush is not None:
            l2_flush.fill_(1)
        ev = evs4[min(i, n2 - 1)]
        ev[0].record()
        lib.dycore_step_w(g, zh, vn, w, ddt, div, vort, ddt_w, nlev)
        ev[1].record()
    barrier()
    t_sw = np.array([e[0].elapsed_time(e[1]) for e in evs4[:-1] or evs4]) * 1e-3
    del ddt_w
    # the metric variant of the tendency call (reading P-20) on seeded terrain-following levels
    t_m, bytes_m = None, None
    if not args.no_metric:
        zh_e, zn_h, zt_h = si.make_metric_heights(args.config, g.table_host("edge_xyz"), g.table_host("edge_normal"), nlev, ldk, ldk_w,
                                                  dtype=cfg["dtype"], pad_value=0.0)
        d_zh = torch.from_numpy(zh_e).to(dev)
        d_wgt = torch.zeros((g.ne, ldk_w), dtype=tdt, device=dev)
        d_inv = torch.zeros((g.ne, ldk), dtype=tdt, device=dev)
        lib.dycore_metric_from_zhalf(g, d_zh, d_wgt, d_inv, nlev)           # set-up, untimed (static in a model run)
        del d_zh, zh_e
        d_zn, d_zt = torch.from_numpy(zn_h).to(dev), torch.from_numpy(zt_h).to(dev)
        del zn_h, zt_h
        evs5 = [[torch.cuda.Event(enable_timing=True) for _ in range(2)] for _ in range(n2)]
        for i in range(n2 + 2):
            if l2_flush is not None:
                l2_flush.fill_(1)
            ev = evs5[min(i, n2 - 1)]
            ev[0].record()
            lib.dycore_velocity_tendencies_metric(g, d_wgt, d_inv, d_zn, d_zt, vn, w, ddt, nlev)
            ev[1].record()
        barrier()
        t_m = np.array([e[0].elapsed_time(e[1]) for e in evs5[:-1] or evs5]) * 1e-3
        # the tendency call's bytes + the four metric columns of every edge (wgt_e on nlev+1 half levels) + cgrad
        bytes_m = bytes_tend + g.ne * (3 * nlev + nlev + 1) * gsize + g.ne * 2 * gsize
        del d_wgt, d_inv, d_zn, d_zt
    t_step_max = max_over_ranks(t_step, dev)
    pts = g.ne * nlev
    value = aggregate_value(pts, t_step_max, world)

    # end to end through the C-ABI with HOST buffers (pinned), copies inside the timed region
    e2e = None
    if not args.no_e2e:
        hv, hw = torch.from_numpy(vn_h).pin_memory(), torch.from_numpy(w_h).pin_memory()
        h_ddt = torch.zeros((g.ne, ldk), dtype=tdt).pin_memory()
        h_div = torch.zeros((g.nc, ldk), dtype=tdt).pin_memory()
        h_vort = torch.zeros((g.nv, ldk), dtype=tdt).pin_memory()
        lib.dycore_step_host(g, zh, hv, hw, h_ddt, h_div, h_vort, nlev)
        barrier()
        n_e2e = max(1, min(args.steps, 3))
        t0 = time.perf_counter()
        for _ in range(n_e2e):
            lib.dycore_step_host(g, zh, hv, hw, h_ddt, h_div, h_vort, nlev)
        torch.cuda.synchronize()
        t_e2e = (time.perf_counter() - t0) / n_e2e
        t_e2e = max_over_ranks(t_e2e, dev)
        e2e = {"value": aggregate_value(pts, t_e2e, world), "unit": UNIT,
               "h2d_bytes_per_step": int(hv.numel() + hw.numel()) * gsize,
               "d2h_bytes_per_step": int(h_ddt.numel() + h_div.numel() + h_vort.numel()) * gsize,
               "ms_per_step": t_e2e * 1e3, "steps": n_e2e}
        del hv, hw, h_ddt, h_div, h_vort

    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return 0

    peak, peak_src = peak_hbm_gbs()
    t_tend_avg = float(t_tend.mean())
    # fused step: vn is read ONCE for all three outputs; its compulsory traffic = the tendency call's + div and vort
    # written once + geofac_div (the cell -> edge ids are the patch's own)
    bytes_fused = bytes_tend + (g.nc + g.nv) * nlev * gsize + g.nc * 3 * gsize
    kname = "dycore_step (fused k_tend_cc)" if fused else "dycore_velocity_tendencies"
    kbytes, ktime = (bytes_fused, t_step) if fused else (bytes_tend, t_tend_avg)
    achieved = kbytes / ktime / 1e9
    traffic, traffic_src = committed_traffic(args.config, "dycore_step" if fused else "dycore_velocity_tendencies")
    kt = (t_steps if fused else t_tend) * 1e3            # per-launch times of the dominant kernel, ms
    # fields-only accounting beside the with-tables one (the fused kernel reads patch records, not the plain tables)
    fields_fused = (2 * g.ne * nlev + g.nc * (nlev + 1) + (g.nc + g.nv) * nlev) * gsize
    fields_tend = (2 * g.ne * nlev + g.nc * (nlev + 1)) * gsize
    kfields = fields_fused if fused else fields_tend
    roofline = {"bound": "hbm", "kernel": kname, "achieved": achieved, "peak": peak, "unit": "GB/s",
                "frac": achieved / peak, "traffic": traffic, "traffic_source": traffic_src, "peak_source": peak_src,
                "algorithmic_bytes_per_launch": kbytes, "kernel_ms": ktime * 1e3,
                "kernel_ms_median": float(np.median(kt)), "kernel_ms_min": float(kt.min()), "kernel_ms_max": float(kt.max()),
                "frac_at_median": kbytes / (float(np.median(kt)) * 1e-3) / 1e9 / peak,
                "frac_at_min": kbytes / (float(kt.min()) * 1e-3) / 1e9 / peak,
                "frac_of_nominal_8TBs": achieved / 8000.0,
                "fields_only": {"bytes_per_launch": kfields, "frac": kfields / ktime / 1e9 / peak,
                                "frac_of_nominal_8TBs": kfields / ktime / 1e9 / 8000.0},
                "two_calls": {"tendencies": {"achieved": bytes_tend / t_tend_avg / 1e9, "frac": bytes_tend / t_tend_avg / 1e9 / peak,
                                             "kernel_ms": t_tend_avg * 1e3, "algorithmic_bytes_per_launch": bytes_tend},
                              "div_vort": {"achieved": bytes_dv / float(t_dv.mean()) / 1e9, "frac": bytes_dv / float(t_dv.mean()) / 1e9 / peak,
                                           "kernel_ms": float(t_dv.mean()) * 1e3, "algorithmic_bytes_per_launch": bytes_dv},
                              "ms_per_step": (t_tend_avg + float(t_dv.mean())) * 1e3},
                "w_tendency": {"call": "dycore_w_tendency (SURVEY 8(f) NEXT-2; not part of the step)", "kernel_ms": float(np.median(t_w)) * 1e3,
                               "algorithmic_bytes_per_launch": bytes_w, "achieved": bytes_w / float(np.median(t_w)) / 1e9,
                               "frac": bytes_w / float(np.median(t_w)) / 1e9 / peak},
                "metric": None if t_m is None else {
                    "call": "dycore_velocity_tendencies_metric (SURVEY 8(f) NEXT-1, reading P-20; not part of the step)",
                    "kernel_ms": float(np.median(t_m)) * 1e3, "algorithmic_bytes_per_launch": bytes_m,
                    "achieved": bytes_m / float(np.median(t_m)) / 1e9, "frac": bytes_m / float(np.median(t_m)) / 1e9 / peak},
                "step_w": {"call": "dycore_step_w: ddt_vn + div + vort + ddt_w from one fused pass (not part of the step)",
                           "kernel_ms": float(np.median(t_sw)) * 1e3,
                           "algorithmic_bytes_per_launch": bytes_fused + g.nc * (nlev + 1) * gsize + g.nc * 3 * gsize,
                           "frac": (bytes_fused + g.nc * (nlev + 1) * gsize + g.nc * 3 * gsize) / float(np.median(t_sw)) / 1e9 / peak}}

    parity_spot = None
    if picks:
        # the oracle (oracle/, test infrastructure) evaluates the same sampled points one by one from the same inputs
        import oracle
        og = oracle.Grid(cfg["k"], si.PERMUTE_SEED if cfg["permute"] else 0, 1 if cfg["permute"] else 0)
        o = og.rounded_f32() if f32 else og
        vn64, w64 = (vn_h.astype(np.float64), w_h.astype(np.float64)) if f32 else (vn_h, w_h)
        tol = 1e-5 if f32 else 1e-12
        parity_spot = {"tolerance": tol, "points_per_output": args.spot_points, "what": "sampled points of the output buffers of "
                       "the last timed launch vs oracle.sample, |gpu - oracle| / M(p) (reading P-16)", "ok": True}
        for what, (idx, lev, got) in picks.items():
            want, m = o.sample(what, idx, lev, vn64, nlev, w=w64, z_half=zh)
            worst = float((np.abs(got - want) / np.maximum(m, 1e-300)).max())
            parity_spot["worst_err_over_M_" + what] = worst
            parity_spot["ok"] = bool(parity_spot["ok"] and worst <= tol and np.isfinite(got).all())
        parity_spot["worst_err_over_M"] = max(v for k_, v in parity_spot.items() if k_.startswith("worst_err_over_M_"))
        del og, o, vn64, w64

    cpu_baseline = None
    if not args.no_cpu_baseline and world == 1:
        k_sample = min(cfg["k"], 6)
        og, ovn, ow, ozh, onlev = oracle_sample(args.config, k_sample)
        oracle_step_seconds(og, ovn, ow, ozh, onlev, 1)
        ts, t_begin = [], time.perf_counter()
        while len(ts) < 3 or (time.perf_counter() - t_begin < 10.0 and len(ts) < 400):
            ts += oracle_step_seconds(og, ovn, ow, ozh, onlev, 1)
        cores = cpu_threads()
        single = None
        if set_oracle_threads(1):                 # the same sample on ONE thread
            t1 = oracle_step_seconds(og, ovn, ow, ozh, onlev, 2)[-1:]
            while sum(t1) < 6.0 and len(t1) < 50:
                t1 += oracle_step_seconds(og, ovn, ow, ozh, onlev, 1)
            set_oracle_threads(cores)
            single = {"value": og.ne * onlev / float(np.mean(t1)) / 1e9, "unit": UNIT, "cores": 1, "steps": len(t1)}
        cpu_baseline = {"value": og.ne * onlev / float(np.mean(ts)) / 1e9, "unit": UNIT, "cores": cores, "kind": "oracle",
                        "sample": "R2B%d x %d levels fp64 oracle, %d timed steps (%.1f s), same field recipe; the full R2B%d "
                                  "grid is not timed because the oracle materialises every intermediate (about 30 GB of host "
                                  "memory and minutes per step at R2B8): a bounded sample of the same recipe instead" % (
                                      k_sample, onlev, len(ts), sum(ts), cfg["k"]),
                        "single_thread": single}
        del og, ovn, ow

    line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
            "ms_per_step": t_step_max * 1e3, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": cfg["dtype"], "data": "synthetic",
            "config": {"workload": workload_name(args.config), "nc": g.nc, "ne": g.ne, "nv": g.nv, "nlev": nlev,
                       "ldk": ldk, "ldk_w": ldk_w, "step": "dycore_step (ddt_vn + div + vort; one fused kernel)" if fused else "dycore_step = dycore_velocity_tendencies + dycore_div_vort",
                       "outputs": ["ddt_vn", "div", "vort"], "l2": "flushed between iterations" if l2_flush is not None else "inputs larger than L2",
                       "parallelism": "replicas only" if world > 1 else "single GPU",
                       "tendency_kernel_variant": args.variant, "cc_tile": args.cc_tile, "cc_pace": args.cc_pace, "grid_create_s": t_grid},
            "gpts_tendency_call_only": pts / t_tend_avg / 1e9,
            "roofline": roofline, "cpu_baseline": cpu_baseline, "e2e": e2e, "gpu_launches": int(launches),
            "step_ms": {"mean": float(t_steps.mean() * 1e3), "median": float(np.median(t_steps) * 1e3),
                        "min": float(t_steps.min() * 1e3), "max": float(t_steps.max() * 1e3),
                        "all": [round(float(x) * 1e3, 4) for x in t_steps]},
            "parity_spot": parity_spot, "clocks": clocks}
    print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()
    return 0


def run_launch_study(args):
    """--launch-study (the paper replays small kernels as CUDA graphs): on the small
    grids the step is one kernel of tens of microseconds, so the launch path matters. Times N dycore_step calls launched
    one by one from Python through the C-ABI against the same N calls captured once into a CUDA graph and replayed, with
    the 126 MB L2 left warm and flushed between steps. One JSON line."""
    import torch
    import paper_2511_02021_b200 as lib
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the product has no CPU path")
    torch.cuda.set_device(0)
    dev = torch.device("cuda", 0)
    lib.load_library()
    n, out = 200, []
    for k in (4, 5):
        g = lib.IconGrid(k)
        nlev, ldk = 90, 96
        vn_h, w_h, zh = si.make_fields(1, g.table_host("edge_xyz"), g.table_host("edge_normal"), g.nc, nlev=nlev, ldk=ldk, ldk_w=ldk, pad_value=0.0)
        vn, w = torch.from_numpy(vn_h).to(dev), torch.from_numpy(w_h).to(dev)
        ddt, div, vort = (torch.zeros((m, ldk), dtype=torch.float64, device=dev) for m in (g.ne, g.nc, g.nv))
        flush = torch.empty(256 * 2 ** 20, dtype=torch.uint8, device=dev)
        step = lambda: lib.dycore_step(g, zh, vn, w, ddt, div, vort, nlev)
        step()
        torch.cuda.synchronize()
        res = {"grid": "R2B%d x %d levels fp64" % (k, nlev), "points": g.ne * nlev, "steps": n}
        for flushed in (False, True):
            def body():
                for _ in range(n):
                    if flushed:
                        flush.fill_(1)
                    step()
            # (a) launched one by one
            body()
            torch.cuda.synchronize()
            t0 = time.perf_counter()
            body()
            torch.cuda.synchronize()
            t_stream = (time.perf_counter() - t0) / n
            # (b) the same sequence captured once, replayed
            side = torch.cuda.Stream()
            side.wait_stream(torch.cuda.current_stream())
            torch.cuda.synchronize()
            graph = torch.cuda.CUDAGraph()
            with torch.cuda.graph(graph):
                body()
            graph.replay()
            torch.cuda.synchronize()
            t0 = time.perf_counter()
            graph.replay()
            torch.cuda.synchronize()
            t_graph = (time.perf_counter() - t0) / n
            # the flush alone, to subtract
            t_flush = 0.0
            if flushed:
                torch.cuda.synchronize()
                t0 = time.perf_counter()
                for _ in range(n):
                    flush.fill_(1)
                torch.cuda.synchronize()
                t_flush = (time.perf_counter() - t0) / n
            key = "l2_flushed" if flushed else "l2_warm"
            res[key] = {"us_per_step_stream": (t_stream - t_flush) * 1e6, "us_per_step_graph": (t_graph - t_flush) * 1e6,
                        "us_flush": t_flush * 1e6, "gpts_stream": g.ne * nlev / (t_stream - t_flush) / 1e9,
                        "gpts_graph": g.ne * nlev / (t_graph - t_flush) / 1e9}
        # device time of one kernel alone (events), L2 warm
        ev = [torch.cuda.Event(enable_timing=True) for _ in range(2)]
        ts = []
        for _ in range(20):
            ev[0].record(); step(); ev[1].record()
            torch.cuda.synchronize()
            ts.append(ev[0].elapsed_time(ev[1]) * 1e3)
        res["us_kernel_events_median"] = float(np.median(ts))
        out.append(res)
        g.close()
    print(json.dumps({"launch_study": out, "what": "wall-clock microseconds per dycore_step over %d back-to-back steps: launched one "
                      "by one through the C-ABI from Python vs captured once into a CUDA graph and replayed" % n}))
    return 0


def run_decomposed(args):
    """--parts R (reading P-21): the fused step on the LOCAL grid of one rank of R, strong scaling
    (total work fixed = the config's grid). Under torchrun with WORLD_SIZE == R every rank holds its part and a step is
    pack(vn) + pack(w) + two all_to_all_single over NCCL + dycore_step; value = the GLOBAL points / the slowest rank's
    time. With one process it times ONE rank's share of that step (--part r, default R // 2) on one GPU: the two pack
    kernels and the local dycore_step, halo rows filled once from the global field; there is no transport on one GPU and
    the line says so. One JSON line."""
    import torch
    import torch.distributed as dist
    import paper_2511_02021_b200 as lib
    from paper_2511_02021_b200.halo import HaloExchange

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the product has no CPU path")
    R = args.parts
    if world > 1 and world != R:
        raise SystemExit("bench.py --parts %d under torchrun needs WORLD_SIZE == %d" % (R, R))
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    if world > 1:
        dist.init_process_group("nccl", device_id=dev)
    lib.load_library()
    cfg = si.CONFIGS[args.config]
    if cfg["permute"]:
        raise SystemExit("bench.py --parts: a decomposed grid keeps the hierarchical numbering (configs without permutation)")
    nlev, f32 = cfg["nlev"], cfg["dtype"] == "f32"
    gsize = 4 if f32 else 8
    line = 32 if f32 else 16
    ldk = args.ldk or (nlev + line - 1) // line * line
    ldk_w = args.ldk_w or (nlev + 1 + line - 1) // line * line
    part = rank if world > 1 else (args.part if args.part >= 0 else R // 2)
    t0 = time.perf_counter()
    g = lib.IconGrid(cfg["k"], n_parts=R, part=part)
    t_grid = time.perf_counter() - t0
    info = g.part_info()
    le, lc = g.part_table("l2g_edge").astype(np.int64), g.part_table("l2g_cell").astype(np.int64)
    # the global synthetic state, of which this rank keeps its rows; geometry from a host-only grid
    gg = lib.IconGrid(cfg["k"], flags=lib.ICON_HOST_ONLY)
    vn_h, w_h, zh = si.make_fields(args.config, gg.table_host("edge_xyz"), gg.table_host("edge_normal"), gg.nc, ldk=ldk, ldk_w=ldk_w,
                                   pad_value=0.0)
    gg.close()
    tdt = torch.float32 if f32 else torch.float64
    vn, w = torch.from_numpy(vn_h[le]).to(dev), torch.from_numpy(w_h[lc]).to(dev)
    del vn_h, w_h
    if world > 1:                     # halo rows must come through the exchange
        vn[info["ne_owned"]:] = float("nan")
        w[info["nc_owned"]:] = float("nan")
    ddt = torch.zeros((g.ne, ldk), dtype=tdt, device=dev)
    div = torch.zeros((g.nc, ldk), dtype=tdt, device=dev)
    vort = torch.zeros((g.nv, ldk), dtype=tdt, device=dev)
    hx = HaloExchange(g)
    sbuf = [hx.send_buffer(0, vn), hx.send_buffer(1, w)]
    l2_flush = torch.empty(256 * 2 ** 20, dtype=torch.uint8, device=dev)      # a rank's share may be L2 resident: flush

    def step(evs=None):
        l2_flush.fill_(1)
        if evs:
            evs[0].record()
        if world > 1:
            hx.exchange(vn, 0)
            hx.exchange(w, 1)
        else:
            lib.dycore_halo_pack(g, 0, vn, sbuf[0])
            lib.dycore_halo_pack(g, 1, w, sbuf[1])
        if evs:
            evs[1].record()
        lib.dycore_step(g, zh, vn, w, ddt, div, vort, nlev)
        if evs:
            evs[2].record()

    for _ in range(max(args.warmup, 3)):
        step()
    torch.cuda.synchronize()
    if world > 1:
        dist.barrier()
    n0 = g.launch_count
    evs = [[torch.cuda.Event(enable_timing=True) for _ in range(3)] for _ in range(args.steps)]
    for i in range(args.steps):
        step(evs[i])
    torch.cuda.synchronize()
    if world > 1:
        dist.barrier()
    t_ex = np.array([e[0].elapsed_time(e[1]) for e in evs]) * 1e-3
    t_st = np.array([e[1].elapsed_time(e[2]) for e in evs]) * 1e-3
    t_all = max_over_ranks(float((t_ex + t_st).mean()), dev)
    launches = g.launch_count - n0
    pts_owned = info["ne_owned"] * nlev
    pts_global = info["ne_global"] * nlev
    send_rows = (sum(hx.send_rows[0]), sum(hx.send_rows[1]))
    recv_rows = (info["ne_local"] - info["ne_owned"], info["nc_local"] - info["nc_owned"])
    bytes_tend, bytes_dv = algorithmic_bytes(info["nc_owned"], info["ne_owned"], info["nv_owned"], nlev, gsize)
    # the fused step's compulsory bytes as run_ours counts them, on the owned points, plus the halo columns it reads
    bytes_step = bytes_tend + (info["nc_owned"] + info["nv_owned"]) * nlev * gsize + info["nc_owned"] * 3 * gsize \
        + (recv_rows[0] * nlev + recv_rows[1] * (nlev + 1)) * gsize
    peak, peak_src = peak_hbm_gbs()
    dec = {"n_parts": R, "part": part, "transport": "nccl all_to_all_single" if world > 1 else "none (one process: one rank's kernels only)",
           "cells_owned": info["nc_owned"], "edges_owned": info["ne_owned"], "edges_halo": recv_rows[0], "cells_halo": recv_rows[1],
           "halo_fraction_edges": recv_rows[0] / info["ne_owned"], "peers": int(sum(1 for x in hx.recv_rows[0] if x)),
           "send_bytes_per_step": (send_rows[0] * ldk + send_rows[1] * ldk_w) * gsize,
           "recv_bytes_per_step": (recv_rows[0] * ldk + recv_rows[1] * ldk_w) * gsize,
           "exchange_ms" if world > 1 else "pack_ms": float(t_ex.mean() * 1e3), "local_step_ms": float(t_st.mean() * 1e3),
           "local_step_ms_min": float(t_st.min() * 1e3),
           "local_step_frac_of_hbm_roofline": bytes_step / float(t_st.mean()) / 1e9 / peak, "peak_source": peak_src,
           "local_grid_build_s": t_grid}
    if rank == 0:
        value = (pts_global if world > 1 else pts_owned) / t_all / 1e9
        print(json.dumps({"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": max(args.warmup, 3),
                          "ms_per_step": t_all * 1e3, "higher_is_better": True, "scaling": "strong", "vs_baseline": None,
                          "dtype": "f32" if f32 else "f64", "data": "synthetic",
                          "config": {"workload": workload_name(args.config) + (", decomposed over %d ranks" % R if world > 1 else
                                                                               ", rank %d of %d only (its owned points)" % (part, R)),
                                     "l2": "flushed between steps", "ldk": ldk, "ldk_w": ldk_w},
                          "gpu_launches": int(launches), "decomposed": dec}))
    g.close()
    if world > 1:
        dist.destroy_process_group()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--config", type=int, default=3, choices=sorted(si.CONFIGS))
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--variant", type=int, default=None, help="ICON_OPT_TENDENCY_KERNEL override")
    ap.add_argument("--cc-tile", type=int, default=None, dest="cc_tile", help="ICON_OPT_CC_TILE override")
    ap.add_argument("--cc-pace", type=int, default=None, dest="cc_pace", help="ICON_OPT_CC_PACE override")
    ap.add_argument("--ldk", type=int, default=0, help="leading dimension of vn/ddt_vn/div/vort (default: padded to 128 B)")
    ap.add_argument("--ldk-w", type=int, default=0, dest="ldk_w")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-parity-spot", action="store_true", dest="no_parity_spot")
    ap.add_argument("--no-metric", action="store_true", dest="no_metric", help="skip the metric-variant leg (saves 4 more field-sized arrays)")
    ap.add_argument("--spot-points", type=int, default=3000, dest="spot_points")
    ap.add_argument("--parts", type=int, default=0, help="decomposed sweep over this many ranks (SURVEY 8(f) NEXT-3); see run_decomposed")
    ap.add_argument("--part", type=int, default=-1, help="with --parts and one process: the rank to time (default parts // 2)")
    ap.add_argument("--launch-study", action="store_true", dest="launch_study", help="CUDA-graph vs stream launches on R2B4 / R2B5")
    args = ap.parse_args()
    if args.launch_study:
        return run_launch_study(args)
    if args.parts:
        return run_decomposed(args)
    if args.warmup < 3 and args.impl == "ours":
        args.warmup = 3
    return run_reference(args) if args.impl == "reference" else run_ours(args)


if __name__ == "__main__":
    sys.exit(main())
