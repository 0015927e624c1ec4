"""ORACLE -- test infrastructure, not the product.

ctypes wrapper around ``oracle/icon_oracle.c`` (plain C, fp64, scalar loops): the slow,
obviously-correct CPU statement of the hot path of arxiv/paper_2511_02021 (PAPER.md:56 C-grid,
PAPER.md:164-167 edge->cell interpolation, PAPER.md:186 dual grid / index arrays; everything
else per the readings P-1..P-17 in DESIGN.md section 3).

Only ``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s ``cpu_baseline`` /
``--impl reference`` legs may import this package. It shares no code with
``paper_2511_02021_b200`` and never imports it.
"""
import ctypes
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "icon_oracle.c")
_LIB = os.path.join(_HERE, "libicon_oracle.so")

PERMUTE = 1
EARTH_RADIUS = 6.371e6
OMEGA = 7.29212e-5


def build(force=False):
    """Compile the oracle with gcc (-O2, no FMA contraction, OpenMP on the entity loops)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        cmd = ["gcc", "-O2", "-ffp-contract=off", "-fopenmp", "-shared", "-fPIC", "-std=c99",
               "-o", _LIB, _SRC, "-lm"]
        subprocess.run(cmd, check=True)
    return _LIB


_lib = None


def _load():
    global _lib
    if _lib is not None:
        return _lib
    build()
    L = ctypes.CDLL(_LIB)
    P = ctypes.c_void_p
    i64 = ctypes.c_int64
    L.og_grid_create.restype = P
    L.og_grid_create.argtypes = [ctypes.c_int, ctypes.c_uint64, ctypes.c_uint]
    L.og_grid_round_f32.restype = P
    L.og_grid_round_f32.argtypes = [P]
    L.og_grid_destroy.restype = None
    L.og_grid_destroy.argtypes = [P]
    for f in (L.og_grid_nc, L.og_grid_ne, L.og_grid_nv):
        f.restype = i64
        f.argtypes = [P]
    L.og_grid_table.restype = P
    L.og_grid_table.argtypes = [P, ctypes.c_char_p]
    L.og_div_vort.restype = ctypes.c_int
    L.og_div_vort.argtypes = [P, ctypes.c_int, i64, P, P, P, P, P]
    L.og_velocity_tendencies.restype = ctypes.c_int
    L.og_velocity_tendencies.argtypes = [P, ctypes.c_int, i64, i64, P, P, P, P, P, P, P, P]
    for f in (L.og_sample_div, L.og_sample_vort):
        f.restype = None
        f.argtypes = [P, ctypes.c_int, i64, P, i64, P, P, P, P]
    L.og_sample_ddt_vn.restype = None
    L.og_sample_ddt_vn.argtypes = [P, ctypes.c_int, i64, i64, P, P, P, i64, P, P, P, P]
    L.og_w_tendency.restype = ctypes.c_int
    L.og_w_tendency.argtypes = [P, ctypes.c_int, i64, i64, P, P, P, P, P]
    L.og_sample_ddt_w.restype = None
    L.og_sample_ddt_w.argtypes = [P, ctypes.c_int, i64, i64, P, P, P, i64, P, P, P, P]
    L.og_ddt_w.restype = None
    L.og_ddt_w.argtypes = [i64, ctypes.c_int, i64, i64, P, P, P, P, P, P, P, P, P]
    L.og_metric_from_zhalf.restype = None
    L.og_metric_from_zhalf.argtypes = [i64, ctypes.c_int, i64, i64, P, P, P]
    L.og_velocity_tendencies_metric.restype = ctypes.c_int
    L.og_velocity_tendencies_metric.argtypes = [P, ctypes.c_int, i64, i64, P, P, P, P, P, P, P, P, P, P, P]
    L.og_sample_ddt_vn_metric.restype = None
    L.og_sample_ddt_vn_metric.argtypes = [P, ctypes.c_int, i64, i64, P, P, P, P, P, P, i64, P, P, P, P]
    L.og_divergence.restype = None
    L.og_divergence.argtypes = [i64, ctypes.c_int, i64, P, P, P, P, P]
    L.og_vorticity.restype = None
    L.og_vorticity.argtypes = [i64, ctypes.c_int, i64, P, P, P, P, P]
    L.og_tangential_wind.restype = None
    L.og_tangential_wind.argtypes = [i64, ctypes.c_int, i64, P, P, P, P]
    L.og_kinetic_energy_edge.restype = None
    L.og_kinetic_energy_edge.argtypes = [i64, ctypes.c_int, i64, P, P, P]
    L.og_kinetic_energy_cell.restype = None
    L.og_kinetic_energy_cell.argtypes = [i64, ctypes.c_int, i64, P, P, P, P]
    L.og_ddt_vn.restype = None
    L.og_ddt_vn.argtypes = [i64, ctypes.c_int, i64, i64, P, P, P, P, P, P, P, P, P, P, P, P, P]
    _lib = L
    return L


# name -> (dtype, entity, cols)
_TABLES = {
    "c2v": (np.int32, "c", 3), "c2e": (np.int32, "c", 3), "e2c": (np.int32, "e", 2),
    "e2v": (np.int32, "e", 2), "e2e4": (np.int32, "e", 4), "v2e": (np.int32, "v", 6),
    "v2c": (np.int32, "v", 6), "v_deg": (np.int32, "v", 1), "c_os": (np.int8, "c", 3),
    "v_os": (np.int8, "v", 6),
    "vert_xyz": (np.float64, "v", 3), "cell_xyz": (np.float64, "c", 3),
    "edge_xyz": (np.float64, "e", 3), "edge_normal": (np.float64, "e", 3),
    "l_e": (np.float64, "e", 1), "d_e": (np.float64, "e", 1), "inv_d_e": (np.float64, "e", 1),
    "f_e": (np.float64, "e", 1), "c_lin": (np.float64, "e", 2), "cgrad": (np.float64, "e", 2), "rbf": (np.float64, "e", 4),
    "a_c": (np.float64, "c", 1), "bln": (np.float64, "c", 3), "adv_c": (np.float64, "c", 3), "a_v": (np.float64, "v", 1),
    "geofac_div": (np.float64, "c", 3), "geofac_rot": (np.float64, "v", 6),
}
TABLE_NAMES = tuple(_TABLES)


def _ptr(a):
    return None if a is None else a.ctypes.data_as(ctypes.c_void_p)


def _f64(a):
    a = np.ascontiguousarray(a, dtype=np.float64)
    return a


class Grid:
    """R2Bk icosahedral C-grid with all tables of SURVEY 8(a) rows G1-G3 (oracle's own generator)."""

    def __init__(self, k, seed=0, flags=0, _handle=None):
        L = _load()
        self._L = L
        self._h = _handle if _handle is not None else L.og_grid_create(int(k), int(seed), int(flags))
        if not self._h:
            raise RuntimeError("oracle: og_grid_create failed for R2B%d" % k)
        self.k = int(k)
        self.nc = int(L.og_grid_nc(self._h))
        self.ne = int(L.og_grid_ne(self._h))
        self.nv = int(L.og_grid_nv(self._h))
        self._cache = {}

    def __del__(self):
        h, self._h = getattr(self, "_h", None), None
        if h:
            self._L.og_grid_destroy(h)

    def rounded_f32(self):
        """P-17: same grid with coefficient arrays rounded to fp32 once (held as fp64)."""
        return Grid(self.k, _handle=self._L.og_grid_round_f32(self._h))

    def table(self, name):
        if name in self._cache:
            return self._cache[name]
        dt, ent, cols = _TABLES[name]
        rows = {"c": self.nc, "e": self.ne, "v": self.nv}[ent]
        p = self._L.og_grid_table(self._h, name.encode())
        if not p:
            raise KeyError(name)
        n = rows * cols
        buf = (ctypes.c_char * (n * np.dtype(dt).itemsize)).from_address(p)
        a = np.frombuffer(buf, dtype=dt, count=n).copy()
        a = a.reshape(rows, cols) if cols > 1 else a
        self._cache[name] = a
        return a

    def __getattr__(self, name):
        if name in _TABLES:
            return self.table(name)
        raise AttributeError(name)

    # ---- whole-call operators (the C-ABI's two calls) ----
    def div_vort(self, vn, nlev, with_scale=False):
        vn = _f64(vn)
        ldk = vn.shape[1]
        div = np.zeros((self.nc, ldk))
        vort = np.zeros((self.nv, ldk))
        md = np.zeros_like(div) if with_scale else None
        mv = np.zeros_like(vort) if with_scale else None
        rc = self._L.og_div_vort(self._h, nlev, ldk, _ptr(vn), _ptr(div), _ptr(vort), _ptr(md), _ptr(mv))
        if rc:
            raise RuntimeError("og_div_vort rc=%d" % rc)
        return (div, vort, md, mv) if with_scale else (div, vort)

    def velocity_tendencies(self, vn, w, z_half, nlev, with_scale=False):
        """returns dict(ddt_vn, vt, ke_c, vort[, m_ddt])"""
        vn = _f64(vn)
        w = _f64(w)
        z_half = _f64(z_half)
        ldk, ldk_w = vn.shape[1], w.shape[1]
        out = {n: np.zeros((self.ne, ldk)) for n in ("ddt_vn", "vt")}
        out["ke_c"] = np.zeros((self.nc, ldk))
        out["vort"] = np.zeros((self.nv, ldk))
        m = np.zeros((self.ne, ldk)) if with_scale else None
        rc = self._L.og_velocity_tendencies(self._h, nlev, ldk, ldk_w, _ptr(z_half), _ptr(vn), _ptr(w),
                                            _ptr(out["ddt_vn"]), _ptr(out["vt"]), _ptr(out["ke_c"]),
                                            _ptr(out["vort"]), _ptr(m))
        if rc:
            raise RuntimeError("og_velocity_tendencies rc=%d" % rc)
        if with_scale:
            out["m_ddt"] = m
        return out

    def w_tendency(self, vn, w, z_half, nlev, with_scale=False):
        """vertical-wind tendency ddt_w [nc][ldk_w] on the nlev+1 half levels (reading P-19)[, m_w]"""
        vn, w, z_half = _f64(vn), _f64(w), _f64(z_half)
        ldk, ldk_w = vn.shape[1], w.shape[1]
        out = np.zeros((self.nc, ldk_w))
        m = np.zeros((self.nc, ldk_w)) if with_scale else None
        rc = self._L.og_w_tendency(self._h, nlev, ldk, ldk_w, _ptr(z_half), _ptr(vn), _ptr(w), _ptr(out), _ptr(m))
        if rc:
            raise RuntimeError("og_w_tendency rc=%d" % rc)
        return (out, m) if with_scale else out

    def velocity_tendencies_metric(self, vn, w, wgt_e, inv_ddqz_e, ddxn_z, ddxt_z, nlev, with_scale=False):
        """metric variant of S3-S7 (reading P-20); returns dict(ddt_vn, vt, ke_c, vort[, m_ddt])"""
        vn, w = _f64(vn), _f64(w)
        wgt_e, inv_ddqz_e, ddxn_z, ddxt_z = _f64(wgt_e), _f64(inv_ddqz_e), _f64(ddxn_z), _f64(ddxt_z)
        ldk, ldk_w = vn.shape[1], w.shape[1]
        assert wgt_e.shape == (self.ne, ldk_w) and inv_ddqz_e.shape == ddxn_z.shape == ddxt_z.shape == (self.ne, ldk)
        out = {n: np.zeros((self.ne, ldk)) for n in ("ddt_vn", "vt")}
        out["ke_c"] = np.zeros((self.nc, ldk))
        out["vort"] = np.zeros((self.nv, ldk))
        m = np.zeros((self.ne, ldk)) if with_scale else None
        rc = self._L.og_velocity_tendencies_metric(self._h, nlev, ldk, ldk_w, _ptr(wgt_e), _ptr(inv_ddqz_e), _ptr(ddxn_z),
                                                   _ptr(ddxt_z), _ptr(vn), _ptr(w), _ptr(out["ddt_vn"]), _ptr(out["vt"]),
                                                   _ptr(out["ke_c"]), _ptr(out["vort"]), _ptr(m))
        if rc:
            raise RuntimeError("og_velocity_tendencies_metric rc=%d" % rc)
        if with_scale:
            out["m_ddt"] = m
        return out

    def sample_metric(self, idx, lev, vn, w, wgt_e, inv_ddqz_e, ddxn_z, ddxt_z, nlev):
        """ddt_vn of the metric variant (P-20) at the points (edge idx[i], level lev[i]); the metric arrays are used as they
        are (any dtype-compatible contiguous float64 arrays of the fields' shapes). Returns (values, M)."""
        vn, w = _f64(vn), _f64(w)
        wgt_e, inv_ddqz_e, ddxn_z, ddxt_z = _f64(wgt_e), _f64(inv_ddqz_e), _f64(ddxn_z), _f64(ddxt_z)
        idx = np.ascontiguousarray(idx, dtype=np.int64)
        lev = np.ascontiguousarray(lev, dtype=np.int32)
        out, m = np.zeros(idx.size), np.zeros(idx.size)
        self._L.og_sample_ddt_vn_metric(self._h, nlev, vn.shape[1], w.shape[1], _ptr(wgt_e), _ptr(inv_ddqz_e), _ptr(ddxn_z),
                                        _ptr(ddxt_z), _ptr(vn), _ptr(w), idx.size, _ptr(idx), _ptr(lev), _ptr(out), _ptr(m))
        return out, m

    # ---- sampled one-by-one evaluation (full-size parity) ----
    def sample(self, what, idx, lev, vn, nlev, w=None, z_half=None):
        vn = _f64(vn)
        idx = np.ascontiguousarray(idx, dtype=np.int64)
        lev = np.ascontiguousarray(lev, dtype=np.int32)
        n = idx.size
        out = np.zeros(n)
        m = np.zeros(n)
        ldk = vn.shape[1]
        if what == "div":
            self._L.og_sample_div(self._h, nlev, ldk, _ptr(vn), n, _ptr(idx), _ptr(lev), _ptr(out), _ptr(m))
        elif what == "vort":
            self._L.og_sample_vort(self._h, nlev, ldk, _ptr(vn), n, _ptr(idx), _ptr(lev), _ptr(out), _ptr(m))
        elif what == "ddt_vn":
            w = _f64(w)
            z_half = _f64(z_half)
            self._L.og_sample_ddt_vn(self._h, nlev, ldk, w.shape[1], _ptr(z_half), _ptr(vn), _ptr(w), n,
                                     _ptr(idx), _ptr(lev), _ptr(out), _ptr(m))
        elif what == "ddt_w":
            w = _f64(w)
            z_half = _f64(z_half)
            self._L.og_sample_ddt_w(self._h, nlev, ldk, w.shape[1], _ptr(z_half), _ptr(vn), _ptr(w), n,
                                    _ptr(idx), _ptr(lev), _ptr(out), _ptr(m))
        else:
            raise ValueError(what)
        return out, m


# ---- stage-by-stage operators on explicit arrays (P-18: feed the oracle someone else's geometry) ----
def divergence(c2e, geofac_div, vn, nlev):
    L = _load()
    c2e = np.ascontiguousarray(c2e, np.int32)
    geofac_div = _f64(geofac_div)
    vn = _f64(vn)
    nc, ldk = c2e.shape[0], vn.shape[1]
    div, m = np.zeros((nc, ldk)), np.zeros((nc, ldk))
    L.og_divergence(nc, nlev, ldk, _ptr(c2e), _ptr(geofac_div), _ptr(vn), _ptr(div), _ptr(m))
    return div, m


def vorticity(v2e, geofac_rot, vn, nlev):
    L = _load()
    v2e = np.ascontiguousarray(v2e, np.int32)
    geofac_rot = _f64(geofac_rot)
    vn = _f64(vn)
    nv, ldk = v2e.shape[0], vn.shape[1]
    vort, m = np.zeros((nv, ldk)), np.zeros((nv, ldk))
    L.og_vorticity(nv, nlev, ldk, _ptr(v2e), _ptr(geofac_rot), _ptr(vn), _ptr(vort), _ptr(m))
    return vort, m


def velocity_tendencies_from_arrays(t, vn, w, z_half, nlev):
    """Same sequence as Grid.velocity_tendencies but on a dict ``t`` of explicit tables
    (c2e, e2c, e2v, e2e4, v2e, rbf, bln, geofac_rot, inv_d_e, f_e, c_lin)."""
    L = _load()
    vn, w, z_half = _f64(vn), _f64(w), _f64(z_half)
    i32 = lambda n: np.ascontiguousarray(t[n], np.int32)
    f64 = lambda n: _f64(t[n])
    c2e, e2c, e2v, e2e4, v2e = i32("c2e"), i32("e2c"), i32("e2v"), i32("e2e4"), i32("v2e")
    rbf, bln, rot, inv_d, f_e, c_lin = f64("rbf"), f64("bln"), f64("geofac_rot"), f64("inv_d_e"), f64("f_e"), f64("c_lin")
    ne, nc, nv = e2c.shape[0], c2e.shape[0], v2e.shape[0]
    ldk, ldk_w = vn.shape[1], w.shape[1]
    vt, ke_e, ddt, m = (np.zeros((ne, ldk)) for _ in range(4))
    ke_c, vort = np.zeros((nc, ldk)), np.zeros((nv, ldk))
    L.og_tangential_wind(ne, nlev, ldk, _ptr(e2e4), _ptr(rbf), _ptr(vn), _ptr(vt))
    L.og_kinetic_energy_edge(ne, nlev, ldk, _ptr(vn), _ptr(vt), _ptr(ke_e))
    L.og_kinetic_energy_cell(nc, nlev, ldk, _ptr(c2e), _ptr(bln), _ptr(ke_e), _ptr(ke_c))
    L.og_vorticity(nv, nlev, ldk, _ptr(v2e), _ptr(rot), _ptr(vn), _ptr(vort), None)
    L.og_ddt_vn(ne, nlev, ldk, ldk_w, _ptr(z_half), _ptr(e2c), _ptr(e2v), _ptr(inv_d), _ptr(f_e), _ptr(c_lin),
                _ptr(vn), _ptr(w), _ptr(vt), _ptr(ke_c), _ptr(vort), _ptr(ddt), _ptr(m))
    return {"ddt_vn": ddt, "vt": vt, "ke_e": ke_e, "ke_c": ke_c, "vort": vort, "m_ddt": m}


def w_tendency_from_arrays(t, vn, w, z_half, nlev):
    """og_ddt_w on a dict ``t`` of explicit tables (c2e, e2c, inv_d_e, adv_c); returns (ddt_w, m_w)"""
    L = _load()
    vn, w, z_half = _f64(vn), _f64(w), _f64(z_half)
    c2e, e2c = np.ascontiguousarray(t["c2e"], np.int32), np.ascontiguousarray(t["e2c"], np.int32)
    inv_d, adv = _f64(t["inv_d_e"]), _f64(t["adv_c"])
    nc, ldk, ldk_w = c2e.shape[0], vn.shape[1], w.shape[1]
    out, m = np.zeros((nc, ldk_w)), np.zeros((nc, ldk_w))
    L.og_ddt_w(nc, nlev, ldk, ldk_w, _ptr(z_half), _ptr(c2e), _ptr(e2c), _ptr(inv_d), _ptr(adv), _ptr(vn), _ptr(w), _ptr(out), _ptr(m))
    return out, m


def metric_from_zhalf(z_half_e, nlev, ldk):
    """(wgt_e [ne][ldk_w], inv_ddqz_e [ne][ldk]) of reading P-20 from the half-level heights z_half_e [ne][ldk_w] of every
    edge column (strictly decreasing in k); pads are NaN"""
    L = _load()
    z = _f64(z_half_e)
    ne, ldk_w = z.shape
    wgt, inv = np.full((ne, ldk_w), np.nan), np.full((ne, ldk), np.nan)
    L.og_metric_from_zhalf(ne, nlev, ldk, ldk_w, _ptr(z), _ptr(wgt), _ptr(inv))
    return wgt, inv
