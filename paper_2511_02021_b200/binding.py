"""Thin ctypes binding over libicon_dycore.so (include/icon_dycore.h). Argument marshalling only:
every step of the hot path runs in the library's CUDA kernels. PyTorch is used by callers for
device memory and streams; this module accepts torch tensors or raw device pointers (ints).

There is no CPU fallback: if the shared library is missing or no CUDA device is usable, calls
raise.
"""
import ctypes
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_LIBPATH = os.path.join(_HERE, "libicon_dycore.so")

ICON_OK, ICON_EINVAL, ICON_ENOMEM, ICON_ECUDA, ICON_EUNSUPPORTED = 0, -1, -2, -3, -4
ICON_F64, ICON_F32 = 0, 1
ICON_T_I32, ICON_T_I8, ICON_T_F64, ICON_T_F32 = 10, 11, 12, 13
ICON_PERMUTE, ICON_LOCALITY_WORKLIST, ICON_HOST_ONLY, ICON_NO_WORKLIST = 1, 2, 4, 8
ICON_OPT_TENDENCY_KERNEL = 0
ICON_OPT_CC_TILE = 1
ICON_OPT_CC_PACE = 2

TABLES = ("c2v", "c2e", "e2c", "e2v", "e2e4", "v2e", "v2c", "v_deg", "c_os", "v_os",
          "vert_xyz", "cell_xyz", "edge_xyz", "edge_normal", "l_e", "d_e", "inv_d_e", "f_e", "c_lin", "rbf",
          "a_c", "bln", "a_v", "geofac_div", "geofac_rot", "adv_c", "cgrad")
TABLE_ID = {n: i for i, n in enumerate(TABLES)}

# every symbol include/icon_dycore.h declares
EXPORTS = ("icon_grid_create", "icon_grid_destroy", "icon_grid_counts", "icon_grid_table_host",
           "icon_grid_table_device", "icon_grid_set_option", "icon_grid_cc_schedule_check", "dycore_div_vort", "dycore_velocity_tendencies",
           "dycore_step", "dycore_step_host", "dycore_step_w", "dycore_w_tendency", "dycore_velocity_tendencies_noalloc", "dycore_metric_from_zhalf", "dycore_velocity_tendencies_metric", "icon_grid_launch_count", "icon_last_error",
           "icon_grid_create_part", "icon_part_info", "icon_part_table", "dycore_halo_pack")


class IconError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__("libicon_dycore error %d: %s" % (code, msg))
        self.code = code


_lib = None


def load_library():
    """dlopen the in-tree CUDA library; fails loudly when it has not been built."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(_LIBPATH):
        raise ImportError("%s is missing: run `python -m paper_2511_02021_b200.build` (needs nvcc). "
                          "There is no CPU fallback." % _LIBPATH)
    L = ctypes.CDLL(_LIBPATH)
    P, i64, ci = ctypes.c_void_p, ctypes.c_int64, ctypes.c_int
    L.icon_grid_create.restype = ci
    L.icon_grid_create.argtypes = [ci, ctypes.c_uint64, ctypes.c_uint, ctypes.POINTER(P)]
    L.icon_grid_destroy.restype = None
    L.icon_grid_destroy.argtypes = [P]
    L.icon_grid_counts.restype = ci
    L.icon_grid_counts.argtypes = [P, ctypes.POINTER(i64), ctypes.POINTER(i64), ctypes.POINTER(i64)]
    L.icon_grid_table_host.restype = ci
    L.icon_grid_table_host.argtypes = [P, ci, ctypes.POINTER(P), ctypes.POINTER(ci), ctypes.POINTER(i64), ctypes.POINTER(ci)]
    L.icon_grid_table_device.restype = ci
    L.icon_grid_table_device.argtypes = [P, ci, ci, ctypes.POINTER(P)]
    L.icon_grid_set_option.restype = ci
    L.icon_grid_set_option.argtypes = [P, ci, ci]
    L.icon_grid_cc_schedule_check.restype = ci
    L.icon_grid_cc_schedule_check.argtypes = [P, ci, ci, ci, ci, ci, ci, ctypes.POINTER(i64)]
    L.icon_grid_launch_count.restype = i64
    L.icon_grid_launch_count.argtypes = [P]
    L.dycore_div_vort.restype = ci
    L.dycore_div_vort.argtypes = [P, ci, ci, ci, P, P, P, P]
    L.dycore_velocity_tendencies.restype = ci
    L.dycore_velocity_tendencies.argtypes = [P, ci, ci, ci, ci, P, P, P, P, P, P, P, P]
    L.dycore_w_tendency.restype = ci
    L.dycore_w_tendency.argtypes = [P, ci, ci, ci, ci, P, P, P, P, P]
    L.dycore_velocity_tendencies_noalloc.restype = ci
    L.dycore_velocity_tendencies_noalloc.argtypes = [P, ci, ci, ci, ci, P, P, P, P, P]
    L.dycore_metric_from_zhalf.restype = ci
    L.dycore_metric_from_zhalf.argtypes = [P, ci, ci, ci, ci, P, P, P, P]
    L.dycore_velocity_tendencies_metric.restype = ci
    L.dycore_velocity_tendencies_metric.argtypes = [P, ci, ci, ci, ci, P, P, P, P, P, P, P, P]
    L.dycore_step_w.restype = ci
    L.dycore_step_w.argtypes = [P, ci, ci, ci, ci, P, P, P, P, P, P, P, P]
    L.dycore_step.restype = ci
    L.dycore_step.argtypes = [P, ci, ci, ci, ci, P, P, P, P, P, P, P]
    L.dycore_step_host.restype = ci
    L.dycore_step_host.argtypes = [P, ci, ci, ci, ci, P, P, P, P, P, P]
    L.icon_grid_create_part.restype = ci
    L.icon_grid_create_part.argtypes = [ci, ctypes.c_uint, ci, ci, ctypes.POINTER(P)]
    L.icon_part_info.restype = ci
    L.icon_part_info.argtypes = [P, ctypes.POINTER(i64)]
    L.icon_part_table.restype = ci
    L.icon_part_table.argtypes = [P, ci, ctypes.POINTER(P), ctypes.POINTER(ci), ctypes.POINTER(i64)]
    L.dycore_halo_pack.restype = ci
    L.dycore_halo_pack.argtypes = [P, ci, ci, ci, P, P, P]
    L.icon_last_error.restype = ctypes.c_char_p
    L.icon_last_error.argtypes = []
    _lib = L
    return L


def _check(rc):
    if rc != ICON_OK:
        raise IconError(rc, load_library().icon_last_error().decode(errors="replace"))


def _dptr(x):
    """device (or host) pointer of a torch tensor / numpy array / int / None"""
    if x is None:
        return None
    if isinstance(x, int):
        return ctypes.c_void_p(x)
    if isinstance(x, np.ndarray):
        return ctypes.c_void_p(x.ctypes.data)
    return ctypes.c_void_p(x.data_ptr())


def _stream_ptr(stream):
    if stream is None:
        import torch
        return ctypes.c_void_p(torch.cuda.current_stream().cuda_stream)
    if isinstance(stream, int):
        return ctypes.c_void_p(stream)
    return ctypes.c_void_p(stream.cuda_stream)


ICON_T_I64 = 14
_NP = {ICON_T_I32: np.int32, ICON_T_I8: np.int8, ICON_T_F64: np.float64, ICON_T_F32: np.float32, ICON_T_I64: np.int64}

# icon_part_table selectors (include/icon_dycore.h)
PART_TABLES = ("l2g_cell", "l2g_edge", "l2g_vert", "recv_begin_edge", "recv_begin_cell", "send_begin_edge", "send_begin_cell",
               "send_ids_edge", "send_ids_cell")
PART_INFO = ("n_parts", "part", "nc_owned", "ne_owned", "nv_owned", "nc_local", "ne_local", "nc_global", "ne_global", "nv_global",
             "parent_lo", "parent_hi")


class IconGrid:
    """icon_grid_t handle (R2Bk grid + tables on host and device)."""

    def __init__(self, k, seed=0, flags=0, n_parts=0, part=0):
        """n_parts > 0: the LOCAL grid of rank `part` of `n_parts` (icon_grid_create_part; counts are local)"""
        self._L = load_library()
        h = ctypes.c_void_p()
        if n_parts:
            if seed:
                raise ValueError("a decomposed grid keeps the hierarchical numbering: no seed")
            _check(self._L.icon_grid_create_part(int(k), int(flags), int(n_parts), int(part), ctypes.byref(h)))
        else:
            _check(self._L.icon_grid_create(int(k), int(seed), int(flags), ctypes.byref(h)))
        self._h = h
        self.k, self.seed, self.flags = int(k), int(seed), int(flags)
        nc, ne, nv = ctypes.c_int64(), ctypes.c_int64(), ctypes.c_int64()
        _check(self._L.icon_grid_counts(h, ctypes.byref(nc), ctypes.byref(ne), ctypes.byref(nv)))
        self.nc, self.ne, self.nv = nc.value, ne.value, nv.value

    def close(self):
        h, self._h = getattr(self, "_h", None), None
        if h:
            self._L.icon_grid_destroy(h)

    def __del__(self):
        self.close()

    def table_host(self, name):
        """numpy view (read-only copy semantics: do not write) of a public table"""
        ptr, dt, rows, cols = ctypes.c_void_p(), ctypes.c_int(), ctypes.c_int64(), ctypes.c_int()
        _check(self._L.icon_grid_table_host(self._h, TABLE_ID[name], ctypes.byref(ptr), ctypes.byref(dt),
                                            ctypes.byref(rows), ctypes.byref(cols)))
        npdt = np.dtype(_NP[dt.value])
        n = rows.value * cols.value
        buf = (ctypes.c_char * (n * npdt.itemsize)).from_address(ptr.value)
        a = np.frombuffer(buf, dtype=npdt, count=n)
        a.flags.writeable = False
        return a.reshape(rows.value, cols.value) if cols.value > 1 else a

    def table_device(self, name, dtype=ICON_F64):
        p = ctypes.c_void_p()
        _check(self._L.icon_grid_table_device(self._h, TABLE_ID[name], dtype, ctypes.byref(p)))
        return p.value

    def part_info(self):
        out = (ctypes.c_int64 * 12)()
        _check(self._L.icon_part_info(self._h, out))
        return dict(zip(PART_INFO, [int(x) for x in out]))

    def part_table(self, name):
        """numpy view (do not write) of a table of the local grid: PART_TABLES"""
        ptr, dt, n = ctypes.c_void_p(), ctypes.c_int(), ctypes.c_int64()
        _check(self._L.icon_part_table(self._h, PART_TABLES.index(name), ctypes.byref(ptr), ctypes.byref(dt), ctypes.byref(n)))
        npdt = np.dtype(_NP[dt.value])
        if n.value == 0:
            return np.zeros(0, dtype=npdt)
        buf = (ctypes.c_char * (n.value * npdt.itemsize)).from_address(ptr.value)
        a = np.frombuffer(buf, dtype=npdt, count=n.value)
        a.flags.writeable = False
        return a

    def set_option(self, option, value):
        _check(self._L.icon_grid_set_option(self._h, option, value))

    def cc_schedule_check(self, dtype, nlev, ldk, ldk_w, n_ctas=148, smem_bytes=232448):
        """build + independently validate the column-cache schedule of tendency kernel 4 (icon_grid_cc_schedule_check)"""
        out = (ctypes.c_int64 * 8)()
        _check(self._L.icon_grid_cc_schedule_check(self._h, dtype, nlev, ldk, ldk_w, n_ctas, smem_bytes, out))
        keys = ("steps", "reduced_steps", "vn_columns", "w_columns", "copies", "slots", "slot_bytes", "ctas")
        return dict(zip(keys, [int(x) for x in out]))

    @property
    def launch_count(self):
        return int(self._L.icon_grid_launch_count(self._h))


def icon_grid_create(k, seed=0, flags=0):
    return IconGrid(k, seed, flags)


def _dtype_of(t):
    import torch
    if t.dtype == torch.float64:
        return ICON_F64
    if t.dtype == torch.float32:
        return ICON_F32
    raise TypeError("fields must be float64 or float32 tensors")


def _check_fields(fields, ldk_of=None):
    """Cheap marshalling checks (no arithmetic): every field is a contiguous 2-D CUDA tensor of one dtype on one device
    with the expected row count; fields that share a leading dimension have the same second dimension.
    fields: (name, tensor or None, rows, group) with group naming the leading dimension the tensor must share."""
    first, widths = None, {}
    for name, t, rows, group in fields:
        if t is None:
            continue
        if not hasattr(t, "is_cuda") or not t.is_cuda:
            raise TypeError("%s must be a CUDA tensor (the library has no CPU path)" % name)
        if t.dim() != 2 or not t.is_contiguous():
            raise ValueError("%s must be a contiguous 2-D tensor [entities][levels]" % name)
        if t.shape[0] != rows:
            raise ValueError("%s has %d rows, the grid has %d" % (name, t.shape[0], rows))
        if first is None:
            first = t
        elif t.dtype != first.dtype or t.device != first.device:
            raise TypeError("%s: all fields must have one dtype and live on one device" % name)
        if widths.setdefault(group, t.shape[1]) != t.shape[1]:
            raise ValueError("%s: leading dimension %d differs from the other %s fields (%d)" % (name, t.shape[1], group, widths[group]))


def dycore_div_vort(grid, vn, div, vort, nlev, stream=None):
    """S1+S2. vn [ne][ldk], div [nc][ldk], vort [nv][ldk]: CUDA tensors of one dtype."""
    _check_fields((("vn", vn, grid.ne, "ldk"), ("div", div, grid.nc, "ldk"), ("vort", vort, grid.nv, "ldk")))
    _check(grid._L.dycore_div_vort(grid._h, _dtype_of(vn), int(nlev), int(vn.shape[1]), _dptr(vn), _dptr(div),
                                   _dptr(vort), _stream_ptr(stream)))


def dycore_velocity_tendencies(grid, z_half, vn, w, ddt_vn, nlev, vt=None, ke_c=None, vort=None, stream=None):
    """S3-S7. z_half: host float64 [nlev+1]; vn/ddt_vn [ne][ldk], w [nc][ldk_w]: CUDA tensors."""
    z = np.ascontiguousarray(z_half, dtype=np.float64)
    if z.size != nlev + 1:
        raise ValueError("z_half must have nlev+1 entries")
    _check_fields((("vn", vn, grid.ne, "ldk"), ("w", w, grid.nc, "ldk_w"), ("ddt_vn", ddt_vn, grid.ne, "ldk"),
                   ("vt", vt, grid.ne, "ldk"), ("ke_c", ke_c, grid.nc, "ldk"), ("vort", vort, grid.nv, "ldk")))
    _check(grid._L.dycore_velocity_tendencies(grid._h, _dtype_of(vn), int(nlev), int(vn.shape[1]), int(w.shape[1]),
                                              _dptr(z), _dptr(vn), _dptr(w), _dptr(ddt_vn), _dptr(vt), _dptr(ke_c),
                                              _dptr(vort), _stream_ptr(stream)))


NOALLOC_SCRATCH_BYTES = 64 << 20     # ICON_NOALLOC_SCRATCH_BYTES of include/icon_dycore.h


def dycore_velocity_tendencies_noalloc(grid, z_half, vn, w, ddt_vn, nlev, stream=None):
    """S3-S7 without any allocation (static device scratch of NOALLOC_SCRATCH_BYTES; see include/icon_dycore.h for the
    limits and the sharing rule: calls that overlap on the GPU race)."""
    z = np.ascontiguousarray(z_half, dtype=np.float64)
    if z.size != nlev + 1:
        raise ValueError("z_half must have nlev+1 entries")
    _check_fields((("vn", vn, grid.ne, "ldk"), ("w", w, grid.nc, "ldk_w"), ("ddt_vn", ddt_vn, grid.ne, "ldk")))
    _check(grid._L.dycore_velocity_tendencies_noalloc(grid._h, _dtype_of(vn), int(nlev), int(vn.shape[1]), int(w.shape[1]),
                                                      _dptr(z), _dptr(vn), _dptr(w), _dptr(ddt_vn), _stream_ptr(stream)))


def dycore_metric_from_zhalf(grid, z_half_e, wgt_e, inv_ddqz_e, nlev, stream=None):
    """Set-up of the metric variant (reading P-20): z_half_e, wgt_e [ne][ldk_w], inv_ddqz_e [ne][ldk]: CUDA tensors."""
    _check_fields((("z_half_e", z_half_e, grid.ne, "ldk_w"), ("wgt_e", wgt_e, grid.ne, "ldk_w"), ("inv_ddqz_e", inv_ddqz_e, grid.ne, "ldk")))
    _check(grid._L.dycore_metric_from_zhalf(grid._h, _dtype_of(z_half_e), int(nlev), int(inv_ddqz_e.shape[1]), int(z_half_e.shape[1]),
                                            _dptr(z_half_e), _dptr(wgt_e), _dptr(inv_ddqz_e), _stream_ptr(stream)))


def dycore_velocity_tendencies_metric(grid, wgt_e, inv_ddqz_e, ddxn_z, ddxt_z, vn, w, ddt_vn, nlev, stream=None):
    """S3-S7 in their metric form (reading P-20): weighted KE gradient, per-edge vertical metrics, contravariant correction."""
    _check_fields((("vn", vn, grid.ne, "ldk"), ("w", w, grid.nc, "ldk_w"), ("ddt_vn", ddt_vn, grid.ne, "ldk"),
                   ("wgt_e", wgt_e, grid.ne, "ldk_w"), ("inv_ddqz_e", inv_ddqz_e, grid.ne, "ldk"), ("ddxn_z", ddxn_z, grid.ne, "ldk"),
                   ("ddxt_z", ddxt_z, grid.ne, "ldk")))
    _check(grid._L.dycore_velocity_tendencies_metric(grid._h, _dtype_of(vn), int(nlev), int(vn.shape[1]), int(w.shape[1]), _dptr(wgt_e),
                                                     _dptr(inv_ddqz_e), _dptr(ddxn_z), _dptr(ddxt_z), _dptr(vn), _dptr(w), _dptr(ddt_vn),
                                                     _stream_ptr(stream)))


def dycore_w_tendency(grid, z_half, vn, w, ddt_w, nlev, stream=None):
    """Vertical-wind tendency (reading P-19). vn [ne][ldk], w and ddt_w [nc][ldk_w] on the nlev+1 half levels."""
    z = np.ascontiguousarray(z_half, dtype=np.float64)
    if z.size != nlev + 1:
        raise ValueError("z_half must have nlev+1 entries")
    _check_fields((("vn", vn, grid.ne, "ldk"), ("w", w, grid.nc, "ldk_w"), ("ddt_w", ddt_w, grid.nc, "ldk_w")))
    _check(grid._L.dycore_w_tendency(grid._h, _dtype_of(vn), int(nlev), int(vn.shape[1]), int(w.shape[1]), _dptr(z), _dptr(vn),
                                     _dptr(w), _dptr(ddt_w), _stream_ptr(stream)))


def dycore_step(grid, z_half, vn, w, ddt_vn, div, vort, nlev, stream=None):
    """S1-S7 in one pass (one fused kernel where the column-cache kernel runs, else the two calls back to back)."""
    z = np.ascontiguousarray(z_half, dtype=np.float64)
    if z.size != nlev + 1:
        raise ValueError("z_half must have nlev+1 entries")
    _check_fields((("vn", vn, grid.ne, "ldk"), ("w", w, grid.nc, "ldk_w"), ("ddt_vn", ddt_vn, grid.ne, "ldk"),
                   ("div", div, grid.nc, "ldk"), ("vort", vort, grid.nv, "ldk")))
    _check(grid._L.dycore_step(grid._h, _dtype_of(vn), int(nlev), int(vn.shape[1]), int(w.shape[1]), _dptr(z), _dptr(vn),
                               _dptr(w), _dptr(ddt_vn), _dptr(div), _dptr(vort), _stream_ptr(stream)))


def dycore_step_w(grid, z_half, vn, w, ddt_vn, div, vort, ddt_w, nlev, stream=None):
    """dycore_step plus ddt_w [nc][ldk_w] (reading P-19) from the same pass (one fused kernel where the column cache runs)."""
    z = np.ascontiguousarray(z_half, dtype=np.float64)
    if z.size != nlev + 1:
        raise ValueError("z_half must have nlev+1 entries")
    _check_fields((("vn", vn, grid.ne, "ldk"), ("w", w, grid.nc, "ldk_w"), ("ddt_vn", ddt_vn, grid.ne, "ldk"),
                   ("div", div, grid.nc, "ldk"), ("vort", vort, grid.nv, "ldk"), ("ddt_w", ddt_w, grid.nc, "ldk_w")))
    _check(grid._L.dycore_step_w(grid._h, _dtype_of(vn), int(nlev), int(vn.shape[1]), int(w.shape[1]), _dptr(z), _dptr(vn),
                                 _dptr(w), _dptr(ddt_vn), _dptr(div), _dptr(vort), _dptr(ddt_w), _stream_ptr(stream)))


def dycore_halo_pack(grid, kind, field, send_buf, stream=None):
    """send side of the halo exchange: send_buf[i] = field[send_ids[i]], whole rows. kind 0 = edge
    field, 1 = cell field; field [n_local][ld], send_buf [n_send][ld]: CUDA tensors of one dtype."""
    rows = grid.ne if kind == 0 else grid.nc
    n_send = len(grid.part_table("send_ids_edge" if kind == 0 else "send_ids_cell"))
    _check_fields((("field", field, rows, "ld"), ("send_buf", send_buf, n_send, "ld")))
    _check(grid._L.dycore_halo_pack(grid._h, _dtype_of(field), int(kind), int(field.shape[1]), _dptr(field), _dptr(send_buf),
                                    _stream_ptr(stream)))


def dycore_step_host(grid, z_half, vn_host, w_host, ddt_vn_host, div_host, vort_host, nlev):
    """End-to-end step on HOST buffers (pinned torch CPU tensors or numpy arrays)."""
    z = np.ascontiguousarray(z_half, dtype=np.float64)
    f64 = (vn_host.dtype == np.float64) if isinstance(vn_host, np.ndarray) else (str(vn_host.dtype) == "torch.float64")
    _check(grid._L.dycore_step_host(grid._h, ICON_F64 if f64 else ICON_F32, int(nlev), int(vn_host.shape[1]),
                                    int(w_host.shape[1]), _dptr(z), _dptr(vn_host), _dptr(w_host), _dptr(ddt_vn_host),
                                    _dptr(div_host), _dptr(vort_host)))
