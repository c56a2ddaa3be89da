"""Thin ctypes binding over the C ABI of include/nbk.h -- argument marshalling only.

Every function here has the name of the C entry point it calls; none contains arithmetic of
the method.  Host variants take numpy arrays, `_dev` variants take raw device addresses
(e.g. `tensor.data_ptr()`).  There is no CPU fallback: if libnbk.so is missing or cannot be
loaded, importing symbols from it raises.
"""
from __future__ import annotations

import ctypes
import os

import numpy as np

from . import build as _build

NBK_OK, NBK_EINVAL, NBK_ERANGE, NBK_ENOMEM, NBK_ECUDA, NBK_ESTATE = 0, -1, -2, -3, -4, -5
NBK_JERK, NBK_POT, NBK_EPS0, NBK_NN = 1, 2, 4, 8
NBK_NOALLOC_MAX_NI, NBK_NOALLOC_MAX_NJ = 4096, 16777216

EXPORTS = [
    "nbk_open", "nbk_open_ws", "nbk_workspace_bytes", "nbk_close", "nbk_npipes", "nbk_set_j_particles", "nbk_set_j_particles_f64",
    "nbk_set_j_particles_dev", "nbk_set_ti", "nbk_predict", "nbk_get_predicted",
    "nbk_calc_firsthalf", "nbk_calc_firsthalf_dev", "nbk_calc_lasthalf", "nbk_calc_lasthalf_f64", "nbk_calc_lasthalf_dev",
    "nbk_calc_noalloc_dev",
    "nbk_get_neighbours", "nbk_get_neighbours_dev", "nbk_calc_batch", "nbk_calc_batch_dev",
    "nbk_shard_gather_i_dev", "nbk_shard_calc_partial_dev", "nbk_shard_finish_dev",
    "nbk_shard_fetch_i_dev", "nbk_shard_combine_dev",
    "nbk_hermite_evolve", "nbk_hermite_evolve_dev", "nbk_sync", "nbk_set_timing", "nbk_get_timing", "nbk_last_launch",
    "nbk_plan", "nbk_set_variant", "nbk_last_cuda_error", "nbk_strerror", "nbk_version",
]

_vp, _i64, _i32, _u32, _f32, _f64 = (ctypes.c_void_p, ctypes.c_int64, ctypes.c_int,
                                     ctypes.c_uint32, ctypes.c_float, ctypes.c_double)


class HermiteStats(ctypes.Structure):
    _fields_ = [("block_steps", _i64), ("particle_steps", _i64), ("interactions", _i64),
                ("wall_seconds", _f64), ("gpu_call_seconds", _f64), ("t_reached", _f64),
                ("ni_histogram", _i64 * 32)]


_SIGS = {
    "nbk_open": (_i32, [ctypes.POINTER(_vp), _i32, _i64, _i64, _vp]),
    "nbk_open_ws": (_i32, [ctypes.POINTER(_vp), _i32, _i64, _i64, _vp, _vp, _i64]),
    "nbk_workspace_bytes": (_i64, [_i32, _i64, _i64]),
    "nbk_close": (_i32, [_vp]),
    "nbk_npipes": (_i32, [_vp]),
    "nbk_set_j_particles": (_i32, [_vp, _i64] + [_vp] * 7),
    "nbk_set_j_particles_f64": (_i32, [_vp, _i64] + [_vp] * 7),
    "nbk_set_j_particles_dev": (_i32, [_vp, _i64] + [_vp] * 7),
    "nbk_set_ti": (_i32, [_vp, _f64]),
    "nbk_predict": (_i32, [_vp, _i64]),
    "nbk_get_predicted": (_i32, [_vp, _i64, _vp, _vp, _vp]),
    "nbk_calc_firsthalf": (_i32, [_vp, _i64, _i64, _vp, _vp, _vp, _f32, _u32]),
    "nbk_calc_firsthalf_dev": (_i32, [_vp, _i64, _i64, _vp, _vp, _vp, _f32, _u32]),
    "nbk_calc_lasthalf": (_i32, [_vp, _i64, _vp, _vp, _vp]),
    "nbk_calc_lasthalf_f64": (_i32, [_vp, _i64, _vp, _vp, _vp]),
    "nbk_calc_lasthalf_dev": (_i32, [_vp, _i64, _vp, _vp, _vp]),
    "nbk_calc_noalloc_dev": (_i32, [_i32, _vp, _i64, _vp, _vp, _vp, _i64, _vp, _f32, _u32, _vp, _vp, _vp,
                                    ctypes.POINTER(_i32)]),
    "nbk_calc_batch": (_i32, [_vp, _i64, _vp, _vp, _vp, _vp, _vp, _f32, _u32, _vp, _vp]),
    "nbk_calc_batch_dev": (_i32, [_vp, _i64, _vp, _vp, _vp, _vp, _vp, _f32, _u32, _vp, _vp]),
    "nbk_get_neighbours": (_i32, [_vp, _i64, _vp, _vp]),
    "nbk_get_neighbours_dev": (_i32, [_vp, _i64, _vp, _vp]),
    "nbk_shard_gather_i_dev": (_i32, [_vp, _i64, _i64, _i64, _vp, _vp, _vp]),
    "nbk_shard_calc_partial_dev": (_i32, [_vp, _i64, _i64, _vp, _vp, _f32, _u32, _vp]),
    "nbk_shard_finish_dev": (_i32, [_vp, _i64, _vp, _vp, _vp, _vp]),
    "nbk_shard_fetch_i_dev": (_i32, [_vp, _i64, _i32, _vp, _vp, _vp, _vp]),
    "nbk_shard_combine_dev": (_i32, [_vp, _i64, _i32, _vp, _vp, _vp, _vp]),
    "nbk_hermite_evolve": (_i32, [_vp, _i64, _vp, _vp, _vp, _f64, _f64, _f64, _f64,
                                  ctypes.POINTER(HermiteStats)]),
    "nbk_hermite_evolve_dev": (_i32, [_vp, _i64, _vp, _vp, _vp, _f64, _f64, _f64, _f64,
                                      ctypes.POINTER(HermiteStats)]),
    "nbk_sync": (_i32, [_vp]),
    "nbk_set_timing": (_i32, [_vp, _i32]),
    "nbk_get_timing": (_i32, [_vp, ctypes.POINTER(_f32 * 4)]),
    "nbk_last_launch": (_i32, [_vp, ctypes.POINTER(_i64 * 8)]),
    "nbk_plan": (_i32, [_i64, _i64, _i32, _i32, ctypes.POINTER(_i64 * 12)]),
    "nbk_set_variant": (_i32, [_vp, _i32]),
    "nbk_last_cuda_error": (_i32, [_vp]),
    "nbk_strerror": (ctypes.c_char_p, [_i32]),
    "nbk_version": (ctypes.c_char_p, []),
}

_lib = None


def library_path() -> str:
    return os.environ.get("NBK_LIB", _build.LIB)


def load(build_if_stale: bool = True):
    """dlopen libnbk.so (building it first if sources are newer and nvcc is here)."""
    global _lib
    if _lib is None:
        path = library_path()
        if build_if_stale and path == _build.LIB and _build.is_stale():
            _build.build()
        if not os.path.exists(path):
            raise RuntimeError(f"{path} not found: build it with `python -m paper_0707_0438_b200.build`"
                               " (the CUDA path has no fallback)")
        lib = ctypes.CDLL(path)
        for name, (res, args) in _SIGS.items():
            fn = getattr(lib, name)  # raises AttributeError if an export is missing
            fn.restype, fn.argtypes = res, args
        _lib = lib
    return _lib


class NbkError(RuntimeError):
    def __init__(self, fn, status, cuda=0):
        msg = load().nbk_strerror(status).decode()
        super().__init__(f"{fn}: {msg} (status {status}" + (f", cudaError {cuda})" if cuda else ")"))
        self.status, self.cuda = status, cuda


def _check(fn, status, ctx=None):
    if status != NBK_OK:
        cuda = load().nbk_last_cuda_error(ctx) if (ctx and status == NBK_ECUDA) else 0
        raise NbkError(fn, status, cuda)


def _host(a, dtype, shape_tail=None):
    if a is None:
        return None, None
    arr = np.ascontiguousarray(a, dtype=dtype)
    if shape_tail is not None and arr.shape[1:] != shape_tail:
        raise ValueError(f"expected shape [n]{list(shape_tail)}, got {arr.shape}")
    return arr, arr.ctypes.data


# ------------------------------------------------------------------ same-name entry points
def nbk_open(device: int, n_max: int, ni_max: int, cuda_stream: int = 0):
    ctx = _vp()
    _check("nbk_open", load().nbk_open(ctypes.byref(ctx), device, n_max, ni_max, cuda_stream or None))
    return ctx


def nbk_workspace_bytes(device: int, n_max: int, ni_max: int) -> int:
    n = load().nbk_workspace_bytes(device, n_max, ni_max)
    if n < 0:
        raise NbkError("nbk_workspace_bytes", int(n))
    return int(n)


def nbk_open_ws(device: int, n_max: int, ni_max: int, cuda_stream: int, workspace: int, workspace_bytes: int):
    """workspace: device address (e.g. tensor.data_ptr()) the caller keeps alive."""
    ctx = _vp()
    _check("nbk_open_ws", load().nbk_open_ws(ctypes.byref(ctx), device, n_max, ni_max, cuda_stream or None,
                                             workspace or None, workspace_bytes))
    return ctx


def nbk_close(ctx):
    _check("nbk_close", load().nbk_close(ctx))


def nbk_npipes(ctx) -> int:
    return load().nbk_npipes(ctx)


def _set_j(fn_name, dtype, ctx, addr, tj, m, x, v, a, jerk):
    m_, pm = _host(m, dtype)
    n = 0 if m_ is None else m_.shape[0]
    ad_, pad = _host(addr, np.int32)
    tj_, ptj = _host(tj, np.float64)
    x_, px = _host(x, dtype, (3,))
    v_, pv = _host(v, dtype, (3,))
    a_, pa = _host(a, dtype, (3,))
    k_, pk = _host(jerk, dtype, (3,))
    for arr in (ad_, tj_, x_, v_, a_, k_):
        if arr is not None and arr.shape[0] != n:
            raise ValueError("set_j: arrays differ in length")
    _check(fn_name, getattr(load(), fn_name)(ctx, n, pad, ptj, pm, px, pv, pa, pk), ctx)


def nbk_set_j_particles(ctx, addr, tj, m, x, v=None, a=None, jerk=None):
    _set_j("nbk_set_j_particles", np.float32, ctx, addr, tj, m, x, v, a, jerk)


def nbk_set_j_particles_f64(ctx, addr, tj, m, x, v=None, a=None, jerk=None):
    _set_j("nbk_set_j_particles_f64", np.float64, ctx, addr, tj, m, x, v, a, jerk)


def nbk_set_j_particles_dev(ctx, n, addr, tj, m, x, v=0, a=0, jerk=0):
    _check("nbk_set_j_particles_dev",
           load().nbk_set_j_particles_dev(ctx, n, addr or None, tj or None, m or None, x or None,
                                          v or None, a or None, jerk or None), ctx)


def nbk_set_ti(ctx, t: float):
    _check("nbk_set_ti", load().nbk_set_ti(ctx, float(t)), ctx)


def nbk_predict(ctx, n_j: int):
    _check("nbk_predict", load().nbk_predict(ctx, n_j), ctx)


def nbk_get_predicted(ctx, n_j: int):
    m = np.empty(n_j, np.float32)
    x = np.empty((n_j, 3), np.float32)
    v = np.empty((n_j, 3), np.float32)
    _check("nbk_get_predicted",
           load().nbk_get_predicted(ctx, n_j, m.ctypes.data, x.ctypes.data, v.ctypes.data), ctx)
    return m, x, v


def nbk_calc_firsthalf(ctx, n_j, n_i, i_index=None, xi=None, vi=None, eps2=0.0, flags=NBK_JERK | NBK_POT):
    ii, pii = _host(i_index, np.int32)
    xi_, pxi = _host(xi, np.float32, (3,))
    vi_, pvi = _host(vi, np.float32, (3,))
    for arr in (ii, xi_, vi_):
        if arr is not None and arr.shape[0] != n_i:
            raise ValueError("firsthalf: i arrays must have n_i rows")
    _check("nbk_calc_firsthalf",
           load().nbk_calc_firsthalf(ctx, n_j, n_i, pii, pxi, pvi, float(eps2), flags), ctx)


def nbk_calc_firsthalf_dev(ctx, n_j, n_i, i_index=0, xi=0, vi=0, eps2=0.0, flags=NBK_JERK | NBK_POT):
    _check("nbk_calc_firsthalf_dev",
           load().nbk_calc_firsthalf_dev(ctx, n_j, n_i, i_index or None, xi or None, vi or None,
                                         float(eps2), flags), ctx)


def nbk_calc_lasthalf(ctx, n_i, out=None):
    """out: optional (acc [n_i,3], jerk [n_i,3], pot [n_i]) float32 C-contiguous arrays to fill, e.g. views
    of pinned memory (the library then copies device -> caller directly); default: fresh arrays."""
    if out is None:
        acc = np.empty((n_i, 3), np.float32)
        jerk = np.empty((n_i, 3), np.float32)
        pot = np.empty(n_i, np.float32)
    else:
        acc, jerk, pot = out
        for arr, shape in ((acc, (n_i, 3)), (jerk, (n_i, 3)), (pot, (n_i,))):
            if not (isinstance(arr, np.ndarray) and arr.dtype == np.float32 and arr.flags.c_contiguous
                    and arr.shape == shape):
                raise ValueError("lasthalf: out arrays must be C-contiguous float32 of shapes [n_i,3], [n_i,3], [n_i]")
    _check("nbk_calc_lasthalf",
           load().nbk_calc_lasthalf(ctx, n_i, acc.ctypes.data, jerk.ctypes.data, pot.ctypes.data), ctx)
    return acc, jerk, pot


def nbk_calc_lasthalf_f64(ctx, n_i):
    acc = np.empty((n_i, 3), np.float64)
    jerk = np.empty((n_i, 3), np.float64)
    pot = np.empty(n_i, np.float64)
    _check("nbk_calc_lasthalf_f64",
           load().nbk_calc_lasthalf_f64(ctx, n_i, acc.ctypes.data, jerk.ctypes.data, pot.ctypes.data), ctx)
    return acc, jerk, pot


def nbk_calc_lasthalf_dev(ctx, n_i, acc=0, jerk=0, pot=0):
    _check("nbk_calc_lasthalf_dev",
           load().nbk_calc_lasthalf_dev(ctx, n_i, acc or None, jerk or None, pot or None), ctx)


def nbk_calc_noalloc_dev(device, cuda_stream, n_j, m, x, v, n_i, i_index=0, eps2=0.0, flags=NBK_JERK | NBK_POT,
                         acc=0, jerk=0, pot=0):
    """The context-free force call for callers that must not allocate device memory (include/nbk.h).
    m, x, v, i_index, acc, jerk, pot: device addresses (0 = NULL); cuda_stream: a cudaStream_t value (0 = the
    legacy default stream).  Enqueues and returns; sizes beyond NBK_NOALLOC_MAX_NI / _NJ raise (NBK_ERANGE)."""
    err = _i32(0)
    st = load().nbk_calc_noalloc_dev(device, cuda_stream or None, n_j, m or None, x or None, v or None, n_i,
                                     i_index or None, float(eps2), flags, acc or None, jerk or None, pot or None,
                                     ctypes.byref(err))
    if st != NBK_OK:
        raise NbkError("nbk_calc_noalloc_dev", st, err.value)


def nbk_calc_batch(ctx, i_offset, xi, j_offset, mj, xj, eps2=0.0, flags=NBK_POT):
    """Host arrays in, (acc[n_i,3], pot[n_i]) out."""
    io, pio = _host(i_offset, np.int64)
    jo, pjo = _host(j_offset, np.int64)
    xi_, pxi = _host(xi, np.float32, (3,))
    mj_, pmj = _host(mj, np.float32)
    xj_, pxj = _host(xj, np.float32, (3,))
    n_groups = io.shape[0] - 1
    if jo.shape[0] != n_groups + 1 or xi_.shape[0] != io[-1] or mj_.shape[0] != jo[-1] or xj_.shape[0] != jo[-1]:
        raise ValueError("calc_batch: offsets and arrays disagree")
    acc = np.empty((xi_.shape[0], 3), np.float32)
    pot = np.empty(xi_.shape[0], np.float32)
    _check("nbk_calc_batch", load().nbk_calc_batch(ctx, n_groups, pio, pxi, pjo, pmj, pxj, float(eps2), flags,
                                                   acc.ctypes.data, pot.ctypes.data), ctx)
    return acc, pot


def nbk_calc_batch_dev(ctx, i_offset, xi, j_offset, mj, xj, eps2, flags, acc, pot):
    """i_offset, j_offset: host int64 arrays; xi, mj, xj, acc, pot: device addresses."""
    io, pio = _host(i_offset, np.int64)
    jo, pjo = _host(j_offset, np.int64)
    _check("nbk_calc_batch_dev", load().nbk_calc_batch_dev(ctx, io.shape[0] - 1, pio, xi or None, pjo, mj or None,
                                                           xj or None, float(eps2), flags, acc or None, pot or None), ctx)


def nbk_get_neighbours(ctx, n_i):
    nn = np.empty(n_i, np.int32)
    r2 = np.empty(n_i, np.float32)
    _check("nbk_get_neighbours", load().nbk_get_neighbours(ctx, n_i, nn.ctypes.data, r2.ctypes.data), ctx)
    return nn, r2


def nbk_get_neighbours_dev(ctx, n_i, nn_index=0, nn_r2=0):
    _check("nbk_get_neighbours_dev",
           load().nbk_get_neighbours_dev(ctx, n_i, nn_index or None, nn_r2 or None), ctx)


def nbk_shard_gather_i_dev(ctx, n_local, j0, n_i, i_global, i_local, xv):
    """All array arguments are device addresses (see include/nbk.h, j-sharding)."""
    _check("nbk_shard_gather_i_dev",
           load().nbk_shard_gather_i_dev(ctx, n_local, j0, n_i, i_global or None, i_local or None, xv or None), ctx)


def nbk_shard_calc_partial_dev(ctx, n_local, n_i, i_local, xv, eps2, flags, sum64):
    _check("nbk_shard_calc_partial_dev",
           load().nbk_shard_calc_partial_dev(ctx, n_local, n_i, i_local or None, xv or None, float(eps2), flags,
                                             sum64 or None), ctx)


def nbk_shard_finish_dev(ctx, n_i, sum64, acc=0, jerk=0, pot=0):
    _check("nbk_shard_finish_dev",
           load().nbk_shard_finish_dev(ctx, n_i, sum64 or None, acc or None, jerk or None, pot or None), ctx)


def nbk_shard_fetch_i_dev(ctx, n_i, i_global, shard_begin, peer_xv, xv):
    """shard_begin: world + 1 global addresses; peer_xv: world device addresses (host sequences)."""
    begin = np.ascontiguousarray(shard_begin, dtype=np.int64)
    ptrs = (_vp * len(peer_xv))(*[int(p) for p in peer_xv])
    if begin.shape[0] != len(peer_xv) + 1:
        raise ValueError("shard_fetch_i: shard_begin must have world + 1 entries")
    _check("nbk_shard_fetch_i_dev",
           load().nbk_shard_fetch_i_dev(ctx, n_i, len(peer_xv), i_global or None, begin.ctypes.data, ptrs, xv or None), ctx)


def nbk_shard_combine_dev(ctx, n_i, peer_sum64, acc=0, jerk=0, pot=0):
    ptrs = (_vp * len(peer_sum64))(*[int(p) for p in peer_sum64])
    _check("nbk_shard_combine_dev",
           load().nbk_shard_combine_dev(ctx, n_i, len(peer_sum64), ptrs, acc or None, jerk or None, pot or None), ctx)


def nbk_hermite_evolve_dev(ctx, m, x, v, eps, t_end, eta=0.01, dt_max=1.0 / 16.0):
    """Device-resident block-step loop; same arguments and return value as nbk_hermite_evolve."""
    return nbk_hermite_evolve(ctx, m, x, v, eps, t_end, eta, dt_max, _fn="nbk_hermite_evolve_dev")


def nbk_hermite_evolve(ctx, m, x, v, eps, t_end, eta=0.01, dt_max=1.0 / 16.0, _fn="nbk_hermite_evolve"):
    """x, v: float64 [n,3] arrays updated IN PLACE.  Returns a dict of nbk_hermite_stats."""
    m = np.ascontiguousarray(m, np.float64)
    if not (isinstance(x, np.ndarray) and x.dtype == np.float64 and x.flags.c_contiguous
            and isinstance(v, np.ndarray) and v.dtype == np.float64 and v.flags.c_contiguous):
        raise ValueError("x, v must be C-contiguous float64 arrays (updated in place)")
    n = m.shape[0]
    if x.shape != (n, 3) or v.shape != (n, 3):
        raise ValueError("x, v must be [n,3]")
    st = HermiteStats()
    _check(_fn,
           getattr(load(), _fn)(ctx, n, m.ctypes.data, x.ctypes.data, v.ctypes.data, float(eps),
                                     float(t_end), float(eta), float(dt_max), ctypes.byref(st)), ctx)
    out = {k: getattr(st, k) for k, _ in HermiteStats._fields_ if k != "ni_histogram"}
    out["ni_histogram"] = list(st.ni_histogram)
    return out


def nbk_sync(ctx):
    _check("nbk_sync", load().nbk_sync(ctx), ctx)


def nbk_set_timing(ctx, enable: bool):
    _check("nbk_set_timing", load().nbk_set_timing(ctx, int(bool(enable))), ctx)


def nbk_get_timing(ctx):
    ms = (_f32 * 4)()
    _check("nbk_get_timing", load().nbk_get_timing(ctx, ctypes.byref(ms)), ctx)
    return dict(scatter=ms[0], predict=ms[1], force=ms[2], reduce=ms[3])


def nbk_last_launch(ctx):
    out = (_i64 * 8)()
    _check("nbk_last_launch", load().nbk_last_launch(ctx, ctypes.byref(out)), ctx)
    keys = ["grid", "threads", "i_per_thread", "j_split_warps", "j_tile", "sms", "smem_bytes", "launches"]
    return dict(zip(keys, list(out)))


def nbk_plan(n_i: int, n_j: int, num_sms: int = 148, force_i: int = 0):
    out = (_i64 * 12)()
    _check("nbk_plan", load().nbk_plan(n_i, n_j, num_sms, force_i, ctypes.byref(out)))
    keys = ["i_per_thread", "threads", "i_tile", "j_tile", "j_split_warps", "i_tiles", "j_tiles", "pairs",
            "grid", "max_segments", "partial_floats", "partial_floats_bound"]
    return dict(zip(keys, list(out)))


def nbk_set_variant(ctx, variant: int):
    _check("nbk_set_variant", load().nbk_set_variant(ctx, variant), ctx)


def nbk_version() -> str:
    return load().nbk_version().decode()
