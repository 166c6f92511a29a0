"""Thin ctypes binding of libtoi (include/toi.h): argument marshalling only.

Function names are the C ABI's.  Tensors are passed as raw pointers (``tensor.data_ptr()``),
streams as ``torch.cuda.Stream.cuda_stream``; torch is used for device/pinned memory and streams
only.  There is no CPU fallback: a missing library or a missing GPU raises.
"""
from __future__ import annotations

import ctypes as C
import os

import torch

from . import build as _build

TOI_OK = 0
TOI_ERR_INVALID_ARG, TOI_ERR_CUDA, TOI_ERR_CUFFT, TOI_ERR_NOMEM = -1, -2, -3, -4
TOI_ERR_DEGENERATE_GEOMETRY, TOI_ERR_CALLBACK, TOI_ERR_UNSUPPORTED = -5, -6, -7
TOI_WEIGHT_NATURAL, TOI_WEIGHT_UNIFORM = 0, 1
TOI_MEM_HOST, TOI_MEM_DEVICE = 0, 1
TOI_GRIDDER_SLIDING, TOI_GRIDDER_ATOMIC = 0, 1
TOI_REPROJECT_EXACT, TOI_REPROJECT_PAPER = 0, 1
TOI_OUT_TILTED, TOI_OUT_REPROJECT_EXACT, TOI_OUT_REPROJECT_PAPER = 0, 1, 2

EXPORTS = ["toi_plan_create", "toi_plan_destroy", "toi_image_snapshot", "toi_plan_sync",
           "toi_copy_image_to_host", "toi_image_stream", "toi_stream_set_output", "toi_image_snapshot_3d",
           "toi_reproject", "toi_difference",
           "toi_last_error", "toi_last_launch_count",
           "toi_debug_set_transform", "toi_debug_cell_indices", "toi_debug_keep_grid",
           "toi_debug_copy_grid", "toi_debug_copy_density", "toi_cell_indices_static"]


class toi_config(C.Structure):
    _fields_ = [("n_baselines", C.c_int32), ("n_channels", C.c_int32), ("n_pols", C.c_int32),
                ("pol_a", C.c_int32), ("pol_b", C.c_int32), ("chan_freq_hz", C.POINTER(C.c_double)),
                ("image_size", C.c_int32), ("cell_size_deg", C.c_double), ("weighting", C.c_int32),
                ("grid_size", C.c_int32), ("kernel_support", C.c_int32), ("apply_jacobian", C.c_int32),
                ("input_location", C.c_int32), ("image_ring_depth", C.c_int32), ("device", C.c_int32),
                ("gridder", C.c_int32), ("enable_3d", C.c_int32), ("debug_keep_grid", C.c_int32),
                ("reserved", C.c_int32 * 5)]


class toi_snapshot_info(C.Structure):
    _fields_ = [("V", C.c_double * 9), ("omega", C.c_double), ("sing", C.c_double * 3),
                ("wsum", C.c_double), ("n_gridded", C.c_int64), ("n_off_grid", C.c_int64),
                ("n_flagged", C.c_int64), ("ms_h2d", C.c_float), ("ms_planefit", C.c_float),
                ("ms_weight", C.c_float), ("ms_grid", C.c_float), ("ms_fft", C.c_float),
                ("ms_crop", C.c_float), ("ms_total", C.c_float), ("ms_clear", C.c_float), ("ms_clear_density", C.c_float)]

    def as_dict(self):
        d = {k: getattr(self, k) for k, _ in self._fields_ if k not in ("V", "sing")}
        d["V"] = [list(self.V[3 * r:3 * r + 3]) for r in range(3)]
        d["sing"] = list(self.sing)
        return d


class toi_3d_info(C.Structure):
    _fields_ = [("n_slab", C.c_int32), ("K", C.c_int32), ("n_passes", C.c_int32), ("reserved", C.c_int32),
                ("phi_max", C.c_double), ("t3_max", C.c_double), ("r3_min", C.c_double), ("r3_max", C.c_double),
                ("alpha_slab", C.c_double), ("expansion_error", C.c_double), ("ms_total", C.c_float)]

    def as_dict(self):
        return {k: getattr(self, k) for k, _ in self._fields_ if k != "reserved"}


class toi_snapshot_buffers(C.Structure):
    _fields_ = [("uvw_m", C.c_void_p), ("vis", C.c_void_p), ("weights", C.c_void_p), ("flags", C.c_void_p)]


class toi_stream_stats(C.Structure):
    _fields_ = [("n_done", C.c_int64), ("wall_s", C.c_double), ("gpu_ms", C.c_double),
                ("h2d_bytes", C.c_double), ("h2d_ms_sum", C.c_double), ("compute_ms_sum", C.c_double),
                ("d2h_bytes", C.c_double), ("d2h_ms_sum", C.c_double)]

    def as_dict(self):
        return {k: getattr(self, k) for k, _ in self._fields_}


toi_fill_fn = C.CFUNCTYPE(C.c_int, C.c_void_p, C.c_int64, C.POINTER(toi_snapshot_buffers))
toi_sink_fn = C.CFUNCTYPE(C.c_int, C.c_void_p, C.c_int64, C.c_void_p, C.c_void_p, C.POINTER(toi_snapshot_info))
toi_host_sink_fn = C.CFUNCTYPE(C.c_int, C.c_void_p, C.c_int64, C.c_void_p)


class toi_stream_output(C.Structure):
    _fields_ = [("product", C.c_int32), ("difference", C.c_int32), ("to_host", C.c_int32),
                ("reserved", C.c_int32 * 5), ("host_sink", toi_host_sink_fn), ("host_user", C.c_void_p)]


_host_sinks = {}      # plan address -> ctypes callback kept alive while the plan may call it

_lib = None


class ToiError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__("libtoi error %d: %s" % (code, msg))
        self.code = code


def library_path() -> str:
    return _build.LIB


def load(build_if_missing: bool = True):
    """dlopen libtoi.so (building it in-tree first if asked and needed) and declare prototypes."""
    global _lib
    if _lib is not None:
        return _lib
    if build_if_missing and _build.needs_build():
        _build.build_library()
    if not os.path.exists(_build.LIB):
        raise RuntimeError("libtoi.so is missing (run python -m paper_2512_06254_b200.build); there is no CPU fallback")
    lib = C.CDLL(_build.LIB)
    vp, i32, i64 = C.c_void_p, C.c_int32, C.c_int64
    lib.toi_plan_create.argtypes = [C.POINTER(toi_config), C.POINTER(vp)]
    lib.toi_plan_destroy.argtypes = [vp]
    lib.toi_image_snapshot.argtypes = [vp, vp, vp, vp, vp, vp, C.POINTER(vp), C.POINTER(toi_snapshot_info)]
    lib.toi_plan_sync.argtypes = [vp]
    lib.toi_copy_image_to_host.argtypes = [vp, vp, vp]
    lib.toi_image_stream.argtypes = [vp, i64, toi_fill_fn, vp, toi_sink_fn, vp, i32, C.POINTER(toi_stream_stats)]
    lib.toi_stream_set_output.argtypes = [vp, C.POINTER(toi_stream_output)]
    lib.toi_image_snapshot_3d.argtypes = [vp, vp, vp, vp, vp, vp, i32, i32, C.POINTER(vp), C.POINTER(toi_3d_info),
                                          C.POINTER(toi_snapshot_info)]
    lib.toi_reproject.argtypes = [vp, vp, vp, i32, vp, vp]
    lib.toi_difference.argtypes = [vp, vp, vp, vp, vp]
    lib.toi_last_error.argtypes = [vp]
    lib.toi_last_error.restype = C.c_char_p
    lib.toi_last_launch_count.argtypes = [vp]
    lib.toi_debug_set_transform.argtypes = [vp, vp]
    lib.toi_debug_cell_indices.argtypes = [vp, vp, vp]
    lib.toi_debug_keep_grid.argtypes = [vp, i32]
    lib.toi_debug_copy_grid.argtypes = [vp, vp]
    lib.toi_debug_copy_density.argtypes = [vp, vp]
    for name in EXPORTS:
        if name != "toi_last_error":
            getattr(lib, name).restype = C.c_int
    _lib = lib
    return lib


def _ptr(t):
    return None if t is None else C.c_void_p(t.data_ptr())


def _check(plan, rc, allow=()):
    if rc != TOI_OK and rc not in allow:
        msg = load().toi_last_error(plan).decode(errors="replace")
        raise ToiError(rc, msg)
    return rc


def toi_plan_create(n_baselines, n_channels, n_pols, chan_freq_hz, image_size, cell_size_deg,
                    weighting=TOI_WEIGHT_NATURAL, pol_a=None, pol_b=None, grid_size=0, kernel_support=0,
                    apply_jacobian=0, input_location=TOI_MEM_DEVICE, image_ring_depth=0, device=0,
                    gridder=TOI_GRIDDER_SLIDING, enable_3d=False, debug_keep_grid=False):
    """-> opaque plan handle (c_void_p).  chan_freq_hz: host float64 tensor/sequence [n_channels]."""
    lib = load()
    freq = torch.as_tensor(chan_freq_hz, dtype=torch.float64, device="cpu").contiguous()
    cfg = toi_config()
    cfg.n_baselines, cfg.n_channels, cfg.n_pols = int(n_baselines), int(n_channels), int(n_pols)
    cfg.pol_a = 0 if pol_a is None else int(pol_a)
    cfg.pol_b = (n_pols - 1) if pol_b is None else int(pol_b)
    cfg.chan_freq_hz = C.cast(C.c_void_p(freq.data_ptr()), C.POINTER(C.c_double))
    cfg.image_size, cfg.cell_size_deg = int(image_size), float(cell_size_deg)
    cfg.weighting, cfg.grid_size, cfg.kernel_support = int(weighting), int(grid_size), int(kernel_support)
    cfg.apply_jacobian, cfg.input_location = int(apply_jacobian), int(input_location)
    cfg.image_ring_depth, cfg.device, cfg.gridder = int(image_ring_depth), int(device), int(gridder)
    cfg.enable_3d, cfg.debug_keep_grid = int(bool(enable_3d)), int(bool(debug_keep_grid))
    plan = C.c_void_p()
    rc = lib.toi_plan_create(C.byref(cfg), C.byref(plan))
    _check(None, rc)
    return plan


def toi_plan_destroy(plan):
    _host_sinks.pop(getattr(plan, "value", None), None)
    return load().toi_plan_destroy(plan)


def toi_image_snapshot(plan, uvw_m, vis, weights=None, flags=None, stream=None, want_info=False,
                       allow_degenerate=False):
    """Tensors live where the plan's input_location says.  -> (device image pointer int, info|None, rc)."""
    lib = load()
    out = C.c_void_p()
    info = toi_snapshot_info() if want_info else None
    s = None if stream is None else C.c_void_p(stream.cuda_stream)
    rc = lib.toi_image_snapshot(plan, _ptr(uvw_m), _ptr(vis), _ptr(weights), _ptr(flags), s, C.byref(out),
                                C.byref(info) if want_info else None)
    _check(plan, rc, allow=(TOI_ERR_DEGENERATE_GEOMETRY,) if allow_degenerate else ())
    return out.value, info, rc


def toi_image_snapshot_3d(plan, uvw_m, vis, weights=None, flags=None, stream=None, n_slab=0, K=0, want_info=True):
    """Near-coplanar (3-D) mode.  -> (device image pointer int, toi_3d_info dict, toi_snapshot_info|None)."""
    lib = load()
    out = C.c_void_p()
    i3 = toi_3d_info()
    info = toi_snapshot_info() if want_info else None
    s = None if stream is None else C.c_void_p(stream.cuda_stream)
    rc = lib.toi_image_snapshot_3d(plan, _ptr(uvw_m), _ptr(vis), _ptr(weights), _ptr(flags), s, int(n_slab), int(K),
                                   C.byref(out), C.byref(i3), C.byref(info) if want_info else None)
    _check(plan, rc)
    return out.value, i3.as_dict(), info


def toi_plan_sync(plan, allow=()):
    return _check(plan, load().toi_plan_sync(plan), allow)


def toi_copy_image_to_host(plan, d_image, image_size, out=None):
    """-> float32 CPU tensor [N, N] (``out`` if given, e.g. a pinned tensor)."""
    h = torch.empty((image_size, image_size), dtype=torch.float32) if out is None else out
    assert h.dtype == torch.float32 and h.numel() == image_size * image_size and h.is_contiguous()
    _check(plan, load().toi_copy_image_to_host(plan, C.c_void_p(d_image), C.c_void_p(h.data_ptr())))
    return h


def toi_image_stream(plan, n_snapshots, fill, sink=None, want_info=False):
    """fill(idx, slot: toi_snapshot_buffers) -> 0/1/<0 ; sink(idx, d_image:int, stream:int, info|None) -> int.
    -> stats dict."""
    lib = load()

    def _fill(user, idx, slot):
        try:
            return int(fill(idx, slot.contents))
        except Exception:      # never unwind through C
            import traceback
            traceback.print_exc()
            return -1

    def _sink(user, idx, d_image, stream, info):
        try:
            r = sink(idx, d_image, stream, info.contents if info else None)
            return 0 if r is None else int(r)
        except Exception:
            import traceback
            traceback.print_exc()
            return -1

    cfill = toi_fill_fn(_fill)
    csink = toi_sink_fn(_sink) if sink is not None else C.cast(None, toi_sink_fn)
    stats = toi_stream_stats()
    rc = lib.toi_image_stream(plan, int(n_snapshots), cfill, None, csink, None, 1 if want_info else 0, C.byref(stats))
    _check(plan, rc)
    return stats.as_dict()


def toi_stream_set_output(plan, product=TOI_OUT_TILTED, difference=False, host_sink=None, image_size=None):
    """Output side of toi_image_stream.  host_sink(idx, image: float32 numpy view [N, N] of the pinned
    slot, valid during the call) -> None/int enables the D2H ring; product/difference as in toi.h.
    Call with no arguments to restore the default."""
    import numpy as np
    cb = C.cast(None, toi_host_sink_fn)
    if host_sink is not None:
        assert image_size, "image_size is needed to view the host image"
        n = int(image_size)

        def _hs(user, idx, h_image):
            try:
                buf = (C.c_float * (n * n)).from_address(h_image)
                r = host_sink(idx, np.frombuffer(buf, dtype=np.float32).reshape(n, n))
                return 0 if r is None else int(r)
            except Exception:      # never unwind through C
                import traceback
                traceback.print_exc()
                return -1

        cb = toi_host_sink_fn(_hs)
    o = toi_stream_output(int(product), 1 if difference else 0, 0 if host_sink is None else 1)
    o.host_sink = cb
    rc = load().toi_stream_set_output(plan, C.byref(o))
    _check(plan, rc)
    _host_sinks[plan.value] = cb
    return rc


def _dev(x):
    """A device address: a CUDA tensor or the int toi_image_snapshot returned."""
    return C.c_void_p(x) if isinstance(x, int) else _ptr(x)


def toi_reproject(plan, d_image, out, V=None, mode=TOI_REPROJECT_EXACT, stream=None):
    """d_image: device pointer (int) or CUDA tensor [N, N] f32 on the tilted plane; out: CUDA tensor
    [N, N] f32 (written); V: 3x3 (host) or None = the plan's last snapshot.  Enqueues only."""
    v = None
    if V is not None:
        v = torch.as_tensor(V, dtype=torch.float64, device="cpu").contiguous().reshape(9)
    s = None if stream is None else C.c_void_p(stream.cuda_stream)
    _check(plan, load().toi_reproject(plan, _dev(d_image), None if v is None else C.c_void_p(v.data_ptr()),
                                      int(mode), s, _dev(out)))
    return out


def toi_difference(plan, d_a, d_b, out, stream=None):
    """out = a - b, device [N, N] f32 each (pointers or CUDA tensors).  Enqueues only."""
    s = None if stream is None else C.c_void_p(stream.cuda_stream)
    _check(plan, load().toi_difference(plan, _dev(d_a), _dev(d_b), s, _dev(out)))
    return out


def toi_last_error(plan=None):
    return load().toi_last_error(plan).decode(errors="replace")


def toi_last_launch_count(plan):
    return load().toi_last_launch_count(plan)


def toi_debug_set_transform(plan, V):
    if V is None:
        return _check(plan, load().toi_debug_set_transform(plan, None))
    v = torch.as_tensor(V, dtype=torch.float64, device="cpu").contiguous().reshape(9)
    return _check(plan, load().toi_debug_set_transform(plan, C.c_void_p(v.data_ptr())))


def toi_debug_cell_indices(plan, n_baselines, n_channels, device="cuda"):
    iu = torch.empty((n_baselines, n_channels), dtype=torch.int32, device=device)
    iv = torch.empty_like(iu)
    _check(plan, load().toi_debug_cell_indices(plan, _ptr(iu), _ptr(iv)))
    return iu, iv


TOI_STATIC_MAX_CHANNELS = 32768


def toi_cell_indices_static(uvw_m, chan_freq_hz, grid_size, cell_size_deg, iu, iv, fit_out=None, stream=None):
    """Steps a1-a3 without a plan and without any allocation (include/toi.h): fills the caller's device
    tensors iu, iv (int32 [n_baselines][n_channels]) and, if given, fit_out (float64 [13]: V, omega, sing)."""
    lib = load()
    freq = torch.as_tensor(chan_freq_hz, dtype=torch.float64, device="cpu").contiguous()
    err = C.create_string_buffer(256)
    st = stream if stream is not None else torch.cuda.current_stream(uvw_m.device)
    rc = lib.toi_cell_indices_static(_ptr(uvw_m), C.c_int32(uvw_m.shape[0]), C.c_void_p(freq.data_ptr()),
                                     C.c_int32(freq.numel()), C.c_int32(grid_size), C.c_double(cell_size_deg),
                                     C.c_void_p(st.cuda_stream), _ptr(iu), _ptr(iv), _ptr(fit_out), err, C.c_int32(256))
    if rc != TOI_OK:
        raise ToiError(rc, err.value.decode(errors="replace"))
    return rc


def toi_debug_keep_grid(plan, on=True):
    return _check(plan, load().toi_debug_keep_grid(plan, 1 if on else 0))


def toi_debug_copy_grid(plan, G, device="cuda"):
    g = torch.empty((G, G), dtype=torch.complex64, device=device)
    _check(plan, load().toi_debug_copy_grid(plan, _ptr(g)))
    return g


def toi_debug_copy_density(plan, G, device="cuda"):
    d = torch.empty((G, G), dtype=torch.float32, device=device)
    _check(plan, load().toi_debug_copy_density(plan, _ptr(d)))
    return d
