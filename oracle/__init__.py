"""oracle -- TEST INFRASTRUCTURE, not product code.

ctypes front end of ``oracle/toi_oracle.c``: the plain fp64 CPU statement of the TOI (2-D)
snapshot imager of arxiv 2512.06254 (readings in DESIGN.md section 3).
Only ``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s ``cpu_baseline`` /
``--impl reference`` legs may import this package.  It imports nothing of
``paper_2512_06254_b200`` and the CUDA path imports nothing of it.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
import threading

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "toi_oracle.c")
_LIB = os.path.join(_HERE, "libtoi_oracle.so")
_lock = threading.Lock()
_lib = None

NATURAL, UNIFORM = 0, 1
BASIS_MINIMAL, BASIS_PRINCIPAL = 0, 1
ERR_DEGENERATE = -5


class OrcConfig(C.Structure):
    _fields_ = [("n_b", C.c_int32), ("n_c", C.c_int32), ("n_p", C.c_int32),
                ("pol_a", C.c_int32), ("pol_b", C.c_int32), ("N", C.c_int32),
                ("cell_size_deg", C.c_double), ("weighting", C.c_int32), ("G", C.c_int32),
                ("W", C.c_int32), ("apply_jacobian", C.c_int32), ("basis", C.c_int32)]


class OrcInfo(C.Structure):
    _fields_ = [("V", C.c_double * 9), ("omega", C.c_double), ("sing", C.c_double * 3),
                ("wsum", C.c_double), ("n_gridded", C.c_int64), ("n_off_grid", C.c_int64),
                ("n_flagged", C.c_int64)]


def build(force: bool = False) -> str:
    """Compile toi_oracle.c into oracle/libtoi_oracle.so (gcc, fp64, OpenMP, no contraction)."""
    with _lock:
        if (not force and os.path.exists(_LIB)
                and os.path.getmtime(_LIB) >= os.path.getmtime(_SRC)):
            return _LIB
        tmp = _LIB + ".tmp.%d" % os.getpid()
        cmd = ["gcc", "-O2", "-ffp-contract=off", "-fopenmp", "-shared", "-fPIC", "-std=c11",
               "-Wall", "-o", tmp, _SRC, "-lm"]
        subprocess.run(cmd, check=True)
        os.replace(tmp, _LIB)
        return _LIB


def lib():
    global _lib
    if _lib is None:
        _lib = C.CDLL(build())
        _lib.toi_oracle_kappa.restype = C.c_double
        _lib.toi_oracle_kappa.argtypes = [C.c_int32, C.c_double]
        _lib.toi_oracle_phi.restype = C.c_double
        _lib.toi_oracle_phi.argtypes = [C.c_double, C.c_int32]
        _lib.toi_oracle_psi.restype = C.c_double
        _lib.toi_oracle_psi.argtypes = [C.c_int32, C.c_int32, C.c_int32, C.c_int32]
        _lib.toi_oracle_num_threads.restype = C.c_int
    return _lib


def _p(a, ctype):
    return None if a is None else a.ctypes.data_as(C.POINTER(ctype))


def _f64(a):
    return np.ascontiguousarray(a, dtype=np.float64)


def _cfg(n_b, n_c, n_p, N, cell_size_deg, weighting=NATURAL, G=0, W=0, pol_a=None, pol_b=None,
         apply_jacobian=1, basis=BASIS_MINIMAL):
    if pol_a is None:
        pol_a = 0
    if pol_b is None:
        pol_b = n_p - 1
    return OrcConfig(n_b, n_c, n_p, pol_a, pol_b, N, float(cell_size_deg), weighting, G, W,
                     apply_jacobian, basis)


def _check_inputs(uvw_m, vis, weights, flags, chan_freq_hz):
    uvw_m = _f64(uvw_m)
    vis = np.ascontiguousarray(vis, dtype=np.complex64)
    n_b, n_c, n_p = vis.shape
    assert uvw_m.shape == (n_b, 3)
    chan_freq_hz = _f64(chan_freq_hz)
    assert chan_freq_hz.shape == (n_c,)
    if weights is not None:
        weights = np.ascontiguousarray(weights, dtype=np.float32)
        assert weights.shape == vis.shape
    if flags is not None:
        flags = np.ascontiguousarray(flags, dtype=np.uint8)
        assert flags.shape == vis.shape
    return uvw_m, vis, weights, flags, chan_freq_hz


def _info_dict(info):
    return {"V": np.array(info.V, dtype=np.float64).reshape(3, 3), "omega": info.omega,
            "sing": np.array(info.sing, dtype=np.float64), "wsum": info.wsum,
            "n_gridded": info.n_gridded, "n_off_grid": info.n_off_grid,
            "n_flagged": info.n_flagged}


def chan_scale(chan_freq_hz):
    f = _f64(chan_freq_hz)
    s = np.empty_like(f)
    lib().toi_oracle_chan_scale(C.c_int32(f.size), _p(f, C.c_double), _p(s, C.c_double))
    return s


def plane_fit(uvw_m, chan_freq_hz, basis=BASIS_MINIMAL):
    """-> (rc, V[3,3], omega, sing[3])."""
    uvw_m = _f64(uvw_m)
    s = chan_scale(chan_freq_hz)
    V = np.zeros(9)
    sing = np.zeros(3)
    om = C.c_double(0.0)
    rc = lib().toi_oracle_plane_fit(C.c_int32(uvw_m.shape[0]), C.c_int32(s.size), _p(uvw_m, C.c_double),
                                    _p(s, C.c_double), C.c_int32(basis), _p(V, C.c_double),
                                    C.byref(om), _p(sing, C.c_double))
    return rc, V.reshape(3, 3), om.value, sing


def rotate(uvw_m, V):
    """rho = V uvw (metres)."""
    uvw_m = _f64(uvw_m)
    V = _f64(V).reshape(9)
    rho = np.empty_like(uvw_m)
    lib().toi_oracle_rotate(C.c_int32(uvw_m.shape[0]), _p(uvw_m, C.c_double), _p(V, C.c_double),
                            _p(rho, C.c_double))
    return rho


def cell_indices(rho, chan_freq_hz, G, cell_size_deg, W=7):
    """-> (iu, iv, on_grid) each [n_b, n_c]; DESIGN.md section 3 step 5."""
    rho = _f64(rho)
    s = chan_scale(chan_freq_hz)
    n_b, n_c = rho.shape[0], s.size
    iu = np.empty((n_b, n_c), np.int32)
    iv = np.empty((n_b, n_c), np.int32)
    on = np.empty((n_b, n_c), np.uint8)
    lib().toi_oracle_cell_indices(C.c_int32(n_b), C.c_int32(n_c), _p(rho, C.c_double), _p(s, C.c_double),
                                  C.c_int32(G), C.c_double(cell_size_deg), C.c_int32(W),
                                  _p(iu, C.c_int32), _p(iv, C.c_int32), _p(on, C.c_uint8))
    return iu, iv, on.astype(bool)


def kappa(G, cell_size_deg):
    return lib().toi_oracle_kappa(G, cell_size_deg)


def phi(x, W=7):
    return lib().toi_oracle_phi(float(x), W)


def psi(n, G, W=7, n_nodes=64):
    return lib().toi_oracle_psi(int(n), int(G), int(W), int(n_nodes))


def fft2(a, sign=+1):
    """Unnormalised 2-D transform, kernel exp(sign 2 pi i (k l + r m)/n); returns a new array."""
    a = np.array(a, dtype=np.complex128, order="C")
    assert a.ndim == 2 and a.shape[0] == a.shape[1]
    rc = lib().toi_oracle_fft2(a.ctypes.data_as(C.c_void_p), C.c_int32(a.shape[0]), C.c_int32(sign))
    assert rc == 0, rc
    return a


def image_gridded(uvw_m, vis, weights, flags, chan_freq_hz, N, cell_size_deg, weighting=NATURAL,
                  G=0, W=0, pol_a=None, pol_b=None, apply_jacobian=1, basis=BASIS_MINIMAL,
                  V_in=None, want_grid=False, want_density=False, want_indices=False):
    """Tier G. -> (rc, image[N,N] f64, info dict, extras dict)."""
    uvw_m, vis, weights, flags, chan_freq_hz = _check_inputs(uvw_m, vis, weights, flags, chan_freq_hz)
    n_b, n_c, n_p = vis.shape
    cfg = _cfg(n_b, n_c, n_p, N, cell_size_deg, weighting, G, W, pol_a, pol_b, apply_jacobian, basis)
    Gr = G if G > 0 else 2 * N
    image = np.zeros((N, N), np.float64)
    info = OrcInfo()
    grid = np.zeros((Gr, Gr), np.complex128) if want_grid else None
    dens = np.zeros((Gr, Gr), np.float64) if want_density else None
    iu = np.zeros((n_b, n_c), np.int32) if want_indices else None
    iv = np.zeros((n_b, n_c), np.int32) if want_indices else None
    Vin = None if V_in is None else _f64(V_in).reshape(9)
    rc = lib().toi_oracle_image_gridded(
        C.byref(cfg), _p(chan_freq_hz, C.c_double), _p(uvw_m, C.c_double),
        vis.ctypes.data_as(C.c_void_p), _p(weights, C.c_float), _p(flags, C.c_uint8),
        _p(Vin, C.c_double), _p(image, C.c_double), C.byref(info),
        None if grid is None else grid.ctypes.data_as(C.c_void_p), _p(dens, C.c_double),
        _p(iu, C.c_int32), _p(iv, C.c_int32))
    extras = {"grid": grid, "density": dens, "iu": iu, "iv": iv}
    return rc, image, _info_dict(info), extras


def image_dft_pixels(uvw_m, vis, weights, flags, chan_freq_hz, N, cell_size_deg, pix_i, pix_j,
                     weighting=NATURAL, G=0, W=0, pol_a=None, pol_b=None, apply_jacobian=1,
                     basis=BASIS_MINIMAL, V_in=None):
    """Tier D at the listed pixels (i = column, j = row). -> (rc, re[n], im[n], info dict)."""
    uvw_m, vis, weights, flags, chan_freq_hz = _check_inputs(uvw_m, vis, weights, flags, chan_freq_hz)
    n_b, n_c, n_p = vis.shape
    cfg = _cfg(n_b, n_c, n_p, N, cell_size_deg, weighting, G, W, pol_a, pol_b, apply_jacobian, basis)
    pi_ = np.ascontiguousarray(pix_i, dtype=np.int32).ravel()
    pj_ = np.ascontiguousarray(pix_j, dtype=np.int32).ravel()
    assert pi_.size == pj_.size
    re = np.zeros(pi_.size)
    im = np.zeros(pi_.size)
    info = OrcInfo()
    Vin = None if V_in is None else _f64(V_in).reshape(9)
    rc = lib().toi_oracle_image_dft_pixels(
        C.byref(cfg), _p(chan_freq_hz, C.c_double), _p(uvw_m, C.c_double),
        vis.ctypes.data_as(C.c_void_p), _p(weights, C.c_float), _p(flags, C.c_uint8),
        _p(Vin, C.c_double), C.c_int64(pi_.size), _p(pi_, C.c_int32), _p(pj_, C.c_int32),
        _p(re, C.c_double), _p(im, C.c_double), C.byref(info))
    return rc, re, im, _info_dict(info)


def image_dft(uvw_m, vis, weights, flags, chan_freq_hz, N, cell_size_deg, **kw):
    """Tier D for the full N x N image. -> (rc, image_re[N,N], image_im[N,N], info dict)."""
    jj, ii = np.meshgrid(np.arange(N, dtype=np.int32), np.arange(N, dtype=np.int32), indexing="ij")
    rc, re, im, info = image_dft_pixels(uvw_m, vis, weights, flags, chan_freq_hz, N, cell_size_deg,
                                        ii.ravel(), jj.ravel(), **kw)
    return rc, re.reshape(N, N), im.reshape(N, N), info


def last_stage_seconds():
    """Wall-clock seconds of the last image_gridded call per stage (instrumentation only)."""
    out = (C.c_double * 5)()
    lib().toi_oracle_last_stage_seconds(out)
    return dict(zip(("fit", "weight", "grid", "fft", "correct"), [float(x) for x in out]))


def num_threads():
    return int(lib().toi_oracle_num_threads())


def set_num_threads(n):
    lib().toi_oracle_set_num_threads(C.c_int(int(n)))
