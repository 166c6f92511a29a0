"""-m gpu parity tests of the re-projection stage (Eqs. 9-16) and the difference
image: libtoi's k_reproject / k_difference through the C ABI against oracle/reproject.py on the
same inputs, element by element.

Bar: the coordinates are fp64 on both sides and the bilinear blend is fp32 on the GPU, so a pixel
differs by a few fp32 roundings of values no larger than the image peak: max abs error
<= 2e-6 * peak (4 roundings of 2^-24 on the blend + the fp32 weights' 6e-8 times the local
contrast); the NaN mask is identical except where the oracle's own position lies within 1e-9 px of
the validity edge (G22).
"""
from __future__ import annotations

import math

import numpy as np
import pytest

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")

import oracle  # noqa: E402
from oracle import reproject as orp  # noqa: E402
from paper_2512_06254_b200 import binding as toi  # noqa: E402
from paper_2512_06254_b200 import synth  # noqa: E402

from gpu_helpers import GpuImager  # noqa: E402
from helpers import snapshot_np  # noqa: E402

MODES = {"exact": toi.TOI_REPROJECT_EXACT, "paper": toi.TOI_REPROJECT_PAPER}
BAR = 2e-6


@pytest.fixture(scope="module", autouse=True)
def _need_gpu():
    assert torch.cuda.is_available(), "the -m gpu tests need a CUDA device"
    toi.load()


def _plan(N, cell_deg):
    freq = np.array([1.0e9, 1.1e9])
    return toi.toi_plan_create(3, 2, 1, freq, N, cell_deg, input_location=toi.TOI_MEM_DEVICE)


def _tilt_V(tilt_deg, az_deg):
    """Inputs only: a rotation whose third row is tilted by tilt_deg (any proper rotation will do)."""
    t, z = math.radians(tilt_deg), math.radians(az_deg)
    a, b = math.sin(t) * math.cos(z), math.sin(t) * math.sin(z)
    c = math.sqrt(1.0 - a * a - b * b)
    return np.array([[1 - a * a / (1 + c), -a * b / (1 + c), -a],
                     [-a * b / (1 + c), 1 - b * b / (1 + c), -b],
                     [a, b, c]])


def _compare(img, V, cell_deg, mode, out_gpu):
    N = img.shape[0]
    mapper = {"exact": orp.map_exact, "paper": orp.map_paper}[mode]
    p1, p2, valid = mapper(V, N, cell_deg)
    ref = orp.bilinear_gather(img, p1, p2, valid)
    nan_o, nan_g = np.isnan(ref), np.isnan(out_gpu)
    mism = nan_o != nan_g
    if mism.any():
        edge = np.minimum.reduce([np.abs(p1 + 1e-6), np.abs(p1 - (N - 1 + 1e-6)),
                                  np.abs(p2 + 1e-6), np.abs(p2 - (N - 1 + 1e-6))])
        assert np.all(edge[mism] < 1e-9), "NaN masks differ away from the validity edge: %d px" % mism.sum()
    both = ~nan_o & ~nan_g
    peak = float(np.max(np.abs(img)))
    err = float(np.max(np.abs(out_gpu[both].astype(np.float64) - ref[both]))) if both.any() else 0.0
    assert err <= BAR * peak, "max abs %.3e > %.0e * peak %.3e" % (err, BAR, peak)
    return both.mean()


@pytest.mark.parametrize("mode", ["exact", "paper"])
@pytest.mark.parametrize("N,cell_deg,tilt,az", [
    (256, 10.0 / 3600, 0.7, 35.0),        # config-1 size, MeerKAT-like near-zenith tilt
    (1024, 1.5 / 3600, 0.3, -120.0),      # several tiles of 256 x 4 pixels
    (250, 0.02, 25.0, 80.0),              # N % 4 != 0 -> scalar path, ragged tail
    (512, 0.05, 62.0, -20.0),             # low elevation: large displacement, NaN border
    (64, 1.9, 10.0, 10.0),                # near all-sky: the SIN domain ends inside the image
])
def test_reproject_matches_oracle(N, cell_deg, tilt, az, mode):
    rng = np.random.default_rng(N + int(tilt * 10))
    img = rng.standard_normal((N, N)).astype(np.float32)
    jj, ii = np.mgrid[0:N, 0:N]
    img += (5.0 * np.exp(-((ii - 0.6 * N) ** 2 + (jj - 0.4 * N) ** 2) / (2 * 9.0))).astype(np.float32)
    V = _tilt_V(tilt, az)
    plan = _plan(N, cell_deg)
    try:
        d_img = torch.from_numpy(img).cuda()
        d_out = torch.full((N, N), -7.0, dtype=torch.float32, device="cuda")
        toi.toi_reproject(plan, d_img, d_out, V=V, mode=MODES[mode])
        toi.toi_plan_sync(plan)
        frac = _compare(img.astype(np.float64), V, cell_deg, mode, d_out.cpu().numpy())
        if tilt < 1.0:
            assert frac > 0.95
    finally:
        toi.toi_plan_destroy(plan)


def test_reproject_identity_transform_returns_the_image():
    N = 128
    rng = np.random.default_rng(1)
    img = rng.standard_normal((N, N)).astype(np.float32)
    plan = _plan(N, 0.01)
    try:
        d_out = torch.empty((N, N), dtype=torch.float32, device="cuda")
        toi.toi_reproject(plan, torch.from_numpy(img).cuda(), d_out, V=np.eye(3))
        toi.toi_plan_sync(plan)
        out = d_out.cpu().numpy()
        assert np.isfinite(out).all()                       # the last row/column too (G22's 1e-6 px)
        assert np.max(np.abs(out - img)) <= 1e-6 * np.max(np.abs(img))
    finally:
        toi.toi_plan_destroy(plan)


def test_reproject_unaligned_output_takes_the_scalar_path():
    N = 64
    rng = np.random.default_rng(2)
    img = rng.standard_normal((N, N)).astype(np.float32)
    V = _tilt_V(5.0, 0.0)
    plan = _plan(N, 0.02)
    try:
        buf = torch.zeros(N * N + 1, dtype=torch.float32, device="cuda")
        d_out = buf[1:]                                     # 4-byte aligned only
        toi.toi_reproject(plan, torch.from_numpy(img).cuda(), d_out, V=V)
        toi.toi_plan_sync(plan)
        _compare(img.astype(np.float64), V, 0.02, "exact", d_out.cpu().numpy().reshape(N, N))
    finally:
        toi.toi_plan_destroy(plan)


@pytest.mark.parametrize("mode", ["exact", "paper"])
def test_snapshot_then_reproject_with_the_plans_own_transform(mode):
    """The whole chain on a low-elevation snapshot: image (tilted plane) -> re-project with V = NULL
    (the V k_planefit left on the device) == oracle image -> oracle re-projection with the oracle's V."""
    wl = synth.reduced(synth.CONFIG5, n_ant=20, n_core=15, n_chan=64, image_size=256)
    snap = snapshot_np(wl)
    N, cell = wl.image_size, wl.cell_size_deg
    rc, img_o, info_o, _ = oracle.image_gridded(snap["uvw_m"], snap["vis"], snap["weights"], snap["flags"],
                                                snap["chan_freq_hz"], N, cell, pol_a=0, pol_b=3)
    assert rc == 0 and info_o["V"][2, 2] < 0.6
    ref = orp.reproject(img_o, info_o["V"], cell, mode)
    with GpuImager(snap, N, cell, "natural", pol_a=0, pol_b=3, apply_jacobian=0) as gi:
        ptr, _, _ = toi.toi_image_snapshot(gi.plan, gi.t["uvw_m"], gi.t["vis"], gi.t["weights"], gi.t["flags"])
        d_out = torch.empty((N, N), dtype=torch.float32, device="cuda")
        toi.toi_reproject(gi.plan, ptr, d_out, V=None, mode=MODES[mode])
        toi.toi_plan_sync(gi.plan)
        out = d_out.cpu().numpy()
    m = ~np.isnan(ref) & ~np.isnan(out)
    assert m.mean() > 0.2 and (np.isnan(ref) != np.isnan(out)).mean() < 1e-3
    peak = float(np.nanmax(np.abs(ref)))
    # imaging parity bar (1e-4 of peak) carries through the interpolation (a convex combination)
    assert float(np.max(np.abs(out[m] - ref[m]))) <= 1e-4 * peak
    assert float(np.linalg.norm(out[m] - ref[m]) / np.linalg.norm(ref[m])) <= 1e-5


def test_reproject_after_degenerate_snapshot_is_nan_and_bad_arguments_are_refused():
    wl = synth.reduced(synth.CONFIG1, n_ant=6, n_core=6, n_chan=4, image_size=32)
    snap = snapshot_np(wl)
    snap["uvw_m"] = np.outer(np.arange(1, snap["uvw_m"].shape[0] + 1), [1.0, 2.0, 0.5])   # collinear
    with GpuImager(snap, 32, wl.cell_size_deg, apply_jacobian=0) as gi:
        ptr, _, rc = toi.toi_image_snapshot(gi.plan, gi.t["uvw_m"], gi.t["vis"], gi.t["weights"], gi.t["flags"])
        d_out = torch.zeros((32, 32), dtype=torch.float32, device="cuda")
        toi.toi_reproject(gi.plan, ptr, d_out)
        toi.toi_plan_sync(gi.plan, allow=(toi.TOI_ERR_DEGENERATE_GEOMETRY,))
        assert torch.isnan(d_out).all()
        lib = toi.load()
        import ctypes as C
        assert lib.toi_reproject(gi.plan, C.c_void_p(ptr), None, 7, None, C.c_void_p(d_out.data_ptr())) == toi.TOI_ERR_INVALID_ARG
        assert lib.toi_reproject(gi.plan, C.c_void_p(ptr), None, 0, None, C.c_void_p(ptr)) == toi.TOI_ERR_INVALID_ARG
        bad = (C.c_double * 9)(1, 0, 0, 0, 1, 0, 0, 0, 0)
        assert lib.toi_reproject(gi.plan, C.c_void_p(ptr), bad, 0, None, C.c_void_p(d_out.data_ptr())) == toi.TOI_ERR_DEGENERATE_GEOMETRY
        assert lib.toi_difference(gi.plan, None, C.c_void_p(ptr), None, C.c_void_p(ptr)) == toi.TOI_ERR_INVALID_ARG


@pytest.mark.parametrize("N,offset", [(256, 0), (250, 0), (64, 1)])
def test_difference_is_bit_exact(N, offset):
    """a - b in fp32 is one correctly rounded operation: identical to numpy's float32 subtraction
    (and to the oracle's fp64 difference rounded to fp32)."""
    rng = np.random.default_rng(N)
    a = rng.standard_normal((N, N)).astype(np.float32)
    b = rng.standard_normal((N, N)).astype(np.float32)
    plan = _plan(N, 0.01)
    try:
        da = torch.zeros(N * N + offset, dtype=torch.float32, device="cuda")
        da[offset:] = torch.from_numpy(a).cuda().reshape(-1)
        db = torch.from_numpy(b).cuda()
        out = torch.empty(N * N, dtype=torch.float32, device="cuda")
        toi.toi_difference(plan, da[offset:], db, out)
        toi.toi_plan_sync(plan)
        got = out.cpu().numpy().reshape(N, N)
        ref = orp.difference(a, b).astype(np.float32)
        assert np.array_equal(got, ref)
    finally:
        toi.toi_plan_destroy(plan)


# ------------------------------------------------------------------------------------------------
# output side of the streamed run (interpolate + copy_cpu stages)
# ------------------------------------------------------------------------------------------------
def _stream_case(n=6, ring=3):
    import ctypes as C
    wl = synth.reduced(synth.CONFIG5, n_ant=12, n_core=9, n_chan=48, image_size=128, dt_s=120.0)
    snaps = [snapshot_np(wl, k) for k in range(n)]
    plan = toi.toi_plan_create(wl.n_baselines, wl.n_chan, wl.n_pol, snaps[0]["chan_freq_hz"], wl.image_size,
                               wl.cell_size_deg, pol_a=0, pol_b=3, input_location=toi.TOI_MEM_HOST,
                               image_ring_depth=ring)

    def fill(idx, slot):
        s = snaps[idx]
        for name, ptr in (("uvw_m", slot.uvw_m), ("vis", slot.vis), ("weights", slot.weights), ("flags", slot.flags)):
            a = np.ascontiguousarray(s[name])
            C.memmove(ptr, a.ctypes.data, a.nbytes)
        return 0

    refs = []
    for s in snaps:
        rc, img_o, info_o, _ = oracle.image_gridded(s["uvw_m"], s["vis"], s["weights"], s["flags"], s["chan_freq_hz"],
                                                    wl.image_size, wl.cell_size_deg, pol_a=0, pol_b=3)
        assert rc == 0
        refs.append((img_o, info_o["V"]))
    return wl, plan, fill, refs


def _close(got, ref, peak):
    m = ~np.isnan(ref) & ~np.isnan(got)
    assert (np.isnan(ref) != np.isnan(got)).mean() < 1e-3 and m.mean() > 0.2
    assert float(np.max(np.abs(got[m] - ref[m]))) <= 1e-4 * peak


@pytest.mark.parametrize("product,difference", [("tilted", False), ("exact", False), ("paper", True), ("tilted", True)])
def test_stream_output_ring_delivers_every_image_to_the_host_in_order(product, difference):
    n = 6
    wl, plan, fill, refs = _stream_case(n)
    N, cell = wl.image_size, wl.cell_size_deg
    code = {"tilted": toi.TOI_OUT_TILTED, "exact": toi.TOI_OUT_REPROJECT_EXACT, "paper": toi.TOI_OUT_REPROJECT_PAPER}[product]
    prods = [img if product == "tilted" else orp.reproject(img, V, cell, product) for img, V in refs]
    host, dev = {}, {}

    def host_sink(idx, image):
        assert idx not in host and (not host or idx == max(host) + 1)      # in order, once
        host[idx] = image.copy()

    def sink(idx, d_image, stream, info):
        dev[idx] = d_image

    try:
        toi.toi_stream_set_output(plan, product=code, difference=difference, host_sink=host_sink, image_size=N)
        stats = toi.toi_image_stream(plan, n, fill, sink)
        first = 1 if difference else 0
        assert sorted(host) == list(range(first, n)) and sorted(dev) == list(range(n))
        assert stats["d2h_bytes"] == (n - first) * N * N * 4 and stats["d2h_ms_sum"] > 0 and stats["gpu_ms"] > 0
        peak = max(float(np.nanmax(np.abs(p))) for p in prods)
        for k in range(first, n):
            ref = orp.difference(prods[k], prods[k - 1]) if difference else prods[k]
            _close(host[k].astype(np.float64), ref, peak)
        # the last delivered device image is still in its ring / ping-pong buffer
        last = toi.toi_copy_image_to_host(plan, dev[n - 1], N).numpy()
        assert np.array_equal(np.nan_to_num(last, nan=-1.0), np.nan_to_num(host[n - 1], nan=-1.0))
        # a second run on the same plan, default output restored: nothing reaches the host sink
        host.clear()
        toi.toi_stream_set_output(plan)
        stats = toi.toi_image_stream(plan, 2, fill, sink)
        assert not host and stats["d2h_bytes"] == 0
    finally:
        toi.toi_plan_destroy(plan)


def test_stream_output_refuses_bad_settings_and_propagates_host_sink_errors():
    wl, plan, fill, _ = _stream_case(3, ring=1)
    try:
        with pytest.raises(toi.ToiError) as ei:
            toi.toi_stream_set_output(plan, difference=True)
        assert ei.value.code == toi.TOI_ERR_INVALID_ARG          # ring depth 1
        with pytest.raises(toi.ToiError):
            toi.toi_stream_set_output(plan, product=9)
    finally:
        toi.toi_plan_destroy(plan)
    wl, plan, fill, _ = _stream_case(3, ring=2)
    try:
        with pytest.raises(toi.ToiError) as ei:      # the D2H ring needs an image ring of depth >= 3
            toi.toi_stream_set_output(plan, host_sink=lambda idx, image: 0, image_size=wl.image_size)
        assert ei.value.code == toi.TOI_ERR_INVALID_ARG
        toi.toi_stream_set_output(plan, difference=True)     # depth 2 is enough for the difference alone
    finally:
        toi.toi_plan_destroy(plan)
    wl, plan, fill, _ = _stream_case(4, ring=3)
    try:
        toi.toi_stream_set_output(plan, host_sink=lambda idx, image: -1, image_size=wl.image_size)
        with pytest.raises(toi.ToiError) as ei:
            toi.toi_image_stream(plan, 4, fill)
        assert ei.value.code == toi.TOI_ERR_CALLBACK
    finally:
        toi.toi_plan_destroy(plan)
