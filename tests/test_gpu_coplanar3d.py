"""-m gpu parity tests of the near-coplanar (3-D) mode, PAPER.md:202-269 (Eqs. 17-27):
libtoi's toi_image_snapshot_3d (Chebyshev-moment passes of the product gridder + cuFFT + the
combination kernels) against oracle/coplanar3d.py on the same inputs, element by element.

The oracle evaluates Eqs. 19-24 by direct Fourier sums (no gridding), with the SAME n_slab and K;
the GPU path differs from it by the gridding error of each moment only (P1's bound per moment,
added over the K orders with |c_k| <= 2 |J_k|) and fp32 accumulation.  Bars: rel-L2 <= 2e-5 and
max-abs <= 2e-5 * sum|z| / Wsum over the valid pixels; NaN masks identical.  Against Eq. 18 itself
(no expansion) the difference is bounded by the sampled expansion error, checked separately.
"""
from __future__ import annotations

import math

import numpy as np
import pytest

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")

import oracle  # noqa: E402
from oracle import coplanar3d as o3  # noqa: E402
from paper_2512_06254_b200 import binding as toi  # noqa: E402

C0 = 299792458.0


@pytest.fixture(scope="module", autouse=True)
def _need_gpu():
    assert torch.cuda.is_available(), "the -m gpu tests need a CUDA device"
    toi.load()


def make_snapshot(seed=1, n_b=40, n_c=8, tilt_deg=55.0, bump_m=2.0, flags=False):
    """Inputs only: a compact array (baselines <= 60 m) on a plane tilted by tilt_deg, with bump_m of
    out-of-plane scatter -- so r3 spans ~ +-10 wavelengths -- 2 pols, random visibilities."""
    rng = np.random.default_rng(seed)
    t = math.radians(tilt_deg)
    ex = np.array([1.0, 0.0, 0.0])
    ey = np.array([0.0, math.cos(t), math.sin(t)])
    nrm = np.cross(ex, ey)
    ab = rng.uniform(-60.0, 60.0, (n_b, 2))
    uvw = ab[:, :1] * ex + ab[:, 1:] * ey + rng.normal(0.0, bump_m, (n_b, 1)) * nrm
    freq = np.linspace(1.30e9, 1.40e9, n_c)
    vis = (rng.normal(size=(n_b, n_c, 2)) + 1j * rng.normal(size=(n_b, n_c, 2))).astype(np.complex64)
    weights = rng.uniform(0.5, 1.5, (n_b, n_c, 2)).astype(np.float32)
    fl = None
    if flags:
        fl = (rng.uniform(size=(n_b, n_c, 2)) < 0.1).astype(np.uint8)
    return {"uvw_m": uvw, "vis": vis, "weights": weights, "flags": fl, "chan_freq_hz": freq}


def oracle_inputs(snap, V):
    """Per-sample (r, z, w_I) for the direct sums: r = (V uvw_j) s_c, z = sum_p w_p Vis_p over unflagged hands."""
    s = snap["chan_freq_hz"] / C0
    rho = snap["uvw_m"] @ V.T                                   # [n_b, 3]
    r = rho[:, None, :] * s[None, :, None]                      # [n_b, n_c, 3]
    w = snap["weights"].astype(np.float64)
    if snap["flags"] is not None:
        w = np.where(snap["flags"] != 0, 0.0, w)
    z = np.sum(w * snap["vis"].astype(np.complex128), axis=2)
    wI = np.sum(w, axis=2)
    keep = wI > 0
    return r[keep], z[keep], wI[keep]


def run_gpu(snap, N, cell, n_slab, K, weighting=toi.TOI_WEIGHT_NATURAL):
    n_b, n_c, n_p = snap["vis"].shape
    plan = toi.toi_plan_create(n_b, n_c, n_p, snap["chan_freq_hz"], N, cell, weighting=weighting,
                               input_location=toi.TOI_MEM_DEVICE, enable_3d=True)
    try:
        t = {k: (None if snap[k] is None else torch.from_numpy(np.ascontiguousarray(snap[k])).cuda())
             for k in ("uvw_m", "vis", "weights", "flags")}
        ptr, i3, info = toi.toi_image_snapshot_3d(plan, t["uvw_m"], t["vis"], t["weights"], t["flags"], n_slab=n_slab, K=K)
        img3 = toi.toi_copy_image_to_host(plan, ptr, N).numpy().copy()
        ptr2, info2, _ = toi.toi_image_snapshot(plan, t["uvw_m"], t["vis"], t["weights"], t["flags"], want_info=True)
        img2 = toi.toi_copy_image_to_host(plan, ptr2, N).numpy().copy()
        return img3, i3, info.as_dict(), img2
    finally:
        toi.toi_plan_destroy(plan)


@pytest.mark.parametrize("n_slab,K,flags", [(1, 16, False), (3, 8, True), (2, 24, False)])
def test_3d_mode_matches_the_chebyshev_oracle(n_slab, K, flags):
    snap = make_snapshot(seed=10 + n_slab, flags=flags)
    N, cell = 64, 200.0 / 3600.0                                # 3.6 deg field: t3 reaches a few 1e-2
    rc, V, omega, _ = oracle.plane_fit(snap["uvw_m"], snap["chan_freq_hz"])
    assert rc == 0 and V[2, 2] < 0.7
    r, z, wI = oracle_inputs(snap, V)
    wsum = float(np.sum(wI))
    img3, i3, info, img2 = run_gpu(snap, N, cell, n_slab, K)
    assert info["n_off_grid"] == 0 and info["n_gridded"] == z.size        # every sample on the grid, counted once
    n_flagged = 0 if snap["flags"] is None else int(np.count_nonzero(np.all(snap["flags"] != 0, axis=2)))
    assert info["n_flagged"] == n_flagged                                   # ... also with several slabs
    assert not flags or n_flagged > 0
    assert abs(info["wsum"] - wsum) <= 2e-6 * wsum
    assert np.max(np.abs(np.array(info["V"]) - V)) < 1e-12
    assert i3["n_slab"] == n_slab and i3["K"] == K and i3["n_passes"] == n_slab * K
    assert abs(i3["r3_min"] - r[:, 2].min()) < 1e-9 and abs(i3["r3_max"] - r[:, 2].max()) < 1e-9
    phi_o, t3max_o = o3.phi_max_of(V, r[:, 2], N, cell)
    assert abs(i3["t3_max"] - t3max_o) < 1e-12 and abs(i3["phi_max"] - phi_o) < 1e-9 * max(1.0, phi_o)
    assert phi_o > 1.0                                                      # a real residual phase
    ref = o3.image_3d_chebyshev(r, z, V, omega, N, cell, n_slab, K, wsum=wsum)
    ok = ~np.isnan(ref.real)
    assert ok.mean() > 0.9 and np.array_equal(np.isnan(img3), ~ok)
    scale = float(np.sum(np.abs(z))) / wsum
    err = img3[ok].astype(np.float64) - ref.real[ok]
    assert np.max(np.abs(err)) <= 2e-5 * scale
    assert np.linalg.norm(err) / np.linalg.norm(ref.real[ok]) <= 2e-5
    # against Eq. 18 itself: within the sampled expansion error
    direct = o3.image_3d_direct(r, z, V, omega, N, cell, wsum=wsum)
    eps = o3.sampled_error(phi_o / n_slab, K)
    assert np.max(np.abs(img3[ok] - direct.real[ok])) <= 1.5 * eps * scale + 2e-5 * scale
    # and the r3 term matters: the 2-D image of the same snapshot is far from Eq. 18
    d2 = np.max(np.abs(img2[ok] - direct.real[ok]))
    assert d2 > 20 * np.max(np.abs(img3[ok] - direct.real[ok])) or K == 8


def test_3d_mode_chooses_the_papers_parameters_and_reduces_to_2d_for_planar_arrays():
    """Automatic n_slab / K follow Eqs. 25-27 (same rule as the oracle's select_parameters); an exactly
    planar array has r3 = 0 everywhere, so the 3-D image equals the 2-D image."""
    snap = make_snapshot(seed=5)
    N, cell = 64, 200.0 / 3600.0
    rc, V, omega, _ = oracle.plane_fit(snap["uvw_m"], snap["chan_freq_hz"])
    r, z, wI = oracle_inputs(snap, V)
    phi_o, _ = o3.phi_max_of(V, r[:, 2], N, cell)
    want = o3.select_parameters(phi_o)
    img3, i3, info, img2 = run_gpu(snap, N, cell, 0, 0)
    assert i3["n_slab"] == want["n_slab"] and i3["K"] == want["K"]
    assert abs(i3["alpha_slab"] - want["alpha_slab"]) < 1e-9 * max(1.0, want["alpha_slab"])
    assert abs(i3["expansion_error"] - want["error"]) <= 1e-6 + 1e-3 * want["error"] and i3["expansion_error"] < 1e-2
    planar = make_snapshot(seed=6, bump_m=0.0)
    img3, i3, info, img2 = run_gpu(planar, N, cell, 0, 0)
    assert i3["n_slab"] == 1 and i3["K"] == 8 and i3["phi_max"] < 1e-6
    ok = ~np.isnan(img3)
    assert ok.mean() > 0.9
    peak = float(np.max(np.abs(img2)))
    assert np.max(np.abs(img3[ok] - img2[ok])) <= 1e-5 * peak


def test_3d_mode_uniform_weighting_and_back_to_back_calls():
    """Uniform weighting reuses the density pass: on a planar array the 3-D image equals the 2-D
    uniform image; a second 3-D call and a 2-D call after it on the same plan still agree (the
    density / grid buffers are handed back in the state the 2-D path expects)."""
    planar = make_snapshot(seed=8, bump_m=0.0, flags=True)
    N, cell = 64, 200.0 / 3600.0
    n_b, n_c, n_p = planar["vis"].shape
    plan = toi.toi_plan_create(n_b, n_c, n_p, planar["chan_freq_hz"], N, cell, weighting=toi.TOI_WEIGHT_UNIFORM,
                               input_location=toi.TOI_MEM_DEVICE, enable_3d=True)
    try:
        t = {k: (None if planar[k] is None else torch.from_numpy(np.ascontiguousarray(planar[k])).cuda())
             for k in ("uvw_m", "vis", "weights", "flags")}
        imgs = []
        for kind in ("2d", "3d", "3d", "2d", "3d"):
            if kind == "2d":
                ptr, info, _ = toi.toi_image_snapshot(plan, t["uvw_m"], t["vis"], t["weights"], t["flags"], want_info=True)
            else:
                ptr, i3, info = toi.toi_image_snapshot_3d(plan, t["uvw_m"], t["vis"], t["weights"], t["flags"])
            imgs.append((kind, toi.toi_copy_image_to_host(plan, ptr, N).numpy().copy(), info.as_dict()))
        ref = imgs[0][1]
        peak = float(np.max(np.abs(ref)))
        assert peak > 0
        for kind, img, info in imgs[1:]:
            ok = ~np.isnan(img)
            assert ok.mean() > 0.9
            assert np.max(np.abs(img[ok] - ref[ok])) <= 1e-5 * peak, kind
            assert info["n_gridded"] == imgs[0][2]["n_gridded"] and info["n_flagged"] == imgs[0][2]["n_flagged"]
            assert abs(info["wsum"] - imgs[0][2]["wsum"]) <= 2e-6 * imgs[0][2]["wsum"]
    finally:
        toi.toi_plan_destroy(plan)


def test_3d_mode_with_host_inputs_equals_device_inputs_and_refuses_bad_arguments():
    import ctypes as C
    snap = make_snapshot(seed=9, flags=True)
    N, cell = 64, 200.0 / 3600.0
    img_dev, i3_dev, info_dev, _ = run_gpu(snap, N, cell, 2, 8)
    n_b, n_c, n_p = snap["vis"].shape
    plan = toi.toi_plan_create(n_b, n_c, n_p, snap["chan_freq_hz"], N, cell, input_location=toi.TOI_MEM_HOST,
                               enable_3d=True)
    try:
        t = {k: (None if snap[k] is None else torch.from_numpy(np.ascontiguousarray(snap[k])).pin_memory())
             for k in ("uvw_m", "vis", "weights", "flags")}
        ptr, i3, info = toi.toi_image_snapshot_3d(plan, t["uvw_m"], t["vis"], t["weights"], t["flags"], n_slab=2, K=8)
        img = toi.toi_copy_image_to_host(plan, ptr, N).numpy()
        assert np.array_equal(np.isnan(img), np.isnan(img_dev))
        ok = ~np.isnan(img)
        assert np.max(np.abs(img[ok] - img_dev[ok])) <= 1e-6 * float(np.max(np.abs(img_dev[ok])))
        assert info.n_gridded == info_dev["n_gridded"]
        lib = toi.load()
        out = C.c_void_p()
        args = (C.c_void_p(t["uvw_m"].data_ptr()), C.c_void_p(t["vis"].data_ptr()), None, None, None)
        assert lib.toi_image_snapshot_3d(plan, *args, 2000, 8, C.byref(out), None, None) == toi.TOI_ERR_INVALID_ARG
        assert lib.toi_image_snapshot_3d(plan, *args, 1, 65, C.byref(out), None, None) == toi.TOI_ERR_INVALID_ARG
        assert lib.toi_image_snapshot_3d(plan, None, args[1], None, None, None, 1, 8, C.byref(out), None, None) == toi.TOI_ERR_INVALID_ARG
    finally:
        toi.toi_plan_destroy(plan)


@pytest.mark.parametrize("weighting", [toi.TOI_WEIGHT_NATURAL, toi.TOI_WEIGHT_UNIFORM])
@pytest.mark.parametrize("order", [("2d", "3d", "2d"), ("3d", "2d", "2d"), ("2d", "3d", "3d", "3d", "2d", "3d")])
def test_2d_and_3d_calls_in_any_order_share_one_clean_grid(weighting, order):
    """2-D and 3-D calls alternate on one plan in every parity: the single gridding grid (and density
    map) must be zero again after each call, whichever mode ran last.  Planar array => both modes give
    the same image."""
    planar = make_snapshot(seed=21, bump_m=0.0, flags=True)
    N, cell = 64, 200.0 / 3600.0
    n_b, n_c, n_p = planar["vis"].shape
    plan = toi.toi_plan_create(n_b, n_c, n_p, planar["chan_freq_hz"], N, cell, weighting=weighting,
                               input_location=toi.TOI_MEM_DEVICE, enable_3d=True)
    try:
        t = {k: (None if planar[k] is None else torch.from_numpy(np.ascontiguousarray(planar[k])).cuda())
             for k in ("uvw_m", "vis", "weights", "flags")}
        ptr, info0, _ = toi.toi_image_snapshot(plan, t["uvw_m"], t["vis"], t["weights"], t["flags"], want_info=True)
        ref = toi.toi_copy_image_to_host(plan, ptr, N).numpy().copy()
        peak = float(np.max(np.abs(ref)))
        for kind in order:
            if kind == "2d":
                ptr, info, _ = toi.toi_image_snapshot(plan, t["uvw_m"], t["vis"], t["weights"], t["flags"], want_info=True)
            else:
                ptr, _, info = toi.toi_image_snapshot_3d(plan, t["uvw_m"], t["vis"], t["weights"], t["flags"])
            img = toi.toi_copy_image_to_host(plan, ptr, N).numpy()
            ok = ~np.isnan(img)
            assert ok.mean() > 0.9
            assert np.max(np.abs(img[ok] - ref[ok])) <= 1e-5 * peak, (kind, order)
            assert info.n_gridded == info0.n_gridded and info.n_flagged == info0.n_flagged
    finally:
        toi.toi_plan_destroy(plan)


def test_stream_after_one_3d_call():
    """toi_image_stream started after a single 3-D call (host-input plan): same images as before it."""
    import ctypes as C
    snap = make_snapshot(seed=23, bump_m=0.0)
    N, cell = 64, 200.0 / 3600.0
    n_b, n_c, n_p = snap["vis"].shape
    plan = toi.toi_plan_create(n_b, n_c, n_p, snap["chan_freq_hz"], N, cell, input_location=toi.TOI_MEM_HOST,
                               enable_3d=True, image_ring_depth=4)
    try:
        t = {k: (None if snap[k] is None else torch.from_numpy(np.ascontiguousarray(snap[k])).pin_memory())
             for k in ("uvw_m", "vis", "weights", "flags")}
        ptr, _, _ = toi.toi_image_snapshot(plan, t["uvw_m"], t["vis"], t["weights"], t["flags"], want_info=True)
        ref = toi.toi_copy_image_to_host(plan, ptr, N).numpy().copy()
        toi.toi_image_snapshot_3d(plan, t["uvw_m"], t["vis"], t["weights"], t["flags"])
        got = {}

        def fill(idx, slot):
            for name, dst in (("uvw_m", slot.uvw_m), ("vis", slot.vis), ("weights", slot.weights)):
                a = np.ascontiguousarray(snap[name])
                C.memmove(dst, a.ctypes.data, a.nbytes)
            slot.flags = None
            return 0

        def sink(idx, d_image, stream, info):
            got[idx] = d_image

        toi.toi_image_stream(plan, 3, fill, sink)
        for k in range(3):
            img = toi.toi_copy_image_to_host(plan, got[k], N).numpy()
            assert np.max(np.abs(img - ref)) <= 2e-6 * float(np.max(np.abs(ref)))
    finally:
        toi.toi_plan_destroy(plan)


@pytest.mark.slow
def test_3d_mode_at_config5_full_size_against_eq18():
    """BASELINE.json configs[4] at full size (2016 baselines x 1024 channels x 4 pols, N = 4096,
    G = 8192, low elevation): the instantiation bench.py times (4 pols, automatic N_slab and K) against
    Eq. 18 ITSELF at sampled pixels -- centre, brightest 2-D pixel, the four corners, seeded others.
    Bound: 1.5 x the sampled expansion error + 2e-5, times sum|z| / Wsum (the gridding + fp32 share)."""
    from paper_2512_06254_b200 import synth
    wl = synth.CONFIG5
    dev = synth.make_snapshot(wl, 0, device="cuda")
    snap = {k: (v.cpu().numpy() if v is not None else None) for k, v in dev.items()}
    N, cell = wl.image_size, wl.cell_size_deg
    plan = toi.toi_plan_create(wl.n_baselines, wl.n_chan, wl.n_pol, snap["chan_freq_hz"], N, cell, pol_a=0, pol_b=3,
                               input_location=toi.TOI_MEM_DEVICE, enable_3d=True)
    try:
        ptr, i3, info = toi.toi_image_snapshot_3d(plan, dev["uvw_m"], dev["vis"], dev["weights"], dev["flags"])
        img3 = toi.toi_copy_image_to_host(plan, ptr, N).numpy().copy()
        ptr2, _, _ = toi.toi_image_snapshot(plan, dev["uvw_m"], dev["vis"], dev["weights"], dev["flags"], want_info=True)
        img2 = toi.toi_copy_image_to_host(plan, ptr2, N).numpy().copy()
    finally:
        toi.toi_plan_destroy(plan)
    del dev
    torch.cuda.empty_cache()
    rc, V, omega, _ = oracle.plane_fit(snap["uvw_m"], snap["chan_freq_hz"])
    assert rc == 0 and np.max(np.abs(np.array(info.as_dict()["V"]) - V)) < 1e-12
    # the samples the gridder keeps: on the grid (G10) and not flagged; hands 0 and 3
    rho = oracle.rotate(snap["uvw_m"], V)
    _, _, on = oracle.cell_indices(rho, snap["chan_freq_hz"], 2 * N, cell)
    s = snap["chan_freq_hz"] / C0
    w = snap["weights"][:, :, [0, 3]].astype(np.float64)
    w = np.where(snap["flags"][:, :, [0, 3]] != 0, 0.0, w)
    z = np.sum(w * snap["vis"][:, :, [0, 3]].astype(np.complex128), axis=2)
    wI = np.sum(w, axis=2)
    keep = (wI > 0) & on
    r = (rho[:, None, :] * s[None, :, None])[keep]
    z, wI = z[keep], wI[keep]
    wsum = float(np.sum(wI))
    assert info.n_gridded == z.size and abs(info.wsum - wsum) <= 2e-6 * wsum
    phi_o, _ = o3.phi_max_of(V, r[:, 2], N, cell)
    want = o3.select_parameters(phi_o)
    assert i3["n_slab"] == want["n_slab"] and i3["K"] == want["K"] and i3["n_passes"] == want["n_slab"] * want["K"]
    rng = np.random.default_rng(55)
    jj, ii = np.unravel_index(np.nanargmax(img2), img2.shape)
    pi = np.concatenate([[N // 2, ii, 0, N - 1, 0, N - 1], rng.integers(0, N, 6)])
    pj = np.concatenate([[N // 2, jj, 0, 0, N - 1, N - 1], rng.integers(0, N, 6)])
    direct = o3.image_3d_direct_pixels(r, z, V, omega, N, cell, pi, pj, wsum=wsum)
    got = img3[pj, pi]
    assert np.array_equal(np.isnan(got), np.isnan(direct.real))
    ok = ~np.isnan(got)
    assert ok.sum() >= 8
    scale = float(np.sum(np.abs(z))) / wsum
    eps = o3.sampled_error(phi_o / i3["n_slab"], i3["K"])
    err = float(np.max(np.abs(got[ok] - direct.real[ok])))
    err2d = float(np.max(np.abs(img2[pj, pi][ok] - direct.real[ok])))
    print("3-D mode, config 5 full size: n_slab %d K %d phi_max %.2f; max |err| vs Eq. 18 = %.3e = %.3e x scale "
          "(sampled expansion error %.3e); the 2-D image is off by %.3e" %
          (i3["n_slab"], i3["K"], phi_o, err, err / scale, eps, err2d))
    assert err <= (1.5 * eps + 2e-5) * scale


def test_3d_mode_on_the_hand_written_transform():
    """N = 512 (G = 1024): the Chebyshev moments go through k_fft_rows / k_fft_cols (complex output in
    place) instead of cuFFT, which the N = 64 cases above use.  Sampled pixels against Eq. 18 itself, and
    the whole image against the cuFFT-sized case's property that a planar array gives the 2-D image."""
    snap = make_snapshot(seed=31, flags=True)
    N, cell = 512, 25.0 / 3600.0                                 # same 3.6 deg field as the N = 64 cases
    rc, V, omega, _ = oracle.plane_fit(snap["uvw_m"], snap["chan_freq_hz"])
    assert rc == 0
    r, z, wI = oracle_inputs(snap, V)
    wsum = float(np.sum(wI))
    img3, i3, info, img2 = run_gpu(snap, N, cell, 2, 16)
    assert info["n_off_grid"] == 0 and info["n_gridded"] == z.size and abs(info["wsum"] - wsum) <= 2e-6 * wsum
    rng = np.random.default_rng(77)
    pi = np.concatenate([[N // 2, 0, N - 1, 0, N - 1], rng.integers(0, N, 60)])
    pj = np.concatenate([[N // 2, 0, 0, N - 1, N - 1], rng.integers(0, N, 60)])
    direct = o3.image_3d_direct_pixels(r, z, V, omega, N, cell, pi, pj, wsum=wsum)
    got = img3[pj, pi]
    assert np.array_equal(np.isnan(got), np.isnan(direct.real))
    ok = ~np.isnan(got)
    assert ok.sum() > 50
    phi_o, _ = o3.phi_max_of(V, r[:, 2], N, cell)
    eps = o3.sampled_error(phi_o / 2, 16)
    scale = float(np.sum(np.abs(z))) / wsum
    assert np.max(np.abs(got[ok] - direct.real[ok])) <= (1.5 * eps + 2e-5) * scale
    planar = make_snapshot(seed=32, bump_m=0.0)
    img3, i3, info, img2 = run_gpu(planar, N, cell, 0, 0)
    ok = ~np.isnan(img3)
    assert ok.mean() > 0.9
    assert np.max(np.abs(img3[ok] - img2[ok])) <= 1e-5 * float(np.max(np.abs(img2)))
