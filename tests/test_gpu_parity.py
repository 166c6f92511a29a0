"""-m gpu parity tests: libtoi (CUDA, through the C ABI via the ctypes binding) against the
fp64 CPU oracle, element by element on the same seeded inputs.

Bars (BASELINE.json north_star): image relative L2 error <= 1e-5 and max abs error <= 1e-4 of the
image peak (fp32 accumulation against fp64); grid-cell indices bit-exact (fp64 on both sides,
protocol G5 of DESIGN.md section 3); counts exact; V within 1e-12.
"""
from __future__ import annotations

import numpy as np
import pytest

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")

import oracle  # noqa: E402
from paper_2512_06254_b200 import binding as toi  # noqa: E402
from paper_2512_06254_b200 import synth  # noqa: E402

from gpu_helpers import GpuImager  # noqa: E402
from helpers import rel_l2, snapshot_np  # noqa: E402

REL_L2_BAR = 1e-5
MAX_ABS_BAR = 1e-4      # of the image peak


@pytest.fixture(scope="module", autouse=True)
def _need_gpu():
    # no skip-on-missing-GPU here: -m gpu is only run on a GPU box, and a silent skip would hide
    # a broken CUDA path.  The library itself fails loudly without a device.
    assert torch.cuda.is_available(), "the -m gpu tests need a CUDA device"
    toi.load()


def _oracle(snap, N, cell, weighting="natural", **kw):
    wt = oracle.UNIFORM if weighting == "uniform" else oracle.NATURAL
    rc, img, info, ex = oracle.image_gridded(snap["uvw_m"], snap["vis"], snap["weights"], snap["flags"],
                                             snap["chan_freq_hz"], N, cell, weighting=wt, **kw)
    return rc, img, info, ex


def _assert_image(img_gpu, img_orc, what=""):
    peak = float(np.max(np.abs(img_orc)))
    err_l2 = rel_l2(img_gpu, img_orc)
    err_max = float(np.max(np.abs(img_gpu.astype(np.float64) - img_orc)))
    assert err_l2 <= REL_L2_BAR, "%s rel-L2 %.3e > %.0e" % (what, err_l2, REL_L2_BAR)
    assert err_max <= MAX_ABS_BAR * peak, "%s max-abs %.3e > %.0e * peak %.3e" % (what, err_max, MAX_ABS_BAR, peak)
    return err_l2, (err_max / peak if peak > 0.0 else 0.0)


def _check_all(snap, wl_N, cell, weighting, gridder, pol_a=None, pol_b=None, location=toi.TOI_MEM_DEVICE,
               check_grid=True):
    """Full protocol for one case: V, indices (injected V), counts, wsum, grid, density, image."""
    rc, img_o, info_o, ex = _oracle(snap, wl_N, cell, weighting, pol_a=pol_a, pol_b=pol_b, want_grid=check_grid,
                                    want_density=(weighting == "uniform"), want_indices=True)
    assert rc == 0
    with GpuImager(snap, wl_N, cell, weighting, gridder, location, pol_a, pol_b,
                   keep_grid=check_grid or weighting == "uniform") as gi:
        # (i) own fit: V within 1e-12 of the oracle's explicit-B fit
        img_g, info_g, _ = gi.image()
        V_g = np.array(info_g["V"])
        assert np.max(np.abs(V_g - info_o["V"])) <= 1e-12
        assert abs(info_g["omega"] - info_o["omega"]) <= 1e-12
        np.testing.assert_allclose(info_g["sing"], info_o["sing"], rtol=1e-9)
        # (iii) indices with each side's own V: report, expect (almost always) zero differences
        iu_g, iv_g = gi.indices()
        n_diff_own = int(np.count_nonzero((iu_g != ex["iu"]) | (iv_g != ex["iv"])))
        assert n_diff_own <= max(2, iu_g.size // 100000), "own-V index mismatches: %d" % n_diff_own
        # (ii) oracle V injected: bit-exact indices for ALL samples, exact counts
        toi.toi_debug_set_transform(gi.plan, info_o["V"])
        img_g, info_g, _ = gi.image()
        iu_g, iv_g = gi.indices()
        assert np.array_equal(iu_g, ex["iu"]) and np.array_equal(iv_g, ex["iv"])
        for k in ("n_gridded", "n_off_grid", "n_flagged"):
            assert info_g[k] == info_o[k], k
        assert abs(info_g["wsum"] - info_o["wsum"]) <= 2e-6 * abs(info_o["wsum"])
        if weighting == "uniform":
            d_g = gi.density_centred()
            np.testing.assert_allclose(d_g, ex["density"], rtol=2e-6, atol=0)
        if check_grid:
            g_g = gi.grid_centred()
            assert rel_l2(g_g.view(np.float32).ravel(), ex["grid"].view(np.float64).ravel()) <= 3e-6
        e_inj = _assert_image(img_g, img_o, "injected-V image")
        # and with its own V again (the product path)
        toi.toi_debug_set_transform(gi.plan, None)
        img_g2, _, _ = gi.image()
        e_own = _assert_image(img_g2, img_o, "own-V image")
    return e_inj, e_own


# ------------------------------------------------------------------------------------------------
# config 1 (BASELINE.json configs[0]): the tiny snapshot, natural weighting, both gridders
# ------------------------------------------------------------------------------------------------
ALL_GRIDDERS = [toi.TOI_GRIDDER_SLIDING, toi.TOI_GRIDDER_ATOMIC]


@pytest.mark.parametrize("gridder", ALL_GRIDDERS)
def test_config1_natural(gridder):
    wl = synth.CONFIG1
    snap = snapshot_np(wl)
    _check_all(snap, wl.image_size, wl.cell_size_deg, "natural", gridder)


def test_config1_point_source_is_1jy():
    """Unit point source at the phase centre, natural weighting: 1 Jy at pixel (N/2, N/2) (P2)."""
    wl = synth.CONFIG1
    snap = snapshot_np(wl)
    snap["vis"] = np.ones_like(snap["vis"])
    with GpuImager(snap, wl.image_size, wl.cell_size_deg) as gi:
        img, info, _ = gi.image()
    c = wl.image_size // 2
    assert abs(img[c, c] * info["omega"] - 1.0) <= 2e-6
    assert np.unravel_index(np.argmax(img), img.shape) == (c, c)


def test_config1_uniform():
    wl = synth.CONFIG1
    snap = snapshot_np(wl)
    _check_all(snap, wl.image_size, wl.cell_size_deg, "uniform", toi.TOI_GRIDDER_SLIDING)


# ------------------------------------------------------------------------------------------------
# reduced config 2: MeerKAT-shaped layout (core + outliers, curved array => tilted plane),
# 4 pols, weights, channel-block flags, wide band; several tiles / strips and ragged tails
# ------------------------------------------------------------------------------------------------
def _reduced2(n_ant=24, n_chan=777, image_size=512, **kw):
    # 777 channels: not a multiple of the 8-sample batch, the 32-lane warp or the 4-strip task
    return synth.reduced(synth.CONFIG2, n_ant=n_ant, n_core=int(0.75 * n_ant), n_chan=n_chan,
                         image_size=image_size, n_src=20, **kw)


@pytest.mark.parametrize("weighting", ["natural", "uniform"])
@pytest.mark.parametrize("gridder", ALL_GRIDDERS)
def test_reduced_config2(weighting, gridder):
    wl = _reduced2()
    snap = snapshot_np(wl)
    assert snap["weights"] is not None and snap["flags"] is not None
    _check_all(snap, wl.image_size, wl.cell_size_deg, weighting, gridder, pol_a=0, pol_b=3)


def test_reduced_config2_long_rows():
    """More channels than one task covers (8 strips x 128): several tasks per baseline row."""
    wl = _reduced2(n_ant=12, n_chan=2500, image_size=1024)
    snap = snapshot_np(wl)
    _check_all(snap, wl.image_size, wl.cell_size_deg, "natural", toi.TOI_GRIDDER_SLIDING, pol_a=0, pol_b=3,
               check_grid=False)


@pytest.mark.parametrize("gridder", ALL_GRIDDERS)
@pytest.mark.parametrize("weighting", ["natural", "uniform"])
def test_coarse_channels_make_the_window_jump(gridder, weighting):
    """16 channels across the whole band: consecutive samples of a long baseline are tens of cells
    apart, so nearly every record takes the "far move" path (flush everything, reopen) instead of
    sliding by one cell; short baselines still slide.  Also mixes diagonal moves."""
    wl = _reduced2(n_ant=14, n_chan=16, image_size=1024)
    snap = snapshot_np(wl)
    _check_all(snap, wl.image_size, wl.cell_size_deg, weighting, gridder, pol_a=0, pol_b=3)


def test_low_elevation_config5_shape():
    """Config 5's geometry (hour angle -83 deg, elevation ~20 deg): the plane is tilted by ~70 deg,
    omega ~ 0.34 -- the SVD transform's stress case."""
    wl = synth.reduced(synth.CONFIG5, n_ant=20, n_core=15, n_chan=256, image_size=512)
    snap = snapshot_np(wl)
    rc, _, info_o, _ = _oracle(snap, wl.image_size, wl.cell_size_deg, pol_a=0, pol_b=3)
    assert rc == 0 and info_o["omega"] < 0.6
    _check_all(snap, wl.image_size, wl.cell_size_deg, "natural", toi.TOI_GRIDDER_SLIDING, pol_a=0, pol_b=3)


# ------------------------------------------------------------------------------------------------
# edge cases of the method
# ------------------------------------------------------------------------------------------------
def _edge_snapshot(seed=7):
    wl = synth.reduced(synth.CONFIG1, n_ant=10, n_core=10, n_chan=37, image_size=128, cell_arcsec=20.0, n_pol=2)
    snap = snapshot_np(wl)
    rng = np.random.default_rng(seed)
    shape = snap["vis"].shape
    snap["weights"] = rng.uniform(0.2, 2.0, shape).astype(np.float32)
    snap["flags"] = np.zeros(shape, np.uint8)
    return wl, snap, rng


def test_edge_single_pol_flags_nan_and_bad_weights():
    """G12: per-pol flags; NaN/Inf data under flags must not leak; weight <= 0 / NaN / Inf = flagged."""
    wl, snap, rng = _edge_snapshot()
    f = snap["flags"]
    f[rng.uniform(size=f.shape) < 0.3] = 1
    f[3, 5, :] = 1                                 # both hands flagged
    snap["vis"][f != 0] = np.nan + 1j * np.inf     # garbage under every flag
    w = snap["weights"]
    w[1, 2, 0] = 0.0
    w[1, 3, 1] = -1.0
    w[2, 4, 0] = np.nan
    w[2, 5, 1] = np.inf
    for gridder in ALL_GRIDDERS:
        e, _ = _check_all(snap, wl.image_size, wl.cell_size_deg, "natural", gridder)
    _check_all(snap, wl.image_size, wl.cell_size_deg, "uniform", toi.TOI_GRIDDER_SLIDING)


def test_edge_off_grid_samples_dropped():
    """G10: a sample whose 7x7 footprint leaves the grid is dropped and counted, never wrapped."""
    wl, snap, _ = _edge_snapshot()
    cell = 3.0 * wl.cell_size_deg                  # grid half-extent shrinks 3x: long baselines fall off
    rc, _, info_o, _ = _oracle(snap, wl.image_size, cell)
    assert rc == 0 and info_o["n_off_grid"] > 0 and info_o["n_gridded"] > 0
    for gridder in ALL_GRIDDERS:
        _check_all(snap, wl.image_size, cell, "natural", gridder)
    _check_all(snap, wl.image_size, cell, "uniform", toi.TOI_GRIDDER_SLIDING)


def test_edge_all_flagged_gives_zero_image():
    wl, snap, _ = _edge_snapshot()
    snap["flags"][:] = 1
    with GpuImager(snap, wl.image_size, wl.cell_size_deg) as gi:
        img, info, rc = gi.image()
    assert rc == toi.TOI_OK and info["wsum"] == 0.0 and info["n_gridded"] == 0
    assert np.all(img == 0.0)


def test_edge_degenerate_geometry():
    """G4: collinear baselines span no plane -> TOI_ERR_DEGENERATE_GEOMETRY and a zero image."""
    wl, snap, _ = _edge_snapshot()
    t = np.linspace(-1.0, 1.0, snap["uvw_m"].shape[0])
    snap["uvw_m"] = np.stack([300.0 * t, 200.0 * t, 10.0 * t], axis=1)
    rc_o = oracle.plane_fit(snap["uvw_m"], snap["chan_freq_hz"])[0]
    assert rc_o == oracle.ERR_DEGENERATE
    with GpuImager(snap, wl.image_size, wl.cell_size_deg) as gi:
        img, _, rc = gi.image(allow_degenerate=True)
        assert rc == toi.TOI_ERR_DEGENERATE_GEOMETRY
        assert np.all(img == 0.0)


@pytest.mark.parametrize("n_pol,pols", [(1, (0, 0)), (4, (0, 3)), (4, (1, 2)), (2, (1, 1))])
def test_edge_polarisation_layouts(n_pol, pols):
    wl = synth.reduced(synth.CONFIG1, n_ant=9, n_core=9, n_chan=19, image_size=64, cell_arcsec=30.0, n_pol=n_pol)
    snap = snapshot_np(wl)
    rng = np.random.default_rng(3)
    snap["vis"] = (rng.normal(size=snap["vis"].shape) + 1j * rng.normal(size=snap["vis"].shape)).astype(np.complex64)
    snap["weights"] = rng.uniform(0.5, 1.5, snap["vis"].shape).astype(np.float32)
    _check_all(snap, wl.image_size, wl.cell_size_deg, "natural", toi.TOI_GRIDDER_SLIDING, pol_a=pols[0], pol_b=pols[1])


@pytest.mark.parametrize("n_chan", [1, 3, 8, 33])
def test_edge_few_channels(n_chan):
    wl = synth.reduced(synth.CONFIG1, n_ant=8, n_core=8, n_chan=n_chan, image_size=64, cell_arcsec=30.0)
    snap = snapshot_np(wl)
    _check_all(snap, wl.image_size, wl.cell_size_deg, "natural", toi.TOI_GRIDDER_SLIDING)


@pytest.mark.parametrize("image_size", [100, 36])
def test_edge_image_size_not_a_multiple_of_8(image_size):
    """Even N that is not a multiple of 8: the scalar correction/crop kernel, a non power-of-two FFT."""
    wl = synth.reduced(synth.CONFIG1, n_ant=8, n_core=8, n_chan=24, image_size=image_size, cell_arcsec=40.0)
    snap = snapshot_np(wl)
    _check_all(snap, wl.image_size, wl.cell_size_deg, "natural", toi.TOI_GRIDDER_SLIDING)


def test_back_to_back_snapshots_find_a_zero_grid():
    """The grid / density map are cleared sparsely (only the tiles the snapshot touched) after the
    first FFT pass: five snapshots in a row (uniform weighting) must all equal the first."""
    wl = _reduced2(n_ant=12, n_chan=130, image_size=256)
    snap = snapshot_np(wl)
    rc, img_o, _, _ = _oracle(snap, wl.image_size, wl.cell_size_deg, "uniform", pol_a=0, pol_b=3)
    assert rc == 0
    with GpuImager(snap, wl.image_size, wl.cell_size_deg, "uniform", pol_a=0, pol_b=3) as gi:
        for _ in range(5):
            img, _, _ = gi.image()
            _assert_image(img, img_o, "repeat")


@pytest.mark.parametrize("weighting", ["natural", "uniform"])
def test_calls_without_info_give_the_same_image(weighting):
    """A call without `info` records no per-stage events and does not synchronise; several of them back to
    back, then a timed one, all against the oracle's image."""
    wl = _reduced2(n_ant=12, n_chan=130, image_size=256)
    snap = snapshot_np(wl)
    rc, img_o, _, _ = _oracle(snap, wl.image_size, wl.cell_size_deg, weighting, pol_a=0, pol_b=3)
    assert rc == 0
    with GpuImager(snap, wl.image_size, wl.cell_size_deg, weighting, pol_a=0, pol_b=3) as gi:
        for k in range(3):
            img, rc_g = gi.image_untimed()
            assert rc_g == 0
            _assert_image(img, img_o, f"untimed call {k}")
        img, info, _ = gi.image()
        _assert_image(img, img_o, "timed call after untimed ones")
        assert info["ms_grid"] > 0.0 and info["ms_fft"] > 0.0
        # a timed call clears the grid and the density map with two launches, each between its own events
        assert info["ms_clear"] > 0.0
        assert (info["ms_clear_density"] > 0.0) == (weighting == "uniform")
        img, rc_g = gi.image_untimed()
        assert rc_g == 0
        _assert_image(img, img_o, "untimed call after a timed one")


def test_edge_non_default_grid_size():
    wl = synth.CONFIG1
    snap = snapshot_np(wl)
    G = 384                                       # 1.5 N, not a power of two
    rc, img_o, info_o, _ = _oracle(snap, wl.image_size, wl.cell_size_deg, G=G)
    assert rc == 0
    with GpuImager(snap, wl.image_size, wl.cell_size_deg, grid_size=G) as gi:
        img, info, _ = gi.image()
    assert info["n_gridded"] == info_o["n_gridded"]
    _assert_image(img, img_o, "G=384")


@pytest.mark.parametrize("N,G", [(528, 1024), (1536, 2048), (752, 2048), (1040, 4096)])
def test_hand_written_transform_with_other_crops(N, G):
    """k_fft_rows / k_fft_cols take G = 2^10 .. 2^14 with G >= 4N/3 and N a multiple of 16; every other
    test runs them at G = 2N.  Here the crop keeps a non-power-of-two N (the two bands of needed columns
    [0, N/2) and [G - N/2, G) and the blocks of the workspace between the passes end on odd multiples
    of the block width), up to the limit N = 3G/4.  Image against the oracle's, natural and uniform."""
    wl = _reduced2(n_ant=12, n_chan=96, image_size=N)
    snap = snapshot_np(wl)
    for weighting in ("natural", "uniform"):
        rc, img_o, info_o, _ = _oracle(snap, N, wl.cell_size_deg, weighting, G=G, pol_a=0, pol_b=3)
        assert rc == 0 and info_o["n_gridded"] > 0
        with GpuImager(snap, N, wl.cell_size_deg, weighting, grid_size=G, pol_a=0, pol_b=3) as gi:
            img, info, _ = gi.image()
            img2, _, _ = gi.image()                  # the workspace and the tile map are reused
        assert info["n_gridded"] == info_o["n_gridded"]
        _assert_image(img, img_o, f"N={N} G={G} {weighting}")
        _assert_image(img2, img_o, f"N={N} G={G} {weighting} (second call)")


@pytest.mark.parametrize("gridder", ALL_GRIDDERS)
@pytest.mark.parametrize("G", [198, 202, 136])
def test_edge_grid_half_size_odd_or_tight(G, gridder):
    """G/2 odd (198, 202): the even-aligned 8x8 register window of the product gridder then starts
    one column/row OUTSIDE the grid for samples on the lowest on-grid cells and overhangs into the
    plan's guard band; G = 136 barely holds the image (G >= N) so many samples sit on the edge
    cells or fall off.  Full protocol (indices, counts, pre-FFT grid, image) for every gridder."""
    wl = synth.reduced(synth.CONFIG1, n_ant=12, n_core=12, n_chan=48, image_size=128, cell_arcsec=25.0)
    snap = snapshot_np(wl)
    rc, img_o, info_o, ex = _oracle(snap, wl.image_size, wl.cell_size_deg, G=G, want_grid=True)
    assert rc == 0 and info_o["n_gridded"] > 0
    if G == 136:
        assert info_o["n_off_grid"] > 0
    with GpuImager(snap, wl.image_size, wl.cell_size_deg, "natural", gridder, grid_size=G, keep_grid=True) as gi:
        img, info, _ = gi.image()
        grid = gi.grid_centred()
    assert info["n_gridded"] == info_o["n_gridded"] and info["n_off_grid"] == info_o["n_off_grid"]
    assert rel_l2(grid.view(np.float32).ravel(), ex["grid"].view(np.float64).ravel()) <= 3e-6
    _assert_image(img, img_o, "G=%d" % G)


def test_no_jacobian_option():
    wl = synth.reduced(synth.CONFIG5, n_ant=12, n_core=9, n_chan=64, image_size=128)
    snap = snapshot_np(wl)
    rc, img_o, info_o, _ = _oracle(snap, wl.image_size, wl.cell_size_deg, pol_a=0, pol_b=3, apply_jacobian=0)
    assert rc == 0
    with GpuImager(snap, wl.image_size, wl.cell_size_deg, pol_a=0, pol_b=3, apply_jacobian=2) as gi:
        img, _, _ = gi.image()
    _assert_image(img, img_o, "no jacobian")


# ------------------------------------------------------------------------------------------------
# boundary behaviour on the device: host inputs (H2D inside the call), image ring, streamed run
# ------------------------------------------------------------------------------------------------
def test_host_inputs_match_device_inputs():
    wl = _reduced2(n_ant=12, n_chan=130, image_size=256)
    snap = snapshot_np(wl)
    with GpuImager(snap, wl.image_size, wl.cell_size_deg, "uniform", pol_a=0, pol_b=3) as a:
        img_d, _, _ = a.image()
    with GpuImager(snap, wl.image_size, wl.cell_size_deg, "uniform", pol_a=0, pol_b=3,
                   location=toi.TOI_MEM_HOST) as b:
        img_h, info, _ = b.image()
        assert info["ms_h2d"] > 0.0
    rc, img_o, _, _ = _oracle(snap, wl.image_size, wl.cell_size_deg, "uniform", pol_a=0, pol_b=3)
    _assert_image(img_h, img_o, "host inputs")
    assert rel_l2(img_h, img_d) <= 2e-6            # fp32 reductions are order-dependent, not bit-equal


def test_image_ring_keeps_previous_images():
    wl = synth.reduced(synth.CONFIG1, n_ant=8, n_core=8, n_chan=16, image_size=64, cell_arcsec=30.0)
    snaps = [snapshot_np(wl, k) for k in range(3)]
    with GpuImager(snaps[0], wl.image_size, wl.cell_size_deg, ring_depth=3) as gi:
        ptrs, imgs = [], []
        for s in snaps:
            gi.set_inputs(s)
            ptr, _, _ = toi.toi_image_snapshot(gi.plan, gi.t["uvw_m"], gi.t["vis"], None, None, want_info=True)
            ptrs.append(ptr)
            imgs.append(toi.toi_copy_image_to_host(gi.plan, ptr, wl.image_size).numpy().copy())
        assert len(set(ptrs)) == 3
        for ptr, img in zip(ptrs, imgs):          # all three still intact after the third call
            again = toi.toi_copy_image_to_host(gi.plan, ptr, wl.image_size).numpy()
            assert np.array_equal(again, img)


def test_stream_matches_single_snapshots():
    """toi_image_stream (pinned ring, copy/compute streams, events) == per-snapshot oracle images."""
    import ctypes as C
    wl = _reduced2(n_ant=10, n_chan=96, image_size=128)
    wl = synth.reduced(wl, pulsar_mjy=50.0)
    n = 5
    snaps = [snapshot_np(wl, k) for k in range(n)]
    plan = toi.toi_plan_create(wl.n_baselines, wl.n_chan, wl.n_pol, snaps[0]["chan_freq_hz"], wl.image_size,
                               wl.cell_size_deg, pol_a=0, pol_b=3, input_location=toi.TOI_MEM_HOST,
                               image_ring_depth=n)
    got = {}

    def fill(idx, slot):
        s = snaps[idx]
        for name, ptr in (("uvw_m", slot.uvw_m), ("vis", slot.vis), ("weights", slot.weights), ("flags", slot.flags)):
            a = np.ascontiguousarray(s[name])
            C.memmove(ptr, a.ctypes.data, a.nbytes)
        return 0

    def sink(idx, d_image, stream, info):
        got[idx] = d_image
        return 0

    try:
        stats = toi.toi_image_stream(plan, n, fill, sink)
        assert stats["n_done"] == n and stats["h2d_bytes"] > 0 and stats["gpu_ms"] > 0
        for k in range(n):
            img = toi.toi_copy_image_to_host(plan, got[k], wl.image_size).numpy()
            rc, img_o, _, _ = _oracle(snaps[k], wl.image_size, wl.cell_size_deg, pol_a=0, pol_b=3)
            assert rc == 0
            _assert_image(img, img_o, "stream snapshot %d" % k)
    finally:
        toi.toi_plan_destroy(plan)


def test_stream_end_of_data_and_callback_error():
    wl = synth.reduced(synth.CONFIG1, n_ant=6, n_core=6, n_chan=8, image_size=32, cell_arcsec=60.0)
    snap = snapshot_np(wl)
    import ctypes as C
    plan = toi.toi_plan_create(wl.n_baselines, wl.n_chan, wl.n_pol, snap["chan_freq_hz"], wl.image_size,
                               wl.cell_size_deg, input_location=toi.TOI_MEM_HOST)

    def fill(idx, slot):
        if idx == 3:
            return 1
        C.memmove(slot.uvw_m, snap["uvw_m"].ctypes.data, snap["uvw_m"].nbytes)
        C.memmove(slot.vis, snap["vis"].ctypes.data, snap["vis"].nbytes)
        slot.weights = None
        slot.flags = None
        return 0

    try:
        stats = toi.toi_image_stream(plan, 10, fill)
        assert stats["n_done"] == 3
        with pytest.raises(toi.ToiError) as ei:
            toi.toi_image_stream(plan, 10, lambda idx, slot: -1)
        assert ei.value.code == toi.TOI_ERR_CALLBACK
    finally:
        toi.toi_plan_destroy(plan)


def test_invalid_arguments_are_refused():
    f = [1.0e9, 1.1e9]
    for kw in (dict(image_size=17), dict(n_pols=3), dict(grid_size=10), dict(cell_size_deg=0.0),
               dict(kernel_support=5), dict(weighting=9), dict(device=99)):
        args = dict(n_baselines=3, n_channels=2, n_pols=2, chan_freq_hz=f, image_size=32, cell_size_deg=0.01)
        args.update(kw)
        with pytest.raises(toi.ToiError):
            toi.toi_plan_create(**args)


# ------------------------------------------------------------------------------------------------
# full size (BASELINE.json configs[1]) in the launch configuration bench.py times
# ------------------------------------------------------------------------------------------------
@pytest.mark.slow
@pytest.mark.parametrize("weighting", ["uniform", "natural"])
def test_config2_full_size(weighting):
    """2016 baselines x 4096 channels x 4 pols, 2048^2 image, G = 4096.  Inputs are generated on the
    GPU by the seeded generator, copied to the host for the oracle; the whole image is compared with
    Tier G, and 12 sampled pixels with the direct DFT of Eq. 7 (Tier D) as an independent check."""
    wl = synth.CONFIG2
    dev = synth.make_snapshot(wl, 0, device="cuda")
    snap = {k: (v.cpu().numpy() if v is not None else None) for k, v in dev.items()}
    N, cell = wl.image_size, wl.cell_size_deg
    rc, img_o, info_o, ex = _oracle(snap, N, cell, weighting, pol_a=0, pol_b=3, want_indices=True)
    assert rc == 0
    with GpuImager(snap, N, cell, weighting, pol_a=0, pol_b=3) as gi:
        img_g, info_g, _ = gi.image()
        assert np.max(np.abs(np.array(info_g["V"]) - info_o["V"])) <= 1e-12
        toi.toi_debug_set_transform(gi.plan, info_o["V"])
        img_g, info_g, _ = gi.image()
        iu_g, iv_g = gi.indices()
        assert np.array_equal(iu_g, ex["iu"]) and np.array_equal(iv_g, ex["iv"])
        for k in ("n_gridded", "n_off_grid", "n_flagged"):
            assert info_g[k] == info_o[k], k
        assert abs(info_g["wsum"] - info_o["wsum"]) <= 2e-6 * abs(info_o["wsum"])
        _assert_image(img_g, img_o, "config 2 %s (injected V)" % weighting)
        toi.toi_debug_set_transform(gi.plan, None)
        img_g, _, _ = gi.image()
        _assert_image(img_g, img_o, "config 2 %s" % weighting)
    # sampled pixels against the definition (Eq. 7): centre, brightest, corners, seeded others
    rng = np.random.default_rng(2)
    jj, ii = np.unravel_index(np.argmax(img_o), img_o.shape)
    pi = np.concatenate([[N // 2, ii, 0, N - 1], rng.integers(0, N, 8)]).astype(np.int32)
    pj = np.concatenate([[N // 2, jj, 0, N - 1], rng.integers(0, N, 8)]).astype(np.int32)
    wt = oracle.UNIFORM if weighting == "uniform" else oracle.NATURAL
    rc, re, _, _ = oracle.image_dft_pixels(snap["uvw_m"], snap["vis"], snap["weights"], snap["flags"],
                                           snap["chan_freq_hz"], N, cell, pi, pj, weighting=wt, pol_a=0, pol_b=3)
    assert rc == 0
    peak = float(np.max(np.abs(img_o)))
    assert np.max(np.abs(img_g[pj, pi] - re)) <= MAX_ABS_BAR * peak


@pytest.mark.slow
@pytest.mark.parametrize("cfg,n_dft", [(5, 8), (4, 6)])
def test_configs_4_and_5_full_size(cfg, n_dft):
    """BASELINE.json configs[3] (2016 x 32768 channels, 8192^2 image, G = 16384: 3.4 GB of inputs, a
    2.1 GB grid) and configs[4] (low elevation, 1024 channels, 4096^2 image, G = 8192) at full size,
    natural weighting, in the launch configuration bench.py times: whole image against Tier G, counts
    and Wsum, and sampled pixels against the direct DFT of Eq. 7 (Tier D)."""
    wl = synth.CONFIGS[cfg]
    dev = synth.make_snapshot(wl, 0, device="cuda")
    snap = {k: (v.cpu().numpy() if v is not None else None) for k, v in dev.items()}
    del dev
    torch.cuda.empty_cache()
    N, cell = wl.image_size, wl.cell_size_deg
    rc, img_o, info_o, _ = _oracle(snap, N, cell, "natural", pol_a=0, pol_b=3)
    assert rc == 0
    with GpuImager(snap, N, cell, "natural", pol_a=0, pol_b=3) as gi:
        img_g, info_g, _ = gi.image()
    assert np.max(np.abs(np.array(info_g["V"]) - info_o["V"])) <= 1e-12
    for k in ("n_gridded", "n_off_grid", "n_flagged"):
        assert abs(info_g[k] - info_o[k]) <= max(2, info_o["n_gridded"] // 100000), k    # own V on both sides (G5 iii)
    assert abs(info_g["wsum"] - info_o["wsum"]) <= 2e-6 * abs(info_o["wsum"])
    _assert_image(img_g, img_o, "config %d natural" % cfg)
    rng = np.random.default_rng(cfg)
    jj, ii = np.unravel_index(np.argmax(img_o), img_o.shape)
    pi = np.concatenate([[N // 2, ii], rng.integers(0, N, n_dft - 2)]).astype(np.int32)
    pj = np.concatenate([[N // 2, jj], rng.integers(0, N, n_dft - 2)]).astype(np.int32)
    rc, re, _, _ = oracle.image_dft_pixels(snap["uvw_m"], snap["vis"], snap["weights"], snap["flags"],
                                           snap["chan_freq_hz"], N, cell, pi, pj, pol_a=0, pol_b=3)
    assert rc == 0
    peak = float(np.max(np.abs(img_o)))
    assert np.max(np.abs(img_g[pj, pi] - re)) <= MAX_ABS_BAR * peak


# ------------------------------------------------------------------------------------------------
# the sparse clear (k_clear.cu): tiles marked by the gridder / the density pass, or all of them
# ------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("weighting", ["natural", "uniform"])
def test_unsorted_channels_take_the_mark_every_tile_path(weighting):
    """The gridder bounds the tiles a strip can touch by the strip's two end samples, which needs
    monotone channel frequencies; a plan with shuffled channels marks every tile instead.  Same image
    as the oracle (which does not care about the channel order), twice in a row, and the same again
    after a DIFFERENT snapshot was imaged in between (nothing of it may be left on the grid)."""
    wl = _reduced2(n_ant=14, n_chan=200, image_size=256)
    snap = snapshot_np(wl)
    other = snapshot_np(wl, 7)
    perm = np.random.default_rng(5).permutation(wl.n_chan)
    for s in (snap, other):
        s["chan_freq_hz"] = np.ascontiguousarray(s["chan_freq_hz"][perm])
        for k in ("vis", "weights", "flags"):
            s[k] = np.ascontiguousarray(s[k][:, perm, :])
    rc, img_o, info_o, _ = _oracle(snap, wl.image_size, wl.cell_size_deg, weighting, pol_a=0, pol_b=3)
    assert rc == 0
    with GpuImager(snap, wl.image_size, wl.cell_size_deg, weighting, pol_a=0, pol_b=3) as gi:
        for k in range(4):
            gi.set_inputs(other if k == 2 else snap)
            img, info, _ = gi.image()
            if k != 2:
                assert info["n_gridded"] == info_o["n_gridded"]
                _assert_image(img, img_o, "shuffled channels, call %d" % k)


@pytest.mark.parametrize("weighting", ["natural", "uniform"])
def test_different_snapshots_in_a_row_leave_nothing_behind(weighting):
    """Sparse clear with the gridder's own tile marks (sorted channels): snapshots with different
    geometry (hour angles 20 min apart: other tiles) alternate on one plan; each image equals its oracle."""
    wl = synth.reduced(_reduced2(n_ant=14, n_chan=160, image_size=256), dt_s=1200.0)
    snaps = [snapshot_np(wl, k) for k in range(3)]
    refs = [_oracle(s, wl.image_size, wl.cell_size_deg, weighting, pol_a=0, pol_b=3)[1] for s in snaps]
    with GpuImager(snaps[0], wl.image_size, wl.cell_size_deg, weighting, pol_a=0, pol_b=3) as gi:
        for k in (0, 1, 2, 0, 2, 1):
            gi.set_inputs(snaps[k])
            img, _, _ = gi.image()
            _assert_image(img, refs[k], "snapshot %d" % k)


def test_debug_exports_need_their_plan_flag():
    wl = synth.reduced(synth.CONFIG1, n_ant=6, n_core=6, n_chan=8, image_size=32, cell_arcsec=60.0)
    snap = snapshot_np(wl)
    with GpuImager(snap, wl.image_size, wl.cell_size_deg) as gi:
        with pytest.raises(toi.ToiError) as ei:
            toi.toi_debug_keep_grid(gi.plan, True)
        assert ei.value.code == toi.TOI_ERR_UNSUPPORTED
        with pytest.raises(toi.ToiError) as ei:
            toi.toi_image_snapshot_3d(gi.plan, gi.t["uvw_m"], gi.t["vis"])
        assert ei.value.code == toi.TOI_ERR_UNSUPPORTED
    with pytest.raises(toi.ToiError) as ei:            # G > 32768: a window base must fit 2 x 16 bits
        toi.toi_plan_create(3, 2, 2, [1.0e9, 1.1e9], 64, 0.01, grid_size=32770)
    assert ei.value.code == toi.TOI_ERR_INVALID_ARG


# ------------------------------------------------------------------------------------------------
# full size: the other configs of BASELINE.json, at the sizes bench.py times
# ------------------------------------------------------------------------------------------------
def _full_size_case(wl, snapshot, weighting, n_dft, what):
    dev = synth.make_snapshot(wl, snapshot, device="cuda")
    snap = {k: (v.cpu().numpy() if v is not None else None) for k, v in dev.items()}
    del dev
    torch.cuda.empty_cache()
    N, cell = wl.image_size, wl.cell_size_deg
    rc, img_o, info_o, _ = _oracle(snap, N, cell, weighting, pol_a=0, pol_b=3)
    assert rc == 0
    with GpuImager(snap, N, cell, weighting, pol_a=0, pol_b=3) as gi:
        img_g, info_g, _ = gi.image()
    assert np.max(np.abs(np.array(info_g["V"]) - info_o["V"])) <= 1e-12
    for k in ("n_gridded", "n_off_grid", "n_flagged"):
        assert abs(info_g[k] - info_o[k]) <= max(2, info_o["n_gridded"] // 100000), k    # own V on both sides (G5 iii)
    assert abs(info_g["wsum"] - info_o["wsum"]) <= 2e-6 * abs(info_o["wsum"])
    e = _assert_image(img_g, img_o, what)
    print("%s: rel-L2 %.3e, max/peak %.3e" % (what, e[0], e[1]))
    if n_dft:
        rng = np.random.default_rng(wl.config_id + snapshot)
        jj, ii = np.unravel_index(np.argmax(img_o), img_o.shape)
        pi = np.concatenate([[N // 2, ii], rng.integers(0, N, n_dft - 2)]).astype(np.int32)
        pj = np.concatenate([[N // 2, jj], rng.integers(0, N, n_dft - 2)]).astype(np.int32)
        wt = oracle.UNIFORM if weighting == "uniform" else oracle.NATURAL
        rc, re, _, _ = oracle.image_dft_pixels(snap["uvw_m"], snap["vis"], snap["weights"], snap["flags"],
                                               snap["chan_freq_hz"], N, cell, pi, pj, weighting=wt, pol_a=0, pol_b=3)
        assert rc == 0
        peak = float(np.max(np.abs(img_o)))
        assert np.max(np.abs(img_g[pj, pi] - re)) <= MAX_ABS_BAR * peak
    return snap, img_g, info_o


@pytest.mark.slow
@pytest.mark.parametrize("snapshot", [0, 749, 1499])
def test_config3_stream_snapshots_full_size(snapshot):
    """BASELINE.json configs[2]: snapshots 0, 749 and 1499 of the 1500-snapshot run (hour angle advanced
    by 0, 25 and 50 minutes; the 5 mJy pulsar is off, ON, off), uniform weighting, against Tier G."""
    wl = synth.CONFIG3
    l, m, flux = synth.sky_model(wl, snapshot)
    assert (float(flux[-1]) > 0.0) == (snapshot == 749)
    _full_size_case(wl, snapshot, "uniform", 0, "config 3 snapshot %d uniform" % snapshot)


@pytest.mark.slow
def test_config4_uniform_full_size():
    """BASELINE.json configs[3] asks for natural AND uniform: the uniform half (density pass over 66 M
    samples, 1 GB density map), whole image against Tier G plus sampled pixels against Tier D."""
    _full_size_case(synth.CONFIG4, 0, "uniform", 4, "config 4 uniform")


@pytest.mark.slow
def test_config5_last_snapshot_full_size():
    """BASELINE.json configs[4]: the other end of the elevation sweep (snapshot 511, elevation 35 deg,
    plane tilt ~55 deg; snapshot 0 at 20 deg / 70 deg is test_configs_4_and_5_full_size)."""
    snap, _, info_o = _full_size_case(synth.CONFIG5, 511, "natural", 6, "config 5 snapshot 511")
    assert 0.5 < info_o["omega"] < 0.65
