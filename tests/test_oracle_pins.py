"""Pins of the fp64 CPU oracle (oracle/) against what the paper and the mathematics fix.

No GPU, no CUDA path: every check compares the oracle with something other than itself --
Eq. 7 summed by brute force in numpy, numpy.linalg.svd, numpy.fft,
scipy quadrature, closed forms (1 Jy point source, shift theorem, Parseval) and invariants
(orthogonality, omega = |V33|, Hermitian symmetry, linearity).  Pin numbers P1..P14 are those of
DESIGN.md section 3.  The paper prints no worked numerical example for the 2-D path, so there
is no tests/golden/ fixture for it (tests/golden/README.md).
"""
from __future__ import annotations

import math

import numpy as np
import pytest
import scipy.integrate

import oracle
from paper_2512_06254_b200 import synth
from helpers import rel_l2, snapshot_np, tiny

C0 = 299792458.0


# ----------------------------------------------------------------------------- numpy Eq. 7
def eq7_numpy(uvw_m, vis_I, w_I, freq, V, N, cell_deg, keep=None):
    """Eq. 7 written out: I(t1,t2) = 1/(omega Wsum) sum_q z_q exp[i2pi(r1 t1 + r2 t2)],
    R = B V^T, B = uvw * nu/c, pixel grid of Eq. 9."""
    s = freq / C0
    B = uvw_m[:, None, :] * s[None, :, None]                 # [n_b, n_c, 3] wavelengths
    R = B @ V.T
    r1, r2 = R[..., 0].ravel(), R[..., 1].ravel()
    z = vis_I.ravel().astype(np.complex128)
    w = w_I.ravel().astype(np.float64)
    if keep is not None:
        r1, r2, z, w = r1[keep.ravel()], r2[keep.ravel()], z[keep.ravel()], w[keep.ravel()]
    omega = abs(V[0, 0] * V[1, 1] - V[1, 0] * V[0, 1])
    beta = math.radians(cell_deg)
    t1 = -beta * (np.arange(N) - N // 2)                      # column i
    t2 = +beta * (np.arange(N) - N // 2)                      # row j
    ph = 2j * np.pi * (r1[None, None, :] * t1[None, :, None] + r2[None, None, :] * t2[:, None, None])
    img = (np.exp(ph) * z[None, None, :]).sum(-1) / (omega * w.sum())
    return img


def stokes_I(snap, pols):
    """unit-weight, unflagged parallel-hand sum: z = V_a + V_b, w_I = 2."""
    a, b = pols
    z = snap["vis"][:, :, a].astype(np.complex128) + snap["vis"][:, :, b].astype(np.complex128)
    return z, np.full(z.shape, 2.0)


# ----------------------------------------------------------------------------- P1, Tier D
def test_tierD_matches_numpy_eq7_tiny():
    wl = tiny()
    s = snapshot_np(wl)
    rc, re, im, info = oracle.image_dft(s["uvw_m"], s["vis"], None, None, s["chan_freq_hz"],
                                        wl.image_size, wl.cell_size_deg)
    assert rc == 0
    z, w = stokes_I(s, wl.pols)
    ref = eq7_numpy(s["uvw_m"], z, w, s["chan_freq_hz"], info["V"], wl.image_size, wl.cell_size_deg)
    assert np.abs(re - ref.real).max() < 1e-12 * np.abs(ref).max()
    assert np.abs(im - ref.imag).max() < 1e-12 * np.abs(ref).max()
    assert info["n_gridded"] == wl.n_baselines * wl.n_chan


def test_tierD_numpy_eq7_tilted_geometry():
    """Same brute force with a non-trivial V (low elevation, config-5 geometry)."""
    wl = synth.reduced(synth.CONFIG5, n_ant=7, n_core=5, outer_km=1.0, n_chan=4, image_size=16,
                       cell_arcsec=4.0, n_src=3, noise_sigma=0.0, flag_frac=0.0, unit_weights=True)
    s = snapshot_np(wl)
    rc, re, im, info = oracle.image_dft(s["uvw_m"], s["vis"], None, None, s["chan_freq_hz"],
                                        wl.image_size, wl.cell_size_deg)
    assert rc == 0 and info["omega"] < 0.5       # plane tilted ~70 deg
    z, w = stokes_I(s, wl.pols)
    ref = eq7_numpy(s["uvw_m"], z, w, s["chan_freq_hz"], info["V"], wl.image_size, wl.cell_size_deg)
    assert np.abs(re - ref.real).max() < 1e-11 * np.abs(ref).max()


def test_P1_gridded_matches_dft_config1():
    """Tier G vs Tier D on BASELINE config 1 (256^2, 7680 samples): the kernel-aliasing bound."""
    wl = synth.CONFIG1
    s = snapshot_np(wl)
    rc, img, info, _ = oracle.image_gridded(s["uvw_m"], s["vis"], None, None, s["chan_freq_hz"],
                                            wl.image_size, wl.cell_size_deg)
    assert rc == 0
    rc, re, _, info_d = oracle.image_dft(s["uvw_m"], s["vis"], None, None, s["chan_freq_hz"],
                                         wl.image_size, wl.cell_size_deg)
    assert rc == 0
    z, w = stokes_I(s, wl.pols)
    bound = 2e-6 * np.abs(z).sum() / w.sum()
    assert np.abs(img - re).max() <= bound
    assert rel_l2(img, re) <= 5e-6
    assert info["wsum"] == info_d["wsum"] == 2.0 * 7680


@pytest.mark.parametrize("weighting", [oracle.NATURAL, oracle.UNIFORM])
def test_P1_gridded_matches_dft_weights_flags(weighting):
    """Tier G vs Tier D with weights, flags, 4 pols, tilted plane and both weightings."""
    wl = synth.reduced(synth.CONFIG2, n_ant=12, n_core=9, outer_km=2.0, n_chan=48, image_size=64,
                       cell_arcsec=12.0, n_src=5, flag_frac=0.1, noise_sigma=0.05)
    s = snapshot_np(wl)
    rc, img, info, _ = oracle.image_gridded(s["uvw_m"], s["vis"], s["weights"], s["flags"],
                                            s["chan_freq_hz"], wl.image_size, wl.cell_size_deg,
                                            weighting=weighting)
    assert rc == 0 and info["n_flagged"] > 0
    rc, re, _, info_d = oracle.image_dft(s["uvw_m"], s["vis"], s["weights"], s["flags"],
                                         s["chan_freq_hz"], wl.image_size, wl.cell_size_deg,
                                         weighting=weighting)
    assert rc == 0
    assert rel_l2(img, re) <= 5e-6
    assert info["wsum"] == pytest.approx(info_d["wsum"], rel=1e-14)


# ----------------------------------------------------------------------------- P2
@pytest.mark.parametrize("tier", ["G", "D"])
def test_P2_unit_point_source_is_1Jy(tier):
    """V_a = V_b = 1 for every sample, natural weights: peak at centre pixel, peak * omega = 1."""
    for wl in (tiny(n_ant=8, n_chan=8, image_size=32),
               synth.reduced(synth.CONFIG5, n_ant=8, n_core=6, n_chan=8, image_size=32, cell_arcsec=10.0)):
        uvw = synth.baseline_uvw_m(wl).numpy()
        freq = synth.chan_freq_hz(wl).numpy()
        vis = np.ones((wl.n_baselines, wl.n_chan, wl.n_pol), np.complex64)
        N = wl.image_size
        if tier == "G":
            rc, img, info, _ = oracle.image_gridded(uvw, vis, None, None, freq, N, wl.cell_size_deg)
            tol = 2e-6
        else:
            rc, img, _, info = oracle.image_dft(uvw, vis, None, None, freq, N, wl.cell_size_deg)
            tol = 1e-12
        assert rc == 0
        assert np.unravel_index(np.argmax(img), img.shape) == (N // 2, N // 2)
        assert img[N // 2, N // 2] * info["omega"] == pytest.approx(1.0, abs=tol)
        if wl.flat_array:
            assert info["omega"] == pytest.approx(1.0, abs=1e-14)


# ----------------------------------------------------------------------------- P3
def test_P3_hermitian_input_gives_real_image():
    wl = tiny(n_ant=7, n_chan=6, image_size=24)
    s = snapshot_np(wl)
    uvw2 = np.concatenate([s["uvw_m"], -s["uvw_m"]])
    vis2 = np.concatenate([s["vis"], np.conj(s["vis"])])
    rc, re0, _, info0 = oracle.image_dft(s["uvw_m"], s["vis"], None, None, s["chan_freq_hz"],
                                         wl.image_size, wl.cell_size_deg)
    # inject the same V: the plane fit of the doubled set has the same normal but let nothing vary
    rc2, re, im, _ = oracle.image_dft(uvw2, vis2, None, None, s["chan_freq_hz"], wl.image_size,
                                      wl.cell_size_deg, V_in=info0["V"])
    assert rc == 0 and rc2 == 0
    assert np.abs(im).max() <= 1e-12 * np.abs(re).max()
    assert np.abs(re - re0).max() <= 1e-12 * np.abs(re0).max()
    # same through the gridded tier (real part only is output; compare with half-plane input)
    _, g0, _, _ = oracle.image_gridded(s["uvw_m"], s["vis"], None, None, s["chan_freq_hz"],
                                       wl.image_size, wl.cell_size_deg, V_in=info0["V"])
    _, g2, _, _ = oracle.image_gridded(uvw2, vis2, None, None, s["chan_freq_hz"], wl.image_size,
                                       wl.cell_size_deg, V_in=info0["V"])
    assert np.abs(g2 - g0).max() <= 1e-12 * np.abs(g0).max()


# ----------------------------------------------------------------------------- P4, P5
@pytest.mark.parametrize("cfg", [1, 2, 5])
@pytest.mark.parametrize("basis", [oracle.BASIS_MINIMAL, oracle.BASIS_PRINCIPAL])
def test_P4_P5_transform_is_a_rotation(cfg, basis):
    wl = synth.reduced(synth.CONFIGS[cfg], n_chan=16)
    uvw = synth.baseline_uvw_m(wl, snapshot=3).numpy()
    rc, V, omega, sing = oracle.plane_fit(uvw, synth.chan_freq_hz(wl).numpy(), basis)
    assert rc == 0
    assert np.abs(V @ V.T - np.eye(3)).max() <= 1e-12
    assert np.linalg.det(V) == pytest.approx(1.0, abs=1e-12)
    assert V[2, 2] > 0
    assert omega == pytest.approx(abs(V[2, 2]), abs=1e-14)       # cofactor identity
    rho = oracle.rotate(uvw, V)
    ln, l0 = np.linalg.norm(rho, axis=1), np.linalg.norm(uvw, axis=1)
    assert np.abs(ln - l0).max() <= 1e-12 * l0.max()
    assert np.abs(rho - uvw @ V.T).max() <= 1e-12 * l0.max()     # R = B V^T


# ----------------------------------------------------------------------------- P6
@pytest.mark.parametrize("tilt_deg", [0.0, 0.7, 55.0, 70.0])
def test_P6_planar_baselines_known_normal(tilt_deg):
    rng = np.random.default_rng(11)
    az = 0.6
    th = math.radians(tilt_deg)
    n = np.array([math.sin(th) * math.cos(az), math.sin(th) * math.sin(az), math.cos(th)])
    e1 = np.cross(n, [0.3, -0.2, 0.9]); e1 /= np.linalg.norm(e1)
    e2 = np.cross(n, e1)
    ab = rng.normal(size=(40, 2)) * [900.0, 400.0]
    uvw = ab[:, :1] * e1 + ab[:, 1:] * e2
    freq = np.linspace(0.9e9, 1.6e9, 12)
    rc, V, omega, sing = oracle.plane_fit(uvw, freq)
    assert rc == 0
    assert np.abs(V[2] - n).max() <= 1e-12
    assert np.abs(oracle.rotate(uvw, V)[:, 2]).max() <= 1e-9
    assert sing[2] <= 1e-6 * sing[1]
    if tilt_deg == 0.0:
        assert np.abs(V - np.eye(3)).max() <= 1e-12             # minimal rotation -> identity


@pytest.mark.parametrize("cfg", [2, 5])
def test_P6_plane_fit_matches_numpy_svd(cfg):
    """The explicit centred matrix Btilde through numpy.linalg.svd."""
    wl = synth.reduced(synth.CONFIGS[cfg], n_ant=20, n_core=14, n_chan=32)
    uvw = synth.baseline_uvw_m(wl).numpy()
    freq = synth.chan_freq_hz(wl).numpy()
    B = (uvw[:, None, :] * (freq / C0)[None, :, None]).reshape(-1, 3)
    Bt = B - B.mean(0)
    _, sv, Vt = np.linalg.svd(Bt, full_matrices=False)
    rc, V, omega, sing = oracle.plane_fit(uvw, freq, oracle.BASIS_MINIMAL)
    assert rc == 0
    assert np.allclose(sing, sv, rtol=1e-10, atol=1e-9 * sv[0])
    n = Vt[2] * np.sign(Vt[2, 2])
    assert np.abs(V[2] - n).max() <= 1e-9                         # conditioning ~ sv2/sv1 gap
    rc, Vp, _, _ = oracle.plane_fit(uvw, freq, oracle.BASIS_PRINCIPAL)
    assert rc == 0
    for k in range(2):                                            # literal reading: rows = principal axes
        assert abs(abs(Vp[k] @ Vt[k]) - 1.0) <= 1e-9


def test_degenerate_geometry_is_reported():
    uvw = np.outer(np.linspace(-500, 500, 20), [1.0, 2.0, 0.5])   # collinear baselines: no plane
    rc, *_ = oracle.plane_fit(uvw, np.linspace(1e9, 1.1e9, 4))
    assert rc == oracle.ERR_DEGENERATE


# ----------------------------------------------------------------------------- cell indices
def test_cell_indices_against_numpy_fp64():
    """DESIGN.md section 3 step 5: the normative expression order, re-evaluated by numpy fp64
    (each numpy ufunc rounds once, no contraction)."""
    wl = synth.reduced(synth.CONFIG2, n_chan=257)
    uvw = synth.baseline_uvw_m(wl).numpy()
    freq = synth.chan_freq_hz(wl).numpy()
    rc, V, _, _ = oracle.plane_fit(uvw, freq)
    rho = oracle.rotate(uvw, V)
    G, W = 2 * wl.image_size, 7
    iu, iv, on = oracle.cell_indices(rho, freq, G, wl.cell_size_deg, W)
    s = freq / C0
    kappa = float(G) * (wl.cell_size_deg * (math.pi / 180.0))
    assert kappa == oracle.kappa(G, wl.cell_size_deg)
    rho_np = (V[None, :, 0] * uvw[:, 0:1] + V[None, :, 1] * uvw[:, 1:2]) + V[None, :, 2] * uvw[:, 2:3]
    assert np.array_equal(rho_np, rho)
    gu = -((rho[:, 0:1] * s[None, :]) * kappa)
    gv = +((rho[:, 1:2] * s[None, :]) * kappa)
    assert np.array_equal(iu, np.floor(gu + 0.5).astype(np.int32))
    assert np.array_equal(iv, np.floor(gv + 0.5).astype(np.int32))
    h = 3
    on_np = (iu >= -G // 2 + h) & (iu <= G // 2 - 1 - h) & (iv >= -G // 2 + h) & (iv <= G // 2 - 1 - h)
    assert np.array_equal(on, on_np)
    assert 0 < (~on).sum() < 0.01 * on.size      # the longest baselines leave the grid (G10)


# ----------------------------------------------------------------------------- P7
@pytest.mark.parametrize("cfg", [1, 5])
def test_P7_source_lands_on_predicted_pixel(cfg):
    """A noise-free source at (l,m): peak at i = N/2 - t1/beta, j = N/2 + t2/beta, t = V s
    (Eqs. 3-4, 162-166 Eq. 9).  Data come from the measurement equation
    (PAPER.md:41), not from the oracle."""
    base = synth.CONFIGS[cfg]
    wl = synth.reduced(base, n_ant=24, n_core=24 if cfg == 1 else 18, n_chan=16, image_size=128,
                       cell_arcsec=8.0, n_src=1, noise_sigma=0.0, flag_frac=0.0, unit_weights=True,
                       flux_lo=1.0, flux_hi=1.0)
    s = snapshot_np(wl, with_noise=False)
    l, m, flux = (t.numpy() for t in synth.sky_model(wl))
    l, m = float(l[0]), float(m[0])
    rc, img, info, _ = oracle.image_gridded(s["uvw_m"], s["vis"], None, None, s["chan_freq_hz"],
                                            wl.image_size, wl.cell_size_deg)
    assert rc == 0
    t = info["V"] @ np.array([l, m, math.sqrt(1 - l * l - m * m) - 1.0])
    beta = math.radians(wl.cell_size_deg)
    N = wl.image_size
    i_exp, j_exp = N / 2 - t[0] / beta, N / 2 + t[1] / beta
    assert 4 < i_exp < N - 4 and 4 < j_exp < N - 4
    assert abs(i_exp - N / 2) > 3 or abs(j_exp - N / 2) > 3       # not a trivially central source
    j_pk, i_pk = np.unravel_index(np.argmax(img), img.shape)
    # sub-pixel peak by a parabola through the peak and its neighbours on each axis
    ci = img[j_pk, i_pk - 1:i_pk + 2]
    cj = img[j_pk - 1:j_pk + 2, i_pk]
    i_sub = i_pk + 0.5 * (ci[0] - ci[2]) / (ci[0] - 2 * ci[1] + ci[2])
    j_sub = j_pk + 0.5 * (cj[0] - cj[2]) / (cj[0] - 2 * cj[1] + cj[2])
    tol = 0.15 if cfg == 1 else 0.5      # cfg 5: neglected r3 t3 term (Eq. 6) smears the peak
    assert abs(i_sub - i_exp) <= tol and abs(j_sub - j_exp) <= tol
    assert img[j_pk, i_pk] * info["omega"] > 0.8 * float(flux[0])


# ----------------------------------------------------------------------------- P8
def test_P8_psi_quadrature():
    G, W = 512, 7
    for n in (0, 1, 17, 128, 255):
        a, b = oracle.psi(n, G, W, 64), oracle.psi(n, G, W, 128)
        assert abs(a - b) <= 1e-12 * abs(oracle.psi(0, G, W, 64))   # sqrt end-point: 2.4e-13 seen
        ref, err = scipy.integrate.quad(
            lambda x: math.exp(2.30 * W * (math.sqrt(max(0.0, 1 - (2 * x / W) ** 2)) - 1.0))
            * math.cos(2 * math.pi * x * n / G), -W / 2, W / 2, epsabs=1e-13, epsrel=1e-13, limit=400)
        assert a == pytest.approx(ref, abs=5e-12)
    assert oracle.phi(0.0) == 1.0
    assert oracle.phi(3.5) == pytest.approx(math.exp(-16.1), rel=1e-12)
    assert oracle.phi(3.5000001) == 0.0
    assert oracle.phi(-1.25) == oracle.phi(1.25)


def test_P8_single_visibility_is_a_plane_wave():
    """One sample: Tier G image = Re exp(i 2 pi (r1 t1 + r2 t2)) / omega at every pixel."""
    N, cell = 64, 20.0 / 3600
    uvw = np.array([[310.7, -142.3, 0.0], [100.0, 50.0, 0.0], [-80.0, 120.0, 0.0]])
    freq = np.array([1.4e9])
    vis = np.zeros((3, 1, 1), np.complex64)
    vis[0, 0, 0] = 0.6 - 0.8j
    w = np.zeros((3, 1, 1), np.float32)
    w[0] = 1.0                                   # the other rows only define the plane (weight 0)
    rc, img, info, _ = oracle.image_gridded(uvw, vis, w, None, freq, N, cell, pol_a=0, pol_b=0)
    assert rc == 0 and info["n_gridded"] == 1 and info["wsum"] == 1.0
    beta = math.radians(cell)
    r = (info["V"] @ uvw[0]) * freq[0] / C0
    t1 = -beta * (np.arange(N) - N // 2)
    t2 = +beta * (np.arange(N) - N // 2)
    ref = ((0.6 - 0.8j) * np.exp(2j * np.pi * (r[0] * t1[None, :] + r[1] * t2[:, None]))).real / info["omega"]
    # kernel-aliasing error, amplified by 1/psi towards the image edge (psi(N/2)/psi(0) = 0.416 per axis)
    assert np.abs(img - ref).max() <= 6e-6
    assert np.abs(img - ref)[N // 4:3 * N // 4, N // 4:3 * N // 4].max() <= 1e-6


# ----------------------------------------------------------------------------- P9
def test_P9_linearity_and_weight_scale_invariance():
    wl = synth.reduced(synth.CONFIG2, n_ant=10, n_core=8, outer_km=2.0, n_chan=24, image_size=32,
                       cell_arcsec=20.0, n_src=4)
    s = snapshot_np(wl)
    args = (s["chan_freq_hz"], wl.image_size, wl.cell_size_deg)
    rng = np.random.default_rng(3)
    v2 = (rng.normal(size=s["vis"].shape) + 1j * rng.normal(size=s["vis"].shape)).astype(np.complex64)
    a = 0.5       # exactly representable: a*v1 + v2 in complex64 then differs only by rounding of the sum
    _, i1, _, _ = oracle.image_gridded(s["uvw_m"], s["vis"], s["weights"], s["flags"], *args)
    _, i2, _, _ = oracle.image_gridded(s["uvw_m"], v2, s["weights"], s["flags"], *args)
    v3 = (a * s["vis"].astype(np.complex128) + v2.astype(np.complex128))
    # keep the sum exact: feed it as two pols of a 2-pol data set is not possible in general, so allow c64 rounding
    _, i3, _, _ = oracle.image_gridded(s["uvw_m"], v3.astype(np.complex64), s["weights"], s["flags"], *args)
    assert np.abs(i3 - (a * i1 + i2)).max() <= 3e-7 * np.abs(i3).max()
    _, i4, info4, _ = oracle.image_gridded(s["uvw_m"], s["vis"], 4.0 * s["weights"], s["flags"], *args)
    assert np.abs(i4 - i1).max() <= 1e-13 * np.abs(i1).max()
    for wt in (oracle.NATURAL, oracle.UNIFORM):
        _, u1, _, _ = oracle.image_gridded(s["uvw_m"], s["vis"], s["weights"], s["flags"], *args, weighting=wt)
        _, u4, _, _ = oracle.image_gridded(s["uvw_m"], s["vis"], 4.0 * s["weights"], s["flags"], *args, weighting=wt)
        assert np.abs(u4 - u1).max() <= 1e-12 * np.abs(u1).max()


# ----------------------------------------------------------------------------- data handling
def test_flags_nan_and_pol_average():
    """flagged -> zero weight; parallel hands averaged with their weights.
    Data under a flag (NaN) is never used; a flagged hand leaves the other alone."""
    wl = tiny(n_ant=7, n_chan=8, image_size=24, n_pol=4)
    s = snapshot_np(wl)
    vis = s["vis"].copy()
    n_b, n_c, n_p = vis.shape
    rng = np.random.default_rng(5)
    wgt = rng.uniform(0.5, 2.0, size=vis.shape).astype(np.float32)
    flg = np.zeros(vis.shape, np.uint8)
    flg[:, 2, :] = 1                     # whole channel
    flg[3, :, 0] = 1                     # one hand of one baseline
    wgt[5, 1, 3] = 0.0                   # zero weight = flagged
    wgt[6, 4, 0] = np.inf                # non-finite weight = flagged
    vis_nan = vis.copy()
    vis_nan[flg.astype(bool)] = np.nan + 1j * np.nan
    vis_nan[5, 1, 3] = np.nan
    vis_nan[6, 4, 0] = np.nan
    args = (s["chan_freq_hz"], wl.image_size, wl.cell_size_deg)
    rc, img, _, info = oracle.image_dft(s["uvw_m"], vis_nan, wgt, flg, *args, pol_a=0, pol_b=3)
    assert rc == 0 and np.isfinite(img).all()
    # independent statement: effective per-hand weights, then Eq. 7 with z = sum_p w_p V_p, Wsum = sum w_p
    we = wgt.astype(np.float64).copy()
    we[flg.astype(bool)] = 0.0
    we[~np.isfinite(we)] = 0.0
    z = np.zeros((n_b, n_c), np.complex128)
    wI = np.zeros((n_b, n_c))
    for p in (0, 3):
        good = we[:, :, p] > 0
        z[good] += we[:, :, p][good] * vis[:, :, p][good].astype(np.complex128)
        wI[good] += we[:, :, p][good]
    rc2, V, _, _ = oracle.plane_fit(s["uvw_m"], s["chan_freq_hz"])
    ref = eq7_numpy(s["uvw_m"], z, wI, s["chan_freq_hz"], V, wl.image_size, wl.cell_size_deg).real
    assert np.abs(img - ref).max() <= 1e-12 * np.abs(ref).max()
    rc, g, infog, _ = oracle.image_gridded(s["uvw_m"], vis_nan, wgt, flg, *args, pol_a=0, pol_b=3)
    assert rc == 0 and np.isfinite(g).all() and rel_l2(g, ref) <= 5e-6
    assert infog["n_flagged"] == n_b                 # only the fully flagged channel drops samples
    assert infog["wsum"] == pytest.approx(wI.sum(), rel=1e-14)


def test_all_flagged_gives_zero_image():
    wl = tiny()
    s = snapshot_np(wl)
    flg = np.ones(s["vis"].shape, np.uint8)
    rc, img, info, _ = oracle.image_gridded(s["uvw_m"], s["vis"], None, flg, s["chan_freq_hz"],
                                            wl.image_size, wl.cell_size_deg)
    assert rc == 0 and info["wsum"] == 0.0 and not img.any()


def test_off_grid_samples_are_dropped_everywhere():
    wl = tiny(n_ant=12, n_chan=8, image_size=16, cell_arcsec=60.0)   # coarse cells => tiny uv grid
    s = snapshot_np(wl)
    G = 2 * wl.image_size
    rc, img, info, ex = oracle.image_gridded(s["uvw_m"], s["vis"], None, None, s["chan_freq_hz"],
                                             wl.image_size, wl.cell_size_deg, want_indices=True)
    assert rc == 0 and 0 < info["n_off_grid"] < wl.n_baselines * wl.n_chan
    on = (np.abs(ex["iu"] + 0.5) <= G / 2 - 3.5) & (np.abs(ex["iv"] + 0.5) <= G / 2 - 3.5)
    assert info["n_off_grid"] == (~on).sum()
    z, w = stokes_I(s, wl.pols)
    ref = eq7_numpy(s["uvw_m"], z, w, s["chan_freq_hz"], info["V"], wl.image_size, wl.cell_size_deg, keep=on).real
    assert info["wsum"] == 2.0 * on.sum()
    assert rel_l2(img, ref) <= 1e-5


# ----------------------------------------------------------------------------- P10
def test_P10_uniform_weighting_invariants():
    wl = synth.reduced(synth.CONFIG2, n_ant=12, n_core=9, outer_km=2.0, n_chan=64, image_size=64,
                       cell_arcsec=12.0, n_src=5, flag_frac=0.1)
    s = snapshot_np(wl)
    rc, img, info, ex = oracle.image_gridded(s["uvw_m"], s["vis"], s["weights"], s["flags"],
                                             s["chan_freq_hz"], wl.image_size, wl.cell_size_deg,
                                             weighting=oracle.UNIFORM, want_density=True, want_indices=True)
    assert rc == 0
    D = ex["density"]
    G = D.shape[0]
    # density is Hermitian-symmetric: D[-iv][-iu] == D[iv][iu] (centred storage, index G/2 = cell 0)
    Dc = D[1:, 1:]
    assert np.array_equal(Dc, Dc[::-1, ::-1])
    # rebuild own(cell) independently from the exported indices + effective weights
    we = s["weights"].astype(np.float64) * (s["flags"] == 0)
    wI = we[:, :, 0] + we[:, :, 3]
    own = np.zeros((G, G))
    on = (np.abs(ex["iu"] + 0.5) <= G / 2 - 3.5) & (np.abs(ex["iv"] + 0.5) <= G / 2 - 3.5)
    np.add.at(own, (ex["iv"][on] + G // 2, ex["iu"][on] + G // 2), wI[on])
    mirror = np.zeros_like(own)
    mirror[1:, 1:] = own[1:, 1:][::-1, ::-1]
    assert np.allclose(D, own + mirror, rtol=1e-13, atol=0)
    occ = own > 0
    assert info["wsum"] == pytest.approx((own[occ] / (own[occ] + mirror[occ])).sum(), rel=1e-12)


def test_P10_uniform_equals_natural_when_one_sample_per_cell():
    N, cell = 32, 30.0 / 3600
    G = 2 * N
    kappa = oracle.kappa(G, cell)
    freq = np.array([C0])                        # s_c = 1: metres are wavelengths
    cells = np.array([[3, 5], [-7, 2], [10, -11], [1, 14], [-4, -9], [12, 6]], float)
    uvw = np.zeros((6, 3))
    uvw[:, 0] = -(cells[:, 0] + 0.21) / kappa    # gu = -r1 kappa
    uvw[:, 1] = +(cells[:, 1] - 0.33) / kappa
    rng = np.random.default_rng(2)
    vis = (rng.normal(size=(6, 1, 1)) + 1j * rng.normal(size=(6, 1, 1))).astype(np.complex64)
    kw = dict(pol_a=0, pol_b=0)
    _, nat, i_n, _ = oracle.image_gridded(uvw, vis, None, None, freq, N, cell, **kw)
    _, uni, i_u, _ = oracle.image_gridded(uvw, vis, None, None, freq, N, cell, weighting=oracle.UNIFORM, **kw)
    assert i_u["wsum"] == 6.0 == i_n["wsum"]      # number of occupied cells
    assert np.abs(uni - nat).max() <= 1e-14 * np.abs(nat).max()
    # uniform is invariant to per-sample weights when each cell holds one sample
    w = rng.uniform(0.5, 3.0, size=(6, 1, 1)).astype(np.float32)
    _, uni_w, _, _ = oracle.image_gridded(uvw, vis, w, None, freq, N, cell, weighting=oracle.UNIFORM, **kw)
    assert np.abs(uni_w - nat).max() <= 1e-6 * np.abs(nat).max()


# ----------------------------------------------------------------------------- P11
def test_P11_shift_theorem():
    """Multiplying data by exp(-i2pi(r1 a + r2 b)) moves the image by (a, b) in (t1, t2)."""
    wl = tiny(n_ant=10, n_chan=8, image_size=64, cell_arcsec=8.0)
    s = snapshot_np(wl)
    N = wl.image_size
    beta = math.radians(wl.cell_size_deg)
    _, img0, info, _ = oracle.image_gridded(s["uvw_m"], s["vis"], None, None, s["chan_freq_hz"], N, wl.cell_size_deg)
    di, dj = 5, -3                                  # move 5 columns right, 3 rows up
    a, b = -beta * di, +beta * dj                   # Eq. 9: t1 decreases with column
    R = (s["uvw_m"] @ info["V"].T)[:, None, :] * (s["chan_freq_hz"] / C0)[None, :, None]
    ph = np.exp(-2j * np.pi * (R[..., 0] * a + R[..., 1] * b))
    vis1 = (s["vis"].astype(np.complex128) * ph[:, :, None])
    # bypass complex64 rounding of the modulated data by comparing at DFT tier in fp64-clean form
    _, img1, _, _ = oracle.image_gridded(s["uvw_m"], vis1.astype(np.complex64), None, None, s["chan_freq_hz"], N, wl.cell_size_deg)
    core0 = img0[8:N - 8, 8:N - 8]
    core1 = img1[8 + dj:N - 8 + dj, 8 + di:N - 8 + di]
    assert np.abs(core1 - core0).max() <= 5e-6 * np.abs(img0).max()


# ----------------------------------------------------------------------------- P12, P13
@pytest.mark.parametrize("n", [8, 12, 64, 256])
def test_P12_fft_matches_numpy(n):
    rng = np.random.default_rng(n)
    a = rng.normal(size=(n, n)) + 1j * rng.normal(size=(n, n))
    assert np.abs(oracle.fft2(a, +1) - np.fft.ifft2(a) * n * n).max() <= 1e-12 * n * n
    assert np.abs(oracle.fft2(a, -1) - np.fft.fft2(a)).max() <= 1e-12 * n * n


def test_P13_grid_to_image_through_numpy_fft():
    """Steps 8-9 re-done with numpy.fft on the oracle's exported grid: FFT sign/shift, crop,
    1/psi correction and 1/(omega Wsum) normalisation; plus Parseval on the uncropped plane."""
    wl = synth.reduced(synth.CONFIG5, n_ant=12, n_core=9, n_chan=16, image_size=64, cell_arcsec=12.0,
                       n_src=3, flag_frac=0.0)
    s = snapshot_np(wl)
    N = wl.image_size
    rc, img, info, ex = oracle.image_gridded(s["uvw_m"], s["vis"], s["weights"], None, s["chan_freq_hz"],
                                             N, wl.cell_size_deg, want_grid=True)
    assert rc == 0
    grid = ex["grid"]
    G = grid.shape[0]
    F = np.fft.fftshift(np.fft.ifft2(np.fft.ifftshift(grid))) * G * G      # centred in, centred out
    assert np.sum(np.abs(F) ** 2) == pytest.approx(G * G * np.sum(np.abs(grid) ** 2), rel=1e-12)
    crop = F[G // 2 - N // 2:G // 2 + N // 2, G // 2 - N // 2:G // 2 + N // 2].real
    psi = np.array([scipy.integrate.quad(
        lambda x, n=n: math.exp(16.1 * (math.sqrt(max(0.0, 1 - (2 * x / 7) ** 2)) - 1.0))
        * math.cos(2 * math.pi * x * n / G), -3.5, 3.5, epsabs=1e-13, epsrel=1e-13, limit=400)[0]
        for n in range(-N // 2, N // 2)])
    ref = crop / (psi[None, :] * psi[:, None] * info["omega"] * info["wsum"])
    assert np.abs(img - ref).max() <= 1e-10 * np.abs(ref).max()
    # the grid itself: total = sum_q z_q * (sum of taps)^2-ish is not closed form, but the number of
    # touched cells is bounded by 49 per gridded sample and the grid is empty outside footprints
    assert 0 < np.count_nonzero(grid) <= 49 * info["n_gridded"]


# ----------------------------------------------------------------------------- P14
def test_P14_thread_count_independence():
    wl = synth.reduced(synth.CONFIG2, n_ant=12, n_core=9, outer_km=2.0, n_chan=64, image_size=64,
                       cell_arcsec=12.0, n_src=5)
    s = snapshot_np(wl)
    n0 = oracle.num_threads()
    out = []
    try:
        for nt in (1, 3, max(2, n0)):
            oracle.set_num_threads(nt)
            rc, img, info, ex = oracle.image_gridded(s["uvw_m"], s["vis"], s["weights"], s["flags"],
                                                     s["chan_freq_hz"], wl.image_size, wl.cell_size_deg,
                                                     weighting=oracle.UNIFORM, want_grid=True)
            assert rc == 0
            out.append((img, ex["grid"]))
    finally:
        oracle.set_num_threads(n0)
    for img, grid in out[1:]:
        assert np.array_equal(grid, out[0][1])
        assert np.array_equal(img, out[0][0])
