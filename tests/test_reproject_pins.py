"""Pins of oracle/reproject.py (CPU only): the re-projection stage of PAPER.md:156-200 (section 3.3,
Eqs. 9-16) and PAPER.md:658-704 (Appendix A).  Each pin ties the oracle to something other than
itself: the appendix' trigonometric route, the sphere constraint Eq. 17, a library interpolator,
closed forms, and the measurement equation through the imaging oracle."""
from __future__ import annotations

import math

import numpy as np
import pytest
import scipy.ndimage

import oracle
from oracle import reproject as orp
from paper_2512_06254_b200 import synth
from helpers import snapshot_np


def minimal_rotation(a, b):
    """V whose third row is the unit normal (a, b, c), c > 0 (G3), typed out here."""
    c = math.sqrt(1.0 - a * a - b * b)
    return np.array([[1 - a * a / (1 + c), -a * b / (1 + c), -a],
                     [-a * b / (1 + c), 1 - b * b / (1 + c), -b],
                     [a, b, c]])


def tilt_V(tilt_deg, az_deg=35.0):
    t, z = math.radians(tilt_deg), math.radians(az_deg)
    return minimal_rotation(math.sin(t) * math.cos(z), math.sin(t) * math.sin(z))


# ----------------------------------------------------------------------------- R1
@pytest.mark.parametrize("tilt_deg", [0.0, 0.7, 20.0, 55.0])
@pytest.mark.parametrize("cell_deg", [1.5 / 3600, 0.05, 0.5])
def test_R1_reduced_mapping_equals_appendix_A_route(tilt_deg, cell_deg):
    """Eqs. 9-16 are 'algebraically equivalent to the SIN geometry used by the conventional WCS
    formulation': the route through (phi, theta), Eqs. A1-A7, must give the same
    output pixel.  Also fixes G16's sign (A6's outer minus)."""
    N = 64
    V = tilt_V(tilt_deg)
    p1, p2, ok = orp.map_paper(V, N, cell_deg)
    q1, q2, ok2 = orp.map_wcs_appendix_a(V, N, cell_deg)
    assert np.array_equal(ok, ok2) and ok.all()
    # acos near 1 loses half the digits: compare in pixels at the accuracy the trig route has
    tol = 1e-6 if cell_deg < 0.01 else 1e-9
    assert np.max(np.abs(p1 - q1)) <= tol and np.max(np.abs(p2 - q2)) <= tol


def test_R2_eq12_equals_eq13():
    h = np.linspace(0.0, 57.0, 2001)
    assert np.max(np.abs(orp.sin_z_eq12(h) - orp.sin_z_eq13(h))) <= 2e-16 * 4
    # and Eq. 13 keeps relative accuracy where Eq. 12 cancels
    hs = 1e-6
    exact = 0.5 * (hs / orp.R0) ** 2                    # series, next term 1e-34
    assert abs(orp.sin_z_eq13(hs) / exact - 1.0) < 1e-12


# ----------------------------------------------------------------------------- R3
@pytest.mark.parametrize("mode", ["exact", "paper"])
def test_R3_no_tilt_is_the_identity(mode):
    rng = np.random.default_rng(3)
    img = rng.standard_normal((48, 48))
    out = orp.reproject(img, np.eye(3), 0.01, mode)
    # V = I: t1 = l, t2 = m up to the n - 1 term times V13 = V23 = 0 -> same pixel
    assert np.isfinite(out).all()
    assert np.max(np.abs(out - img)) <= 1e-9


# ----------------------------------------------------------------------------- R4
def eq17_t3(V, t1, t2):
    """PAPER.md:208 Eq. 17, typed out."""
    return -V[2, 2] + np.sign(V[2, 2]) * np.sqrt(1.0 - (t1 + V[0, 2]) ** 2 - (t2 + V[1, 2]) ** 2)


@pytest.mark.parametrize("tilt_deg", [0.7, 25.0, 60.0])
def test_R4_exact_map_inverts_the_sphere_constraint(tilt_deg):
    """Go the OTHER way with the paper's own formulas: a tilted-plane position (t1, t2) has t3 by
    Eq. 17 and direction s = V^T t (Eq. 4).  Mapping that direction's (l, m) with map_exact must
    return the (t1, t2) we started from.  Catches a transposed V, a wrong sign of n - 1, swapped
    axes."""
    V = tilt_V(tilt_deg, az_deg=-70.0)
    N, cell = 96, 0.02
    beta = math.radians(cell)
    rng = np.random.default_rng(4)
    t1 = (rng.uniform(-0.3, 0.3, 200)) * N * beta
    t2 = (rng.uniform(-0.3, 0.3, 200)) * N * beta
    t3 = eq17_t3(V, t1, t2)
    s = V.T @ np.stack([t1, t2, t3])                    # Eq. 4
    l, m = s[0], s[1]
    assert np.max(np.abs(s[2] - (np.sqrt(1 - l * l - m * m) - 1.0))) < 1e-12     # really on the sphere
    got1, got2, ok = orp.tilted_pixel_of_direction(V, l, m, N, cell)
    assert ok.all()
    want1 = N / 2 - t1 / beta
    want2 = N / 2 + t2 / beta
    assert np.max(np.abs(got1 - want1)) < 1e-9 and np.max(np.abs(got2 - want2)) < 1e-9


# ----------------------------------------------------------------------------- R5
def test_R5_paper_map_is_the_small_tilt_limit_of_the_exact_map():
    """Eq. 15 keeps only xi, eta: it must agree with t = V s to first order in the tilt and differ
    at large tilt by the in-plane terms (V11 - 1) l etc.."""
    N, cell = 128, 0.01
    for tilt, bound in [(0.05, 2e-4), (0.7, 2e-2)]:
        V = tilt_V(tilt)
        a1, a2, _ = orp.map_exact(V, N, cell)
        b1, b2, _ = orp.map_paper(V, N, cell)
        d = max(np.max(np.abs(a1 - b1)), np.max(np.abs(a2 - b2)))
        assert d < bound, (tilt, d)
    V = tilt_V(60.0)
    a1, _, _ = orp.map_exact(V, N, cell)
    b1, _, _ = orp.map_paper(V, N, cell)
    assert np.max(np.abs(a1 - b1)) > 5.0                 # pixels: the reduced form is NOT exact there


# ----------------------------------------------------------------------------- R6
def test_R6_bilinear_gather_matches_scipy():
    rng = np.random.default_rng(6)
    N = 40
    img = rng.standard_normal((N, N))
    p1 = rng.uniform(-2.0, N + 1.0, (N, N))
    p2 = rng.uniform(-2.0, N + 1.0, (N, N))
    p1[0, :4] = [0.0, N - 1.0, 5.0, N - 1.0]             # exact edges are inside
    p2[0, :4] = [0.0, N - 1.0, N - 1.0, 7.25]
    valid = np.ones((N, N), bool)
    valid[3, 3] = False
    out = orp.bilinear_gather(img, p1, p2, valid)
    inside = valid & (p1 >= 0) & (p1 <= N - 1) & (p2 >= 0) & (p2 <= N - 1)
    ref = scipy.ndimage.map_coordinates(img, [p2, p1], order=1, mode="nearest")
    assert np.array_equal(np.isnan(out), ~inside)
    assert inside[0, :4].all()
    assert np.max(np.abs(out[inside] - ref[inside])) < 1e-12


def test_R8_edge_rule_of_reading_G22():
    """DESIGN.md G22: a position within 1e-6 px outside [0, N-1]^2 counts as on the edge (and is clipped
    to it), anything further out is NaN.  (a) With V = I the map must be the identity INCLUDING the
    last row and column, whatever the rounding: for N = 250 and this cell size the fp64 evaluation of
    Eq. 16 puts the last column 1.4e-14 px outside -- without the tolerance that column would be lost;
    (b) a position 5e-7 px outside takes the edge value, one 1e-5 px outside is NaN -- a tolerance of
    1e-3 would keep it."""
    N, cell = 250, 0.1061373992010266
    p1, p2, ok = orp.map_exact(np.eye(3), N, cell)
    over = max(p1.max() - (N - 1), -p1.min(), p2.max() - (N - 1), -p2.min())
    assert 0.0 < over < 1e-12                                   # the rounding this rule exists for
    rng = np.random.default_rng(4)
    img = rng.normal(size=(N, N))
    out = orp.reproject(img, np.eye(3), cell, "exact")
    assert not np.isnan(out).any()
    assert np.max(np.abs(out - img)) < 1e-9
    M = 8
    small = rng.normal(size=(M, M))
    p1 = np.full((1, 6), 3.0)
    p2 = np.full((1, 6), 2.0)
    p1[0, :] = [M - 1 + 5e-7, M - 1 + 1e-5, -5e-7, -1e-5, 3.0, 3.0]
    p2[0, 4:] = [M - 1 + 5e-7, -1e-5]
    got = orp.bilinear_gather(small, p1, p2, np.ones((1, 6), bool))[0]
    assert got[0] == small[2, M - 1] and got[2] == small[2, 0] and abs(got[4] - small[M - 1, 3]) < 1e-15
    assert np.isnan(got[1]) and np.isnan(got[3]) and np.isnan(got[5])


def test_R6_bilinear_reproduces_affine_images_exactly():
    N = 32
    jj, ii = np.mgrid[0:N, 0:N].astype(np.float64)
    img = 2.0 - 0.5 * ii + 0.25 * jj
    V = tilt_V(3.0)
    p1, p2, ok = orp.map_exact(V, N, 0.05)
    out = orp.bilinear_gather(img, p1, p2, ok)
    m = np.isfinite(out)
    assert m.sum() > 0.5 * N * N
    assert np.max(np.abs(out[m] - (2.0 - 0.5 * p1[m] + 0.25 * p2[m]))) < 1e-12


# ----------------------------------------------------------------------------- R7
def test_R7_reprojected_source_sits_at_its_true_lm_pixel():
    """End to end through the imaging oracle: a noise-free source at (l, m) observed at low
    elevation (config-5 geometry, plane tilt ~70 deg) peaks, after re-projection, at the pixel of
    its TRUE direction, i = N/2 - l/beta, j = N/2 + m/beta -- where P7 showed that before
    re-projection it sits at t = V s.  Data come from the measurement equation."""
    wl = synth.reduced(synth.CONFIGS[5], n_ant=24, n_core=18, n_chan=16, image_size=128,
                       cell_arcsec=8.0, n_src=1, noise_sigma=0.0, flag_frac=0.0, unit_weights=True,
                       flux_lo=1.0, flux_hi=1.0)
    s = snapshot_np(wl, with_noise=False)
    l, m, _ = (t.numpy() for t in synth.sky_model(wl))
    l, m = float(l[0]), float(m[0])
    rc, img, info, _ = oracle.image_gridded(s["uvw_m"], s["vis"], None, None, s["chan_freq_hz"],
                                            wl.image_size, wl.cell_size_deg)
    assert rc == 0
    V = info["V"]
    assert math.degrees(math.acos(V[2, 2])) > 50.0          # a real tilt
    beta = math.radians(wl.cell_size_deg)
    N = wl.image_size
    i_true, j_true = N / 2 - l / beta, N / 2 + m / beta
    t = V @ np.array([l, m, math.sqrt(1 - l * l - m * m) - 1.0])
    i_tilt, j_tilt = N / 2 - t[0] / beta, N / 2 + t[1] / beta
    assert math.hypot(i_true - i_tilt, j_true - j_tilt) > 8.0  # the two differ by many pixels
    out = orp.reproject(img, V, wl.cell_size_deg, "exact")
    j_pk, i_pk = np.unravel_index(np.nanargmax(out), out.shape)
    # P7 allows the tilted peak 0.5 px of smear from the neglected r3 t3 term (Eq. 6); the map
    # stretches that by up to 1/V33, plus half a pixel of rounding to the nearest pixel
    tol = 0.5 / V[2, 2] + 0.5
    assert tol < 2.5
    assert abs(i_pk - i_true) <= tol and abs(j_pk - j_true) <= tol
    # the tilted image's own peak is elsewhere
    j0, i0 = np.unravel_index(np.argmax(img), img.shape)
    assert abs(i0 - i_tilt) <= 1.0 and abs(j0 - j_tilt) <= 1.0


def test_difference_is_elementwise():
    a = np.arange(12.0).reshape(3, 4)
    b = np.ones((3, 4))
    assert np.array_equal(orp.difference(a, b), a - 1.0)
