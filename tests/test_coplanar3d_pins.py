"""Pins of oracle/coplanar3d.py (CPU only): the near-coplanar 3-D mode of PAPER.md:202-269
(section 3.4, Eqs. 17-27).  Pins: the paper's own worked numbers (Table 1, tests/golden/), the sphere
constraint, the Jacobi-Anger identity against direct evaluation, and Eq. 23 against Eq. 18."""
from __future__ import annotations

import math
import os

import numpy as np
import pytest
import scipy.special

from oracle import coplanar3d as o3

GOLDEN = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden", "table1_chebyshev.txt")


def minimal_rotation(a, b):
    c = math.sqrt(1.0 - a * a - b * b)
    return np.array([[1 - a * a / (1 + c), -a * b / (1 + c), -a],
                     [-a * b / (1 + c), 1 - b * b / (1 + c), -b],
                     [a, b, c]])


def table1():
    rows = []
    for line in open(GOLDEN):
        if line.startswith("#") or not line.strip():
            continue
        name, phi, n_slab, alpha, K, nk = line.split()
        rows.append((name, float(phi), int(n_slab), float(alpha), int(K), int(nk)))
    return rows


@pytest.mark.parametrize("row", table1(), ids=lambda r: r[0])
def test_C1_table1_of_the_paper_is_reproduced(row):
    """Phi_max -> (N_slab, alpha_slab, K, N_slab K) with alpha_target = 10,
    gamma = 0.01, K in {8, 16, 24, 32} (Eq. 27 and the sampled-error rule of PAPER.md:267)."""
    name, phi, n_slab, alpha, K, nk = row
    got = o3.select_parameters(phi)
    assert got["n_slab"] == n_slab
    assert abs(got["alpha_slab"] - alpha) < 0.005           # printed to two decimals
    assert got["K"] == K and got["n_slab"] * got["K"] == nk
    assert got["error"] < o3.GAMMA
    assert o3.sampled_error(got["alpha_slab"], 8) > o3.GAMMA    # the next smaller order really fails


@pytest.mark.parametrize("tilt_deg", [0.7, 30.0, 65.0])
def test_C2_t3_satisfies_the_sphere_constraint(tilt_deg):
    """Eq. 17 is the solution of |s + (0,0,1)| = 1 for s = V^T t (App. B1): take
    directions (l, m), form t = V s, and Eq. 17 must return t3 from (t1, t2)."""
    t = math.radians(tilt_deg)
    V = minimal_rotation(math.sin(t) * 0.6, math.sin(t) * 0.8)
    rng = np.random.default_rng(2)
    l = rng.uniform(-0.05, 0.05, 300)
    m = rng.uniform(-0.05, 0.05, 300)
    s = np.stack([l, m, np.sqrt(1 - l * l - m * m) - 1.0])
    tt = V @ s
    assert np.max(np.abs(o3.t3_of(V, tt[0], tt[1]) - tt[2])) < 1e-13


def test_C3_jacobi_anger_expansion_converges_to_the_exponential():
    """Eqs. 21-22 against the exponential itself; the truncation error is bounded by the tail
    2 sum_{k>=K} |J_k(alpha)|."""
    rng = np.random.default_rng(3)
    alpha = rng.uniform(0.0, 12.0, 40)
    s = rng.uniform(-1.0, 1.0, 40)
    for K in (8, 16, 24, 32, 48):
        approx = np.sum(o3.cheb_coeffs(alpha, K) * o3.cheb_T(s, K), axis=-1)
        err = np.abs(np.exp(1j * alpha * s) - approx)
        tail = 2.0 * np.sum(np.abs(scipy.special.jv(np.arange(K, 200)[None, :], alpha[:, None])), axis=1)
        assert np.all(err <= tail + 1e-14)
    assert np.max(err) < 1e-13                               # K = 48 at alpha <= 12
    # T_k against its three-term recurrence
    T = o3.cheb_T(s, 6)
    assert np.max(np.abs(T[:, 5] - (2 * s * T[:, 4] - T[:, 3]))) < 1e-13


def test_C4_slabs_partition_the_r3_range():
    rng = np.random.default_rng(4)
    r3 = rng.normal(0.0, 3.0, 500)
    for n_slab in (1, 3, 17):
        p, centres, d, s = o3.slabs(r3, n_slab)
        assert centres.size == n_slab and p.min() == 0 and p.max() == n_slab - 1
        assert np.all(np.abs(s) <= 1.0 + 1e-12)
        assert np.allclose(centres[p] + s * d, r3, atol=1e-12)       # Eq. 19 inverted
    p, centres, d, s = o3.slabs(np.full(5, 2.5), 4)
    assert d == 0.0 and np.all(s == 0.0) and np.all(p == 0)


@pytest.mark.parametrize("n_slab,K", [(1, 16), (3, 8), (2, 24)])
def test_C5_chebyshev_image_equals_the_direct_3d_sum(n_slab, K):
    """Eq. 23 (slabs + moments) against Eq. 18 (direct sum with r3 t3) on a tiny tilted snapshot:
    the difference is bounded by the sampled expansion error times the mean |Vis|."""
    rng = np.random.default_rng(5)
    t = math.radians(40.0)
    V = minimal_rotation(math.sin(t), 0.0)
    n, N, cell = 60, 24, 0.5
    r = np.column_stack([rng.normal(0, 40, n), rng.normal(0, 40, n), rng.normal(0, 6.0, n)])
    vis = rng.normal(size=n) + 1j * rng.normal(size=n)
    omega = abs(V[0, 0] * V[1, 1] - V[1, 0] * V[0, 1])
    direct = o3.image_3d_direct(r, vis, V, omega, N, cell)
    cheb = o3.image_3d_chebyshev(r, vis, V, omega, N, cell, n_slab, K)
    ok = ~np.isnan(direct)
    assert ok.mean() > 0.9 and np.array_equal(np.isnan(cheb), ~ok)
    phi_max, t3_max = o3.phi_max_of(V, r[:, 2], N, cell)
    eps = o3.sampled_error(phi_max / n_slab, K)
    bound = (eps + 1e-12) * np.sum(np.abs(vis)) / (omega * n)
    assert np.max(np.abs(cheb[ok] - direct[ok])) <= 1.5 * bound
    # and the r3 term matters here: dropping it (the 2-D approximation, Eq. 7) is far off
    flat = o3.image_3d_direct(np.column_stack([r[:, 0], r[:, 1], np.zeros(n)]), vis, V, omega, N, cell)
    assert np.max(np.abs(flat[ok] - direct[ok])) > 100 * np.max(np.abs(cheb[ok] - direct[ok]))


def test_C6_pixel_list_form_of_eq18_equals_the_full_image_form():
    """image_3d_direct_pixels (used where the full N x N sum is too large) is the same Eq. 18 sum as
    image_3d_direct, pixel by pixel -- including the NaN outside the sphere constraint and the
    chunking over samples."""
    rng = np.random.default_rng(11)
    t = math.radians(50.0)
    V = minimal_rotation(math.sin(t) * 0.8, -math.sin(t) * 0.6)
    n, N, cell = 45, 20, 3.0                                    # 60 deg field: some pixels leave the sphere
    r = np.column_stack([rng.normal(0, 10, n), rng.normal(0, 10, n), rng.normal(0, 3.0, n)])
    vis = rng.normal(size=n) + 1j * rng.normal(size=n)
    omega = abs(V[0, 0] * V[1, 1] - V[1, 0] * V[0, 1])
    full = o3.image_3d_direct(r, vis, V, omega, N, cell, wsum=17.5)
    jj, ii = np.mgrid[0:N, 0:N]
    got = o3.image_3d_direct_pixels(r, vis, V, omega, N, cell, ii.ravel(), jj.ravel(), wsum=17.5, chunk=7).reshape(N, N)
    assert np.isnan(full).any() and not np.isnan(full).all()
    assert np.array_equal(np.isnan(got), np.isnan(full))
    ok = ~np.isnan(full)
    assert np.max(np.abs(got[ok] - full[ok])) <= 1e-12 * np.max(np.abs(full[ok]))
    # transposed pixel arguments would show: the image is not symmetric
    swapped = o3.image_3d_direct_pixels(r, vis, V, omega, N, cell, jj.ravel(), ii.ravel(), wsum=17.5).reshape(N, N)
    both = ok & ~np.isnan(swapped)
    assert np.max(np.abs(swapped[both] - full[both])) > 1e-3 * np.max(np.abs(full[ok]))
