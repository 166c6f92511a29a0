"""oracle.coplanar3d -- TEST INFRASTRUCTURE, not product code.

Plain fp64 numpy statement of TOI's near-coplanar ("3-D") mode, PAPER.md:202-269 (section 3.4,
Eqs. 17-27) and PAPER.md:706-796 (Appendix B): the residual coordinate r3 is kept, its range is cut
into slabs, and inside a slab the residual phase exp(i alpha s_q) is expanded in Chebyshev
polynomials (Jacobi-Anger), so that the image is a sum of N_slab * K two-dimensional
reconstructions ("Chebyshev moments").

Written and pinned before the CUDA path of this mode (``toi_image_snapshot_3d``), which is checked
against it in ``tests/test_gpu_coplanar3d.py``.  Only ``tests/`` may import it; it shares no code
with the CUDA path.

Everything here is brute force (direct Fourier sums, no gridding, no FFT) and follows the paper's
order and notation: it is the definition the future gridded/FFT path must reach.
Library primitives used as steps: scipy.special.jv (Bessel J_k), numpy.cos/arccos (T_k).

Readings (the paper leaves these open):
  G24  slabs: N_slab equal-width slabs over [r3_min, r3_max], half-width
       Delta_r3 = (r3_max - r3_min) / (2 N_slab), centres r3_min + (2p + 1) Delta_r3; a sample on an
       interior boundary belongs to the upper slab, r3_max to the last.  A snapshot with
       r3_max = r3_min has Delta_r3 = 0: s_q = 0, one moment.
  G25  K selection samples |exp(i alpha s) - sum_k c_k T_k(s)| on a 129 x 257 grid of
       [0, alpha_slab] x [-1, 1]; alpha_slab = Phi_max / N_slab (Table 1's third column).  This
       rule reproduces all three rows of Table 1.
  G26  valid image region D of Eq. 25: every pixel of the N x N image whose (t1, t2) lies inside
       the sphere constraint of Eq. 17.
"""
from __future__ import annotations

import numpy as np
import scipy.special

ALPHA_TARGET = 10.0
GAMMA = 1e-2
K_CHOICES = (8, 16, 24, 32)


def t3_of(V, t1, t2):
    """Eq. 17: t3(t1, t2) = -V33 + sgn(V33) sqrt(1 - (t1 + V13)^2 - (t2 + V23)^2); NaN outside."""
    V = np.asarray(V, dtype=np.float64).reshape(3, 3)
    rad = 1.0 - (np.asarray(t1) + V[0, 2]) ** 2 - (np.asarray(t2) + V[1, 2]) ** 2
    with np.errstate(invalid="ignore"):
        return -V[2, 2] + np.sign(V[2, 2]) * np.sqrt(rad)


def cheb_coeffs(alpha, K):
    """Eq. 22: c_0 = J_0(alpha), c_k = 2 i^k J_k(alpha).  alpha: array [...]; -> complex [..., K]."""
    alpha = np.asarray(alpha, dtype=np.float64)
    k = np.arange(K)
    return np.where(k == 0, 1.0, 2.0) * (1j ** k) * scipy.special.jv(k, alpha[..., None])


def cheb_T(s, K):
    """T_k(s) = cos(k arccos s) for k < K, -1 <= s <= 1.  s: array [...]; -> [..., K]."""
    s = np.clip(np.asarray(s, dtype=np.float64), -1.0, 1.0)
    return np.cos(np.arange(K) * np.arccos(s)[..., None])


def sampled_error(alpha_slab, K, n_alpha=129, n_s=257):
    """max over the sampling grid of |exp(i alpha s) - sum_{k<K} c_k(alpha) T_k(s)| (Eq. 21; G25)."""
    a = np.linspace(0.0, alpha_slab, n_alpha)
    s = np.linspace(-1.0, 1.0, n_s)
    approx = cheb_coeffs(a, K) @ cheb_T(s, K).T                     # [n_alpha, n_s]
    return float(np.max(np.abs(np.exp(1j * a[:, None] * s[None, :]) - approx)))


def select_parameters(phi_max, alpha_target=ALPHA_TARGET, gamma=GAMMA, k_choices=K_CHOICES):
    """Eq. 27 and the K rule of PAPER.md:267. -> dict(n_slab, alpha_slab, K, error)."""
    n_slab = max(1, int(np.ceil(phi_max / alpha_target)))
    alpha_slab = phi_max / n_slab
    K, err = k_choices[-1], None
    for cand in k_choices:
        e = sampled_error(alpha_slab, cand)
        if e < gamma:
            K, err = cand, e
            break
    if err is None:
        err = sampled_error(alpha_slab, K)
    return {"n_slab": n_slab, "alpha_slab": alpha_slab, "K": K, "error": err}


def phi_max_of(V, r3, N, cell_size_deg):
    """Eqs. 25-26: Phi_max = 2 pi t3_max (r3_max - r3_min) / 2 over the valid pixels of the image."""
    beta = np.radians(cell_size_deg)
    k = np.arange(N, dtype=np.float64) - (N // 2)
    t3 = t3_of(V, (-beta * k)[None, :], (beta * k)[:, None])
    t3_max = float(np.nanmax(np.abs(t3)))
    r3 = np.asarray(r3, dtype=np.float64)
    return 2.0 * np.pi * t3_max * (r3.max() - r3.min()) / 2.0, t3_max


def slabs(r3, n_slab):
    """G24. -> (p[q] slab index, centres[n_slab], half-width Delta_r3, s_q of Eq. 19)."""
    r3 = np.asarray(r3, dtype=np.float64)
    lo, hi = r3.min(), r3.max()
    d = (hi - lo) / (2.0 * n_slab)
    if d == 0.0:
        return np.zeros(r3.shape, np.int64), np.array([lo]), 0.0, np.zeros_like(r3)
    p = np.minimum(np.floor((r3 - lo) / (2.0 * d)).astype(np.int64), n_slab - 1)
    centres = lo + (2.0 * np.arange(n_slab) + 1.0) * d
    return p, centres, d, (r3 - centres[p]) / d


def image_3d_direct(r, vis, V, omega, N, cell_size_deg, wsum=None):
    """Eq. 18 by brute force: I(t1,t2) = 1/(omega N_vis) sum_q Vis_q exp[i 2 pi (r1 t1 + r2 t2 + r3 t3)].
    r: [n, 3] transformed baselines (wavelengths), vis: complex [n].  -> complex [N, N] (NaN outside
    the sphere constraint)."""
    beta = np.radians(cell_size_deg)
    k = np.arange(N, dtype=np.float64) - (N // 2)
    t1 = np.broadcast_to((-beta * k)[None, :], (N, N))
    t2 = np.broadcast_to((beta * k)[:, None], (N, N))
    t3 = t3_of(V, t1, t2)
    r = np.asarray(r, dtype=np.float64)
    vis = np.asarray(vis, dtype=np.complex128)
    norm = omega * (vis.size if wsum is None else wsum)
    img = np.zeros((N, N), np.complex128)
    for q in range(vis.size):
        img += vis[q] * np.exp(2j * np.pi * (r[q, 0] * t1 + r[q, 1] * t2 + r[q, 2] * t3))
    return img / norm


def image_3d_direct_pixels(r, vis, V, omega, N, cell_size_deg, pix_i, pix_j, wsum=None, chunk=1 << 18):
    """Eq. 18 at the listed pixels only (i = column, j = row), for inputs too large for the full image:
    the same sum as image_3d_direct, pixel by pixel.  -> complex [n_pix] (NaN outside the sphere constraint)."""
    beta = np.radians(cell_size_deg)
    pix_i = np.asarray(pix_i, dtype=np.int64).ravel()
    pix_j = np.asarray(pix_j, dtype=np.int64).ravel()
    t1 = -beta * (pix_i - (N // 2)).astype(np.float64)
    t2 = beta * (pix_j - (N // 2)).astype(np.float64)
    t3 = t3_of(V, t1, t2)
    r = np.asarray(r, dtype=np.float64)
    vis = np.asarray(vis, dtype=np.complex128)
    norm = omega * (vis.size if wsum is None else wsum)
    out = np.zeros(pix_i.size, np.complex128)
    for q0 in range(0, vis.size, chunk):
        rq, vq = r[q0:q0 + chunk], vis[q0:q0 + chunk]
        ph = rq[:, 0:1] * t1[None, :] + rq[:, 1:2] * t2[None, :] + rq[:, 2:3] * t3[None, :]     # [n, n_pix]
        out += vq @ np.exp(2j * np.pi * ph)
    return out / norm


def image_3d_chebyshev(r, vis, V, omega, N, cell_size_deg, n_slab, K, wsum=None):
    """Eqs. 19-24 step by step: slabs, s_q, moments M_{p,k} (each a 2-D Fourier sum, Eq. 24), then
    I = 1/(omega N_vis) sum_p exp(i 2 pi r3_p t3) sum_k c_k(2 pi Delta_r3 t3) M_{p,k} (Eq. 23)."""
    beta = np.radians(cell_size_deg)
    kpx = np.arange(N, dtype=np.float64) - (N // 2)
    t1 = np.broadcast_to((-beta * kpx)[None, :], (N, N))
    t2 = np.broadcast_to((beta * kpx)[:, None], (N, N))
    t3 = t3_of(V, t1, t2)
    r = np.asarray(r, dtype=np.float64)
    vis = np.asarray(vis, dtype=np.complex128)
    norm = omega * (vis.size if wsum is None else wsum)
    p, centres, d, s = slabs(r[:, 2], n_slab)
    Tk = cheb_T(s, K)                                                    # [n, K]
    ck = cheb_coeffs(2.0 * np.pi * d * np.nan_to_num(t3), K)             # [N, N, K]  (Eq. 20: alpha)
    img = np.zeros((N, N), np.complex128)
    for sp in range(centres.size):
        sel = np.nonzero(p == sp)[0]
        if sel.size == 0:
            continue
        M = np.zeros((N, N, K), np.complex128)                           # Eq. 24
        for q in sel:
            plane = vis[q] * np.exp(2j * np.pi * (r[q, 0] * t1 + r[q, 1] * t2))
            M += plane[:, :, None] * Tk[q][None, None, :]
        img += np.exp(2j * np.pi * centres[sp] * t3) * np.sum(ck * M, axis=2)   # Eq. 23
    return np.where(np.isnan(t3), np.nan, img / norm)
