"""oracle.reproject -- TEST INFRASTRUCTURE, not product code.

Plain fp64 numpy statement of TOI's re-projection ("interpolate") stage
(section 3.3, Eqs. 9-16) and PAPER.md:658-704 (Appendix A, Eqs. A1-A7): the dirty image that the
2-D Fourier reconstruction leaves on the tilted (t1, t2) plane is resampled onto the standard
(l, m) grid.  Only ``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s CPU legs may import
this module; it shares no code with the CUDA path.

Readings (G20-G23; the paper leaves all four open):
  G20  direction: GATHER.  Output pixel (i, j) of the standard grid looks up the tilted image at
       the fractional pixel (p1', p2') the mapping gives.  Eq. 15's x' = x + r0 z xi is, to first
       order in the tilt, t1 = V11 l + V12 m + V13 (n - 1) of Eq. 4 (t = V s) -- i.e. the map from a
       true (l, m) to where that direction sits on the tilted plane.
  G21  two mappings: "exact" (default) evaluates t = V s of Eqs. 3-4 with no small-tilt assumption;
       "paper" evaluates Eqs. 9-16 literally (tilt enters only through xi = V31/V33, eta = V32/V33).
  G16  Eq. 11/15 sign garble: y' = y + r0 z eta (Appendix A6 has the outer minus), x' = x + r0 z xi.
  G22  interpolation: bilinear on the four neighbours (the paper names none); a pixel whose source
       position falls outside [0, N-1]^2, or outside the SIN domain h <= r0, is NaN.  A position
       within 1e-6 px outside the edge is taken as on the edge (with V = I the positions are the
       integers up to rounding, and the last row/column must not depend on that rounding).
  G23  pixel convention as everywhere else (G6): 0-based, centre N/2, x = -beta (i - N/2),
       y = +beta (j - N/2); Eq. 9's 1-based (N/2 + 1) is the same pixel.

Functions follow the paper's order and notation; nothing is fused or reordered.
"""
from __future__ import annotations

import numpy as np

R0 = 180.0 / np.pi          # Eq. 10


def pixel_to_angle(N, cell_size_deg):
    """Eq. 9 (0-based): x[i] = -beta (i - N/2), y[j] = +beta (j - N/2), degrees. -> (x[N], y[N])."""
    k = np.arange(N, dtype=np.float64) - (N // 2)
    return -cell_size_deg * k, cell_size_deg * k


def sin_z_eq12(h):
    """Eq. 12: z = 1 - sqrt(1 - (h/r0)^2)."""
    return 1.0 - np.sqrt(1.0 - (h / R0) ** 2)


def sin_z_eq13(h):
    """Eq. 13: z = (h/r0)^2 / (1 + sqrt(1 - (h/r0)^2))."""
    q = (h / R0) ** 2
    return q / (1.0 + np.sqrt(1.0 - q))


def map_paper(V, N, cell_size_deg):
    """Eqs. 9-16 at every pixel. -> (p1'[N,N], p2'[N,N], valid[N,N]); arrays are [j][i], 0-based."""
    V = np.asarray(V, dtype=np.float64).reshape(3, 3)
    beta = float(cell_size_deg)
    xs, ys = pixel_to_angle(N, beta)
    x = np.broadcast_to(xs[None, :], (N, N))
    y = np.broadcast_to(ys[:, None], (N, N))
    h = np.sqrt(x * x + y * y)                                    # Eq. 10
    valid = h <= R0
    hs = np.where(valid, h, 0.0)
    nz = hs != 0.0
    xhat = np.where(nz, x / np.where(nz, hs, 1.0), 0.0)           # Eq. 11
    yhat = np.where(nz, y / np.where(nz, hs, 1.0), 1.0)           # Eq. 11 with G16's sign (+y/h)
    z = sin_z_eq13(hs)                                            # Eq. 13 (== Eq. 12)
    xi = V[2, 0] / V[2, 2]                                        # Eq. 14
    eta = V[2, 1] / V[2, 2]
    xp = hs * xhat + R0 * z * xi                                  # Eq. 15
    yp = hs * yhat + R0 * z * eta
    p1 = -xp / beta + N // 2                                      # Eq. 16 (0-based)
    p2 = yp / beta + N // 2
    return p1, p2, valid


def map_wcs_appendix_a(V, N, cell_size_deg):
    """The conventional route through native spherical coordinates, Eqs. A1-A7, written out with
    atan2 / acos / asin exactly as the appendix lists them (its special cases are the limits of the
    general expressions).  Independent of map_paper: used to pin it.  -> (p1', p2', valid)."""
    V = np.asarray(V, dtype=np.float64).reshape(3, 3)
    beta = float(cell_size_deg)
    k = np.arange(N, dtype=np.float64) - (N // 2)
    xr = np.broadcast_to((-(np.pi / 180.0) * beta * k)[None, :], (N, N))      # A1, radians
    yr = np.broadcast_to(((np.pi / 180.0) * beta * k)[:, None], (N, N))
    r2 = xr * xr + yr * yr
    valid = r2 <= 1.0
    r2s = np.where(valid, r2, 0.0)
    phi = np.degrees(np.arctan2(xr, -yr))                                     # A2
    phi = np.where((xr == 0.0) & (yr <= 0.0), 0.0, phi)
    phi = np.where((xr == 0.0) & (yr > 0.0), 180.0, phi)
    r = np.sqrt(r2s)
    theta_a = np.degrees(np.arccos(np.clip(r, -1.0, 1.0)))                    # A3 (x^2 + y^2 < 0.5)
    theta_b = np.degrees(np.arcsin(np.clip(np.sqrt(1.0 - r2s), -1.0, 1.0)))   # A4 (0.5 <= . <= 1)
    theta = np.where(r2s < 0.5, theta_a, theta_b)
    xi = V[2, 0] / V[2, 2]                                                    # A5
    eta = V[2, 1] / V[2, 2]
    th, ph = np.radians(theta), np.radians(phi)
    x = R0 * (np.cos(th) * np.sin(ph) + xi * (1.0 - np.sin(th)))              # A6
    y = -R0 * (np.cos(th) * np.cos(ph) - eta * (1.0 - np.sin(th)))
    p1 = -x / beta + N // 2                                                   # A7 (0-based)
    p2 = y / beta + N // 2
    return p1, p2, valid


def tilted_pixel_of_direction(V, l, m, N, cell_size_deg):
    """Eqs. 3-4 with no approximation, for directions (l, m) (arrays, direction cosines):
    s = (l, m, n - 1), n = sqrt(1 - l^2 - m^2); t = V s; the place of t on the tilted image is
    p1' = N/2 - t1/beta_rad, p2' = N/2 + t2/beta_rad (Eq. 9 inverted). -> (p1', p2', valid)."""
    V = np.asarray(V, dtype=np.float64).reshape(3, 3)
    beta_rad = float(cell_size_deg) * (np.pi / 180.0)
    l = np.asarray(l, dtype=np.float64)
    m = np.asarray(m, dtype=np.float64)
    q = l * l + m * m
    valid = q <= 1.0
    qs = np.where(valid, q, 0.0)
    n = np.sqrt(1.0 - qs)                                         # Eq. 3
    s3 = n - 1.0
    t1 = V[0, 0] * l + V[0, 1] * m + V[0, 2] * s3                 # Eq. 4: t = V s
    t2 = V[1, 0] * l + V[1, 1] * m + V[1, 2] * s3
    p1 = -t1 / beta_rad + N // 2
    p2 = t2 / beta_rad + N // 2
    return p1, p2, valid


def map_exact(V, N, cell_size_deg):
    """tilted_pixel_of_direction at every output pixel: (l, m) = (x, y) * pi/180 of Eq. 9."""
    beta_rad = float(cell_size_deg) * (np.pi / 180.0)
    k = np.arange(N, dtype=np.float64) - (N // 2)
    l = np.broadcast_to((-beta_rad * k)[None, :], (N, N))
    m = np.broadcast_to((beta_rad * k)[:, None], (N, N))
    return tilted_pixel_of_direction(V, l, m, N, cell_size_deg)


def bilinear_gather(image, p1, p2, valid):
    """G22: out[j][i] = bilinear(image at column p1[j][i], row p2[j][i]); NaN where the position is
    invalid or outside [0, N-1]^2 (by more than 1e-6 px).  Plain definition, no vector tricks beyond numpy indexing."""
    img = np.asarray(image, dtype=np.float64)
    N = img.shape[0]
    assert img.shape == (N, N)
    eps = 1e-6          # G22: a position within 1e-6 px outside the edge counts as on the edge
    inside = valid & (p1 >= -eps) & (p1 <= N - 1.0 + eps) & (p2 >= -eps) & (p2 <= N - 1.0 + eps)
    a = np.clip(np.where(inside, p1, 0.0), 0.0, N - 1.0)
    b = np.clip(np.where(inside, p2, 0.0), 0.0, N - 1.0)
    i0 = np.minimum(np.floor(a), N - 2).astype(np.int64)
    j0 = np.minimum(np.floor(b), N - 2).astype(np.int64)
    fx = a - i0
    fy = b - j0
    top = (1.0 - fx) * img[j0, i0] + fx * img[j0, i0 + 1]
    bot = (1.0 - fx) * img[j0 + 1, i0] + fx * img[j0 + 1, i0 + 1]
    out = (1.0 - fy) * top + fy * bot
    return np.where(inside, out, np.nan)


def reproject(image, V, cell_size_deg, mode="exact"):
    """Tilted-plane image [N][N] -> standard (l, m) grid [N][N] (fp64)."""
    N = np.asarray(image).shape[0]
    mapper = {"exact": map_exact, "paper": map_paper}[mode]
    p1, p2, valid = mapper(V, N, cell_size_deg)
    return bilinear_gather(image, p1, p2, valid)


def difference(image_a, image_b):
    """Difference image of two consecutive snapshots (the quantity the downstream transient search
    consumes): a - b, element by element."""
    return np.asarray(image_a, dtype=np.float64) - np.asarray(image_b, dtype=np.float64)
