"""Seeded synthetic snapshots (inputs only).

This module serves BOTH the CUDA path's tests/bench and the oracle's tests.  It holds none of
the imaging method's arithmetic: it builds telescope geometry (textbook ENU -> uvw), a
point-source sky, and visibilities by the measurement equation PAPER.md:41 (Eq. 1)
``Vis = sum_k S_k exp(-i 2 pi (u l + v m + w (n - 1)))`` plus noise, weights and flags.

The inputs stand in for the paper's private MeerKAT Measurement Sets and OSKAR/PulSKASim
simulations, which are not available; shapes follow BASELINE.json's configs
(recipe in DESIGN.md section 4).  Every random draw is a counter-based hash of
(seed, stream, index) (SplitMix64 finaliser), so any snapshot can be regenerated anywhere, on
CPU or GPU, without generator state.
"""
from __future__ import annotations

import dataclasses
import math

import torch

SEED_BASE = 251206254 * 10
C0 = 299792458.0
EARTH_R = 6.371e6
_M64 = (1 << 64) - 1


def _wrap(v: int) -> int:
    """Python int -> the int64 with the same low 64 bits."""
    v &= _M64
    return v - (1 << 64) if v >= (1 << 63) else v


def _lsr(x: torch.Tensor, k: int) -> torch.Tensor:
    """Logical right shift of int64 (torch's >> is arithmetic)."""
    return (x >> k) & ((1 << (64 - k)) - 1)


def _mix64(x: torch.Tensor) -> torch.Tensor:
    x = x + _wrap(0x9E3779B97F4A7C15)
    x = (x ^ _lsr(x, 30)) * _wrap(0xBF58476D1CE4E5B9)
    x = (x ^ _lsr(x, 27)) * _wrap(0x94D049BB133111EB)
    return x ^ _lsr(x, 31)


def hash_uniform(seed: int, stream: int, idx: torch.Tensor) -> torch.Tensor:
    """Uniform doubles in (0,1), one per int64 index; stateless."""
    idx = idx.to(torch.int64)
    key = _wrap((seed * 0x632BE59BD9B4E019 + stream * 0xD1342543DE82EF95) & _M64)
    h = _mix64(_mix64(idx ^ key) + key)
    return (_lsr(h, 11).to(torch.float64) + 0.5) * (1.0 / 9007199254740992.0)


def hash_normal(seed: int, stream: int, idx: torch.Tensor) -> torch.Tensor:
    """Standard normal doubles by Box-Muller on two hashed uniforms."""
    u1 = hash_uniform(seed, 2 * stream, idx)
    u2 = hash_uniform(seed, 2 * stream + 1, idx)
    return torch.sqrt(-2.0 * torch.log(u1)) * torch.cos(2.0 * math.pi * u2)


@dataclasses.dataclass(frozen=True)
class Workload:
    """One of BASELINE.json's configs (or a reduced variant for tests)."""
    name: str
    config_id: int
    n_ant: int = 64
    n_core: int = 48              # antennas uniform in a 1 km disk; the rest U(1, outer_km) km
    outer_km: float = 8.0
    flat_array: bool = False      # config 1: heights 0, latitude = dec (zenith => w = 0)
    lat_deg: float = -30.713
    dec_deg: float = -30.0
    ha0_deg: float = -7.5         # hour angle of snapshot 0 (H_0 = -0.5 h)
    dt_s: float = 2.0
    n_chan: int = 4096
    f_lo_hz: float = 856e6
    f_hi_hz: float = 1712e6
    n_pol: int = 4
    n_src: int = 200
    flux_lo: float = 1e-3
    flux_hi: float = 1.0
    noise_sigma: float = 0.5
    flag_frac: float = 0.05
    unit_weights: bool = False
    image_size: int = 2048
    cell_arcsec: float = 1.5
    weighting: str = "uniform"
    pulsar_mjy: float = 0.0       # config 3: on/off pulsar flux (on in 30 % of snapshots)
    pulsar_ramp_mjy: tuple = ()   # config 4: (first, last) flux of a pulsar ramping linearly over the run
    n_transients: int = 0         # config 5: faint transients (2-10 mJy), each on in one seeded window of 8-64 snapshots
    n_snapshots: int = 1

    @property
    def seed(self) -> int:
        return SEED_BASE + self.config_id

    @property
    def n_baselines(self) -> int:
        return self.n_ant * (self.n_ant - 1) // 2

    @property
    def cell_size_deg(self) -> float:
        return self.cell_arcsec / 3600.0

    @property
    def pols(self):
        return (0, self.n_pol - 1)


CONFIG1 = Workload("tiny", 1, n_ant=16, n_core=16, flat_array=True, lat_deg=-30.0, dec_deg=-30.0,
                   ha0_deg=0.0, n_chan=64, f_lo_hz=1.30e9, f_hi_hz=1.40e9, n_pol=2, n_src=3,
                   noise_sigma=0.05, flag_frac=0.0, unit_weights=True, image_size=256,
                   cell_arcsec=10.0, weighting="natural")
CONFIG2 = Workload("meerkat_snapshot", 2)
CONFIG3 = Workload("meerkat_stream", 3, pulsar_mjy=5.0, n_snapshots=1500)
CONFIG4 = Workload("wide_deep", 4, n_chan=32768, n_src=400, flag_frac=0.08, image_size=8192,
                   weighting="natural", pulsar_ramp_mjy=(1.0, 20.0), n_snapshots=64)
CONFIG5 = Workload("low_elevation", 5, n_chan=1024, n_src=10, flux_lo=1.0, flux_hi=5.0,
                   ha0_deg=-83.3, image_size=4096, weighting="natural", n_transients=12, n_snapshots=512)
CONFIGS = {1: CONFIG1, 2: CONFIG2, 3: CONFIG3, 4: CONFIG4, 5: CONFIG5}


def chan_freq_hz(wl: Workload) -> torch.Tensor:
    c = torch.arange(wl.n_chan, dtype=torch.float64)
    return wl.f_lo_hz + (c + 0.5) * ((wl.f_hi_hz - wl.f_lo_hz) / wl.n_chan)


def antenna_enu(wl: Workload) -> torch.Tensor:
    """[n_ant, 3] East, North, Up in metres."""
    k = torch.arange(wl.n_ant, dtype=torch.int64)
    u_r, u_az = hash_uniform(wl.seed, 1, k), hash_uniform(wl.seed, 2, k)
    r_core = 1000.0 * torch.sqrt(u_r)
    r_out = 1000.0 * (1.0 + (wl.outer_km - 1.0) * u_r)
    r = torch.where(k < wl.n_core, r_core, r_out)
    az = 2.0 * math.pi * u_az
    e, n = r * torch.sin(az), r * torch.cos(az)
    if wl.flat_array:
        up = torch.zeros_like(e)
    else:
        up = -(e * e + n * n) / (2.0 * EARTH_R) + 2.0 * hash_normal(wl.seed, 3, k)
    return torch.stack([e, n, up], dim=1)


def hour_angle_deg(wl: Workload, snapshot: int) -> float:
    if wl.config_id == 5:   # sweep -83.3 -> -64.7 deg over the run (elevation 20 -> 35 deg)
        return wl.ha0_deg + (18.6 * snapshot) / max(1, wl.n_snapshots - 1)
    return wl.ha0_deg + snapshot * wl.dt_s * (360.0 / 86164.0905)


def baseline_uvw_m(wl: Workload, snapshot: int = 0) -> torch.Tensor:
    """[n_b, 3] fp64 metres, rows (i<j) in row-major pair order, uvw = p_j - p_i, no autos."""
    enu = antenna_enu(wl)
    lat, dec = math.radians(wl.lat_deg), math.radians(wl.dec_deg)
    H = math.radians(hour_angle_deg(wl, snapshot))
    e, n, up = enu[:, 0], enu[:, 1], enu[:, 2]
    X = -math.sin(lat) * n + math.cos(lat) * up
    Y = e
    Z = math.cos(lat) * n + math.sin(lat) * up
    u = math.sin(H) * X + math.cos(H) * Y
    v = -math.sin(dec) * math.cos(H) * X + math.sin(dec) * math.sin(H) * Y + math.cos(dec) * Z
    w = math.cos(dec) * math.cos(H) * X - math.cos(dec) * math.sin(H) * Y + math.sin(dec) * Z
    p = torch.stack([u, v, w], dim=1)
    ii, jj = torch.triu_indices(wl.n_ant, wl.n_ant, offset=1)
    return (p[jj] - p[ii]).contiguous()


def sky_model(wl: Workload, snapshot: int = 0):
    """-> (l, m, flux) fp64 [n_src(+1)]; flat spectrum, unpolarised point sources."""
    k = torch.arange(wl.n_src, dtype=torch.int64)
    beta = math.radians(wl.cell_size_deg)
    if wl.config_id == 1 or wl.n_src == 3:
        flux = torch.tensor([1.0, 0.3, 0.1], dtype=torch.float64)[: wl.n_src]
        rad = math.radians(0.25) * torch.sqrt(hash_uniform(wl.seed, 10, k))
    else:
        a = 1.0 - 1.6   # inverse CDF of N(S) ~ S^-1.6 on [flux_lo, flux_hi]
        uu = hash_uniform(wl.seed, 12, k)
        flux = (wl.flux_lo ** a + uu * (wl.flux_hi ** a - wl.flux_lo ** a)) ** (1.0 / a)
        rad = 0.45 * wl.image_size * beta * torch.sqrt(hash_uniform(wl.seed, 10, k))
    ang = 2.0 * math.pi * hash_uniform(wl.seed, 11, k)
    l, m = rad * torch.cos(ang), rad * torch.sin(ang)
    if wl.pulsar_mjy > 0.0:
        one = torch.zeros(1, dtype=torch.int64)
        on = float(hash_uniform(wl.seed, 20, one + snapshot)) < 0.3
        pr = 0.3 * wl.image_size * beta * math.sqrt(float(hash_uniform(wl.seed, 21, one)))
        pa = 2.0 * math.pi * float(hash_uniform(wl.seed, 22, one))
        l = torch.cat([l, torch.tensor([pr * math.cos(pa)], dtype=torch.float64)])
        m = torch.cat([m, torch.tensor([pr * math.sin(pa)], dtype=torch.float64)])
        flux = torch.cat([flux, torch.tensor([wl.pulsar_mjy * 1e-3 if on else 0.0], dtype=torch.float64)])
    if wl.pulsar_ramp_mjy:
        one = torch.zeros(1, dtype=torch.int64)
        lo, hi = wl.pulsar_ramp_mjy
        f = lo + (hi - lo) * min(max(snapshot, 0), wl.n_snapshots - 1) / max(1, wl.n_snapshots - 1)
        pr = 0.3 * wl.image_size * beta * math.sqrt(float(hash_uniform(wl.seed, 21, one)))
        pa = 2.0 * math.pi * float(hash_uniform(wl.seed, 22, one))
        l = torch.cat([l, torch.tensor([pr * math.cos(pa)], dtype=torch.float64)])
        m = torch.cat([m, torch.tensor([pr * math.sin(pa)], dtype=torch.float64)])
        flux = torch.cat([flux, torch.tensor([f * 1e-3], dtype=torch.float64)])
    if wl.n_transients > 0:
        t = torch.arange(wl.n_transients, dtype=torch.int64)
        tr = 0.4 * wl.image_size * beta * torch.sqrt(hash_uniform(wl.seed, 23, t))
        ta = 2.0 * math.pi * hash_uniform(wl.seed, 24, t)
        tf = (2.0 + 8.0 * hash_uniform(wl.seed, 25, t)) * 1e-3
        width = 8 + torch.floor(57.0 * hash_uniform(wl.seed, 26, t)).to(torch.int64)            # 8 .. 64 snapshots
        start = torch.floor(hash_uniform(wl.seed, 27, t) * (wl.n_snapshots - width).clamp(min=1).to(torch.float64)).to(torch.int64)
        on = (snapshot >= start) & (snapshot < start + width)
        l = torch.cat([l, tr * torch.cos(ta)])
        m = torch.cat([m, tr * torch.sin(ta)])
        flux = torch.cat([flux, torch.where(on, tf, torch.zeros_like(tf))])
    return l, m, flux


def flag_channels(wl: Workload) -> torch.Tensor:
    """bool [n_chan]: seeded contiguous blocks of 16-128 channels until flag_frac is covered
    (blocks are capped at flag_frac * n_chan + 1 channels so reduced test shapes are not all-flagged)."""
    flagged = torch.zeros(wl.n_chan, dtype=torch.bool)
    if wl.flag_frac <= 0.0:
        return flagged
    one = torch.zeros(1, dtype=torch.int64)
    k = 0
    while flagged.double().mean().item() < wl.flag_frac and k < 10000:
        width = min(int(wl.flag_frac * wl.n_chan) + 1, 16 + int(float(hash_uniform(wl.seed, 30, one + k)) * 113))
        start = int(float(hash_uniform(wl.seed, 31, one + k)) * max(1, wl.n_chan - width))
        flagged[start:start + width] = True
        k += 1
    return flagged


def make_snapshot(wl: Workload, snapshot: int = 0, device="cpu", with_noise: bool = True):
    """One time sample in Measurement-Set column shapes.

    -> dict(uvw_m f64 [n_b,3], vis c64 [n_b,n_c,n_p], weights f32 [n_b,n_c,n_p] | None,
            flags u8 [n_b,n_c,n_p] | None, chan_freq_hz f64 [n_c]) on ``device``.
    """
    dev = torch.device(device)
    uvw = baseline_uvw_m(wl, snapshot).to(dev)
    freq = chan_freq_hz(wl).to(dev)
    s = freq / C0
    l, m, flux = (t.to(dev) for t in sky_model(wl, snapshot))
    nm1 = torch.sqrt(1.0 - l * l - m * m) - 1.0
    n_b, n_c, n_p = wl.n_baselines, wl.n_chan, wl.n_pol
    vis = torch.empty((n_b, n_c, n_p), dtype=torch.complex64, device=dev)
    # metres of path difference per (baseline, source); phase = -2 pi s_c * path
    path = uvw[:, 0:1] * l[None, :] + uvw[:, 1:2] * m[None, :] + uvw[:, 2:3] * nm1[None, :]
    chunk = max(1, int(2.0e7 // max(1, n_c * flux.numel())))
    par = (0, n_p - 1)
    for b0 in range(0, n_b, chunk):
        b1 = min(n_b, b0 + chunk)
        ph = (-2.0 * math.pi) * path[b0:b1, None, :] * s[None, :, None]       # [b, c, k]
        val = torch.complex(torch.cos(ph) @ flux, torch.sin(ph) @ flux)         # [b, c]
        block = torch.zeros((b1 - b0, n_c, n_p), dtype=torch.complex128, device=dev)
        for p in set(par):
            block[:, :, p] = val
        if with_noise and wl.noise_sigma > 0.0:
            idx = (torch.arange(b0 * n_c * n_p, b1 * n_c * n_p, dtype=torch.int64, device=dev)
                   + snapshot * (n_b * n_c * n_p))
            nre = hash_normal(wl.seed, 40, idx).reshape(b1 - b0, n_c, n_p)
            nim = hash_normal(wl.seed, 41, idx).reshape(b1 - b0, n_c, n_p)
            block = block + wl.noise_sigma * torch.complex(nre, nim)
        vis[b0:b1] = block.to(torch.complex64)
    weights = flags = None
    if not wl.unit_weights:
        jp = torch.arange(n_b * n_p, dtype=torch.int64, device=dev)
        g = (0.5 + hash_uniform(wl.seed, 50, jp)).reshape(n_b, 1, n_p)
        c = torch.arange(n_c, dtype=torch.float64, device=dev)
        h = (1.0 - 0.3 * torch.cos(2.0 * math.pi * c / n_c)).reshape(1, n_c, 1)
        weights = (g * h).to(torch.float32).contiguous()
    if wl.flag_frac > 0.0:
        fc = flag_channels(wl).to(dev)
        flags = fc.reshape(1, n_c, 1).expand(n_b, n_c, n_p).to(torch.uint8).contiguous()
    return {"uvw_m": uvw.contiguous(), "vis": vis, "weights": weights, "flags": flags,
            "chan_freq_hz": freq.contiguous()}


def reduced(wl: Workload, **kw) -> Workload:
    """A smaller variant of a config for tests (same recipe, fewer antennas/channels/pixels)."""
    return dataclasses.replace(wl, **kw)
