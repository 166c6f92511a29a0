"""Shared test helpers (inputs only; no imaging arithmetic of either side)."""
from __future__ import annotations

import numpy as np

from paper_2512_06254_b200 import synth


def snapshot_np(wl, snapshot=0, with_noise=True):
    """synth.make_snapshot -> dict of numpy arrays (None stays None)."""
    s = synth.make_snapshot(wl, snapshot, device="cpu", with_noise=with_noise)
    return {k: (v.numpy() if v is not None else None) for k, v in s.items()}


def tiny(n_ant=6, n_chan=4, image_size=16, cell_arcsec=4.0, **kw):
    """A config-1-shaped workload small enough for O(N^2 S) brute force."""
    return synth.reduced(synth.CONFIG1, n_ant=n_ant, n_core=n_ant, n_chan=n_chan,
                         image_size=image_size, cell_arcsec=cell_arcsec, **kw)


def rel_l2(a, b):
    a = np.asarray(a, dtype=np.float64)
    b = np.asarray(b, dtype=np.float64)
    return float(np.linalg.norm(a - b) / max(np.linalg.norm(b), 1e-300))
