"""Helpers of the -m gpu parity tests: run libtoi through the Python binding (C ABI) on numpy
inputs and hand the results back as numpy.  Marshalling only; no imaging arithmetic."""
from __future__ import annotations

import numpy as np
import torch

from paper_2512_06254_b200 import binding as toi


def to_dev(a, device):
    return None if a is None else torch.from_numpy(np.ascontiguousarray(a)).to(device)


class GpuImager:
    """One plan + resident inputs; ``image()`` images the snapshot and returns numpy results."""

    def __init__(self, snap, N, cell_size_deg, weighting="natural", gridder=toi.TOI_GRIDDER_SLIDING,
                 location=toi.TOI_MEM_DEVICE, pol_a=None, pol_b=None, grid_size=0, apply_jacobian=0,
                 ring_depth=0, keep_grid=False, enable_3d=False):
        vis = snap["vis"]
        self.n_b, self.n_c, self.n_p = vis.shape
        self.N = N
        self.G = grid_size if grid_size else 2 * N
        self.location = location
        wt = toi.TOI_WEIGHT_UNIFORM if weighting == "uniform" else toi.TOI_WEIGHT_NATURAL
        self.plan = toi.toi_plan_create(self.n_b, self.n_c, self.n_p, snap["chan_freq_hz"], N, cell_size_deg,
                                        weighting=wt, pol_a=pol_a, pol_b=pol_b, grid_size=grid_size,
                                        apply_jacobian=apply_jacobian, input_location=location,
                                        image_ring_depth=ring_depth, gridder=gridder, enable_3d=enable_3d,
                                        debug_keep_grid=keep_grid)
        if keep_grid:
            toi.toi_debug_keep_grid(self.plan, True)
        self.set_inputs(snap)

    def set_inputs(self, snap):
        if self.location == toi.TOI_MEM_DEVICE:
            dev = "cuda"
            self.t = {k: to_dev(snap[k], dev) for k in ("uvw_m", "vis", "weights", "flags")}
        else:
            self.t = {k: (None if snap[k] is None else torch.from_numpy(np.ascontiguousarray(snap[k])).pin_memory())
                      for k in ("uvw_m", "vis", "weights", "flags")}

    def image(self, allow_degenerate=False):
        ptr, info, rc = toi.toi_image_snapshot(self.plan, self.t["uvw_m"], self.t["vis"], self.t["weights"],
                                               self.t["flags"], want_info=True,
                                               allow_degenerate=allow_degenerate)
        img = toi.toi_copy_image_to_host(self.plan, ptr, self.N).numpy()
        return img, info.as_dict(), rc

    def image_untimed(self):
        """The call without `info`: no per-stage timing events, no synchronisation inside the call."""
        ptr, _, rc = toi.toi_image_snapshot(self.plan, self.t["uvw_m"], self.t["vis"], self.t["weights"],
                                            self.t["flags"], want_info=False)
        return toi.toi_copy_image_to_host(self.plan, ptr, self.N).numpy(), rc

    def indices(self):
        iu, iv = toi.toi_debug_cell_indices(self.plan, self.n_b, self.n_c)
        return iu.cpu().numpy(), iv.cpu().numpy()

    def grid_centred(self):
        """Pre-FFT grid of the last snapshot; libtoi stores it centred (cell k at k + G/2) like the oracle."""
        return toi.toi_debug_copy_grid(self.plan, self.G).cpu().numpy()

    def density_centred(self):
        return toi.toi_debug_copy_density(self.plan, self.G).cpu().numpy()

    def close(self):
        if self.plan is not None:
            toi.toi_plan_destroy(self.plan)
            self.plan = None

    def __enter__(self):
        return self

    def __exit__(self, *exc):
        self.close()
