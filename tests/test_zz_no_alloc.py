"""-m gpu: toi_cell_indices_static -- the entry point that allocates nothing (its scratch is a file-scope
__device__ array, include/toi.h) -- against the plan's own path (toi_image_snapshot +
toi_debug_cell_indices).  Index work: bit-exact, the bar of tests/test_gpu_parity.py; V within 1e-12.
Collected last on purpose (the suite runs with pytest -x).  Passes alone in a fresh process (the first
call then does the per-device cudaGetSymbolAddress set-up) and after the other tests."""
from __future__ import annotations

import numpy as np
import pytest

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")

from paper_2512_06254_b200 import binding as toi  # noqa: E402
from paper_2512_06254_b200 import synth  # noqa: E402

from gpu_helpers import GpuImager  # noqa: E402
from helpers import snapshot_np  # noqa: E402


@pytest.fixture(scope="module", autouse=True)
def _need_gpu():
    assert torch.cuda.is_available(), "the -m gpu tests need a CUDA device"
    toi.load()


def _plan_path(snap, wl):
    """The existing path: a plan images the snapshot, then exports the centre cells and V."""
    with GpuImager(snap, wl.image_size, wl.cell_size_deg, "natural", pol_a=0, pol_b=wl.n_pol - 1) as gi:
        _, info, _ = gi.image()
        iu, iv = gi.indices()
    return iu, iv, info


def _static_path(snap, wl, iu, iv, fit):
    """The allocation-free entry point; iu, iv, fit are the caller's (pre-allocated) device tensors."""
    uvw = torch.from_numpy(np.ascontiguousarray(snap["uvw_m"])).cuda()
    n_b, n_c = uvw.shape[0], len(snap["chan_freq_hz"])
    iu_v, iv_v = iu[: n_b * n_c].view(n_b, n_c), iv[: n_b * n_c].view(n_b, n_c)
    toi.toi_cell_indices_static(uvw, snap["chan_freq_hz"], 2 * wl.image_size, wl.cell_size_deg, iu_v, iv_v, fit)
    torch.cuda.synchronize()
    return iu_v.cpu().numpy(), iv_v.cpu().numpy(), fit.cpu().numpy()


def test_static_entry_point_matches_the_plan_on_two_calls_in_a_row():
    """Two different snapshots back to back through the same static scratch: the second has fewer channels,
    another array layout and another hour angle, so anything left over from the first call would show."""
    wl_a = synth.reduced(synth.CONFIG2, n_ant=14, n_core=10, n_chan=777, image_size=512, n_src=5)
    wl_b = synth.reduced(synth.CONFIG5, n_ant=11, n_core=8, n_chan=130, image_size=256, n_src=5)
    # outputs allocated once, before either call, for the larger case
    n_max = max(wl.n_baselines * wl.n_chan for wl in (wl_a, wl_b))
    iu = torch.empty(n_max, dtype=torch.int32, device="cuda")
    iv = torch.empty_like(iu)
    fit = torch.empty(13, dtype=torch.float64, device="cuda")
    for k, (wl, snapshot) in enumerate(((wl_a, 0), (wl_b, 3), (wl_a, 0))):
        snap = snapshot_np(wl, snapshot)
        iu.fill_(-12345)
        iv.fill_(-12345)
        iu_s, iv_s, fit_s = _static_path(snap, wl, iu, iv, fit)
        iu_p, iv_p, info = _plan_path(snap, wl)
        assert np.array_equal(iu_s, iu_p), "call %d: iu differs in %d samples" % (k, int(np.sum(iu_s != iu_p)))
        assert np.array_equal(iv_s, iv_p), "call %d: iv differs in %d samples" % (k, int(np.sum(iv_s != iv_p)))
        assert np.max(np.abs(fit_s[:9] - np.asarray(info["V"]).reshape(9))) <= 1e-12
        assert abs(fit_s[9] - info["omega"]) <= 1e-12
        assert np.allclose(fit_s[10:13], np.asarray(info["sing"]), rtol=1e-12, atol=0.0)


def test_static_entry_point_rejects_what_its_scratch_cannot_hold():
    uvw = torch.zeros((6, 3), dtype=torch.float64, device="cuda")
    n_c = toi.TOI_STATIC_MAX_CHANNELS + 1
    iu = torch.empty((6, 4), dtype=torch.int32, device="cuda")
    iv = torch.empty_like(iu)
    with pytest.raises(toi.ToiError) as e:
        toi.toi_cell_indices_static(uvw, np.linspace(1.0e9, 1.1e9, n_c), 64, 0.01, iu, iv)
    assert e.value.code == toi.TOI_ERR_UNSUPPORTED and "TOI_STATIC_MAX_CHANNELS" in str(e.value)
    with pytest.raises(toi.ToiError) as e:
        toi.toi_cell_indices_static(uvw, [1.0e9, -1.0, 1.1e9, 1.2e9], 64, 0.01, iu, iv)
    assert e.value.code == toi.TOI_ERR_INVALID_ARG
