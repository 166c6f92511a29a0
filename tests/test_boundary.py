"""-m "not gpu": the C-ABI library builds, loads and exports every symbol include/toi.h declares;
the Python binding mirrors the header; without a GPU the product path fails loudly (no CPU
fallback); the oracle and the CUDA path share no code."""
from __future__ import annotations

import ctypes as C
import os
import re

import pytest

torch = pytest.importorskip("torch")

from paper_2512_06254_b200 import binding as toi  # noqa: E402
from paper_2512_06254_b200 import build as toi_build  # noqa: E402

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
HEADER = os.path.join(ROOT, "include", "toi.h")


def _declared_functions():
    src = open(HEADER).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    names = re.findall(r"^\s*(?:const\s+char\s*\*|int)\s*(toi_[a-z0-9_]+)\s*\(", src, flags=re.M)
    names = [n for n in names if not n.endswith("_fn")]
    return sorted(set(names))


def test_header_declares_the_four_entry_points():
    names = _declared_functions()
    for need in ("toi_plan_create", "toi_image_snapshot", "toi_image_stream", "toi_plan_destroy"):
        assert need in names


def test_library_builds_and_exports_every_declared_symbol():
    lib_path = toi_build.build_library()
    assert os.path.exists(lib_path)
    lib = C.CDLL(lib_path)
    for name in _declared_functions():
        assert hasattr(lib, name), "libtoi.so does not export %s" % name
    assert sorted(toi.EXPORTS) == _declared_functions()


def test_library_is_built_for_sm_100a():
    import subprocess
    out = subprocess.run(["cuobjdump", "--list-elf", toi_build.build_library()], capture_output=True, text=True).stdout
    assert "sm_100a" in out


def test_struct_layouts_match_the_header(tmp_path):
    """sizeof/offsetof as gcc sees include/toi.h == the ctypes mirrors of the binding."""
    import subprocess
    src = tmp_path / "layout.c"
    src.write_text(
        '#include <stdio.h>\n#include <stddef.h>\n#include "toi.h"\n'
        'int main(void){printf("%zu %zu %zu %zu %zu %zu %zu %zu %zu %zu %zu\\n", sizeof(toi_3d_info), offsetof(toi_3d_info, ms_total), sizeof(toi_config), sizeof(toi_snapshot_info),'
        ' sizeof(toi_snapshot_buffers), sizeof(toi_stream_stats), offsetof(toi_config, chan_freq_hz),'
        ' offsetof(toi_config, debug_keep_grid), offsetof(toi_snapshot_info, ms_clear_density), sizeof(toi_stream_output),'
        ' offsetof(toi_stream_output, host_sink));return 0;}\n')
    exe = tmp_path / "layout"
    subprocess.run(["gcc", "-I", os.path.join(ROOT, "include"), str(src), "-o", str(exe)], check=True)
    got = [int(x) for x in subprocess.run([str(exe)], capture_output=True, text=True, check=True).stdout.split()]
    want = [C.sizeof(toi.toi_3d_info), toi.toi_3d_info.ms_total.offset, C.sizeof(toi.toi_config), C.sizeof(toi.toi_snapshot_info), C.sizeof(toi.toi_snapshot_buffers),
            C.sizeof(toi.toi_stream_stats), toi.toi_config.chan_freq_hz.offset, toi.toi_config.debug_keep_grid.offset,
            toi.toi_snapshot_info.ms_clear_density.offset, C.sizeof(toi.toi_stream_output), toi.toi_stream_output.host_sink.offset]
    assert got == want


@pytest.mark.skipif(torch.cuda.is_available(), reason="checks the no-GPU behaviour")
def test_no_gpu_means_loud_failure_not_cpu_fallback():
    with pytest.raises(toi.ToiError) as ei:
        toi.toi_plan_create(3, 2, 2, [1.0e9, 1.1e9], 32, 0.01)
    assert ei.value.code == toi.TOI_ERR_CUDA
    assert "no CPU fallback" in str(ei.value)


def test_invalid_config_is_refused_before_touching_the_device():
    with pytest.raises(toi.ToiError) as ei:
        toi.toi_plan_create(3, 2, 3, [1.0e9, 1.1e9], 32, 0.01)      # n_pols = 3
    assert ei.value.code == toi.TOI_ERR_INVALID_ARG


def test_oracle_and_cuda_path_share_no_code():
    pkg = os.path.join(ROOT, "paper_2512_06254_b200")
    for dirpath, _, files in os.walk(pkg):
        if "build" in dirpath.split(os.sep)[-1:]:
            continue
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h", ".cpp")):
                text = open(os.path.join(dirpath, f), errors="replace").read()
                assert not re.search(r"^\s*(from|import)\s+oracle\b", text, flags=re.M), f
                assert "toi_oracle" not in text, f
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith((".py", ".c", ".h")):
            text = open(os.path.join(ROOT, "oracle", f), errors="replace").read()
            assert not re.search(r"^\s*(from|import)\s+paper_2512_06254_b200", text, flags=re.M), f
            assert '#include "toi' not in text and "csrc/" not in text.replace("paper_2512_06254_b200/csrc", ""), f


@pytest.mark.parametrize("G", [16, 18, 136, 198, 202, 384, 4096, 4098, 32766, 32768])
def test_gridder_window_overhang_stays_inside_the_guard_band(G):
    """The product gridder flushes an 8 x 8-cell register window whose corner sits on even cells,
    base = (centre - 3) & ~1, so it can overhang the grid by one row / column (of zeros).  The plan
    allocates grid_guard(G) = ceil((G + 8) / 32) * 32 cells in front of and behind the grid for that.
    compute-sanitizer is closed on this GPU pool, so the bound is checked here by enumeration: over all
    on-grid centre cells (-G/2 + 3 <= i <= G/2 - 4 on both axes) the lowest and highest flat cell index a
    window can touch must stay within [-guard, G*G + guard)."""
    h = G // 2
    guard = (G + 8 + 31) // 32 * 32
    centres = range(-h + 3, h - 3)                     # on-grid centre cells (reading G10)
    bases = sorted({(c - 3) & ~1 for c in centres})    # Python's & on negative ints is two's complement, like the kernel's
    lo_b, hi_b = bases[0], bases[-1]
    assert lo_b >= -h - 1 and hi_b + 7 <= h           # at most one cell outside on either side
    lowest = (lo_b + h) * G + (lo_b + h)
    highest = (hi_b + 7 + h) * G + (hi_b + 7 + h)
    assert lowest >= -guard and highest < G * G + guard
