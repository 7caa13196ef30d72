"""Host-side check of the tensor-core engine's tap-row ring protocol (gm_tc.cuh): the producer order and the
ring split must never make the MMA warps wait for a row whose slot they still hold.  tests/tc_ring_check.cu
models both sides with the kernels' own constexpr mapping; built with nvcc as host code, run on the CPU."""
import shutil
import subprocess
from pathlib import Path

import pytest

ROOT = Path(__file__).resolve().parents[1]
CSRC = ROOT / "paper_2404_07780_b200" / "csrc"


def _nvcc():
    for cand in ("/usr/local/cuda/bin/nvcc", shutil.which("nvcc")):
        if cand and Path(cand).exists():
            return cand
    return None


@pytest.mark.parametrize("tile", [(4, 32), (8, 16)])
def test_tap_row_rings_never_deadlock(tmp_path, tile):
    nvcc = _nvcc()
    if nvcc is None:
        pytest.skip("nvcc not found")
    src = (CSRC / "gm_tc.cuh").read_text()
    # the shipped tile shape, and the taller one that exposed the deadlock: same header, other constants
    want = f"constexpr int kTileR = {tile[0]}, kTileC = {tile[1]};"
    assert "constexpr int kTileR = 4, kTileC = 32;" in src
    inc = tmp_path / "pkg" / "csrc"                      # the headers reach gm.h as ../../include/gm.h
    inc.mkdir(parents=True)
    (tmp_path / "include").mkdir()
    (tmp_path / "include" / "gm.h").write_text((ROOT / "include" / "gm.h").read_text())
    (inc / "gm_tc.cuh").write_text(src.replace("constexpr int kTileR = 4, kTileC = 32;", want))
    for name in ("gm_device.cuh", "gm_prologue.cuh"):
        if (CSRC / name).exists():
            (inc / name).write_text((CSRC / name).read_text())
    exe = tmp_path / "ring_check"
    r = subprocess.run([nvcc, "-std=c++20", "-O1", "-gencode", "arch=compute_100a,code=sm_100a", f"-I{inc}",
                        f"-I{ROOT / 'include'}", "-o", str(exe), str(ROOT / "tests" / "tc_ring_check.cu")],
                       capture_output=True, text=True)
    assert r.returncode == 0, r.stderr[-2000:]
    r = subprocess.run([str(exe)], capture_output=True, text=True)
    assert r.returncode == 0, r.stdout
    assert f"tile {tile[0]} x {tile[1]}: ok" in r.stdout
