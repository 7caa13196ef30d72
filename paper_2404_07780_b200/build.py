"""Build libgm.so (hand-written CUDA for sm_100a) in-tree with nvcc.

``python -m paper_2404_07780_b200.build`` or ``build()``.  One object per PSF
side (gm_tiles.cu with -DGM_K=..) so the heavy, fully unrolled convolution
kernels compile in parallel; nvcc cross-compiles without a GPU.
"""
from __future__ import annotations

import hashlib
import os
import subprocess
import sys
from concurrent.futures import ThreadPoolExecutor
from pathlib import Path

PKG = Path(__file__).resolve().parent
CSRC = PKG / "csrc"
OBJ = PKG / "build"
LIB = PKG / "libgm.so"
INCLUDE = PKG.parent / "include"

KS = (5, 9, 15, 21, 25, 33, 41)          # keep in sync with kCompiledK in gm_api.cu
TC_KS = (9, 17, 25, 33, 41)              # tensor-core engine: padded sides with (K - 1) / 2 a multiple of 4
EXTRA = os.environ.get("GM_NVCC_EXTRA", "").split()
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++20",
              "-Xcompiler", "-fPIC", *EXTRA]


def _nvcc() -> str:
    for cand in (os.environ.get("NVCC"), "/usr/local/cuda/bin/nvcc", "nvcc"):
        if cand and (os.path.sep not in cand or os.path.exists(cand)):
            return cand
    raise RuntimeError("nvcc not found")


def _stamp(files=None) -> str:
    h = hashlib.sha256()
    if files is None:
        files = sorted(list(CSRC.glob("*.cu")) + list(CSRC.glob("*.cuh")))
    for p in list(files) + [INCLUDE / "gm.h", Path(__file__)]:
        h.update(p.name.encode()); h.update(p.read_bytes())
    h.update(" ".join(EXTRA).encode())
    return h.hexdigest()


# what each object is compiled from (an object is rebuilt only when one of these changed)
_DEPS = {
    "gm_api": ["gm_api.cu", "gm_fused.cuh", "gm_kernels.cuh", "gm_device.cuh", "gm_prologue.cuh", "gm_boot.cuh",
               "gm_tc.cuh", "gm_tc_fused.cuh"],
    "gm_tc": ["gm_tc.cu", "gm_tc.cuh", "gm_tc_fused.cuh", "gm_kernels.cuh", "gm_device.cuh"],
    "gm_tiles": ["gm_tiles.cu", "gm_fused.cuh", "gm_kernels.cuh", "gm_device.cuh"],
}


def build(force: bool = False, verbose: bool = False) -> Path:
    stamp_file = OBJ / "stamp"
    stamp = _stamp()
    if not force and LIB.exists() and stamp_file.exists() and stamp_file.read_text() == stamp:
        return LIB
    OBJ.mkdir(exist_ok=True)
    nvcc = _nvcc()
    jobs = [([nvcc, *NVCC_FLAGS, "-c", str(CSRC / "gm_api.cu"), "-o", str(OBJ / "gm_api.o")], "gm_api")]
    for k in TC_KS:
        jobs.append(([nvcc, *NVCC_FLAGS, f"-I{INCLUDE}", f"-DGM_TC_K={k}", "-c", str(CSRC / "gm_tc.cu"),
                      "-o", str(OBJ / f"gm_tc_{k}.o")], f"gm_tc K={k}"))
    for k in KS:
        jobs.append(([nvcc, *NVCC_FLAGS, f"-DGM_K={k}", "-c", str(CSRC / "gm_tiles.cu"),
                      "-o", str(OBJ / f"gm_tiles_{k}.o")], f"gm_tiles K={k}"))

    def run(job):
        cmd, name = job
        obj = Path(cmd[cmd.index("-o") + 1])
        key = name.split()[0]
        want = _stamp([CSRC / f for f in _DEPS[key]]) + " " + " ".join(cmd)
        ostamp = obj.with_suffix(".stamp")
        if not force and obj.exists() and ostamp.exists() and ostamp.read_text() == want:
            return name
        r = subprocess.run(cmd, capture_output=True, text=True)
        if r.returncode != 0:
            raise RuntimeError(f"nvcc failed for {name}:\n{r.stdout}\n{r.stderr}")
        ostamp.write_text(want)
        if verbose:
            print(f"[build] {name} ok", file=sys.stderr)
        return name

    with ThreadPoolExecutor(max_workers=min(len(jobs), os.cpu_count() or 4)) as ex:
        list(ex.map(run, jobs))
    objs = [str(OBJ / "gm_api.o")] + [str(OBJ / f"gm_tc_{k}.o") for k in TC_KS] + [str(OBJ / f"gm_tiles_{k}.o") for k in KS]
    tmp = LIB.with_suffix(f".tmp{os.getpid()}.so")
    r = subprocess.run([nvcc, "-shared", "-gencode", "arch=compute_100a,code=sm_100a", "-o", str(tmp), *objs],
                       capture_output=True, text=True)
    if r.returncode != 0:
        raise RuntimeError(f"link failed:\n{r.stdout}\n{r.stderr}")
    os.replace(tmp, LIB)
    stamp_file.write_text(stamp)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose=True))
