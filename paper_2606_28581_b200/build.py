"""Build libsatsplat.so (hand-written sm_100a kernels + the C ABI) in-tree with nvcc.

    python -m paper_2606_28581_b200.build [--force]

nvcc cross-compiles without a GPU.  The .so is git-ignored but travels to the GPU box with the snapshot.
"""
from __future__ import annotations

import os
import subprocess
import sys
from concurrent.futures import ThreadPoolExecutor

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
OUT = os.path.join(HERE, "libsatsplat.so")
SOURCES = ["api.cu", "preprocess.cu", "binning.cu", "blend_forward.cu", "blend_backward.cu", "chain_backward.cu", "adam.cu", "losses.cu", "init.cu", "relocate.cu", "relocate_static.cu", "peaks.cu", "camera.cu"]
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17", "-Xcompiler", "-fPIC,-ffp-contract=off",
              "--expt-relaxed-constexpr"]


def _newest_dep() -> float:
    deps = [os.path.join(CSRC, f) for f in os.listdir(CSRC)] + [os.path.join(HERE, "..", "include", "satsplat.h")]
    return max(os.path.getmtime(d) for d in deps)


def _flags_stamp() -> str:
    """Everything besides the sources that decides what the .so contains: a tuning build (SATSPLAT_NVCC_FLAGS=-D...) must not
    survive as the library a later default test or bench run loads."""
    return " ".join(NVCC_FLAGS + os.environ.get("SATSPLAT_NVCC_FLAGS", "").split() + SOURCES)


def build(force: bool = False, verbose: bool = False) -> str:
    objdir = os.path.join(HERE, "build")
    stamp_file = os.path.join(objdir, "flags.stamp")
    stamp_ok = os.path.exists(stamp_file) and open(stamp_file).read() == _flags_stamp()
    if not force and stamp_ok and os.path.exists(OUT) and os.path.getmtime(OUT) >= _newest_dep():
        return OUT
    nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
    os.makedirs(objdir, exist_ok=True)

    def compile_one(src):
        obj = os.path.join(objdir, src.replace(".cu", ".o"))
        extra = os.environ.get("SATSPLAT_NVCC_FLAGS", "").split()     # e.g. -DSATSPLAT_BWD_MINB=8 (tuning experiments)
        cmd = [nvcc, *NVCC_FLAGS, *extra, *( ["-Xptxas", "-v"] if verbose else []), "-c", os.path.join(CSRC, src), "-o", obj]
        r = subprocess.run(cmd, capture_output=True, text=True)
        if r.returncode != 0:
            raise RuntimeError(f"nvcc failed for {src}:\n{r.stdout}\n{r.stderr}")
        if verbose:
            sys.stderr.write(r.stderr)
        return obj

    with ThreadPoolExecutor(max_workers=len(SOURCES)) as ex:
        objs = list(ex.map(compile_one, SOURCES))
    tmp = OUT + f".tmp{os.getpid()}"
    r = subprocess.run([nvcc, "-shared", "-o", tmp, *objs, "-lcudart"], capture_output=True, text=True)
    if r.returncode != 0:
        raise RuntimeError(f"link failed:\n{r.stdout}\n{r.stderr}")
    os.replace(tmp, OUT)
    with open(stamp_file, "w") as f:
        f.write(_flags_stamp())
    return OUT


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
