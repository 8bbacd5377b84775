"""Build libqlga.so (hand-written CUDA for sm_100a + the C ABI) in-tree with nvcc.

    python -m paper_1907_12834_b200.build [--force] [-v]

nvcc cross-compiles without a GPU; the resulting .so sits beside this file so it
travels with the source tree to the GPU box.  The translation units compile in
parallel to objects under csrc/build/ (git-ignored) and are linked into one library.
"""
from __future__ import annotations

import os
import subprocess
import sys
from concurrent.futures import ThreadPoolExecutor

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
OBJ = os.path.join(CSRC, "build")
LIB = os.path.join(HERE, "libqlga.so")
SOURCES = ["qlga_api.cu", "qlga_step.cu", "qlga_step_f32.cu", "qlga_step_mixed.cu", "qlga_diag.cu", "qlga_peak.cu", "qlga_track.cu", "qlga_march.cu"]
HEADERS = ["qlga_math.cuh", "qlga_internal.h", "qlga_pass.cuh", os.path.join("..", "..", "include", "qlga.h")]
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17",
              "-Xcompiler", "-fPIC"]


def _newest_header() -> float:
    return max(os.path.getmtime(os.path.join(CSRC, h)) for h in HEADERS)


def _extra() -> list:
    return os.environ.get("QLGA_NVCC_EXTRA", "").split()       # experiment knobs, e.g. -DQLGA_MINB128=4


def build(force: bool = False, verbose: bool = False) -> str:
    nvcc = os.environ.get("NVCC", "nvcc")
    os.makedirs(OBJ, exist_ok=True)
    stamp = os.path.join(OBJ, "flags.txt")
    flags = " ".join(NVCC_FLAGS + _extra())
    if not os.path.exists(stamp) or open(stamp).read() != flags:
        force = True
    hdr = _newest_header()
    jobs = []
    for s in SOURCES:
        src, obj = os.path.join(CSRC, s), os.path.join(OBJ, s[:-3] + ".o")
        if force or not os.path.exists(obj) or os.path.getmtime(obj) < max(os.path.getmtime(src), hdr):
            cmd = [nvcc, *NVCC_FLAGS, *_extra(), "-c", src, "-o", obj]
            if verbose:
                cmd[1:1] = ["-Xptxas", "-v"]
            jobs.append(cmd)
    objs = [os.path.join(OBJ, s[:-3] + ".o") for s in SOURCES]
    if not jobs and os.path.exists(LIB) and os.path.getmtime(LIB) >= max(os.path.getmtime(o) for o in objs):
        return LIB

    def run(cmd):
        if verbose:
            print(" ".join(cmd))
        r = subprocess.run(cmd, cwd=CSRC, capture_output=True, text=True)
        return cmd, r

    with ThreadPoolExecutor(max_workers=max(1, min(len(jobs), os.cpu_count() or 1))) as ex:
        for cmd, r in ex.map(run, jobs):
            if verbose or r.returncode != 0:
                sys.stderr.write(r.stdout + r.stderr)
            if r.returncode != 0:
                raise subprocess.CalledProcessError(r.returncode, cmd)
    subprocess.run([nvcc, "-gencode", "arch=compute_100a,code=sm_100a", "-shared", "-o", LIB, *objs],
                   check=True, cwd=CSRC)
    with open(stamp, "w") as f:
        f.write(flags)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
