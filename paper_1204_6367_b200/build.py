"""Builds libgdrr_b200.so (the C-ABI library of include/gdrr.h) in-tree with nvcc
for sm_100a.  nvcc cross-compiles without a GPU.

    python paper_1204_6367_b200/build.py [--force] [--verbose]

(run as a file: importing the package first would load the library that is being replaced)
"""
import os
import shutil
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(HERE)
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libgdrr_b200.so")
SOURCES = ["gdrr_api.cu", "project_fused.cu", "project_packed.cu", "project_staged.cu", "project_siddon.cu", "project_texture.cu", "denoise.cu", "volume_layout.cu", "debug_cells.cu", "energy_sum.cu"]
HEADERS = ["gdrr_internal.h", "denoise_static.h", "ray_setup.cuh", "project_common.cuh", "packed_sampler.cuh", os.path.join(ROOT, "include", "gdrr.h")]

NVCC_FLAGS = [
    "-gencode", "arch=compute_100a,code=sm_100a",
    "-O3", "-std=c++17", "-lineinfo", "-ftz=true",
    "-Xcompiler", "-fPIC,-ffp-contract=off,-fvisibility=hidden",
    "-Xptxas", "-v",
]


def find_nvcc() -> str:
    for cand in (os.environ.get("NVCC"), shutil.which("nvcc"), "/usr/local/cuda/bin/nvcc"):
        if cand and os.path.exists(cand):
            return cand
    raise RuntimeError("nvcc not found; libgdrr_b200.so cannot be built")


def _stale() -> bool:
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    deps = [os.path.join(CSRC, s) for s in SOURCES] + [
        h if os.path.isabs(h) else os.path.join(CSRC, h) for h in HEADERS] + [__file__]
    return any(os.path.getmtime(d) > t for d in deps)


def build(force: bool = False, verbose: bool = False) -> str:
    if not force and not _stale():
        return LIB
    nvcc = find_nvcc()
    cmd = [nvcc] + NVCC_FLAGS + ["-shared", "-o", LIB] + [os.path.join(CSRC, s) for s in SOURCES]
    res = subprocess.run(cmd, cwd=CSRC, capture_output=True, text=True)
    if verbose or res.returncode:
        sys.stderr.write(res.stdout + res.stderr)
    if res.returncode:
        raise RuntimeError("nvcc failed building libgdrr_b200.so")
    # registers / spills / shared memory per kernel (ptxas -v): a build log, kept out of the tracked tree
    os.makedirs(os.path.join(HERE, "build"), exist_ok=True)
    with open(os.path.join(HERE, "build", "ptxas_info.txt"), "w") as f:
        f.write("$ " + " ".join(cmd) + "\n" + res.stderr)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="--verbose" in sys.argv))
