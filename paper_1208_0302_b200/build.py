"""Builds paper_1208_0302_b200/libme_b200.so (the C-ABI library of include/me.h) with nvcc for sm_100a.

`python -m paper_1208_0302_b200.build [--force] [-v]`.  Translation units compile in parallel; the library is built
in-tree so that it travels to the GPU box.
"""
import os
import subprocess
import sys
from concurrent.futures import ThreadPoolExecutor

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
OBJ = os.path.join(HERE, "build")
LIB = os.path.join(HERE, "libme_b200.so")
SOURCES = ["me_api.cu", "me_kernels.cu", "me_probe.cu"] + ["me_inst_%d_%s_%d.cu" % (nl, t, m) for m in (9, 11) for nl in (2, 1, 4) for t in ("t", "g")]
HEADERS = ["me_device.cuh", "me_inst.cuh", "me_launch.h", "faddeeva_table.h", os.path.join("..", "..", "include", "me.h")]
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17", "-Xptxas=-v",
              "-Xcompiler", "-fPIC"]


def needs_build():
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    return any(os.path.getmtime(os.path.join(CSRC, d)) > t for d in SOURCES + HEADERS)


def build(force=False, verbose=False):
    if not force and not needs_build():
        return LIB
    nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
    os.makedirs(OBJ, exist_ok=True)

    def compile_one(src):
        obj = os.path.join(OBJ, src.replace(".cu", ".o"))
        r = subprocess.run([nvcc] + NVCC_FLAGS + ["-c", "-o", obj, os.path.join(CSRC, src)], capture_output=True, text=True)
        return src, obj, r

    with ThreadPoolExecutor(max_workers=min(8, os.cpu_count() or 1)) as ex:
        results = list(ex.map(compile_one, SOURCES))
    log = "".join(r.stdout + r.stderr for _, _, r in results)
    with open(os.path.join(OBJ, "nvcc.log"), "w") as fh:
        fh.write(log)
    if verbose or any(r.returncode for _, _, r in results):
        sys.stderr.write(log)
    if any(r.returncode for _, _, r in results):
        raise RuntimeError("nvcc failed building libme_b200.so")
    r = subprocess.run([nvcc, "-gencode", "arch=compute_100a,code=sm_100a", "-shared", "-o", LIB] + [o for _, o, _ in results],
                       capture_output=True, text=True)
    if r.returncode != 0:
        sys.stderr.write(r.stdout + r.stderr)
        raise RuntimeError("nvcc failed linking libme_b200.so")
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
