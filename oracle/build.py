"""oracle/build.py — TEST INFRASTRUCTURE. Compiles the CPU oracle into oracle/liboracle.so with g++.

Run as `python -m oracle.build` or through `__graft_entry__.build()` (building the checker is not using it).
"""
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
SOURCES = ["faddeeva.cpp", "zeeman.cpp", "synth.cpp", "philox.cpp", "sobol.cpp", "ga.cpp", "uncertainty.cpp", "capi.cpp"]
LIB = os.path.join(HERE, "liboracle.so")


def needs_build():
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    deps = [os.path.join(HERE, s) for s in SOURCES] + [os.path.join(HERE, "oracle.hpp")]
    return any(os.path.getmtime(d) > t for d in deps)


def build(force=False):
    if not force and not needs_build():
        return LIB
    # -ffp-contract=off: the binary32 gene arithmetic of ga.cpp must not be fused behind our back.
    cmd = ["g++", "-std=c++17", "-O2", "-ffp-contract=off", "-fPIC", "-shared", "-pthread", "-Wall", "-Wextra",
           "-o", LIB] + [os.path.join(HERE, s) for s in SOURCES]
    subprocess.run(cmd, check=True)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv))
