"""Build the CPU oracle (test infrastructure; see kho.h).

    python oracle/build.py            -> oracle/libkho.so (single thread) and oracle/libkho_omp.so
    python oracle/build.py --sanitize -> also oracle/libkho_san.so (-fsanitize=address,undefined -O1 -g); the oracle tests
                                         run against it with
        KHO_SANITIZE=1 LD_PRELOAD=$(gcc -print-file-name=libasan.so):$(gcc -print-file-name=libubsan.so) \
            ASAN_OPTIONS=detect_leaks=0 python -m pytest tests -m "not gpu" -q -k oracle

Flags: -O2 -ffp-contract=off (no FMA contraction: the oracle's rounding is the plain IEEE one).
The OpenMP build only parallelises zone-independent outer loops; results are bit-identical.
"""
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))


def _stale(target, sources):
    if not os.path.exists(target):
        return True
    t = os.path.getmtime(target)
    return any(os.path.getmtime(s) > t for s in sources)


def build(verbose=False, sanitize=False):
    src = [os.path.join(HERE, "kho.cpp"), os.path.join(HERE, "kho.h")]
    base = ["g++", "-std=c++17", "-O2", "-ffp-contract=off", "-fPIC", "-shared", "-Wall", "-Wno-unused-variable"]
    outs = []
    variants = [("libkho.so", []), ("libkho_omp.so", ["-fopenmp"])]
    if sanitize:
        variants.append(("libkho_san.so", ["-O1", "-g", "-fno-omit-frame-pointer", "-fsanitize=address,undefined", "-fno-sanitize-recover=undefined"]))
    for name, extra in variants:
        out = os.path.join(HERE, name)
        if _stale(out, src):
            cmd = base + extra + ["-o", out, src[0]]
            if verbose:
                print(" ".join(cmd))
            subprocess.check_call(cmd)
        outs.append(out)
    return outs


if __name__ == "__main__":
    build(verbose=True, sanitize="--sanitize" in sys.argv)
    sys.exit(0)
