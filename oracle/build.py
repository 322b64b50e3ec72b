"""Build the oracle (test infrastructure) with gcc: liboracle.so (FP64) and liboracle_ld.so (x87 80-bit).

Flags follow SURVEY.md sec. 8(c) R21: -O2 -ffp-contract=off (no FMA contraction, no fast-math).
"""
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "vg_oracle.c")
LIB = os.path.join(HERE, "liboracle.so")
LIB_LD = os.path.join(HERE, "liboracle_ld.so")
LIB_SAN = os.path.join(HERE, "liboracle_san.so")  # AddressSanitizer + UndefinedBehaviorSanitizer build
SAN_FLAGS = ["-O1", "-g", "-fno-omit-frame-pointer", "-fsanitize=address,undefined", "-fno-sanitize-recover=undefined",
             "-ffp-contract=off", "-fopenmp", "-fPIC", "-shared", "-std=c99", "-Wall", "-Wextra"]
CFLAGS = ["-O2", "-ffp-contract=off", "-fopenmp", "-fPIC", "-shared", "-std=c99", "-Wall", "-Wextra"]


def _stale(lib):
    return not os.path.exists(lib) or os.path.getmtime(lib) < os.path.getmtime(SRC)


def build(force=False):
    for lib, extra in ((LIB, []), (LIB_LD, ["-DORC_LONG_DOUBLE"])):
        if force or _stale(lib):
            cmd = ["gcc"] + CFLAGS + extra + [SRC, "-o", lib, "-lm"]
            subprocess.run(cmd, check=True)
    return LIB, LIB_LD


def build_sanitized(force=False):
    """The same source with ASan + UBSan.  A process that loads it must have the ASan runtime loaded first
    (LD_PRELOAD=$(gcc -print-file-name=libasan.so)); oracle/__init__.py loads it when ORACLE_SANITIZE=1."""
    if force or _stale(LIB_SAN):
        subprocess.run(["gcc"] + SAN_FLAGS + [SRC, "-o", LIB_SAN, "-lm"], check=True)
    return LIB_SAN


def asan_runtime():
    return subprocess.run(["gcc", "-print-file-name=libasan.so"], check=True, capture_output=True, text=True).stdout.strip()


if __name__ == "__main__":
    build(force="--force" in sys.argv)
    print(LIB)
    print(LIB_LD)
