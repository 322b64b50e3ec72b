"""Build libvg.so (the C-ABI CUDA library) for sm_100a with nvcc, in-tree.

    python -m paper_1512_06637_b200.build [--force] [--verbose]

One object per translation unit (compiled in parallel), linked with the static CUDA runtime so that the
library loads (and its symbols can be inspected) on a box without a GPU.  No fast-math: FMA contraction only.
"""
import concurrent.futures as cf
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
OBJ = os.path.join(HERE, "build")
LIB = os.path.join(HERE, "libvg.so")
INCLUDE = os.path.join(os.path.dirname(HERE), "include")
UNITS = ["vg_api", "vg_host", "vg_static", "vg_nav", "vg_world", "vg_bool", "vg_boolx", "vg_csg", "vg_bool_k0", "vg_bool_k1", "vg_bool_k2", "vg_bool_k3", "vg_bool_k4", "vg_probe", "vg_k_box", "vg_k_orb", "vg_k_tube", "vg_k_cone", "vg_k_trd", "vg_k_polycone"]
NVCC = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17", "-Xcompiler", "-fPIC",
         "-Xptxas", "-v", "-I", INCLUDE]


def _deps_mtime():
    names = [f for f in os.listdir(CSRC) if f.endswith((".cuh", ".h"))] + ["../../include/vg.h"]
    return max(os.path.getmtime(os.path.join(CSRC, f)) for f in names)


def _compile(unit, force, extra):
    src = os.path.join(CSRC, unit + ".cu")
    obj = os.path.join(OBJ, unit + ".o")
    if not force and os.path.exists(obj) and os.path.getmtime(obj) >= max(os.path.getmtime(src), _deps_mtime()):
        return unit, False, ""
    cmd = [NVCC] + FLAGS + list(extra) + ["-c", src, "-o", obj]
    r = subprocess.run(cmd, capture_output=True, text=True)
    if r.returncode != 0:
        raise RuntimeError("nvcc failed for %s:\n%s\n%s" % (unit, r.stdout, r.stderr))
    with open(os.path.join(OBJ, unit + ".ptxas.log"), "w") as f:
        f.write(" ".join(cmd) + "\n" + r.stderr)
    return unit, True, r.stderr


def build(force=False, verbose=False, extra=()):
    # VG_NVCC_EXTRA="-DVG_IEEE_MATH ..." adds compile flags (tuning sweeps, bisecting a parity failure); the objects are
    # keyed by time stamp only, so combine it with force / --force
    extra = list(extra) + os.environ.get("VG_NVCC_EXTRA", "").split()
    os.makedirs(OBJ, exist_ok=True)
    with cf.ThreadPoolExecutor(max_workers=min(len(UNITS), os.cpu_count() or 4)) as ex:
        results = list(ex.map(lambda u: _compile(u, force, extra), UNITS))
    rebuilt = [u for u, did, _ in results if did]
    objs = [os.path.join(OBJ, u + ".o") for u in UNITS]
    if rebuilt or not os.path.exists(LIB):
        cmd = [NVCC, "-shared", "-gencode", "arch=compute_100a,code=sm_100a", "-cudart", "static", "-o", LIB] + objs
        r = subprocess.run(cmd, capture_output=True, text=True)
        if r.returncode != 0:
            raise RuntimeError("link failed:\n%s\n%s" % (r.stdout, r.stderr))
    if verbose:
        for u, did, log in results:
            if did:
                print("== %s\n%s" % (u, log))
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="--verbose" in sys.argv))
