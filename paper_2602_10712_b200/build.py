"""Builds the C-ABI library ``libsrp_b200.so`` in-tree with nvcc for sm_100a.

    python -m paper_2602_10712_b200.build [--force] [--bounds-check]

``--bounds-check`` builds ``libsrp_b200_chk.so`` instead, with -DSRP_BOUNDS_CHECK: every write into a
fixed-capacity list of the trace kernels traps with a message when out of range (debug aid; load it by
setting ``paper_2602_10712_b200.binding.LIB_PATH`` before the first call).

No GPU is needed to build (nvcc cross-compiles).  The library is git-ignored but travels to the
GPU box with the working tree.
"""
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
INCLUDE = os.path.join(os.path.dirname(HERE), "include")
LIB_PATH = os.path.join(HERE, "libsrp_b200.so")
OBJ_DIR = os.path.join(HERE, "build")

ARCH = ["-gencode", "arch=compute_100a,code=sm_100a"]
COMMON = ["-O3", "-std=c++17", "-lineinfo", "-Xcompiler", "-fPIC", "-I", INCLUDE, "-I", CSRC]
# per-file extra flags: the mesh generator is evaluated in plain IEEE fp64 (no FMA contraction)
SOURCES = {
    "srp_api.cu": [],
    "mesh_gen.cu": ["--fmad=false"],
    "lbvh.cu": [],
    "bvh_sah.cu": [],
    "bvh4.cu": [],
    "escape_mask.cu": [],
    "trace.cu": [],
    "trace_perray.cu": [],
    "trace_beam.cu": [],
    "trace_bounce.cu": [],
    "trace_small.cu": [],
    "trace_sample.cu": [],
    "trace_thermal.cu": [],
}


def _nvcc():
    for cand in (os.environ.get("NVCC"), "/usr/local/cuda/bin/nvcc", "nvcc"):
        if cand and (os.path.isabs(cand) and os.path.exists(cand) or not os.path.isabs(cand)):
            return cand
    raise RuntimeError("nvcc not found")


def _stale(target, deps):
    if not os.path.exists(target):
        return True
    t = os.path.getmtime(target)
    return any(os.path.getmtime(d) > t for d in deps)


def build_library(force=False, verbose=False, bounds_check=False):
    """Compile csrc/*.cu -> build/*.o -> libsrp_b200.so.  Returns the library path."""
    global OBJ_DIR, LIB_PATH
    extra_all = []
    if bounds_check:
        OBJ_DIR = os.path.join(HERE, "build_chk")
        LIB_PATH = os.path.join(HERE, "libsrp_b200_chk.so")
        extra_all = ["-DSRP_BOUNDS_CHECK"]
    os.makedirs(OBJ_DIR, exist_ok=True)
    headers = [os.path.join(CSRC, "srp_internal.cuh"), os.path.join(CSRC, "trace_common.cuh"), os.path.join(CSRC, "escape_bins.cuh"), os.path.join(INCLUDE, "srp.h"), os.path.abspath(__file__)]
    nvcc = _nvcc()
    objs, procs = [], []
    for src, extra in SOURCES.items():
        s = os.path.join(CSRC, src)
        o = os.path.join(OBJ_DIR, src.replace(".cu", ".o"))
        objs.append(o)
        if force or _stale(o, [s] + headers):
            cmd = [nvcc, *ARCH, *COMMON, *extra, *extra_all, "-c", s, "-o", o]
            if verbose:
                print(" ".join(cmd))
            procs.append((src, subprocess.Popen(cmd, stdout=subprocess.PIPE, stderr=subprocess.STDOUT)))
    for src, p in procs:
        out, _ = p.communicate()
        if p.returncode != 0:
            raise RuntimeError("nvcc failed on %s:\n%s" % (src, out.decode()))
    if force or procs or _stale(LIB_PATH, objs):
        tmp = LIB_PATH + ".tmp.%d" % os.getpid()
        cmd = [nvcc, *ARCH, "-shared", "-o", tmp, *objs]
        r = subprocess.run(cmd, stdout=subprocess.PIPE, stderr=subprocess.STDOUT)
        if r.returncode != 0:
            raise RuntimeError("link failed:\n%s" % r.stdout.decode())
        os.replace(tmp, LIB_PATH)
    return LIB_PATH


if __name__ == "__main__":
    print(build_library(force="--force" in sys.argv, verbose=True, bounds_check="--bounds-check" in sys.argv))
