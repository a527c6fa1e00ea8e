"""Builds paper_2110_00853_b200/libcm_dg.so in-tree with nvcc for sm_100a (cross-compiles without a GPU).

One object per polynomial order (the kernel templates are instantiated per order) so the build
parallelises; sources under csrc/, public header under include/.
"""
import os
import subprocess
import sys
from concurrent.futures import ThreadPoolExecutor

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
OBJ = os.path.join(HERE, "build")
LIB = os.path.join(HERE, "libcm_dg.so")
NQS = (3, 4, 5, 6, 7, 8)
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17",
              "-Xcompiler", "-fPIC", "-Xptxas", "-v"]


def _sources():
    return [os.path.join(CSRC, f) for f in sorted(os.listdir(CSRC))] + \
           [os.path.join(os.path.dirname(HERE), "include", "cm_dg.h")]


def _stale(target):
    if not os.path.exists(target):
        return True
    t = os.path.getmtime(target)
    return any(os.path.getmtime(s) > t for s in _sources())


def _run(cmd, log):
    r = subprocess.run(cmd, stdout=subprocess.PIPE, stderr=subprocess.STDOUT, text=True)
    with open(log, "w") as f:
        f.write(" ".join(cmd) + "\n" + r.stdout)
    if r.returncode != 0:
        raise RuntimeError("nvcc failed:\n" + " ".join(cmd) + "\n" + r.stdout[-4000:])


def build(force=False, verbose=False):
    """CM_DG_NVCC_EXTRA (extra nvcc flags, e.g. tuning macros) and CM_DG_LIB_OUT (output path) serve kernel experiments."""
    nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
    extra = os.environ.get("CM_DG_NVCC_EXTRA", "").split()
    LIB = os.environ.get("CM_DG_LIB_OUT", globals()["LIB"])
    if extra and LIB == globals()["LIB"]:
        raise RuntimeError("CM_DG_NVCC_EXTRA builds an experimental variant: set CM_DG_LIB_OUT to a path other than the "
                           "default library, which tests and bench load")
    if not force and not extra and not _stale(LIB):
        return LIB
    os.makedirs(OBJ, exist_ok=True)
    jobs = []
    for nq in NQS:
        o = os.path.join(OBJ, "kernels_nq%d.o" % nq)
        jobs.append(([nvcc] + NVCC_FLAGS + extra + ["-DCM_NQ=%d" % nq, "-c", os.path.join(CSRC, "cm_dg_kernels_inst.cu"), "-o", o],
                     os.path.join(OBJ, "kernels_nq%d.log" % nq)))
    o_lib = os.path.join(OBJ, "lib.o")
    jobs.append(([nvcc] + NVCC_FLAGS + ["-c", os.path.join(CSRC, "cm_dg_lib.cu"), "-o", o_lib], os.path.join(OBJ, "lib.log")))
    with ThreadPoolExecutor(max_workers=min(8, os.cpu_count() or 2)) as ex:
        list(ex.map(lambda j: _run(*j), jobs))
    objs = [os.path.join(OBJ, "kernels_nq%d.o" % nq) for nq in NQS] + [o_lib]
    _run([nvcc, "-shared", "-gencode", "arch=compute_100a,code=sm_100a", "-o", LIB] + objs + ["-lcudart"],
         os.path.join(OBJ, "link.log"))
    if verbose:
        print("built", LIB)
    return LIB


if __name__ == "__main__":
    build(force="--force" in sys.argv, verbose=True)
