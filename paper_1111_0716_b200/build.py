"""Builds libexx.so (the C-ABI CUDA library) in-tree with nvcc for sm_100a.

    python -m paper_1111_0716_b200.build [--force]

nvcc cross-compiles without a GPU.  The built library sits next to this file so that it travels with the repo.

Build knobs (supported, for tuning sweeps on a new GPU; libexx.so itself is always built without them): a variant library is
built with `build(extra=["-D..."], out="/some/libexx_variant.so")` and loaded by setting EXX_LIB to its path.
    -DEXX_TUNE_R1=<R1> with any of -DEXX_TUNE_{U1,NT1,U3,NT3,NT2,MINB1,MINB2,MINB3,TWREG,ACCREG,STAGE3}=<v>
                          launch geometry of the fused passes for the grid N = 8 R1 (FusedCfg in csrc/exx_fused_phases.h)
    -DEXX_STAGE3_ALL=<0|1|2>   cp.async staging level of pass C for every grid
    -DEXX_DUAL_RG_ALL=<0|1|2|4>  rows per CTA of the dual sweep for every grid (0 = two single sweeps)
    -DEXX_DEFAULT_TILE=<n>, -DEXX_SHARD_TILE=<n>, -DEXX_WORK_CAP_GIB=<n>   batch tiles and the pair-workspace cap (csrc/exx_internal.h)
"""
import hashlib
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libexx.so")
STAMP = LIB + ".srchash"   # hash of what LIB was built from (git-ignored like the library, travels with it)
SOURCES = ["exx_api.cu", "exx_kernels.cu", "exx_fused.cu", "exx_subspace.cu", "exx_static.cu"]
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17", "--fmad=true",
              "-Xcompiler", "-fPIC,-ffp-contract=off,-Wall,-Wno-unknown-pragmas", "-shared", "-cudart", "shared", "--threads", "4"]


def _nvcc():
    for p in (os.environ.get("NVCC"), "/usr/local/cuda/bin/nvcc", "nvcc"):
        if p and (os.path.isabs(p) and os.path.exists(p) or not os.path.isabs(p)):
            return p
    return "nvcc"


def _source_hash():
    """sha256 over the sources, the public header and the compiler flags: what the library was built from."""
    h = hashlib.sha256(" ".join(NVCC_FLAGS).encode())
    deps = sorted(os.path.join(CSRC, f) for f in os.listdir(CSRC)) + [os.path.join(os.path.dirname(HERE), "include", "exx.h")]
    for d in deps:
        h.update(os.path.basename(d).encode())
        with open(d, "rb") as f:
            h.update(f.read())
    return h.hexdigest()


def needs_build():
    """Stale iff the library is missing or was built from other sources.  Decided by content (a hash kept beside the library), not
    by modification times: a copy of the tree (e.g. onto the GPU box) does not keep them, and a needless rebuild costs ~20 s."""
    if not os.path.exists(LIB) or not os.path.exists(STAMP):
        return True
    with open(STAMP) as f:
        return f.read().strip() != _source_hash()


def build(force=False, verbose=False, extra=(), out=None):
    """Build libexx.so (or `out`, e.g. a variant compiled with extra flags; such a variant never replaces libexx.so itself)."""
    if extra and out is None and [str(x) for x in extra] != ["-Xptxas", "-v"]:   # ptxas verbosity only: it cannot change the code
        raise ValueError("build(extra=...) needs out=...: libexx.so is only ever built with the stamped flags")
    if out is None and not force and not needs_build():
        return LIB
    target = out or LIB
    tmp = target + ".tmp.%d" % os.getpid()
    cmd = [_nvcc()] + NVCC_FLAGS + list(extra) + ["-o", tmp] + [os.path.join(CSRC, s) for s in SOURCES]
    if verbose:
        print(" ".join(cmd))
    digest = _source_hash()
    subprocess.check_call(cmd)
    os.replace(tmp, target)
    if out is None:   # extra can only be ptxas verbosity here (checked above): same code
        with open(STAMP + ".tmp.%d" % os.getpid(), "w") as f:
            f.write(digest + "\n")
        os.replace(STAMP + ".tmp.%d" % os.getpid(), STAMP)
    return target


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose=True, extra=["-Xptxas", "-v"] if "-v" in sys.argv else []))
