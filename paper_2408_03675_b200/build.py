"""Build libnacl_evict.so (the product: hand-written sm_100a CUDA kernels + the C ABI) in-tree.

    python -m paper_2408_03675_b200.build [--force]

Diagnostics variants of the kernels (NACL_NVCC_EXTRA="-DNACL_...") are built only with NACL_DIAGNOSTICS=1 in the
environment: some of them give wrong results by design and none of them is the product.

nvcc cross-compiles for sm_100a without a GPU.  The library is git-ignored but travels to the GPU
box with the gpurun snapshot.
"""
from __future__ import annotations

import glob
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(HERE)
CSRC = os.path.join(HERE, "csrc")
INCLUDE = os.path.join(ROOT, "include")
LIB = os.path.join(HERE, "libnacl_evict.so")

NVCC_FLAGS = [
    "-gencode", "arch=compute_100a,code=sm_100a",
    "-O3", "-std=c++17", "-lineinfo",
    "-Xcompiler", "-fPIC", "-Xcompiler", "-fvisibility=hidden",
    "-shared", "-cudart", "static",
    "--expt-relaxed-constexpr", "--extended-lambda",
]


def sources() -> list[str]:
    return sorted(glob.glob(os.path.join(CSRC, "*.cu")))


def needs_build() -> bool:
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    deps = sources() + glob.glob(os.path.join(CSRC, "*.cuh")) + glob.glob(os.path.join(CSRC, "*.inc")) + glob.glob(os.path.join(INCLUDE, "*.h"))
    return any(os.path.getmtime(p) > t for p in deps)


def build(force: bool = False, verbose: bool = False) -> str:
    if not force and not needs_build():
        return LIB
    nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
    cmd = [nvcc] + NVCC_FLAGS + ["-I", INCLUDE, "-I", CSRC]
    extra = os.environ.get("NACL_NVCC_EXTRA", "").split()
    # Diagnostics builds (-DNACL_TC_TRACE, -DNACL_TC_STAMPS, -DNACL_SEL_TRACE, -DNACL_DIAG_*, -DNACL_EPI_TRIVIAL,
    # -DNACL_FORCE_CLUSTER=n ...) add undeclared debug exports and, some of them, compute WRONG results on purpose (they
    # switch parts of a kernel off to time the rest).  They reproduce the tables under profiles/ and are never the product:
    # the build refuses them unless NACL_DIAGNOSTICS=1 says the caller knows what the resulting library is.
    if any(f.startswith("-DNACL_") for f in extra) and os.environ.get("NACL_DIAGNOSTICS") != "1":
        raise RuntimeError("NACL_NVCC_EXTRA asks for a diagnostics build of libnacl_evict.so (results may be wrong by design); "
                           "set NACL_DIAGNOSTICS=1 to build it, and rebuild without both afterwards")
    cmd += extra
    if verbose:
        cmd += ["-Xptxas", "-v"]
    cmd += ["-o", LIB + ".tmp"] + sources()
    subprocess.run(cmd, check=True, cwd=HERE)
    os.replace(LIB + ".tmp", LIB)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
