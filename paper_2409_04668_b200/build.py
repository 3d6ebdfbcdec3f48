"""Build libmcdc.so (the C-ABI CUDA library) in-tree with nvcc for sm_100a.

The host file and the four k_warp instantiation units (one per VARIANT) are compiled in parallel and linked into one
shared library; objects go to csrc/_obj (git-ignored)."""
from __future__ import annotations

import os
import subprocess
import sys
from concurrent.futures import ThreadPoolExecutor

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
OBJ = os.path.join(CSRC, "_obj")
LIB = os.path.join(HERE, "libmcdc.so")
# (source, object name, extra defines)
UNITS = [("mcdc_host.cu", "mcdc_host.o", []), ("mcdc_lattice.cu", "mcdc_lattice.o", [])] + \
        [("mcdc_warp_inst.cu", f"mcdc_warp_v{v}.o", [f"-DMCDC_WARP_VARIANT={v}"]) for v in range(4)]
HEADERS = ["mcdc_types.h", "mcdc_device.cuh", "mcdc_step.cuh", "mcdc_kernels.cuh", "mcdc_warp.cuh", "mcdc_warp_inst.cuh"]

ARCH = ["-gencode", "arch=compute_100a,code=sm_100a"]
NVCC_FLAGS = ARCH + ["-O3", "-lineinfo", "-std=c++17", "--compiler-options", "-fPIC"]
LINK_FLAGS = ARCH + ["-shared", "-cudart", "static", "--compiler-options", "-fPIC"]


def kernel_rev() -> str:
    """First 12 hex digits of the SHA-1 over the kernel sources (headers + instantiation unit): the library reports it
    through mcdc_kernel_info_get, and profiles/ncu_constants.json records the revision each capture was made from."""
    import hashlib
    h = hashlib.sha1()
    for f in HEADERS + ["mcdc_warp_inst.cu"]:
        with open(os.path.join(CSRC, f), "rb") as fh:
            h.update(fh.read())
    return h.hexdigest()[:12]


def lib_path() -> str:
    return LIB


def _stale() -> bool:
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    deps = [os.path.join(CSRC, f) for f in sorted(set(u[0] for u in UNITS)) + HEADERS]
    deps.append(os.path.join(os.path.dirname(HERE), "include", "mcdc.h"))
    return any(os.path.getmtime(d) > t for d in deps)


def build(force: bool = False, verbose: bool = False, defines=()) -> str:
    """defines: extra -D flags for tuning builds (e.g. ["-DMCDC_WARP_THREADS=576"])."""
    if not force and not _stale() and not defines:
        return LIB
    nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
    os.makedirs(OBJ, exist_ok=True)
    rev = [f'-DMCDC_KERNEL_REV="{kernel_rev()}"']

    def compile_unit(u):
        src, obj, defs = u
        cmd = [nvcc] + NVCC_FLAGS + (["-Xptxas", "-v"] if verbose else []) + list(defs) + rev + list(defines) + \
              ["-c", os.path.join(CSRC, src), "-o", os.path.join(OBJ, obj)]
        r = subprocess.run(cmd, cwd=CSRC, capture_output=True, text=True)
        return u, r

    with ThreadPoolExecutor(max_workers=len(UNITS)) as ex:
        results = list(ex.map(compile_unit, UNITS))
    for u, r in results:
        if verbose or r.returncode != 0:
            sys.stderr.write(r.stdout + r.stderr)
        if r.returncode != 0:
            raise subprocess.CalledProcessError(r.returncode, f"nvcc {u[0]} {' '.join(u[2])}")
    subprocess.check_call([nvcc] + LINK_FLAGS + ["-o", LIB] + [os.path.join(OBJ, u[1]) for u in UNITS], cwd=CSRC)
    return LIB


if __name__ == "__main__":
    defs = [a for a in sys.argv[1:] if a.startswith("-D")]
    print(build(force="--force" in sys.argv or bool(defs), verbose="-v" in sys.argv, defines=defs))
