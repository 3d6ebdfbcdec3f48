"""Build libmcdc.so (the C-ABI CUDA library) in-tree with nvcc for sm_100a.

The host file and the four k_warp instantiation units (one per VARIANT) are compiled in parallel and linked into one
shared library; objects go to csrc/_obj (git-ignored).

A tuning build (extra -D defines) never touches that library: it goes to libmcdc_tuned.so with its objects in
csrc/_obj_tuned, and is used only by a process that sets MCDC_LIB_PATH to it.  The default library therefore always
is the default configuration, and the revision it reports covers everything that shapes a launch: the kernel headers,
the instantiation unit, the host file (pool, reserve and grid plans) and the defines."""
from __future__ import annotations

import os
import subprocess
import sys
from concurrent.futures import ThreadPoolExecutor

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
OBJ = os.path.join(CSRC, "_obj")
LIB = os.path.join(HERE, "libmcdc.so")
OBJ_TUNED = os.path.join(CSRC, "_obj_tuned")
LIB_TUNED = os.path.join(HERE, "libmcdc_tuned.so")
# (source, object name, extra defines)
UNITS = [("mcdc_host.cu", "mcdc_host.o", []), ("mcdc_lattice.cu", "mcdc_lattice.o", [])] + \
        [("mcdc_warp_inst.cu", f"mcdc_warp_v{v}.o", [f"-DMCDC_WARP_VARIANT={v}"]) for v in range(4)]
HEADERS = ["mcdc_types.h", "mcdc_device.cuh", "mcdc_step.cuh", "mcdc_kernels.cuh", "mcdc_warp.cuh", "mcdc_warp_inst.cuh"]

ARCH = ["-gencode", "arch=compute_100a,code=sm_100a"]
NVCC_FLAGS = ARCH + ["-O3", "-lineinfo", "-std=c++17", "--compiler-options", "-fPIC"]
LINK_FLAGS = ARCH + ["-shared", "-cudart", "static", "--compiler-options", "-fPIC"]


def kernel_rev(defines=()) -> str:
    """First 12 hex digits of the SHA-1 over what decides a launch: the kernel headers, the instantiation unit, the host
    file (it holds the pool / reserve / grid plan) and the sorted -D defines of a tuning build.  The library reports it
    through mcdc_kernel_info_get, and profiles/ncu_constants.json records the revision each capture was made from."""
    import hashlib
    h = hashlib.sha1()
    for f in HEADERS + ["mcdc_warp_inst.cu", "mcdc_host.cu"]:
        with open(os.path.join(CSRC, f), "rb") as fh:
            h.update(fh.read())
    for d in sorted(defines):
        h.update(b"\0" + d.encode())
    return h.hexdigest()[:12]


def lib_path() -> str:
    return LIB


def _stale() -> bool:
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    deps = [os.path.join(CSRC, f) for f in sorted(set(u[0] for u in UNITS)) + HEADERS]
    deps.append(os.path.join(os.path.dirname(HERE), "include", "mcdc.h"))
    deps.append(os.path.abspath(__file__))                  # flags and the revision recipe live here
    return any(os.path.getmtime(d) > t for d in deps)


def build(force: bool = False, verbose: bool = False, defines=()) -> str:
    """defines: extra -D flags for a tuning build (e.g. ["-DMCDC_WARP_THREADS=576"]): built into libmcdc_tuned.so /
    csrc/_obj_tuned, never over the default library; returns the path of what was built."""
    defines = list(defines)
    if not force and not _stale() and not defines:
        return LIB
    nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
    obj_dir, lib = (OBJ_TUNED, LIB_TUNED) if defines else (OBJ, LIB)
    os.makedirs(obj_dir, exist_ok=True)
    rev = [f'-DMCDC_KERNEL_REV="{kernel_rev(defines)}"']

    def compile_unit(u):
        src, obj, defs = u
        cmd = [nvcc] + NVCC_FLAGS + (["-Xptxas", "-v"] if verbose else []) + list(defs) + rev + list(defines) + \
              ["-c", os.path.join(CSRC, src), "-o", os.path.join(obj_dir, obj)]
        r = subprocess.run(cmd, cwd=CSRC, capture_output=True, text=True)
        return u, r

    with ThreadPoolExecutor(max_workers=len(UNITS)) as ex:
        results = list(ex.map(compile_unit, UNITS))
    for u, r in results:
        if verbose or r.returncode != 0:
            sys.stderr.write(r.stdout + r.stderr)
        if r.returncode != 0:
            raise subprocess.CalledProcessError(r.returncode, f"nvcc {u[0]} {' '.join(u[2])}")
    subprocess.check_call([nvcc] + LINK_FLAGS + ["-o", lib] + [os.path.join(obj_dir, u[1]) for u in UNITS], cwd=CSRC)
    return lib


if __name__ == "__main__":
    defs = [a for a in sys.argv[1:] if a.startswith("-D")]
    print(build(force="--force" in sys.argv or bool(defs), verbose="-v" in sys.argv, defines=defs))
