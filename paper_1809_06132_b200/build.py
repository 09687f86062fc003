"""Builds libfsw.so (the C-ABI library of include/fsw.h) for sm_100a with nvcc, in-tree, and libfsw_probe.so (the
bench-only FP32-peak probe of csrc/probe_fp32_peak.cu, which is not part of the library's ABI).

    python -m paper_1809_06132_b200.build [--force]

Every translation unit is compiled with `-gencode arch=compute_100a,code=sm_100a -lineinfo`; the sweep kernel is
instantiated once per (matching-window size, view count) in its own object so the instantiations build in parallel.
"""
from __future__ import annotations

import os
import shutil
import subprocess
import sys
from concurrent.futures import ThreadPoolExecutor

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(HERE)
CSRC = os.path.join(HERE, "csrc")
INCLUDE = os.path.join(ROOT, "include")
OBJ = os.path.join(HERE, "build")
LIB = os.path.join(HERE, "libfsw.so")
PROBE_LIB = os.path.join(HERE, "libfsw_probe.so")
PROBE_SRC = os.path.join(CSRC, "probe_fp32_peak.cu")
WINDOWS = (3, 5, 7, 9, 11, 13, 15)

# -compress-all: the library holds some 350 instantiations of the sweep kernel with line information; compressed it is
# a third of the size (it travels to the GPU box with every gpurun snapshot)
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17",
              "-Xcompiler", "-fPIC", "-Xfatbin", "-compress-all", "-I" + INCLUDE, "-I" + CSRC]


def _nvcc() -> str:
    for cand in (os.environ.get("NVCC"), shutil.which("nvcc"), "/usr/local/cuda/bin/nvcc"):
        if cand and os.path.exists(cand):
            return cand
    raise RuntimeError("nvcc not found: the CUDA extension cannot be built (there is no CPU fallback)")


def _sources():
    deps = [os.path.join(CSRC, f) for f in os.listdir(CSRC) if f != os.path.basename(PROBE_SRC)]
    deps += [os.path.join(INCLUDE, "fsw.h"), os.path.abspath(__file__)]
    units = [("fsw_api.o", "fsw_api.cu", []), ("fsw_aux.o", "fsw_aux.cu", []), ("fsw_tsdf.o", "fsw_tsdf.cu", []),
             ("fsw_sweep_dispatch.o", "fsw_sweep_dispatch.cu", [])]
    # one object per (window, view count): views 1..4 unrolled (3 and 4 only where two views share a pass, i.e. for
    # windows up to 9), 0 = the run-time view loop; the heaviest objects first
    for n in (4, 3, 0, 2, 1):
        for w in WINDOWS:
            if n in (3, 4) and w > 9:
                continue
            units.append(("fsw_sweep_w%d_v%d.o" % (w, n), "fsw_sweep_inst.cu", ["-DFSW_WIN=%d" % w, "-DFSW_NVT=%d" % n]))
    return deps, units


def build(force: bool = False, verbose: bool = False) -> str:
    deps, units = _sources()
    newest = max(os.path.getmtime(p) for p in deps)
    if not force and os.path.exists(LIB) and os.path.getmtime(LIB) >= newest and os.path.exists(PROBE_LIB) \
            and os.path.getmtime(PROBE_LIB) >= os.path.getmtime(PROBE_SRC):
        return LIB
    nvcc = _nvcc()
    if force or not os.path.exists(PROBE_LIB) or os.path.getmtime(PROBE_LIB) < os.path.getmtime(PROBE_SRC):
        tmp = PROBE_LIB + ".tmp.%d" % os.getpid()
        res = subprocess.run([nvcc, "-shared"] + NVCC_FLAGS + [PROBE_SRC, "-o", tmp], capture_output=True, text=True)
        if res.returncode != 0:
            raise RuntimeError("nvcc failed for the probe:\n%s\n%s" % (res.stdout, res.stderr))
        os.replace(tmp, PROBE_LIB)
    if not force and os.path.exists(LIB) and os.path.getmtime(LIB) >= newest:
        return LIB
    os.makedirs(OBJ, exist_ok=True)

    def compile_one(unit):
        obj, src, extra = unit
        out = os.path.join(OBJ, obj)
        if not force and os.path.exists(out) and os.path.getmtime(out) >= newest:
            return out
        cmd = [nvcc] + NVCC_FLAGS + extra + (["-Xptxas", "-v"] if verbose else []) + ["-c", os.path.join(CSRC, src), "-o", out]
        res = subprocess.run(cmd, capture_output=True, text=True)
        if res.returncode != 0:
            raise RuntimeError("nvcc failed for %s:\n%s\n%s" % (src, res.stdout, res.stderr))
        if verbose:
            sys.stderr.write(res.stderr)
        return out

    with ThreadPoolExecutor(max_workers=min(8, os.cpu_count() or 2)) as pool:
        objs = list(pool.map(compile_one, units))
    tmp = LIB + ".tmp.%d" % os.getpid()
    cmd = [nvcc, "-shared", "-gencode", "arch=compute_100a,code=sm_100a", "-o", tmp] + objs
    res = subprocess.run(cmd, capture_output=True, text=True)
    if res.returncode != 0:
        raise RuntimeError("link failed:\n%s\n%s" % (res.stdout, res.stderr))
    os.replace(tmp, LIB)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
