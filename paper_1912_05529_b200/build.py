"""Build libpdm.so in-tree with nvcc for sm_100a (called by __graft_entry__.build()).

The unrolled kernel families live in their own translation units (csrc/tu_*.cu) so that the
objects compile in parallel; they are linked into one shared library.
"""
from __future__ import annotations

import os
import shutil
import subprocess
from concurrent.futures import ThreadPoolExecutor

_HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(_HERE, "csrc")
LIB = os.path.join(_HERE, "libpdm.so")
OBJDIR = os.path.join(_HERE, "build")
# (source, extra defines, object name)
UNITS = [("pdm_api.cu", [], "pdm_api.o"),
         ("pdm_design.cu", [], "pdm_design.o"),
         ("pdm3_api.cu", [], "pdm3_api.o"),
         ("pdm_static.cu", [], "pdm_static.o"),
         ("tu_march.cu", ["-DPDM_TU_PART=0"], "tu_march0.o"),
         ("tu_march.cu", ["-DPDM_TU_PART=1"], "tu_march1.o"),
         ("tu_march.cu", ["-DPDM_TU_PART=2"], "tu_march2.o"),
         ("tu_asym.cu", ["-DPDM_TU_PART=0"], "tu_asym0.o"),
         ("tu_asym.cu", ["-DPDM_TU_PART=1"], "tu_asym1.o"),
         ("tu_asym.cu", ["-DPDM_TU_PART=2"], "tu_asym2.o"),
         ("tu_pack.cu", ["-DPDM_TU_PART=0"], "tu_pack0.o"),
         ("tu_pack.cu", ["-DPDM_TU_PART=1"], "tu_pack1.o"),
         ("tu_pack.cu", ["-DPDM_TU_PART=2"], "tu_pack2.o"),
         ("tu_cluster.cu", [], "tu_cluster.o"),
         ("tu_tiled.cu", [], "tu_tiled.o")]
HEADERS = ["pdm_common.cuh", "pdm_dispatch.cuh", "kern_naive.cuh", "kern_peak.cuh", "kern_march.cuh",
           "kern_tiled.cuh", "kern_tf.cuh", "kern_cluster.cuh", "kern_reduce.cuh", "kern_pack.cuh", "kern_fft.cuh", "kern_3d.cuh"]
NVCC_FLAGS = ["-std=c++17", "-O3", "-lineinfo", "-gencode", "arch=compute_100a,code=sm_100a",
              "-Xcompiler", "-fPIC"]


def _nvcc() -> str:
    for cand in (shutil.which("nvcc"), "/usr/local/cuda/bin/nvcc"):
        if cand and os.path.exists(cand):
            return cand
    raise RuntimeError("nvcc not found: libpdm.so cannot be built")


def _stale() -> bool:
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    deps = [os.path.join(CSRC, f) for f in sorted({u[0] for u in UNITS}) + HEADERS]
    deps.append(os.path.join(os.path.dirname(_HERE), "include", "pdm.h"))
    return any(os.path.getmtime(d) > t for d in deps)


def build_lib(force: bool = False, verbose: bool = False) -> str:
    """nvcc -gencode arch=compute_100a,code=sm_100a -lineinfo ... -> paper_1912_05529_b200/libpdm.so"""
    if not force and not _stale():
        return LIB
    nvcc = _nvcc()
    os.makedirs(OBJDIR, exist_ok=True)
    tag = f".tmp{os.getpid()}"

    def compile_unit(unit):
        src, defines, obj = unit
        out = os.path.join(OBJDIR, obj[:-2] + tag + ".o")
        cmd = [nvcc, *NVCC_FLAGS, *(["-Xptxas", "-v"] if verbose else []), *defines,
               "-c", "-o", out, os.path.join(CSRC, src)]
        subprocess.run(cmd, check=True)
        return out

    with ThreadPoolExecutor(max_workers=min(len(UNITS), os.cpu_count() or 1)) as pool:
        objs = list(pool.map(compile_unit, UNITS))
    tmp = LIB + tag
    try:
        subprocess.run([nvcc, "-shared", "-gencode", "arch=compute_100a,code=sm_100a", "-o", tmp, *objs],
                       check=True)
        os.replace(tmp, LIB)
    finally:
        for o in objs:
            if os.path.exists(o):
                os.remove(o)
    return LIB


if __name__ == "__main__":
    print(build_lib(force=True, verbose=True))
