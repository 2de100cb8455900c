"""Build the sm_100a SLDG library in-tree: paper_2110_14557_b200/libsldg_b200.so.

nvcc cross-compiles without a GPU.  -lineinfo so ncu's source page maps to csrc/; static cudart so the
library loads (and exports its symbols) on a box without a CUDA driver.
"""
import os
import subprocess
import sys
from concurrent.futures import ThreadPoolExecutor

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libsldg_b200.so")
SOURCES = ["sldg_api.cu", "sldg_sweep_walk.cu", "sldg_sweep_tma.cu", "sldg_sweep_line.cu", "sldg_sweep_fused.cu", "sldg_sweep_fused_cell.cu", "sldg_sweep_fused3.cu", "sldg_sweep_fused3d.cu", "sldg_sweep_fusedv.cu", "sldg_sweep_fusedv3.cu", "sldg_field.cu", "sldg_density_static.cu", "sldg_cgdg.cu", "sldg_tables.cpp"]
DUAL = ["sldg_sweep_walk.cu", "sldg_sweep_line.cu", "sldg_sweep_fused_cell.cu", "sldg_sweep_fused3.cu", "sldg_sweep_fused3d.cu", "sldg_sweep_fusedv.cu", "sldg_sweep_fusedv3.cu"]
HEADERS = [os.path.join(CSRC, "sldg_real.h"), os.path.join(CSRC, "sldg_internal.h"), os.path.join(CSRC, "sldg_async.h"), os.path.join(CSRC, "sldg_tmap.h"), os.path.join(HERE, "..", "include", "sldg.h")]
NVCC = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
FLAGS = ["-O3", "-std=c++17", "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo",
         "-Xcompiler", "-fPIC,-ffp-contract=off", "-cudart", "static"]


def _stale(target, deps):
    if not os.path.exists(target):
        return True
    t = os.path.getmtime(target)
    return any(os.path.getmtime(d) > t for d in deps)


def build(force=False, verbose=False):
    objs, jobs = [], []
    extra = ["-Xptxas", "-v"] if verbose else []
    for s in SOURCES:
        src = os.path.join(CSRC, s)
        obj = os.path.join(CSRC, os.path.splitext(s)[0] + ".o")
        if force or _stale(obj, [src] + HEADERS):
            jobs.append([NVCC] + FLAGS + extra + ["-c", src, "-o", obj])
        objs.append(obj)
        if s in DUAL:          # second compilation: real = float (single precision mode, sldg_real.h)
            obj32 = os.path.join(CSRC, os.path.splitext(s)[0] + "_f32.o")
            if force or _stale(obj32, [src] + HEADERS):
                jobs.append([NVCC] + FLAGS + extra + ["-DSLDG_REAL_FLOAT", "-c", src, "-o", obj32])
            objs.append(obj32)
    # the translation units are independent: compile them side by side
    with ThreadPoolExecutor(max_workers=max(1, min(len(jobs), os.cpu_count() or 1))) as pool:
        for rc in pool.map(lambda cmd: subprocess.run(cmd, capture_output=not verbose, text=True), jobs):
            if rc.returncode != 0:
                sys.stderr.write((rc.stdout or "") + (rc.stderr or ""))
                raise subprocess.CalledProcessError(rc.returncode, rc.args)
    if force or _stale(LIB, objs):
        subprocess.check_call([NVCC, "-shared", "-cudart", "static", "-gencode", "arch=compute_100a,code=sm_100a", "-o", LIB] + objs)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
