"""Builds paper_2509_25347_b200/libdg.so (the C-ABI library of include/dg.h) in-tree with nvcc for sm_100a.

    python -m paper_2509_25347_b200.build [--force] [--verbose]

One object per translation unit, compiled in parallel: dg_kernels.cu, dg_wpc_kernels.cu, dg_paper_kernels.cu and
dg_f32_kernels.cu once per species count N (-DDG_N=<N>), dg_ppc_kernels.cu once per even number of dust slots
(-DDG_NP=<NP>), dg_tps_kernels.cu once per N <= 12 in double and once in single precision (-DDG_TPS_F32), plus dg_api.cu,
dg_peaks.cu, dg_host.cu, dg_host_static.cu, dg_energy.cu.  Objects are cached under csrc/build/ and rebuilt when a source or header is newer.
nvcc cross-compiles without a GPU.  Never --use_fast_math: fp64 arithmetic must stay IEEE (the kernels' own Newton
reciprocals are explicit, dg_params.cuh).  Extra nvcc flags for an experiment can be passed in DG_EXTRA_FLAGS.
"""
import argparse
import os
import subprocess
import sys
from concurrent.futures import ThreadPoolExecutor

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
OBJDIR = os.path.join(CSRC, "build")
LIB = os.path.join(HERE, "libdg.so")
INCLUDE = os.path.join(os.path.dirname(HERE), "include")
NMAX = 16
TPS_NMAX = 12  # dg_internal.h kTpsMaxN

NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17", "--fmad=true",
              "-Xcompiler", "-fPIC", "-Xptxas", "-v"]


def _nvcc():
    for cand in (os.environ.get("NVCC"), "/usr/local/cuda/bin/nvcc", "nvcc"):
        if cand and (os.path.isabs(cand) and os.path.exists(cand) or not os.path.isabs(cand)):
            return cand
    raise RuntimeError("nvcc not found")


def _units():
    """(object name, source, extra flags)"""
    units = [("dg_api.o", "dg_api.cu", []), ("dg_peaks.o", "dg_peaks.cu", []), ("dg_host.o", "dg_host.cu", []),
             ("dg_energy.o", "dg_energy.cu", []), ("dg_host_static.o", "dg_host_static.cu", [])]
    for n in range(1, NMAX + 1):
        units.append((f"dg_kernels_N{n}.o", "dg_kernels.cu", [f"-DDG_N={n}"]))
        units.append((f"dg_wpc_kernels_N{n}.o", "dg_wpc_kernels.cu", [f"-DDG_N={n}"]))
        units.append((f"dg_paper_kernels_N{n}.o", "dg_paper_kernels.cu", [f"-DDG_N={n}"]))
        units.append((f"dg_f32_kernels_N{n}.o", "dg_f32_kernels.cu", [f"-DDG_N={n}"]))
    for n in range(1, TPS_NMAX + 1):
        units.append((f"dg_tps_kernels_N{n}.o", "dg_tps_kernels.cu", [f"-DDG_N={n}"]))
        units.append((f"dg_tps_f32_kernels_N{n}.o", "dg_tps_kernels.cu", [f"-DDG_N={n}", "-DDG_TPS_F32"]))
    for np_ in range(2, NMAX + 1, 2):
        units.append((f"dg_ppc_kernels_NP{np_}.o", "dg_ppc_kernels.cu", [f"-DDG_NP={np_}"]))
    return units


def _newest_dep():
    deps = [os.path.join(CSRC, f) for f in os.listdir(CSRC) if f.endswith((".cu", ".cuh", ".h"))]
    deps += [os.path.join(INCLUDE, "dg.h"), os.path.abspath(__file__)]
    return max(os.path.getmtime(d) for d in deps)


def build(force: bool = False, verbose: bool = False) -> str:
    newest = _newest_dep()
    if not force and os.path.exists(LIB) and os.path.getmtime(LIB) >= newest:
        return LIB  # up to date (the objects need not exist: only libdg.so travels to the GPU box)
    os.makedirs(OBJDIR, exist_ok=True)
    nvcc = _nvcc()
    todo = []
    objs = []
    for obj, src, extra in _units():
        objp = os.path.join(OBJDIR, obj)
        objs.append(objp)
        if force or not os.path.exists(objp) or os.path.getmtime(objp) < newest:
            todo.append((objp, os.path.join(CSRC, src), extra))

    def compile_one(job):
        objp, src, extra = job
        cmd = [nvcc] + NVCC_FLAGS + extra + os.environ.get("DG_EXTRA_FLAGS", "").split() + ["-c", src, "-o", objp]
        r = subprocess.run(cmd, capture_output=True, text=True)
        log = r.stdout + r.stderr
        with open(objp[:-2] + ".ptxas.log", "w") as f:
            f.write(" ".join(cmd) + "\n" + log)
        if r.returncode != 0:
            raise RuntimeError(f"nvcc failed for {os.path.basename(objp)}:\n{log}")
        return objp, log

    if todo:
        with ThreadPoolExecutor(max_workers=min(len(todo), os.cpu_count() or 4)) as ex:
            for objp, log in ex.map(compile_one, todo):
                if verbose:
                    print(f"== {os.path.basename(objp)}\n{log}")
    if todo or force or not os.path.exists(LIB):
        cmd = [nvcc, "-shared", "-o", LIB + ".tmp"] + objs
        r = subprocess.run(cmd, capture_output=True, text=True)
        if r.returncode != 0:
            raise RuntimeError("link failed:\n" + r.stdout + r.stderr)
        os.replace(LIB + ".tmp", LIB)
    return LIB


if __name__ == "__main__":
    ap = argparse.ArgumentParser()
    ap.add_argument("--force", action="store_true")
    ap.add_argument("--verbose", action="store_true")
    a = ap.parse_args()
    print(build(force=a.force, verbose=a.verbose))
    sys.exit(0)
