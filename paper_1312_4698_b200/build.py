"""Build libsc_ivr.so (the C-ABI CUDA library) in-tree with nvcc for sm_100a.

    python -m paper_1312_4698_b200.build [--force]

nvcc cross-compiles without a GPU.  The .so is git-ignored but travels to the GPU box with gpurun.
"""
from __future__ import annotations

import os
import subprocess
import sys
from concurrent.futures import ThreadPoolExecutor

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libsc_ivr.so")
SOURCES = ["api.cu", "propagate_cml.cu", "propagate_tpt.cu", "spectrum.cu", "chirp.cu", "fourier_static.cu"]
HEADERS = [os.path.join(CSRC, "common.cuh"), os.path.join(CSRC, "tmem_ldst.cuh"), os.path.join(CSRC, "cml_table.h"),
           os.path.join(HERE, "..", "include", "sc_ivr.h")]


def cml_table():
    """(F, L) rows of csrc/cml_table.h: propagate_cml.cu is compiled once per row (-DSCI_CML_INST_F, -DSCI_CML_INST_L)."""
    import re
    with open(os.path.join(CSRC, "cml_table.h")) as f:
        line = [ln for ln in f if ln.startswith("#define SCI_CML_FOR_EACH")][0]
    return [(int(a), int(b)) for a, b in re.findall(r"X\((\d+),\s*(\d+)\)", line)]
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-std=c++17", "-lineinfo",
              "-Xcompiler", "-fPIC"]


def _nvcc() -> str:
    for cand in (os.environ.get("NVCC"), "/usr/local/cuda/bin/nvcc", "nvcc"):
        if cand and (os.path.sep not in cand or os.path.exists(cand)):
            return cand
    return "nvcc"


def _stale(target: str, deps) -> bool:
    if not os.path.exists(target):
        return True
    t = os.path.getmtime(target)
    return any(os.path.getmtime(d) > t for d in deps)


def build(force: bool = False, verbose: bool = False) -> str:
    objdir = os.path.join(HERE, "build")
    os.makedirs(objdir, exist_ok=True)
    nvcc = _nvcc()
    jobs = []
    units = [(src, src.replace(".cu", ".o"), []) for src in SOURCES]
    units += [("propagate_cml.cu", f"propagate_cml_f{f}.o", [f"-DSCI_CML_INST_F={f}", f"-DSCI_CML_INST_L={l}"]) for f, l in cml_table()]
    for src, obj, flags in units:
        s = os.path.join(CSRC, src)
        o = os.path.join(objdir, obj)
        if force or _stale(o, [s] + HEADERS):
            jobs.append([nvcc] + NVCC_FLAGS + flags + (["-Xptxas", "-v"] if verbose else []) + ["-c", s, "-o", o])

    def run(cmd):
        r = subprocess.run(cmd, capture_output=True, text=True)
        if r.returncode != 0:
            raise RuntimeError("nvcc failed:\n" + " ".join(cmd) + "\n" + r.stdout + r.stderr)
        return r.stderr

    if jobs:
        with ThreadPoolExecutor(max_workers=min(len(jobs), os.cpu_count() or 4)) as ex:
            for out in ex.map(run, jobs):
                if verbose:
                    sys.stderr.write(out)
    objs = [os.path.join(objdir, obj) for _, obj, _ in units]
    if force or jobs or _stale(LIB, objs):
        run([nvcc, "-shared", "-o", LIB] + objs)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
