"""Build step: compiles csrc/*.cu|*.cpp into paper_2502_06073_b200/liballegro_b200.so for sm_100a.

Run as ``python -m paper_2502_06073_b200.build`` (or through ``__graft_entry__.build()``).  nvcc
cross-compiles without a GPU.  The library links cudart statically and exposes only the C-ABI of
include/allegro.h.
"""
from __future__ import annotations

import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "liballegro_b200.so")
SOURCES = ["plan.cpp", "neighbor.cu", "network.cu", "tp_kernels.cu", "tp3_fwd.cu", "tp3_bwd.cu", "gemm_tc.cu", "gemm_f16s.cu", "decomp.cu", "virial_noalloc.cu", "tp_mix.cu", "md.cu", "api.cu"]
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17",
              "-Xcompiler", "-fPIC", "--expt-relaxed-constexpr", "-Xptxas", "-v" if os.environ.get("ALLEGRO_PTXAS_V") else "-O3"]
if os.environ.get("ALLEGRO_F16S_TRACE"):   # developer build: gemm_f16s.cu prints the per-tile timeline of CTA 0 after every launch
    NVCC_FLAGS.append("-DF16S_TRACE")
if os.environ.get("ALLEGRO_X_TRACE"):   # developer build: tp_mix.cu prints the wait times of CTA 0
    NVCC_FLAGS.append("-DX_TRACE"); NVCC_FLAGS.append("-DX_FEWMMA") if os.environ.get("ALLEGRO_X_FEWMMA") else None
if os.environ.get("ALLEGRO_F16S_DBGWAIT"):   # developer build: barrier waits time out and report their source line instead of trapping
    NVCC_FLAGS.append("-DF16S_DBGWAIT")


STAMP = os.path.join(HERE, "build", "flags.txt")


def _stale() -> bool:
    if not os.path.exists(LIB):
        return True
    if not os.path.exists(STAMP) or open(STAMP).read() != " ".join(NVCC_FLAGS):   # a developer build is replaced by a normal one
        return True
    t = os.path.getmtime(LIB)
    deps = [os.path.join(CSRC, f) for f in os.listdir(CSRC)] + [os.path.join(HERE, "..", "include", "allegro.h"), __file__]
    return any(os.path.getmtime(d) > t for d in deps)


def build(force: bool = False, verbose: bool = False) -> str:
    if not force and not _stale():
        return LIB
    nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
    objs = []
    procs = []
    bdir = os.path.join(HERE, "build")
    os.makedirs(bdir, exist_ok=True)
    # generated coupling code: host generator built from plan.cpp, run once -> build/tp_gen.cuh
    gen = os.path.join(bdir, "gen_tp")
    for cmd in (["g++", "-O1", "-std=c++17", os.path.join(CSRC, "gen_tp.cpp"), os.path.join(CSRC, "plan.cpp"), "-o", gen],
                [gen, os.path.join(bdir, "tp_gen.cuh")]):
        r = subprocess.run(cmd, stdout=subprocess.PIPE, stderr=subprocess.STDOUT, text=True)
        if r.returncode != 0:
            raise RuntimeError("tensor-product code generation failed:\n" + r.stdout)
    for src in SOURCES:
        obj = os.path.join(HERE, "build", src.rsplit(".", 1)[0] + ".o")
        cmd = [nvcc, *NVCC_FLAGS, "-I", bdir, "-x", "cu", "-c", os.path.join(CSRC, src), "-o", obj]
        procs.append((src, subprocess.Popen(cmd, stdout=subprocess.PIPE, stderr=subprocess.STDOUT, text=True)))
        objs.append(obj)
    for src, p in procs:
        out, _ = p.communicate()
        if p.returncode != 0:
            raise RuntimeError(f"nvcc failed on {src}:\n{out}")
        if verbose and out.strip():
            print(out)
    cmd = [nvcc, "-shared", "-o", LIB, *objs, "-gencode", "arch=compute_100a,code=sm_100a", "-Xcompiler", "-fPIC"]
    r = subprocess.run(cmd, stdout=subprocess.PIPE, stderr=subprocess.STDOUT, text=True)
    if r.returncode != 0:
        raise RuntimeError("link failed:\n" + r.stdout)
    with open(STAMP, "w") as f:
        f.write(" ".join(NVCC_FLAGS))
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose=True))
