"""Build paper_2112_08926_b200/liblbm_b200.so (the C-ABI library of include/lbm.h) for sm_100a, in-tree.

    python -m paper_2112_08926_b200.build [--force] [--verbose]

One object per (velocity set, storage format) pair is compiled from csrc/lbm_unit.cu, in parallel, plus
the aux / table / API objects; they are linked into one shared library next to this file, so that the
built library travels with the repository snapshot to the GPU box.  nvcc cross-compiles without a GPU.

Flags that matter for bit-level parity with the oracle: `--fmad=false` (the only fused operations are
the explicit __fmaf_rn calls), no fast-math, `-prec-div=true`, `-ftz=false` (FP16C decoding goes through
FP32 denormals).
"""
from __future__ import annotations

import concurrent.futures as cf
import hashlib
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
OBJ = os.path.join(HERE, "build")
LIB = os.path.join(HERE, "liblbm_b200.so")
NVCC = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
ARCH = ["-gencode", "arch=compute_100a,code=sm_100a"]
FLAGS = ARCH + (["-DLBM_SELFTEST_DEBUG"] if os.environ.get("LBM_SELFTEST_DEBUG") else []) + ["-O3", "-std=c++17", "-lineinfo", "--fmad=false", "-prec-div=true", "-prec-sqrt=true", "-ftz=false",
                "-Xcompiler", "-fPIC", "-Xcompiler", "-Wall", "-Xptxas", "-v"]
VELSETS = (9, 19, 27)
FORMATS = (0, 1, 2, 3, 4, 5, 6)
FORMATS64 = (7, 8)          # FP64 arithmetic: double / float storage (csrc/lbm_unit64.cu)
HEADERS = ["lbm_codecs.cuh", "lbm_lattice.cuh", "lbm_kernels.cuh", "lbm_internal.h"]


def _jobs():
    jobs = []
    for q in VELSETS:
        for f in FORMATS:
            jobs.append((os.path.join(CSRC, "lbm_unit.cu"), os.path.join(OBJ, f"unit_q{q}_f{f}.o"), [f"-DLBM_Q={q}", f"-DLBM_F={f}"]))
    for q in VELSETS:
        for f in FORMATS64:
            jobs.append((os.path.join(CSRC, "lbm_unit64.cu"), os.path.join(OBJ, f"unit_q{q}_f{f}.o"), [f"-DLBM_Q={q}", f"-DLBM_F={f}"]))
    for name in ("lbm_aux", "lbm_units", "lbm_api"):
        jobs.append((os.path.join(CSRC, name + ".cu"), os.path.join(OBJ, name + ".o"), []))
    return jobs


def _stamp() -> str:
    h = hashlib.sha256()
    for name in sorted(os.listdir(CSRC)):
        with open(os.path.join(CSRC, name), "rb") as fh:
            h.update(name.encode() + b"\0" + fh.read())
    with open(os.path.join(os.path.dirname(HERE), "include", "lbm.h"), "rb") as fh:
        h.update(fh.read())
    h.update(" ".join(FLAGS).encode())
    return h.hexdigest()


def needs_build() -> bool:
    stamp = os.path.join(OBJ, "stamp")
    return not (os.path.exists(LIB) and os.path.exists(stamp) and open(stamp).read() == _stamp())


def _compile(job):
    src, obj, defs = job
    cmd = [NVCC] + FLAGS + defs + ["-c", src, "-o", obj]
    r = subprocess.run(cmd, capture_output=True, text=True)
    return job, r.returncode, r.stdout + r.stderr


def build(force: bool = False, verbose: bool = False) -> str:
    if not force and not needs_build():
        return LIB
    os.makedirs(OBJ, exist_ok=True)
    jobs = _jobs()
    logs = []
    with cf.ThreadPoolExecutor(max_workers=max(1, os.cpu_count() or 1)) as ex:
        for job, rc, out in ex.map(_compile, jobs):
            logs.append(f"==== {os.path.basename(job[1])}\n{out}")
            if rc != 0:
                sys.stderr.write(out)
                raise RuntimeError(f"nvcc failed on {job[0]} {job[2]}")
    with open(os.path.join(OBJ, "ptxas.log"), "w") as fh:
        fh.write("\n".join(logs))
    if verbose:
        print("\n".join(logs))
    cmd = [NVCC] + ARCH + ["-shared", "-o", LIB] + [j[1] for j in jobs] + ["-lcudart_static", "-lpthread", "-ldl", "-lrt"]
    subprocess.run(cmd, check=True)
    with open(os.path.join(OBJ, "stamp"), "w") as fh:
        fh.write(_stamp())
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="--verbose" in sys.argv))
