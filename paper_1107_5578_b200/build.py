"""Builds paper_1107_5578_b200/libcwo.so from csrc/ with nvcc for sm_100a (cross-compiles without a GPU).

    python -m paper_1107_5578_b200.build [--force] [--verbose]

One object per transform length (pass_inst.cu with -DCWO_LOGN=k) so the lengths compile in parallel.
"""
from __future__ import annotations

import concurrent.futures as cf
import hashlib
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
OBJ = os.path.join(HERE, "_build")
LIB = os.path.join(HERE, "libcwo.so")
ROOT = os.path.dirname(HERE)

NVCC_FLAGS = ["-O3", "-std=c++17", "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo",
              "--expt-relaxed-constexpr", "-Xcompiler", "-fPIC", "-I", os.path.join(ROOT, "include")]
LOGNS = list(range(5, 15))


def _sources():
    out = []
    for f in sorted(os.listdir(CSRC)):
        if f.endswith((".cu", ".cuh", ".h")):
            out.append(os.path.join(CSRC, f))
    out.append(os.path.join(ROOT, "include", "cwo.h"))
    out.append(os.path.join(ROOT, "include", "cwo_debug.h"))
    return out


def _stamp() -> str:
    h = hashlib.sha256()
    for s in _sources():
        h.update(s.encode()); h.update(open(s, "rb").read())
    h.update(" ".join(NVCC_FLAGS).encode())
    return h.hexdigest()


def _run(cmd, verbose):
    if verbose:
        print(" ".join(cmd), flush=True)
    r = subprocess.run(cmd, stdout=subprocess.PIPE, stderr=subprocess.STDOUT, text=True)
    if r.returncode != 0:
        raise RuntimeError("command failed: %s\n%s" % (" ".join(cmd), r.stdout))
    return r.stdout


def build(force: bool = False, verbose: bool = False, ptxas_v: bool = False) -> str:
    os.makedirs(OBJ, exist_ok=True)
    stamp_file = os.path.join(OBJ, "stamp")
    stamp = _stamp()
    if (not force and os.path.exists(LIB) and os.path.exists(stamp_file)
            and open(stamp_file).read() == stamp):
        return LIB
    flags = NVCC_FLAGS + (["-Xptxas", "-v"] if ptxas_v else [])
    jobs = []
    for k in LOGNS:
        o = os.path.join(OBJ, "pass_%d.o" % k)
        jobs.append((["nvcc"] + flags + ["-DCWO_LOGN=%d" % k, "-c", os.path.join(CSRC, "pass_inst.cu"), "-o", o], o))
    for name in ("tables", "transpose", "outputs", "scale_static", "cwo"):
        o = os.path.join(OBJ, name + ".o")
        jobs.append((["nvcc"] + flags + ["-c", os.path.join(CSRC, name + ".cu"), "-o", o], o))
    logs = []
    with cf.ThreadPoolExecutor(max_workers=min(len(jobs), os.cpu_count() or 4)) as ex:
        for out in ex.map(lambda j: _run(j[0], verbose), jobs):
            logs.append(out)
    tmp = LIB + ".tmp%d" % os.getpid()
    _run(["nvcc", "-shared", "-gencode", "arch=compute_100a,code=sm_100a", "-o", tmp] + [j[1] for j in jobs]
         + ["-lcudart"], verbose)
    os.replace(tmp, LIB)
    open(stamp_file, "w").write(stamp)
    if ptxas_v:
        open(os.path.join(OBJ, "ptxas.log"), "w").write("\n".join(logs))
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="--verbose" in sys.argv, ptxas_v="--ptxas" in sys.argv))
