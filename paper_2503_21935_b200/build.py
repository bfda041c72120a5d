"""Build step: generate the per-process sources and compile libme_b200.so for sm_100a (in-tree).

    python -m paper_2503_21935_b200.build [--force] [--only gg_ttgg,...] [--verbose]

nvcc cross-compiles without a GPU.  One translation unit per (process, precision) is compiled in parallel.
"""
from __future__ import annotations

import argparse
import hashlib
import os
import subprocess
import sys
from concurrent.futures import ThreadPoolExecutor

from .codegen.generate import GROUP_LAYOUT, generate_all

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
OBJ = os.path.join(HERE, "build")
LIB = os.path.join(HERE, "libme_b200.so")

PROCS = ["ee_mumu", "gg_tt", "gg_ttg", "gg_ttgg", "gg_ttggg", "gux_taptamux", "gux_taptamgux", "gux_taptamggux"]
DIAG_PROCS = ["gg_tt", "gg_ttg", "gg_ttgg", "gg_ttggg"]   # multichannel (diagram-by-diagram) kernels
NVCC_BASE = ["nvcc", "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17",
             "--expt-relaxed-constexpr", "--extended-lambda", "-Xcompiler", "-fPIC", "-Xptxas", "-v"]

# launch configuration per (process, precision): threads per block, min blocks per SM (register cap)
TUNE = {
    # lane-group pipeline: the amplitude kernel runs one warp per block; min blocks/SM caps its registers
    # (gg_ttgg fp32: 18 -> 95 registers, 19 resident warps (shared memory), +4 % over 16; fp64 / mixed: 9 forces 168
    # registers with spills, -17 %)
    ("gg_ttggg", 0): (32, 9), ("gg_ttggg", 1): (32, 16), ("gg_ttggg", 2): (32, 9),
    ("gg_ttgg", 0): (32, 8), ("gg_ttgg", 1): (32, 18), ("gg_ttgg", 2): (32, 8),
}
DEFAULT_TUNE = (128, 1)
# lane-group units whose colour kernel runs on the amplitude kernel's own stream rather than on the high-priority one
# (round 3, 262144 / 2^20 events: gg_ttggg fp64 242.2 -> 239.9 ms, gg_ttgg fp32 22.85 -> 22.61 ms; gg_ttgg fp64 loses
# 9 % (47.3 -> 52.0 ms) and gg_ttggg fp32 gains 0.3 %, so they keep the high-priority stream; mixed not measured)
K2_SAME_STREAM = {("gg_ttggg", 0), ("gg_ttgg", 1)}
# extra nvcc flags for experiments, e.g. ME_B200_NVCC_FLAGS="-DME_UNROLL_T=2" (part of the units' hashes)
# for the units whose name starts with one of ME_B200_NVCC_UNITS (comma separated; default: all)
EXTRA = os.environ.get("ME_B200_NVCC_FLAGS", "").split()
EXTRA_UNITS = [u for u in os.environ.get("ME_B200_NVCC_UNITS", "").split(",") if u]


def _extra(name):
    return EXTRA if (not EXTRA_UNITS or any(name.startswith(u) for u in EXTRA_UNITS)) else []


def _units():
    for p in PROCS:
        for prec in (0, 1, 2):
            nt, minb = TUNE.get((p, prec), DEFAULT_TUNE)
            defs = [f"-DME_PROC={p}", f"-DME_PROC_UP={p.upper()}", f"-DME_PREC={prec}", f"-DME_NT={nt}", f"-DME_MINB={minb}"]
            if p == "ee_mumu":
                defs.append("-DME_IS_EE_MUMU")
            if p == "gg_ttg" and prec != 1:
                # complex Minkowski products as product + subtraction: with the all-FMA form this unit spills 130 bytes
                # more per thread and runs 13 % slower (measured); every other unit gains from the FMA form
                defs.append("-DME_MDOT_FMA=0")
            if (p, prec) in K2_SAME_STREAM:
                defs.append("-DME_K2_SAME_STREAM")
            src = "me_proc_group.cu" if p in GROUP_LAYOUT else "me_proc.cu"
            yield f"{p}_p{prec}", os.path.join(CSRC, src), defs
    for p in DIAG_PROCS:
        yield f"{p}_diag", os.path.join(CSRC, "me_proc_diag.cu"), [f"-DME_PROC={p}"]
    yield "api", os.path.join(CSRC, "me_api.cu"), []
    yield "peak", os.path.join(CSRC, "me_peak.cu"), []
    yield "rambo", os.path.join(CSRC, "me_rambo.cu"), []
    # me_compute_noalloc: the gg_ttg fp64 kernel with its scratch in a static device array (flags of the gg_ttg_p0 unit)
    yield "noalloc", os.path.join(CSRC, "me_noalloc.cu"), ["-DME_PROC=gg_ttg", "-DME_MDOT_FMA=0"]


def _deps_hash(defs, extra=()):
    h = hashlib.sha256()
    for root, _, files in sorted(os.walk(CSRC)):
        for f in sorted(files):
            if f.endswith((".cu", ".cuh", ".h")):
                # a unit depends on the shared headers and on its own generated header only
                if f.startswith(("proc_", "grp_", "cmat_", "diag_")) and not any(
                        f in (f"proc_{d.split('=')[1]}.cuh", f"grp_{d.split('=')[1]}.cuh", f"cmat_{d.split('=')[1]}.h",
                              f"diag_{d.split('=')[1]}.cuh")
                        for d in defs if d.startswith("-DME_PROC=")):
                    continue
                if f == "me_tables.h" and defs:
                    continue
                with open(os.path.join(root, f), "rb") as fh:
                    h.update(f.encode() + fh.read())
    with open(os.path.join(os.path.dirname(HERE), "include", "me_b200.h"), "rb") as fh:
        h.update(fh.read())
    h.update(" ".join(NVCC_BASE + defs + list(extra)).encode())
    return h.hexdigest()


def _compile(unit, force, verbose):
    name, src, defs = unit
    obj = os.path.join(OBJ, name + ".o")
    stamp = obj + ".hash"
    want = _deps_hash(defs, _extra(name))
    if not force and os.path.exists(obj) and os.path.exists(stamp) and open(stamp).read() == want:
        return name, "cached", ""
    cmd = NVCC_BASE + defs + _extra(name) + ["-c", src, "-o", obj]
    r = subprocess.run(cmd, capture_output=True, text=True)
    log = r.stdout + r.stderr
    with open(os.path.join(OBJ, name + ".ptxas.txt"), "w") as f:
        f.write(" ".join(cmd) + "\n" + log)
    if r.returncode != 0:
        raise RuntimeError(f"nvcc failed for {name}:\n{log[-4000:]}")
    with open(stamp, "w") as f:
        f.write(want)
    return name, "built", log if verbose else ""


def build(force=False, only=None, verbose=False, jobs=None) -> str:
    generate_all()
    os.makedirs(OBJ, exist_ok=True)
    units = [u for u in _units() if not only or u[0] == "api" or any(u[0].startswith(o + "_p") for o in only)]
    if only:  # the library always needs every unit: build the rest too, after the requested ones
        units += [u for u in _units() if u not in units]
    jobs = jobs or max(1, min(len(units), os.cpu_count() or 1))
    with ThreadPoolExecutor(jobs) as ex:
        for name, what, log in ex.map(lambda u: _compile(u, force, verbose), units):
            if verbose:
                print(f"[build] {name}: {what}", file=sys.stderr)
                if log:
                    print(log, file=sys.stderr)
    objs = [os.path.join(OBJ, u[0] + ".o") for u in _units()]
    if force or not os.path.exists(LIB) or any(os.path.getmtime(o) > os.path.getmtime(LIB) for o in objs):
        tmp = LIB + ".tmp%d" % os.getpid()
        cmd = ["nvcc", "-gencode", "arch=compute_100a,code=sm_100a", "-shared", "-o", tmp] + objs + ["-lcudart"]
        subprocess.check_call(cmd)
        os.replace(tmp, LIB)
    return LIB


if __name__ == "__main__":
    ap = argparse.ArgumentParser()
    ap.add_argument("--force", action="store_true")
    ap.add_argument("--only", default="")
    ap.add_argument("--verbose", action="store_true")
    ap.add_argument("--jobs", type=int, default=0)
    a = ap.parse_args()
    print(build(a.force, [x for x in a.only.split(",") if x] or None, a.verbose, a.jobs or None))
