"""Builds libcf_b200.so in-tree with nvcc for sm_100a (`python -m paper_2512_14098_b200.build`).

Every kernel family is its own translation unit; they are compiled in parallel into
`csrc/build/*.o` and linked into one shared library. `cf_k32.cu` (the fast simulation kernel) is
compiled once per (VMAX, CMAX) template pair."""
from __future__ import annotations

import concurrent.futures as cf
import os
import subprocess
import sys

_HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(_HERE, "csrc")
OBJ = os.path.join(CSRC, "build")
LIB = os.path.join(_HERE, "libcf_b200.so")
HEADERS = ["cf_device.cuh", "cf_rel32.cuh", "cf_scan.cuh", "cf_launch.h", "cf_aux.cuh", "cf_fcfs.cuh",
           os.path.join("..", "..", "include", "cf.h"), os.path.join("..", "..", "include", "cf_debug.h")]
# (object name, source, extra defines)
UNITS = [("cf_api", "cf_api.cu", []),
         ("cf_k64", "cf_k64.cu", []),
         ("cf_scan", "cf_scan.cu", []),
         ("cf_fcfs", "cf_fcfs.cu", []),
         ("cf_noalloc", "cf_noalloc.cu", [])] + \
        [(f"cf_k32_v{v}c{c}", "cf_k32.cu", [f"-DCF_VMAX={v}", f"-DCF_CMAX={c}"])
         for v, c in ((2, 6), (4, 6), (6, 6), (8, 6), (8, 8))]
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17",
              "--compiler-options", "-fPIC"]


def _newest_header() -> float:
    return max(os.path.getmtime(os.path.join(CSRC, h)) for h in HEADERS if os.path.exists(os.path.join(CSRC, h)))


def build(force: bool = False, verbose: bool = False) -> str:
    nvcc = os.environ.get("NVCC", "nvcc")
    os.makedirs(OBJ, exist_ok=True)
    hdr = max(_newest_header(), os.path.getmtime(os.path.abspath(__file__)))
    jobs = []
    units = [u for u in UNITS if os.path.exists(os.path.join(CSRC, u[1]))]
    for name, src, defs in units:
        obj = os.path.join(OBJ, name + ".o")
        srcp = os.path.join(CSRC, src)
        if force or not os.path.exists(obj) or os.path.getmtime(obj) < max(hdr, os.path.getmtime(srcp)):
            cmd = [nvcc] + NVCC_FLAGS + (["-Xptxas", "-v"] if verbose else []) + defs + ["-c", "-o", obj, src]
            jobs.append(cmd)
    if jobs:
        with cf.ThreadPoolExecutor(max_workers=min(len(jobs), os.cpu_count() or 1)) as ex:
            futs = [ex.submit(subprocess.run, cmd, cwd=CSRC, capture_output=True, text=True) for cmd in jobs]
            fail = False
            for cmd, f in zip(jobs, futs):
                r = f.result()
                if verbose or r.returncode:
                    sys.stderr.write(r.stdout + r.stderr)
                fail = fail or r.returncode != 0
            if fail:
                raise RuntimeError("nvcc failed")
    objs = [os.path.join(OBJ, name + ".o") for name, _, _ in units]
    if jobs or not os.path.exists(LIB) or os.path.getmtime(LIB) < max(os.path.getmtime(o) for o in objs):
        subprocess.run([nvcc, "-gencode", "arch=compute_100a,code=sm_100a", "-shared", "-o", LIB] + objs,
                       check=True, cwd=CSRC)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
