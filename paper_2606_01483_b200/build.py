"""In-tree build of libmurmur.so (hand-written CUDA for sm_100a) with nvcc.

The shared library lands next to this file so that it travels with the repository snapshot
to the GPU box.  No torch extension machinery: the boundary is a plain C ABI loaded with
ctypes (see binding.py).  Sources are compiled to objects in parallel (one nvcc per .cu,
only the stale ones) and linked into one shared library.

    python -m paper_2606_01483_b200.build [-v] [--trace]

``--trace`` (or MURMUR_TRACE=1 in the environment) compiles the per-CTA ``globaltimer`` stamps and
the two ``murmur_debug_*`` exports in (profiling builds only; see include/murmur.h).  ``--pftrace`` compiles
the prefill kernel's clock stamps in (``-DMURMUR_PFTRACE``: per-item and per-tile stamps of CTA 0's issuer and
of one softmax warp, read back with ``murmur_debug_pftrace`` / ``murmur_debug_pftile``; profiles/r02_prefill_ncu.md).
"""
from __future__ import annotations

import concurrent.futures
import os
import shutil
import subprocess
import sys
from typing import List, Sequence

_HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(_HERE, "csrc")
INCLUDE = os.path.join(os.path.dirname(_HERE), "include")
LIB = os.path.join(_HERE, "libmurmur.so")
OBJ_DIR = os.path.join(_HERE, "_obj")

SOURCES = ["murmur_api.cu", "kv_append.cu", "kv_evict.cu", "decode_attn_generic.cu", "decode_attn_mma.cu",
           "attn_profile.cu", "prefill_attn.cu", "prefill_attn_umma.cu", "chunk_plan.cu", "kv_indexed.cu",
           "decode_attn_indexed.cu"]
HEADERS = ["device_state.cuh", "policy_math.cuh", "evict_body.cuh", "ptx_utils.cuh", "umma_utils.cuh"]

NVCC_FLAGS = [
    "-O3", "-std=c++17", "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo",
    "-Xcompiler", "-fPIC,-fvisibility=hidden",
]
LINK_FLAGS = ["--shared", "-cudart", "static", "-gencode", "arch=compute_100a,code=sm_100a"]


def _nvcc() -> str:
    for cand in (shutil.which("nvcc"), "/usr/local/cuda/bin/nvcc"):
        if cand and os.path.exists(cand):
            return cand
    raise RuntimeError("nvcc not found: the CUDA extension cannot be built")


def _sources() -> List[str]:
    return [f for f in SOURCES if os.path.exists(os.path.join(CSRC, f))]


def _deps() -> List[str]:
    return [os.path.join(CSRC, f) for f in HEADERS if os.path.exists(os.path.join(CSRC, f))] + [
        os.path.join(INCLUDE, "murmur.h"), os.path.abspath(__file__)]


def _flag_file() -> str:
    return os.path.join(OBJ_DIR, "flags.txt")


def _stale() -> bool:
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    deps = [os.path.join(CSRC, f) for f in _sources()] + _deps()
    return any(os.path.getmtime(d) > t for d in deps)


def build(force: bool = False, verbose: bool = False, extra: Sequence[str] = (), trace: bool = False) -> str:
    trace = trace or os.environ.get("MURMUR_TRACE", "") not in ("", "0")
    flags = list(NVCC_FLAGS) + list(extra) + (["-DMURMUR_TRACE=1"] if trace else [])
    os.makedirs(OBJ_DIR, exist_ok=True)
    flag_str = " ".join(flags)
    try:
        with open(_flag_file()) as f:
            same_flags = f.read() == flag_str
    except OSError:
        same_flags = False
    if not force and same_flags and not _stale():
        return LIB
    nvcc = _nvcc()
    hdr_t = max(os.path.getmtime(d) for d in _deps())
    jobs = []
    objs = []
    for src in _sources():
        sp = os.path.join(CSRC, src)
        op = os.path.join(OBJ_DIR, src[:-3] + ".o")
        objs.append(op)
        fresh = (not force and same_flags and os.path.exists(op)
                 and os.path.getmtime(op) >= max(os.path.getmtime(sp), hdr_t))
        if not fresh:
            jobs.append([nvcc, *flags, "-I", INCLUDE, "-c", sp, "-o", op])

    def run(cmd):
        if verbose:
            print(" ".join(cmd), file=sys.stderr)
        r = subprocess.run(cmd, capture_output=True, text=True)
        return cmd, r

    with concurrent.futures.ThreadPoolExecutor(max_workers=min(8, max(1, len(jobs)))) as ex:
        for cmd, r in ex.map(run, jobs):
            if verbose or r.returncode != 0:
                sys.stderr.write(r.stdout + r.stderr)
            if r.returncode != 0:
                raise RuntimeError("nvcc failed: " + " ".join(cmd))
    link = [nvcc, *LINK_FLAGS, "-o", LIB, *objs]
    if verbose:
        print(" ".join(link), file=sys.stderr)
    subprocess.run(link, check=True)
    with open(_flag_file(), "w") as f:
        f.write(flag_str)
    return LIB


if __name__ == "__main__":
    build(force="-f" in sys.argv, verbose=True,
          extra=(["-Xptxas", "-v"] if "-v" in sys.argv else []) + (["-DMURMUR_PFTRACE=1"] if "--pftrace" in sys.argv else []),
          trace="--trace" in sys.argv)
    print(LIB)
