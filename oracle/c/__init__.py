"""Build + ctypes loader for the plain-C oracle twin (TEST INFRASTRUCTURE).

``build()`` compiles ``murmur_oracle.c`` with gcc (``-O2 -fopenmp``) into
``libmurmur_oracle.so`` next to the source; ``load()`` returns a small wrapper.  Used by
``tests/``, ``__graft_entry__`` and ``bench.py``'s ``cpu_baseline`` leg only.
"""
from __future__ import annotations

import ctypes
import os
import subprocess
from typing import Optional, Sequence, Tuple

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "murmur_oracle.c")
_LIB = os.path.join(_HERE, "libmurmur_oracle.so")


def build(force: bool = False) -> str:
    if not force and os.path.exists(_LIB) and os.path.getmtime(_LIB) >= os.path.getmtime(_SRC):
        return _LIB
    cmd = ["gcc", "-O2", "-std=c99", "-fopenmp", "-shared", "-fPIC", "-o", _LIB, _SRC, "-lm"]
    subprocess.run(cmd, check=True)
    return _LIB


class COracle:
    def __init__(self, lib: ctypes.CDLL):
        self._lib = lib
        lib.murmur_oracle_retained.restype = ctypes.c_int
        lib.murmur_oracle_retained.argtypes = [ctypes.c_int] * 10 + [ctypes.c_void_p, ctypes.c_int]
        lib.murmur_oracle_prefill.restype = ctypes.c_int
        lib.murmur_oracle_prefill.argtypes = [
            ctypes.c_int, ctypes.c_int, ctypes.c_int, ctypes.c_int, ctypes.c_void_p, ctypes.c_void_p,
            ctypes.c_int64, ctypes.c_int, ctypes.c_int, ctypes.c_void_p, ctypes.c_double,
            ctypes.c_void_p, ctypes.c_void_p, ctypes.c_int,
        ]
        lib.murmur_oracle_attend.restype = ctypes.c_int
        lib.murmur_oracle_attend.argtypes = [
            ctypes.c_int, ctypes.c_int, ctypes.c_int, ctypes.c_int, ctypes.c_void_p, ctypes.c_void_p,
            ctypes.c_int64, ctypes.c_void_p, ctypes.c_int, ctypes.c_void_p, ctypes.c_double,
            ctypes.c_void_p, ctypes.c_void_p, ctypes.c_int,
        ]

    def prefill(self, q_bits: np.ndarray, k_bits: np.ndarray, v_bits: np.ndarray, pos_begin: int, scale: float,
                n_threads: int = 0) -> Tuple[np.ndarray, np.ndarray, int]:
        """Causal prefill attention, several layers at once: q [L, n_tok, n_q, d], k/v [L, n_pos, n_kv, d] uint16 ->
        (out [L, n_tok, n_q, d] f64, lse [L, n_tok, n_q] f64, threads)."""
        q_bits = np.ascontiguousarray(q_bits, dtype=np.uint16)
        k_bits = np.ascontiguousarray(k_bits, dtype=np.uint16)
        v_bits = np.ascontiguousarray(v_bits, dtype=np.uint16)
        L, n_tok, n_q, d = q_bits.shape
        _, n_pos, n_kv, _ = k_bits.shape
        out = np.empty((L, n_tok, n_q, d), dtype=np.float64)
        lse = np.empty((L, n_tok, n_q), dtype=np.float64)
        used = self._lib.murmur_oracle_prefill(
            L, n_q, n_kv, d, k_bits.ctypes.data, v_bits.ctypes.data, n_pos, int(pos_begin), n_tok,
            q_bits.ctypes.data, float(scale), out.ctypes.data, lse.ctypes.data, int(n_threads))
        if used < 0:
            raise RuntimeError("murmur_oracle_prefill failed")
        return out, lse, used

    def retained(self, P: int, S: int, M: int, t: int, pol, length: Optional[int] = None) -> np.ndarray:
        total = P + S + M + t
        length = total if length is None else length
        out = np.empty((max(total, 1),), dtype=np.int32)
        n = self._lib.murmur_oracle_retained(
            P, S, M, t, pol.w_speech, pol.delay, pol.n_sink_speech, pol.w_out, pol.n_sink_out,
            length, out.ctypes.data, out.size)
        if n < 0:
            raise RuntimeError("murmur_oracle_retained: capacity")
        return out[:n].copy()

    def attend(self, q_bits: np.ndarray, k_bits: np.ndarray, v_bits: np.ndarray,
               retained: Sequence[int], scale: float, n_threads: int = 0) -> Tuple[np.ndarray, np.ndarray, int]:
        """q [L, n_q, d], k/v [L, n_pos, n_kv, d] uint16 -> (out [L, n_q, d] f64, lse [L, n_q], threads)."""
        q_bits = np.ascontiguousarray(q_bits, dtype=np.uint16)
        k_bits = np.ascontiguousarray(k_bits, dtype=np.uint16)
        v_bits = np.ascontiguousarray(v_bits, dtype=np.uint16)
        L, n_q, d = q_bits.shape
        _, n_pos, n_kv, _ = k_bits.shape
        ret = np.ascontiguousarray(np.asarray(retained, dtype=np.int32))
        out = np.empty((L, n_q, d), dtype=np.float64)
        lse = np.empty((L, n_q), dtype=np.float64)
        used = self._lib.murmur_oracle_attend(
            L, n_q, n_kv, d, k_bits.ctypes.data, v_bits.ctypes.data, n_pos, ret.ctypes.data, ret.size,
            q_bits.ctypes.data, float(scale), out.ctypes.data, lse.ctypes.data, int(n_threads))
        if used < 0:
            raise RuntimeError("murmur_oracle_attend failed")
        return out, lse, used


_cached: Optional[COracle] = None


def load() -> COracle:
    global _cached
    if _cached is None:
        _cached = COracle(ctypes.CDLL(build()))
    return _cached
