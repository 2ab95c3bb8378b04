"""Thin ctypes binding over the C ABI of include/murmur.h.

Argument marshalling only: every step of the path runs in the CUDA kernels of libmurmur.so.
PyTorch is used for device memory (pools, workspace, Q/O tensors) and the current stream.
There is no CPU fallback: if the library cannot be loaded, importing ``lib()`` raises.
"""
from __future__ import annotations

import ctypes as C
import math
import os
from typing import Optional, Sequence, Tuple

import numpy as np
import torch

from . import build as _build

MURMUR_WINDOW_OFF = 0x7FFFFFFF
MURMUR_OPT_ATTN_VARIANT = 1
MURMUR_OPT_ATTN_GRID = 2
MURMUR_OPT_PDL = 3
MURMUR_OPT_FUSE_STEP = 4
MURMUR_OPT_PREFILL_VARIANT = 5
MURMUR_OPT_HOST_ZERO_COPY = 6
MURMUR_OPT_L2_KEEP_PCT = 7
MURMUR_PREFILL_AUTO, MURMUR_PREFILL_MMA_SYNC, MURMUR_PREFILL_UMMA = 0, 1, 2
MURMUR_ATTN_AUTO, MURMUR_ATTN_GENERIC, MURMUR_ATTN_MMA = 0, 1, 2

STATUS_NAMES = {0: "MURMUR_OK", 1: "MURMUR_ERR_INVALID_ARG", 2: "MURMUR_ERR_STATE", 3: "MURMUR_ERR_OOM_PAGES",
                4: "MURMUR_ERR_CUDA", 5: "MURMUR_ERR_UNSUPPORTED", 6: "MURMUR_ERR_SCRATCH_LIMIT"}
MURMUR_PROFILE_NOALLOC_MAX_BYTES = 8 << 20

# every symbol include/murmur.h declares (checked by tests/test_abi.py)
EXPORTED_SYMBOLS = [
    "murmur_pool_bytes", "murmur_workspace_bytes", "murmur_cache_create", "murmur_cache_destroy",
    "murmur_seq_begin", "murmur_seq_end", "murmur_kv_append", "murmur_kv_evict", "murmur_decode_attn",
    "murmur_decode_step", "murmur_decode_step_layers", "murmur_decode_step_chunked", "murmur_decode_step_host", "murmur_mirror_sync", "murmur_seq_get_state", "murmur_kv_get_retained", "murmur_kv_get_page_list",
    "murmur_kv_get_runs", "murmur_kv_get_free_stack", "murmur_kv_gather", "murmur_get_last_error",
    "murmur_profile_scratch_bytes", "murmur_attn_profile", "murmur_attn_profile_noalloc",
    "murmur_decode_attn_windowed", "murmur_prefill_attn", "murmur_chunk_plan", "murmur_batch_plan",
    "murmur_indexed_bytes", "murmur_indexed_enable", "murmur_select_scratch_bytes", "murmur_select_mass_sets",
    "murmur_kv_evict_indexed", "murmur_kv_append_indexed", "murmur_decode_attn_indexed", "murmur_kv_get_indexed",
    "murmur_kv_gather_indexed",
    "murmur_set_option", "murmur_get_stats", "murmur_reset_stats", "murmur_status_str",
    "murmur_last_cuda_error", "murmur_version",
]


class CacheDesc(C.Structure):
    _fields_ = [("n_layers", C.c_int32), ("n_q_heads", C.c_int32), ("n_kv_heads", C.c_int32),
                ("head_dim", C.c_int32), ("page_size", C.c_int32), ("max_seqs", C.c_int32),
                ("max_blocks_per_seq", C.c_int32), ("n_pages", C.c_int64), ("k_pool", C.c_void_p),
                ("v_pool", C.c_void_p), ("workspace", C.c_void_p), ("workspace_bytes", C.c_size_t)]


class Policy(C.Structure):
    _fields_ = [("w_speech", C.c_int32), ("delay", C.c_int32), ("n_sink_speech", C.c_int32),
                ("w_out", C.c_int32), ("n_sink_out", C.c_int32)]


class Stats(C.Structure):
    _fields_ = [("kernel_launches", C.c_int64), ("append_calls", C.c_int64), ("evict_calls", C.c_int64),
                ("attn_calls", C.c_int64), ("free_pages", C.c_int64), ("attn_grid", C.c_int32),
                ("attn_smem_bytes", C.c_int32), ("attn_variant", C.c_int32), ("sm_count", C.c_int32),
                ("host_zero_copy_steps", C.c_int64)]


class MurmurError(RuntimeError):
    def __init__(self, status: int, what: str = ""):
        self.status = status
        super().__init__(f"{STATUS_NAMES.get(status, status)} {what}".strip())


_lib: Optional[C.CDLL] = None


def lib() -> C.CDLL:
    """Loads (building if needed) libmurmur.so.  Raises if it cannot - there is no fallback."""
    global _lib
    if _lib is not None:
        return _lib
    path = _build.LIB
    if not os.path.exists(path) or _build._stale():
        path = _build.build()
    L = C.CDLL(path)
    vp, i32, i64 = C.c_void_p, C.c_int32, C.c_int64
    L.murmur_pool_bytes.restype = C.c_size_t
    L.murmur_pool_bytes.argtypes = [C.POINTER(CacheDesc)]
    L.murmur_workspace_bytes.restype = C.c_size_t
    L.murmur_workspace_bytes.argtypes = [C.POINTER(CacheDesc)]
    L.murmur_cache_create.argtypes = [C.POINTER(CacheDesc), C.POINTER(vp), vp]
    L.murmur_cache_destroy.argtypes = [vp]
    L.murmur_seq_begin.argtypes = [vp, i32, i32, i32, i32, C.POINTER(Policy), vp]
    L.murmur_seq_end.argtypes = [vp, i32, vp]
    L.murmur_kv_append.argtypes = [vp, vp, vp, i32, vp, vp, i32, i32, vp]
    L.murmur_kv_evict.argtypes = [vp, vp, i32, vp]
    L.murmur_decode_attn.argtypes = [vp, vp, i32, vp, vp, vp, i32, i32, C.c_float, vp]
    L.murmur_decode_step.argtypes = [vp, vp, i32, vp, vp, vp, vp, vp, C.c_float, vp]
    L.murmur_decode_step_layers.argtypes = [vp, vp, i32, vp, vp, vp, vp, vp, i32, i32, C.c_float, vp]
    L.murmur_decode_step_chunked.argtypes = [vp, vp, i32, vp, vp, vp, vp, vp, i32, C.c_float, vp]
    L.murmur_mirror_sync.argtypes = [vp, vp]
    L.murmur_decode_step_host.argtypes = [vp, vp, i32, vp, vp, vp, vp, C.c_float, vp]
    L.murmur_seq_get_state.argtypes = [vp, i32, vp, vp]
    L.murmur_kv_get_retained.argtypes = [vp, i32, vp, i32, vp, vp]
    L.murmur_kv_get_page_list.argtypes = [vp, i32, vp, vp, i32, vp, vp]
    L.murmur_kv_get_runs.argtypes = [vp, i32, vp, i32, vp, vp]
    L.murmur_kv_get_free_stack.argtypes = [vp, vp, i64, vp, vp]
    L.murmur_kv_gather.argtypes = [vp, i32, vp, i32, i32, i32, vp, vp, vp]
    L.murmur_get_last_error.argtypes = [vp, vp, vp]
    if hasattr(L, "murmur_debug_attn_timeline"):  # profiling builds only (-DMURMUR_TRACE)
        L.murmur_debug_attn_timeline.argtypes = [vp, vp, i32, vp, vp]
        L.murmur_debug_step_trace.argtypes = [vp, vp, vp]
    L.murmur_decode_attn_windowed.argtypes = [vp, vp, i32, vp, vp, vp, i32, i32, C.c_float, vp, vp]
    L.murmur_chunk_plan.argtypes = [vp, vp, i32, C.c_float, vp, i32, vp]
    L.murmur_batch_plan.argtypes = [vp, vp, i32, vp, i32, i32, C.c_double, i32, C.c_double, i32, i32, i32, vp, vp]
    L.murmur_prefill_attn.argtypes = [vp, i32, i32, i32, vp, vp, vp, i32, i32, C.c_float, vp]
    L.murmur_profile_scratch_bytes.argtypes = [vp, vp, i32, i32, i32]
    L.murmur_profile_scratch_bytes.restype = C.c_size_t
    L.murmur_attn_profile.argtypes = [vp, vp, i32, vp, vp, C.c_float, vp, vp, C.c_size_t, i32, i32, C.c_float, vp]
    L.murmur_attn_profile_noalloc.argtypes = [vp, vp, i32, vp, vp, C.c_float, vp, i32, i32, C.c_float, vp]
    L.murmur_indexed_bytes.restype = C.c_size_t
    L.murmur_indexed_bytes.argtypes = [C.POINTER(CacheDesc)]
    L.murmur_indexed_enable.argtypes = [vp, vp, C.c_size_t, vp]
    L.murmur_select_scratch_bytes.restype = C.c_size_t
    L.murmur_select_scratch_bytes.argtypes = [vp, i32]
    L.murmur_select_mass_sets.argtypes = [vp, i32, vp, C.c_float, i32, vp, vp, i32, vp, C.c_size_t, C.c_float, vp]
    L.murmur_kv_evict_indexed.argtypes = [vp, i32, vp, vp, i32, vp, vp]
    L.murmur_kv_append_indexed.argtypes = [vp, vp, i32, vp, vp, vp]
    L.murmur_decode_attn_indexed.argtypes = [vp, vp, i32, vp, vp, vp, C.c_float, vp]
    L.murmur_kv_get_indexed.argtypes = [vp, i32, i32, i32, vp, i32, vp, vp]
    L.murmur_kv_gather_indexed.argtypes = [vp, i32, vp, vp, i32, vp]
    L.murmur_set_option.argtypes = [vp, i32, i32]
    L.murmur_get_stats.argtypes = [vp, C.POINTER(Stats)]
    L.murmur_reset_stats.argtypes = [vp]
    L.murmur_status_str.restype = C.c_char_p
    L.murmur_status_str.argtypes = [C.c_int]
    L.murmur_last_cuda_error.restype = C.c_char_p
    L.murmur_last_cuda_error.argtypes = [vp]
    L.murmur_version.restype = C.c_char_p
    for name in EXPORTED_SYMBOLS:
        fn = getattr(L, name)
        if fn.restype is C.c_int:  # default restype: status codes
            fn.restype = C.c_int
    _lib = L
    return L


def _ids(a: Sequence[int]) -> np.ndarray:
    return np.ascontiguousarray(np.asarray(a, dtype=np.int32))


def _stream() -> int:
    return int(torch.cuda.current_stream().cuda_stream)


class MurmurCache:
    """Owns the device buffers (torch tensors) and the murmur_cache_t handle."""

    def __init__(self, n_layers: int, n_q_heads: int, n_kv_heads: int, head_dim: int, page_size: int,
                 max_seqs: int, max_blocks_per_seq: int, n_pages: int, device="cuda:0"):
        self.L = lib()
        self.device = torch.device(device)
        torch.cuda.set_device(self.device)
        self.n_layers, self.n_q, self.n_kv, self.d = n_layers, n_q_heads, n_kv_heads, head_dim
        self.page_size, self.max_seqs, self.max_blocks, self.n_pages = page_size, max_seqs, max_blocks_per_seq, n_pages
        d = CacheDesc(n_layers, n_q_heads, n_kv_heads, head_dim, page_size, max_seqs, max_blocks_per_seq, n_pages,
                      None, None, None, 0)
        pool_bytes = self.L.murmur_pool_bytes(C.byref(d))
        ws_bytes = self.L.murmur_workspace_bytes(C.byref(d))
        if pool_bytes == 0 or ws_bytes == 0:
            raise MurmurError(5, "unsupported geometry")
        self.k_pool = torch.empty(pool_bytes, dtype=torch.uint8, device=self.device)
        self.v_pool = torch.empty(pool_bytes, dtype=torch.uint8, device=self.device)
        self.workspace = torch.empty(ws_bytes, dtype=torch.uint8, device=self.device)
        d.k_pool, d.v_pool, d.workspace = self.k_pool.data_ptr(), self.v_pool.data_ptr(), self.workspace.data_ptr()
        d.workspace_bytes = ws_bytes
        self.desc = d
        h = C.c_void_p()
        self._check(self.L.murmur_cache_create(C.byref(d), C.byref(h), _stream()))
        self.h = h

    def close(self):
        if getattr(self, "h", None):
            torch.cuda.synchronize(self.device)
            self.L.murmur_cache_destroy(self.h)
            self.h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def _check(self, st: int):
        if st != 0:
            what = ""
            if st == 4 and getattr(self, "h", None):
                what = self.L.murmur_last_cuda_error(self.h).decode()
            raise MurmurError(st, what)

    # ---- lifecycle ----------------------------------------------------------------------
    def seq_begin(self, seq: int, n_prefix: int, n_speech: int, n_mid: int, policy: Tuple[int, int, int, int, int]):
        pol = Policy(*policy)
        self._check(self.L.murmur_seq_begin(self.h, seq, n_prefix, n_speech, n_mid, C.byref(pol), _stream()))

    def seq_end(self, seq: int):
        self._check(self.L.murmur_seq_end(self.h, seq, _stream()))

    # ---- hot path -----------------------------------------------------------------------
    def kv_append(self, seq_ids, n_tokens, k_new: torch.Tensor, v_new: torch.Tensor, layer_begin: int = 0,
                  layer_end: Optional[int] = None):
        layer_end = self.n_layers if layer_end is None else layer_end
        ids, nt = _ids(seq_ids), _ids(n_tokens)
        total = int(nt.sum())
        for t in (k_new, v_new):
            assert t.dtype == torch.bfloat16 and t.is_cuda and t.is_contiguous()
            assert t.numel() == (layer_end - layer_begin) * total * self.n_kv * self.d, "k_new/v_new shape"
        self._check(self.L.murmur_kv_append(self.h, ids.ctypes.data, nt.ctypes.data, len(ids), k_new.data_ptr(),
                                            v_new.data_ptr(), layer_begin, layer_end, _stream()))

    def kv_evict(self, seq_ids):
        ids = _ids(seq_ids)
        self._check(self.L.murmur_kv_evict(self.h, ids.ctypes.data, len(ids), _stream()))

    def decode_attn(self, seq_ids, q: torch.Tensor, out: Optional[torch.Tensor] = None,
                    lse: Optional[torch.Tensor] = None, sm_scale: Optional[float] = None, layer_begin: int = 0,
                    layer_end: Optional[int] = None, window=None) -> torch.Tensor:
        """window: optional 5-tuple policy -> murmur_decode_attn_windowed (per-layer windows)."""
        layer_end = self.n_layers if layer_end is None else layer_end
        ids = _ids(seq_ids)
        shape = (layer_end - layer_begin, len(ids), self.n_q, self.d)
        assert q.dtype == torch.bfloat16 and q.is_cuda and q.is_contiguous() and tuple(q.shape) == shape
        if out is None:
            out = torch.empty(shape, dtype=torch.bfloat16, device=self.device)
        assert out.dtype == torch.bfloat16 and out.is_contiguous() and tuple(out.shape) == shape
        if lse is not None:
            assert lse.dtype == torch.float32 and lse.is_contiguous() and tuple(lse.shape) == shape[:3]
        sm_scale = 1.0 / math.sqrt(self.d) if sm_scale is None else sm_scale
        if window is not None:
            pol = (C.c_int32 * 5)(*window)
            self._check(self.L.murmur_decode_attn_windowed(self.h, ids.ctypes.data, len(ids), q.data_ptr(), out.data_ptr(),
                                                           lse.data_ptr() if lse is not None else None, layer_begin,
                                                           layer_end, C.c_float(sm_scale), pol, _stream()))
            return out
        self._check(self.L.murmur_decode_attn(self.h, ids.ctypes.data, len(ids), q.data_ptr(), out.data_ptr(),
                                              lse.data_ptr() if lse is not None else None, layer_begin, layer_end,
                                              C.c_float(sm_scale), _stream()))
        return out

    def prefill_attn(self, seq: int, pos_begin: int, pos_end: int, q: torch.Tensor, out: Optional[torch.Tensor] = None,
                     lse: Optional[torch.Tensor] = None, sm_scale: Optional[float] = None, layer_begin: int = 0,
                     layer_end: Optional[int] = None) -> torch.Tensor:
        """Causal attention of the prefill positions [pos_begin, pos_end): q, out [layers, n_tok, n_q, d] bf16."""
        layer_end = self.n_layers if layer_end is None else layer_end
        shape = (layer_end - layer_begin, pos_end - pos_begin, self.n_q, self.d)
        assert q.dtype == torch.bfloat16 and q.is_cuda and q.is_contiguous() and tuple(q.shape) == shape
        if out is None:
            out = torch.empty(shape, dtype=torch.bfloat16, device=self.device)
        assert out.dtype == torch.bfloat16 and out.is_contiguous() and tuple(out.shape) == shape
        if lse is not None:
            assert lse.dtype == torch.float32 and lse.is_contiguous() and tuple(lse.shape) == shape[:3]
        sm_scale = 1.0 / math.sqrt(self.d) if sm_scale is None else sm_scale
        self._check(self.L.murmur_prefill_attn(self.h, seq, pos_begin, pos_end, q.data_ptr(), out.data_ptr(),
                                               lse.data_ptr() if lse is not None else None, layer_begin, layer_end,
                                               C.c_float(sm_scale), _stream()))
        return out

    def attn_profile(self, seq_ids, q: torch.Tensor, candidate=None, mass_frac: float = 0.99,
                     sm_scale: Optional[float] = None, layer_begin: int = 0, layer_end: Optional[int] = None) -> np.ndarray:
        """Attention-sparsity profile of the step whose queries are q: structured array
        [layers, n_seqs, n_q] with the fields of murmur_profile_t.  candidate: 5-tuple policy or None."""
        layer_end = self.n_layers if layer_end is None else layer_end
        ids = _ids(seq_ids)
        shape = (layer_end - layer_begin, len(ids), self.n_q, self.d)
        assert q.dtype == torch.bfloat16 and q.is_cuda and q.is_contiguous() and tuple(q.shape) == shape
        sm_scale = 1.0 / math.sqrt(self.d) if sm_scale is None else sm_scale
        nbytes = self.L.murmur_profile_scratch_bytes(self.h, ids.ctypes.data, len(ids), layer_begin, layer_end)
        if nbytes == 0:
            raise MurmurError(1, "murmur_profile_scratch_bytes: bad arguments")
        scratch = torch.empty(nbytes, dtype=torch.uint8, device=self.device)
        out = torch.zeros(shape[:3] + (12,), dtype=torch.int32, device=self.device)
        pol = (C.c_int32 * 5)(*candidate) if candidate is not None else None
        self._check(self.L.murmur_attn_profile(self.h, ids.ctypes.data, len(ids), q.data_ptr(), pol, C.c_float(mass_frac),
                                               out.data_ptr(), scratch.data_ptr(), nbytes, layer_begin, layer_end,
                                               C.c_float(sm_scale), _stream()))
        torch.cuda.synchronize(self.device)
        dt = np.dtype([(n, np.int32) for n in ("n_resident", "n_prompt", "n_speech", "n_text", "k_mass", "k_prompt",
                                               "k_speech", "k_text")] +
                      [(n, np.float32) for n in ("coverage", "mass_prompt", "mass_speech", "mass_text")])
        return out.cpu().numpy().view(dt).reshape(shape[:3])

    def attn_profile_noalloc(self, seq_ids, q: torch.Tensor, out: torch.Tensor, candidate=None, mass_frac: float = 0.99,
                             sm_scale: Optional[float] = None, layer_begin: int = 0, layer_end: Optional[int] = None):
        """murmur_attn_profile_noalloc: the same profile for callers that may not allocate device memory (a hook
        inside an engine that owns all of HBM, a latency-critical loop where cudaMalloc would stall the GPU).  The
        scratch is a fixed MURMUR_PROFILE_NOALLOC_MAX_BYTES array inside the library, so this method allocates
        nothing either: `out` is the caller's int32 tensor [layers, n_seqs, n_q, 12] (12 words = murmur_profile_t)
        and is filled asynchronously on the current stream; view it with `profile_view` after synchronising.
        Raises MurmurError(6) when the sequences are too long for the built-in array.  Calls that overlap on the
        GPU share that array and race; the first call on a device should precede any stream capture."""
        layer_end = self.n_layers if layer_end is None else layer_end
        ids = _ids(seq_ids)
        shape = (layer_end - layer_begin, len(ids), self.n_q, self.d)
        assert q.dtype == torch.bfloat16 and q.is_cuda and q.is_contiguous() and tuple(q.shape) == shape
        assert out.dtype == torch.int32 and out.is_cuda and out.is_contiguous() and tuple(out.shape) == shape[:3] + (12,)
        sm_scale = 1.0 / math.sqrt(self.d) if sm_scale is None else sm_scale
        pol = (C.c_int32 * 5)(*candidate) if candidate is not None else None
        st = self.L.murmur_attn_profile_noalloc(self.h, ids.ctypes.data, len(ids), q.data_ptr(), pol,
                                                C.c_float(mass_frac), out.data_ptr(), layer_begin, layer_end,
                                                C.c_float(sm_scale), _stream())
        if st == 6:
            raise MurmurError(st, f"the profile needs more than the built-in {MURMUR_PROFILE_NOALLOC_MAX_BYTES} bytes of "
                                  "scratch: use fewer layers or sequences per call, or murmur_attn_profile with your own buffer")
        self._check(st)

    @staticmethod
    def profile_view(out: torch.Tensor) -> np.ndarray:
        """Structured view (fields of murmur_profile_t) of an `out` tensor of attn_profile_noalloc; synchronises."""
        dt = np.dtype([(n, np.int32) for n in ("n_resident", "n_prompt", "n_speech", "n_text", "k_mass", "k_prompt",
                                               "k_speech", "k_text")] +
                      [(n, np.float32) for n in ("coverage", "mass_prompt", "mass_speech", "mass_text")])
        return out.cpu().numpy().view(dt).reshape(tuple(out.shape[:3]))

    def decode_step(self, seq_ids, k_new: torch.Tensor, v_new: torch.Tensor, q: torch.Tensor, out: torch.Tensor,
                    lse: Optional[torch.Tensor] = None, sm_scale: Optional[float] = None):
        """append (1 token per sequence, all layers) -> evict -> decode_attn in one C call; DEVICE tensors."""
        ids = seq_ids if isinstance(seq_ids, np.ndarray) and seq_ids.dtype == np.int32 else _ids(seq_ids)
        sm_scale = 1.0 / math.sqrt(self.d) if sm_scale is None else sm_scale
        self._check(self.L.murmur_decode_step(self.h, ids.ctypes.data, len(ids), k_new.data_ptr(), v_new.data_ptr(),
                                              q.data_ptr(), out.data_ptr(),
                                              lse.data_ptr() if lse is not None else None, C.c_float(sm_scale),
                                              _stream()))

    def decode_step_layers(self, seq_ids, k_new: torch.Tensor, v_new: torch.Tensor, q: torch.Tensor, out: torch.Tensor,
                           layer_begin: int, layer_end: int, lse: Optional[torch.Tensor] = None,
                           sm_scale: Optional[float] = None):
        """The decode step restricted to layers [layer_begin, layer_end), one launch; layer_begin == 0 opens the step."""
        ids = seq_ids if isinstance(seq_ids, np.ndarray) and seq_ids.dtype == np.int32 else _ids(seq_ids)
        sm_scale = 1.0 / math.sqrt(self.d) if sm_scale is None else sm_scale
        self._check(self.L.murmur_decode_step_layers(self.h, ids.ctypes.data, len(ids), k_new.data_ptr(), v_new.data_ptr(),
                                                     q.data_ptr(), out.data_ptr(),
                                                     lse.data_ptr() if lse is not None else None, layer_begin, layer_end,
                                                     C.c_float(sm_scale), _stream()))

    def decode_step_chunked(self, seq_ids, k_new: torch.Tensor, v_new: torch.Tensor, q: torch.Tensor, out: torch.Tensor,
                            layers_per_launch: int, lse: Optional[torch.Tensor] = None, sm_scale: Optional[float] = None):
        """The whole step issued from C as ceil(L / layers_per_launch) launches (1 = layer-by-layer engine pattern)."""
        ids = seq_ids if isinstance(seq_ids, np.ndarray) and seq_ids.dtype == np.int32 else _ids(seq_ids)
        sm_scale = 1.0 / math.sqrt(self.d) if sm_scale is None else sm_scale
        self._check(self.L.murmur_decode_step_chunked(self.h, ids.ctypes.data, len(ids), k_new.data_ptr(), v_new.data_ptr(),
                                                      q.data_ptr(), out.data_ptr(),
                                                      lse.data_ptr() if lse is not None else None, layers_per_launch,
                                                      C.c_float(sm_scale), _stream()))

    def mirror_sync(self):
        """After replaying captured steps (CUDA graph): re-reads lengths and the free-page count from the device."""
        self._check(self.L.murmur_mirror_sync(self.h, _stream()))

    def decode_step_host(self, seq_ids, k_new: torch.Tensor, v_new: torch.Tensor, q: torch.Tensor,
                         out: torch.Tensor, sm_scale: Optional[float] = None):
        """All tensors are HOST (ideally pinned) bf16; enqueues H2D + append + evict + attn + D2H."""
        ids = _ids(seq_ids)
        for t in (k_new, v_new, q, out):
            assert t.dtype == torch.bfloat16 and not t.is_cuda and t.is_contiguous()
        sm_scale = 1.0 / math.sqrt(self.d) if sm_scale is None else sm_scale
        self._check(self.L.murmur_decode_step_host(self.h, ids.ctypes.data, len(ids), k_new.data_ptr(),
                                                   v_new.data_ptr(), q.data_ptr(), out.data_ptr(),
                                                   C.c_float(sm_scale), _stream()))

    # ---- general index-set eviction (indexed mode) ------------------------------------------
    def indexed_enable(self):
        """Allocates the indexed-mode tables (a torch tensor owned by this object) and hands them to the handle."""
        n = self.L.murmur_indexed_bytes(C.byref(self.desc))
        self.indexed_buf = torch.empty(n, dtype=torch.uint8, device=self.device)
        self._check(self.L.murmur_indexed_enable(self.h, self.indexed_buf.data_ptr(), n, _stream()))

    def select_mass_sets(self, seq: int, q: torch.Tensor, mass_frac: float, n_recent: int, cap: int,
                         sm_scale: Optional[float] = None) -> Tuple[torch.Tensor, torch.Tensor]:
        """Query-aware index sets of one positional sequence: (sel_pos int32 [L, n_kv, cap], sel_cnt int32 [L, n_kv]) on the device."""
        assert q.dtype == torch.bfloat16 and q.is_cuda and q.is_contiguous() and tuple(q.shape) == (self.n_layers, self.n_q, self.d)
        sm_scale = 1.0 / math.sqrt(self.d) if sm_scale is None else sm_scale
        nb = self.L.murmur_select_scratch_bytes(self.h, seq)
        if nb == 0:
            raise MurmurError(2, "murmur_select_scratch_bytes: sequence not active or already indexed")
        scratch = torch.empty(nb, dtype=torch.uint8, device=self.device)
        sel_pos = torch.zeros(self.n_layers, self.n_kv, cap, dtype=torch.int32, device=self.device)
        sel_cnt = torch.zeros(self.n_layers, self.n_kv, dtype=torch.int32, device=self.device)
        self._check(self.L.murmur_select_mass_sets(self.h, seq, q.data_ptr(), C.c_float(mass_frac), n_recent, sel_pos.data_ptr(),
                                                   sel_cnt.data_ptr(), cap, scratch.data_ptr(), nb, C.c_float(sm_scale), _stream()))
        torch.cuda.synchronize(self.device)
        return sel_pos, sel_cnt

    def kv_evict_indexed(self, seq: int, sel_pos: torch.Tensor, sel_cnt: torch.Tensor) -> int:
        """Applies per-(layer, KV head) index sets (device int32 tensors); returns the bytes of K/V rows moved."""
        assert sel_pos.dtype == torch.int32 and sel_pos.is_cuda and sel_pos.is_contiguous() and sel_pos.dim() == 3
        assert sel_cnt.dtype == torch.int32 and sel_cnt.is_cuda and sel_cnt.is_contiguous()
        assert tuple(sel_pos.shape[:2]) == (self.n_layers, self.n_kv) == tuple(sel_cnt.shape)
        moved = C.c_int64(0)
        self._check(self.L.murmur_kv_evict_indexed(self.h, seq, sel_pos.data_ptr(), sel_cnt.data_ptr(), sel_pos.shape[2],
                                                   C.byref(moved), _stream()))
        return moved.value

    def kv_append_indexed(self, seq_ids, k_new: torch.Tensor, v_new: torch.Tensor):
        ids = _ids(seq_ids)
        for t in (k_new, v_new):
            assert t.dtype == torch.bfloat16 and t.is_cuda and t.is_contiguous()
            assert tuple(t.shape) == (self.n_layers, len(ids), self.n_kv, self.d)
        self._check(self.L.murmur_kv_append_indexed(self.h, ids.ctypes.data, len(ids), k_new.data_ptr(), v_new.data_ptr(), _stream()))

    def decode_attn_indexed(self, seq_ids, q: torch.Tensor, lse: Optional[torch.Tensor] = None,
                            sm_scale: Optional[float] = None) -> torch.Tensor:
        ids = _ids(seq_ids)
        shape = (self.n_layers, len(ids), self.n_q, self.d)
        assert q.dtype == torch.bfloat16 and q.is_cuda and q.is_contiguous() and tuple(q.shape) == shape
        out = torch.empty(shape, dtype=torch.bfloat16, device=self.device)
        sm_scale = 1.0 / math.sqrt(self.d) if sm_scale is None else sm_scale
        self._check(self.L.murmur_decode_attn_indexed(self.h, ids.ctypes.data, len(ids), q.data_ptr(), out.data_ptr(),
                                                      lse.data_ptr() if lse is not None else None, C.c_float(sm_scale), _stream()))
        return out

    def indexed_positions(self, seq: int, layer: int, kv_head: int) -> np.ndarray:
        cap = self.max_blocks * self.page_size
        a = np.zeros(cap, dtype=np.int32)
        n = C.c_int32(0)
        self._check(self.L.murmur_kv_get_indexed(self.h, seq, layer, kv_head, a.ctypes.data, cap, C.byref(n), _stream()))
        return a[: n.value].copy()

    def gather_indexed(self, seq: int, cap_rows: int) -> Tuple[torch.Tensor, torch.Tensor]:
        shape = (self.n_layers, self.n_kv, cap_rows, self.d)
        k = torch.empty(shape, dtype=torch.bfloat16, device=self.device)
        v = torch.empty(shape, dtype=torch.bfloat16, device=self.device)
        self._check(self.L.murmur_kv_gather_indexed(self.h, seq, k.data_ptr(), v.data_ptr(), cap_rows, _stream()))
        return k, v

    # ---- introspection ------------------------------------------------------------------
    def seq_state(self, seq: int) -> dict:
        a = np.zeros(6, dtype=np.int32)
        self._check(self.L.murmur_seq_get_state(self.h, seq, a.ctypes.data, _stream()))
        return dict(zip(("length", "t", "n_live", "n_runs", "n_tiles", "n_retained"), (int(x) for x in a)))

    def retained(self, seq: int) -> np.ndarray:
        cap = self.max_blocks * self.page_size
        a = np.zeros(cap, dtype=np.int32)
        n = C.c_int32(0)
        self._check(self.L.murmur_kv_get_retained(self.h, seq, a.ctypes.data, cap, C.byref(n), _stream()))
        return a[: n.value].copy()

    def page_list(self, seq: int) -> Tuple[np.ndarray, np.ndarray]:
        pages = np.zeros(self.max_blocks, dtype=np.int32)
        blocks = np.zeros(self.max_blocks, dtype=np.int32)
        n = C.c_int32(0)
        self._check(self.L.murmur_kv_get_page_list(self.h, seq, pages.ctypes.data, blocks.ctypes.data,
                                                   self.max_blocks, C.byref(n), _stream()))
        return pages[: n.value].copy(), blocks[: n.value].copy()

    def runs(self, seq: int):
        a = np.zeros(18, dtype=np.int32)
        n = C.c_int32(0)
        self._check(self.L.murmur_kv_get_runs(self.h, seq, a.ctypes.data, 6, C.byref(n), _stream()))
        return [tuple(int(x) for x in a[3 * r: 3 * r + 3]) for r in range(n.value)]

    def free_stack(self) -> np.ndarray:
        a = np.zeros(self.n_pages, dtype=np.int32)
        n = C.c_int64(0)
        self._check(self.L.murmur_kv_get_free_stack(self.h, a.ctypes.data, self.n_pages, C.byref(n), _stream()))
        return a[: n.value].copy()

    def gather(self, seq: int, positions, layer_begin: int = 0, layer_end: Optional[int] = None):
        layer_end = self.n_layers if layer_end is None else layer_end
        pos = _ids(positions)
        shape = (layer_end - layer_begin, len(pos), self.n_kv, self.d)
        k = torch.empty(shape, dtype=torch.bfloat16, device=self.device)
        v = torch.empty(shape, dtype=torch.bfloat16, device=self.device)
        self._check(self.L.murmur_kv_gather(self.h, seq, pos.ctypes.data, len(pos), layer_begin, layer_end,
                                            k.data_ptr(), v.data_ptr(), _stream()))
        return k, v

    def last_error(self) -> int:
        e = C.c_int32(0)
        self._check(self.L.murmur_get_last_error(self.h, C.byref(e), _stream()))
        return e.value

    def attn_timeline(self) -> np.ndarray:
        """uint64 [n_ctas, 8] = (start ns, end ns, SM id, tiles, entry ns, set-up done, keeper begin, keeper end) of the
        last tensor-core attention launch.
        Needs a profiling build of the library (python -m paper_2606_01483_b200.build --trace)."""
        if not hasattr(self.L, "murmur_debug_attn_timeline"):
            raise MurmurError(5, "library built without MURMUR_TRACE")
        a = np.zeros((1024, 8), dtype=np.uint64)
        n = C.c_int32(0)
        self._check(self.L.murmur_debug_attn_timeline(self.h, a.ctypes.data, 1024, C.byref(n), _stream()))
        return a[: n.value].copy()

    def step_trace(self) -> np.ndarray:
        """uint64 [16]: globaltimer stamps of the last step prologue (see murmur_debug_step_trace)."""
        if not hasattr(self.L, "murmur_debug_step_trace"):
            raise MurmurError(5, "library built without MURMUR_TRACE")
        a = np.zeros(16, dtype=np.uint64)
        self._check(self.L.murmur_debug_step_trace(self.h, a.ctypes.data, _stream()))
        return a

    def set_option(self, option: int, value: int):
        self._check(self.L.murmur_set_option(self.h, option, value))

    def stats(self) -> dict:
        s = Stats()
        self._check(self.L.murmur_get_stats(self.h, C.byref(s)))
        return {f: getattr(s, f) for f, _ in Stats._fields_}

    def reset_stats(self):
        self._check(self.L.murmur_reset_stats(self.h))


def chunk_plan(segments, max_len: float = 300.0):
    """Greedy VAD-segment merge (murmur_chunk_plan): list of (start, end) seconds -> list of lists of segment indices."""
    seg = np.ascontiguousarray(np.asarray(segments, dtype=np.float32).reshape(-1, 2))
    a, b = np.ascontiguousarray(seg[:, 0]), np.ascontiguousarray(seg[:, 1])
    first = np.zeros(max(1, len(seg)), dtype=np.int32)
    n = C.c_int32(0)
    st = lib().murmur_chunk_plan(a.ctypes.data, b.ctypes.data, len(seg), C.c_float(max_len), first.ctypes.data, len(first),
                                 C.byref(n))
    if st != 0:
        raise MurmurError(st, "murmur_chunk_plan")
    cuts = list(first[: n.value]) + [len(seg)]
    return [list(range(cuts[j], cuts[j + 1])) for j in range(n.value)]


def batch_plan(segments, chunks, batch_size: int = 16, tokens_per_s: float = 7.5, max_new_nominal: int = 32768,
               d_nominal: float = 3600.0, n_prefix: int = 0, n_mid: int = 0, page_size: int = 64):
    """murmur_batch_plan: chunks (lists of segment indices, as chunk_plan returns them) -> list of batches, each a list
    of dicts {chunk, slot, n_speech, max_new, max_blocks}."""
    seg = np.ascontiguousarray(np.asarray(segments, dtype=np.float32).reshape(-1, 2))
    a, b = np.ascontiguousarray(seg[:, 0]), np.ascontiguousarray(seg[:, 1])
    first = np.ascontiguousarray(np.asarray([ch[0] for ch in chunks], dtype=np.int32))
    ent = np.zeros((max(1, len(first)), 6), dtype=np.int32)
    nb = C.c_int32(0)
    st = lib().murmur_batch_plan(a.ctypes.data, b.ctypes.data, len(seg), first.ctypes.data, len(first), batch_size,
                                 C.c_double(tokens_per_s), max_new_nominal, C.c_double(d_nominal), n_prefix, n_mid,
                                 page_size, ent.ctypes.data, C.byref(nb))
    if st != 0:
        raise MurmurError(st, "murmur_batch_plan")
    batches = [[] for _ in range(nb.value)]
    for j in range(len(first)):
        ch, bt, slot, S, T, mb = (int(x) for x in ent[j])
        batches[bt].append({"chunk": ch, "slot": slot, "n_speech": S, "max_new": T, "max_blocks": mb})
    return batches


def version() -> str:
    return lib().murmur_version().decode()
