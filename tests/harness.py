"""Side-by-side driver: runs one workloads.Config through the CUDA path (C ABI via the binding)
and through the oracle on the same seeded bits, and compares them.

Used by the ``-m gpu`` parity tests and by ``__graft_entry__.smoke()``.  The two sides meet
only here: integer state must be bit-exact, attention within the stated tolerance
(max-abs <= 2e-2, mean-abs <= 2e-3 on unit-scale bf16 outputs - BASELINE.json north_star).
"""
from __future__ import annotations

import math
import os
import sys
from typing import Dict, Iterable, List, Optional, Sequence

import numpy as np
import torch

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import workloads  # noqa: E402
from oracle import attention as o_attn  # noqa: E402
from oracle import paged_cache as o_cache  # noqa: E402
from oracle import policy as o_policy  # noqa: E402

MAX_ABS_TOL = 2e-2
MEAN_ABS_TOL = 2e-3


def out_to_f64(out_bf16: torch.Tensor) -> np.ndarray:
    return o_attn.bf16_bits_to_f64(workloads.to_bits(out_bf16))


class RowStore:
    """K (or V) rows of one sequence by absolute position, uint16 [L, n_pos, n_kv, d], grown in place
    (the full-size cases hold ~100 MB per sequence: no re-concatenation per step)."""

    def __init__(self):
        self.buf: Optional[np.ndarray] = None
        self.n = 0

    def append(self, bits: np.ndarray):
        n_new = bits.shape[1]
        if self.buf is None or self.n + n_new > self.buf.shape[1]:
            cap = self.n + n_new + max(64, (self.n + n_new) // 4)
            nb = np.empty((bits.shape[0], cap) + bits.shape[2:], dtype=np.uint16)
            if self.buf is not None:
                nb[:, : self.n] = self.buf[:, : self.n]
            self.buf = nb
        self.buf[:, self.n: self.n + n_new] = bits
        self.n += n_new

    def rows(self) -> np.ndarray:
        return self.buf[:, : self.n]


class SideBySide:
    def __init__(self, cfg: workloads.Config, device="cuda:0", n_pages: Optional[int] = None, max_seqs: Optional[int] = None,
                 extra_tokens: int = 0, variant: Optional[int] = None, grid: Optional[int] = None, use_c_oracle: bool = False,
                 data: Optional[list] = None, bulk_bits: Optional[dict] = None):
        """data: SeqData list shared between cases that use the same seeded values (the config-4 sweep);
        bulk_bits: {(seq, n_tokens): (k_bits, v_bits)} host copies of bulk appends, filled and re-used
        across such cases (saves the device-to-host copy of ~2 GB per case)."""
        from paper_2606_01483_b200 import MurmurCache, binding

        self.cfg = cfg
        self.device = torch.device(device)
        g = cfg.geom
        self.p = cfg.page_size
        n_pages = workloads.unevicted_blocks(cfg, extra_tokens) + 2 if n_pages is None else n_pages
        max_blocks = workloads.max_blocks_per_seq(cfg, extra_tokens) + 1
        max_seqs = cfg.batch if max_seqs is None else max_seqs
        self.gpu = MurmurCache(g.n_layers, g.n_q_heads, g.n_kv_heads, g.head_dim, cfg.page_size, max_seqs, max_blocks,
                               n_pages, device=device)
        if variant is not None:
            self.gpu.set_option(binding.MURMUR_OPT_ATTN_VARIANT, variant)
        if grid is not None:
            self.gpu.set_option(binding.MURMUR_OPT_ATTN_GRID, grid)
        self.oracle = o_cache.OraclePagedCache(n_pages, cfg.page_size, max_seqs, max_blocks)
        self.data = data if data is not None else [workloads.SeqData(cfg, i, device=device) for i in range(cfg.batch)]
        self.bulk_bits = bulk_bits
        # oracle-side K/V by absolute position: uint16 [L, n_pos, n_kv, d] per sequence
        self.k_store: Dict[int, RowStore] = {i: RowStore() for i in range(cfg.batch)}
        self.v_store: Dict[int, RowStore] = {i: RowStore() for i in range(cfg.batch)}
        self.scale = 1.0 / math.sqrt(g.head_dim)
        self.use_c_oracle = use_c_oracle
        self.max_abs_seen = 0.0
        self.mean_abs_seen = 0.0
        for i, s in enumerate(cfg.seqs):
            self.gpu.seq_begin(i, s.P, s.S, s.M, s.policy_tuple)
            self.oracle.seq_begin(i, s.P, s.S, s.M, o_policy.Policy(*s.policy_tuple))

    # ---- helpers ---------------------------------------------------------------------------
    def _store(self, i: int, k: torch.Tensor, v: torch.Tensor):
        key = (i, k.shape[1])
        if self.bulk_bits is not None and k.shape[1] > 64:
            if key not in self.bulk_bits:
                self.bulk_bits[key] = (workloads.to_bits(k), workloads.to_bits(v))
            kb, vb = self.bulk_bits[key]
        else:
            kb, vb = workloads.to_bits(k), workloads.to_bits(v)
        self.k_store[i].append(kb)
        self.v_store[i].append(vb)

    def kv_by_position(self, i: int):
        return self.k_store[i].rows(), self.v_store[i].rows()

    def t_of(self, i: int) -> int:
        return self.oracle.seqs[i].t

    # ---- phases ----------------------------------------------------------------------------
    def bulk_prefill(self, seq_ids: Sequence[int], t0: int, evict: bool = True):
        """Appends prefix + speech + mid + the first t0 output tokens of every listed sequence in
        ONE call (P4: bulk-append-then-evict == step-by-step)."""
        ks, vs, nt = [], [], []
        for i in seq_ids:
            sd = self.data[i]
            kp, vp = sd.prefill_kv()
            ko, vo = sd.out_kv(0, t0)
            k = torch.cat([kp, ko], dim=1)
            v = torch.cat([vp, vo], dim=1)
            ks.append(k)
            vs.append(v)
            nt.append(k.shape[1])
            self._store(i, k, v)
        k_new = torch.cat(ks, dim=1).contiguous()
        v_new = torch.cat(vs, dim=1).contiguous()
        self.gpu.kv_append(seq_ids, nt, k_new, v_new)
        self.oracle.append(seq_ids, nt)
        if evict:
            self.gpu.kv_evict(seq_ids)
            self.oracle.evict(seq_ids)

    def append_step(self, seq_ids: Sequence[int]):
        """One new output token for each listed sequence (both sides)."""
        ks, vs = [], []
        for i in seq_ids:
            u = self.t_of(i)  # index of the token about to be appended
            k, v = self.data[i].out_kv(u, u + 1)
            ks.append(k)
            vs.append(v)
            self._store(i, k, v)
        k_new = torch.cat(ks, dim=1).contiguous()
        v_new = torch.cat(vs, dim=1).contiguous()
        self.gpu.kv_append(seq_ids, [1] * len(seq_ids), k_new, v_new)
        self.oracle.append(seq_ids, [1] * len(seq_ids))

    def evict(self, seq_ids: Sequence[int]):
        self.gpu.kv_evict(seq_ids)
        self.oracle.evict(seq_ids)

    def fused_step(self, seq_ids: Sequence[int], want_lse: bool = False):
        """One whole decode step through murmur_decode_step (prologue = append+evict, attention);
        the oracle side does append -> evict.  Returns (q, out, lse)."""
        ks, vs = [], []
        for i in seq_ids:
            u = self.t_of(i)
            k, v = self.data[i].out_kv(u, u + 1)
            ks.append(k)
            vs.append(v)
            self._store(i, k, v)
        k_new = torch.cat(ks, dim=1).contiguous()
        v_new = torch.cat(vs, dim=1).contiguous()
        self.oracle.append(seq_ids, [1] * len(seq_ids))
        self.oracle.evict(seq_ids)
        q = self.queries(seq_ids)
        out = torch.empty_like(q)
        lse = torch.empty(q.shape[:3], dtype=torch.float32, device=self.device) if want_lse else None
        self.gpu.decode_step(seq_ids, k_new, v_new, q, out, lse, self.scale)
        return q, out, lse

    def per_layer_step(self, seq_ids: Sequence[int], want_lse: bool = False):
        """One decode step issued the way an engine that produces layer l's K/V at layer l would:
        append(layer 0) reserves the slots, evict, attention(layer 0); then for every further layer
        append(layer l) only writes rows, attention(layer l).  The oracle side does append -> evict.
        Returns (q, out, lse) over all layers."""
        ks, vs = [], []
        for i in seq_ids:
            u = self.t_of(i)
            k, v = self.data[i].out_kv(u, u + 1)
            ks.append(k)
            vs.append(v)
            self._store(i, k, v)
        k_new = torch.cat(ks, dim=1).contiguous()  # [L, n_seqs, kv, d]
        v_new = torch.cat(vs, dim=1).contiguous()
        ones = [1] * len(seq_ids)
        self.oracle.append(seq_ids, ones)
        self.oracle.evict(seq_ids)
        q = self.queries(seq_ids)
        out = torch.empty_like(q)
        lse = torch.empty(q.shape[:3], dtype=torch.float32, device=self.device) if want_lse else None
        for l in range(q.shape[0]):
            self.gpu.kv_append(seq_ids, ones, k_new[l:l + 1].contiguous(), v_new[l:l + 1].contiguous(), layer_begin=l, layer_end=l + 1)
            if l == 0:
                self.gpu.kv_evict(seq_ids)
            self.gpu.decode_attn(seq_ids, q[l:l + 1].contiguous(), out=out[l:l + 1], lse=lse[l:l + 1] if want_lse else None,
                                 sm_scale=self.scale, layer_begin=l, layer_end=l + 1)
        return q, out, lse

    def layer_range_step(self, seq_ids: Sequence[int], ranges: Sequence, want_lse: bool = False):
        """One decode step through murmur_decode_step_layers, one call (= one launch) per layer range;
        ranges[0] must start at layer 0 (it opens the step)."""
        ks, vs = [], []
        for i in seq_ids:
            u = self.t_of(i)
            k, v = self.data[i].out_kv(u, u + 1)
            ks.append(k)
            vs.append(v)
            self._store(i, k, v)
        k_new = torch.cat(ks, dim=1).contiguous()
        v_new = torch.cat(vs, dim=1).contiguous()
        self.oracle.append(seq_ids, [1] * len(seq_ids))
        self.oracle.evict(seq_ids)
        q = self.queries(seq_ids)
        out = torch.empty_like(q)
        lse = torch.empty(q.shape[:3], dtype=torch.float32, device=self.device) if want_lse else None
        for a, b in ranges:
            self.gpu.decode_step_layers(seq_ids, k_new[a:b].contiguous(), v_new[a:b].contiguous(), q[a:b].contiguous(),
                                        out[a:b], a, b, lse=lse[a:b] if want_lse else None, sm_scale=self.scale)
        return q, out, lse

    def queries(self, seq_ids: Sequence[int]) -> torch.Tensor:
        """[L, n_seqs, n_q, d]: query of each sequence's newest output token."""
        qs = [self.data[i].q_step(max(1, self.t_of(i))) for i in seq_ids]
        return torch.stack(qs, dim=1).contiguous()

    def attend(self, seq_ids: Sequence[int], want_lse: bool = False):
        q = self.queries(seq_ids)
        lse = None
        if want_lse:
            lse = torch.empty(q.shape[:3], dtype=torch.float32, device=self.device)
        out = self.gpu.decode_attn(seq_ids, q, lse=lse, sm_scale=self.scale)
        return q, out, lse

    # ---- comparisons -----------------------------------------------------------------------
    def check_integer_state(self, seq_ids: Iterable[int], check_free_stack: bool = True):
        for i in seq_ids:
            st = self.gpu.seq_state(i)
            assert st["length"] == self.oracle.seqs[i].length, (i, st)
            assert st["t"] == self.oracle.seqs[i].t, (i, st)
            ret = self.gpu.retained(i)
            want = np.asarray(self.oracle.retained(i), dtype=np.int32)
            assert np.array_equal(ret, want), f"retained set differs for seq {i} at t={st['t']}"
            pages, blocks = self.gpu.page_list(i)
            assert list(blocks) == self.oracle.live_blocks(i), f"live blocks differ for seq {i}"
            assert list(pages) == self.oracle.live_pages(i), f"live pages differ for seq {i}"
            assert self.gpu.runs(i) == self.oracle.runs(i), f"runs differ for seq {i}"
        if check_free_stack:
            fs = self.gpu.free_stack()
            assert list(fs) == self.oracle.free_stack, "free stack differs"
        assert self.gpu.last_error() == 0
        assert self.gpu.stats()["free_pages"] == len(self.oracle.free_stack), "host mirror of free pages is off"

    def check_gather(self, i: int, layers: Optional[Sequence[int]] = (0,)):
        """Rows gathered through the GPU's tables == the rows handed to append (bit-exact); layers=None: all."""
        if layers is None:
            layers = range(self.cfg.geom.n_layers)
        res = sorted(o_policy.resident_positions(*self._regions(i), self.t_of(i), self.oracle.seqs[i].pol))
        res = [x for x in res if x < self.oracle.seqs[i].length]
        kb, vb = self.kv_by_position(i)
        for layer in layers:
            k, v = self.gpu.gather(i, res, layer, layer + 1)
            assert np.array_equal(workloads.to_bits(k)[0], kb[layer][res])
            assert np.array_equal(workloads.to_bits(v)[0], vb[layer][res])

    def _regions(self, i: int):
        s = self.oracle.seqs[i]
        return s.P, s.S, s.M

    def oracle_attend(self, i: int, q_bits_layer: np.ndarray, layer: int):
        kb, vb = self.kv_by_position(i)
        return o_attn.attend_retained(q_bits_layer, kb[layer], vb[layer], self.oracle.retained(i), self.scale)

    def check_attention(self, seq_ids: Sequence[int], q: torch.Tensor, out: torch.Tensor, lse: Optional[torch.Tensor] = None,
                        layers: Optional[Sequence[int]] = None, seq_subset: Optional[Sequence[int]] = None,
                        retained: Optional[Dict[int, Sequence[int]]] = None):
        """Compares out[l, j] with the fp64 oracle for the chosen layers / sequences (default: all of
        them).  retained: the oracle's retained sets as recorded at the step `out` belongs to, when that
        is not the oracle's current step (outputs of earlier steps checked after the fact)."""
        ret_of = (lambda i: retained[i]) if retained is not None else self.oracle.retained
        L = q.shape[0]
        layers = range(L) if layers is None else layers
        got = out_to_f64(out)
        q_bits = workloads.to_bits(q)
        lse_np = lse.cpu().numpy().astype(np.float64) if lse is not None else None
        errs = []
        for j, i in enumerate(seq_ids):
            if seq_subset is not None and i not in seq_subset:
                continue
            if self.use_c_oracle:
                from oracle import c as oc

                kb, vb = self.kv_by_position(i)
                ls = list(layers)
                full = ls == list(range(kb.shape[0]))
                o_all, lse_all, _ = oc.load().attend(q_bits[ls][:, j], kb if full else kb[ls], vb if full else vb[ls],
                                                     ret_of(i), self.scale)
                for a, layer in enumerate(ls):
                    errs.append(np.abs(got[layer, j] - o_all[a]))
                    if lse_np is not None:
                        assert np.max(np.abs(lse_np[layer, j] - lse_all[a])) < 2e-3
            else:
                for layer in layers:
                    kb, vb = self.kv_by_position(i)
                    o_ref, lse_ref, _ = o_attn.attend_retained(q_bits[layer, j], kb[layer], vb[layer], ret_of(i), self.scale)
                    errs.append(np.abs(got[layer, j] - o_ref))
                    if lse_np is not None:
                        assert np.max(np.abs(lse_np[layer, j] - lse_ref)) < 2e-3, "lse mismatch"
        e = np.stack(errs)
        assert np.all(np.isfinite(got)), "non-finite attention output"
        mx, mean = float(e.max()), float(e.mean())
        self.max_abs_seen = max(self.max_abs_seen, mx)
        self.mean_abs_seen = max(self.mean_abs_seen, mean)
        assert mx <= MAX_ABS_TOL, f"max-abs error {mx:.4g} > {MAX_ABS_TOL}"
        assert mean <= MEAN_ABS_TOL, f"mean-abs error {mean:.4g} > {MEAN_ABS_TOL}"
        return mx, mean

    def close(self):
        self.gpu.close()
