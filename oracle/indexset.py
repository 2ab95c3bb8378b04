"""General index-set eviction with dense stable compaction (oracle).

TEST INFRASTRUCTURE - see ``oracle/__init__.py``.

PAPER.md:224 (Discussion): "the evictable tokens are not contiguous and cannot be captured by a simple
positional policy. This motivates future work on adaptive speech token selection strategies, such as
query-aware ... eviction policies"; the sparsity the paper measures differs by layer ("on 24 of
28 layers"; "particularly in deeper layers") and is a per-head quantity (Fig. 5).
The paper defines no such policy or cache layout, so everything below except Eq. 1 is a CONVENTION of this
build ("f3"): parity unpinned against the paper, pinned against the properties listed in
tests/test_oracle_indexset.py.

Definitions
  index set      per (layer l, KV head h): an ascending list sel[l][h] of ORIGINAL absolute positions to keep.
  indexed mode   a sequence whose rows are stored DENSELY per (l, h): slot s of slab (l, h) holds the row of
                 the s-th smallest retained position  pos[l][h][s]  ("dense stable defrag": order preserved).
                 Slab lengths differ by (l, h) (a head-ragged cache).
  evict_indexed  sel[l][h] must be a subset of what slab (l, h) holds.  Afterwards pos[l][h] = sel[l][h] and
                 slot s holds the row that position sel[l][h][s] had before; every other row is gone.
  pages          one page id still addresses the same logical block in every layer and head (reading C2), so a
                 sequence keeps the blocks 0 .. ceil(max_lh len(l,h) / p) - 1.  Entering indexed mode re-uses the
                 sequence's LIVE pages in ascending logical-block order as blocks 0, 1, ...; surplus pages are
                 pushed on the free stack in that order (reading C3).  Later evictions free the trailing blocks,
                 ascending.
  append_indexed the next token (absolute position next_pos) is appended to EVERY slab, at slot len(l,h); a page
                 is popped when the longest slab crosses a block boundary (call order, as in C3).
  attention      Eq. 1 of query head hq over the rows of slab (l, hq // G).
  bytes moved    rows that change their (block, slot) address x 2 (K and V) x 256 bytes: the "cache management
                 overhead" of PAPER.md:154, 214 made countable.
  mass sets      a producer of query-aware sets from the quantity the paper measures (Fig. 5): per
                 (l, h) the union over the G query heads of the group of each head's fewest-token set holding
                 >= frac of its Eq. 1 mass (oracle.sparsity.mass_set_indices), plus both system prompts (never
                 evicted) and the n_recent newest positions.
"""
from __future__ import annotations

from typing import Dict, List, Sequence, Tuple

import numpy as np

from . import paged_cache as _pc
from . import sparsity as _sp
from .attention import bf16_bits_to_f64, softmax_weights


class IndexedSeq:
    def __init__(self, n_layers: int, n_kv: int, pos: List[List[List[int]]], blocks: List[int], next_pos: int):
        self.n_layers, self.n_kv = n_layers, n_kv
        self.pos = pos          # pos[l][h]: ascending original positions, by slot
        self.blocks = blocks    # page id of logical block 0, 1, ...
        self.next_pos = next_pos

    def max_len(self) -> int:
        return max(len(self.pos[l][h]) for l in range(self.n_layers) for h in range(self.n_kv))


def _check_sets(sel, n_layers: int, n_kv: int):
    if len(sel) != n_layers or any(len(sel[l]) != n_kv for l in range(n_layers)):
        raise ValueError("index sets must be given for every (layer, KV head)")
    for l in range(n_layers):
        for h in range(n_kv):
            s = list(sel[l][h])
            if any(s[i] >= s[i + 1] for i in range(len(s) - 1)):
                raise ValueError("an index set must be strictly ascending")


class OracleIndexedCache:
    """Indexed-mode bookkeeping on top of an ``OraclePagedCache`` (they share the free stack)."""

    def __init__(self, paged: _pc.OraclePagedCache, n_layers: int, n_kv: int):
        self.pc = paged
        self.p = paged.p
        self.n_layers, self.n_kv = n_layers, n_kv
        self.seqs: Dict[int, IndexedSeq] = {}

    # ---- entering indexed mode / evicting --------------------------------------------------------
    def evict_indexed(self, seq: int, sel) -> int:
        """Applies the index sets; returns the number of rows that changed address (per K or V pool)."""
        _check_sets(sel, self.n_layers, self.n_kv)
        sel = [[list(int(x) for x in sel[l][h]) for h in range(self.n_kv)] for l in range(self.n_layers)]
        p = self.p
        if seq not in self.seqs:
            st = self.pc._get(seq)  # positional sequence: must be evicted up to date (its live list is the source)
            resident = set(_pc._pol.resident_positions(st.P, st.S, st.M, st.t, st.pol))
            live = self.pc.live_blocks(seq)
            pages = self.pc.live_pages(seq)
            rank = {b: k for k, b in enumerate(live)}  # logical block -> index in the live list

            def old_addr(x: int) -> Tuple[int, int]:
                return rank[x // p], x % p

            for l in range(self.n_layers):
                for h in range(self.n_kv):
                    for x in sel[l][h]:
                        if not (0 <= x < st.length) or x not in resident or (x // p) not in rank:
                            raise _pc.BadState(f"position {x} is not resident")
            blocks = list(pages)
            next_pos = st.length
            del self.pc.seqs[seq]  # the positional bookkeeping ends here; its pages live on in `blocks`
        else:
            cur = self.seqs[seq]
            slot_of = [[{x: s for s, x in enumerate(cur.pos[l][h])} for h in range(self.n_kv)] for l in range(self.n_layers)]
            for l in range(self.n_layers):
                for h in range(self.n_kv):
                    for x in sel[l][h]:
                        if x not in slot_of[l][h]:
                            raise _pc.BadState(f"position {x} is not held by slab ({l}, {h})")
            blocks = list(cur.blocks)
            next_pos = cur.next_pos
            old_addr = None
        moved = 0
        for l in range(self.n_layers):
            for h in range(self.n_kv):
                for s, x in enumerate(sel[l][h]):
                    a = old_addr(x) if old_addr is not None else divmod(slot_of[l][h][x], p)
                    if a != (s // p, s % p):
                        moved += 1
        new = IndexedSeq(self.n_layers, self.n_kv, sel, blocks, next_pos)
        need = -(-new.max_len() // p)
        for page in blocks[need:]:  # surplus blocks, ascending
            self.pc.free_stack.append(page)
        new.blocks = blocks[:need]
        self.seqs[seq] = new
        return moved

    # ---- append ------------------------------------------------------------------------------------
    def append_indexed(self, seq_ids: Sequence[int]) -> None:
        if len(set(seq_ids)) != len(seq_ids):
            raise _pc.BadState("duplicate sequence in one call")
        need = 0
        for s in seq_ids:
            st = self.seqs[s]
            need += -(-(st.max_len() + 1) // self.p) - len(st.blocks)
        if need > len(self.pc.free_stack):
            raise _pc.OutOfPages()
        for s in seq_ids:  # call order
            st = self.seqs[s]
            while -(-(st.max_len() + 1) // self.p) > len(st.blocks):
                st.blocks.append(self.pc.free_stack.pop())
            for l in range(self.n_layers):
                for h in range(self.n_kv):
                    st.pos[l][h].append(st.next_pos)
            st.next_pos += 1

    def seq_end(self, seq: int) -> None:
        for page in self.seqs[seq].blocks:
            self.pc.free_stack.append(page)
        del self.seqs[seq]

    # ---- views -------------------------------------------------------------------------------------
    def positions(self, seq: int, l: int, h: int) -> List[int]:
        return list(self.seqs[seq].pos[l][h])

    def check_invariants(self) -> None:
        used = [pg for st in self.seqs.values() for pg in st.blocks]
        used += [pg for st in self.pc.seqs.values() for pg in st.block_table if pg >= 0]
        assert len(used) == len(set(used)), "physical page referenced twice"
        assert not (set(used) & set(self.pc.free_stack)), "page both live and free"
        assert len(used) + len(self.pc.free_stack) == self.pc.N, "page conservation violated"


def attend_indexed(q_bits: np.ndarray, k_bits: np.ndarray, v_bits: np.ndarray, pos_lh: Sequence[Sequence[int]], scale: float
                   ) -> Tuple[np.ndarray, np.ndarray]:
    """One layer.  q_bits [n_q, d]; k_bits, v_bits [n_pos, n_kv, d] by ORIGINAL position; pos_lh[h] = positions of
    slab h.  Eq. 1 of query head hq over the rows of slab hq // G.  Returns (o [n_q, d], lse [n_q]) in fp64."""
    n_q, d = q_bits.shape
    n_kv = k_bits.shape[1]
    G = n_q // n_kv
    q = bf16_bits_to_f64(q_bits)
    o = np.empty((n_q, d), dtype=np.float64)
    lse = np.empty((n_q,), dtype=np.float64)
    for hq in range(n_q):
        h = hq // G
        idx = np.asarray(list(pos_lh[h]), dtype=np.int64)
        if idx.size == 0:
            raise ValueError("attention over an empty slab is undefined")
        k = bf16_bits_to_f64(k_bits[idx, h])
        v = bf16_bits_to_f64(v_bits[idx, h])
        s = (k @ q[hq]) * scale
        a = softmax_weights(s)
        o[hq] = a @ v
        m = np.max(s)
        lse[hq] = m + np.log(np.sum(np.exp(s - m)))
    return o, lse


def select_mass_sets(q_bits: np.ndarray, k_bits: np.ndarray, resident: Sequence[int], P: int, S: int, M: int, length: int,
                     scale: float, frac: float, n_recent: int) -> List[List[int]]:
    """One layer.  q_bits [n_q, d], k_bits [n_pos, n_kv, d].  Returns sel[h] (ascending) per KV head: union over the
    group's query heads of their fewest-token >= frac mass sets over `resident`, plus both system prompts and the
    n_recent newest positions (all restricted to `resident`)."""
    n_q = q_bits.shape[0]
    n_kv = k_bits.shape[1]
    G = n_q // n_kv
    res = sorted(int(x) for x in resident)
    res_set = set(res)
    always = {x for x in res if x < P or P + S <= x < P + S + M or x >= length - n_recent}
    out: List[List[int]] = []
    for h in range(n_kv):
        keep = set(always)
        k = bf16_bits_to_f64(k_bits[np.asarray(res, dtype=np.int64), h])
        for g in range(G):
            q = bf16_bits_to_f64(q_bits[h * G + g])
            alpha = softmax_weights((k @ q) * scale)
            keep.update(res[i] for i in _sp.mass_set_indices(alpha, frac))
        out.append(sorted(keep & res_set))
    return out
