"""Plain-integer simulation of the paged KV-cache bookkeeping (oracle).

TEST INFRASTRUCTURE - see ``oracle/__init__.py``.

The paper gives no cache layout ("custom KV cache management"); it only
says that eviction happens at every decode step and that managing it
costs time.  The canonical, history-free bookkeeping simulated here is
reading C2/C3 of DESIGN.md:

C2  position-paged, tokens never move: absolute position x lives in logical block
    x // p, slot x % p.  ``block_table[blk]`` is a physical page id or -1.  A block is
    *dead* iff it is allocated, completely filled ((blk+1)*p <= len) and every position in
    it is dead under the policy; evict frees dead blocks.  ``live_blocks`` / ``live_pages``
    list the allocated blocks in ascending logical order (the compacted page table).
    ``runs`` are the maximal intervals of A(t): (first_pos, n_tok, index of the interval's
    first block in live_blocks).
C3  deterministic allocator: ``free_stack[i] = N-1-i`` initially, pop from the top (so
    pops return 0,1,2,...); append walks the sequences of a call in order and, per
    sequence, new logical blocks ascending; if the call as a whole needs more pages than
    are free nothing changes and OutOfPages is raised; evict walks the sequences in call
    order and pushes dead blocks ascending; seq_end pushes the live blocks ascending.

Everything is Python ints and lists: no vectorisation, no shared code with the CUDA path.
"""
from __future__ import annotations

from dataclasses import dataclass, field
from typing import Dict, List, Sequence, Tuple

from . import policy as _pol


class OutOfPages(Exception):
    pass


class BadState(Exception):
    pass


@dataclass
class SeqState:
    P: int
    S: int
    M: int
    pol: _pol.Policy
    length: int = 0  # tokens appended so far (positions 0..length-1 exist)
    block_table: List[int] = field(default_factory=list)  # logical block -> page id / -1

    @property
    def t(self) -> int:
        """Output tokens in the cache, including the newest (0 while prefilling)."""
        return max(0, self.length - (self.P + self.S + self.M))


class OraclePagedCache:
    def __init__(self, n_pages: int, page_size: int, max_seqs: int, max_blocks_per_seq: int):
        if page_size <= 0 or n_pages < 0:
            raise ValueError("bad geometry")
        self.N = n_pages
        self.p = page_size
        self.max_seqs = max_seqs
        self.max_blocks_per_seq = max_blocks_per_seq
        self.free_stack: List[int] = [n_pages - 1 - i for i in range(n_pages)]
        self.seqs: Dict[int, SeqState] = {}

    # ---- lifecycle -----------------------------------------------------------------
    def seq_begin(self, seq: int, P: int, S: int, M: int, pol: _pol.Policy) -> None:
        if not (0 <= seq < self.max_seqs) or seq in self.seqs:
            raise BadState(f"seq {seq} out of range or already active")
        if min(P, S, M) < 0:
            raise ValueError("negative region size")
        self.seqs[seq] = SeqState(P, S, M, pol)

    def seq_end(self, seq: int) -> None:
        st = self._get(seq)
        for blk, page in enumerate(st.block_table):  # live blocks ascending
            if page >= 0:
                self.free_stack.append(page)
        del self.seqs[seq]

    def _get(self, seq: int) -> SeqState:
        if seq not in self.seqs:
            raise BadState(f"seq {seq} not active")
        return self.seqs[seq]

    # ---- append (C3) ----------------------------------------------------------------
    def blocks_needed(self, seq_ids: Sequence[int], n_tokens: Sequence[int]) -> int:
        need = 0
        for s, n in zip(seq_ids, n_tokens):
            st = self._get(s)
            new_len = st.length + n
            need += -(-new_len // self.p) - (-(-st.length // self.p))
        return need

    def append(self, seq_ids: Sequence[int], n_tokens: Sequence[int]) -> List[List[int]]:
        """Reserve slots for n_tokens[i] new tokens of seq_ids[i].  Returns, per sequence,
        the absolute positions the new tokens occupy.  All-or-nothing on page exhaustion."""
        if len(set(seq_ids)) != len(seq_ids):
            raise BadState("duplicate sequence in one call")
        for s, n in zip(seq_ids, n_tokens):
            st = self._get(s)
            if n < 0:
                raise ValueError("negative token count")
            if -(-(st.length + n) // self.p) > self.max_blocks_per_seq:
                raise BadState("max_blocks_per_seq exceeded")
        if self.blocks_needed(seq_ids, n_tokens) > len(self.free_stack):
            raise OutOfPages()
        positions: List[List[int]] = []
        for s, n in zip(seq_ids, n_tokens):  # sequences in call order
            st = self.seqs[s]
            first_new_blk = -(-st.length // self.p)
            new_len = st.length + n
            last_blk_excl = -(-new_len // self.p)
            for blk in range(first_new_blk, last_blk_excl):  # new blocks ascending
                assert blk == len(st.block_table)
                st.block_table.append(self.free_stack.pop())
            positions.append(list(range(st.length, new_len)))
            st.length = new_len
        return positions

    # ---- policy views -----------------------------------------------------------------
    def retained(self, seq: int) -> List[int]:
        """A(t) restricted to the positions that exist."""
        st = self._get(seq)
        return [x for x in _pol.retained_positions(st.P, st.S, st.M, st.t, st.pol) if x < st.length]

    def _dead_set(self, st: SeqState) -> set:
        return {x for x in _pol.dead_positions(st.P, st.S, st.M, st.t, st.pol) if x < st.length}

    # ---- evict (C2/C3) ------------------------------------------------------------------
    def evict(self, seq_ids: Sequence[int]) -> None:
        if len(set(seq_ids)) != len(seq_ids):
            raise BadState("duplicate sequence in one call")
        for s in seq_ids:  # sequences in call order
            st = self._get(s)
            dead = self._dead_set(st)
            for blk, page in enumerate(st.block_table):  # dead blocks ascending
                if page < 0:
                    continue
                lo, hi = blk * self.p, (blk + 1) * self.p
                if hi <= st.length and all(x in dead for x in range(lo, hi)):
                    self.free_stack.append(page)
                    st.block_table[blk] = -1

    # ---- compacted tables ---------------------------------------------------------------
    def live_blocks(self, seq: int) -> List[int]:
        return [b for b, pg in enumerate(self._get(seq).block_table) if pg >= 0]

    def live_pages(self, seq: int) -> List[int]:
        return [pg for pg in self._get(seq).block_table if pg >= 0]

    def runs(self, seq: int) -> List[Tuple[int, int, int]]:
        """Maximal intervals of A(t): (first_pos, n_tok, index of first block in live_blocks)."""
        pos = self.retained(seq)
        lb = self.live_blocks(seq)
        out: List[Tuple[int, int, int]] = []
        i = 0
        while i < len(pos):
            j = i
            while j + 1 < len(pos) and pos[j + 1] == pos[j] + 1:
                j += 1
            out.append((pos[i], j - i + 1, lb.index(pos[i] // self.p)))
            i = j + 1
        return out

    def slot_of(self, seq: int, x: int) -> Tuple[int, int]:
        """(physical page, slot) holding absolute position x; raises if x was evicted."""
        st = self._get(seq)
        page = st.block_table[x // self.p]
        if page < 0:
            raise BadState(f"position {x} is in a freed block")
        return page, x % self.p

    # ---- invariants (P6) ------------------------------------------------------------------
    def check_invariants(self) -> None:
        used: List[int] = []
        for st in self.seqs.values():
            used.extend(pg for pg in st.block_table if pg >= 0)
        assert len(used) == len(set(used)), "physical page referenced twice"
        assert not (set(used) & set(self.free_stack)), "page both live and free"
        assert len(set(self.free_stack)) == len(self.free_stack), "page twice on the free stack"
        assert len(used) + len(self.free_stack) == self.N, "page conservation violated"
