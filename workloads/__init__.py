"""Seeded synthetic workloads: the five BASELINE.json configs and their input generators.

This module serves BOTH the oracle-side tests and the CUDA-side tests / bench, so it holds
none of the method's arithmetic: no eviction rule, no page bookkeeping, no attention.  It
only (a) names the shapes and policy parameters of each configuration and (b) draws the
seeded random Q/K/V values, which are handed - the same bits - to both sides.

Stand-ins: the paper measures on AMI-IHM audio with VibeVoice-ASR weights;
neither is available, so these inputs take the paper's *shapes* (300 s chunk ~ 2250 speech
tokens, T up to ~2700 output tokens, 60 min ~ 27000 speech tokens, a batch of concurrent
chunks) with geometry 28 q / 4 KV heads, d = 128, bf16 from
BASELINE.json.  The recipe is restated in DESIGN.md section "Input recipe".

Values: iid N(0,1) rounded to bf16 (round-to-nearest-even); the first 4 prefix keys are
scaled x4 (attention sinks); with ``locality_rho`` > 0 the output keys of each 256-token
output block share a latent direction with the queries issued inside that block
(k_u = sqrt(rho) c_b + sqrt(1-rho) eta_u, q = sqrt(rho) c_b(t) + sqrt(1-rho) eps), so the
attention mass concentrates in the recent window.
Seeds: 1000 * config + sequence index, mixed with a stream id per chunk (see ``_seed``).
"""
from __future__ import annotations

from dataclasses import dataclass, field, replace
from typing import Dict, List, Optional, Tuple

import numpy as np
import torch

WINDOW_OFF = 0x7FFFFFFF  # API sentinel: window >= any length
OUT_BLOCK = 256  # granularity of output-token generation and of the locality latent
N_SINK_KEYS = 4  # first prefix keys scaled x4
SINK_SCALE = 4.0


@dataclass(frozen=True)
class Geometry:
    n_layers: int = 28
    n_q_heads: int = 28
    n_kv_heads: int = 4
    head_dim: int = 128


@dataclass(frozen=True)
class SeqSpec:
    P: int  # prefix system-prompt tokens
    S: int  # speech tokens
    M: int  # second system-prompt tokens
    T: int  # output tokens this sequence decodes
    w_speech: int
    delay: int
    n_sink_speech: int
    w_out: int
    n_sink_out: int

    @property
    def policy_tuple(self) -> Tuple[int, int, int, int, int]:
        return (self.w_speech, self.delay, self.n_sink_speech, self.w_out, self.n_sink_out)


def seq_spec(P, S, T, w_speech, w_out, *, M=0, delay=None, n_sink_speech=0, n_sink_out=4) -> SeqSpec:
    """Defaults where BASELINE.json is silent: k_o = 4 ("s4"), k_s = 0 (Alg. 2 has no
    sinks), d = w_s // 2 (the paper's operating point is d512 / w1024), M = 0."""
    if delay is None:
        delay = 0 if w_speech >= WINDOW_OFF else w_speech // 2
    return SeqSpec(P, S, M, T, w_speech, delay, n_sink_speech, w_out, n_sink_out)


@dataclass(frozen=True)
class Config:
    name: str
    config_id: int
    geom: Geometry
    page_size: int
    seqs: Tuple[SeqSpec, ...]
    locality_rho: float = 0.0
    note: str = ""

    @property
    def batch(self) -> int:
        return len(self.seqs)

    def with_layers(self, n_layers: int) -> "Config":
        return replace(self, geom=replace(self.geom, n_layers=n_layers))

    def with_seqs(self, seqs) -> "Config":
        return replace(self, seqs=tuple(seqs))


# ------------------------------------------------------------------------------------------
# The five configurations of BASELINE.json
# ------------------------------------------------------------------------------------------
def config1() -> Config:
    """Tiny single chunk: 1 layer, 64 + 450 + 128 tokens, w_s 128 / w_o 64; 32 decode steps are run
    from t = 128 (bulk) to t = 160."""
    return Config("tiny_single_chunk", 1, Geometry(n_layers=1), 64,
                  (seq_spec(64, 450, 160, 128, 64),))


def config2(w_speech: int = 512, w_out: int = 256) -> Config:
    """Chunked parallel decode: 12 x 300 s chunks, p = 64, locality-biased keys."""
    return Config("chunked_12x300s", 2, Geometry(), 64,
                  tuple(seq_spec(64, 2250, 1500, w_speech, w_out) for _ in range(12)),
                  locality_rho=0.5)


def config3(evicted: bool) -> Config:
    """Single-pass long context: 1 x 60 min; (a) no eviction, (b) w_s 2048 / w_o 512."""
    if evicted:
        s = seq_spec(64, 27000, 4000, 2048, 512)
    else:
        s = seq_spec(64, 27000, 4000, WINDOW_OFF, WINDOW_OFF)
    return Config("single_pass_60min_" + ("evicted" if evicted else "full"), 3, Geometry(), 64, (s,))


def config4_points() -> List[Tuple[int, int]]:
    """Window sweep over the config-2 shape: (w_speech, w_out); 2250 = no speech eviction."""
    return [(ws, wo) for ws in (128, 256, 512, 1024, 2250) for wo in (64, 256, 1024)]


def config4(w_speech: int, w_out: int) -> Config:
    c = config2(w_speech, w_out)
    return replace(c, name=f"sweep_ws{w_speech}_wo{w_out}", config_id=4)


def config5() -> Config:
    """Ragged mixed batch: 32 sequences, chunk lengths U[60 s, 600 s] (450..4500 speech tokens),
    output counts U[200, 3000], per-sequence windows from {256, 512, 1024}, p = 16."""
    rng = np.random.default_rng(5000)
    S = rng.integers(450, 4501, size=32)
    T = rng.integers(200, 3001, size=32)
    ws = rng.choice([256, 512, 1024], size=32)
    wo = rng.choice([256, 512, 1024], size=32)
    seqs = tuple(seq_spec(64, int(S[i]), int(T[i]), int(ws[i]), int(wo[i])) for i in range(32))
    return Config("ragged_mixed_32", 5, Geometry(), 16, seqs)


ALL_CONFIG_BUILDERS = {
    "config1": config1, "config2": config2, "config3a": lambda: config3(False),
    "config3b": lambda: config3(True), "config5": config5,
}


# ------------------------------------------------------------------------------------------
# Seeded value generators
# ------------------------------------------------------------------------------------------
def _seed(cfg: Config, seq_index: int, stream: int) -> int:
    base = 1000 * cfg.config_id + seq_index
    return (base * 1_000_003 + stream * 7919 + 12345) % (2**63 - 1)


def to_bits(x: torch.Tensor) -> np.ndarray:
    """bf16 tensor -> uint16 numpy bit patterns (host copy)."""
    assert x.dtype == torch.bfloat16
    return x.detach().contiguous().cpu().view(torch.int16).numpy().view(np.uint16)


def from_bits(bits: np.ndarray, device="cpu") -> torch.Tensor:
    return torch.from_numpy(np.ascontiguousarray(bits).view(np.int16)).view(torch.bfloat16).to(device)


class SeqData:
    """Lazily generated, cached, seeded Q/K/V of one sequence of a config.

    Layouts (bf16): K, V ``[n_layers, n_tokens, n_kv_heads, head_dim]``;
    Q ``[n_tokens, n_layers, n_q_heads, head_dim]`` (one query token per decode step).
    """

    def __init__(self, cfg: Config, seq_index: int, device="cpu"):
        self.cfg = cfg
        self.idx = seq_index
        self.spec = cfg.seqs[seq_index]
        self.device = torch.device(device)
        self._chunks: Dict[int, Dict[str, torch.Tensor]] = {}
        self._prefill: Optional[Tuple[torch.Tensor, torch.Tensor]] = None

    def _gen(self, stream: int) -> torch.Generator:
        g = torch.Generator(device=self.device)
        g.manual_seed(_seed(self.cfg, self.idx, stream))
        return g

    def _randn(self, g, *shape) -> torch.Tensor:
        return torch.randn(*shape, generator=g, device=self.device, dtype=torch.float32)

    @property
    def n_prefill(self) -> int:
        return self.spec.P + self.spec.S + self.spec.M

    def prefill_kv(self) -> Tuple[torch.Tensor, torch.Tensor]:
        """K, V of [prefix][speech][mid]; first 4 prefix keys x4."""
        if self._prefill is None:
            ge = self.cfg.geom
            g = self._gen(0)
            n = self.n_prefill
            k = self._randn(g, ge.n_layers, n, ge.n_kv_heads, ge.head_dim)
            v = self._randn(g, ge.n_layers, n, ge.n_kv_heads, ge.head_dim)
            k[:, : min(N_SINK_KEYS, self.spec.P)] *= SINK_SCALE
            self._prefill = (k.to(torch.bfloat16), v.to(torch.bfloat16))
        return self._prefill

    def out_chunk(self, b: int) -> Dict[str, torch.Tensor]:
        """Output tokens u in [256 b, 256 b + 256): their K, V and the queries issued when each is
        the newest token (query of step t belongs to u = t - 1)."""
        if b not in self._chunks:
            ge = self.cfg.geom
            g = self._gen(1 + b)
            rho = self.cfg.locality_rho
            k = self._randn(g, ge.n_layers, OUT_BLOCK, ge.n_kv_heads, ge.head_dim)
            v = self._randn(g, ge.n_layers, OUT_BLOCK, ge.n_kv_heads, ge.head_dim)
            q = self._randn(g, OUT_BLOCK, ge.n_layers, ge.n_q_heads, ge.head_dim)
            if rho > 0.0:
                c = self._randn(g, ge.n_layers, ge.n_kv_heads, ge.head_dim)  # latent of block b
                a, bb = float(np.sqrt(rho)), float(np.sqrt(1.0 - rho))
                k = a * c[:, None, :, :] + bb * k
                G = ge.n_q_heads // ge.n_kv_heads
                cq = c.repeat_interleave(G, dim=1)  # q head h shares the latent of KV head h // G
                q = a * cq[None, :, :, :] + bb * q
            self._chunks = {b: {"k": k.to(torch.bfloat16), "v": v.to(torch.bfloat16), "q": q.to(torch.bfloat16)}}
        return self._chunks[b]

    def out_kv(self, u0: int, u1: int) -> Tuple[torch.Tensor, torch.Tensor]:
        """K, V ``[n_layers, u1-u0, n_kv, d]`` of output tokens u0 <= u < u1."""
        ks, vs = [], []
        u = u0
        while u < u1:
            b = u // OUT_BLOCK
            hi = min(u1, (b + 1) * OUT_BLOCK)
            ch = self.out_chunk(b)
            ks.append(ch["k"][:, u - b * OUT_BLOCK: hi - b * OUT_BLOCK])
            vs.append(ch["v"][:, u - b * OUT_BLOCK: hi - b * OUT_BLOCK])
            u = hi
        if not ks:
            ge = self.cfg.geom
            e = torch.empty(ge.n_layers, 0, ge.n_kv_heads, ge.head_dim, dtype=torch.bfloat16, device=self.device)
            return e, e.clone()
        return torch.cat(ks, dim=1), torch.cat(vs, dim=1)

    def q_step(self, t: int) -> torch.Tensor:
        """Query ``[n_layers, n_q, d]`` of decode step t (newest output token u = t - 1), t >= 1."""
        u = t - 1
        return self.out_chunk(u // OUT_BLOCK)["q"][u % OUT_BLOCK]

    def q_steps(self, t0: int, t1: int) -> torch.Tensor:
        """Queries of steps t0 <= t < t1: ``[t1-t0, n_layers, n_q, d]``."""
        return torch.stack([self.q_step(t) for t in range(t0, t1)], dim=0)


def unevicted_blocks(cfg: Config, extra_tokens: int = 0) -> int:
    """Pages needed to hold every sequence of the config with nothing evicted (pool sizing)."""
    p = cfg.page_size
    return sum(-(-(s.P + s.S + s.M + s.T + extra_tokens) // p) for s in cfg.seqs)


def max_blocks_per_seq(cfg: Config, extra_tokens: int = 0) -> int:
    p = cfg.page_size
    return max(-(-(s.P + s.S + s.M + s.T + extra_tokens) // p) for s in cfg.seqs)
