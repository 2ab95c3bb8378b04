"""Per-layer attention-sparsity report (the analysis of PAPER.md:77-87, Fig. 5) on a synthetic workload.

    python -m paper_2606_01483_b200.sparsity_report [--workload config2] [--seqs 4] [--t 600] [--frac 0.99]

Builds the workload's sequences WITHOUT eviction (windows off), appends the prefill and the first t
output tokens, and runs ``murmur_attn_profile`` for the query of step t with the workload's own
window policy as the candidate.  Prints, per layer (mean over sequences and heads): the share of
speech / text tokens inside the 99 %-mass set ("kept") and outside it ("evictable"), and the
attention mass the candidate policy's retained set preserves ("coverage").  Needs a GPU.
"""
from __future__ import annotations

import argparse
import os
import sys
import time

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def main() -> int:
    import numpy as np
    import torch

    import workloads
    from paper_2606_01483_b200 import MURMUR_WINDOW_OFF, MurmurCache

    ap = argparse.ArgumentParser()
    ap.add_argument("--workload", default="config2", choices=sorted(workloads.ALL_CONFIG_BUILDERS))
    ap.add_argument("--seqs", type=int, default=4)
    ap.add_argument("--t", type=int, default=600)
    ap.add_argument("--frac", type=float, default=0.99)
    args = ap.parse_args()
    if not torch.cuda.is_available():
        raise SystemExit("sparsity_report: no CUDA device")
    dev = torch.device("cuda:0")
    cfg = workloads.ALL_CONFIG_BUILDERS[args.workload]()
    n = min(args.seqs, cfg.batch)
    cfg = cfg.with_seqs(cfg.seqs[:n])
    g = cfg.geom
    blocks = max(-(-(s.P + s.S + s.M + args.t) // cfg.page_size) for s in cfg.seqs) + 1
    cache = MurmurCache(g.n_layers, g.n_q_heads, g.n_kv_heads, g.head_dim, cfg.page_size, n, blocks, n * blocks + 2, device=dev)
    qs = []
    for i, s in enumerate(cfg.seqs):
        cache.seq_begin(i, s.P, s.S, s.M, (MURMUR_WINDOW_OFF, 0, 0, MURMUR_WINDOW_OFF, 0))
        d = workloads.SeqData(cfg, i, device=dev)
        kp, vp = d.prefill_kv()
        ko, vo = d.out_kv(0, args.t)
        k = torch.cat([kp, ko], dim=1).contiguous()
        v = torch.cat([vp, vo], dim=1).contiguous()
        cache.kv_append([i], [k.shape[1]], k, v)
        qs.append(d.q_step(args.t))
    q = torch.stack(qs, dim=1).contiguous()
    ids = list(range(n))
    cand = cfg.seqs[0].policy_tuple
    cache.attn_profile(ids, q, candidate=cand, mass_frac=args.frac)  # warm-up
    t0 = time.perf_counter()
    pr = cache.attn_profile(ids, q, candidate=cand, mass_frac=args.frac)
    dt = time.perf_counter() - t0
    s0 = cfg.seqs[0]
    print(f"# {cfg.name}: {n} sequences x {g.n_layers} layers x {g.n_q_heads} heads, P={s0.P} S={s0.S} t={args.t}, "
          f"mass fraction {args.frac}, candidate policy (w_s, d, k_s, w_o, k_o) = {cand}")
    print(f"# murmur_attn_profile: {dt * 1e3:.2f} ms for {pr.size} (layer, sequence, head) profiles")
    print("| layer | kept speech % | evictable speech % | kept text % | evictable text % | speech tokens in the mass set % | coverage of the candidate window % |")
    print("|---|---|---|---|---|---|---|")
    for layer in range(g.n_layers):
        p = pr[layer]
        tot = (p["n_speech"] + p["n_text"]).astype(np.float64)
        ks, kt = p["k_speech"] / tot, p["k_text"] / tot
        es, et = (p["n_speech"] - p["k_speech"]) / tot, (p["n_text"] - p["k_text"]) / tot
        print("| %d | %.1f | %.1f | %.1f | %.1f | %.1f | %.1f |" % (
            layer, 100 * ks.mean(), 100 * es.mean(), 100 * kt.mean(), 100 * et.mean(),
            100 * (p["k_speech"] / np.maximum(p["n_speech"], 1)).mean(), 100 * p["coverage"].mean()))
    cache.close()
    return 0


if __name__ == "__main__":
    sys.exit(main())
