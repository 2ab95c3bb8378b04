#!/usr/bin/env python
"""bench.py - decode-attention us/step and HBM GB/s on the 12 x 300 s-chunk evicted-KV workload.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl murmur|reference] [--workload NAME]

A *step* is one pass of the whole hot path over one batch of synthetic input:
``murmur_decode_step`` = append one token per sequence (all 28 layers) -> evict -> decode attention
(all 28 layers), ONE kernel launch per step.  Prints ONE JSON line (rank 0).

Timed regions (CUDA events on the stream the kernels are launched on, W >= 3 warm-up steps,
barrier + synchronize on both sides, max over ranks):
  A  K consecutive steps, inputs resident in HBM, each followed by a one-element kernel that makes the next
     step's q depend on this step's out (what an autoregressive loop has between two steps, at its smallest:
     consecutive step launches cannot overlap)                            -> value, ms_per_step, roofline
  A2 K more steps with nothing in between (chained launches overlap one step's tail with the next step's
     stream - possible only because the bench has all inputs in advance)  -> chained_back_to_back_us (secondary)
  B  K more steps with one event pair around every launch                 -> isolated launch duration;
     then <= 100 steps as three separate API calls (append, evict, attention), one event pair each
  P  <= 50 steps issued layer by layer from C (murmur_decode_step_chunked, 28 launches per step)
                                                                         -> per_layer_mode_us
  C  K_e steps through murmur_decode_step_host from pinned HOST buffers, stream-synchronised
     every step (the caller reads `out`)                                  -> e2e
Every step re-reads ~575 MB of retained K/V (>> 126 MB L2), so inputs are larger than L2 and no
explicit flush is needed; t advances every step, so windows slide and pages are freed/reused.

Checks against the oracle (rank 0, N = 1; all outside the timed regions; SURVEY.md 8(d) "Protocol"):
  parity    the outputs the TIMED launches produced - region A's last `out` (murmur_decode_step) and
            region C's last host `out` (murmur_decode_step_host) - compared with the fp64 oracle for
            every (sequence, layer, head); integer state of every sequence after region A bit-exact
  replay    region A re-run on a second cache from the same seeded inputs, integer state compared
            with the oracle at EVERY step; its last output must equal region A's bit for bit
  protocol  the whole decode t = 1..T on a third cache; full-tensor attention check at the steps
            {1, 2, k_o+w_o, k_o+w_o+1, d, d+1, d+2, T/2, T-1, T}, retained sets at those steps
  cpu_baseline  the same oracle (policy + plain-C fp64 attention) timed on the host cores
  other_workloads  configs 3a, 3b, 5 and two sweep points: us/step, roofline fraction, clocks, oracle check

Multi-GPU: the path has no exchange step: "replicas only".  Under torchrun every
rank runs an independent replica of the workload on its own GPU; time = max over ranks.

`--impl reference` times the oracle itself (oracle/: Python integer bookkeeping + plain-C fp64
attention) on the host cores, each step a bounded sample of the same workload.
"""
from __future__ import annotations

import argparse
import hashlib
import json
import math
import os
import subprocess
import sys
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "decode-attn us/step (whole step: append+evict+attn), 12x300s chunks, evicted KV"
UNIT = "us/step"
BYTES_PER_TOKEN_LAYER = 4 * 128 * 2 * 2  # 4 KV heads x 128 x bf16 x {K, V}
HBM_FALLBACK_GBS = 6650.0  # /opt/skills/guides/B200_PROFILING.md fallback when MEASURED_PEAKS.json is absent
OTHER_WORKLOADS = ["config3a", "config3b", "config5", "sweep_128_64", "sweep_2250_1024"]
# sources whose change invalidates an ncu traffic capture of the step kernel (profiles/traffic.md)
KERNEL_SOURCES = ["decode_attn_mma.cu", "evict_body.cuh", "device_state.cuh", "policy_math.cuh", "ptx_utils.cuh"]
# ... and of the prefill kernel (workload prefill_300s)
PREFILL_SOURCES = ["prefill_attn_umma.cu", "umma_utils.cuh", "ptx_utils.cuh"]


def kernel_source_hash(sources=None) -> str:
    h = hashlib.sha256()
    for f in (sources or KERNEL_SOURCES):
        with open(os.path.join(ROOT, "paper_2606_01483_b200", "csrc", f), "rb") as fh:
            h.update(fh.read())
    return h.hexdigest()[:16]


def ncu_traffic_bytes(workload: str, sources=None):
    """dram__bytes_read.sum + dram__bytes_write.sum of ONE launch of the dominant kernel from the committed
    `ncu --set full` capture (profiles/traffic.md), or None when there is no capture for this workload or
    the kernel sources have changed since it was taken (the row carries their hash)."""
    try:
        with open(os.path.join(ROOT, "profiles", "traffic.md")) as f:
            for ln in f:
                if not (ln.startswith("| `") and ln.count("|") >= 5):
                    continue
                c = [x.strip() for x in ln.strip().strip("|").split("|")]
                if c[0].strip("`") == workload and c[2].strip("`") == kernel_source_hash(sources):
                    return float(c[1])
    except (OSError, ValueError, IndexError):
        pass
    return None


# ------------------------------------------------------------------------------------------------
# clock sampler (separate process: NVML polled every few ms, so that the short timed regions
# still get samples; nvidia-smi -lms cannot go that fast)
# ------------------------------------------------------------------------------------------------
SAMPLER_SRC = r"""
import sys, time
import pynvml as nv
nv.nvmlInit()
h = nv.nvmlDeviceGetHandleByIndex(int(sys.argv[1]))
try:
    reasons = nv.nvmlDeviceGetCurrentClocksEventReasons
except AttributeError:
    reasons = nv.nvmlDeviceGetCurrentClocksThrottleReasons
mx = nv.nvmlDeviceGetMaxClockInfo(h, nv.NVML_CLOCK_SM)
out = open(sys.argv[2], "w")
while True:
    try:
        sm = nv.nvmlDeviceGetClockInfo(h, nv.NVML_CLOCK_SM)
        r = reasons(h)
        try:
            pw = nv.nvmlDeviceGetPowerUsage(h) / 1000.0
        except Exception:
            pw = -1.0
        out.write("%.6f %d %d %d %.1f\n" % (time.time(), sm, mx, r, pw))
        out.flush()
    except Exception as e:
        out.write("# %r\n" % (e,))
        out.flush()
    time.sleep(0.004)
"""
REASON_BITS = {0x1: "gpu_idle", 0x2: "applications_clocks_setting", 0x4: "sw_power_cap", 0x8: "hw_slowdown",
               0x10: "sync_boost", 0x20: "sw_thermal_slowdown", 0x40: "hw_thermal_slowdown",
               0x80: "hw_power_brake_slowdown", 0x100: "display_clock_setting"}


class ClockSampler:
    def __init__(self, dev_index: int):
        self.path = f"/tmp/murmur_clocks_{os.getpid()}.txt"
        self.windows = {}
        self.proc = None
        try:
            self.proc = subprocess.Popen([sys.executable, "-c", SAMPLER_SRC, str(dev_index), self.path],
                                         stdout=subprocess.DEVNULL, stderr=subprocess.DEVNULL)
        except Exception:
            self.proc = None

    def wait_ready(self, timeout_s: float = 3.0):
        """Blocks until the sampler process has written its first sample (it takes ~0.1-0.5 s to start)."""
        t_end = time.time() + timeout_s
        while self.proc is not None and time.time() < t_end:
            try:
                if os.path.getsize(self.path) > 0:
                    return
            except OSError:
                pass
            time.sleep(0.01)

    def window(self, t0: float, t1: float, tag: str = "main"):
        self.windows.setdefault(tag, []).append((t0, t1))

    def finish(self) -> dict:
        """{tag: summary of the samples that fell inside that tag's timed regions}."""
        if self.proc is None:
            return {}
        time.sleep(0.02)
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except Exception:
            self.proc.kill()
        rows = []
        try:
            with open(self.path) as f:
                for ln in f:
                    if ln.startswith("#"):
                        continue
                    p = ln.split()
                    if len(p) == 5:
                        rows.append((float(p[0]), int(p[1]), int(p[2]), int(p[3]), float(p[4])))
            os.unlink(self.path)
        except OSError:
            pass
        out = {}
        for tag, wins in self.windows.items():
            under = [r for r in rows if any(a <= r[0] <= b for a, b in wins)]
            if not under:
                out[tag] = {"sm_mhz": None, "sm_max_mhz": rows[0][2] if rows else None, "reasons": [], "samples": 0,
                            "note": "no sample fell inside a timed region"}
                continue
            sms = sorted(r[1] for r in under)
            mask = 0
            for r in under:
                mask |= r[3]
            reasons = [name for bit, name in REASON_BITS.items() if mask & bit and name != "gpu_idle"]
            out[tag] = {"sm_mhz": sms[len(sms) // 2], "sm_min_mhz": sms[0], "sm_max_mhz": under[0][2], "reasons": reasons,
                        "samples": len(under), "power_w_max": max(r[4] for r in under), "how": "NVML polled every ~4 ms"}
        return out


# ------------------------------------------------------------------------------------------------
def max_over_ranks(values, dist, device):
    """MAX over ranks of a list of floats (every timing is reported as the slowest rank's); identity
    when dist is None.  Works with any torch.distributed backend (nccl on the GPUs, gloo in the CPU test)."""
    import torch

    t = torch.tensor(list(values), dtype=torch.float64, device=device)
    if dist is not None:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return [float(x) for x in t.tolist()]


def whole_job_tokens_per_s(world: int, batch_per_rank: int, us_step: float) -> float:
    """Replicas only: every rank decodes its own batch, one token per sequence
    per step; the job's throughput is all ranks' tokens over the slowest rank's step time."""
    return world * batch_per_rank / (us_step * 1e-6)


def pick_workload(name: str):
    import workloads

    if name == "config2":
        return workloads.config2(), 300
    if name == "config3a":
        return workloads.config3(False), 1030
    if name == "config3b":
        return workloads.config3(True), 1030
    if name == "config5":  # the full-batch point: all 32 sequences active (windows already sliding for most)
        return workloads.config5(), 700
    if name.startswith("sweep_"):  # sweep_<w_s>_<w_o>
        _, ws, wo = name.split("_")
        return workloads.config4(int(ws), int(wo)), 1100
    raise SystemExit(f"unknown workload {name}")


def config_keys(cfg, world: int = 1) -> dict:
    """The workload description both arms print under `config` (same keys, same values)."""
    g = cfg.geom
    d = {"workload": cfg.name, "batch": cfg.batch, "n_layers": g.n_layers, "n_q_heads": g.n_q_heads,
         "n_kv_heads": g.n_kv_heads, "head_dim": g.head_dim, "page_size": cfg.page_size,
         "parallelism": "replicas only" if world > 1 else "single GPU"}
    s0 = cfg.seqs[0]
    if len({(x.S, x.w_speech, x.w_out) for x in cfg.seqs}) == 1:
        d.update({"speech_tokens": s0.S, "prefix_tokens": s0.P, "w_speech": s0.w_speech, "w_out": s0.w_out,
                  "delay": s0.delay, "n_sink_out": s0.n_sink_out})
    else:
        d.update({"ragged": True, "speech_tokens": [min(x.S for x in cfg.seqs), max(x.S for x in cfg.seqs)],
                  "prefix_tokens": s0.P, "w_speech": sorted({x.w_speech for x in cfg.seqs}),
                  "w_out": sorted({x.w_out for x in cfg.seqs}), "n_sink_out": s0.n_sink_out,
                  "note": "all sequences kept active at a common t (the full-batch point of config 5)"})
    return d


def load_peak():
    try:
        with open(os.path.join(ROOT, "MEASURED_PEAKS.json")) as f:
            pk = json.load(f)
        return float(pk["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs, torch copy)"
    except Exception:
        return HBM_FALLBACK_GBS, "fallback (B200_PROFILING.md 6.65 TB/s)"


# ------------------------------------------------------------------------------------------------
# reference arm: the oracle, as it stands, on the host cores
# ------------------------------------------------------------------------------------------------
def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return 0
    import numpy as np

    import workloads
    from oracle import c as oracle_c
    from oracle import paged_cache as o_cache
    from oracle import policy as o_policy

    cfg, t0 = pick_workload(args.workload)
    g = cfg.geom
    co = oracle_c.load()
    K, W = args.steps, args.warmup
    n_items_step = cfg.batch * g.n_layers  # (sequence, layer) items of one step
    budget_s = float(args.ref_budget_s)
    # data of sequence 0 only (the sample never leaves it): CPU generator, same recipe
    sd = workloads.SeqData(cfg, 0, device="cpu")
    kp, vp = sd.prefill_kv()
    ko, vo = sd.out_kv(0, t0 + K + W + 2)
    k_bits = np.concatenate([workloads.to_bits(kp), workloads.to_bits(ko)], axis=1)
    v_bits = np.concatenate([workloads.to_bits(vp), workloads.to_bits(vo)], axis=1)
    n_pages = workloads.unevicted_blocks(cfg, 2) + 2
    oc = o_cache.OraclePagedCache(n_pages, cfg.page_size, cfg.batch, workloads.max_blocks_per_seq(cfg, 2) + 1)
    ids = list(range(cfg.batch))
    for i, s in enumerate(cfg.seqs):
        oc.seq_begin(i, s.P, s.S, s.M, o_policy.Policy(*s.policy_tuple))
    oc.append(ids, [s.P + s.S + s.M + t0 for s in cfg.seqs])
    oc.evict(ids)
    scale = 1.0 / math.sqrt(g.head_dim)

    def step(n_layers_sample: int):
        oc.append(ids, [1] * len(ids))
        oc.evict(ids)
        ret = oc.retained(0)
        t = oc.seqs[0].t
        q = workloads.to_bits(sd.q_step(t))[:n_layers_sample]
        _, _, used = co.attend(q, k_bits[:n_layers_sample], v_bits[:n_layers_sample], ret, scale)
        return used

    # calibrate: one layer of sequence 0
    tc = time.perf_counter()
    used = step(1)
    per_item = max(time.perf_counter() - tc, 1e-4)
    n_sample = int(max(1, min(g.n_layers, budget_s / max(1, K + W) / per_item)))
    for _ in range(max(0, W - 1)):
        step(n_sample)
    n_ret0 = sum(len(oc.retained(i)) for i in ids)  # outside the timed region: the same |A(t)| the CUDA arm reads off the device
    t_start = time.perf_counter()
    for _ in range(K):
        used = step(n_sample)
    el = time.perf_counter() - t_start
    n_ret = (n_ret0 + sum(len(oc.retained(i)) for i in ids)) // 2
    kv_bytes = n_ret * BYTES_PER_TOKEN_LAYER * g.n_layers
    us_step = el / K * (n_items_step / n_sample) * 1e6
    sample = (f"per step: Python integer bookkeeping (oracle.paged_cache append + evict) of all {cfg.batch} sequences "
              f"+ fp64 attention of sequence 0, layers 0..{n_sample - 1} (all 28 q heads); the whole time is scaled "
              f"x{n_items_step / n_sample:.1f} to the {n_items_step} (sequence, layer) items of a step - so, unlike the CUDA "
              f"arm's cpu_baseline key (policy + attention only), this value includes the Python bookkeeping")
    line = {
        "impl": "reference", "metric": METRIC, "value": us_step, "unit": UNIT, "n_gpus": args.gpus, "steps": K,
        "warmup": W, "ms_per_step": us_step / 1e3, "higher_is_better": False, "scaling": "weak",
        "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        # the same keys and values as the CUDA arm's `config` (same workload, same t)
        "config": dict(config_keys(cfg, int(os.environ.get("WORLD_SIZE", "1"))), retained_tokens_per_seq=n_ret // cfg.batch,
                       t_first_timed=t0 + max(W, 1) + 1,
                       l2="inputs larger than L2 (each step re-reads %.0f MB of K/V)" % (kv_bytes / 1e6)),
        "what": "fp64 CPU oracle (oracle/), bounded sample per step",
        "cpu_baseline": {"value": us_step, "unit": UNIT, "cores": int(used), "kind": "oracle", "sample": sample},
        "e2e": {"value": us_step, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line), flush=True)
    return 0


# ------------------------------------------------------------------------------------------------
# the CUDA arm
# ------------------------------------------------------------------------------------------------
class Workbench:
    """One cache filled by a bulk append to t = t0 plus pre-generated step inputs resident in HBM."""

    def __init__(self, cfg, t0: int, n_steps: int, dev, n_gen_cap: int = 1100):
        import numpy as np
        import torch

        import workloads
        from paper_2606_01483_b200 import MurmurCache

        self.cfg, self.t0, self.dev = cfg, t0, dev
        g = cfg.geom
        self.B = cfg.batch
        self.n_gen = max(1, min(n_steps, n_gen_cap))  # distinct step inputs (re-used cyclically beyond that)
        Tmin = min(s.T for s in cfg.seqs)
        extra = max(2, t0 + n_steps + 2 - Tmin)  # a long run decodes past the config's T
        self.ids = np.arange(self.B, dtype=np.int32)
        self.n_pages = workloads.unevicted_blocks(cfg, extra) + 2
        self.max_blocks = workloads.max_blocks_per_seq(cfg, extra) + 1
        self.cache = MurmurCache(g.n_layers, g.n_q_heads, g.n_kv_heads, g.head_dim, cfg.page_size, self.B,
                                 self.max_blocks, self.n_pages, device=dev)
        self.data = [workloads.SeqData(cfg, i, device=dev) for i in range(self.B)]
        k_steps, v_steps, q_steps = [], [], []
        for i, s in enumerate(cfg.seqs):
            self.cache.seq_begin(i, s.P, s.S, s.M, s.policy_tuple)
            k, v = self._bulk(i)
            if k.shape[1]:
                self.cache.kv_append([i], [k.shape[1]], k, v)
            del k, v
            ks, vs = self.data[i].out_kv(t0, t0 + self.n_gen)  # [L, steps, kv, d]
            k_steps.append(ks)
            v_steps.append(vs)
            q_steps.append(self.data[i].q_steps(t0 + 1, t0 + self.n_gen + 1))  # [steps, L, n_q, d]
        self.cache.kv_evict(self.ids)
        self.k_all = torch.stack(k_steps, dim=2).permute(1, 0, 2, 3, 4).contiguous()  # [steps, L, B, kv, d]
        self.v_all = torch.stack(v_steps, dim=2).permute(1, 0, 2, 3, 4).contiguous()
        self.q_all = torch.stack(q_steps, dim=2).contiguous()  # [steps, L, B, n_q, d]
        self.out = torch.empty_like(self.q_all[0])
        self.scale = 1.0 / math.sqrt(g.head_dim)
        self.step_no = 0

    def _bulk(self, i: int):
        import torch

        kp, vp = self.data[i].prefill_kv()
        ko, vo = self.data[i].out_kv(0, self.t0)
        return torch.cat([kp, ko], dim=1).contiguous(), torch.cat([vp, vo], dim=1).contiguous()

    def inputs(self, s: int):
        j = s % self.n_gen
        return self.k_all[j], self.v_all[j], self.q_all[j]

    def step(self, out=None, lse=None, dependent: bool = False):
        """One murmur_decode_step.  dependent=True puts what an autoregressive loop has between two steps behind
        it, at its smallest: a one-element kernel (torch's, not counted in gpu_launches) that makes the NEXT step's
        q a function of THIS step's out (q += 0 * out, values unchanged).  The next launch then cannot overlap this
        one's tail - the overlap chained back-to-back launches get, which no real decoder can have."""
        import torch

        k, v, q = self.inputs(self.step_no)
        o = self.out if out is None else out
        self.cache.decode_step(self.ids, k, v, q, o, lse, self.scale)
        self.step_no += 1
        if dependent:
            qn = self.inputs(self.step_no)[2].view(-1)[:1]
            torch.add(qn, o.view(-1)[:1], alpha=0.0, out=qn)

    def n_retained(self) -> int:
        return sum(self.cache.seq_state(i)["n_retained"] for i in range(self.B))

    def host_kv(self, i: int, n_steps_done: int):
        """uint16 [L, n_pos, kv, d] bit patterns of every row appended to sequence i so far, by position."""
        import torch

        import workloads

        k, v = self._bulk(i)
        if n_steps_done:
            order = torch.arange(n_steps_done, device=self.dev) % self.n_gen
            k = torch.cat([k, self.k_all[order][:, :, i].permute(1, 0, 2, 3)], dim=1)
            v = torch.cat([v, self.v_all[order][:, :, i].permute(1, 0, 2, 3)], dim=1)
        return workloads.to_bits(k), workloads.to_bits(v)

    def close(self):
        self.cache.close()


class Shadow:
    """The oracle's integer bookkeeping (oracle.paged_cache) advanced beside a Workbench."""

    def __init__(self, wb: Workbench):
        from oracle import paged_cache as o_cache
        from oracle import policy as o_policy

        cfg = wb.cfg
        self.ids = list(range(cfg.batch))
        self.oc = o_cache.OraclePagedCache(wb.n_pages, cfg.page_size, cfg.batch, wb.max_blocks)
        for i, s in enumerate(cfg.seqs):
            self.oc.seq_begin(i, s.P, s.S, s.M, o_policy.Policy(*s.policy_tuple))
            n = s.P + s.S + s.M + wb.t0
            if n:
                self.oc.append([i], [n])  # same call pattern as Workbench: one bulk append per sequence
        self.oc.evict(self.ids)

    def advance(self, n: int = 1):
        for _ in range(n):
            self.oc.append(self.ids, [1] * len(self.ids))
            self.oc.evict(self.ids)

    def retained(self) -> dict:
        return {i: list(self.oc.retained(i)) for i in self.ids}

    def check(self, cache) -> None:
        """Integer state of every sequence, bit-exact: length, t, retained set, compacted page table,
        run descriptors; the free stack; the device error word; the host mirror of the free count."""
        import numpy as np

        for i in self.ids:
            st = cache.seq_state(i)
            o = self.oc.seqs[i]
            assert st["length"] == o.length and st["t"] == o.t, (i, st, o.length, o.t)
            assert np.array_equal(cache.retained(i), np.asarray(self.oc.retained(i), dtype=np.int32)), f"retained set, seq {i}"
            pages, blocks = cache.page_list(i)
            assert list(blocks) == self.oc.live_blocks(i), f"live blocks, seq {i}"
            assert list(pages) == self.oc.live_pages(i), f"live pages, seq {i}"
            assert cache.runs(i) == self.oc.runs(i), f"runs, seq {i}"
        assert list(cache.free_stack()) == self.oc.free_stack, "free stack"
        assert cache.last_error() == 0
        assert cache.stats()["free_pages"] == len(self.oc.free_stack)


def oracle_compare(wb: Workbench, host_kv: dict, q, out, retained: dict, n_threads: int = 0):
    """out [L, B, n_q, d] (bf16 tensor, device or host) vs Eq. 1 over `retained` in fp64 (plain-C oracle),
    every (sequence, layer, head).  Returns (parity dict, oracle attention seconds, threads used)."""
    import numpy as np

    import workloads
    from oracle import attention as o_attn
    from oracle import c as oracle_c

    co = oracle_c.load()
    got = o_attn.bf16_bits_to_f64(workloads.to_bits(out))
    q_bits = workloads.to_bits(q)
    mx, sm, n, secs, used = 0.0, 0.0, 0, 0.0, 1
    assert np.all(np.isfinite(got))
    for i in range(wb.B):
        kb, vb = host_kv[i]
        tc = time.perf_counter()
        o_ref, _, used = co.attend(q_bits[:, i], kb, vb, retained[i], wb.scale, n_threads=n_threads)
        secs += time.perf_counter() - tc
        e = np.abs(got[:, i] - o_ref)
        mx = max(mx, float(e.max()))
        sm += float(e.sum())
        n += e.size
    return {"max_abs": mx, "mean_abs": sm / n, "tol_max_abs": 2e-2, "tol_mean_abs": 2e-3,
            "ok": bool(mx <= 2e-2 and sm / n <= 2e-3), "items": f"{wb.B} sequences x {q.shape[0]} layers x {q.shape[2]} heads"}, secs, used


def timed_steps(wb: Workbench, K: int, barrier, stream, torch, dependent: bool = False):
    barrier()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    w0 = time.time()
    e0.record(stream)
    for _ in range(K):
        wb.step(dependent=dependent)
    e1.record(stream)
    barrier()
    return e0.elapsed_time(e1) / K * 1e3, (w0, time.time())


def spin_up(wb: Workbench, torch, seconds: float = 0.25):
    """Untimed, state not advanced: repeat attention on the current state until the clocks are up."""
    t_spin = time.perf_counter()
    while time.perf_counter() - t_spin < seconds:
        for _ in range(20):
            wb.cache.decode_attn(wb.ids, wb.q_all[0], out=wb.out, sm_scale=wb.scale)
        torch.cuda.synchronize(wb.dev)


def alg_bytes_of(cfg, n_ret_total: int) -> int:
    g = cfg.geom
    return n_ret_total * BYTES_PER_TOKEN_LAYER * g.n_layers + 2 * g.n_layers * cfg.batch * g.n_q_heads * g.head_dim * 2


def run_other_workload(name: str, dev, sampler, peak: float, check: bool, torch) -> dict:
    """One of the other BASELINE.json configurations: 5 warm-up + 50 timed one-launch steps, roofline
    fraction, and the oracle check of the last timed output (every sequence, layer, head)."""
    cfg, t0 = pick_workload(name)
    K, W = 50, 5
    wb = Workbench(cfg, t0, W + 3 * K + 6, dev)
    stream = torch.cuda.current_stream()

    def barrier():
        torch.cuda.synchronize(dev)

    spin_up(wb, torch, 0.1)
    for _ in range(W):
        wb.step()
    us_chain, _ = timed_steps(wb, K, barrier, stream, torch)  # back-to-back chained launches (secondary figure)
    n0 = wb.n_retained()
    us, win = timed_steps(wb, K, barrier, stream, torch, dependent=True)
    if sampler:
        sampler.window(win[0], win[1], name)
    n_ret = (n0 + wb.n_retained()) // 2
    ab = alg_bytes_of(cfg, n_ret)
    gbs = ab / (us * 1e-6) / 1e9
    # opt-in L2 pinning (MURMUR_OPT_L2_KEEP_PCT = -1, automatic): the same dependent steps again, reported beside the
    # default (0 = pure evict_first, so that `frac` stays a pure HBM fraction)
    from paper_2606_01483_b200 import binding as _b
    wb.cache.set_option(_b.MURMUR_OPT_L2_KEEP_PCT, -1)
    for _ in range(3):
        wb.step()
    us_l2, _ = timed_steps(wb, K, barrier, stream, torch, dependent=True)
    wb.cache.set_option(_b.MURMUR_OPT_L2_KEEP_PCT, 0)
    n_extra = 3 + K
    res = {"workload": cfg.name, "us_per_step": us, "steps": K, "retained_tokens_per_seq": n_ret // cfg.batch,
           "algorithmic_bytes_per_step": ab, "achieved_gbs": gbs, "frac": min(1.0, gbs / peak), "frac_uncapped": gbs / peak,
           "frac_note": "peak is a measured COPY figure (read + write); a read-only stream can exceed it, so frac is capped at 1",
           "frac_of_nominal_8000": gbs / 8000.0, "l2_keep_pct": 0, "us_per_step_with_l2_keep_auto": us_l2,
           "timing": "each step followed by a one-element kernel that makes the next step's q depend on this step's out",
           "chained_back_to_back_us": us_chain,
           "tokens_per_s": cfg.batch / (us * 1e-6), "launches_per_step": 1}
    if check:
        n_done = W + 2 * K + n_extra
        sh = Shadow(wb)
        sh.advance(n_done)
        sh.check(wb.cache)
        hk = {i: wb.host_kv(i, n_done) for i in range(cfg.batch)}
        par, secs, used = oracle_compare(wb, hk, wb.inputs(n_done - 1)[2], wb.out, sh.retained())
        par["compared"] = ("output of the LAST TIMED murmur_decode_step launch (of the L2-keep run, which follows the "
                           "default run on the same cache); integer state of every sequence bit-exact")
        res["parity"] = par
        res["cpu_baseline"] = {"value": secs * 1e6, "unit": UNIT, "cores": int(used), "kind": "oracle",
                               "sample": f"the WHOLE last timed step: plain-C fp64 attention (oracle/c) of all {cfg.batch} "
                                         f"sequences x {cfg.geom.n_layers} layers x {cfg.geom.n_q_heads} heads over the oracle's "
                                         "retained sets, once, not scaled"}
        del hk
    res["device_error_word"] = wb.cache.last_error()
    wb.close()
    del wb
    torch.cuda.empty_cache()
    return res


def run_murmur(args):
    import numpy as np
    import torch

    from paper_2606_01483_b200 import binding

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device (the product path has no CPU fallback)")
    dev = torch.device(f"cuda:{local_rank}")
    torch.cuda.set_device(dev)
    dist = None
    if world > 1:
        import torch.distributed as dist_mod

        dist_mod.init_process_group("nccl", device_id=dev)
        dist = dist_mod
    binding.lib()  # fail loudly if libmurmur.so is missing

    cfg, t0 = pick_workload(args.workload)
    g = cfg.geom
    K, W = args.steps, max(3, args.warmup)
    Ke, We = args.e2e_steps, 3
    Kb2, Kp = min(K, 100), min(K, 50)
    n_steps_total = W + 3 * K + Kb2 + 3 + Kp + We + Ke + 1
    B = cfg.batch
    check = rank == 0 and world == 1 and not args.no_cpu_baseline
    wb = Workbench(cfg, t0, n_steps_total, dev)
    cache, ids, scale = wb.cache, wb.ids, wb.scale
    stream = torch.cuda.current_stream()
    peak, peak_src = load_peak()

    def barrier():
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize(dev)

    sampler = ClockSampler(local_rank) if rank == 0 else None
    if sampler:
        sampler.wait_ready()
    spin_up(wb, torch)
    for _ in range(W):
        wb.step()
    # ---- region A: K steps, whole-step timing -----------------------------------------------
    cache.reset_stats()
    n_ret_a0 = wb.n_retained()
    # every step is followed by a one-element kernel that makes the next step's q depend on this step's out: the
    # launch pattern of an autoregressive loop at its tightest (no overlap of step t+1's stream with step t's tail)
    us_a, win = timed_steps(wb, K, barrier, stream, torch, dependent=True)
    launches = cache.stats()["kernel_launches"]
    if sampler:
        sampler.window(win[0], win[1])
    st = cache.stats()
    n_ret_a1 = wb.n_retained()
    steps_a = wb.step_no  # steps applied to the cache when region A's last output was produced
    out_a = wb.out.clone()
    shadow, parity_int = None, None
    if check:
        shadow = Shadow(wb)
        shadow.advance(steps_a)
        shadow.check(cache)  # integer state of every sequence after the timed region, bit-exact
        ret_a = shadow.retained()
        parity_int = f"bit-exact after region A (all {B} sequences: lengths, retained sets, page tables, runs, free stack)"

    # ---- region A2: K steps back to back with nothing in between (chained launches overlap) --------
    us_chain, win2 = timed_steps(wb, K, barrier, stream, torch)
    if sampler:
        sampler.window(win2[0], win2[1])

    # ---- region B: K steps with one event pair around every launch --------------------------------
    # B1: the step as the library runs it (ONE launch) -> isolated launch duration, no PDL overlap
    # B2: the same step as three separate calls (append, evict, attention) -> per-stage breakdown
    ones = [1] * B
    evs1 = [[torch.cuda.Event(enable_timing=True) for _ in range(2)] for _ in range(K)]
    evs = [[torch.cuda.Event(enable_timing=True) for _ in range(4)] for _ in range(Kb2)]
    barrier()
    w0 = time.time()
    torch.cuda._sleep(int(1e8))  # ~50 ms of GPU spin so the host runs ahead: event pairs then see kernels, not launch gaps
    cache.reset_stats()
    for j in range(K):
        evs1[j][0].record(stream)
        wb.step()
        evs1[j][1].record(stream)
    launches_per_step_b1 = cache.stats()["kernel_launches"] / K
    barrier()
    torch.cuda._sleep(int(1e8))
    for j in range(Kb2):
        k, v, q = wb.inputs(wb.step_no)
        evs[j][0].record(stream)
        cache.kv_append(ids, ones, k, v)
        evs[j][1].record(stream)
        cache.kv_evict(ids)
        evs[j][2].record(stream)
        cache.decode_attn(ids, q, out=wb.out, sm_scale=scale)
        evs[j][3].record(stream)
        wb.step_no += 1
    barrier()
    if sampler:
        sampler.window(w0, time.time())
    step_list = sorted(e[0].elapsed_time(e[1]) * 1e3 for e in evs1)
    t_stepk = sum(step_list) / K
    t_stepk_med = step_list[K // 2]
    stepk_p10, stepk_p90 = step_list[K // 10], step_list[min(K - 1, (9 * K) // 10)]
    t_app = sum(e[0].elapsed_time(e[1]) for e in evs) / Kb2 * 1e3
    t_evi = sum(e[1].elapsed_time(e[2]) for e in evs) / Kb2 * 1e3
    attn_list = sorted(e[2].elapsed_time(e[3]) * 1e3 for e in evs)
    t_att = sum(attn_list) / Kb2
    t_att_med = attn_list[Kb2 // 2]

    # ---- region P: the step as a layer-by-layer engine issues it, from C ---------------------------
    # (layer l's K/V exist only when layer l runs: murmur_decode_step_layers once per layer = 28 launches
    # per step, issued by murmur_decode_step_chunked(layers_per_launch = 1) without leaving the library)
    for _ in range(3):
        k, v, q = wb.inputs(wb.step_no)
        cache.decode_step_chunked(ids, k, v, q, wb.out, 1, None, scale)
        wb.step_no += 1
    barrier()
    p0, p1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    cache.reset_stats()
    p0.record(stream)
    for _ in range(Kp):
        k, v, q = wb.inputs(wb.step_no)
        cache.decode_step_chunked(ids, k, v, q, wb.out, 1, None, scale)
        wb.step_no += 1
    p1.record(stream)
    barrier()
    us_per_layer_mode = p0.elapsed_time(p1) / Kp * 1e3
    per_layer_launches = cache.stats()["kernel_launches"] / Kp

    # ---- region C: end to end from pinned host buffers -------------------------------------------
    s0 = wb.step_no
    sel = torch.arange(s0, s0 + We + Ke, device=dev) % wb.n_gen
    # per step: k_new | v_new | q packed back to back in one pinned block
    kv_n, q_n = wb.k_all[0].numel(), wb.q_all[0].numel()
    hb = torch.empty((We + Ke, 2 * kv_n + q_n), dtype=torch.bfloat16).pin_memory()
    hb[:, :kv_n] = wb.k_all[sel].reshape(We + Ke, -1).cpu()
    hb[:, kv_n:2 * kv_n] = wb.v_all[sel].reshape(We + Ke, -1).cpu()
    hb[:, 2 * kv_n:] = wb.q_all[sel].reshape(We + Ke, -1).cpu()
    kh = [hb[j, :kv_n].view(wb.k_all[0].shape) for j in range(We + Ke)]
    vh = [hb[j, kv_n:2 * kv_n].view(wb.v_all[0].shape) for j in range(We + Ke)]
    qh = [hb[j, 2 * kv_n:].view(wb.q_all[0].shape) for j in range(We + Ke)]
    oh = torch.empty(wb.out.shape, dtype=torch.bfloat16).pin_memory()
    for j in range(We):
        cache.decode_step_host(ids, kh[j], vh[j], qh[j], oh, scale)
        torch.cuda.synchronize(dev)
    barrier()
    c0, c1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    cache.reset_stats()
    w0 = time.time()
    c0.record(stream)
    for j in range(We, We + Ke):
        cache.decode_step_host(ids, kh[j], vh[j], qh[j], oh, scale)
        stream.synchronize()  # the caller reads `oh` every step
    c1.record(stream)
    barrier()
    w1 = time.time()
    if sampler:
        sampler.window(w0, w1)
    e2e_launches = cache.stats()["kernel_launches"] / Ke
    e2e_zero_copy = cache.stats()["host_zero_copy_steps"] == Ke
    us_e2e_dev = c0.elapsed_time(c1) / Ke * 1e3
    us_e2e_wall = (w1 - w0) / Ke * 1e6
    us_e2e = max(us_e2e_dev, us_e2e_wall)
    wb.step_no = s0 + We + Ke
    steps_c = wb.step_no
    h2d = (kh[0].numel() + vh[0].numel() + qh[0].numel()) * 2
    d2h = oh.numel() * 2

    # ---- reduce over ranks ---------------------------------------------------------------------
    us_step, us_e2e, t_att, t_app, t_evi, t_att_med, t_stepk, t_stepk_med, us_per_layer_mode, us_chain = max_over_ranks(
        [us_a, us_e2e, t_att, t_app, t_evi, t_att_med, t_stepk, t_stepk_med, us_per_layer_mode, us_chain], dist, dev)

    # ---- algorithmic bytes of one step launch -----------------------------------
    n_ret = (n_ret_a0 + n_ret_a1) // 2  # the device's own |A(t)|, mean over region A
    alg_bytes = alg_bytes_of(cfg, n_ret)
    kv_bytes = n_ret * BYTES_PER_TOKEN_LAYER * g.n_layers
    one_launch = launches_per_step_b1 < 1.5
    if one_launch:
        # region A is K launches of this one kernel, each followed by a one-element dependent kernel: its average
        # launch duration over the timed region is region A's time / K (this slightly over-states the kernel: the
        # one-element kernel and two launch gaps are inside).  The event-pair-per-launch figure of region B1 is kept
        # beside it as isolated_launch_us, and the back-to-back figure of region A2 (chained launches overlap one
        # step's tail with the next step's stream - something a real decoder cannot do) as chained_back_to_back_us
        dom_kernel, dom_us, dom_med = "attn_mma_kernel<step> (append + evict + attention, one launch)", us_step, t_stepk_med
    else:
        dom_kernel = "attn_mma_kernel" if st["attn_variant"] == 2 else "attn_generic_kernel"
        dom_us, dom_med = t_att, t_att_med
    achieved = alg_bytes / (dom_us * 1e-6) / 1e9
    attn_only = alg_bytes / (t_att * 1e-6) / 1e9
    roofline = {"bound": "hbm", "kernel": dom_kernel,
                "achieved": achieved, "peak": peak, "unit": "GB/s", "frac": min(1.0, achieved / peak), "frac_uncapped": achieved / peak,
                "traffic": ncu_traffic_bytes(cfg.name), "kernel_source_hash": kernel_source_hash(),
                "peak_source": peak_src, "algorithmic_bytes_per_launch": alg_bytes,
                "avg_launch_us": dom_us, "median_launch_us": dom_med, "isolated_launch_us": t_stepk if one_launch else t_att,
                "how": ("region A time / K launches: one launch per step, CUDA events around the K steps, every step "
                        "followed by a one-element kernel that makes the next step's q depend on this step's out (no "
                        "overlap between consecutive steps)" if one_launch
                        else "mean of per-launch CUDA event pairs (region B2)"),
                "frac_of_nominal_8000": achieved / 8000.0,
                "frac_isolated_launch": alg_bytes / ((t_stepk if one_launch else t_att) * 1e-6) / 1e9 / peak,
                "l2_keep_pct": 0,
                "chained_back_to_back_us": us_chain,
                "chained_back_to_back_gbs": alg_bytes / (us_chain * 1e-6) / 1e9,
                "note": ("peak is a COPY figure (read + write streams).  chained_back_to_back_* is the same kernel launched "
                         "K times with nothing in between: consecutive launches overlap (step t+1 streams K/V under step "
                         "t's tail), which needs the next step's inputs before this step's output exists - it is a property "
                         "of the launch chain, not bandwidth of the kernel, and is not the headline")}

    # ---- oracle: parity of the timed outputs, CPU baseline, replay, protocol, other workloads -----
    cpu_baseline = parity = replay = protocol = others = index_sets = None
    if check:
        import workloads
        from oracle import c as oracle_c
        from oracle import policy as o_policy

        shadow.advance(steps_c - steps_a)
        ret_c = shadow.retained()
        hk = {i: wb.host_kv(i, steps_c) for i in range(B)}
        # region A's last output (the timed murmur_decode_step launches) and region C's (murmur_decode_step_host)
        q_a = wb.inputs(steps_a - 1)[2]
        best = None
        for _ in range(2):
            par_a, secs, used = oracle_compare(wb, hk, q_a, out_a, ret_a)
            best = secs if best is None else min(best, secs)
        par_c, _, _ = oracle_compare(wb, hk, wb.inputs(steps_c - 1)[2], oh, ret_c)
        parity = {"compared": "murmur_decode_step: output of the LAST TIMED launch of region A; murmur_decode_step_host: "
                              "host output of the last timed step of region C; every (sequence, layer, head), fp64 oracle",
                  "decode_step": par_a, "decode_step_host": par_c, "integer_state": parity_int,
                  "ok": bool(par_a["ok"] and par_c["ok"])}
        # CPU baseline: the oracle's work for the same step = retained sets (oracle.policy) + plain-C attention
        s0_ = cfg.seqs[0]
        tp = time.perf_counter()
        for s in cfg.seqs:
            o_policy.retained_positions(s.P, s.S, s.M, t0 + steps_a, o_policy.Policy(*s.policy_tuple))
        t_policy = time.perf_counter() - tp
        co = oracle_c.load()
        import workloads as _w
        qb0 = _w.to_bits(q_a[:, 0])
        n_l1 = max(1, min(g.n_layers, 4))
        t1 = time.perf_counter()
        co.attend(qb0[:n_l1], hk[0][0][:n_l1], hk[0][1][:n_l1], ret_a[0], scale, n_threads=1)
        us_1t = ((time.perf_counter() - t1) / n_l1 * g.n_layers * B + t_policy) * 1e6
        cpu_baseline = {"value": (best + t_policy) * 1e6, "unit": UNIT, "cores": int(used), "kind": "oracle",
                        "single_thread_value": us_1t,
                        "sample": f"the WHOLE last step of region A (t={t0 + steps_a}): oracle.policy retained sets + plain-C "
                                  f"fp64 attention (oracle/c) of all {B} sequences x {g.n_layers} layers x {g.n_q_heads} heads, "
                                  f"best of 2, not scaled; single_thread_value = sequence 0, layers 0..{n_l1 - 1} on one thread, "
                                  f"scaled; host cores = {os.cpu_count()}"}
        del hk
        wb_err = cache.last_error()
        wb.close()
        torch.cuda.empty_cache()

        # replay of region A on a second cache: integer state at EVERY step, final output bit-identical
        wb2 = Workbench(cfg, t0, steps_a + 1, dev)
        sh2 = Shadow(wb2)
        for _ in range(steps_a):
            wb2.step()
            sh2.advance(1)
            sh2.check(wb2.cache)
        torch.cuda.synchronize(dev)
        replay = {"steps": steps_a, "integer_state": "bit-exact vs oracle.paged_cache at every step (warm-up + region A)",
                  "last_output_bit_identical_to_region_A": bool(torch.equal(wb2.out, out_a))}
        wb2.close()
        del wb2
        torch.cuda.empty_cache()

        if not args.no_protocol:
            protocol = run_protocol(cfg, dev, torch)
        if cfg.name == "chunked_12x300s" and not args.no_others:
            others = {}
            for name in OTHER_WORKLOADS:
                others[name] = run_other_workload(name, dev, sampler, peak, True, torch)
            index_sets = run_index_set_eviction(dev, torch)
    else:
        wb_err = cache.last_error()
        wb.close()
    clocks_all = sampler.finish() if sampler else {}
    if others:
        for name in others:
            others[name]["clocks"] = clocks_all.get(name)
    if dist is not None:
        dist.destroy_process_group()
    if rank != 0:
        return 0
    line = {
        "metric": METRIC, "value": us_step, "unit": UNIT, "n_gpus": world, "steps": K, "warmup": W,
        "ms_per_step": us_step / 1e3, "higher_is_better": False, "scaling": "weak", "vs_baseline": None,
        "dtype": "bf16", "data": "synthetic",
        "config": dict(config_keys(cfg, world), retained_tokens_per_seq=n_ret // B, t_first_timed=t0 + W + 1,
                       l2="inputs larger than L2 (each step re-reads %.0f MB of K/V)" % (kv_bytes / 1e6)),
        "tokens_per_s": whole_job_tokens_per_s(world, B, us_step),
        "step_kernel_us": t_stepk, "step_kernel_us_p10_p50_p90": [stepk_p10, t_stepk_med, stepk_p90],
        "launches_per_step": launches_per_step_b1,
        "separate_calls": {"append_us": t_app, "evict_us": t_evi, "attn_us": t_att, "attn_median_us": t_att_med,
                           "attn_hbm_gbs": attn_only, "attn_pct_of_measured_peak": 100.0 * attn_only / peak,
                           "note": "the same step as three API calls, one event pair per call (includes launch gaps)"},
        "per_layer_mode_us": us_per_layer_mode,
        "per_layer_mode": {"us_per_step": us_per_layer_mode, "launches_per_step": per_layer_launches, "steps": Kp,
                           "achieved_gbs": alg_bytes / (us_per_layer_mode * 1e-6) / 1e9,
                           "frac": alg_bytes / (us_per_layer_mode * 1e-6) / 1e9 / peak,
                           "api": "murmur_decode_step_chunked(layers_per_launch=1): murmur_decode_step_layers once per layer, "
                                  "issued from C (append-write + attention of layer l in ONE launch; the layer-0 launch "
                                  "also reserves, commits and evicts)"},
        "step_hbm_gbs": alg_bytes / (us_step * 1e-6) / 1e9,
        "chained_back_to_back_us": us_chain,
        "timing": "value = region A: K steps, each followed by a one-element kernel (out -> next q), CUDA events around "
                  "the region, barrier + synchronize on both sides; chained_back_to_back_us = region A2, the same K steps "
                  "with nothing in between",
        "roofline": roofline, "cpu_baseline": cpu_baseline, "parity": parity, "parity_last_step": parity,
        "replay": replay, "protocol": protocol, "other_workloads": others, "index_set_eviction": index_sets,
        "e2e": {"value": us_e2e, "unit": UNIT, "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h,
                "device_us": us_e2e_dev, "wall_us": us_e2e_wall, "steps": Ke, "launches_per_step": e2e_launches,
                "path": ("zero-copy: the step kernel reads k_new / v_new / q from the pinned host buffers and stores out to the "
                         "pinned host buffer through their device-mapped addresses (the declared bytes cross PCIe inside the "
                         "timed kernel; no staging copies)" if e2e_zero_copy else
                         "staged: cudaMemcpyAsync host->device, step, cudaMemcpyAsync device->host"),
                "api": "murmur_decode_step_host (pinned host k_new | v_new | q -> out), stream-synchronised per step"},
        "gpu_launches": int(launches), "attn_grid": st["attn_grid"], "attn_smem_bytes": st["attn_smem_bytes"],
        "device_error_word": wb_err, "clocks": clocks_all.get("main"),
        "paper_context": "paper reports end-to-end only: 88.43 s (chunked + speech eviction) vs 370.73 s single pass, "
                         "1x H100 80GB, batch 16, AMI-IHM (PAPER.md:201-206)",
    }
    print(json.dumps(line), flush=True)
    return 0


def run_protocol(cfg, dev, torch) -> dict:
    """SURVEY.md 8(d) "Protocol": the whole decode t = 1 .. T through one-launch steps; at the steps
    {1, 2, k_o+w_o, k_o+w_o+1, d, d+1, d+2, T/2, T-1, T} the retained sets are compared with oracle.policy
    and the output of EVERY (sequence, layer, head) with the fp64 oracle."""
    import numpy as np

    from oracle import policy as o_policy

    s0 = cfg.seqs[0]
    T = min(s.T for s in cfg.seqs)
    marks = sorted({x for x in (1, 2, s0.n_sink_out + s0.w_out, s0.n_sink_out + s0.w_out + 1, s0.delay, s0.delay + 1,
                                s0.delay + 2, T // 2, T - 1, T) if 1 <= x <= T})
    wb = Workbench(cfg, 0, T, dev, n_gen_cap=T)
    saved = {}
    t_run = time.perf_counter()
    for t in range(1, T + 1):
        if t in marks:
            out = torch.empty_like(wb.out)
            wb.step(out=out)
            ret = {}
            for i, s in enumerate(cfg.seqs):
                want = [x for x in o_policy.retained_positions(s.P, s.S, s.M, t, o_policy.Policy(*s.policy_tuple))
                        if x < s.P + s.S + s.M + t]
                assert np.array_equal(wb.cache.retained(i), np.asarray(want, dtype=np.int32)), f"retained set, seq {i}, t={t}"
                assert wb.cache.seq_state(i)["t"] == t
                ret[i] = want
            saved[t] = (out, ret)
        else:
            wb.step()
    torch.cuda.synchronize(dev)
    gpu_s = time.perf_counter() - t_run
    assert wb.cache.last_error() == 0
    hk = {i: wb.host_kv(i, T) for i in range(cfg.batch)}
    worst_max, worst_mean, ok = 0.0, 0.0, True
    for t in marks:
        out, ret = saved[t]
        par, _, _ = oracle_compare(wb, hk, wb.inputs(t - 1)[2], out, ret)
        worst_max, worst_mean, ok = max(worst_max, par["max_abs"]), max(worst_mean, par["mean_abs"]), ok and par["ok"]
    wb.close()
    del hk
    torch.cuda.empty_cache()
    return {"decode_steps": T, "checked_steps_t": marks, "full_tensor_steps": len(marks),
            "retained_sets": "bit-exact vs oracle.policy at every checked step",
            "attention": {"max_abs": worst_max, "mean_abs": worst_mean, "tol_max_abs": 2e-2, "tol_mean_abs": 2e-3, "ok": ok,
                          "items": f"{cfg.batch} sequences x {cfg.geom.n_layers} layers x {cfg.geom.n_q_heads} heads per step"},
            "wall_s_gpu_loop": gpu_s}


def run_index_set_eviction(dev, torch) -> dict:
    """SURVEY 8f-3 on the config-2 shape: query-aware index sets (>= 99 % of every query head's Eq. 1 mass, both
    prompts, the 16 newest positions) for every sequence of an un-evicted cache, applied by the in-place dense
    compaction; reports the bytes the compaction moved next to the bytes it retains, and checks sequence 0's slabs
    and attention against oracle/indexset.py."""
    import numpy as np

    import workloads
    from oracle import indexset as o_ix
    from oracle import paged_cache as o_cache
    from oracle import policy as o_policy

    W = workloads.WINDOW_OFF
    cfg = workloads.config2(W, W)
    t0 = 300
    wb = Workbench(cfg, t0, 2, dev)
    g = cfg.geom
    L, H = g.n_layers, g.n_kv_heads
    wb.cache.indexed_enable()
    n = cfg.seqs[0].P + cfg.seqs[0].S + cfg.seqs[0].M + t0
    frac, n_recent = 0.99, 16
    e0, e1, e2, e3 = (torch.cuda.Event(enable_timing=True) for _ in range(4))
    stream = torch.cuda.current_stream()
    sets = []
    torch.cuda.synchronize(dev)
    e0.record(stream)
    for i in range(cfg.batch):
        sets.append(wb.cache.select_mass_sets(i, wb.data[i].q_step(t0).contiguous(), frac, n_recent, cap=n, sm_scale=wb.scale))
    e1.record(stream)
    torch.cuda.synchronize(dev)
    moved = 0
    t_def = time.perf_counter()
    for i in range(cfg.batch):
        moved += wb.cache.kv_evict_indexed(i, sets[i][0], sets[i][1])
    t_def = time.perf_counter() - t_def
    rows = sum(int(sets[i][1].sum()) for i in range(cfg.batch))
    q = wb.q_all[0]  # [L, B, n_q, d]: the queries of step t0 + 1 (any queries do for a timing + parity check)
    for _ in range(3):
        out = wb.cache.decode_attn_indexed(wb.ids, q, sm_scale=wb.scale)
    torch.cuda.synchronize(dev)
    e2.record(stream)
    for _ in range(10):
        out = wb.cache.decode_attn_indexed(wb.ids, q, sm_scale=wb.scale)
    e3.record(stream)
    torch.cuda.synchronize(dev)
    # parity of sequence 0 against the oracle, with the sets the GPU selected
    oc = o_cache.OraclePagedCache(wb.n_pages, cfg.page_size, cfg.batch, wb.max_blocks)
    s0 = cfg.seqs[0]
    oc.seq_begin(0, s0.P, s0.S, s0.M, o_policy.Policy(*s0.policy_tuple))
    oc.append([0], [n])
    oc.evict([0])
    oix = o_ix.OracleIndexedCache(oc, L, H)
    sel = [[sets[0][0][l, h, : int(sets[0][1][l, h])].cpu().tolist() for h in range(H)] for l in range(L)]
    oix.evict_indexed(0, sel)
    kb, vb = wb.host_kv(0, 0)
    gk, gv = wb.cache.gather_indexed(0, oix.seqs[0].max_len())
    gk, gv = workloads.to_bits(gk), workloads.to_bits(gv)
    rows_ok = all(np.array_equal(gk[l, h, : len(sel[l][h])], kb[l][sel[l][h], h]) and
                  np.array_equal(gv[l, h, : len(sel[l][h])], vb[l][sel[l][h], h]) and
                  wb.cache.indexed_positions(0, l, h).tolist() == sel[l][h] for l in range(L) for h in range(H))
    got = workloads.to_bits(out[:, 0])
    from oracle import attention as o_attn

    gotf = o_attn.bf16_bits_to_f64(got)
    qb = workloads.to_bits(q[:, 0])
    mx, sm = 0.0, 0.0
    for l in range(L):
        o_ref, _ = o_ix.attend_indexed(qb[l], kb[l], vb[l], sel[l], wb.scale)
        e = np.abs(gotf[l] - o_ref)
        mx, sm = max(mx, float(e.max())), sm + float(e.sum())
    mean = sm / (L * g.n_q_heads * g.head_dim)
    res = {"workload": "config-2 shape, un-evicted (%d tokens / sequence), sets selected at t = %d" % (n, t0),
           "mass_frac": frac, "n_recent": n_recent,
           "rows_before": cfg.batch * n * L * H, "rows_retained": rows, "kept_pct": 100.0 * rows / (cfg.batch * n * L * H),
           "retained_bytes": rows * 512, "defrag_bytes_moved": moved, "moved_over_retained": moved / max(1, rows * 512),
           "select_us_per_sequence": e0.elapsed_time(e1) * 1e3 / cfg.batch,
           "evict_indexed_wall_us_per_sequence": t_def * 1e6 / cfg.batch,
           "decode_attn_indexed_us": e2.elapsed_time(e3) * 1e3 / 10,
           "decode_attn_indexed_gbs": rows * 512 / (e2.elapsed_time(e3) * 1e-3 / 10) / 1e9,
           "pages_freed": int(wb.cache.stats()["free_pages"]) - 2,
           "parity_sequence_0": {"slab_tables_and_rows_bit_exact": bool(rows_ok), "max_abs": mx, "mean_abs": mean,
                                 "ok": bool(rows_ok and mx <= 2e-2 and mean <= 2e-3)},
           "device_error_word": wb.cache.last_error(),
           "note": "attention over the slabs: streaming tensor-core kernel, one CTA per (layer, sequence, KV head) slab; "
                   "the point of the line is the cache-management cost (PAPER.md:154, 214) next to what it buys"}
    wb.close()
    del wb
    torch.cuda.empty_cache()
    return res


def run_prefill(args):
    """--workload prefill_300s: causal prefill attention of one 300 s chunk (64 prompt + 2250 speech tokens, 28 layers)
    over the paged cache, murmur_prefill_attn (tcgen05 + TMEM).  A step = one call over all layers.  Bound: tensor."""
    import numpy as np
    import torch

    import workloads
    from paper_2606_01483_b200 import MURMUR_WINDOW_OFF, MurmurCache, binding

    dev = torch.device("cuda:%d" % int(os.environ.get("LOCAL_RANK", "0")))
    torch.cuda.set_device(dev)
    binding.lib()
    cfg = workloads.config2()
    g = cfg.geom
    K, W = args.steps, max(3, args.warmup)
    d = workloads.SeqData(cfg, 0, device=dev)
    k, v = d.prefill_kv()
    n, L = k.shape[1], g.n_layers
    nb = (n + cfg.page_size - 1) // cfg.page_size + 2
    c = MurmurCache(L, g.n_q_heads, g.n_kv_heads, g.head_dim, cfg.page_size, 1, nb, nb + 2, device=dev)
    c.seq_begin(0, cfg.seqs[0].P, cfg.seqs[0].S, 0, (MURMUR_WINDOW_OFF, 0, 0, MURMUR_WINDOW_OFF, 0))
    c.kv_append([0], [n], k.contiguous(), v.contiguous())
    gen = torch.Generator(device=dev)
    gen.manual_seed(2606)
    q = torch.randn(L, n, g.n_q_heads, g.head_dim, generator=gen, device=dev).to(torch.bfloat16)
    out = torch.empty_like(q)
    lse = torch.empty(L, n, g.n_q_heads, dtype=torch.float32, device=dev)
    stream = torch.cuda.current_stream()
    sampler = ClockSampler(dev.index or 0)
    for _ in range(W):
        c.prefill_attn(0, 0, n, q, out=out, lse=lse)
    torch.cuda.synchronize(dev)
    sampler.wait_ready()
    for _ in range(20):  # clocks up and the sampler inside a loaded stretch before the timed region
        c.prefill_attn(0, 0, n, q, out=out, lse=lse)
    torch.cuda.synchronize(dev)
    c.reset_stats()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    w0 = time.time()
    e0.record(stream)
    for _ in range(K):
        c.prefill_attn(0, 0, n, q, out=out, lse=lse)
    e1.record(stream)
    torch.cuda.synchronize(dev)
    sampler.window(w0, time.time())
    launches = c.stats()["kernel_launches"]
    ms = e0.elapsed_time(e1) / K
    # the round-1 mma.sync kernel, for context
    c.set_option(binding.MURMUR_OPT_PREFILL_VARIANT, binding.MURMUR_PREFILL_MMA_SYNC)
    out_old = torch.empty_like(q)
    for _ in range(2):
        c.prefill_attn(0, 0, n, q, out=out_old)
    torch.cuda.synchronize(dev)
    e0.record(stream)
    for _ in range(5):
        c.prefill_attn(0, 0, n, q, out=out_old)
    e1.record(stream)
    torch.cuda.synchronize(dev)
    ms_old = e0.elapsed_time(e1) / 5
    flops = 4.0 * g.head_dim * (n * (n + 1) / 2) * g.n_q_heads * L  # causal: QK^T + PV over y <= x
    tfs = flops / (ms * 1e-3) / 1e12
    try:
        with open(os.path.join(ROOT, "MEASURED_PEAKS.json")) as f:
            pk = json.load(f)
        peak, peak_src = float(pk["bf16_tflops"]), ("measured (MEASURED_PEAKS.json bf16_tflops, the BURST figure - the conservative "
                                                     "denominator: K launches back to back run into the power cap like the sustained one)")
        peak_sus = float(pk["bf16_tflops_sustained"]) if "bf16_tflops_sustained" in pk else None
    except Exception:
        peak, peak_src, peak_sus = 1590.0, "fallback (B200_PROFILING.md 1.59 PFLOP/s)", None
    # oracle: sampled rows (first, tile / page boundaries, last) of 3 layers, all heads, fp64
    from oracle import attention as o_attn

    rows = [0, 1, 63, 64, 127, 128, 129, 1000, 2047, 2048, n - 2, n - 1]
    layers = [0, L // 2, L - 1]
    kb, vb, qb = workloads.to_bits(k), workloads.to_bits(v), workloads.to_bits(q[layers][:, rows])
    got = o_attn.bf16_bits_to_f64(workloads.to_bits(out[layers][:, rows]))
    lse_np = lse[layers][:, rows].cpu().numpy().astype(np.float64)
    mx, sm, cnt, lse_mx = 0.0, 0.0, 0, 0.0
    t_or = time.perf_counter()
    for a, l in enumerate(layers):
        for b, x in enumerate(rows):
            o_ref, lse_ref, _ = o_attn.attend_retained(qb[a, b], kb[l], vb[l], range(x + 1), 1.0 / math.sqrt(g.head_dim))
            e = np.abs(got[a, b] - o_ref)
            mx, sm, cnt = max(mx, float(e.max())), sm + float(e.sum()), cnt + e.size
            lse_mx = max(lse_mx, float(np.max(np.abs(lse_np[a, b] - lse_ref))))
    t_or = time.perf_counter() - t_or
    pairs = sum(x + 1 for x in rows) * len(layers) * g.n_q_heads
    all_pairs = n * (n + 1) / 2 * L * g.n_q_heads
    cpu_ms = t_or * all_pairs / pairs * 1e3
    clocks = sampler.finish().get("main")
    err = c.last_error()
    c.close()
    line = {
        "metric": "prefill-attn ms per 300 s chunk (causal, 28 layers, 2314 tokens)", "value": ms, "unit": "ms/chunk",
        "n_gpus": 1, "steps": K, "warmup": W, "ms_per_step": ms, "higher_is_better": False, "scaling": "weak",
        "vs_baseline": None, "dtype": "bf16", "data": "synthetic",
        "config": {"workload": "prefill_300s", "tokens": n, "n_layers": L, "n_q_heads": g.n_q_heads, "n_kv_heads": g.n_kv_heads,
                   "head_dim": g.head_dim, "page_size": cfg.page_size, "l2": "q + out = 2 x 464 MB per call (> 126 MB L2); K/V 133 MB"},
        "tflops": tfs, "tokens_per_s": n / (ms * 1e-3),
        "roofline": {"bound": "tensor", "kernel": "prefill_umma_kernel (tcgen05.mma, accumulators in TMEM, TMA-fed)",
                     "achieved": tfs, "peak": peak, "unit": "TFLOP/s", "frac": tfs / peak,
                     "traffic": ncu_traffic_bytes("prefill_300s", PREFILL_SOURCES),
                     "kernel_source_hash": kernel_source_hash(PREFILL_SOURCES),
                     "peak_source": peak_src, "peak_sustained": peak_sus,
                     "frac_of_sustained_peak": (tfs / peak_sus) if peak_sus else None, "algorithmic_flops_per_launch": flops,
                     "how": "causal flops 4 d sum_x (x + 1) per head and layer / mean launch duration (CUDA events, %d launches)" % K},
        "mma_sync_kernel_ms": ms_old, "speedup_vs_mma_sync": ms_old / ms,
        "max_abs_diff_vs_mma_sync": float((out.float() - out_old.float()).abs().max()),
        "cpu_baseline": {"value": cpu_ms, "unit": "ms/chunk", "cores": 1, "kind": "oracle",
                         "sample": f"oracle.attention (numpy fp64) on {len(rows)} query rows x {len(layers)} layers x {g.n_q_heads} heads, "
                                   f"scaled by (query, key) pairs x{all_pairs / pairs:.0f}"},
        "parity": {"max_abs": mx, "mean_abs": sm / cnt, "lse_max_abs": lse_mx, "tol_max_abs": 2e-2, "tol_mean_abs": 2e-3,
                   "ok": bool(mx <= 2e-2 and sm / cnt <= 2e-3 and lse_mx < 2e-3),
                   "compared": f"output of the last timed launch: rows {rows} of layers {layers}, all heads, vs Eq. 1 in fp64"},
        "e2e": {"value": ms, "unit": "ms/chunk", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0,
                "note": "prefill Q/K/V are produced on the device by the model's projections; no host entry exists for this call"},
        "gpu_launches": int(launches), "device_error_word": err, "clocks": clocks,
    }
    print(json.dumps(line), flush=True)
    return 0


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=300)
    ap.add_argument("--warmup", type=int, default=20)
    ap.add_argument("--impl", default="murmur", choices=["murmur", "reference"])
    ap.add_argument("--workload", default="config2")
    ap.add_argument("--e2e-steps", type=int, default=100)
    ap.add_argument("--no-cpu-baseline", action="store_true", help="skip every oracle leg (parity, cpu_baseline, replay, protocol, others)")
    ap.add_argument("--no-protocol", action="store_true", help="skip the whole-decode protocol pass")
    ap.add_argument("--no-others", action="store_true", help="skip the other_workloads block")
    ap.add_argument("--cpu-budget-s", default="12", help="(kept for old command lines; the baseline now times one whole step)")
    ap.add_argument("--ref-budget-s", default="120")
    args = ap.parse_args()
    if args.impl == "reference":
        return run_reference(args)
    if args.workload == "prefill_300s":
        return run_prefill(args)
    return run_murmur(args)


if __name__ == "__main__":
    sys.exit(main())
