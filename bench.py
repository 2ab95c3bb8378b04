#!/usr/bin/env python
"""bench.py - decode-attention us/step and HBM GB/s on the 12 x 300 s-chunk evicted-KV workload.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl murmur|reference] [--workload NAME]

A *step* is one pass of the whole hot path over one batch of synthetic input:
``murmur_decode_step`` = append one token per sequence (all 28 layers) -> evict -> decode attention
(all 28 layers), ONE kernel launch per step by default (MURMUR_OPT_FUSE_STEP; --fuse 1 / 0 give the
two- and three-launch forms).  Prints ONE JSON line (rank 0).

Timed regions (CUDA events on the stream the kernels are launched on, W >= 3 warm-up steps,
barrier + synchronize on both sides, max over ranks):
  A  K consecutive steps, inputs resident in HBM                          -> value, ms_per_step
  B  K more steps with one event pair around every launch                 -> roofline (the fused
     step kernel's average launch duration); then <= 100 steps as three separate API calls
     (append, evict, attention) with one event pair each                  -> per-stage breakdown
  C  K_e steps through murmur_decode_step_host from pinned HOST buffers, stream-synchronised
     every step (the caller reads `out`)                                  -> e2e
Every step re-reads ~575 MB of retained K/V (>> 126 MB L2), so inputs are larger than L2 and no
explicit flush is needed; t advances every step, so windows slide and pages are freed/reused.
After the timed regions rank 0 (N = 1) times the fp64 CPU oracle on a bounded sample of the last
step and compares the GPU output of that step against it (cpu_baseline + parity keys).

Multi-GPU: the path has no exchange step: "replicas only".  Under torchrun every
rank runs an independent replica of the workload on its own GPU; time = max over ranks.

`--impl reference` times the oracle itself (oracle/: Python integer bookkeeping + plain-C fp64
attention) on the host cores, each step a bounded sample of the same workload.
"""
from __future__ import annotations

import argparse
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

# dram__bytes_read.sum + dram__bytes_write.sum of ONE attention launch from the committed
# `ncu --set full` capture (profiles/), keyed by workload; None until a capture exists.
NCU_TRAFFIC_BYTES = {}
try:
    with open(os.path.join(ROOT, "profiles", "traffic.md")) as _f:
        for _ln in _f:
            if _ln.startswith("| `") and _ln.count("|") >= 4:
                _c = [x.strip() for x in _ln.strip().strip("|").split("|")]
                try:
                    NCU_TRAFFIC_BYTES[_c[0].strip("`")] = float(_c[1])
                except ValueError:
                    pass
except OSError:
    pass


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
        self.windows = []
        self.proc = None
        try:
            self.proc = subprocess.Popen([sys.executable, "-c", SAMPLER_SRC, str(dev_index), self.path],
                                         stdout=subprocess.DEVNULL, stderr=subprocess.DEVNULL)
        except Exception:
            self.proc = None

    def window(self, t0: float, t1: float):
        self.windows.append((t0, t1))

    def finish(self) -> dict:
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": [], "note": "sampler unavailable"}
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
        under = [r for r in rows if any(a <= r[0] <= b for a, b in self.windows)]
        if not under:
            return {"sm_mhz": None, "sm_max_mhz": rows[0][2] if rows else None, "reasons": [],
                    "samples": 0, "note": "no sample fell inside a timed region"}
        sms = sorted(r[1] for r in under)
        mask = 0
        for r in under:
            mask |= r[3]
        reasons = [name for bit, name in REASON_BITS.items() if mask & bit and name != "gpu_idle"]
        return {"sm_mhz": sms[len(sms) // 2], "sm_min_mhz": sms[0], "sm_max_mhz": under[0][2], "reasons": reasons,
                "samples": len(under), "power_w_max": max(r[4] for r in under), "how": "NVML polled every ~4 ms"}


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
    import torch

    import workloads
    from oracle import c as oracle_c
    from oracle import paged_cache as o_cache
    from oracle import policy as o_policy

    cfg, t0 = pick_workload(args.workload)
    if t0 is None:
        t0 = 200
    g = cfg.geom
    co = oracle_c.load()
    K, W = args.steps, args.warmup
    n_items_step = cfg.batch * g.n_layers  # (sequence, layer) items of one step
    budget_s = float(args.ref_budget_s)
    # data of sequence 0 only (the sample never leaves it): CPU generator, same recipe
    sd = workloads.SeqData(cfg, 0, device="cpu")
    spec = cfg.seqs[0]
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
    t_start = time.perf_counter()
    for _ in range(K):
        used = step(n_sample)
    el = time.perf_counter() - t_start
    us_step = el / K * (n_items_step / n_sample) * 1e6
    sample = (f"per step: integer bookkeeping of all {cfg.batch} sequences + fp64 attention of sequence 0, layers "
              f"0..{n_sample - 1} (all 28 q heads), scaled x{n_items_step / n_sample:.1f} to the "
              f"{n_items_step} (sequence, layer) items of a step")
    line = {
        "impl": "reference", "metric": METRIC, "value": us_step, "unit": UNIT, "n_gpus": args.gpus, "steps": K,
        "warmup": W, "ms_per_step": us_step / 1e3, "higher_is_better": False, "scaling": "weak",
        "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": cfg.name, "batch": cfg.batch, "n_layers": g.n_layers, "page_size": cfg.page_size,
                   "what": "fp64 CPU oracle (oracle/), bounded sample per step"},
        "cpu_baseline": {"value": us_step, "unit": UNIT, "cores": int(used), "kind": "oracle", "sample": sample},
        "e2e": {"value": us_step, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line), flush=True)
    return 0


# ------------------------------------------------------------------------------------------------
# the CUDA arm
# ------------------------------------------------------------------------------------------------
def run_murmur(args):
    import numpy as np
    import torch

    import workloads
    from paper_2606_01483_b200 import MurmurCache, binding

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
    n_steps_total = W + 2 * K + We + Ke + 1 + (56 if args.per_layer else 0)
    n_gen = min(n_steps_total, 1100)  # distinct pre-generated step inputs (re-used cyclically beyond that)
    Tmin = min(s.T for s in cfg.seqs)
    extra = max(2, t0 + n_steps_total + 2 - Tmin)  # a long --steps run decodes past the config's T
    B = cfg.batch
    ids = np.arange(B, dtype=np.int32)

    cache = MurmurCache(g.n_layers, g.n_q_heads, g.n_kv_heads, g.head_dim, cfg.page_size, B,
                        workloads.max_blocks_per_seq(cfg, extra) + 1, workloads.unevicted_blocks(cfg, extra) + 2,
                        device=dev)
    if args.variant:
        cache.set_option(binding.MURMUR_OPT_ATTN_VARIANT, {"generic": 1, "mma": 2}[args.variant])
    if args.grid:
        cache.set_option(binding.MURMUR_OPT_ATTN_GRID, args.grid)
    if args.no_pdl:
        cache.set_option(binding.MURMUR_OPT_PDL, 0)
    if args.no_fuse:
        cache.set_option(binding.MURMUR_OPT_FUSE_STEP, 0)
    elif args.fuse >= 0:
        cache.set_option(binding.MURMUR_OPT_FUSE_STEP, args.fuse)
    data = [workloads.SeqData(cfg, i, device=dev) for i in range(B)]
    k_steps, v_steps, q_steps = [], [], []
    for i, s in enumerate(cfg.seqs):
        cache.seq_begin(i, s.P, s.S, s.M, s.policy_tuple)
        kp, vp = data[i].prefill_kv()
        ko, vo = data[i].out_kv(0, t0)
        k = torch.cat([kp, ko], dim=1).contiguous()
        v = torch.cat([vp, vo], dim=1).contiguous()
        cache.kv_append([i], [k.shape[1]], k, v)
        del k, v, kp, vp
        ks, vs = data[i].out_kv(t0, t0 + n_gen)  # [L, steps, kv, d]
        k_steps.append(ks)
        v_steps.append(vs)
        q_steps.append(data[i].q_steps(t0 + 1, t0 + n_gen + 1))  # [steps, L, n_q, d]
    cache.kv_evict(ids)
    k_all = torch.stack(k_steps, dim=2).permute(1, 0, 2, 3, 4).contiguous()  # [steps, L, B, kv, d]
    v_all = torch.stack(v_steps, dim=2).permute(1, 0, 2, 3, 4).contiguous()
    q_all = torch.stack(q_steps, dim=2).contiguous()  # [steps, L, B, n_q, d]
    del k_steps, v_steps, q_steps
    out = torch.empty_like(q_all[0])
    scale = 1.0 / math.sqrt(g.head_dim)
    stream = torch.cuda.current_stream()
    step_no = [0]

    def one_step():
        s = step_no[0]
        j = s % n_gen
        cache.decode_step(ids, k_all[j], v_all[j], q_all[j], out, None, scale)
        step_no[0] = s + 1

    def barrier():
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize(dev)

    sampler = ClockSampler(local_rank) if rank == 0 else None

    # spin the clocks up (untimed, state not advanced): repeat attention on the current state
    t_spin = time.perf_counter()
    while time.perf_counter() - t_spin < 0.25:
        for _ in range(20):
            cache.decode_attn(ids, q_all[0], out=out, sm_scale=scale)
        torch.cuda.synchronize(dev)

    for _ in range(W):
        one_step()
    # ---- region A: K steps, whole-step timing -----------------------------------------------
    cache.reset_stats()
    barrier()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    w0 = time.time()
    e0.record(stream)
    for _ in range(K):
        one_step()
    e1.record(stream)
    barrier()
    w1 = time.time()
    ms_a = e0.elapsed_time(e1)
    launches = cache.stats()["kernel_launches"]
    if sampler:
        sampler.window(w0, w1)
    st = cache.stats()
    if args.timeline and rank == 0:  # per-CTA trace of the last attention launch of region A (profiling aid)
        tl = cache.attn_timeline().astype(np.int64)
        t_first = int(tl[:, 0].min())
        tr = cache.step_trace().astype(np.int64)
        with open(args.timeline, "w") as f:
            f.write("# step prologue stamps (ns relative to the first attention CTA start): append_start %d ticket %d "
                    "commit %d evict_start %d evict_end %d | last CTA: wait_done %d state_loaded %d prefix %d loads_issued %d "
                    "tasks %d pages_consumed %d block %d\n" % (tuple(int(x) - t_first for x in tr[:11]) + (int(tr[11]),)))
            f.write("# cta start_ns end_ns smid tiles   (ns relative to the first CTA start)\n")
            for b in range(tl.shape[0]):
                f.write("%d %d %d %d %d\n" % (b, tl[b, 0] - t_first, tl[b, 1] - t_first if tl[b, 1] else -1,
                                            tl[b, 2] - t_first if tl[b, 2] > (1 << 20) else tl[b, 2], tl[b, 3]))

    # ---- region B: K steps with one event pair around every launch --------------------------------
    # B1: the step as the library runs it by default (murmur_decode_step = ONE launch of the fused
    #     step kernel) -> duration of the dominant kernel for `roofline`
    # B2: the same step as three separate calls (append, evict, attention) -> per-stage breakdown
    n_ret_b0 = sum(cache.seq_state(i)["n_retained"] for i in range(B))
    ones = [1] * B
    Kb2 = min(K, 100)
    evs1 = [[torch.cuda.Event(enable_timing=True) for _ in range(2)] for _ in range(K)]
    evs = [[torch.cuda.Event(enable_timing=True) for _ in range(4)] for _ in range(Kb2)]
    barrier()
    w0 = time.time()
    torch.cuda._sleep(int(1e8))  # ~50 ms of GPU spin so the host runs ahead: event pairs then see kernels, not launch gaps
    cache.reset_stats()
    for j in range(K):
        s = step_no[0] % n_gen
        evs1[j][0].record(stream)
        cache.decode_step(ids, k_all[s], v_all[s], q_all[s], out, None, scale)
        evs1[j][1].record(stream)
        step_no[0] += 1
    launches_per_step_b1 = cache.stats()["kernel_launches"] / K
    barrier()
    n_ret_b1 = sum(cache.seq_state(i)["n_retained"] for i in range(B))
    torch.cuda._sleep(int(1e8))
    for j in range(Kb2):
        s = step_no[0] % n_gen
        evs[j][0].record(stream)
        cache.kv_append(ids, ones, k_all[s], v_all[s])
        evs[j][1].record(stream)
        cache.kv_evict(ids)
        evs[j][2].record(stream)
        cache.decode_attn(ids, q_all[s], out=out, sm_scale=scale)
        evs[j][3].record(stream)
        step_no[0] += 1
    barrier()
    w1 = time.time()
    if sampler:
        sampler.window(w0, w1)
    step_list = sorted(e[0].elapsed_time(e[1]) * 1e3 for e in evs1)
    t_stepk = sum(step_list) / K
    t_stepk_med = step_list[K // 2]
    stepk_p10, stepk_p90 = step_list[K // 10], step_list[min(K - 1, (9 * K) // 10)]
    t_app = sum(e[0].elapsed_time(e[1]) for e in evs) / Kb2 * 1e3
    t_evi = sum(e[1].elapsed_time(e[2]) for e in evs) / Kb2 * 1e3
    attn_list = sorted(e[2].elapsed_time(e[3]) * 1e3 for e in evs)
    t_att = sum(attn_list) / Kb2
    t_att_med = attn_list[Kb2 // 2]

    # ---- optional region P: the step as a per-layer engine would issue it -------------------------
    # (layer l's K/V exist only when layer l runs: append(layer l) + attention(layer l), 28 times,
    # with the eviction right after the first layer's append has reserved the slots)
    us_per_layer_mode = None
    if args.per_layer:
        Kp = min(K, 50)
        L = g.n_layers

        def layer_step(s_idx):
            for l in range(L):
                cache.kv_append(ids, ones, k_all[s_idx][l:l + 1], v_all[s_idx][l:l + 1], layer_begin=l, layer_end=l + 1)
                if l == 0:
                    cache.kv_evict(ids)
                cache.decode_attn(ids, q_all[s_idx][l:l + 1], out=out[l:l + 1], sm_scale=scale, layer_begin=l, layer_end=l + 1)

        for _ in range(3):
            layer_step(step_no[0] % n_gen)
            step_no[0] += 1
        barrier()
        p0, p1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        p0.record(stream)
        for _ in range(Kp):
            layer_step(step_no[0] % n_gen)
            step_no[0] += 1
        p1.record(stream)
        barrier()
        us_per_layer_mode = p0.elapsed_time(p1) / Kp * 1e3

    # ---- region C: end to end from pinned host buffers -------------------------------------------
    s0 = step_no[0]
    sel = torch.arange(s0, s0 + We + Ke, device=dev) % n_gen
    # per step: k_new | v_new | q packed back to back in one pinned block (moved with ONE host-to-device copy)
    kv_n, q_n = k_all[0].numel(), q_all[0].numel()
    hb = torch.empty((We + Ke, 2 * kv_n + q_n), dtype=torch.bfloat16).pin_memory()
    hb[:, :kv_n] = k_all[sel].reshape(We + Ke, -1).cpu()
    hb[:, kv_n:2 * kv_n] = v_all[sel].reshape(We + Ke, -1).cpu()
    hb[:, 2 * kv_n:] = q_all[sel].reshape(We + Ke, -1).cpu()
    kh = [hb[j, :kv_n].view(k_all[0].shape) for j in range(We + Ke)]
    vh = [hb[j, kv_n:2 * kv_n].view(v_all[0].shape) for j in range(We + Ke)]
    qh = [hb[j, 2 * kv_n:].view(q_all[0].shape) for j in range(We + Ke)]
    oh = torch.empty(out.shape, dtype=torch.bfloat16).pin_memory()
    for j in range(We):
        cache.decode_step_host(ids, kh[j], vh[j], qh[j], oh, scale)
        torch.cuda.synchronize(dev)
    barrier()
    c0, c1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
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
    us_e2e_dev = c0.elapsed_time(c1) / Ke * 1e3
    us_e2e_wall = (w1 - w0) / Ke * 1e6
    us_e2e = max(us_e2e_dev, us_e2e_wall)
    step_no[0] = s0 + We + Ke
    h2d = (kh[0].numel() + vh[0].numel() + qh[0].numel()) * 2
    d2h = oh.numel() * 2
    clocks = sampler.finish() if sampler else None

    # ---- reduce over ranks ---------------------------------------------------------------------
    us_step = ms_a / K * 1e3
    us_step, us_e2e, t_att, t_app, t_evi, t_att_med, t_stepk, t_stepk_med = max_over_ranks(
        [us_step, us_e2e, t_att, t_app, t_evi, t_att_med, t_stepk, t_stepk_med], dist, dev)

    # ---- algorithmic bytes of one attention launch ------------------------------
    # retained tokens per launch: the device's own |A(t)|, mean of the first and last step of region B
    n_ret = (n_ret_b0 + n_ret_b1) // 2
    kv_bytes = n_ret * BYTES_PER_TOKEN_LAYER * g.n_layers
    qo_bytes = 2 * g.n_layers * B * g.n_q_heads * g.head_dim * 2
    alg_bytes = kv_bytes + qo_bytes
    peak, peak_src = load_peak()
    # dominant kernel of the timed step: the fused step kernel when the step is one launch, else the
    # attention kernel of the multi-launch step
    one_launch = launches_per_step_b1 < 1.5
    if one_launch:
        # region A is K back-to-back launches of this one kernel: its average launch duration over the
        # timed region is region A's time / K (consecutive launches overlap their set-up through PDL);
        # the event-pair-per-launch figure of region B1 (no overlap, includes the launch gap) is kept beside it
        dom_kernel, dom_us, dom_med = "attn_mma_kernel<step> (append + evict + attention, one launch)", us_step, t_stepk_med
    else:
        dom_kernel = "attn_mma_kernel" if st["attn_variant"] == 2 else "attn_generic_kernel"
        dom_us, dom_med = t_att, t_att_med
    achieved = alg_bytes / (dom_us * 1e-6) / 1e9
    attn_only = alg_bytes / (t_att * 1e-6) / 1e9
    traffic = NCU_TRAFFIC_BYTES.get(cfg.name)
    roofline = {"bound": "hbm", "kernel": dom_kernel,
                "achieved": achieved, "peak": peak, "unit": "GB/s", "frac": achieved / peak, "traffic": traffic,
                "peak_source": peak_src, "algorithmic_bytes_per_launch": alg_bytes,
                "avg_launch_us": dom_us, "median_launch_us": dom_med, "isolated_launch_us": t_stepk if one_launch else t_att,
                "how": ("region A time / K launches (one launch per step, CUDA events around the K steps)" if one_launch
                        else "mean of per-launch CUDA event pairs (region B2)"),
                "frac_of_nominal_8000": achieved / 8000.0}

    # ---- CPU oracle on a bounded sample of the last step + parity of that step -----------------
    cpu_baseline, parity = None, None
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        # K/V of sequence 0 exactly as appended: prefill + first t0 outputs, then the step inputs in order
        kp, vp = data[0].prefill_kv()
        ko, vo = data[0].out_kv(0, t0)
        order = torch.arange(step_no[0], device=dev) % n_gen
        k_seq0 = torch.cat([kp, ko, k_all[order][:, :, 0].permute(1, 0, 2, 3)], dim=1)  # [L, n_pos, kv, d]
        v_seq0 = torch.cat([vp, vo, v_all[order][:, :, 0].permute(1, 0, 2, 3)], dim=1)
        cpu_baseline, parity = oracle_sample(cfg, cache, k_seq0, v_seq0, ids, q_all[(step_no[0] - 1) % n_gen], scale,
                                             t0 + step_no[0], dev, float(args.cpu_budget_s))
    err = cache.last_error()
    cache.close()
    if dist is not None:
        dist.destroy_process_group()
    if rank != 0:
        return 0
    line = {
        "metric": METRIC, "value": us_step, "unit": UNIT, "n_gpus": world, "steps": K, "warmup": W,
        "ms_per_step": us_step / 1e3, "higher_is_better": False, "scaling": "weak", "vs_baseline": None,
        "dtype": "bf16", "data": "synthetic",
        "config": dict({"workload": cfg.name, "batch": B, "n_layers": g.n_layers, "n_q_heads": g.n_q_heads,
                        "n_kv_heads": g.n_kv_heads, "head_dim": g.head_dim, "page_size": cfg.page_size,
                        "retained_tokens_per_seq": n_ret // B, "t_first_timed": t0 + W + 1,
                        "l2": "inputs larger than L2 (each step re-reads %.0f MB of K/V)" % (kv_bytes / 1e6),
                        "parallelism": "replicas only" if world > 1 else "single GPU"},
                       **({"speech_tokens": cfg.seqs[0].S, "prefix_tokens": cfg.seqs[0].P,
                           "w_speech": cfg.seqs[0].w_speech, "w_out": cfg.seqs[0].w_out, "delay": cfg.seqs[0].delay,
                           "n_sink_out": cfg.seqs[0].n_sink_out}
                          if len({(x.S, x.w_speech, x.w_out) for x in cfg.seqs}) == 1 else
                          {"ragged": True, "speech_tokens": [min(x.S for x in cfg.seqs), max(x.S for x in cfg.seqs)],
                           "prefix_tokens": cfg.seqs[0].P, "w_speech": sorted({x.w_speech for x in cfg.seqs}),
                           "w_out": sorted({x.w_out for x in cfg.seqs}), "n_sink_out": cfg.seqs[0].n_sink_out,
                           "note": "all sequences kept active at a common t (the full-batch point of config 5)"})),
        "tokens_per_s": whole_job_tokens_per_s(world, B, us_step),
        "step_kernel_us": t_stepk, "step_kernel_us_p10_p50_p90": [stepk_p10, t_stepk_med, stepk_p90],
        "launches_per_step": launches_per_step_b1,
        "separate_calls": {"append_us": t_app, "evict_us": t_evi, "attn_us": t_att, "attn_median_us": t_att_med,
                           "attn_hbm_gbs": attn_only, "attn_pct_of_measured_peak": 100.0 * attn_only / peak,
                           "note": "the same step as three API calls, one event pair per call (includes launch gaps)"},
        "per_layer_mode_us": us_per_layer_mode,
        "attn_us": t_att, "append_us": t_app, "evict_us": t_evi,
        "attn_hbm_gbs": attn_only, "attn_pct_of_measured_peak": 100.0 * attn_only / peak,
        "step_hbm_gbs": alg_bytes / (us_step * 1e-6) / 1e9,
        "roofline": roofline, "cpu_baseline": cpu_baseline, "parity_last_step": parity,
        "e2e": {"value": us_e2e, "unit": UNIT, "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h,
                "device_us": us_e2e_dev, "wall_us": us_e2e_wall, "steps": Ke,
                "api": "murmur_decode_step_host (pinned host k_new | v_new | q packed in one block -> one H2D copy, one launch, "
                       "one D2H copy of out), stream-synchronised per step"},
        "gpu_launches": int(launches), "attn_grid": st["attn_grid"], "attn_smem_bytes": st["attn_smem_bytes"],
        "device_error_word": err, "clocks": clocks,
        "paper_context": "paper reports end-to-end only: 88.43 s (chunked + speech eviction) vs 370.73 s single pass, "
                         "1x H100 80GB, batch 16, AMI-IHM (PAPER.md:201-206)",
    }
    print(json.dumps(line), flush=True)
    return 0


def oracle_sample(cfg, cache, k_seq0, v_seq0, ids, q_last, scale, t_now, dev, budget_s):
    """Times oracle (policy + plain-C fp64 attention) on sequence 0 of the last step, as many layers
    as fit the budget, and compares the GPU output of the same step with it."""
    import numpy as np
    import torch

    import workloads
    from oracle import attention as o_attn
    from oracle import c as oracle_c
    from oracle import policy as o_policy

    g = cfg.geom
    co = oracle_c.load()
    spec = cfg.seqs[0]
    out = cache.decode_attn(ids, q_last, sm_scale=scale)  # recompute the last step's output (state unchanged)
    torch.cuda.synchronize(dev)
    got = o_attn.bf16_bits_to_f64(workloads.to_bits(out[:, 0]))  # [L, n_q, d]
    k_bits = workloads.to_bits(k_seq0)
    v_bits = workloads.to_bits(v_seq0)
    assert k_bits.shape[1] == spec.P + spec.S + spec.M + t_now
    q_bits = workloads.to_bits(q_last[:, 0])
    t_or = time.perf_counter()
    ret = o_policy.retained_positions(spec.P, spec.S, spec.M, t_now, o_policy.Policy(*spec.policy_tuple))
    t_policy = time.perf_counter() - t_or
    assert list(cache.retained(0)) == list(ret), "retained set differs from the oracle"
    # calibrate on one layer, then as many layers as fit the budget
    tc = time.perf_counter()
    o1, _, used = co.attend(q_bits[:1], k_bits[:1], v_bits[:1], ret, scale)
    per_layer = max(time.perf_counter() - tc, 1e-5)
    n_l = int(max(1, min(g.n_layers, budget_s / per_layer)))
    best = None
    for _ in range(2 if per_layer * n_l < budget_s / 2 else 1):
        tc = time.perf_counter()
        o_ref, _, used = co.attend(q_bits[:n_l], k_bits[:n_l], v_bits[:n_l], ret, scale)
        el = time.perf_counter() - tc
        best = el if best is None else min(best, el)
    n_items = cfg.batch * g.n_layers
    us_step = (best / n_l * n_items + t_policy * cfg.batch) * 1e6
    # the same oracle on ONE thread, on a slice small enough for ~2 s
    n_l1 = int(max(1, min(n_l, 2.0 / max(per_layer * used, 1e-5))))
    tc = time.perf_counter()
    co.attend(q_bits[:n_l1], k_bits[:n_l1], v_bits[:n_l1], ret, scale, n_threads=1)
    us_step_1t = ((time.perf_counter() - tc) / n_l1 * n_items + t_policy * cfg.batch) * 1e6
    e = np.abs(got[:n_l] - o_ref)
    parity = {"max_abs": float(e.max()), "mean_abs": float(e.mean()), "tol_max_abs": 2e-2, "tol_mean_abs": 2e-3,
              "compared": f"sequence 0, layers 0..{n_l - 1}, all {g.n_q_heads} heads of the last step (t={t_now}); "
                          "retained set bit-exact"}
    cpu = {"value": us_step, "unit": UNIT, "cores": int(used), "kind": "oracle", "single_thread_value": us_step_1t,
           "sample": f"oracle.policy retained set + plain-C fp64 attention (oracle/c) of sequence 0, layers 0..{n_l - 1} of "
                     f"the last step ({len(ret)} retained tokens), best of runs, scaled x{n_items / n_l:.1f} to the "
                     f"{n_items} (sequence, layer) items of a step; host cores = {os.cpu_count()}"}
    return cpu, parity


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=300)
    ap.add_argument("--warmup", type=int, default=20)
    ap.add_argument("--impl", default="murmur", choices=["murmur", "reference"])
    ap.add_argument("--workload", default="config2")
    ap.add_argument("--e2e-steps", type=int, default=100)
    ap.add_argument("--variant", default="", choices=["", "generic", "mma"])
    ap.add_argument("--grid", type=int, default=0)
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--per-layer", action="store_true",
                    help="also time the step issued layer by layer (append(l) + attention(l) x 28, 57 launches)")
    ap.add_argument("--no-pdl", action="store_true", help="A/B: launch the step's kernels without programmatic dependent launch")
    ap.add_argument("--fuse", type=int, default=-1, help="A/B: MURMUR_OPT_FUSE_STEP value (2 = one launch per step, default)")
    ap.add_argument("--no-fuse", action="store_true", help="A/B: murmur_decode_step as three launches (append, evict, attention)")
    ap.add_argument("--timeline", default="", help="write the per-CTA trace of one attention launch to this file")
    ap.add_argument("--cpu-budget-s", default="12")
    ap.add_argument("--ref-budget-s", default="120")
    args = ap.parse_args()
    if args.impl == "reference":
        return run_reference(args)
    return run_murmur(args)


if __name__ == "__main__":
    sys.exit(main())
