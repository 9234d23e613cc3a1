#!/usr/bin/env python
"""bench.py -- MoE-layer tokens/s of the grouped (and ungrouped) layer on B200, % of roofline.

A "step" is one pass of the whole hot path (bm_route + bm_moe_forward: SURVEY.md 8(a) rows 1-13) over one
batch of synthetic tokens.  Headline workload at N=1: BASELINE.json configs[2] (Mixtral-8x7B-shaped prefill
layer, T=8192, G=4 united groups) -- BASELINE.json's metric names no config, so the largest single-GPU one is
taken; it is the tensor-bound regime.  The HBM-bound regime, configs[1] (the same layer as a T=64 decode batch),
is measured in the same run and reported in `roofline.decode` / `roofline_decode` / `decode`; both layers are
also run ungrouped (G=8, identity map) for the speed-up ratio.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--no-extras]

For N>1 launch under torchrun (one rank per GPU); tokens are sharded across ranks with no data-path
collective (weak scaling: every rank runs the same layer on its own batch).
Prints ONE JSON line on rank 0.
"""
from __future__ import annotations

import argparse
import json
import os
import statistics
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import numpy as np
import torch

from bm_inputs import CONFIGS, bf16_bits, get_config, identity_variant, make_layer

METRIC = "moe_layer_tokens_per_s"
UNIT = "tokens/s"
L2_BYTES = 126e6


# ---------------------------------------------------------------------------------------------------
# peaks, roofline arithmetic
# ---------------------------------------------------------------------------------------------------
def load_peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        with open(path) as fh:
            p = json.load(fh)
        return dict(hbm_gbs=float(p["hbm_gbs"]), bf16_tflops=float(p["bf16_tflops"]),
                    bf16_tflops_sustained=float(p.get("bf16_tflops_sustained", p["bf16_tflops"])),
                    source="measured (MEASURED_PEAKS.json)")
    # B200_PROFILING.md fallback: an earlier measurement on this pool
    return dict(hbm_gbs=6650.0, bf16_tflops=1590.0, bf16_tflops_sustained=1400.0, source="fallback (B200_PROFILING.md)")


def layer_work(cfg, A, G_act):
    """Algorithmic FLOPs and bytes of one layer call; H, xs and split-K partials are
    implementation traffic and are not counted."""
    T, D, F, E, S = cfg.T, cfg.D, cfg.F, cfg.E, cfg.S
    flops = A * 6 * D * F + S * T * 6 * D * F + 2 * T * E * D
    nbytes = (G_act + S) * 3 * D * F * 2 + T * D * 2 + T * D * 2 + E * D * 2
    return flops, nbytes


def gemm1_work(cfg, A, G_act):
    """Algorithmic work of the dominant kernel (GEMM1 + SwiGLU): W1, W3 of the active groups once, the
    gathered rows in, H out (bf16)."""
    T, D, F, S = cfg.T, cfg.D, cfg.F, cfg.S
    rows = A + S * T
    return rows * 4 * D * F, (G_act + S) * 2 * D * F * 2 + rows * D * 2 + rows * F * 2


# ---------------------------------------------------------------------------------------------------
# clocks during the timed region (NVML polling thread)
# ---------------------------------------------------------------------------------------------------
class ClockSampler:
    REASONS = {0x1: "gpu_idle", 0x2: "applications_clocks_setting", 0x4: "sw_power_cap", 0x8: "hw_slowdown",
               0x10: "sync_boost", 0x20: "sw_thermal_slowdown", 0x40: "hw_thermal_slowdown",
               0x80: "hw_power_brake_slowdown", 0x100: "display_clock_setting"}

    def __init__(self, index: int):
        self.samples, self.reasons, self.ok = [], set(), False
        self._stop = threading.Event()
        try:
            import pynvml
            pynvml.nvmlInit()
            self.nv = pynvml
            vis = os.environ.get("CUDA_VISIBLE_DEVICES")
            phys = index
            if vis:
                ids = [v for v in vis.split(",") if v.strip()]
                if index < len(ids) and ids[index].strip().isdigit():
                    phys = int(ids[index])
            self.h = pynvml.nvmlDeviceGetHandleByIndex(phys)
            self.max_mhz = int(pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM))
            self.ok = True
        except Exception as exc:  # NVML missing: report that clocks were not sampled
            self.err = repr(exc)
            self.max_mhz = None

    def _run(self):
        nv = self.nv
        while not self._stop.is_set():
            try:
                self.samples.append(int(nv.nvmlDeviceGetClockInfo(self.h, nv.NVML_CLOCK_SM)))
                mask = int(nv.nvmlDeviceGetCurrentClocksEventReasons(self.h)) if hasattr(
                    nv, "nvmlDeviceGetCurrentClocksEventReasons") else int(nv.nvmlDeviceGetCurrentClocksThrottleReasons(self.h))
                for bit, name in self.REASONS.items():
                    if mask & bit and name != "gpu_idle":
                        self.reasons.add(name)
            except Exception:
                pass
            self._stop.wait(0.005)

    def __enter__(self):
        if self.ok:
            self.t = threading.Thread(target=self._run, daemon=True)
            self.t.start()
        return self

    def __exit__(self, *a):
        if self.ok:
            self._stop.set()
            self.t.join()

    def summary(self):
        if not self.ok or not self.samples:
            return {"sm_mhz": None, "sm_max_mhz": self.max_mhz, "reasons": [], "note": "NVML sampling unavailable"}
        return {"sm_mhz": statistics.median(self.samples), "sm_max_mhz": self.max_mhz,
                "reasons": sorted(self.reasons), "samples": len(self.samples)}


# ---------------------------------------------------------------------------------------------------
# distributed plumbing
# ---------------------------------------------------------------------------------------------------
def dist_env():
    return int(os.environ.get("RANK", 0)), int(os.environ.get("LOCAL_RANK", 0)), int(os.environ.get("WORLD_SIZE", 1))


def barrier(ws):
    if ws > 1:
        torch.distributed.barrier()


def max_over_ranks(v: float, ws: int, device) -> float:
    if ws == 1:
        return v
    t = torch.tensor([v], dtype=torch.float64, device=device)
    torch.distributed.all_reduce(t, op=torch.distributed.ReduceOp.MAX)
    return float(t.item())


# ---------------------------------------------------------------------------------------------------
# our arm
# ---------------------------------------------------------------------------------------------------
class DeviceLayer:
    """One layer resident in HBM: weights, router, group map, workspace, routing arrays."""

    def __init__(self, cfg, seed, x_seed, weights_from=None, keep_host_weights=False, tp=None):
        import paper_2607_04164_b200 as bm
        self.bm, self.cfg = bm, cfg
        self.tp = tp                       # (rank, world): tensor parallelism over F, else None
        L = make_layer(cfg, seed, weights=weights_from is None)
        if tp is not None:
            L.W1, L.W3, L.W2 = bm.shard_f(L.W1, L.W3, L.W2, *tp)
        if x_seed != seed:   # ranks share the layer, not the tokens
            L.x = make_layer(cfg, x_seed, weights=False).x
        self.host = L
        self.x = L.x.cuda()
        self.W_router = L.W_router.cuda()
        self.bias = None if L.router_bias is None else L.router_bias.cuda()
        self.gmap = L.group_map.cuda()
        if weights_from is None:
            self.W1, self.W3, self.W2 = L.W1.cuda(), L.W3.cuda(), L.W2.cuda()
            if not keep_host_weights:
                L.W1 = L.W3 = L.W2 = None      # free the host copies (1.4 - 2.8 GB)
        else:
            self.W1, self.W3, self.W2 = weights_from.W1, weights_from.W3, weights_from.W2
        self.ws = bm.alloc_workspace(cfg.T, cfg.D, cfg.F, cfg.E, cfg.K, cfg.G, cfg.S)
        self.routing = bm.Routing(cfg.T, cfg.K, cfg.G)
        self.out = torch.empty((cfg.T, cfg.D), dtype=torch.bfloat16, device="cuda")
        self.x_pinned = L.x.pin_memory()
        self.out_pinned = torch.empty((cfg.T, cfg.D), dtype=torch.bfloat16).pin_memory()
        self.x_stage = torch.empty_like(self.x)
        self.partial = (torch.empty((cfg.T, cfg.D), dtype=torch.float32, device="cuda") if tp is not None else None)

    def step(self):
        bm, c = self.bm, self.cfg
        if self.tp is not None:     # F-sharded weights: fp32 partial, NCCL all-reduce, one rounding
            bm.bm_route(self.x, self.W_router, self.bias, c.K, self.gmap, c.G, self.routing, self.ws)
            bm.tp_moe_forward(self.x, self.routing, self.W1, self.W3, self.W2, self.out, self.ws, S=c.S, partial=self.partial)
        else:                       # the whole hot path: bm_route + bm_moe_forward (one call; one kernel for single-token decode)
            bm.bm_moe_layer(self.x, self.W_router, self.bias, c.K, self.gmap, c.G, self.W1, self.W3, self.W2, self.out,
                            self.routing, self.ws, S=c.S)

    def step_host(self):
        bm, c = self.bm, self.cfg
        bm.bm_moe_layer_host(self.x_pinned, self.W_router, self.bias, c.K, self.gmap, c.G, self.W1, self.W3, self.W2,
                             c.S, self.out_pinned, self.x_stage, self.out, self.routing, self.ws)

    def realised(self):
        counts = self.routing.counts.cpu().numpy()
        return int(counts.sum()), int((counts > 0).sum()), counts.tolist()


def timed_loop(fn, steps, warmup, ws, device, sampler=None):
    """W warm-up steps, then exactly `steps` steps between barrier+synchronize, timed with CUDA events on
    the launching stream; returns the max over ranks in seconds."""
    for _ in range(warmup):
        fn()
    torch.cuda.synchronize()
    barrier(ws)
    torch.cuda.synchronize()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    ctx = sampler if sampler is not None else _Null()
    with ctx:
        e0.record()
        for _ in range(steps):
            fn()
        e1.record()
        torch.cuda.synchronize()
    barrier(ws)
    torch.cuda.synchronize()
    return max_over_ranks(e0.elapsed_time(e1) / 1e3, ws, device)


class _Null:
    def __enter__(self):
        return self

    def __exit__(self, *a):
        return False


def settle(fn, seconds):
    """Run `fn` back to back for at least `seconds` of wall time (clocks and power settle into the steady state a
    long-running job sees: a tensor-bound kernel on this 1 kW part sits on the power cap after a few hundred ms).
    Returns (steps run, seconds per step)."""
    torch.cuda.synchronize()
    t0 = time.perf_counter()
    n = 0
    while True:
        for _ in range(4):
            fn()
        n += 4
        torch.cuda.synchronize()
        dt = time.perf_counter() - t0
        if dt >= seconds:
            return n, dt / n


def kernel_breakdown(layer, seconds, step_guess_s):
    """Average device time per step of every kernel kind, each launch bracketed by CUDA events recorded inside the
    library on the launching stream (bm_profile_*, which also switches programmatic dependent launch off, so the
    kernels run one after the other) over >= `seconds` of steps.  Returns ({kind: us per step}, steps)."""
    bm = layer.bm
    n = max(3, min(2000, int(seconds / max(step_guess_s, 1e-6)) + 1))
    bm.profile_enable("all", n * 8 + 16)
    for _ in range(2):
        layer.step()
    torch.cuda.synchronize()
    bm.profile_read_kinds()
    for _ in range(n):
        layer.step()
    torch.cuda.synchronize()
    kinds = bm.profile_read_kinds()
    bm.profile_enable(None)
    return {k: ms * 1e3 / n for k, (ms, cnt) in kinds.items()}, n


def roofline_times(cfg, A, G_act, peaks):
    flops, nbytes = layer_work(cfg, A, G_act)
    t_flop = flops / (peaks["bf16_tflops"] * 1e12)
    t_hbm = nbytes / (peaks["hbm_gbs"] * 1e9)
    return flops, nbytes, t_flop, t_hbm


def measure(layer, steps, warmup, ws, device, peaks, sampler=None, with_e2e=True, settle_s=0.5, sustain_s=1.0,
            profile_s=0.5):
    """One workload, four timed regions on the same resident layer:
      contract   exactly `steps` steps after `warmup` (+ >= settle_s of clock settling) steps  -> value / ms_per_step
      sustained  >= sustain_s of back-to-back steps (NVML clocks sampled)                       -> roofline fractions
      kernels    >= profile_s with every launch bracketed by events, PDL off                    -> per-kernel times
      e2e        through bm_moe_layer_host (pinned host x -> device -> layer -> host out)
    and the reconciliation  sum of per-kernel times (serialised) >= step (PDL on) >= dominant kernel."""
    cfg = layer.cfg
    bm = layer.bm
    tp = getattr(layer, "tp", None)
    n_settle, t_guess = settle(layer.step, settle_s)
    l0 = bm.launch_count()
    t = timed_loop(layer.step, steps, warmup, ws, device, sampler)
    launches_per_step = (bm.launch_count() - l0) // (steps + warmup)
    status = bm.bm_device_status(layer.ws)
    A, G_act, counts = layer.realised()
    flops, nbytes, t_flop, t_hbm = roofline_times(cfg, A, G_act, peaks)
    if tp is not None:      # F sharded over ws GPUs: the roofline of the whole job has ws x the peaks
        t_flop, t_hbm = t_flop / ws, t_hbm / ws
    t_step = t / steps
    n_rep = 1 if tp is not None else ws      # tp: all ranks work on the same tokens
    # sustained region
    n_sus = max(steps, int(sustain_s / max(t_step, 1e-6)) + 1)
    sus_sampler = ClockSampler(torch.cuda.current_device())
    t_sus = timed_loop(layer.step, n_sus, 0, ws, device, sus_sampler) / n_sus
    bound = "hbm" if t_hbm >= t_flop else "tensor"
    t_flop_sus = flops / (peaks["bf16_tflops_sustained"] * 1e12) / (ws if tp is not None else 1)
    res = dict(tokens_per_s=n_rep * cfg.T / t_step, ms_per_step=t_step * 1e3, A=A, G_act=G_act, counts=counts,
               flops=flops, bytes=nbytes, t_flop_us=t_flop * 1e6, t_hbm_us=t_hbm * 1e6, bound=bound,
               roofline_frac=max(t_flop, t_hbm) / t_sus, roofline_frac_contract_region=max(t_flop, t_hbm) / t_step,
               roofline_frac_vs_sustained_peak=max(t_flop_sus, t_hbm) / t_sus,
               sustained=dict(steps=n_sus, seconds=t_sus * n_sus, us_per_step=t_sus * 1e6,
                              tokens_per_s=n_rep * cfg.T / t_sus, clocks=sus_sampler.summary()),
               settle_steps=n_settle, achieved_gbs=nbytes / t_sus / 1e9, achieved_tflops=flops / t_sus / 1e12,
               launches_per_step=launches_per_step, gpu_launches=launches_per_step * steps, device_status=status)
    if with_e2e and tp is None:
        n_e = max(3, min(steps, int(0.5 / max(t_step * 3, 1e-6)) + 1))
        te = timed_loop(layer.step_host, n_e, 3, ws, device)
        res["e2e_tokens_per_s"] = n_rep * cfg.T / (te / n_e)
        res["e2e_steps"] = n_e
    # per-kernel times in the same steady state (PDL off: kernels serialised)
    if tp is None:
        kinds, n_prof = kernel_breakdown(layer, profile_s, t_sus)
        kflops, kbytes = gemm1_work(cfg, A, G_act)
        k1 = kinds["gemm1"] / 1e6
        res["gemm1"] = dict(avg_us=kinds["gemm1"], launches_timed=n_prof, alg_bytes=kbytes, alg_flops=kflops,
                            gbs=kbytes / k1 / 1e9, tflops=kflops / k1 / 1e12)
        res["gemm2"] = dict(avg_us=kinds["gemm2"], launches_timed=n_prof)
        res["breakdown_us"] = kinds
        total = sum(kinds.values())
        dominant = max(kinds.values())
        ok = total >= 0.97 * t_sus * 1e6 and t_sus * 1e6 >= 0.97 * dominant
        res["reconcile"] = dict(sum_kernels_us=total, step_us=t_sus * 1e6, dominant_us=dominant,
                                sum_over_step=total / (t_sus * 1e6), dominant_over_step=dominant / (t_sus * 1e6), ok=ok,
                                rule="sum of per-kernel times (events per launch, PDL off) >= step (PDL on) >= dominant kernel, 3% slack")
        if not ok:
            sys.stderr.write(f"bench.py: kernel times do not reconcile with the step for {cfg.name}: {res['reconcile']}\n")
    return res


def roofline_block(cfg_key, m, peaks):
    """The judged roofline object for one measured workload: the dominant kernel (GEMM1 + SwiGLU)."""
    g1 = m["gemm1"]
    traffic, traffic_src = load_traffic(cfg_key + "_gemm1")
    if m["bound"] == "hbm":
        roof = dict(bound="hbm", achieved=g1["gbs"], peak=peaks["hbm_gbs"], unit="GB/s", frac=g1["gbs"] / peaks["hbm_gbs"])
    else:
        roof = dict(bound="tensor", achieved=g1["tflops"], peak=peaks["bf16_tflops"], unit="TFLOP/s",
                    frac=g1["tflops"] / peaks["bf16_tflops"], peak_sustained=peaks["bf16_tflops_sustained"],
                    frac_of_sustained_peak=g1["tflops"] / peaks["bf16_tflops_sustained"])
    roof.update(traffic=traffic, traffic_source=traffic_src, kernel="gemm_kernel<GEMM1+SwiGLU>", avg_launch_us=g1["avg_us"],
                launches_timed=g1["launches_timed"], alg_bytes_per_launch=g1["alg_bytes"], alg_flops_per_launch=g1["alg_flops"],
                peak_source=peaks["source"], peak_kind="burst (bf16_tflops / hbm_gbs of MEASURED_PEAKS.json); the kernel is "
                "timed inside a >= 0.5 s run of whole steps, so frac_of_sustained_peak is the like-for-like figure",
                layer_frac=m["roofline_frac"], layer_frac_vs_sustained_peak=m["roofline_frac_vs_sustained_peak"],
                layer_bound=m["bound"], layer_us_per_step=m["sustained"]["us_per_step"],
                layer_tokens_per_s=m["sustained"]["tokens_per_s"], layer_timed_seconds=m["sustained"]["seconds"],
                clocks=m["sustained"]["clocks"], workload=cfg_key, reconcile=m.get("reconcile"))
    return roof


def load_traffic(kind):
    """(dram bytes per launch of the dominant kernel, where the figure comes from).  The bytes are
    dram__bytes_read.sum + dram__bytes_write.sum of one `ncu --set full` capture (never taken inside a timed run: ncu
    replays kernels); profiles/traffic.json names the capture and the commit it was taken on."""
    path = os.path.join(ROOT, "profiles", "traffic.json")
    if os.path.exists(path):
        try:
            with open(path) as fh:
                d = json.load(fh)
            return d.get(kind), d.get("_source", "profiles/traffic.json")
        except Exception:
            pass
    return None, "no ncu capture committed for this kernel/config"


def cpu_baseline(L, budget_s=20.0):
    """The oracle as it stands (never tuned for this), timed on this box's host cores on a bounded sample
    of the same workload: whole batches of the layer if one takes seconds, else a token prefix."""
    import oracle
    cfg = L.cfg
    xb, wr = bf16_bits(L.x), bf16_bits(L.W_router)
    bias = None if L.router_bias is None else L.router_bias.numpy()
    W1, W3, W2 = bf16_bits(L.W1), bf16_bits(L.W3), bf16_bits(L.W2)
    gm = L.group_map.numpy()
    cores = oracle.num_threads()

    def run(n):
        t0 = time.perf_counter()
        r = oracle.route(xb[:n], wr, bias, cfg.K, gm, cfg.G)
        oracle.moe_forward(xb[:n], r, W1, W3, W2, cfg.S)
        return time.perf_counter() - t0

    n0 = min(cfg.T, max(2, cores // max(cfg.K, 1)))
    t_probe = run(n0)                                   # also warms the page cache
    n = int(min(cfg.T, max(n0, n0 * budget_s / max(t_probe, 1e-3))))
    reps = max(1, int(budget_s / max(t_probe * n / n0, 1e-3))) if n == cfg.T else 1
    t = sum(run(n) for _ in range(reps))
    return dict(value=n * reps / t, unit=UNIT, cores=cores, kind="oracle",
                sample=f"{reps} x the first {n} of {cfg.T} tokens of '{cfg.name}' (oracle route + forward), {t:.1f} s")


CFG_INDEX = {"tiny": 0, "decode": 1, "prefill": 2, "finegrained": 3}


def run_ours(args):
    rank, local_rank, ws = dist_env()
    torch.cuda.set_device(local_rank)
    device = torch.device("cuda", local_rank)
    if ws > 1:
        torch.distributed.init_process_group("nccl", device_id=device)
    import paper_2607_04164_b200 as bm
    bm.lib()
    peaks = load_peaks()
    headline = args.config == "headline"
    main_key = "prefill" if headline else args.config
    cfg = get_config(main_key)
    steps, warmup = args.steps, max(args.warmup, 3)

    tp = (rank, ws) if (args.parallel == "tp" and ws > 1) else None
    # dp: every rank its own tokens (weak scaling); tp: the same tokens on every rank, F sharded (strong scaling)
    layer = DeviceLayer(cfg, seed=0, x_seed=0 if tp else rank, keep_host_weights=(rank == 0 and ws == 1 and not args.no_cpu), tp=tp)
    sampler = ClockSampler(local_rank)
    main = measure(layer, steps, warmup, ws, device, peaks, sampler)
    clocks = sampler.summary()

    extras = {}
    dec = None
    if headline and tp is None:
        # the HBM-bound regime on the same layer (BJ:configs[1], T = 64): shares the weights already in HBM
        dl = DeviceLayer(CONFIGS["decode"], seed=0, x_seed=rank, weights_from=layer)
        dec = measure(dl, max(steps, 200), warmup, ws, device, peaks, sustain_s=0.5)
        del dl
    if not args.no_extras and ws == 1:
        # the ungrouped comparison runs (zero brownout: G = E, identity map)
        ul = DeviceLayer(identity_variant(cfg), seed=0, x_seed=rank)
        extras[main_key + "_ungrouped"] = measure(ul, steps, warmup, ws, device, peaks, with_e2e=False, sustain_s=0.5, profile_s=0.25)
        extras[main_key + "_grouped_over_ungrouped"] = (main["sustained"]["tokens_per_s"] /
                                                        extras[main_key + "_ungrouped"]["sustained"]["tokens_per_s"])
        if headline:
            udl = DeviceLayer(identity_variant(CONFIGS["decode"]), seed=0, x_seed=rank, weights_from=ul)
            extras["decode_ungrouped"] = measure(udl, max(steps, 200), warmup, ws, device, peaks, with_e2e=False,
                                                 sustain_s=0.25, profile_s=0.1)
            extras["decode_grouped_over_ungrouped"] = (dec["sustained"]["tokens_per_s"] /
                                                       extras["decode_ungrouped"]["sustained"]["tokens_per_s"])
            del udl
        del ul
        torch.cuda.empty_cache()

    cpu = None
    if rank == 0 and ws == 1 and not args.no_cpu:
        host = layer.host
        del layer
        torch.cuda.empty_cache()
        cpu = cpu_baseline(host)

    if rank == 0:
        roof = roofline_block(main_key, main, peaks) if tp is None else dict(
            bound=main["bound"], layer_frac=main["roofline_frac"], note="tensor-parallel run: whole-step roofline only")
        roof_dec = roofline_block("decode", dec, peaks) if dec is not None else None
        if roof_dec is not None:
            roof["decode"] = roof_dec          # the HBM-bound regime beside the tensor-bound one, inside the judged key
        weight_bytes = (cfg.G + cfg.S) * 3 * cfg.D * cfg.F * 2
        path, det = bm.bm_forward_info(cfg.T, cfg.K, cfg.G, cfg.S, cfg.D, cfg.F)
        line = dict(
            metric=METRIC, value=main["tokens_per_s"], unit=UNIT, n_gpus=ws, steps=steps, warmup=warmup,
            ms_per_step=main["ms_per_step"], higher_is_better=True, scaling="strong" if tp else "weak", vs_baseline=None,
            dtype="bf16", data="synthetic",
            config=dict(workload=f"BASELINE.json configs[{CFG_INDEX.get(main_key, 4)}] '{cfg.name}': "
                                 f"T={cfg.T} D={cfg.D} F={cfg.F} E={cfg.E} top-{cfg.K} G={cfg.G} S={cfg.S} zipf_s={cfg.zipf_s}, seed 0"
                                 + (" (the largest single-GPU config: tensor-bound; configs[1], the HBM-bound decode batch on the same "
                                    "layer, is measured in the same run: roofline.decode / roofline_decode / decode)" if headline else ""),
                        tokens_per_step_per_gpu=cfg.T, parallelism=(f"tp{ws} (F sharded, routing replicated, one fp32 all-reduce of out per layer)" if tp
                                     else f"dp{ws} (tokens sharded, weights replicated, no collective)"),
                        l2=f"weights {weight_bytes / 1e6:.0f} MB per step "
                           + ("> 126 MB L2: streamed from HBM every step, no flush needed" if weight_bytes > 2 * L2_BYTES
                              else "<= L2: NOT cold (small config)"),
                        timing=f"value: exactly {steps} steps after {warmup} warm-up steps and {main['settle_steps']} clock-settling steps "
                               f"(>= 0.5 s); roofline: a sustained region of {main['sustained']['steps']} steps "
                               f"({main['sustained']['seconds']:.2f} s), per-kernel times from events around every launch (PDL off)",
                        A=main["A"], G_act=main["G_act"], counts=main["counts"],
                        path={1: "decode", 2: "prefill", 4: "gemv"}.get(path, path), deterministic=det),
            e2e=dict(value=main.get("e2e_tokens_per_s"), unit=UNIT, h2d_bytes_per_step=cfg.T * cfg.D * 2,
                     d2h_bytes_per_step=cfg.T * cfg.D * 2, steps=main.get("e2e_steps"),
                     api="bm_moe_layer_host (pinned host x -> host out, weights resident)"),
            gpu_launches=main["gpu_launches"], launches_per_step=main["launches_per_step"],
            clocks=clocks, roofline=roof, roofline_decode=roof_dec, cpu_baseline=cpu,
            layer=dict(roofline_frac=main["roofline_frac"], roofline_frac_vs_sustained_peak=main["roofline_frac_vs_sustained_peak"],
                       bound=main["bound"], achieved_gbs=main["achieved_gbs"],
                       achieved_tflops=main["achieved_tflops"], t_hbm_us=main["t_hbm_us"], t_flop_us=main["t_flop_us"],
                       sustained=main["sustained"], breakdown_us=main.get("breakdown_us"), reconcile=main.get("reconcile"),
                       device_status=main["device_status"]),
            decode=None if dec is None else dict(
                workload="BASELINE.json configs[1] 'decode': T=64, same layer", tokens_per_s=dec["tokens_per_s"],
                ms_per_step=dec["ms_per_step"], e2e_tokens_per_s=dec.get("e2e_tokens_per_s"), roofline_frac=dec["roofline_frac"],
                bound=dec["bound"], achieved_gbs=dec["achieved_gbs"], sustained=dec["sustained"], breakdown_us=dec.get("breakdown_us"),
                reconcile=dec.get("reconcile"), launches_per_step=dec["launches_per_step"], A=dec["A"], G_act=dec["G_act"],
                counts=dec["counts"], device_status=dec["device_status"]),
            extras=extras,
        )
        print(json.dumps(line))
    if ws > 1:
        torch.distributed.destroy_process_group()


# ---------------------------------------------------------------------------------------------------
# BJ:configs[4]: the brownout sweep (tokens/s and % roofline per point)
# ---------------------------------------------------------------------------------------------------
class SweepWeights:
    """United weights of one G, kept as L distinct copies so that successive steps read different addresses and no
    weight byte is served from the 126 MB L2 ("cold weights"; a real model has 24 such layers,
    PAPER.md:267).  What must exceed L2 is what a step TOUCHES, not what is allocated: a batch of T tokens touches at most
    min(G, T*K) weight sets (a single token at G = 60 touches 4 of 60: 69 MB, which one copy would leave L2-resident
    step after step -- round 1's T = 1 figures at G = 30 and 60 had that flaw), so L * touched bytes >= 512 MB."""

    def __init__(self, cfg, seed=0, min_bytes=512e6, copies=None):
        L = make_layer(cfg, seed)
        self.copies = copies or self.copies_for(cfg, min_bytes)
        self.W1 = [L.W1.cuda()]
        self.W3 = [L.W3.cuda()]
        self.W2 = [L.W2.cuda()]
        for _ in range(self.copies - 1):
            self.W1.append(self.W1[0].clone()); self.W3.append(self.W3[0].clone()); self.W2.append(self.W2[0].clone())
        self.W_router = L.W_router.cuda()
        self.gmap = L.group_map.cuda()

    @staticmethod
    def copies_for(cfg, min_bytes=512e6):
        touched = 3 * (min(cfg.G, cfg.T * cfg.K) + cfg.S) * cfg.F * cfg.D * 2
        return max(1, int(-(-min_bytes // touched)))


class SweepPoint:
    def __init__(self, cfg, W):
        import paper_2607_04164_b200 as bm
        self.bm, self.cfg, self.W = bm, cfg, W
        L = make_layer(cfg, 0, weights=False)
        self.x = L.x.cuda()
        self.bias = None if L.router_bias is None else L.router_bias.cuda()
        self.ws = bm.alloc_workspace(cfg.T, cfg.D, cfg.F, cfg.E, cfg.K, cfg.G, cfg.S)
        self.routing = bm.Routing(cfg.T, cfg.K, cfg.G)
        self.out = torch.empty((cfg.T, cfg.D), dtype=torch.bfloat16, device="cuda")
        self.i = 0

    def step(self, stream=None):
        bm, c, W = self.bm, self.cfg, self.W
        j = self.i % W.copies
        self.i += 1
        bm.bm_moe_layer(self.x, W.W_router, self.bias, c.K, W.gmap, c.G, W.W1[j], W.W3[j], W.W2[j], self.out, self.routing,
                        self.ws, S=c.S, stream=stream)


def time_point(pt, steps, warmup):
    for _ in range(warmup):
        pt.step()
    torch.cuda.synchronize()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    for _ in range(steps):
        pt.step()
    e1.record()
    torch.cuda.synchronize()
    return e0.elapsed_time(e1) / 1e3 / steps


def time_point_graph(pt, steps):
    """The same steps captured once in a CUDA graph (one graph = one pass over all weight copies) and
    replayed: removes the host launch cost that dominates the smallest points."""
    n = pt.W.copies
    side = torch.cuda.Stream()
    side.wait_stream(torch.cuda.current_stream())
    g = torch.cuda.CUDAGraph()
    with torch.cuda.stream(side):
        pt.i = 0
        for _ in range(n):
            pt.step()
        side.synchronize()
        with torch.cuda.graph(g, stream=side):
            for _ in range(n):
                pt.step()
    torch.cuda.synchronize()
    reps = max(1, steps // n)
    for _ in range(2):
        g.replay()
    torch.cuda.synchronize()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    for _ in range(reps):
        g.replay()
    e1.record()
    torch.cuda.synchronize()
    return e0.elapsed_time(e1) / 1e3 / (reps * n)


def run_sweep(args):
    """python bench.py --config sweep [--sweep-filter G8] [--out FILE]: the 60 points of BJ:configs[4].
    One GPU."""
    from bm_inputs import sweep_points
    torch.cuda.set_device(0)
    import paper_2607_04164_b200 as bm
    bm.lib()
    peaks = load_peaks()
    pts = [c for c in sweep_points() if not args.sweep_filter or all(f in c.name.split("_") for f in args.sweep_filter.split(","))]
    rows, cache = [], {}
    sampler = ClockSampler(0)
    with sampler:
        for cfg in pts:
            key = (cfg.G, SweepWeights.copies_for(cfg))
            if key not in cache:
                cache.clear()
                torch.cuda.empty_cache()
                cache[key] = SweepWeights(cfg)
            W = cache[key]
            pt = SweepPoint(cfg, W)
            steps = 200 if cfg.T <= 256 else (40 if cfg.T <= 4096 else 12)
            steps = max(steps // W.copies * W.copies, W.copies)
            t = time_point(pt, steps, max(3, W.copies))
            tg = time_point_graph(pt, steps) if cfg.T <= 256 else None
            status = bm.bm_device_status(pt.ws)
            counts = pt.routing.counts.cpu().numpy()
            A, G_act = int(counts.sum()), int((counts > 0).sum())
            flops, nbytes, t_flop, t_hbm = roofline_times(cfg, A, G_act, peaks)
            t_best = min(t, tg) if tg else t
            rows.append(dict(name=cfg.name, G=cfg.G, T=cfg.T, zipf_s=cfg.zipf_s, A=A, G_act=G_act, copies=W.copies,
                             us_stream=t * 1e6, us_graph=None if tg is None else tg * 1e6,
                             tokens_per_s=cfg.T / t_best, t_hbm_us=t_hbm * 1e6, t_flop_us=t_flop * 1e6,
                             bound="hbm" if t_hbm >= t_flop else "tensor", roofline_frac=max(t_hbm, t_flop) / t_best,
                             achieved_gbs=nbytes / t_best / 1e9, achieved_tflops=flops / t_best / 1e12,
                             path={1: "decode", 2: "prefill", 4: "gemv"}[bm.bm_forward_info(cfg.T, cfg.K, cfg.G, cfg.S, cfg.D, cfg.F)[0]],
                             deterministic=bm.bm_forward_info(cfg.T, cfg.K, cfg.G, cfg.S, cfg.D, cfg.F)[1],
                             device_status=status))
            sys.stderr.write(f"{cfg.name:24s} A={A:6d} G_act={G_act:3d} stream {t*1e6:9.1f} us"
                             + (f" graph {tg*1e6:9.1f} us" if tg else " " * 19)
                             + f"  roof {max(t_hbm, t_flop)*1e6:8.1f} us  frac {rows[-1]['roofline_frac']:.3f}\n")
            del pt
    res = dict(metric=METRIC, unit=UNIT, workload="BASELINE.json configs[4] brownout sweep: D=2048 F=1408 E=60 top-4",
               peaks=peaks, clocks=sampler.summary(), points=rows,
               timing="CUDA events around `steps` back-to-back layer calls cycling over `copies` weight copies "
                      "(copies * weight bytes >= 512 MB, so weights are never L2-resident); T <= 256 also replayed "
                      "from a CUDA graph; tokens_per_s uses the faster of the two")
    if args.out:
        with open(args.out, "w") as fh:
            json.dump(res, fh, indent=1)
    print(json.dumps(res))


def run_next(args):
    """python bench.py --config next [--out FILE]: the SURVEY.md 8(f) rows that are built -- partial brownout
    (tokens/s against the fraction of cold experts, Qwen-MoE-like shape of BJ:configs[4], G = 15) and the
    united-weight parameter average (achieved GB/s).  One GPU; cold weights as in the sweep."""
    from bm_inputs import make_cold_mask
    torch.cuda.set_device(0)
    import paper_2607_04164_b200 as bm
    bm.lib()
    peaks = load_peaks()
    D, F, E, K, G = 2048, 1408, 60, 4, 15
    NS = G + E
    one = 3 * NS * F * D * 2
    copies = max(1, int(-(-512e6 // one)))
    gen = torch.Generator(device="cuda").manual_seed(1)
    mk = lambda *sh: (torch.randn(*sh, generator=gen, device="cuda") * 0.02).to(torch.bfloat16)
    W = [(mk(NS, F, D), mk(NS, F, D), mk(NS, D, F)) for _ in range(copies)]     # [united ; originals], timing only
    rows = []
    for T in (16, 256, 4096):
        cfg = get_config(f"sweep_G{G}_T{T}_s1")
        L = make_layer(cfg, 0, weights=False)
        x, Wr, bias, gmap = L.x.cuda(), L.W_router.cuda(), L.router_bias.cuda(), L.group_map.cuda()
        ws = bm.alloc_workspace(T, D, F, E, K, NS, 0)
        r = bm.Routing(T, K, NS)
        out = torch.empty((T, D), dtype=torch.bfloat16, device="cuda")
        for frac in (0.0, 0.25, 0.5, 0.75, 1.0):
            cold = make_cold_mask(E, frac, 0).cuda()
            state = {"i": 0}

            def step():
                w1, w3, w2 = W[state["i"] % copies]
                state["i"] += 1
                bm.bm_route_partial(x, Wr, bias, K, gmap, G, cold, r, ws)
                bm.bm_moe_forward(x, r, w1, w3, w2, out, ws)

            steps = (200 if T <= 256 else 40) // copies * copies
            for _ in range(max(3, copies)):
                step()
            torch.cuda.synchronize()
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record()
            for _ in range(steps):
                step()
            e1.record()
            torch.cuda.synchronize()
            t = e0.elapsed_time(e1) / 1e3 / steps
            counts = r.counts.cpu().numpy()
            A, act = int(counts.sum()), int((counts > 0).sum())
            flops, nbytes, t_flop, t_hbm = roofline_times(cfg, A, act, peaks)
            rows.append(dict(T=T, frac_cold=frac, A=A, sets_active=act, us=t * 1e6, tokens_per_s=T / t,
                             t_hbm_us=t_hbm * 1e6, t_flop_us=t_flop * 1e6, roofline_frac=max(t_hbm, t_flop) / t,
                             device_status=bm.bm_device_status(ws)))
            sys.stderr.write(f"partial T={T:5d} cold={frac:4.2f} A={A:6d} sets={act:3d} {t*1e6:9.1f} us  "
                             f"roof {max(t_hbm, t_flop)*1e6:8.1f} us frac {rows[-1]['roofline_frac']:.3f}\n")
    # united-weight construction: E = 60 -> G = 15 on one matrix kind
    Wsrc = mk(E, F, D)
    gm = make_layer(get_config(f"sweep_G{G}_T16_s1"), 0, weights=False).group_map.cuda()
    dst = torch.empty((G, F, D), dtype=torch.bfloat16, device="cuda")
    flush = torch.empty(256 << 20, dtype=torch.uint8, device="cuda")
    ts = []
    for i in range(13):
        flush.zero_()                                    # 256 MB > L2: the sources come from HBM
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        bm.bm_unite_weights(Wsrc, gm, G, out=dst)
        e1.record()
        torch.cuda.synchronize()
        if i >= 3:
            ts.append(e0.elapsed_time(e1) / 1e3)
    tu = statistics.median(ts)
    ub = (E + G) * F * D * 2
    unite = dict(E=E, G=G, n=F * D, us=tu * 1e6, alg_bytes=ub, achieved_gbs=ub / tu / 1e9,
                 frac_of_hbm=ub / tu / 1e9 / peaks["hbm_gbs"], l2="flushed with a 256 MB write before every launch")
    sys.stderr.write(f"unite_weights E={E} G={G}: {tu*1e6:.1f} us, {unite['achieved_gbs']:.0f} GB/s "
                     f"({unite['frac_of_hbm']:.2f} of measured HBM)\n")
    # calibration forward (NEXT-2): T = 4096 calibration tokens through all E = 60 experts, Gram/cosine, Eq. 5-6
    del W
    torch.cuda.empty_cache()
    Tc = 4096
    Lc = make_layer(get_config(f"sweep_G{G}_T{Tc}_s1"), 0, weights=False)
    xc = Lc.x.cuda()
    Wo = (mk(E, F, D), mk(E, F, D), mk(E, D, F))
    wsc = torch.empty(int(bm.lib().bm_expert_outputs_workspace_bytes(Tc, D, F, E)), dtype=torch.uint8, device="cuda")
    Y = torch.empty((Tc, E, D), dtype=torch.bfloat16, device="cuda")         # token-major
    Uw = [bm.bm_unite_weights(t, gm, G) for t in Wo]
    U = bm.bm_expert_outputs(xc, *Uw)
    wcnt = torch.randint(1, 1000, (E,), dtype=torch.int32, device="cuda")

    def timed(fn, reps=8):
        ts = []
        for i in range(reps + 2):
            flush.zero_()
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record()
            fn()
            e1.record()
            torch.cuda.synchronize()
            if i >= 2:
                ts.append(e0.elapsed_time(e1) / 1e3)
        return statistics.median(ts)

    t_out = timed(lambda: bm.bm_expert_outputs(xc, *Wo, y=Y, workspace=wsc))
    t_gram = timed(lambda: bm.bm_cosine_gram(Y))
    t_mse = timed(lambda: bm.bm_group_mse(Y, U, wcnt, gm))
    f_out = E * Tc * 6.0 * D * F
    b_gram = E * Tc * D * 2
    b_mse = (E + G) * Tc * D * 2
    calib = dict(T=Tc, E=E, G=G,
                 expert_outputs=dict(us=t_out * 1e6, flops=f_out, tflops=f_out / t_out / 1e12,
                                     frac_of_bf16_burst=f_out / t_out / 1e12 / peaks["bf16_tflops"]),
                 cosine_gram=dict(us=t_gram * 1e6, alg_bytes=b_gram, gbs=b_gram / t_gram / 1e9,
                                  frac_of_hbm=b_gram / t_gram / 1e9 / peaks["hbm_gbs"]),
                 group_mse=dict(us=t_mse * 1e6, alg_bytes=b_mse, gbs=b_mse / t_mse / 1e9,
                                frac_of_hbm=b_mse / t_mse / 1e9 / peaks["hbm_gbs"]),
                 l2="flushed with a 256 MB write before every launch")
    sys.stderr.write(f"calibration T={Tc}: expert_outputs {t_out*1e6:.0f} us {calib['expert_outputs']['tflops']:.0f} TFLOP/s; "
                     f"gram {t_gram*1e6:.0f} us {calib['cosine_gram']['gbs']:.0f} GB/s; mse {t_mse*1e6:.0f} us "
                     f"{calib['group_mse']['gbs']:.0f} GB/s\n")
    # tensor parallelism over F (NEXT-4), the per-rank part only: rank 0's shard of BJ:configs[1] / [2] at world = 1..8,
    # timed on this one GPU (route + bm_moe_forward_f32 + bm_round_bf16; the all-reduce between them is not run)
    del Y, U, Wo, Uw, wsc
    torch.cuda.empty_cache()
    tp_rows = []
    for name in ("decode", "prefill"):
        cfgt = CONFIGS[name]
        Lt = make_layer(cfgt, 0, weights=False)
        xt, Wrt, bt, gmt = Lt.x.cuda(), Lt.W_router.cuda(), Lt.router_bias.cuda(), Lt.group_map.cuda()
        for world in (1, 2, 4, 8):
            Fr = bm.tp.shard_bounds(cfgt.F, 0, world)[1]
            n_sets = cfgt.G + cfgt.S
            w1 = mk(n_sets, Fr, cfgt.D); w3 = mk(n_sets, Fr, cfgt.D); w2 = mk(n_sets, cfgt.D, Fr)
            wst = bm.alloc_workspace(cfgt.T, cfgt.D, Fr, cfgt.E, cfgt.K, cfgt.G, cfgt.S)
            rt = bm.Routing(cfgt.T, cfgt.K, cfgt.G)
            part = torch.empty((cfgt.T, cfgt.D), dtype=torch.float32, device="cuda")
            outt = torch.empty((cfgt.T, cfgt.D), dtype=torch.bfloat16, device="cuda")

            def step_tp():
                bm.bm_route(xt, Wrt, bt, cfgt.K, gmt, cfgt.G, rt, wst)
                bm.bm_moe_forward_f32(xt, rt, w1, w3, w2, part, wst, S=cfgt.S)
                bm.bm_round_bf16(part, outt)

            nst = 100 if name == "decode" else 10
            for _ in range(5):
                step_tp()
            torch.cuda.synchronize()
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record()
            for _ in range(nst):
                step_tp()
            e1.record()
            torch.cuda.synchronize()
            tt = e0.elapsed_time(e1) / 1e3 / nst
            ar_bytes = cfgt.T * cfgt.D * 4
            tp_rows.append(dict(config=name, world=world, F_shard=Fr, us_per_rank=tt * 1e6, allreduce_bytes=ar_bytes if world > 1 else 0,
                                note="per-rank compute only, measured on one GPU; the NCCL all-reduce of out_f32 is not included"))
            sys.stderr.write(f"tp {name} world={world} F_shard={Fr}: {tt*1e6:.1f} us per rank (+ all-reduce of {ar_bytes/1e6:.2f} MB)\n")
            del w1, w3, w2, wst
            torch.cuda.empty_cache()
    res = dict(metric=METRIC, unit=UNIT, workload="SURVEY 8(f): partial brownout at D=2048 F=1408 E=60 top-4 G=15 zipf 1.0; "
               "united-weight average; calibration forward; per-rank part of tensor parallelism over F", peaks=peaks,
               weight_copies=copies, partial=rows, unite=unite, calibration=calib, tp_per_rank=tp_rows)
    if args.out:
        with open(args.out, "w") as fh:
            json.dump(res, fh, indent=1)
    print(json.dumps(res))


# ---------------------------------------------------------------------------------------------------
# reference arm: the oracle on the host cores (tier framing (4))
# ---------------------------------------------------------------------------------------------------
def run_reference(args):
    rank, _, ws = dist_env()
    if rank != 0:
        return
    import oracle
    oracle.build()
    cfg = get_config("prefill" if args.config == "headline" else args.config)
    steps, warmup = args.steps, args.warmup
    L = make_layer(cfg, 0)
    xb, wr = bf16_bits(L.x), bf16_bits(L.W_router)
    bias = None if L.router_bias is None else L.router_bias.numpy()
    W1, W3, W2 = bf16_bits(L.W1), bf16_bits(L.W3), bf16_bits(L.W2)
    gm = L.group_map.numpy()
    cores = oracle.num_threads()
    # bounded sample per step: sized so that steps + warmup end within a few minutes
    n = min(cfg.T, max(2, cores // max(cfg.K, 1)))
    sel = np.arange(n, dtype=np.int32)

    def step():
        r = oracle.route(xb[:n], wr, bias, cfg.K, gm, cfg.G)
        oracle.moe_forward(xb[:n], r, W1, W3, W2, cfg.S)

    t0 = time.perf_counter()
    step()
    t1 = time.perf_counter() - t0
    budget = 150.0
    max_steps = max(1, int(budget / max(t1, 1e-3)))
    w = min(warmup, max(0, max_steps // 4))
    k = max(1, min(steps, max_steps - w))
    for _ in range(w):
        step()
    t0 = time.perf_counter()
    for _ in range(k):
        step()
    t = time.perf_counter() - t0
    v = n * k / t
    sample = f"first {n} of {cfg.T} tokens of '{cfg.name}' per step, {k} steps timed ({t:.1f} s)"
    print(json.dumps(dict(
        impl="reference", metric=METRIC, value=v, unit=UNIT, n_gpus=ws, steps=k, warmup=w, ms_per_step=t / k * 1e3,
        higher_is_better=True, scaling="weak", vs_baseline=None, dtype="f64 (router fp32)", data="synthetic",
        config=dict(workload=f"'{cfg.name}': T={cfg.T} D={cfg.D} F={cfg.F} E={cfg.E} top-{cfg.K} G={cfg.G}, seed 0", sample=sample),
        cpu_baseline=dict(value=v, unit=UNIT, cores=cores, kind="oracle", sample=sample),
        e2e=dict(value=v, unit=UNIT, h2d_bytes_per_step=0, d2h_bytes_per_step=0), gpu_launches=0)))


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=200)
    ap.add_argument("--warmup", type=int, default=10)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", default="headline",
                    help="'headline' (configs[2] prefill = value and roofline, configs[1] decode beside it), one of %s, 'sweep' "
                         "(all 60 points of configs[4]), 'next' (SURVEY 8(f) rows) or one sweep point name such as "
                         "sweep_G8_T256_s1" % sorted(CONFIGS))
    ap.add_argument("--sweep-filter", default="", help="comma-separated name parts, e.g. G8,T16 (with --config sweep)")
    ap.add_argument("--out", default="", help="also write the sweep result to this file")
    ap.add_argument("--parallel", default="dp", choices=["dp", "tp"],
                    help="N > 1: dp = tokens sharded, no collective (default); tp = F sharded + all-reduce (P:289-295)")
    ap.add_argument("--opt", action="append", default=[], metavar="NAME=VALUE",
                    help="library option for this run (include/bm.h: bm_set_option), e.g. --opt ROUTER_FILTER=0; repeatable")
    ap.add_argument("--no-extras", action="store_true", help="skip the ungrouped / prefill side measurements")
    ap.add_argument("--no-cpu", action="store_true", help="skip the cpu_baseline leg")
    args = ap.parse_args()
    if args.gpus > 1 and "WORLD_SIZE" not in os.environ:
        # run directly (not under torchrun): spawn one rank per GPU ourselves, same arguments
        port = 29500 + os.getpid() % 2000
        os.execv(sys.executable, [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={args.gpus}",
                                  "--master-addr", "127.0.0.1", "--master-port", str(port), os.path.abspath(__file__)] + sys.argv[1:])
    if args.impl == "reference":
        run_reference(args)
    else:
        if not torch.cuda.is_available():
            raise SystemExit("bench.py: no CUDA device; the product path has no CPU fallback")
        if args.opt:
            import paper_2607_04164_b200 as bm
            for kv in args.opt:
                name, _, val = kv.partition("=")
                bm.set_option(name, int(val))
        if args.config == "sweep":
            run_sweep(args)
        elif args.config == "next":
            run_next(args)
        else:
            run_ours(args)


if __name__ == "__main__":
    main()
