#!/usr/bin/env python
"""bench.py -- one D2SD verification step (select -> build -> 36x cascade attention -> accept).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config 2] [--impl d2sd|reference]

Prints ONE JSON line (rank 0).  A "step" is one pass of the whole hot path over one batch of
synthetic input shaped like BASELINE.json config 2 (Qwen3-8B verification step, L=4096, gamma=16,
K=4, 36 layers with distinct KV, vocab 151936).  `value` = tree tokens verified per second with all
inputs resident in HBM (CUDA-graph replay of the step, CUDA events, max over ranks); `e2e` = the
same through the C-ABI binding with HOST (pinned) buffers and the copies inside the timed region;
`roofline` = the dominant kernel (the cascade attention launch) against the measured peaks; `cpu_baseline` = the CPU
oracle timed on this box's host cores on a bounded sample.  N>1: independent replicas, one per
rank, no data-path collective ("replicas only").
"""
from __future__ import annotations

import argparse
import json
import math
import os
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import d2sd_synth as synth  # noqa: E402

METRIC = "tree_tokens_per_s (cascade tree-verify step: select+build+36x attention+accept)"
UNIT = "tokens/s"
L2_BYTES = 126 * 1024 * 1024


# ------------------------------------------------------------------------------- multi-rank helpers

def shard_range(n_units: int, rank: int, world: int):
    """Contiguous, balanced partition of n_units independent units (requests) over ranks."""
    base, rem = divmod(n_units, world)
    lo = rank * base + min(rank, rem)
    return lo, lo + base + (1 if rank < rem else 0)


def _reduce(x: float, op) -> float:
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return float(x)
    dev = "cuda" if dist.get_backend() == "nccl" else "cpu"
    t = torch.tensor([x], dtype=torch.float64, device=dev)
    dist.all_reduce(t, op=op)
    return float(t.item())


def max_over_ranks(x: float) -> float:
    import torch.distributed as dist
    return _reduce(x, dist.ReduceOp.MAX)


def sum_over_ranks(x: float) -> float:
    import torch.distributed as dist
    return _reduce(x, dist.ReduceOp.SUM)


def _barrier():
    import torch
    import torch.distributed as dist
    if dist.is_available() and dist.is_initialized() and dist.get_world_size() > 1:
        dist.barrier()
    torch.cuda.synchronize()


# ------------------------------------------------------------------------------- clocks

class ClockSampler:
    """Samples SM clock and throttle reasons DURING the timed region (NVML, 10 ms period)."""

    REASONS = {0x8: "hw_slowdown", 0x40: "hw_thermal_slowdown", 0x20: "sw_thermal_slowdown",
               0x4: "sw_power_cap", 0x80: "hw_power_brake_slowdown"}

    def __init__(self, device_index: int):
        self.samples, self.reasons, self.max_mhz = [], set(), None
        self._stop = threading.Event()
        self._thread = None
        try:
            import pynvml
            pynvml.nvmlInit()
            self.nv = pynvml
            vis = os.environ.get("CUDA_VISIBLE_DEVICES")
            idx = device_index
            if vis:
                try:
                    idx = int(vis.split(",")[device_index])
                except ValueError:
                    idx = device_index
            self.h = pynvml.nvmlDeviceGetHandleByIndex(idx)
            self.max_mhz = int(pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM))
        except Exception:
            self.nv = None

    def _poll(self):
        while not self._stop.is_set():
            self.sample()
            time.sleep(0.01)

    def sample(self):
        if self.nv is None:
            return
        try:
            self.samples.append(int(self.nv.nvmlDeviceGetClockInfo(self.h, self.nv.NVML_CLOCK_SM)))
            r = int(self.nv.nvmlDeviceGetCurrentClocksEventReasons(self.h))
            for bit, name in self.REASONS.items():
                if r & bit:
                    self.reasons.add(name)
        except Exception:
            pass

    def start(self):
        if self.nv is not None:
            self._stop.clear()
            self._thread = threading.Thread(target=self._poll, daemon=True)
            self._thread.start()

    def stop(self):
        if self._thread is not None:
            self.sample()
            self._stop.set()
            self._thread.join()
            self._thread = None

    def summary(self):
        if not self.samples:
            return {"sm_mhz": None, "sm_max_mhz": self.max_mhz, "reasons": sorted(self.reasons), "samples": 0}
        return {"sm_mhz": float(np.median(self.samples)), "sm_max_mhz": self.max_mhz,
                "reasons": sorted(self.reasons), "samples": len(self.samples)}


# ------------------------------------------------------------------------------- peaks

def measured_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        d = json.load(open(p))
        return {"hbm_gbs": float(d["hbm_gbs"]), "bf16_tflops": float(d["bf16_tflops"]),
                "bf16_tflops_sustained": float(d.get("bf16_tflops_sustained", d["bf16_tflops"])),
                "source": "measured"}
    # fallback stated in the B200 profiling recipe
    return {"hbm_gbs": 6650.0, "bf16_tflops": 1590.0, "bf16_tflops_sustained": 1400.0, "source": "fallback"}


def ncu_traffic(kernel: str, cfg_no: int):
    """DRAM bytes per launch of the dominant kernel from the committed ncu --set full capture
    (profiles/traffic.csv: kernel,config,dram_bytes_read,dram_bytes_write), or None."""
    p = os.path.join(ROOT, "profiles", "traffic.csv")
    if not os.path.exists(p):
        return None
    for line in open(p):
        f = [x.strip() for x in line.split(",")]
        if len(f) >= 4 and f[0] == kernel and f[1] == str(cfg_no):
            return float(f[2]) + float(f[3])
    return None


# ------------------------------------------------------------------------------- workload (GPU arm)

class Workload:
    """All tensors of one verification step, resident in HBM, plus pinned host copies for e2e."""

    def __init__(self, cfg: synth.Config, d2sd, torch, host_copies: bool = True):
        self.cfg, self.d2sd, self.torch = cfg, d2sd, torch
        dev = "cuda"
        st = synth.make_step_inputs(cfg)
        self.st = st
        self.max_ctx = int(st["ctx_len"].max())

        def bf(bits):
            return torch.from_numpy(np.ascontiguousarray(bits).view(np.int16)).view(torch.bfloat16)

        def dev_of(host):
            return {k: v.to(dev, non_blocking=True) for k, v in host.items()}

        # host (pinned) originals
        self.h_step = {"conf": torch.from_numpy(st["conf"]), "draft1": torch.from_numpy(st["draft1"]),
                       "draft2": torch.from_numpy(st["draft2"]), "ctx_len": torch.from_numpy(st["ctx_len"])}
        self.h_layers = []
        self.page_size = 0
        for layer in range(cfg.layers):
            ti = synth.make_tree_inputs(cfg, layer)
            kv = synth.make_kv_cache(cfg, st["ctx_len"], layer)
            self.page_size = kv["page_size"]
            h = {"q": bf(ti["q"]), "tree_k": bf(ti["tree_k"]), "tree_v": bf(ti["tree_v"]),
                 "k_cache": bf(kv["k_cache"]), "v_cache": bf(kv["v_cache"])}
            if layer == 0:
                self.h_kvmeta = {"kv_indptr": torch.from_numpy(kv["kv_indptr"])}
                if kv["kv_indices"] is not None:
                    self.h_kvmeta["kv_indices"] = torch.from_numpy(kv["kv_indices"])
            self.h_layers.append(h)
        # The step's own per-layer inputs (Q, tree K, tree V of every layer) live in ONE packed buffer on each side, so
        # the end-to-end path moves them with one copy per layer slice instead of three; the per-layer tensors the calls
        # take are views into it.  The committed KV caches stay separate tensors (they are state, not step input).
        names = ("q", "tree_k", "tree_v")
        sizes = [self.h_layers[0][n].numel() for n in names]
        self.pack_stride = sum(sizes)
        h_pack = torch.empty((cfg.layers, self.pack_stride), dtype=torch.bfloat16)
        for l, h in enumerate(self.h_layers):
            off = 0
            for n, sz in zip(names, sizes):
                h_pack[l, off:off + sz] = h[n].reshape(-1)
                off += sz
        if host_copies:
            self.h_step = {k: v.pin_memory() for k, v in self.h_step.items()}
            h_pack = h_pack.pin_memory()
            for h in self.h_layers:
                for n in ("k_cache", "v_cache"):
                    h[n] = h[n].pin_memory()
        self.h_pack = h_pack
        self.step_in = dev_of(self.h_step)
        self.kvmeta = dev_of(self.h_kvmeta)
        self.pack = h_pack.to(dev)
        self.layers = []
        for l, h in enumerate(self.h_layers):
            d_l, off = {}, 0
            for n, sz in zip(names, sizes):
                d_l[n] = self.pack[l, off:off + sz].view(h[n].shape)
                off += sz
                del h[n]  # the packed host buffer holds it
            d_l["k_cache"] = h["k_cache"].to(dev, non_blocking=True)
            d_l["v_cache"] = h["v_cache"].to(dev, non_blocking=True)
            self.layers.append(d_l)
        self.e2e_graphs = {}
        torch.cuda.synchronize()

        B, T, Hq, Hkv, d = cfg.B, cfg.T_cap, cfg.Hq, cfg.Hkv, cfg.d
        kv_rows = self.layers[0]["k_cache"].shape[0] * (cfg.page_size if cfg.paged else 1)
        self.attn_impl = int(os.environ.get("D2SD_BENCH_ATTN_IMPL", "0"))  # kernel A/B runs only (d2sd.h: test knob)
        self.attn_splits = int(os.environ.get("D2SD_BENCH_ATTN_SPLITS", "0"))  # chunk-count sweeps only (d2sd.h: test knob)
        self.ws_attn = d2sd.cascade_workspace(B, T, Hq, Hkv, d, self.max_ctx, device=dev,
                                              page_size=self.page_size, kv_rows=kv_rows, impl=self.attn_impl,
                                              num_splits=self.attn_splits)
        self.ws_acc = torch.empty(d2sd.accept_workspace_bytes(B, T, cfg.V), dtype=torch.uint8, device=dev)
        self.prefix_len = torch.empty((B, cfg.K), dtype=torch.int32, device=dev)
        self.tree = None
        self.outs = [torch.zeros((B, T, Hq, d), dtype=torch.bfloat16, device=dev) for _ in range(cfg.layers)]
        self.lse = torch.empty((B, T, Hq), dtype=torch.float32, device=dev)
        self.acc = None

        # Logits: planted on the tree the CUDA path itself builds (a real target model consumes the
        # tree and emits the logits; no oracle on the product path).
        self.select_build()
        torch.cuda.synchronize()
        tree_h = {k: v.cpu().numpy() for k, v in self.tree.items()}
        logits = synth.make_logits(cfg)
        self.n_plants = synth.plant_acceptance(cfg, logits, st["conf"], tree_h["tokens"], tree_h["parent"],
                                               tree_h["depth"], tree_h["tree_len"])
        self.h_logits = bf(logits).pin_memory() if host_copies else bf(logits)
        self.logits = self.h_logits.to(dev)
        self.tree_len_host = tree_h["tree_len"].copy()
        self.tree_tokens = int(tree_h["tree_len"].sum())
        torch.cuda.synchronize()

    # --- the hot path ---------------------------------------------------------------------------
    def select_build(self):
        d, s, c = self.d2sd, self.step_in, self.cfg
        d.select_prefixes(s["conf"], c.K, prefix_len=self.prefix_len)
        self.tree = d.build_tree(s["draft1"], s["draft2"], self.prefix_len, s["ctx_len"], c.T_cap, out=self.tree)

    def attention(self, layer: int, phases: int = 0):
        L, t = self.layers[layer], self.tree
        self.d2sd.cascade_verify_attn(L["q"], L["k_cache"], L["v_cache"], self.kvmeta.get("kv_indptr"),
                                      self.kvmeta.get("kv_indices"), self.step_in["ctx_len"], L["tree_k"],
                                      L["tree_v"], t["mask"], t["tree_len"], self.max_ctx,
                                      page_size=self.page_size, phases=phases, out=self.outs[layer],
                                      lse=self.lse, workspace=self.ws_attn, impl=self.attn_impl,
                                      num_splits=self.attn_splits)

    def accept(self):
        t = self.tree
        self.acc = self.d2sd.accept(self.logits, t["tokens"], t["parent"], t["depth"], t["tree_len"],
                                    self.cfg.gamma, out=self.acc, workspace=self.ws_acc)

    def step(self):
        self.select_build()
        for layer in range(self.cfg.layers):
            self.attention(layer)
        self.accept()

    @property
    def attn_kernel(self) -> str:
        return self.attn_kernel_for(self.cfg)

    @staticmethod
    def attn_kernel_for(cfg) -> str:
        # api.cu: paged KV with more (request, kv head) pairs than one wave holds runs the two-tiles-per-CTA kernel
        return "attn_duo_kernel" if cfg.paged and cfg.B * cfg.Hkv * 4 > 148 else "attn_stream_kernel"

    @property
    def launches_per_step(self) -> int:
        # select, build, per layer: one fused tcgen05 launch (contiguous KV) or mma.sync pass + merge
        # (paged KV), argmax, walk
        return 2 + self.cfg.layers + 2

    # --- e2e: host buffers in, host results out ---------------------------------------------------
    def h2d_bytes(self, with_kv: bool) -> int:
        n = sum(v.numel() * v.element_size() for v in self.h_step.values()) + self.h_logits.numel() * 2
        n += self.h_pack.numel() * 2
        if with_kv:
            for h in self.h_layers:
                n += h["k_cache"].numel() * 2 + h["v_cache"].numel() * 2
        return n

    def _e2e_enqueue(self, with_kv: bool, k_stream, c_stream):
        """Host buffers -> device -> step -> host results.  Copies run on a second stream, one event per layer, so
        layer l's attention waits only for layer l's inputs and the transfers overlap the kernels."""
        torch = self.torch
        c_stream.wait_stream(k_stream)
        evs = []
        with torch.cuda.stream(c_stream):
            for k, v in self.h_step.items():
                self.step_in[k].copy_(v, non_blocking=True)
            e0 = torch.cuda.Event()
            e0.record(c_stream)
            for l, h in enumerate(self.h_layers):
                self.pack[l].copy_(self.h_pack[l], non_blocking=True)
                if with_kv:
                    self.layers[l]["k_cache"].copy_(h["k_cache"], non_blocking=True)
                    self.layers[l]["v_cache"].copy_(h["v_cache"], non_blocking=True)
                e = torch.cuda.Event()
                e.record(c_stream)
                evs.append(e)
            self.logits.copy_(self.h_logits, non_blocking=True)
            e_log = torch.cuda.Event()
            e_log.record(c_stream)
        k_stream.wait_event(e0)
        self.select_build()
        for l in range(self.cfg.layers):
            k_stream.wait_event(evs[l])
            self.attention(l)
        k_stream.wait_event(e_log)
        self.accept()
        for k, v in self.acc.items():
            self.h_res[k].copy_(v, non_blocking=True)
        self.h_res["out_last"].copy_(self.outs[-1], non_blocking=True)
        k_stream.wait_stream(c_stream)

    def e2e_step(self, with_kv: bool):
        """One end-to-end step through the public API, replayed from a CUDA graph that holds the copies (pinned host
        memory in, pinned host memory out) and the calls (the paper runs its verify pass from pre-warmed CUDA
        graphs)."""
        torch = self.torch
        if with_kv not in self.e2e_graphs:
            if not hasattr(self, "h_res"):
                self.accept()
                self.h_res = {k: torch.empty_like(v, device="cpu").pin_memory() for k, v in self.acc.items()}
                self.h_res["out_last"] = torch.empty_like(self.outs[-1], device="cpu").pin_memory()
            ks, cs = torch.cuda.Stream(), torch.cuda.Stream()
            ks.wait_stream(torch.cuda.current_stream())
            with torch.cuda.stream(ks):
                self._e2e_enqueue(with_kv, ks, cs)  # warm, outside capture
            torch.cuda.synchronize()
            g = torch.cuda.CUDAGraph()
            with torch.cuda.graph(g, stream=ks):
                self._e2e_enqueue(with_kv, ks, cs)
            torch.cuda.synchronize()
            self.e2e_graphs[with_kv] = g
        self.e2e_graphs[with_kv].replay()
        return self.h_res

    def d2h_bytes(self) -> int:
        n = sum(v.numel() * v.element_size() for v in self.acc.values())
        return n + self.outs[-1].numel() * 2


def workload_config(cfg, ctx_len, tree_tokens: int, planted: int, world: int) -> dict:
    """The workload description both arms print (same keys, same values for the same config)."""
    return {"workload": f"BASELINE.json configs[{cfg.number - 1}] ({cfg.name})", "B": cfg.B, "layers": cfg.layers,
            "gamma": cfg.gamma, "K": cfg.K, "ctx": [int(x) for x in ctx_len[:4]], "V": cfg.V,
            "tree_tokens": int(tree_tokens), "planted_accepts": int(planted),
            "kv": "paged(16)" if cfg.paged else "contiguous", "parallelism": f"replicas x{world}"}


def capture(torch, fn):
    s = torch.cuda.Stream()
    s.wait_stream(torch.cuda.current_stream())
    with torch.cuda.stream(s):
        fn()  # warm (lazy module load, attribute opt-ins) outside capture
        torch.cuda.synchronize()
        g = torch.cuda.CUDAGraph()
        with torch.cuda.graph(g, stream=s):
            fn()
    torch.cuda.current_stream().wait_stream(s)
    torch.cuda.synchronize()
    return g


def time_replays(torch, g, n: int, flush=None) -> float:
    """Milliseconds for n replays of graph g on the current stream (CUDA events).  With `flush`
    (a callable writing a buffer larger than L2) each replay is timed on its own, flush excluded."""
    if flush is None:
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        for _ in range(n):
            g.replay()
        e1.record()
        torch.cuda.synchronize()
        return e0.elapsed_time(e1)
    pairs = []
    for _ in range(n):
        flush()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        g.replay()
        e1.record()
        pairs.append((e0, e1))
    torch.cuda.synchronize()
    return sum(a.elapsed_time(b) for a, b in pairs)



# ------------------------------------------------------------------------------- roofline + extra measurements

NOMINAL_HBM_GBS = 8000.0  # the north star's "roughly 8 TB/s" (stretch basis)


def attn_roofline(cfg, wl, us_per_launch: float, peaks, traffic):
    """Algorithmic bytes / flops of ONE cascade-attention launch against the measured peaks."""
    T_rows = wl.tree_tokens
    kv_bytes = 2 * int(wl.st["ctx_len"].sum()) * cfg.Hkv * cfg.d * 2
    q_bytes = T_rows * cfg.Hq * cfg.d * 2                     # Q in; O out is the same size
    tree_kv_bytes = 2 * T_rows * cfg.Hkv * cfg.d * 2
    alg_bytes = kv_bytes + 2 * q_bytes + tree_kv_bytes + T_rows * cfg.Hq * 4
    alg_flops = 4.0 * cfg.Hq * cfg.d * float(sum(int(t) * int(l) for t, l in zip(wl.tree_len_host, wl.st["ctx_len"])))
    ach_gbs = alg_bytes / (us_per_launch * 1e-6) / 1e9
    ach_tf = alg_flops / (us_per_launch * 1e-6) / 1e12
    t_hbm_us = alg_bytes / (peaks["hbm_gbs"] * 1e9) * 1e6
    t_tc_us = alg_flops / (peaks["bf16_tflops_sustained"] * 1e12) * 1e6
    hbm = {"bound": "hbm", "achieved": ach_gbs, "peak": peaks["hbm_gbs"], "unit": "GB/s",
           "frac": ach_gbs / peaks["hbm_gbs"], "frac_of_nominal_8TBs": ach_gbs / NOMINAL_HBM_GBS, "traffic": traffic,
           "peak_source": peaks["source"], "kernel": wl.attn_kernel, "us_per_launch": us_per_launch,
           "alg_bytes_per_launch": alg_bytes}
    tc = {"bound": "tensor", "achieved": ach_tf, "peak": peaks["bf16_tflops_sustained"], "unit": "TFLOP/s",
          "frac": ach_tf / peaks["bf16_tflops_sustained"], "traffic": traffic,
          "peak_source": peaks["source"] + " (sustained bf16)", "kernel": wl.attn_kernel,
          "us_per_launch": us_per_launch, "alg_flops_per_launch": alg_flops}
    return (tc if t_tc_us > t_hbm_us else hbm), hbm, tc  # "the slower of" the two bounds first


def attention_only(torch, d2sd, cfg, peaks, steps: int, layers: int):
    """Attention launches of one config alone (graph replay, CUDA events): us per launch + rooflines."""
    import dataclasses
    sub = dataclasses.replace(cfg, layers=min(cfg.layers, layers))
    wl = Workload(sub, d2sd, torch, host_copies=False)
    kv_bytes = 2 * int(wl.st["ctx_len"].sum()) * sub.Hkv * sub.d * 2 * sub.layers
    flush = None
    if kv_bytes < 2 * L2_BYTES:
        fbuf = torch.empty(2 * L2_BYTES, dtype=torch.uint8, device="cuda")
        flush = lambda: fbuf.fill_(1)  # noqa: E731
    g = capture(torch, lambda: [wl.attention(i) for i in range(sub.layers)])
    for _ in range(3):
        g.replay()
    torch.cuda.synchronize()
    us = time_replays(torch, g, steps, flush) / (steps * sub.layers) * 1e3
    roof, hbm, tc = attn_roofline(sub, wl, us, peaks, ncu_traffic(wl.attn_kernel_for(sub), sub.number))
    out = {"workload": f"BASELINE.json configs[{cfg.number - 1}] ({cfg.name})", "attn_us_per_layer": us,
           "layers_timed": sub.layers, "tree_tokens": wl.tree_tokens, "kernel": wl.attn_kernel_for(sub),
           "l2": "flushed between replays" if flush else "distinct KV per layer, larger than L2",
           "roofline_bound": roof["bound"], "roofline_frac": roof["frac"],
           "roofline_hbm": {k: hbm[k] for k in ("achieved", "frac", "frac_of_nominal_8TBs", "traffic", "alg_bytes_per_launch")},
           "roofline_tensor": {k: tc[k] for k in ("achieved", "frac", "alg_flops_per_launch")}}
    del wl, g
    torch.cuda.empty_cache()
    return out


# prefix sets that give T = gamma + sum(gamma-1-i) tree nodes at gamma = 16, K = 4 (intensity is 4T
# flop per KV byte, so the bound moves from HBM to the tensor pipe inside this range)
T_SWEEP = {26: (11, 12, 13, 14), 40: (7, 8, 9, 12), 54: (3, 4, 6, 9), 64: (0, 2, 3, 7), 70: (0, 1, 2, 3)}


def tree_size_sweep(torch, d2sd, cfg, peaks, steps: int, layers: int = 8):
    """Attention us per layer at L = 4096 for forced prefix sets (harness input: the tree is built from a given
    prefix_len instead of the selected one)."""
    import dataclasses
    sub = dataclasses.replace(cfg, layers=min(cfg.layers, layers))
    wl = Workload(sub, d2sd, torch, host_copies=False)
    rows = []
    for T, prefixes in T_SWEEP.items():
        pl_t = torch.tensor([list(prefixes)] * sub.B, dtype=torch.int32, device="cuda")
        s = wl.step_in
        wl.tree = d2sd.build_tree(s["draft1"], s["draft2"], pl_t, s["ctx_len"], sub.T_cap, out=wl.tree)
        torch.cuda.synchronize()
        assert int(wl.tree["tree_len"][0]) == T
        wl.tree_len_host = wl.tree["tree_len"].cpu().numpy()
        wl.tree_tokens = int(wl.tree_len_host.sum())
        g = capture(torch, lambda: [wl.attention(i) for i in range(sub.layers)])
        for _ in range(3):
            g.replay()
        torch.cuda.synchronize()
        us = time_replays(torch, g, steps, None) / (steps * sub.layers) * 1e3
        roof, hbm, tc = attn_roofline(sub, wl, us, peaks, None)
        rows.append({"T": T, "attn_us_per_layer": us, "bound": roof["bound"], "frac": roof["frac"],
                     "frac_hbm": hbm["frac"], "frac_tensor": tc["frac"]})
        del g
    del wl
    torch.cuda.empty_cache()
    return rows


def stage_times(torch, wl, steps: int, flush):
    """us per call of the launch-latency-sized stages, each as its own CUDA graph (L2 flushed between replays)."""
    d, cfg = wl.d2sd, wl.cfg
    out = {}
    def timed(fn):
        g = capture(torch, fn)
        for _ in range(3):
            g.replay()
        torch.cuda.synchronize()
        return time_replays(torch, g, steps, flush) / steps * 1e3
    s = wl.step_in
    out["select_prefixes"] = timed(lambda: d.select_prefixes(s["conf"], cfg.K, prefix_len=wl.prefix_len))
    out["build_tree"] = timed(lambda: d.build_tree(s["draft1"], s["draft2"], wl.prefix_len, s["ctx_len"], cfg.T_cap, out=wl.tree))
    out["accept (argmax + walk)"] = timed(wl.accept)
    # the steps around the path: drafter confidence extraction and KV commit of one layer set
    dl = torch.randn((cfg.B, cfg.gamma - 1, cfg.V), device="cuda").to(torch.bfloat16)
    anchor = torch.zeros((cfg.B,), dtype=torch.int32, device="cuda")
    ws = torch.empty(d.confidence_workspace_bytes(cfg.B, cfg.gamma, cfg.V), dtype=torch.uint8, device="cuda")
    dr = torch.empty((cfg.B, cfg.gamma), dtype=torch.int32, device="cuda")
    cf = torch.empty((cfg.B, cfg.gamma), dtype=torch.float32, device="cuda")
    out["draft_confidence"] = timed(lambda: d.draft_confidence(dl, anchor, draft=dr, conf=cf, workspace=ws))
    return out

# ------------------------------------------------------------------------------- CPU oracle legs

def oracle_sample_seconds(cfg: synth.Config, layers_sampled: int = 1):
    """Time the oracle, as it stands, on a bounded sample of the step: select + build (whole),
    `layers_sampled` of the cfg.layers attention layers (every row), argmax + walk (whole).
    Returns (extrapolated seconds per step, measured seconds, tree tokens, description, cores)."""
    import oracle
    st = synth.make_step_inputs(cfg)
    t0 = time.perf_counter()
    pl, _ = oracle.select_prefixes(st["conf"], cfg.K)
    tree = oracle.build_tree(st["draft1"], st["draft2"], pl, st["ctx_len"], cfg.T_cap)
    t_sb = time.perf_counter() - t0
    t_attn = 0.0
    for layer in range(layers_sampled):
        ti = synth.make_tree_inputs(cfg, layer)
        kv = synth.make_kv_cache(cfg, st["ctx_len"], layer)
        t0 = time.perf_counter()
        oracle.attention(ti["q"], kv["k_cache"], kv["v_cache"], kv["kv_indptr"], kv["kv_indices"], kv["page_size"],
                         st["ctx_len"], ti["tree_k"], ti["tree_v"], tree["mask"], tree["tree_len"])
        t_attn += time.perf_counter() - t0
    logits = synth.make_logits(cfg)
    synth.plant_acceptance(cfg, logits, st["conf"], tree["tokens"], tree["parent"], tree["depth"], tree["tree_len"])
    t0 = time.perf_counter()
    oracle.accept(logits, tree["tokens"], tree["parent"], tree["depth"], tree["tree_len"], cfg.gamma)
    t_acc = time.perf_counter() - t0
    measured = t_sb + t_attn + t_acc
    step_s = t_sb + t_attn * (cfg.layers / layers_sampled) + t_acc
    desc = (f"config {cfg.number}: select+build and argmax+walk in full, {layers_sampled} of {cfg.layers} attention "
            f"layers (all {int(tree['tree_len'].sum())}x{cfg.Hq} rows), attention time scaled x{cfg.layers}/{layers_sampled}")
    return step_s, measured, int(tree["tree_len"].sum()), desc, oracle.num_threads()


def oracle_layers_within(cfg: synth.Config, budget_s: float) -> int:
    """How many of the cfg.layers attention layers the oracle gets through in about budget_s seconds on this
    host (one layer is timed first, which also warms the OpenMP pool and pages the library in)."""
    _, measured, _, _, _ = oracle_sample_seconds(cfg, 1)
    return max(1, min(cfg.layers, int(budget_s / max(measured, 1e-3))))


def run_reference(args, cfg):
    """The oracle as the reference arm: every step times select + build, as many of the cfg.layers attention layers
    (every row) as fit the run's budget of about two minutes, and argmax + walk; when fewer than cfg.layers are
    timed the step time scales the attention part (stated in `extrapolated`)."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return 0
    n_layers = oracle_layers_within(cfg, 120.0 / max(1, args.steps))  # (this first sample is the warm-up)
    ts, meas, tokens, desc, cores = [], [], 0, "", 1
    for _ in range(args.steps):
        step_s, measured, tokens, desc, cores = oracle_sample_seconds(cfg, n_layers)
        ts.append(step_s)
        meas.append(measured)
    step_s = float(np.mean(ts))
    value = tokens / step_s
    st = synth.make_step_inputs(cfg)
    import oracle
    pl_, _ = oracle.select_prefixes(st["conf"], cfg.K)
    tr_ = oracle.build_tree(st["draft1"], st["draft2"], pl_, st["ctx_len"], cfg.T_cap)
    plants = synth.plant_acceptance(cfg, synth.make_logits(cfg), st["conf"], tr_["tokens"], tr_["parent"], tr_["depth"],
                                    tr_["tree_len"])
    line = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": step_s * 1e3, "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": workload_config(cfg, st["ctx_len"], tokens, plants, 1),
            "measurement": {"timing": "time.perf_counter around the oracle calls on the host cores"},
            "extrapolated": {"what": (f"ms_per_step = select + build + {cfg.layers}/{n_layers} x ({n_layers} timed attention "
                                      f"layers) + accept") if n_layers < cfg.layers else "nothing: the whole step is timed",
                             "measured_ms_per_step": float(np.mean(meas)) * 1e3, "attention_layers_timed": n_layers,
                             "attention_layers_per_step": cfg.layers},
            "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": desc},
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line))
    return 0


# ------------------------------------------------------------------------------- main (GPU arm)

def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=200)
    ap.add_argument("--warmup", type=int, default=10)
    ap.add_argument("--config", type=int, default=2, choices=sorted(synth.CONFIGS))
    ap.add_argument("--impl", default="d2sd", choices=["d2sd", "reference"])
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-extras", action="store_true", help="skip stage times, the tree-size sweep and the per-config block")
    args = ap.parse_args()
    cfg = synth.CONFIGS[args.config]
    if args.impl == "reference":
        return run_reference(args, cfg)
    args.warmup = max(args.warmup, 3)

    import torch
    import torch.distributed as dist
    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    import paper_2606_04446_b200 as d2sd
    d2sd.lib()  # no fallback: fails here if libd2sd.so is missing

    peaks = measured_peaks()
    wl = Workload(cfg, d2sd, torch, host_copies=not args.no_e2e)
    kv_bytes_layer = 2 * int(wl.st["ctx_len"].sum()) * cfg.Hkv * cfg.d * 2
    step_bytes = kv_bytes_layer * cfg.layers
    flush = None
    if step_bytes < 2 * L2_BYTES:
        fbuf = torch.empty(2 * L2_BYTES, dtype=torch.uint8, device="cuda")
        flush = lambda: fbuf.fill_(1)  # noqa: E731

    g_step = capture(torch, wl.step)
    g_attn = capture(torch, lambda: [wl.attention(i) for i in range(cfg.layers)])

    clocks = ClockSampler(local)
    for _ in range(args.warmup):
        g_step.replay()
    _barrier()
    clocks.start()
    ms = time_replays(torch, g_step, args.steps, flush)
    _barrier()
    # dominant kernel (the cascade attention launch) alone: same launch configuration, same
    # distinct-per-layer KV, back to back as in the step
    for _ in range(3):
        g_attn.replay()
    torch.cuda.synchronize()
    ms_prefix = time_replays(torch, g_attn, args.steps, flush)
    clocks.stop()
    ms = max_over_ranks(ms)
    tokens_all = sum_over_ranks(float(wl.tree_tokens))
    ms_per_step = ms / args.steps
    value = tokens_all / (ms_per_step * 1e-3)

    # roofline of the dominant kernel (algorithmic bytes and flops per launch)
    us_prefix = ms_prefix / (args.steps * cfg.layers) * 1e3
    roofline, roof_hbm, roof_tc = attn_roofline(cfg, wl, us_prefix, peaks, ncu_traffic(wl.attn_kernel, cfg.number))

    line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": ms_per_step, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "bf16", "data": "synthetic",
            "config": workload_config(cfg, wl.st["ctx_len"], wl.tree_tokens, wl.n_plants, world),
            "measurement": {"l2": ("flushed between steps (256 MiB write)" if flush else
                                   f"inputs larger than L2 ({step_bytes / 2**20:.0f} MiB of distinct KV per step)"),
                            "timing": "CUDA-graph replay of the whole step, CUDA events on the replay stream"},
            "us_per_step": ms_per_step * 1e3,
            "attn_us_per_layer": us_prefix,
            "roofline": roofline, "roofline_hbm": roof_hbm, "roofline_tensor": roof_tc,
            "gpu_launches": wl.launches_per_step * args.steps,
            "clocks": clocks.summary()}
    if not args.no_extras:
        line["stage_us"] = stage_times(torch, wl, min(args.steps, 30), flush)
        line["stage_us"]["cascade_verify_attn (per layer)"] = us_prefix
        line["non_attention_us_per_step"] = ms_per_step * 1e3 - us_prefix * cfg.layers

    # e2e: host buffers -> device -> step -> host results, everything inside the timed region
    if not args.no_e2e:
        for name, with_kv in (("e2e", True), ("e2e_kv_resident", False)):
            n = max(3, min(args.steps, 20 if with_kv else 50))
            for _ in range(2):
                wl.e2e_step(with_kv)
            _barrier()
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            t0 = time.perf_counter()
            e0.record()
            for _ in range(n):
                wl.e2e_step(with_kv)
                torch.cuda.synchronize()  # the result is on the host when the step ends
            e1.record()
            torch.cuda.synchronize()
            wall = max(time.perf_counter() - t0, e0.elapsed_time(e1) * 1e-3)
            wall = max_over_ranks(wall)
            line[name] = {"value": tokens_all / (wall / n), "unit": UNIT, "h2d_bytes_per_step": wl.h2d_bytes(with_kv),
                          "d2h_bytes_per_step": wl.d2h_bytes(), "ms_per_step": wall / n * 1e3, "steps": n,
                          "kv_cache": "copied from pinned host memory every step" if with_kv else
                          "resident in HBM (committed state, PAPER.md:119); only the step's own inputs are copied"}

    if rank == 0 and world == 1 and not args.no_extras and cfg.number == 2:
        # the other single-GPU configs (attention launches only) and the tree-size sweep, driver-verifiable in this line
        del g_step, g_attn
        wl.layers = None
        wl.outs = None
        torch.cuda.empty_cache()
        line["tree_size_sweep_L4096"] = tree_size_sweep(torch, d2sd, cfg, peaks, min(args.steps, 30))
        line["per_config"] = [attention_only(torch, d2sd, synth.CONFIGS[n], peaks, min(args.steps, 20), layers=4)
                              for n in (3, 4, 5)]
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        step_s, measured, tokens, desc, cores = oracle_sample_seconds(cfg, oracle_layers_within(cfg, 15.0))
        line["cpu_baseline"] = {"value": tokens / step_s, "unit": UNIT, "cores": cores, "kind": "oracle",
                                "sample": desc, "sample_seconds": measured}
    if rank == 0:
        print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()
    return 0


if __name__ == "__main__":
    sys.exit(main())
