#!/usr/bin/env python
"""bench.py -- STAR-KV latent-cache decode step on B200 (contract: task prompt "Measurement").

A STEP is one pass of the whole hot path (rows A1-A4 then D1-D9) over one batch:
``starkv_append`` compresses the batch's newest token (dense-KV mode, one token per sequence,
written at position context-1) and ``starkv_decode_attn`` then attends over [0, context).

  value   = algorithmic bytes the step must move (latent + scale bytes of every cached token
            + factor bytes; synth.algorithmic_bytes_per_token / synth.factor_bytes) / step time,
            summed over ranks.  Inputs resident in HBM; the K steps are CUDA-graph launches.
  e2e     = same metric through the HOST-buffer C-ABI calls (starkv_append_host +
            starkv_decode_attn_host): pinned host q / new K,V in, out back, every step.
  roofline= the split-K decode kernel (rows D2-D7) alone, timed by CUDA events recorded by the
            library directly around that launch, against the measured HBM copy bandwidth.
  cpu_baseline / --impl reference = the CPU oracle (``oracle/``) as it stands on the host cores.

L2: every step reads a different replica of the cache (distinct seeded sequences); replicas are
sized so the footprint is >= 3x the 126 MB L2 and the cache a step reads was last touched
n_replicas steps ago.
"""
from __future__ import annotations

import argparse
import dataclasses
import json
import os
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import synth  # noqa: E402

METRIC = "decode_attn_latent_kv_hbm_gbs"
UNIT = "GB/s"
L2_BYTES = 126 * 1024 * 1024
NOMINAL_HBM_GBS = 8000.0          # north_star's denominator (context; the roofline uses the measured one)
FALLBACK_HBM_GBS = 6650.0         # B200_PROFILING.md fallback when MEASURED_PEAKS.json is absent
HEADLINE = "C3"                   # north_star target configs are C2, C3, C5; C3 (128K, int8/int4, batch 1) is the hardest


def step_bytes(cfg) -> int:
    """Algorithmic bytes of one step: every cached token's latent+scale bytes, plus per-step factor
    bytes (B_k, B_v, q, out).  DESIGN.md section 6."""
    return cfg.batch * cfg.context * synth.algorithmic_bytes_per_token(cfg)["total"] + synth.factor_bytes(cfg)


def kernel_bytes(cfg) -> int:
    """Algorithmic bytes of one launch of the split-K decode kernel: the latent cache only."""
    return cfg.batch * cfg.context * synth.algorithmic_bytes_per_token(cfg)["total"]


def measured_peak():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        try:
            with open(p) as f:
                return float(json.load(f)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
        except Exception:
            pass
    return FALLBACK_HBM_GBS, "fallback (B200_PROFILING.md)"


def stored_traffic(workload: str):
    """dram bytes per launch of the decode kernel from the committed ncu --set full summary."""
    p = os.path.join(ROOT, "profiles", "traffic.json")
    if os.path.exists(p):
        try:
            with open(p) as f:
                return json.load(f).get(workload)
        except Exception:
            return None
    return None


# ------------------------------------------------------------------------------------------------
# clocks (NVML through nvidia_ml_py; sampled in a thread during the measured phases)
# ------------------------------------------------------------------------------------------------
class ClockSampler:
    def __init__(self, device_index: int):
        self.samples = []
        self.stop = threading.Event()
        self.ok = False
        try:
            import pynvml
            import torch
            pynvml.nvmlInit()
            self.nv = pynvml
            h = None
            try:
                uuid = str(torch.cuda.get_device_properties(device_index).uuid)
                if not uuid.startswith("GPU-"):
                    uuid = "GPU-" + uuid
                h = pynvml.nvmlDeviceGetHandleByUUID(uuid)
            except Exception:
                h = pynvml.nvmlDeviceGetHandleByIndex(device_index)
            self.h = h
            self.max_mhz = int(pynvml.nvmlDeviceGetMaxClockInfo(h, pynvml.NVML_CLOCK_SM))
            self.ok = True
        except Exception as e:  # noqa: BLE001
            self.err = repr(e)
        self.thread = threading.Thread(target=self._run, daemon=True)
        self.timed = False

    def _reasons(self):
        nv = self.nv
        try:
            return int(nv.nvmlDeviceGetCurrentClocksEventReasons(self.h))
        except Exception:
            return int(nv.nvmlDeviceGetCurrentClocksThrottleReasons(self.h))

    def _run(self):
        nv = self.nv
        while not self.stop.is_set():
            try:
                self.samples.append((self.timed, int(nv.nvmlDeviceGetClockInfo(self.h, nv.NVML_CLOCK_SM)),
                                     self._reasons(), nv.nvmlDeviceGetPowerUsage(self.h) / 1000.0))
            except Exception:
                pass
            time.sleep(0.004)

    def start(self):
        if self.ok:
            self.thread.start()

    def finish(self):
        if not self.ok:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": [], "error": getattr(self, "err", "nvml")}
        self.stop.set()
        self.thread.join()
        names = {0x1: "gpu_idle", 0x2: "applications_clocks_setting", 0x4: "sw_power_cap", 0x8: "hw_slowdown",
                 0x10: "sync_boost", 0x20: "sw_thermal_slowdown", 0x40: "hw_thermal_slowdown",
                 0x80: "hw_power_brake_slowdown", 0x100: "display_clock_setting"}
        load = [s for s in self.samples if s[0]]
        use = load if load else self.samples
        mask = 0
        for s in use:
            mask |= s[2]
        reasons = [n for b, n in names.items() if mask & b and n != "gpu_idle"]
        mhz = sorted(s[1] for s in use)
        return {"sm_mhz": mhz[len(mhz) // 2] if mhz else None, "sm_max_mhz": self.max_mhz, "reasons": reasons,
                "samples_under_load": len(load), "power_w_max": max((s[3] for s in use), default=None),
                "window": "timed device loop, e2e loop, kernel-timing loop and a same-load dwell"}


# ------------------------------------------------------------------------------------------------
# device workload
# ------------------------------------------------------------------------------------------------
class Workload:
    """Device-resident replicas of one config's cache + everything a step needs."""

    def __init__(self, cfg, sk, torch, device, n_rep=None, verbose=False, stream=None):
        self.cfg, self.sk, self.torch = cfg, sk, torch
        B, ctxlen, P = cfg.batch, cfg.context, cfg.page_tokens
        self.stream = stream if stream is not None else torch.cuda.Stream(device=device)
        self.ctx = sk.create_from_config(cfg, stream=self.stream)
        page_bytes = sk.starkv_page_bytes(self.ctx)
        cache_bytes = kernel_bytes(cfg)
        self.n_rep = n_rep or max(2, -(-3 * L2_BYTES // cache_bytes))
        R = self.n_rep
        call = dataclasses.replace(cfg, batch=R * B)
        lens_all = np.full(R * B, ctxlen, np.int32)
        table, n_pool = synth.make_block_table(call, lens_all)
        self.max_pages = table.shape[1]
        self.table = torch.from_numpy(table).to(device)
        self.pool = torch.zeros((n_pool, page_bytes), dtype=torch.uint8, device=device)
        self.seq_lens = torch.full((B,), ctxlen, dtype=torch.int32, device=device)
        n_pages = (ctxlen + P - 1) // P
        tmp = torch.empty((n_pages, page_bytes), dtype=torch.uint8, device=device)
        t0 = time.time()
        with torch.cuda.stream(self.stream):
            for s in range(R * B):
                lk, lv = synth.make_latents(cfg, ctxlen, seq=s)
                dk = torch.from_numpy(lk.view(np.int16)).to(device).view(torch.float16)
                dv = torch.from_numpy(lv.view(np.int16)).to(device).view(torch.float16)
                sk.starkv_pack(self.ctx, dk, dv, ctxlen, tmp)
                self.pool[self.table[s, :n_pages].long()] = tmp
            self.stream.synchronize()
        if verbose:
            print(f"# built {R} replicas x {B} sequences x {ctxlen} tokens in {time.time() - t0:.1f}s "
                  f"({R * cache_bytes / 1e6:.0f} MB of cache)", file=sys.stderr)
        bk, bv = synth.make_factors(cfg)
        dk_in, dv_in = cfg.head_dim, cfg.n_kv_heads * cfg.head_dim
        ak, av = synth.make_append_factors(cfg, dk_in, dv_in)
        kn, vn = synth.make_append_inputs(cfg, B, mode="dense")
        q = synth.make_q(cfg, B)
        f16 = lambda a: torch.from_numpy(np.ascontiguousarray(a).view(np.int16)).to(device).view(torch.float16)  # noqa: E731
        self.bk, self.bv, self.ak, self.av = f16(bk), f16(bv), f16(ak), f16(av)
        self.q, self.k_new, self.v_new = f16(q), f16(kn), f16(vn)
        self.d_in_k, self.d_in_v = dk_in, dv_in
        self.seq_ids = torch.arange(B, dtype=torch.int32, device=device)
        self.positions = torch.full((B,), ctxlen - 1, dtype=torch.int32, device=device)
        self.wsb = sk.starkv_workspace_bytes(self.ctx, B, self.max_pages)
        self.ws = torch.empty(self.wsb, dtype=torch.uint8, device=device)
        self.awsb = max(sk.starkv_append_workspace_bytes(self.ctx, B),
                        sk.starkv_append_host_workspace_bytes(self.ctx, B, cfg.n_kv_heads * cfg.head_dim, dv_in))
        self.aws = torch.empty(self.awsb, dtype=torch.uint8, device=device)
        self.out = torch.zeros((B, cfg.n_q_heads, cfg.head_dim), dtype=torch.float16, device=device)
        # pinned host buffers for the e2e leg
        pin = lambda a: torch.from_numpy(np.ascontiguousarray(a).view(np.int16)).pin_memory()  # noqa: E731
        self.h_q, self.h_k, self.h_v = pin(q), pin(kn), pin(vn)
        self.h_seq = torch.arange(B, dtype=torch.int32).pin_memory()
        self.h_pos = torch.full((B,), ctxlen - 1, dtype=torch.int32).pin_memory()
        self.h_lens = torch.full((B,), ctxlen, dtype=torch.int32).pin_memory()
        self.h_out = torch.zeros((B, cfg.n_q_heads, cfg.head_dim), dtype=torch.float16).pin_memory()
        self.launches_per_step = 0

    def table_of(self, rep):
        return self.table[rep * self.cfg.batch:].data_ptr()

    def step(self, rep):
        """One whole-path step on replica ``rep`` with device-resident inputs (enqueue only)."""
        sk, c, B = self.sk, self.cfg, self.cfg.batch
        sk.starkv_decode_step(self.ctx, self.pool, self.table_of(rep), self.max_pages, self.seq_ids, self.positions, B,
                              self.k_new, c.n_kv_heads * c.head_dim, c.head_dim, self.d_in_k, self.v_new, self.d_in_v,
                              self.d_in_v, self.ak, self.av, self.aws, self.awsb, self.q, self.seq_lens, self.bk, self.bv,
                              self.ws, self.wsb, self.out)
        self.launches_per_step = sk.starkv_last_launches(self.ctx)

    def step_host(self, rep):
        """Same step through the HOST-buffer entry point (starkv_decode_step_host); returns after `out` is back on the host."""
        sk, c, B = self.sk, self.cfg, self.cfg.batch
        sk.starkv_decode_step_host(self.ctx, self.pool, self.table_of(rep), self.max_pages, self.h_seq, self.h_pos, B,
                                   self.h_k, c.n_kv_heads * c.head_dim, c.head_dim, self.d_in_k, self.h_v, self.d_in_v,
                                   self.d_in_v, self.ak, self.av, self.aws, self.awsb, self.h_q, self.h_lens, self.bk, self.bv,
                                   self.ws, self.wsb, self.h_out)

    def h2d_bytes(self):
        return int(self.h_q.numel() * 2 + self.h_k.numel() * 2 + self.h_v.numel() * 2 + 3 * self.cfg.batch * 4)

    def d2h_bytes(self):
        return int(self.h_out.numel() * 2)


# ------------------------------------------------------------------------------------------------
# CPU oracle legs (cpu_baseline at N=1, and --impl reference)
# ------------------------------------------------------------------------------------------------
class OracleSample:
    """A bounded sample of the workload on the host: ``n_seq`` sequences of ``tokens`` cached tokens,
    packed by the oracle's own codec, decoded by the oracle's plain-definition attention (all heads)."""

    def __init__(self, cfg, n_seq, tokens):
        from oracle import codec as ocodec
        from oracle.layout import CacheDesc
        self.cfg = dataclasses.replace(cfg, batch=n_seq, context=tokens)
        self.d = CacheDesc.from_config(self.cfg)
        lens = np.full(n_seq, tokens, np.int32)
        self.table, n_pool = synth.make_block_table(self.cfg, lens)
        from oracle.layout import page_layout
        self.pool = np.zeros((n_pool, page_layout(self.d).page_bytes), np.uint8)
        for s in range(n_seq):
            lk, lv = synth.make_latents(cfg, tokens, seq=s)
            pages = ocodec.pack_pages(self.d, lk, lv)
            self.pool[self.table[s, :pages.shape[0]]] = pages
        self.lens = lens
        self.bk, self.bv = synth.make_factors(cfg)
        self.q = synth.make_q(cfg, n_seq)
        self.bytes = step_bytes(self.cfg)
        self.sample = f"{n_seq} sequence(s) x {tokens} cached tokens of {cfg.name}, all {cfg.n_q_heads} query heads"

    def run(self):
        from oracle import attention as oattn
        return oattn.decode_attn(self.d, self.q, self.pool, self.table, self.lens, self.bk, self.bv)


def oracle_cores() -> int:
    try:
        return len(os.sched_getaffinity(0))
    except AttributeError:
        return os.cpu_count() or 1


def cpu_baseline(cfg, budget_s=15.0):
    """Oracle timed on a bounded sample sized for ~budget_s seconds of CPU work."""
    probe = OracleSample(cfg, 1, min(cfg.context, 4096))
    t0 = time.perf_counter()
    probe.run()
    tok_per_s = probe.cfg.context / max(time.perf_counter() - t0, 1e-6)
    total = cfg.batch * cfg.context
    want = int(min(total, max(4096, tok_per_s * budget_s / 3)))      # run it 3 times, keep the best
    n_seq = max(1, min(cfg.batch, want // cfg.context)) if want >= cfg.context else 1
    tokens = cfg.context if want >= cfg.context else max(64, want // 64 * 64)
    smp = OracleSample(cfg, n_seq, tokens)
    best = float("inf")
    for _ in range(3):
        t0 = time.perf_counter()
        smp.run()
        best = min(best, time.perf_counter() - t0)
    return {"value": smp.bytes / best / 1e9, "unit": UNIT, "cores": oracle_cores(), "kind": "oracle",
            "sample": smp.sample + f"; best of 3 runs, {best:.2f} s per run",
            "us_per_step_per_layer_extrapolated": best * 1e6 * total / (n_seq * tokens)}


def run_reference(args, cfg):
    """--impl reference: the oracle, as it stands, on the host cores; each step = one decode of a
    bounded sample sized so that steps+warmup finish within ~2 minutes."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    probe = OracleSample(cfg, 1, min(cfg.context, 2048))
    t0 = time.perf_counter()
    probe.run()
    tok_per_s = probe.cfg.context / max(time.perf_counter() - t0, 1e-6)
    per_step = 120.0 / max(1, args.steps + args.warmup)
    want = int(tok_per_s * per_step)
    total = cfg.batch * cfg.context
    if want >= total:
        n_seq, tokens = cfg.batch, cfg.context
    elif want >= cfg.context:
        n_seq, tokens = want // cfg.context, cfg.context
    else:
        n_seq, tokens = 1, max(64, want // 64 * 64)
    smp = OracleSample(cfg, n_seq, tokens)
    for _ in range(args.warmup):
        smp.run()
    t0 = time.perf_counter()
    for _ in range(args.steps):
        smp.run()
    dt = (time.perf_counter() - t0) / max(1, args.steps)
    v = smp.bytes / dt / 1e9
    line = {"impl": "reference", "metric": METRIC, "value": v, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": dt * 1e3, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": workload_name(cfg), "sample": smp.sample},
            "cpu_baseline": {"value": v, "unit": UNIT, "cores": oracle_cores(), "kind": "oracle", "sample": smp.sample},
            "e2e": {"value": v, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line))


def prefill_append_leg(wl, sk, torch, device, T):
    """starkv_append on T new tokens spread over the batch (positions at the end of each sequence), in dense-KV
    mode (K/V rows in, north_star's call) and hidden-state mode (x in).  Device-resident inputs,
    CUDA events around 20 calls; flops = 2 * T * d_in * columns of the projections only."""
    cfg = wl.cfg
    B, per = cfg.batch, T // cfg.batch
    T = per * B
    seq = torch.arange(B, dtype=torch.int32, device=device).repeat_interleave(per)
    pos = (torch.arange(per, dtype=torch.int32, device=device) + (cfg.context - per)).repeat(B)
    wsb = sk.starkv_append_workspace_bytes(wl.ctx, T)
    ws = torch.empty(wsb, dtype=torch.uint8, device=device)
    f16 = lambda a: torch.from_numpy(np.ascontiguousarray(a).view(np.int16)).to(device).view(torch.float16)  # noqa: E731
    out = {"tokens": T}
    for mode in ("dense", "hidden"):
        if mode == "dense":
            dk, dv, khs = cfg.head_dim, cfg.n_kv_heads * cfg.head_dim, cfg.head_dim
            kn, vn = synth.make_append_inputs(cfg, T, mode="dense")
            k, v = f16(kn.reshape(T, -1)), f16(vn)
            ak, av = wl.ak, wl.av
            flops = 2.0 * T * (cfg.head_dim * cfg.sum_rank_k + dv * cfg.rank_v)
        else:
            dk = dv = cfg.d_model
            khs = 0
            xn, _ = synth.make_append_inputs(cfg, T, mode="hidden")
            k = v = f16(xn)
            a1, a2 = synth.make_append_factors(cfg, dk, dv)
            ak, av = f16(a1), f16(a2)
            flops = 2.0 * T * cfg.d_model * (cfg.sum_rank_k + cfg.rank_v)
        call = lambda: sk.starkv_append(wl.ctx, wl.pool, wl.table_of(0), wl.max_pages, seq, pos, T, k, k.shape[1], khs,  # noqa: E731
                                        dk, v, v.shape[1], dv, ak, av, ws, wsb)
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        with torch.cuda.stream(wl.stream):
            for _ in range(3):
                call()
            e0.record(wl.stream)
            for _ in range(20):
                call()
            e1.record(wl.stream)
            wl.stream.synchronize()
        us = e0.elapsed_time(e1) * 1e3 / 20
        out[mode] = {"us_per_call": us, "projection_tflops": flops / (us * 1e-6) / 1e12, "d_in_k": dk, "d_in_v": dv,
                     "kernel": sk.starkv_last_append_kernel_name(wl.ctx), "launches": sk.starkv_last_launches(wl.ctx)}
    return out


def latent_output_leg(wl, sk, torch, device, K=300):
    """NEXT-3: decode attention alone (no append), once with the B_v up-projection (starkv_decode_attn) and once in
    latent-output mode (starkv_decode_attn_latent: merge-only combine, o~ [batch, H_q, r_v]); one CUDA graph per cache
    replica, K replays each, CUDA events on the workload's stream."""
    cfg, B, R = wl.cfg, wl.cfg.batch, wl.n_rep
    out_lat = torch.zeros((B, cfg.n_q_heads, cfg.rank_v), dtype=torch.float16, device=device)
    calls = {
        "decode_attn_us": lambda rep: sk.starkv_decode_attn(wl.ctx, wl.q, wl.pool, wl.table_of(rep), wl.max_pages, wl.seq_lens, B,
                                                             wl.bk, wl.bv, wl.ws, wl.wsb, wl.out),
        "decode_attn_latent_us": lambda rep: sk.starkv_decode_attn_latent(wl.ctx, wl.q, wl.pool, wl.table_of(rep), wl.max_pages,
                                                                           wl.seq_lens, B, wl.bk, wl.ws, wl.wsb, out_lat),
    }
    res = {"calls_timed": K, "out_latent_shape": [B, cfg.n_q_heads, cfg.rank_v]}
    with torch.cuda.stream(wl.stream):
        for key, fn in calls.items():
            graphs = []
            for rep in range(R):
                fn(rep)
            wl.stream.synchronize()
            for rep in range(R):
                g = torch.cuda.CUDAGraph()
                with torch.cuda.graph(g, stream=wl.stream):
                    fn(rep)
                graphs.append(g)
            for i in range(10):
                graphs[i % R].replay()
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record(wl.stream)
            for i in range(K):
                graphs[i % R].replay()
            e1.record(wl.stream)
            wl.stream.synchronize()
            res[key] = e0.elapsed_time(e1) * 1e3 / K
            del graphs
    return res


def workload_name(cfg) -> str:
    kind = "fp16 latents" if not cfg.quantized else f"int{cfg.bits_hi}/int{cfg.bits_lo} latents"
    return (f"{cfg.name}: BASELINE.json configs[{int(cfg.name[1]) - 1}], 1 layer, batch {cfg.batch}, "
            f"{cfg.n_q_heads}q/{cfg.n_kv_heads}kv heads x {cfg.head_dim}, context {cfg.context}, "
            f"key ranks {cfg.rank_k}, value rank {cfg.rank_v}, {kind}")


# ------------------------------------------------------------------------------------------------
# our arm
# ------------------------------------------------------------------------------------------------
def run_ours(args, cfg, env, K, with_cpu):
    """One single-layer workload (C2, C3 or C4) on every rank; returns the JSON line as a dict (rank 0) or None."""
    import torch
    import torch.distributed as dist

    import paper_2606_08382_b200 as sk      # raises if libstarkv.so is missing: there is no fallback
    from paper_2606_08382_b200.sharding import max_over_ranks

    world, rank, local, device = env
    W = max(args.warmup, 3)

    # weak scaling: every rank owns one full BASELINE batch (sequences are independent: no collective)
    wl = Workload(cfg, sk, torch, device, n_rep=args.replicas or None, verbose=(rank == 0 and args.verbose))
    R = wl.n_rep
    with torch.cuda.stream(wl.stream):
        for i in range(W):
            wl.step(i % R)
        wl.stream.synchronize()
        graphs = []
        for rep in range(R):
            g = torch.cuda.CUDAGraph()
            with torch.cuda.graph(g, stream=wl.stream):
                wl.step(rep)
            graphs.append(g)
        for i in range(W):
            graphs[i % R].replay()
        wl.stream.synchronize()
    launches_per_step = wl.launches_per_step

    sampler = ClockSampler(local)
    sampler.start()

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    # ---- device-resident timed region: exactly K steps ----
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier()
    sampler.timed = True
    with torch.cuda.stream(wl.stream):
        ev0.record(wl.stream)
        for i in range(K):
            graphs[i % R].replay()
        ev1.record(wl.stream)
    barrier()
    sampler.timed = False
    ms_total = max_over_ranks(ev0.elapsed_time(ev1), device)
    ms_step = ms_total / K
    value = world * step_bytes(cfg) / (ms_step * 1e-3) / 1e9

    # ---- e2e: HOST buffers through the C ABI, copies inside the timed region ----
    Ke = min(K, 2000)
    for i in range(3):
        wl.step_host(i % R)
    barrier()
    sampler.timed = True
    ev0.record(wl.stream)
    for i in range(Ke):
        wl.step_host(i % R)
    ev1.record(wl.stream)
    barrier()
    sampler.timed = False
    ms_e2e = max_over_ranks(ev0.elapsed_time(ev1), device) / Ke
    e2e = world * step_bytes(cfg) / (ms_e2e * 1e-3) / 1e9

    # ---- roofline: the split-K decode kernel alone (events recorded by the library around it) ----
    Kr = min(K, 200)
    sk.starkv_set_kernel_timing(wl.ctx, True)
    kms = []
    sampler.timed = True
    with torch.cuda.stream(wl.stream):
        for i in range(Kr + 3):
            torch.cuda._sleep(300000)   # ~150 us spin kernel: the host runs ahead, so the library's events sit
                                        # directly around the kernel; L2 is defeated by the replica rotation
            wl.step(i % R)
            ms = sk.starkv_last_decode_kernel_ms(wl.ctx)
            if i >= 3:
                kms.append(ms)
    sampler.timed = False
    sk.starkv_set_kernel_timing(wl.ctx, False)
    k_ms = float(np.mean(kms))
    peak, peak_src = measured_peak()
    achieved = kernel_bytes(cfg) / (k_ms * 1e-3) / 1e9

    # ---- C4: the compress-on-append kernel on a prefill chunk (BASELINE.json configs[3]) ----
    prefill = prefill_append_leg(wl, sk, torch, device, args.prefill_tokens) if (cfg.name == "C4" or args.prefill) else None
    # ---- headline config: latent-output mode beside the plain decode ----
    latent = latent_output_leg(wl, sk, torch, device) if cfg.name == HEADLINE else None

    # ---- clocks: if the timed loops were too short to be sampled, dwell on the same load ----
    if sampler.ok and sum(1 for s in sampler.samples if s[0]) < 8:
        sampler.timed = True
        t_end = time.time() + 0.6
        with torch.cuda.stream(wl.stream):
            while time.time() < t_end:
                for i in range(64):
                    graphs[i % R].replay()
                wl.stream.synchronize()
        sampler.timed = False
    clocks = sampler.finish()
    torch.cuda.synchronize()

    h2d_b, d2h_b, kname = wl.h2d_bytes(), wl.d2h_bytes(), sk.starkv_decode_kernel_name(wl.ctx)
    del graphs, wl
    torch.cuda.empty_cache()
    if rank != 0:
        return None
    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": K, "warmup": W,
        "ms_per_step": ms_step, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f16", "data": "synthetic",
        "config": {"workload": workload_name(cfg), "parallelism": f"dp{world} (batch-sharded replicas, no collective)",
                   "step": "starkv_decode_step = starkv_append (1 new token / sequence, dense-KV mode) + starkv_decode_attn, launch-fused",
                   "l2": f"each step reads a different one of {R} cache replicas "
                         f"({R * kernel_bytes(cfg) / 1e6:.0f} MB footprint vs 126 MB L2)",
                   "launch": "CUDA graph per step (device-resident leg)", "bytes_per_step": step_bytes(cfg)},
        "us_per_step_per_layer": ms_step * 1e3,
        "tokens_per_s_attn_only_32_layers": world * cfg.batch / (32 * ms_step * 1e-3),
        "frac_of_nominal_8TBs": value / world / NOMINAL_HBM_GBS,
        "e2e": {"value": e2e, "unit": UNIT, "h2d_bytes_per_step": h2d_b, "d2h_bytes_per_step": d2h_b,
                "ms_per_step": ms_e2e, "steps": Ke},
        "gpu_launches": K * launches_per_step,
        "clocks": clocks,
        "roofline": {"bound": "hbm", "kernel": kname + " (rows D2-D7)", "achieved": achieved,
                     "peak": peak,
                     "unit": "GB/s", "frac": achieved / peak, "traffic": stored_traffic(cfg.name),
                     "peak_source": peak_src, "kernel_us": k_ms * 1e3, "kernel_us_min": float(np.min(kms)) * 1e3,
                     "launches_timed": Kr, "algorithmic_bytes_per_launch": kernel_bytes(cfg),
                     "frac_of_nominal_8TBs": achieved / NOMINAL_HBM_GBS},
    }
    if prefill is not None:
        line["append_prefill"] = prefill
    if latent is not None:
        line["latent_output"] = latent
    if world == 1 and with_cpu:
        line["cpu_baseline"] = cpu_baseline(cfg)
    return line


# ------------------------------------------------------------------------------------------------
# C5: the full 32-layer decode step (BASELINE.json configs[4])
# ------------------------------------------------------------------------------------------------
N_LAYERS_C5 = 32
# LLaMA-3.1-8B-shaped weights read once per decode step: 32 x (q,o 2 x 4096^2 + k,v 2 x 4096 x 1024
# + mlp 3 x 4096 x 14336) + lm_head 128256 x 4096, fp16
NON_ATTN_WEIGHT_BYTES = 2 * (32 * (2 * 4096 * 4096 + 2 * 4096 * 1024 + 3 * 4096 * 14336) + 128256 * 4096)


def run_c5(args, env, K):
    """One step = starkv_append + starkv_decode_attn for each of the 32 layers (each layer its own rank table,
    context and cache), captured as one CUDA graph.  The 32 caches (2.9 GB) are the L2 defeat."""
    import torch
    import torch.distributed as dist

    import paper_2606_08382_b200 as sk
    from paper_2606_08382_b200.sharding import max_over_ranks

    world, rank, local, device = env
    W = max(args.warmup, 3)
    n_layers = args.layers or N_LAYERS_C5
    stream = torch.cuda.Stream(device=device)
    layers = []
    t0 = time.time()
    for l in range(n_layers):
        cfg = synth.make_config("C5", layer=l)
        layers.append(Workload(cfg, sk, torch, device, n_rep=1, stream=stream))
    if rank == 0 and args.verbose:
        print(f"# built {n_layers} layer caches in {time.time() - t0:.1f}s", file=sys.stderr)
    bytes_step = sum(step_bytes(w.cfg) for w in layers)
    bytes_kern = sum(kernel_bytes(w.cfg) for w in layers)

    def step():
        for w in layers:
            w.step(0)

    with torch.cuda.stream(stream):
        for _ in range(W):
            step()
        stream.synchronize()
        g = torch.cuda.CUDAGraph()
        with torch.cuda.graph(g, stream=stream):
            step()
        for _ in range(W):
            g.replay()
        stream.synchronize()
    launches = sum(w.launches_per_step for w in layers)
    sampler = ClockSampler(local)
    sampler.start()

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier()
    sampler.timed = True
    with torch.cuda.stream(stream):
        ev0.record(stream)
        for _ in range(K):
            g.replay()
        ev1.record(stream)
    barrier()
    sampler.timed = False
    ms_step = max_over_ranks(ev0.elapsed_time(ev1), device) / K
    value = world * bytes_step / (ms_step * 1e-3) / 1e9

    Ke = min(K, 200)
    for _ in range(2):
        for w in layers:
            w.step_host(0)
    barrier()
    sampler.timed = True
    ev0.record(stream)
    for _ in range(Ke):
        for w in layers:
            w.step_host(0)
    ev1.record(stream)
    barrier()
    sampler.timed = False
    ms_e2e = max_over_ranks(ev0.elapsed_time(ev1), device) / Ke
    e2e = world * bytes_step / (ms_e2e * 1e-3) / 1e9

    kms = []
    sampler.timed = True
    with torch.cuda.stream(stream):
        for it in range(4):
            tot = 0.0
            for w in layers:
                sk.starkv_set_kernel_timing(w.ctx, True)
                torch.cuda._sleep(300000)
                w.step(0)
                tot += sk.starkv_last_decode_kernel_ms(w.ctx)
                sk.starkv_set_kernel_timing(w.ctx, False)
            if it:
                kms.append(tot)
    sampler.timed = False
    k_ms = float(np.mean(kms))
    peak, peak_src = measured_peak()
    achieved = bytes_kern / (k_ms * 1e-3) / 1e9
    clocks = sampler.finish()
    torch.cuda.synchronize()
    h2d_b, d2h_b = sum(w.h2d_bytes() for w in layers), sum(w.d2h_bytes() for w in layers)
    kname, c0 = sk.starkv_decode_kernel_name(layers[0].ctx), layers[0].cfg
    del g, layers
    torch.cuda.empty_cache()
    if rank != 0:
        return None
    non_attn_ms = NON_ATTN_WEIGHT_BYTES / (peak * 1e9) * 1e3
    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": K, "warmup": W,
        "ms_per_step": ms_step, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f16", "data": "synthetic",
        "config": {"workload": f"C5: BASELINE.json configs[4], {n_layers} layers, batch {c0.batch}, {c0.n_q_heads}q/{c0.n_kv_heads}kv "
                               f"heads x {c0.head_dim}, context {c0.context}, per-layer key ranks from the seeded profile "
                               f"(mean 32), value rank {c0.rank_v}, int8/int4 latents",
                   "parallelism": f"dp{world} (batch-sharded replicas, no collective)",
                   "step": f"{n_layers} x starkv_decode_step (append of 1 new token / sequence + decode attention)",
                   "l2": f"{n_layers} distinct layer caches, {bytes_kern / 1e6:.0f} MB per step vs 126 MB L2",
                   "launch": "one CUDA graph per step", "bytes_per_step": bytes_step},
        "us_per_step_per_layer": ms_step * 1e3 / n_layers,
        "tokens_per_s_attn_only": world * c0.batch / (ms_step * 1e-3) * (N_LAYERS_C5 / n_layers),
        "attention_share_model": {"attention_ms": ms_step * N_LAYERS_C5 / n_layers, "non_attention_ms_bandwidth_model": non_attn_ms,
                                  "share": ms_step * N_LAYERS_C5 / n_layers / (ms_step * N_LAYERS_C5 / n_layers + non_attn_ms),
                                  "tokens_per_s": world * c0.batch / ((ms_step * N_LAYERS_C5 / n_layers + non_attn_ms) * 1e-3),
                                  "model": "LLaMA-3.1-8B-shaped fp16 weights (%.1f GB) read once per step at the measured HBM "
                                           "bandwidth; the library holds no such code" % (NON_ATTN_WEIGHT_BYTES / 1e9)},
        "frac_of_nominal_8TBs": value / world / NOMINAL_HBM_GBS,
        "e2e": {"value": e2e, "unit": UNIT, "h2d_bytes_per_step": h2d_b, "d2h_bytes_per_step": d2h_b, "ms_per_step": ms_e2e,
                "steps": Ke},
        "gpu_launches": K * launches,
        "clocks": clocks,
        "roofline": {"bound": "hbm", "kernel": kname + " (rows D2-D7), summed over the layers of a step",
                     "achieved": achieved, "peak": peak, "unit": "GB/s", "frac": achieved / peak,
                     "traffic": stored_traffic("C5"), "peak_source": peak_src, "kernel_us": k_ms * 1e3,
                     "launches_timed": len(kms) * n_layers, "algorithmic_bytes_per_launch": bytes_kern / n_layers,
                     "frac_of_nominal_8TBs": achieved / NOMINAL_HBM_GBS},
    }
    return line


def summary(d):
    """What the per_config block keeps of a workload's line."""
    r = d["roofline"]
    out = {"workload": d["config"]["workload"], "steps": d["steps"], "step_us": d["ms_per_step"] * 1e3,
           "us_per_step_per_layer": d["us_per_step_per_layer"], "value": d["value"], "unit": d["unit"],
           "frac_of_nominal_8TBs": d["frac_of_nominal_8TBs"],
           "roofline": {k: r[k] for k in ("kernel", "kernel_us", "achieved", "peak", "frac", "traffic", "frac_of_nominal_8TBs")},
           "e2e": {"value": d["e2e"]["value"], "ms_per_step": d["e2e"]["ms_per_step"]},
           "gpu_launches_per_step": d["gpu_launches"] // max(1, d["steps"])}
    for k in ("append_prefill", "latent_output", "attention_share_model", "tokens_per_s_attn_only", "tokens_per_s_attn_only_32_layers"):
        if k in d:
            out[k] = d[k]
    return out


def spawn_ranks(n):
    """`bench.py --gpus N` outside torchrun: start the N ranks ourselves (one process per GPU, NCCL rendezvous on
    127.0.0.1) with the same arguments."""
    import socket
    with socket.socket() as so:
        so.bind(("127.0.0.1", 0))
        port = so.getsockname()[1]
    os.execvp(sys.executable, [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={n}",
                               "--master-addr", "127.0.0.1", "--master-port", str(port), os.path.abspath(__file__)] + sys.argv[1:])


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=2000)
    ap.add_argument("--warmup", type=int, default=20)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="all",
                    help="all (default: headline C3 + per_config block with C2, C4, C5), or one of C2, C3, C4, C5")
    ap.add_argument("--replicas", type=int, default=0)
    ap.add_argument("--layers", type=int, default=0, help="C5 only: number of layers (default 32)")
    ap.add_argument("--no-cpu", action="store_true", help="skip the cpu_baseline leg")
    ap.add_argument("--prefill", action="store_true", help="also time starkv_append on a prefill chunk (always on for C4)")
    ap.add_argument("--prefill-tokens", type=int, default=2048)
    ap.add_argument("--verbose", action="store_true")
    args = ap.parse_args()
    if args.impl == "reference":
        run_reference(args, synth.make_config(HEADLINE if args.workload == "all" else args.workload))
        return
    if args.gpus > 1 and "WORLD_SIZE" not in os.environ:
        spawn_ranks(args.gpus)
    import torch
    import torch.distributed as dist
    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the product path has no CPU fallback")
    torch.cuda.set_device(local)
    device = torch.device("cuda", local)
    if world > 1:
        dist.init_process_group("nccl", device_id=device)
    env = (world, rank, local, device)

    def measure(name, K, with_cpu):
        if name == "C5":
            return run_c5(args, env, K)
        return run_ours(args, synth.make_config(name), env, K, with_cpu)

    if args.workload != "all":
        line = measure(args.workload, args.steps, not args.no_cpu)
    else:
        # headline = the hardest target configuration (C3: 128K context, int8/int4): exactly --steps timed steps.  The other
        # BASELINE.json configurations are measured the same way with a bounded number of steps and reported in per_config.
        line = measure(HEADLINE, args.steps, not args.no_cpu)
        per = {HEADLINE: summary(line)} if line is not None else {}
        for name in ("C2", "C4", "C5"):
            d = measure(name, min(args.steps, 200 if name == "C5" else 500), False)
            if d is not None:
                per[name] = summary(d)
        if line is not None:
            line["per_config"] = per
    if rank == 0 and line is not None:
        print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
