#!/usr/bin/env python
"""bench.py -- the pre-position hot path on B200, measured.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config c1|c2|c3|c4|c5] [--impl reference]

A step is one pass of the whole hot path over one batch of synthetic
sessions, every stage through the C ABI of libprepos (ctypes binding, paper_2606_29565_b200.prepos):

    prepos_invalidate   the data update commits: version bump (a6)
    prepos_entry_attn   budget check, Append(E), entry attention over the paged KV, all layers (a0-a2)
    prepos_ready_dist   LM head at the last entry position fused with the vocabulary reduction (a3-a4)
    prepos_gate_serve   the request(s) that arrive next are answered from the cached record (a5)

It prints ONE compact JSON line on stdout (a few KB: the contract fields of the headline workload, which the driver
parses) and writes every side measurement to gpurun_out/bench_detail.json.  Without --config the headline is
configs[4] (70B-shaped: the paper's measured model class, and the largest per-session pass: 7.56 GB),
timed with the caller's --steps / --warmup; the other four configs then run with their own defaults and appear in the
line only as `other_configs` (us/session + roofline fraction; everything else about them is in the detail file).
--config cN runs that one config alone (what the ncu captures under profiles/ use).  See DESIGN.md "Measurement".
`--impl reference` times the CPU oracle (oracle/) on a bounded sample of the headline workload instead.
"""
from __future__ import annotations

import argparse
import json
import math
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

from paper_2606_29565_b200 import synth

METRIC = "prepos_entry_us_per_session"
UNIT = "us/session"
L2_BYTES = 126 << 20
HEADLINE = "c5"
ALL_CONFIGS = ["c1", "c2", "c3", "c4", "c5"]
DEFAULT_STEPS = {"c1": (200, 20), "c2": (100, 10), "c3": (40, 5), "c4": (10, 3), "c5": (40, 5)}


# ----------------------------------------------------------------------------------------------------
# workloads (BASELINE.json configs; recipe in DESIGN.md "Input recipe")
# ----------------------------------------------------------------------------------------------------
def workload_spec(name: str):
    seed = synth.SEED_BASE + int(name[1])
    if name == "c1":
        return dict(name=name, shape=synth.C1, n_s=[256], l_entry=[8], resident=4, serves=1, seed=seed, flush_l2=True,
                    text="configs[0] tiny: 1 session, n_s=256, L=8, 4/2 heads, d=64, H=256, V=1024")
    if name == "c2":
        return dict(name=name, shape=synth.C2, n_s=[4096], l_entry=[24], resident=4, serves=1, seed=seed, flush_l2=False,
                    text="configs[1] Llama-3-8B-shaped streaming session: 32 layers, 32/8 heads, d=128, page 16, "
                         "n_s=4096, L_entry=24, H=4096, V=128256")
    if name == "c3":
        return dict(name=name, shape=synth.C3, n_s=[32768], l_entry=[16], resident=2, serves=1, seed=seed, flush_l2=False,
                    text="configs[2] long streaming session: 8B shapes, n_s=32768, L_entry=16")
    if name == "c4":
        return dict(name=name, shape=synth.C4, n_s=synth.lognormal_ns(64, seed), l_entry=synth.uniform_l(64, seed),
                    resident=1, serves=4096, seed=seed, flush_l2=False,
                    text="configs[3] agentic batch: 64 sessions, 8B shapes, n_s~lognormal[1024,16384], L~U{32..96}, "
                         "shuffled pages, one batched ready-dist, 4096 gate serves")
    if name == "c5":
        return dict(name=name, shape=synth.C5, n_s=[16384], l_entry=[32], resident=4, serves=1, seed=seed, flush_l2=False,
                    text="configs[4] 70B-shaped: 80 layers, 64/8 heads, d=128, n_s=16384, L_entry=32, H=8192, V=128256, "
                         "sessions pre-positioned back to back")
    raise SystemExit(f"unknown config {name}")


def algorithmic_bytes(spec):
    """Bytes the pass must move once: every cached K/V byte + Q read + O write + entry K/V read
    and append write for attention; W once per ready-dist launch + hidden + records."""
    s = spec["shape"]
    kv = sum(spec["n_s"]) * s.layers * s.Hkv * s.d * 2 * 2
    sum_l = sum(spec["l_entry"])
    qo = sum_l * s.layers * s.Hq * s.d * 2 * 2
    new = sum_l * s.layers * s.Hkv * s.d * 2 * 2 * 2
    n = len(spec["n_s"])
    rd = s.V * s.H * 2 + n * s.H * 2 + n * 48
    return {"entry_attn": kv + qo + new, "ready_dist": rd, "kv": kv}


def attention_flops(spec):
    """2 GEMMs (QK^T and PV) over cached tokens, plus the causal entry triangle."""
    s = spec["shape"]
    f = 0
    for n_s, L in zip(spec["n_s"], spec["l_entry"]):
        f += 4 * s.Hq * s.d * (L * n_s + L * (L + 1) // 2)
    return f * s.layers


def ncu_traffic(config, kernel):
    """DRAM bytes (dram__bytes_read.sum + dram__bytes_write.sum) of ONE launch of `kernel` on `config`, from the
    committed summary of the `ncu --set full` captures, profiles/ncu_traffic.csv (columns: config, kernel,
    dram_read_bytes, dram_write_bytes, capture = the .md under profiles/ that documents the command, commit).  It is a
    measurement of THAT capture, not of this run: the source is returned with it.  (None, None) without a row."""
    path = os.path.join(ROOT, "profiles", "ncu_traffic.csv")
    if not os.path.exists(path):
        return None, None
    best = None
    with open(path) as f:
        for ln in f:
            parts = [x.strip() for x in ln.split(",")]
            if len(parts) < 6 or parts[0].startswith("#") or parts[0] == "config":
                continue
            if parts[0] == config and parts[1] == kernel:
                best = parts            # the last row wins (newest capture)
    if best is None:
        return None, None
    return int(float(best[2])) + int(float(best[3])), f"profiles/{best[4]}@{best[5]}"


def peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        with open(p) as f:
            m = json.load(f)
        return dict(hbm=float(m["hbm_gbs"]), bf16=float(m["bf16_tflops"]),
                    bf16_sustained=float(m.get("bf16_tflops_sustained", m["bf16_tflops"])), source="measured")
    return dict(hbm=6650.0, bf16=1590.0, bf16_sustained=1400.0, source="fallback")


# ----------------------------------------------------------------------------------------------------
# clocks during the timed region
# ----------------------------------------------------------------------------------------------------
class ClockSampler:
    def __init__(self, index: int, period_s: float = 0.005):
        self.samples, self.reasons, self.max_mhz = [], set(), None
        self._stop = threading.Event()
        self._t = None
        self.period = period_s
        try:
            import pynvml
            pynvml.nvmlInit()
            self.nv = pynvml
            # honour CUDA_VISIBLE_DEVICES: map the torch index to the NVML device through its UUID
            uuid = torch.cuda.get_device_properties(index).uuid
            try:
                self.h = pynvml.nvmlDeviceGetHandleByUUID("GPU-" + str(uuid))
            except Exception:  # noqa: BLE001  (older bindings want bytes)
                self.h = pynvml.nvmlDeviceGetHandleByUUID(("GPU-" + str(uuid)).encode())
            self.max_mhz = pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM)
        except Exception as e:  # noqa: BLE001
            self.nv, self.err = None, repr(e)

    def _loop(self):
        nv = self.nv
        names = {
            getattr(nv, "nvmlClocksEventReasonHwSlowdown", 0x8): "hw_slowdown",
            getattr(nv, "nvmlClocksEventReasonHwThermalSlowdown", 0x40): "hw_thermal_slowdown",
            getattr(nv, "nvmlClocksEventReasonSwThermalSlowdown", 0x20): "sw_thermal_slowdown",
            getattr(nv, "nvmlClocksEventReasonSwPowerCap", 0x4): "sw_power_cap",
        }
        get_reasons = getattr(nv, "nvmlDeviceGetCurrentClocksEventReasons", None) or \
            getattr(nv, "nvmlDeviceGetCurrentClocksThrottleReasons")
        while not self._stop.is_set():
            try:
                self.samples.append(nv.nvmlDeviceGetClockInfo(self.h, nv.NVML_CLOCK_SM))
                r = get_reasons(self.h)
                for bit, name in names.items():
                    if r & bit:
                        self.reasons.add(name)
            except Exception:  # noqa: BLE001
                pass
            time.sleep(self.period)

    def __enter__(self):
        if self.nv is not None:
            self._t = threading.Thread(target=self._loop, daemon=True)
            self._t.start()
        return self

    def __exit__(self, *a):
        self._stop.set()
        if self._t is not None:
            self._t.join()

    def summary(self):
        if not self.samples:
            return {"sm_mhz": None, "sm_max_mhz": self.max_mhz, "reasons": [], "note": "no NVML samples"}
        return {"sm_mhz": int(statistics.median(self.samples)), "sm_max_mhz": self.max_mhz,
                "reasons": sorted(self.reasons), "samples": len(self.samples)}


# ----------------------------------------------------------------------------------------------------
# device-side workload
# ----------------------------------------------------------------------------------------------------
class Workload:
    """`resident` independent copies of the batch (distinct pools, Q, hidden) that the steps rotate over, so
    that no step finds its inputs in L2; W_vocab is shared (model weights)."""

    def __init__(self, spec, device, prepos):
        self.spec, self.dev = spec, device
        s = spec["shape"]
        seed = spec["seed"]
        n = len(spec["n_s"])
        self.n = n
        self.sets = []
        self.w = synth.make_w_vocab(s, seed, device)
        self.fast = synth.make_fast_set(s, seed)
        self.bitmap = prepos.fastset_build(self.fast, s.V).to(device)
        for r in range(spec["resident"]):
            sb = synth.make_sessions(s, spec["n_s"], spec["l_entry"], seed + 100003 * (r + 1), device)
            hidden, planted, _ = synth.make_hidden(s, n, self.w, self.fast, seed + 100003 * (r + 1))
            self.sets.append(dict(sb=sb, hidden=hidden, planted=planted,
                                  out=torch.zeros(sb.q.shape, dtype=torch.bfloat16, device=device)))
        self.n_s_h = torch.tensor(spec["n_s"], dtype=torch.int32)
        self.l_h = torch.tensor(spec["l_entry"], dtype=torch.int32)
        self.cap_h = torch.tensor(self.sets[0]["sb"].capacity, dtype=torch.int32)
        self.sid = torch.arange(n, dtype=torch.int32, device=device)
        self.records = prepos.new_records(n, device)
        self.version = torch.zeros(n, dtype=torch.int64, device=device)
        self.position = torch.tensor([a + b for a, b in zip(spec["n_s"], spec["l_entry"])], dtype=torch.int64, device=device)
        self.req = synth.serve_requests(spec["serves"], n, seed).to(device)
        self.dec = torch.zeros(spec["serves"], dtype=torch.int32, device=device)
        self.tok = torch.zeros(spec["serves"], dtype=torch.int32, device=device)
        self.ctx = prepos.Context(s.layers, s.Hq, s.Hkv, s.d, s.H, s.V, s.page, max_sessions=n)
        # rows of `hidden` fed to the LM head: the last entry position of each session (reading Q7)

    def step(self, i, ev=None):
        st = self.sets[i % len(self.sets)]
        sb, ctx = st["sb"], self.ctx
        if ev:
            ev[0].record()
        ctx.invalidate(self.sid, self.version, self.records)
        if ev:
            ev[1].record()
        ctx.entry_attn(sb.q, sb.k_new, sb.v_new, sb.k_pool, sb.v_pool, sb.page_table, self.n_s_h, self.l_h, self.cap_h,
                       st["out"])
        if ev:
            ev[2].record()
        ctx.ready_dist(self.sid, st["hidden"], self.w, self.records, self.version, position_p=self.position)
        if ev:
            ev[3].record()
        ctx.gate_serve(self.req, self.records, self.version, self.bitmap, self.spec["shape"].tau, self.dec, self.tok)
        if ev:
            ev[4].record()


def run_device_timed(wl, steps, warmup, dist_ctx):
    """K steps with inputs resident in HBM, timed with CUDA events on the launch stream.

    Pass A (the reported `value`): the K steps back to back with one event before the first and one after the
    last call -- nothing between the four calls of a step, so that each kernel's prologue may overlap its
    predecessor's tail (programmatic dependent launch) exactly as in a caller's stream.  With an L2 flush between
    steps (c1) the events bracket each step instead and the flushes stay outside.
    Pass B (the per-kernel breakdown and the roofline): the same K steps again with an event between the calls;
    a kernel's duration is the mean over those K launches."""
    flush = torch.empty(2 * L2_BYTES, dtype=torch.uint8, device=wl.dev) if wl.spec["flush_l2"] else None
    for i in range(warmup):
        wl.step(i)
    torch.cuda.synchronize()
    launches0 = wl.ctx.launch_count()
    dist_ctx.barrier()
    torch.cuda.synchronize()
    t_wall0 = time.perf_counter()
    with ClockSampler(torch.cuda.current_device()) as clk:
        if flush is None:
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record()
            for i in range(steps):
                wl.step(warmup + i)
            e1.record()
            torch.cuda.synchronize()
            total_ms = e0.elapsed_time(e1)
            per_step = [total_ms / steps] * steps
        else:
            ev = [[torch.cuda.Event(enable_timing=True) for _ in range(2)] for _ in range(steps)]
            for i in range(steps):
                flush.fill_(i & 0xFF)  # evict L2 between timed iterations (outside the per-step events)
                ev[i][0].record()
                wl.step(warmup + i)
                ev[i][1].record()
            torch.cuda.synchronize()
            per_step = [a.elapsed_time(b) for a, b in ev]
            total_ms = sum(per_step)
    dist_ctx.barrier()
    wall = time.perf_counter() - t_wall0
    launches = wl.ctx.launch_count() - launches0
    # pass B: per-call events (after half a second of idle: the long HBM- and tensor-bound steps of pass A leave the
    # board at its power cap, and a kernel timed between two events is meant to be the kernel alone)
    time.sleep(0.5)
    evs = [[torch.cuda.Event(enable_timing=True) for _ in range(5)] for _ in range(steps)]
    with ClockSampler(torch.cuda.current_device()) as clk_b:
        for i in range(steps):
            if flush is not None:
                flush.fill_(i & 0xFF)
            wl.step(warmup + steps + i, evs[i])
        torch.cuda.synchronize()
    spans = (("invalidate", 0, 1), ("entry_attn", 1, 2), ("ready_dist", 2, 3), ("gate_serve", 3, 4))
    calls = {name: statistics.fmean(e[a].elapsed_time(e[b]) for e in evs) for name, a, b in spans}
    calls_median = {name: statistics.median(e[a].elapsed_time(e[b]) for e in evs) for name, a, b in spans}
    calls_min = {name: min(e[a].elapsed_time(e[b]) for e in evs) for name, a, b in spans}
    return dict(total_ms=total_ms, per_step=per_step, calls=calls, calls_median=calls_median, calls_min=calls_min,
                launches=launches, wall_s=wall, clocks=clk.summary(), clocks_per_call_pass=clk_b.summary())


def run_e2e(wl, steps, warmup, dist_ctx):
    """Same step through the public binding with HOST inputs: every step copies that step's Q/K_new/V_new,
    hidden and request ids from pinned host memory and reads back the attention output, the records and the
    decisions.  The copies run on their own streams, chained to the step by events (H2D(i) -> step(i) -> D2H(i)),
    so the transfers of neighbouring steps overlap the kernels as a serving loop would arrange it; the host waits
    for the results of step i - 2 before it issues step i (at most two steps in flight)."""
    R = len(wl.sets)
    host = []
    for st in wl.sets:
        sb = st["sb"]
        h = {k: getattr(sb, k).cpu().pin_memory() for k in ("q", "k_new", "v_new")}
        h["hidden"] = st["hidden"].cpu().pin_memory()
        h["out"] = torch.empty(sb.q.shape, dtype=torch.bfloat16).pin_memory()
        h["rec"] = torch.empty(wl.records.shape, dtype=torch.uint8).pin_memory()
        h["dec"] = torch.empty(wl.dec.shape, dtype=torch.int32).pin_memory()
        h["tok"] = torch.empty(wl.tok.shape, dtype=torch.int32).pin_memory()
        host.append(h)
    req_h = wl.req.cpu().pin_memory()
    h0 = host[0]
    h2d = sum(h0[k].numel() * h0[k].element_size() for k in ("q", "k_new", "v_new", "hidden")) + req_h.numel() * 4
    d2h = sum(h0[k].numel() * h0[k].element_size() for k in ("out", "rec", "dec", "tok"))
    cur = torch.cuda.current_stream()
    s_in, s_out = torch.cuda.Stream(), torch.cuda.Stream()
    step_done = [None] * R      # per resident set: the step that last used its device buffers
    out_read = [None] * R       # per resident set: its attention output has been copied out
    small_read = [None]         # records / decisions of the previous step have been copied out
    prev_step = [None]
    results = []                # per step: the event after its last D2H

    def one(i):
        k = i % R
        st, h = wl.sets[k], host[k]
        sb = st["sb"]
        if len(results) >= 2:
            results[-2].synchronize()           # the caller consumes the result of step i - 2
        with torch.cuda.stream(s_in):
            if step_done[k] is not None:
                s_in.wait_event(step_done[k])   # the set's inputs are no longer being read
            sb.q.copy_(h["q"], non_blocking=True)
            sb.k_new.copy_(h["k_new"], non_blocking=True)
            sb.v_new.copy_(h["v_new"], non_blocking=True)
            st["hidden"].copy_(h["hidden"], non_blocking=True)
            if prev_step[0] is not None:
                s_in.wait_event(prev_step[0])   # the shared request buffer is free
            wl.req.copy_(req_h, non_blocking=True)
            e_in = torch.cuda.Event()
            e_in.record(s_in)
        cur.wait_event(e_in)
        if out_read[k] is not None:
            cur.wait_event(out_read[k])         # the set's output buffer has been read
        if small_read[0] is not None:
            cur.wait_event(small_read[0])       # the shared records / decisions have been read
        wl.step(i)
        e_step = torch.cuda.Event()
        e_step.record(cur)
        step_done[k] = e_step
        prev_step[0] = e_step
        with torch.cuda.stream(s_out):
            s_out.wait_event(e_step)
            h["rec"].copy_(wl.records, non_blocking=True)
            h["dec"].copy_(wl.dec, non_blocking=True)
            h["tok"].copy_(wl.tok, non_blocking=True)
            e_small = torch.cuda.Event()
            e_small.record(s_out)
            small_read[0] = e_small
            h["out"].copy_(st["out"], non_blocking=True)
            e_out = torch.cuda.Event()
            e_out.record(s_out)
            out_read[k] = e_out
        results.append(e_out)

    for i in range(warmup):
        one(i)
    torch.cuda.synchronize()
    dist_ctx.barrier()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record(cur)
    for i in range(steps):
        one(warmup + i)
    cur.wait_event(results[-1])     # the last step's results are on the host
    e1.record(cur)
    torch.cuda.synchronize()
    dist_ctx.barrier()
    return dict(ms_per_step=e0.elapsed_time(e1) / steps, h2d=h2d, d2h=d2h)


def run_gate_serve(wl, prepos, reps=200):
    """prepos_gate_serve alone over a 64-record table (config 4's serve side): device time per call, and wall
    time per call including the D2H of the decisions into pinned memory + sync, for B = 1, 64, 4096."""
    dev, s = wl.dev, wl.spec["shape"]
    n_sess = 64
    ctx = prepos.Context(s.layers, s.Hq, s.Hkv, s.d, s.H, s.V, s.page, max_sessions=n_sess)
    sid = torch.arange(n_sess, dtype=torch.int32, device=dev)
    recs = prepos.new_records(n_sess, dev)
    ver = torch.zeros(n_sess, dtype=torch.int64, device=dev)
    hidden, _, _ = synth.make_hidden(s, n_sess, wl.w, wl.fast, wl.spec["seed"] + 9)
    ctx.ready_dist(sid, hidden, wl.w, recs, ver)
    res = {}
    for B in (1, 64, 4096):
        req = synth.serve_requests(B, n_sess, wl.spec["seed"] + B).to(dev)
        # decisions and tokens in one device buffer and one pinned host buffer: a serve is answered with ONE D2H copy
        both = torch.zeros((2, B), dtype=torch.int32, device=dev)
        dec, tok = both[0], both[1]
        both_h = torch.empty((2, B), dtype=torch.int32).pin_memory()
        dec_h = both_h[0]
        for _ in range(10):
            ctx.gate_serve(req, recs, ver, wl.bitmap, s.tau, dec, tok)
        torch.cuda.synchronize()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        for _ in range(reps):
            ctx.gate_serve(req, recs, ver, wl.bitmap, s.tau, dec, tok)
        e1.record()
        torch.cuda.synchronize()
        dev_us = e0.elapsed_time(e1) * 1e3 / reps
        walls = []
        for _ in range(reps):
            t0 = time.perf_counter()
            ctx.gate_serve(req, recs, ver, wl.bitmap, s.tau, dec, tok)
            both_h.copy_(both, non_blocking=True)
            torch.cuda.synchronize()
            walls.append((time.perf_counter() - t0) * 1e6)
        # the same serve with the decisions written straight into pinned host memory (the outputs are plain pointers:
        # pinned memory is device-addressable), so a serve is ONE launch + one sync, no copy call
        zc = torch.zeros((2, B), dtype=torch.int32).pin_memory()
        walls_zc = []
        for _ in range(reps):
            t0 = time.perf_counter()
            ctx.gate_serve(req, recs, ver, wl.bitmap, s.tau, zc[0], zc[1])
            torch.cuda.synchronize()
            walls_zc.append((time.perf_counter() - t0) * 1e6)
        assert torch.equal(zc, both_h), "zero-copy serve disagrees with the copied one"
        res[f"B{B}"] = {"device_us_per_call": round(dev_us, 3), "device_us_per_serve": round(dev_us / B, 5),
                        "wall_us_per_call_p50": round(statistics.median(walls), 2),
                        "wall_us_per_serve_p50": round(statistics.median(walls) / B, 5),
                        "wall_us_per_call_pinned_out_p50": round(statistics.median(walls_zc), 2),
                        "served": int((dec_h == 0).sum())}
    ctx.close()
    return res


def run_co_schedule(wl, prepos, n_serves=300):
    """SURVEY.md 8(f) NEXT-2 (the pass runs in the idle window and "yields to any request"):
    wall latency of one gate serve (launch on a high-priority stream + D2H of the decisions + sync) while the
    low-priority stream is kept full of pre-position steps, beside the same serve on an idle GPU.  The persistent
    kernels leave room for one small CTA per SM, so the serve does not wait for a pre-position to finish."""
    dev, s = wl.dev, wl.spec["shape"]
    s_lo, s_hi = torch.cuda.Stream(priority=0), torch.cuda.Stream(priority=-1)
    n = 64
    ctx2 = prepos.Context(s.layers, s.Hq, s.Hkv, s.d, s.H, s.V, s.page, max_sessions=n)
    sid = torch.arange(n, dtype=torch.int32, device=dev)
    recs = prepos.new_records(n, dev)
    ver = torch.zeros(n, dtype=torch.int64, device=dev)
    hidden, _, _ = synth.make_hidden(s, n, wl.w, wl.fast, wl.spec["seed"] + 9)
    ctx2.ready_dist(sid, hidden, wl.w, recs, ver)
    torch.cuda.synchronize()
    req = synth.serve_requests(n, n, wl.spec["seed"] + 3).to(dev)
    dec = torch.zeros(n, dtype=torch.int32, device=dev)
    tok = torch.zeros(n, dtype=torch.int32, device=dev)
    dec_h = torch.empty(n, dtype=torch.int32).pin_memory()

    def serve_once():
        t0 = time.perf_counter()
        with torch.cuda.stream(s_hi):
            ctx2.gate_serve(req, recs, ver, wl.bitmap, s.tau, dec, tok)
            dec_h.copy_(dec, non_blocking=True)
        s_hi.synchronize()
        return (time.perf_counter() - t0) * 1e6

    for _ in range(20):
        serve_once()
    idle = sorted(serve_once() for _ in range(n_serves))
    # the low-priority stream gets ~15 ms of pre-position steps in one go (no second host thread competing for the
    # interpreter), and the serves are issued for as long as that work is running
    t0 = time.perf_counter()
    wl.step(0)
    torch.cuda.synchronize()
    per_step = max(time.perf_counter() - t0, 1e-4)
    n_bg = max(4, min(400, int(0.015 / per_step)))
    busy, i, rounds = [], 0, 0
    while len(busy) < n_serves and rounds < 200:
        rounds += 1
        end = torch.cuda.Event()
        with torch.cuda.stream(s_lo):
            for _ in range(n_bg):
                wl.step(i)
                i += 1
            end.record(s_lo)
        while not end.query() and len(busy) < n_serves:
            v = serve_once()
            if not end.query():          # the pre-position was still running when the serve returned
                busy.append(v)
        torch.cuda.synchronize()
    ctx2.close()
    busy.sort()
    q = lambda v, p: round(v[min(len(v) - 1, int(len(v) * p))], 1) if v else None
    # A request that needs whole SMs -- the fall-through decode step of one session (L = 1, all layers) -- has to wait
    # for pre-position CTAs to retire.  The caller bounds that wait by issuing the pre-position in layer chunks
    # (`layer_begin/layer_end`): measured for one launch per step and for chunks of layers / 8.
    decode = {}
    if wl.n_s_h.numel() >= 1 and s.layers >= 8:
        sb0 = wl.sets[0]["sb"]
        ctx3 = prepos.Context(s.layers, s.Hq, s.Hkv, s.d, s.H, s.V, s.page, max_sessions=1)
        q1 = sb0.q[:, :1].contiguous()
        k1, v1 = sb0.k_new[:, :1].contiguous(), sb0.v_new[:, :1].contiguous()
        o1 = torch.empty_like(q1)
        ns1, l1, cap1 = wl.n_s_h[:1].clone(), torch.ones(1, dtype=torch.int32), wl.cap_h[:1].clone()

        def decode_once():
            t0 = time.perf_counter()
            with torch.cuda.stream(s_hi):
                ctx3.entry_attn(q1, k1, v1, sb0.k_pool, sb0.v_pool, sb0.page_table[:1], ns1, l1, cap1, o1)
            s_hi.synchronize()
            return (time.perf_counter() - t0) * 1e6

        def step_chunked(i, chunk):
            st = wl.sets[i % len(wl.sets)]
            sb = st["sb"]
            wl.ctx.invalidate(wl.sid, wl.version, wl.records)
            for l0 in range(0, s.layers, chunk):
                wl.ctx.entry_attn(sb.q, sb.k_new, sb.v_new, sb.k_pool, sb.v_pool, sb.page_table, wl.n_s_h, wl.l_h, wl.cap_h,
                                  st["out"], layer_begin=l0, layer_end=min(s.layers, l0 + chunk))
            wl.ctx.ready_dist(wl.sid, st["hidden"], wl.w, wl.records, wl.version, position_p=wl.position)
            wl.ctx.gate_serve(wl.req, wl.records, wl.version, wl.bitmap, s.tau, wl.dec, wl.tok)

        for _ in range(5):
            decode_once()
        d_idle = sorted(decode_once() for _ in range(40))
        decode["idle_wall_us_p50"] = q(d_idle, 0.5)
        for label, chunk in (("one_launch", s.layers), ("layer_chunks_of_%d" % (s.layers // 8), s.layers // 8)):
            got, i, rounds = [], 0, 0
            while len(got) < 40 and rounds < 100:
                rounds += 1
                end = torch.cuda.Event()
                with torch.cuda.stream(s_lo):
                    for _ in range(n_bg):
                        step_chunked(i, chunk)
                        i += 1
                    end.record(s_lo)
                while not end.query() and len(got) < 40:
                    v = decode_once()
                    if not end.query():
                        got.append(v)
                torch.cuda.synchronize()
            got.sort()
            decode["during_preposition_" + label] = {"p50": q(got, 0.5), "p90": q(got, 0.9), "samples": len(got)}
        ctx3.close()
    # (a launch-bound workload such as c1 never gets ahead of the host: no serve falls inside a running step)
    return {"requests_per_serve": n, "idle_wall_us": {"p50": q(idle, 0.5), "p99": q(idle, 0.99)},
            "during_preposition_wall_us": {"p50": q(busy, 0.5), "p90": q(busy, 0.9), "p99": q(busy, 0.99),
                                           "samples": len(busy)},
            "decode_step_wall_us": decode}


def run_layer_sequential(wl, reps=10):
    """SURVEY.md 8(d) schedule (S): the attention of the step as one launch PER LAYER (what an engine whose layer
    l + 1 queries depend on layer l must issue; the timed step uses schedule (F), all layers in one launch, valid
    for the synthetic where per-layer Q/K/V are pre-drawn).  Same kernel, `layer_begin = l, layer_end = l + 1`.
    Timed twice: the calls issued one by one from Python (host-bound: ~19 us per call), and the same launches
    captured once into a CUDA graph and replayed (what the device needs: programmatic dependent launch overlaps
    the prologues, units spread over many CTAs take the cooperative merge)."""
    s = wl.spec["shape"]
    ab = algorithmic_bytes(wl.spec)["entry_attn"]

    def issue(st):
        sb = st["sb"]
        for l in range(s.layers):
            wl.ctx.entry_attn(sb.q, sb.k_new, sb.v_new, sb.k_pool, sb.v_pool, sb.page_table, wl.n_s_h, wl.l_h, wl.cap_h,
                              st["out"], layer_begin=l, layer_end=l + 1)

    def timed(fn):
        ev = []
        for i in range(reps + 2):
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record()
            fn(i)
            e1.record()
            ev.append((e0, e1))
        torch.cuda.synchronize()
        return statistics.fmean(a.elapsed_time(b) for a, b in ev[2:])

    ms = timed(lambda i: issue(wl.sets[i % len(wl.sets)]))
    out = {"launches": s.layers, "attn_ms": round(ms, 5), "achieved_gbs": round(ab / (ms * 1e-3) / 1e9, 1),
           "frac_of_measured_hbm": round(ab / (ms * 1e-3) / 1e9 / peaks()["hbm"], 4)}
    try:
        graphs = []
        side = torch.cuda.Stream()
        for st in wl.sets:
            g = torch.cuda.CUDAGraph()
            side.wait_stream(torch.cuda.current_stream())
            with torch.cuda.graph(g, stream=side):
                issue(st)
            graphs.append(g)
        torch.cuda.current_stream().wait_stream(side)
        gms = timed(lambda i: graphs[i % len(graphs)].replay())
        out["graph_replay"] = {"attn_ms": round(gms, 5), "achieved_gbs": round(ab / (gms * 1e-3) / 1e9, 1),
                               "frac_of_measured_hbm": round(ab / (gms * 1e-3) / 1e9 / peaks()["hbm"], 4)}
        # the same graph with prepos_ctx_set_kv_prefetch: a layer's launch requests its cached K/V tiles while the previous
        # layer's merge is still running (legal between the layers of one pass: layer l appends to layer l's pages only)
        wl.ctx.set_kv_prefetch(True)
        graphs2 = []
        for st in wl.sets:
            g = torch.cuda.CUDAGraph()
            side.wait_stream(torch.cuda.current_stream())
            with torch.cuda.graph(g, stream=side):
                issue(st)
            graphs2.append(g)
        torch.cuda.current_stream().wait_stream(side)
        gms2 = timed(lambda i: graphs2[i % len(graphs2)].replay())
        wl.ctx.set_kv_prefetch(False)
        out["graph_replay_kv_prefetch"] = {"attn_ms": round(gms2, 5), "achieved_gbs": round(ab / (gms2 * 1e-3) / 1e9, 1),
                                           "frac_of_measured_hbm": round(ab / (gms2 * 1e-3) / 1e9 / peaks()["hbm"], 4)}
    except Exception as e:  # capture is a convenience of this measurement, not part of the path
        out["graph_replay"] = {"unavailable": str(e)[:120]}
        wl.ctx.set_kv_prefetch(False)
        torch.cuda.synchronize()
    return out


def run_fall_through(wl, reps=20):
    """SURVEY.md 8(f) NEXT-1, the step after a gate miss (Eq. 5): prepos_entry_attn with a delta of
    8 tokens, and with the single decode token, over the same cached sessions (all layers, one launch each).
    G * L is 32 / 4 rows per KV head here: the streaming-HBM regime of the same kernel."""
    res = {}
    ab = algorithmic_bytes(wl.spec)
    s = wl.spec["shape"]
    kv_bytes = sum(wl.spec["n_s"]) * s.layers * s.Hkv * s.d * 2 * 2
    for L in (8, 1):
        if min(wl.spec["l_entry"]) < L or wl.n != 1:
            continue
        l_h = [L] * wl.n
        ev = []
        for i in range(reps + 3):
            st = wl.sets[i % len(wl.sets)]
            sb = st["sb"]
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record()
            wl.ctx.entry_attn(sb.q[:, :L], sb.k_new[:, :L], sb.v_new[:, :L], sb.k_pool, sb.v_pool, sb.page_table,
                              wl.n_s_h, l_h, wl.cap_h, st["out"][:, :L])
            e1.record()
            ev.append((e0, e1))
        torch.cuda.synchronize()
        ms = statistics.fmean(a.elapsed_time(b) for a, b in ev[3:])
        res[f"L{L}"] = {"attn_ms": round(ms, 5), "kv_gbs": round(kv_bytes / (ms * 1e-3) / 1e9, 1),
                        "frac_of_measured_hbm": round(kv_bytes / (ms * 1e-3) / 1e9 / peaks()["hbm"], 4)}
    return res


# ----------------------------------------------------------------------------------------------------
# the CPU oracle, timed on a bounded sample (cpu_baseline leg and --impl reference)
# ----------------------------------------------------------------------------------------------------
class OracleSample:
    """Holds host copies of ONE session of the workload and times the oracle, as it stands, on a sample of it:
    `units` (layer, kv head) slices of the entry attention and `rows` vocabulary rows of the LM head, plus the
    record and one gate decision; the per-session figure scales each part to the full session."""

    def __init__(self, spec):
        from oracle import oracle as o
        self.o = o
        o.lib()
        self.spec = spec
        s = spec["shape"]
        self.s = s
        seed = spec["seed"] + 100003
        # one session, a few layers are enough for any sample the budget allows
        self.max_layers = min(s.layers, 2)
        sb = synth.make_sessions(s, spec["n_s"][:1], spec["l_entry"][:1], seed, "cpu", layers=self.max_layers)
        self.sb = sb
        self.bits = lambda t: t.contiguous().view(torch.int16).numpy().view(np.uint16)
        self.w = self.bits(synth.make_w_vocab(s, spec["seed"], "cpu"))
        self.fast = synth.make_fast_set(s, spec["seed"])
        g = synth.gen(seed + 5, "cpu")
        self.x = self.bits(synth.randn_bf16((s.H,), g))
        self.bitmap = o.fastset_bitmap(self.fast.numpy(), s.V)
        self.total_units = s.layers * s.Hkv
        self.cores = o.num_threads()

    def attn_unit(self, u):
        s, sb = self.s, self.sb
        layer, g = (u // s.Hkv) % self.max_layers, u % s.Hkv
        G = s.G
        kp = self.bits(sb.k_pool[layer][:, g:g + 1]).copy()
        vp = self.bits(sb.v_pool[layer][:, g:g + 1]).copy()
        t0 = time.perf_counter()
        self.o.entry_attn(self.bits(sb.q[layer][:, g * G:(g + 1) * G]), self.bits(sb.k_new[layer][:, g:g + 1]),
                          self.bits(sb.v_new[layer][:, g:g + 1]), kp, vp, sb.page_table[0].numpy(), sb.n_s[0],
                          sb.capacity[0])
        return time.perf_counter() - t0

    def vocab(self, rows):
        t0 = time.perf_counter()
        lg = self.o.logits(self.w[:rows], self.x)
        rec = self.o.record(lg)
        self.o.gate(rec.gap, rec.top1, True, rec.nonfinite, 1, 1, 0, 0, self.bitmap, self.s.V, self.s.tau)
        return time.perf_counter() - t0

    def plan(self, budget_s):
        """Calibrates on one attention unit and 8192 vocabulary rows, then sizes the sample to the budget."""
        t_u = self.attn_unit(0)
        r0 = min(8192, self.s.V)
        t_r = self.vocab(r0) / r0
        units = max(1, min(self.total_units, int(0.7 * budget_s / max(t_u, 1e-9))))
        rows = max(min(1024, self.s.V), min(self.s.V, int(0.3 * budget_s / max(t_r, 1e-12))))
        return units, rows

    def run(self, units, rows):
        """One sampled step -> estimated seconds for one full session."""
        ta = sum(self.attn_unit(u) for u in range(units))
        tv = self.vocab(rows)
        full = ta * self.total_units / units + tv * self.s.V / rows
        return full, ta + tv

    def describe(self, units, rows):
        return (f"{units} of {self.total_units} (layer, kv-head) attention slices + {rows} of {self.s.V} vocabulary rows "
                f"of one session, each part scaled to the full session; oracle as it stands (C, fp64, OpenMP)")


# ----------------------------------------------------------------------------------------------------
class Dist:
    def __init__(self, gpus):
        self.world = int(os.environ.get("WORLD_SIZE", "1"))
        self.rank = int(os.environ.get("RANK", "0"))
        self.local_rank = int(os.environ.get("LOCAL_RANK", "0"))
        self.on = self.world > 1
        if self.on:
            import torch.distributed as dist
            self.dist = dist
            os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
            os.environ.setdefault("MASTER_PORT", "29511")

    def init(self, backend):
        if self.on:
            self.dist.init_process_group(backend=backend)

    def barrier(self):
        if self.on:
            self.dist.barrier()

    def max(self, v, device):
        if not self.on:
            return v
        t = torch.tensor([v], dtype=torch.float64, device=device)
        self.dist.all_reduce(t, op=self.dist.ReduceOp.MAX)
        return float(t[0])

    def close(self):
        if self.on:
            self.dist.destroy_process_group()


def run_graph_replay(wl, replays=24):
    """SURVEY.md 8(d) timing protocol: the whole per-session pass (the four calls of a step) captured once per resident
    set into a CUDA graph and replayed, CUDA events around every replay: median and min over `replays` (>= 20).
    c1 flushes L2 before every replay."""
    flush = torch.empty(2 * L2_BYTES, dtype=torch.uint8, device=wl.dev) if wl.spec["flush_l2"] else None
    try:
        graphs = []
        side = torch.cuda.Stream()
        for k in range(len(wl.sets)):
            g = torch.cuda.CUDAGraph()
            side.wait_stream(torch.cuda.current_stream())
            with torch.cuda.graph(g, stream=side):
                wl.step(k)
            graphs.append(g)
        torch.cuda.current_stream().wait_stream(side)
        ev = []
        for i in range(replays + 3):
            if flush is not None:
                flush.fill_(i & 0xFF)
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record()
            graphs[i % len(graphs)].replay()
            e1.record()
            ev.append((e0, e1))
        torch.cuda.synchronize()
        us = sorted(a.elapsed_time(b) * 1e3 / wl.n for a, b in ev[3:])
        return {"replays": replays, "median_us_per_session": round(statistics.median(us), 3),
                "min_us_per_session": round(us[0], 3), "max_us_per_session": round(us[-1], 3)}
    except Exception as e:  # noqa: BLE001  (capture is a convenience of this measurement, not part of the path)
        torch.cuda.synchronize()
        return {"unavailable": str(e)[:160]}


def run_scan_logits(wl, prepos, reps=50):
    """a4' -- the paper's serve-time vocabulary scan T_scan(V) (Eq. 3; 0.664 ms derived on its host,
    PAPER.md:276): prepos_scan_logits over stored fp32 logits, n = 1 and n = 64 rows.  Device time per call with
    the logits L2-resident (back-to-back calls) and after an L2 flush (the logits come from HBM), and wall time of
    call + D2H of the record(s) into pinned memory + sync."""
    dev, s = wl.dev, wl.spec["shape"]
    res = {}
    flush = torch.empty(2 * L2_BYTES, dtype=torch.uint8, device=dev)
    for n in (1, 64):
        ctx = prepos.Context(s.layers, s.Hq, s.Hkv, s.d, s.H, s.V, s.page, max_sessions=n)
        lg = torch.randn((n, s.V), generator=synth.gen(wl.spec["seed"] + 31 + n, dev), device=dev, dtype=torch.float32)
        recs = prepos.new_records(n, dev)
        rec_h = torch.empty(recs.shape, dtype=torch.uint8).pin_memory()
        for _ in range(5):
            ctx.scan_logits(lg, recs)
        torch.cuda.synchronize()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        for _ in range(reps):
            ctx.scan_logits(lg, recs)
        e1.record()
        torch.cuda.synchronize()
        warm = e0.elapsed_time(e1) * 1e3 / reps
        cold = []
        for i in range(10):
            flush.fill_(i)
            a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            a.record()
            ctx.scan_logits(lg, recs)
            b.record()
            torch.cuda.synchronize()
            cold.append(a.elapsed_time(b) * 1e3)
        walls = []
        for _ in range(reps):
            t0 = time.perf_counter()
            ctx.scan_logits(lg, recs)
            rec_h.copy_(recs, non_blocking=True)
            torch.cuda.synchronize()
            walls.append((time.perf_counter() - t0) * 1e6)
        nbytes = n * s.V * 4
        res[f"n{n}"] = {"logit_bytes": nbytes, "device_us_l2_resident": round(warm, 2),
                        "device_us_from_hbm_median": round(statistics.median(cold), 2),
                        "hbm_gbs_from_hbm": round(nbytes / (statistics.median(cold) * 1e-6) / 1e9, 1),
                        "wall_us_call_d2h_sync_p50": round(statistics.median(walls), 2)}
        ctx.close()
    return res


def run_ready_dist_w4(wl, prepos, reps=30):
    """SURVEY.md 8(f) NEXT-4 (the paper's headline model "runs at 4-bit precision"; format per
    DESIGN.md reading Q21): prepos_ready_dist_w4 -- the same record from int4 codes + one bf16 scale per (row, 128 k)
    -- beside the bf16 call it replaces.  Algorithmic bytes: V*H/2 codes + V*H/64 scale bytes + the hidden rows, read
    ONCE (a batch of more than 8 rows takes ceil(n / 8) passes over the codes: `passes_over_codes`; the extra reads are
    the kernel's, not the algorithm's, and count against `frac_of_measured_hbm`).  Rotates over two copies of the codes
    (each is larger than L2)."""
    dev, s = wl.dev, wl.spec["shape"]
    n = min(wl.n, 64)   # config 4: its whole 64-session batch, which this kernel serves in ceil(n / 8) passes over the codes
    sets = [synth.make_w_vocab_w4(s, wl.spec["seed"] + 11 * r, dev) for r in range(2)]
    hidden = wl.sets[0]["hidden"][:n].contiguous()
    sid = torch.arange(n, dtype=torch.int32, device=dev)
    recs = prepos.new_records(n, dev)
    ver = torch.zeros(n, dtype=torch.int64, device=dev)
    ctx = prepos.Context(s.layers, s.Hq, s.Hkv, s.d, s.H, s.V, s.page, max_sessions=n)
    ev = []
    for i in range(reps + 5):
        w4, sc = sets[i % 2]
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a.record()
        ctx.ready_dist_w4(sid, hidden, w4, sc, recs, ver)
        b.record()
        ev.append((a, b))
    torch.cuda.synchronize()
    ms = sorted(a.elapsed_time(b) for a, b in ev[5:])
    ctx.close()
    nbytes = s.V * s.H // 2 + s.V * (s.H // 128) * 2 + n * s.H * 2 + n * 48
    med = statistics.median(ms)
    return {"rows": n, "passes_over_codes": (n + 7) // 8, "ms_median": round(med, 5), "ms_min": round(ms[0], 5),
            "algorithmic_bytes": nbytes,
            "achieved_gbs": round(nbytes / (med * 1e-3) / 1e9, 1),
            "frac_of_measured_hbm": round(nbytes / (med * 1e-3) / 1e9 / peaks()["hbm"], 4),
            "bf16_call_algorithmic_bytes": s.V * s.H * 2 + n * s.H * 2 + n * 48}


def run_attn_fp8(wl, prepos, reps=12):
    """prepos_entry_attn_fp8 -- the same pass over an e4m3 KV cache (reading Q20: one
    fp32 scale per (layer, page, kv head)), all layers in one launch, on the workload's sessions quantised in place of
    their bf16 pools.  Algorithmic bytes: every cached code once (half the bf16 bytes) + the page scales + Q / O +
    the entry K/V read and their codes written."""
    s, spec = wl.spec["shape"], wl.spec
    chunk = max(64, (1 << 28) // (s.layers * s.Hkv * s.page * s.d))   # <= 1 GiB of fp32 per quantiser chunk
    n_sets = 1 if wl.n > 8 else 2   # config 4's pools are far larger than L2 on their own (and 23 GB per quantised copy)
    reps = 4 if wl.n > 8 else reps
    sets = [synth.quantise_sessions_fp8(st["sb"], chunk_pages=chunk) for st in wl.sets[:n_sets]]
    ctx = prepos.Context(s.layers, s.Hq, s.Hkv, s.d, s.H, s.V, s.page, max_sessions=wl.n)
    ev = []
    for i in range(reps + 3):
        fb, st = sets[i % len(sets)], wl.sets[i % len(sets)]
        sb = fb.base
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a.record()
        ctx.entry_attn_fp8(sb.q, sb.k_new, sb.v_new, fb.k_pool8, fb.v_pool8, fb.k_scale, fb.v_scale, sb.page_table,
                           wl.n_s_h, wl.l_h, wl.cap_h, st["out"])
        b.record()
        ev.append((a, b))
    torch.cuda.synchronize()
    ms = sorted(a.elapsed_time(b) for a, b in ev[3:])
    ctx.close()
    sum_l, sum_n = sum(spec["l_entry"]), sum(spec["n_s"])
    n_pages_used = sum(-(-(a + b) // s.page) for a, b in zip(spec["n_s"], spec["l_entry"]))
    nbytes = (sum_n * s.layers * s.Hkv * s.d * 2                    # K and V codes, one byte each
              + n_pages_used * s.layers * s.Hkv * 4 * 2             # page scales
              + sum_l * s.layers * s.Hq * s.d * 2 * 2               # Q read, O written
              + sum_l * s.layers * s.Hkv * s.d * 2 * (2 + 1 + 1))   # entry K/V read (bf16), codes written and read back
    med = statistics.median(ms)
    fl = attention_flops(spec)
    return {"ms_median": round(med, 5), "ms_min": round(ms[0], 5), "algorithmic_bytes": nbytes,
            "achieved_gbs": round(nbytes / (med * 1e-3) / 1e9, 1),
            "frac_of_measured_hbm": round(nbytes / (med * 1e-3) / 1e9 / peaks()["hbm"], 4),
            "tflops": round(fl / (med * 1e-3) / 1e12, 1),
            "bf16_call_algorithmic_bytes": algorithmic_bytes(spec)["entry_attn"]}


def run_yield(wl, prepos, trials=40):
    """SURVEY.md 8(f) NEXT-2, the request that needs whole SMs ("yields immediately"; Eq. 5 / Eq. 7): the
    fall-through decode step of one session (L = 1, all layers, its own ctx) issued on a high-priority stream while the
    pre-position's attention pass (ONE launch, all layers: no caller-side layer chopping) runs on the low-priority
    stream.  The request first calls prepos_ctx_request_yield: the pass stops at its next segment boundaries, the
    decode step takes the SMs, and prepos_entry_attn_resume finishes the pass afterwards.  Reported: wall time of the
    decode step idle / behind the un-yielded pass / with the yield; and what the yield costs the pass (device time of
    launch + resume against the uninterrupted launch)."""
    dev, s = wl.dev, wl.spec["shape"]
    if s.layers < 8:
        return None
    s_lo, s_hi = torch.cuda.Stream(priority=0), torch.cuda.Stream(priority=-1)
    sb0 = wl.sets[0]["sb"]
    ctx3 = prepos.Context(s.layers, s.Hq, s.Hkv, s.d, s.H, s.V, s.page, max_sessions=1)
    q1 = sb0.q[:, :1].contiguous()
    k1, v1 = sb0.k_new[:, :1].contiguous(), sb0.v_new[:, :1].contiguous()
    o1 = torch.empty_like(q1)
    ns1, l1, cap1 = wl.n_s_h[:1].clone(), torch.ones(1, dtype=torch.int32), wl.cap_h[:1].clone()
    q = lambda v, p: round(v[min(len(v) - 1, int(len(v) * p))], 1) if v else None

    def attn(i):
        st = wl.sets[i % len(wl.sets)]
        sb = st["sb"]
        wl.ctx.entry_attn(sb.q, sb.k_new, sb.v_new, sb.k_pool, sb.v_pool, sb.page_table, wl.n_s_h, wl.l_h, wl.cap_h, st["out"])

    def decode(yield_first):
        t0 = time.perf_counter()
        with torch.cuda.stream(s_hi):
            if yield_first:
                wl.ctx.request_yield()
            ctx3.entry_attn(q1, k1, v1, sb0.k_pool, sb0.v_pool, sb0.page_table[:1], ns1, l1, cap1, o1)
        s_hi.synchronize()
        return (time.perf_counter() - t0) * 1e6

    for _ in range(5):
        decode(False)
    idle = sorted(decode(False) for _ in range(trials))
    # the uninterrupted pass, device time
    ev = []
    for i in range(6):
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        with torch.cuda.stream(s_lo):
            a.record(s_lo)
            attn(i)
            b.record(s_lo)
        ev.append((a, b))
    torch.cuda.synchronize()
    pass_ms = statistics.median(a.elapsed_time(b) for a, b in ev[1:])
    res = {"idle_wall_us_p50": q(idle, 0.5), "pass_ms_uninterrupted": round(pass_ms, 4)}
    rng = np.random.default_rng(wl.spec["seed"])
    for label, use_yield in (("behind_the_pass_no_yield", False), ("with_yield", True)):
        got, cost, caught = [], [], 0
        for i in range(trials):
            a, b, c = (torch.cuda.Event(enable_timing=True) for _ in range(3))
            with torch.cuda.stream(s_lo):
                a.record(s_lo)
                attn(i)
                b.record(s_lo)
            # the request arrives somewhere inside the pass
            time.sleep(float(rng.uniform(0.15, 0.7)) * pass_ms * 1e-3)
            running = not b.query()
            v = decode(use_yield)
            if use_yield:
                with torch.cuda.stream(s_lo):
                    pend = wl.ctx.entry_attn_pending()
                    caught += int(pend)
                    wl.ctx.entry_attn_resume()
                    c.record(s_lo)
            torch.cuda.synchronize()
            if running:
                got.append(v)
                if use_yield:
                    cost.append(a.elapsed_time(c))
        got.sort()
        res[label] = {"p50": q(got, 0.5), "p90": q(got, 0.9), "samples": len(got)}
        if use_yield:
            res[label]["passes_caught_running"] = caught
            if cost:
                # start of the pass to end of its resume, which includes the decode step that ran in between
                res[label]["pass_plus_decode_plus_resume_ms_median"] = round(statistics.median(cost), 4)
    ctx3.close()
    return res


def run_update_trace(wl, prepos, n_steps=1000):
    """BASELINE configs[2]'s trace at the config's real vocabulary shape (reading Q16; "triggered after a
    data update"): per update, with probability 0.3 the state version is bumped (prepos_invalidate); then one gate
    serve; if that serve was refused as stale, the session is re-pre-positioned with the next of 16 hidden rows
    (prepos_ready_dist only: the attention of the update is the step timed above).  Wall time of the whole trace, the
    decisions' counts, and two invariants checked on the spot: every serve right after a bump is STALE, no other is."""
    dev, s = wl.dev, wl.spec["shape"]
    seed = wl.spec["seed"]
    bumps = synth.bump_trace(n_steps, seed)
    pool, _, _ = synth.make_hidden(s, 16, wl.w, wl.fast, seed + 17)
    ctx = prepos.Context(s.layers, s.Hq, s.Hkv, s.d, s.H, s.V, s.page, max_sessions=1)
    recs = prepos.new_records(1, dev)
    ver = torch.zeros(1, dtype=torch.int64, device=dev)
    sid = torch.zeros(1, dtype=torch.int32, device=dev)
    decs = torch.full((n_steps,), -9, dtype=torch.int32, device=dev)
    toks = torch.full((n_steps,), -9, dtype=torch.int32, device=dev)
    exp = torch.arange(0, n_steps + 1, dtype=torch.int64, device=dev)
    ctx.ready_dist(sid, pool[0:1], wl.w, recs, ver, expected_version=exp[0:1])
    torch.cuda.synchronize()
    cur, nb = 0, 0
    t0 = time.perf_counter()
    for t, b in enumerate(bumps):
        if b:
            ctx.invalidate(sid, ver, recs)
            nb += 1
        ctx.gate_serve(sid, recs, ver, wl.bitmap, s.tau, decs[t:t + 1], toks[t:t + 1])
        if b:   # the serve above was refused (stale): pre-position again on the new state
            cur = (cur + 1) % 16
            ctx.ready_dist(sid, pool[cur:cur + 1], wl.w, recs, ver, expected_version=exp[nb:nb + 1])
    torch.cuda.synchronize()
    wall = time.perf_counter() - t0
    d = decs.cpu().tolist()
    stale_ok = all((d[t] == prepos.STALE_OR_INVALID) == bool(b) for t, b in enumerate(bumps))
    ctx.close()
    counts = {name: sum(1 for x in d if x == code) for name, code in
              (("served", 0), ("gap_below_tau", 1), ("not_in_fast_set", 2), ("stale_or_invalid", 3), ("ineligible", 4))}
    return {"updates": n_steps, "bumps": nb, "wall_us_per_update": round(wall * 1e6 / n_steps, 2),
            "ready_dist_calls": nb + 1, "decisions": counts, "stale_iff_bumped": stale_ok,
            "final_version": int(ver[0])}


def run_c2_variants(spec, dev, prepos, steps=40):
    """What the steady-state step of config 2 does not show: (a) a session whose n_s advances by L after every
    pre-position, as a real one does (the host rebuilds and uploads the attention plan on every call); (b) n_s = 4100,
    where the units do not divide evenly over the CTAs and the general stream-K grid runs (cut segments + merges)
    instead of the whole-unit grid of n_s = 4096."""
    s = spec["shape"]
    res = {}
    L = spec["l_entry"][0]
    # (a)
    n0 = spec["n_s"][0]
    sb = synth.make_sessions(s, [n0], [L], spec["seed"] + 5, dev, extra_pages=(steps + 12) * L // s.page + 2)
    ctx = prepos.Context(s.layers, s.Hq, s.Hkv, s.d, s.H, s.V, s.page, max_sessions=1)
    out = torch.empty_like(sb.q)
    for i in range(10):
        ctx.entry_attn(sb.q, sb.k_new, sb.v_new, sb.k_pool, sb.v_pool, sb.page_table, [n0 + i * L], [L], sb.capacity, out)
    torch.cuda.synchronize()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    t0 = time.perf_counter()
    e0.record()
    for i in range(steps):
        ctx.entry_attn(sb.q, sb.k_new, sb.v_new, sb.k_pool, sb.v_pool, sb.page_table, [n0 + (10 + i) * L], [L],
                       sb.capacity, out)
    e1.record()
    torch.cuda.synchronize()
    res["advancing_n_s"] = {"attn_ms_per_call_device": round(e0.elapsed_time(e1) / steps, 5),
                            "attn_ms_per_call_wall": round((time.perf_counter() - t0) * 1e3 / steps, 5),
                            "n_s_from_to": [n0 + 10 * L, n0 + (10 + steps) * L]}
    ctx.close()
    del sb, out
    # (b)
    spec_b = dict(spec, n_s=[4100])
    ab = algorithmic_bytes(spec_b)["entry_attn"]
    sets = [synth.make_sessions(s, [4100], [L], spec["seed"] + 7 + r, dev) for r in range(3)]
    ctx = prepos.Context(s.layers, s.Hq, s.Hkv, s.d, s.H, s.V, s.page, max_sessions=1)
    outs = [torch.empty_like(x.q) for x in sets]
    ev = []
    for i in range(steps + 5):
        sb = sets[i % 3]
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a.record()
        ctx.entry_attn(sb.q, sb.k_new, sb.v_new, sb.k_pool, sb.v_pool, sb.page_table, sb.n_s, sb.l_entry, sb.capacity,
                       outs[i % 3])
        b.record()
        ev.append((a, b))
    torch.cuda.synchronize()
    ms = statistics.median(a.elapsed_time(b) for a, b in ev[5:])
    res["n_s_4100_general_grid"] = {"attn_ms_median": round(ms, 5), "achieved_gbs": round(ab / (ms * 1e-3) / 1e9, 1),
                                    "frac_of_measured_hbm": round(ab / (ms * 1e-3) / 1e9 / peaks()["hbm"], 4)}
    ctx.close()
    return res


def headline_config_dict(spec, world):
    return {"workload": spec["text"], "sessions_per_step": len(spec["n_s"]), "gate_serves_per_step": spec["serves"],
            "resident_sets": spec["resident"],
            "l2": "flushed between timed steps" if spec["flush_l2"] else
                  "inputs larger than L2 (rotating resident sets; W_vocab alone is 8x L2)",
            "parallelism": f"session-sharded replicas x{world}, no collective"}


def main_reference(args, d):
    """--impl reference: the CPU oracle on this arm's config/metric/unit, each step a bounded sample."""
    if d.rank != 0:
        return
    name = args.config or HEADLINE
    spec = workload_spec(name)
    os_ = OracleSample(spec)
    steps = args.steps if args.steps is not None else 3
    warmup = args.warmup if args.warmup is not None else 1
    budget = 120.0 / max(1, steps + warmup)
    units, rows = os_.plan(min(budget, 15.0))
    for _ in range(warmup):
        os_.run(units, rows)
    t0 = time.perf_counter()
    fulls = [os_.run(units, rows)[0] for _ in range(steps)]
    wall = time.perf_counter() - t0
    value = statistics.fmean(fulls) * 1e6
    line = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus, "steps": steps,
        "warmup": warmup, "ms_per_step": wall * 1e3 / steps, "higher_is_better": False, "scaling": "weak",
        "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": headline_config_dict(spec, d.world),
        "sampling": "ms_per_step is the sampled step's wall time; value is the per-session estimate from the sample",
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": os_.cores, "kind": "oracle", "sample": os_.describe(units, rows)},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line))


def cpu_baseline_leg(spec, budget_s):
    """The oracle as it stands on the box's host cores: all cores on a bounded sample, and one thread on a smaller one."""
    osmp = OracleSample(spec)
    units, rows = osmp.plan(budget_s)
    full, spent = osmp.run(units, rows)
    out = {"value": full * 1e6, "unit": UNIT, "cores": osmp.cores, "kind": "oracle",
           "sample": osmp.describe(units, rows), "sample_seconds": round(spent, 2)}
    try:
        osmp.o.set_num_threads(1)
        u1 = max(1, min(units, max(1, units // osmp.cores)))
        r1 = max(min(1024, spec["shape"].V), rows // osmp.cores)
        full1, spent1 = osmp.run(u1, r1)
        out["one_thread"] = {"value": full1 * 1e6, "unit": UNIT, "cores": 1, "sample": osmp.describe(u1, r1),
                             "sample_seconds": round(spent1, 2)}
    finally:
        osmp.o.set_num_threads(osmp.cores)
    return out


def run_config(name, args, d, dev, prepos, steps=None, warmup=None):
    """One BASELINE config -> the dict of its JSON fields (rank 0; other ranks return None).  `steps` / `warmup`
    None = the config's own defaults (--steps / --warmup bind the headline config only)."""
    spec = workload_spec(name)
    steps = steps if steps is not None else DEFAULT_STEPS[name][0]
    warmup = max(warmup if warmup is not None else DEFAULT_STEPS[name][1], 3)
    wl = Workload(spec, dev, prepos)
    if args.attn_path:
        wl.ctx.set_attn_path(args.attn_path)
    n_sess = wl.n
    res = run_device_timed(wl, steps, warmup, d)
    total_ms = d.max(res["total_ms"], dev)
    ms_per_step = total_ms / steps
    # weak scaling: every rank pre-positions its own sessions; whole-job us/session = time / (N * sessions)
    value = ms_per_step * 1e3 / (n_sess * d.world)

    e2e = None
    if not args.no_e2e:
        e = run_e2e(wl, max(3, min(steps, 30)), 3, d)
        e_ms = d.max(e["ms_per_step"], dev)
        e2e = {"value": e_ms * 1e3 / (n_sess * d.world), "unit": UNIT, "h2d_bytes_per_step": e["h2d"], "d2h_bytes_per_step": e["d2h"],
               "timing": "CUDA events from before the first H2D to after the last D2H; copies on their own streams, two steps in flight"}
    if d.rank != 0:
        del wl
        torch.cuda.empty_cache()
        return None

    pk = peaks()
    ab = algorithmic_bytes(spec)
    calls = res["calls"]
    kern = {}
    for kname_ in ("entry_attn", "ready_dist"):
        gbs = ab[kname_] / (calls[kname_] * 1e-3) / 1e9
        kern[kname_] = {"ms": round(calls[kname_], 5), "ms_median": round(res["calls_median"][kname_], 5),
                        "ms_min": round(res["calls_min"][kname_], 5), "algorithmic_bytes": ab[kname_],
                        "achieved_gbs": round(gbs, 1), "frac_of_measured_hbm": round(gbs / pk["hbm"], 4)}
    fl = attention_flops(spec)
    kern["entry_attn"]["tflops"] = round(fl / (calls["entry_attn"] * 1e-3) / 1e12, 1)
    kern["entry_attn"]["frac_of_measured_bf16"] = round(kern["entry_attn"]["tflops"] / pk["bf16"], 4)
    kern["invalidate"] = {"ms": round(calls["invalidate"], 5)}
    kern["gate_serve"] = {"ms": round(calls["gate_serve"], 5), "requests": spec["serves"]}
    dom = max(("entry_attn", "ready_dist"), key=lambda k: calls[k])
    intensity = fl / max(1, ab["entry_attn"])   # flop per algorithmic byte of the attention call
    ridge = pk["bf16"] * 1e12 / (pk["hbm"] * 1e9)
    kname = ("attn_generic_kernel" if name == "c1" else "attn_umma_kernel") if dom == "entry_attn" else (
        "ready_dist_batch_kernel" if n_sess > 8 else "ready_dist_kernel")
    if dom == "entry_attn" and intensity >= 0.9 * ridge:
        # G * L_entry at or above the ridge: the attention is a tensor-bound dense contraction;
        # the kernel is timed alone between events: burst peak
        roofline = {"kernel": kname, "bound": "tensor", "achieved": kern[dom]["tflops"], "peak": pk["bf16"],
                    "unit": "TFLOP/s", "frac": kern[dom]["frac_of_measured_bf16"]}
    else:
        roofline = {"kernel": kname, "bound": "hbm", "achieved": kern[dom]["achieved_gbs"], "peak": pk["hbm"],
                    "unit": "GB/s", "frac": kern[dom]["frac_of_measured_hbm"]}
    traffic, traffic_src = ncu_traffic(name, kname)
    roofline.update({"traffic": traffic, "traffic_source": traffic_src, "algorithmic_bytes": ab[dom],
                     "flop_per_byte": round(intensity, 1) if dom == "entry_attn" else round(2.0 * n_sess, 1),
                     "peak_source": pk["source"], "share_of_step": round(calls[dom] / sum(calls.values()), 4)})
    step_bytes = ab["entry_attn"] + ab["ready_dist"]
    step_gbs = step_bytes / (ms_per_step * 1e-3) / 1e9
    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": d.world, "steps": steps, "warmup": warmup,
        "ms_per_step": ms_per_step, "higher_is_better": False, "scaling": "weak", "vs_baseline": None,
        "dtype": "bf16", "data": "synthetic",
        "config": headline_config_dict(spec, d.world),
        "roofline": roofline,
        "entry_pass_roofline": {"algorithmic_bytes": step_bytes, "achieved_gbs": round(step_gbs, 1),
                                "frac_of_measured_hbm": round(step_gbs / pk["hbm"], 4),
                                "frac_of_8tbs_nominal": round(step_gbs / 8000.0, 4)},
        "timing": {"mean_us_per_session": round(value, 3), "graph_replay": run_graph_replay(wl)},
        "kernels": kern,
        "clocks": res["clocks"],
        "clocks_per_call_pass": res["clocks_per_call_pass"],
        "gpu_launches": res["launches"],
    }
    if e2e:
        line["e2e"] = e2e
    if not args.quick:
        line["gate_serve"] = run_gate_serve(wl, prepos)
        line["attn_layer_sequential"] = run_layer_sequential(wl)
        ft = run_fall_through(wl)
        if ft:
            line["fall_through"] = ft
        if d.world == 1:
            line["co_schedule"] = run_co_schedule(wl, prepos)
            y = run_yield(wl, prepos)
            if y:
                line["co_schedule"]["decode_step_with_yield_wall_us"] = y
        if name in ("c2", "c5"):
            line["scan_logits"] = run_scan_logits(wl, prepos)
        if name in ("c2", "c4", "c5"):
            line["ready_dist_w4"] = run_ready_dist_w4(wl, prepos)
        if name in ("c2", "c3", "c4", "c5"):
            line["entry_attn_fp8"] = run_attn_fp8(wl, prepos)
        if name == "c3":
            line["update_trace"] = run_update_trace(wl, prepos)
    del wl
    torch.cuda.empty_cache()
    if name == "c2" and not args.quick:
        line["variants"] = run_c2_variants(spec, dev, prepos)
        torch.cuda.empty_cache()
    if not args.no_cpu_baseline:
        line["cpu_baseline"] = cpu_baseline_leg(spec, 12.0 if name == (args.config or HEADLINE) else 5.0)
    return line


DETAIL_REL = "gpurun_out/bench_detail.json"
DETAIL_PATH = os.path.join(ROOT, "gpurun_out", "bench_detail.json")
CONTRACT_KEYS = ("metric", "value", "unit", "n_gpus", "steps", "warmup", "ms_per_step", "higher_is_better", "scaling",
                 "vs_baseline", "dtype", "data", "config", "roofline", "entry_pass_roofline", "cpu_baseline", "e2e",
                 "clocks", "gpu_launches")


def _finite(x):
    """Non-finite floats -> None, so that the line is strict JSON."""
    if isinstance(x, float):
        return x if math.isfinite(x) else None
    if isinstance(x, dict):
        return {k: _finite(v) for k, v in x.items()}
    if isinstance(x, (list, tuple)):
        return [_finite(v) for v in x]
    return x


def contract_line(full, others):
    """The ONE stdout line: the headline config's contract fields only, a few KB (the driver parses this line; every
    side measurement and the other configs go to DETAIL_PATH).  `others`: {config: full dict} of the rest of the run."""
    line = {k: full[k] for k in CONTRACT_KEYS if k in full}
    if "cpu_baseline" in line:
        line["cpu_baseline"] = {k: v for k, v in line["cpu_baseline"].items() if k != "one_thread"}
    if "e2e" in line:
        line["e2e"] = {k: v for k, v in line["e2e"].items() if k != "timing"}
    line["kernels"] = {k: {kk: v[kk] for kk in ("ms", "frac_of_measured_hbm", "frac_of_measured_bf16") if kk in v}
                       for k, v in full["kernels"].items()}
    if "gate_serve" in full:
        line["gate_serve"] = {b: {"device_us_per_call": v["device_us_per_call"], "device_us_per_serve": v["device_us_per_serve"],
                                  "wall_us_per_call_p50": v["wall_us_per_call_p50"]}
                              for b, v in full["gate_serve"].items() if isinstance(v, dict) and "device_us_per_call" in v}
    if others:
        line["other_configs"] = {n: {"us_per_session": round(o["value"], 2), "roofline_bound": o["roofline"]["bound"],
                                     "roofline_frac": o["roofline"]["frac"],
                                     "step_frac_of_measured_hbm": o["entry_pass_roofline"]["frac_of_measured_hbm"]}
                                 for n, o in others.items()}
    line["detail"] = DETAIL_REL
    return _finite(line)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=None)
    ap.add_argument("--warmup", type=int, default=None)
    ap.add_argument("--config", default=None, choices=ALL_CONFIGS,
                    help="run this one config alone (default: all five, headline " + HEADLINE + ")")
    ap.add_argument("--impl", default="prepos", choices=["prepos", "reference"])
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--quick", action="store_true", help="the timed step only: no side measurements (for ncu runs)")
    ap.add_argument("--attn-path", type=int, default=0, help="0 auto, 1 generic CUDA-core kernel, 2 tcgen05 kernel")
    ap.add_argument("--section", default=None, choices=["entry_attn_fp8", "ready_dist_w4"],
                    help="run ONE side measurement of --config alone and print it (what the ncu captures of the "
                         "NEXT-4 kernels use)")
    args = ap.parse_args()

    d = Dist(args.gpus)
    if args.impl == "reference":
        main_reference(args, d)
        return

    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device -- libprepos has no CPU fallback (use --impl reference for the oracle)")
    from paper_2606_29565_b200 import prepos
    prepos.lib()  # fail loudly if the extension is missing
    torch.cuda.set_device(d.local_rank)
    dev = torch.device("cuda", d.local_rank)
    d.init("nccl")

    if args.section:
        spec = workload_spec(args.config or HEADLINE)
        spec = dict(spec, resident=min(spec["resident"], 2))
        wl = Workload(spec, dev, prepos)
        fn = {"entry_attn_fp8": run_attn_fp8, "ready_dist_w4": run_ready_dist_w4}[args.section]
        print(json.dumps({"config": spec["name"], args.section: fn(wl, prepos)}))
        return
    head = args.config or HEADLINE
    # the headline first, with the caller's --steps / --warmup; in the default run the other four follow with their
    # own defaults, so that steps x ms_per_step of the printed line is the headline's timed region
    names = [head] if args.config else [head] + [n for n in ALL_CONFIGS if n != head]
    lines = {}
    for name in names:
        mine = name == head
        lines[name] = run_config(name, args, d, dev, prepos, args.steps if mine else None, args.warmup if mine else None)
    if d.rank == 0:
        others = {n: lines[n] for n in names if n != head}
        detail = _finite({"headline": head, "configs": lines})
        try:
            os.makedirs(os.path.dirname(DETAIL_PATH), exist_ok=True)
            with open(DETAIL_PATH, "w") as f:
                json.dump(detail, f, allow_nan=False)
            sys.stderr.write(f"bench.py: every section of every config -> {DETAIL_PATH}\n")
        except OSError as e:   # a read-only tree: the contract line below does not depend on the side file
            sys.stderr.write(f"bench.py: could not write {DETAIL_PATH}: {e}\n")
        sys.stdout.write(json.dumps(contract_line(lines[head], others), allow_nan=False, separators=(",", ":")) + "\n")
        sys.stdout.flush()
    d.barrier()
    d.close()


if __name__ == "__main__":
    main()
