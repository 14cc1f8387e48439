#!/usr/bin/env python
"""bench.py -- one JSON line for BASELINE.json's metric: global-attention layer ms (and dense-equivalent / executed
TFLOP/s) at 100 frames.

A "step" is one pass of the whole hot path over one synthetic global-attention layer of config C3
(S=100 frames x 1374 tokens, N=137400, H=16, D=64, B=128): saf3r_select (pool -> score -> select) followed by
saf3r_sparse_attn, with a seeded per-layer mix of head types and sparsity.

  python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--config c2|c3|c4|c5]

N > 1 (torchrun): every rank runs the same number of independent layers (the path shards over independent
layers/heads with no data-path collective) -> "scaling": "weak".
--impl reference times the CPU oracle (oracle/), as it stands, on the host cores on a bounded sample of the workload.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

import numpy as np  # noqa: E402

import saf3r_synth as sy  # noqa: E402

METRIC = "global_attn_layer_ms"
UNIT = "ms/layer"


def load_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        d = json.load(open(p))
        return {"hbm_gbs": d["hbm_gbs"], "tflops_burst": d["bf16_tflops"], "tflops_sustained": d["bf16_tflops_sustained"],
                "source": "measured"}
    return {"hbm_gbs": 6650.0, "tflops_burst": 1590.0, "tflops_sustained": 1400.0, "source": "fallback"}


def shape_for(name: str) -> sy.Shape:
    return {"c2": sy.shape_c2, "c3": sy.shape_c3, "c4": sy.shape_c4, "c5": sy.shape_c5}[name]()


def make_layers(name: str, count: int, gen: str | None = None, ratio: float | None = None):
    sh = shape_for(name)
    layers = []
    for l in range(count):
        if name == "c3" and gen is None:
            layers.append(sy.config_c3_layer(l, sh=sh))
        else:
            gens, cfgs = sy.sweep_heads(sh, gen, ratio) if gen is not None else sy.mixed_heads(sh)
            layers.append(sy.make_layer(sh, gens, cfgs, seed={"c2": 2, "c3": 3, "c4": 4, "c5": 5}[name] * 1000 + l, layer=l))
    return layers


class ClockSampler:
    """Samples SM clock / throttle reasons / power during the timed region (NVML every 20 ms; nvidia-smi as a fallback)."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.index, self.rows, self.stop, self.t = index, [], threading.Event(), None
        self.nvml = None
        try:
            import pynvml
            pynvml.nvmlInit()
            self.nvml = pynvml
            self.handle = pynvml.nvmlDeviceGetHandleByIndex(index)
        except Exception:
            self.nvml = None

    def _sample_nvml(self):
        n = self.nvml
        sm = n.nvmlDeviceGetClockInfo(self.handle, n.NVML_CLOCK_SM)
        mx = n.nvmlDeviceGetMaxClockInfo(self.handle, n.NVML_CLOCK_SM)
        pw = n.nvmlDeviceGetPowerUsage(self.handle) / 1000.0
        r = n.nvmlDeviceGetCurrentClocksThrottleReasons(self.handle)
        flag = lambda b: "Active" if (r & b) else "Not Active"
        return [str(sm), str(mx), f"{pw:.1f}", flag(n.nvmlClocksThrottleReasonHwSlowdown),
                flag(n.nvmlClocksThrottleReasonHwThermalSlowdown), flag(n.nvmlClocksThrottleReasonSwThermalSlowdown),
                flag(n.nvmlClocksThrottleReasonSwPowerCap)]

    def _run(self):
        while not self.stop.is_set():
            try:
                if self.nvml is not None:
                    self.rows.append(self._sample_nvml())
                else:
                    o = subprocess.run(["nvidia-smi", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits", "-i", str(self.index)],
                                       capture_output=True, text=True, timeout=5).stdout.strip()
                    if o:
                        self.rows.append([x.strip() for x in o.split(",")])
            except Exception:
                pass
            self.stop.wait(0.02 if self.nvml is not None else 0.2)

    def __enter__(self):
        self.t = threading.Thread(target=self._run, daemon=True)
        self.t.start()
        return self

    def __exit__(self, *a):
        self.stop.set()
        self.t.join(timeout=6)

    def summary(self):
        sm = [float(r[0]) for r in self.rows if r and r[0].replace(".", "").isdigit()]
        mx = [float(r[1]) for r in self.rows if len(r) > 1 and r[1].replace(".", "").isdigit()]
        pw = [float(r[2]) for r in self.rows if len(r) > 2 and r[2].replace(".", "").isdigit()]
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        reasons = sorted({n for r in self.rows if len(r) >= 7 for n, v in zip(names, r[3:7]) if v.lower().startswith("active")})
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(mx) if mx else None, "reasons": reasons,
                "samples": len(sm), "power_w_max": max(pw) if pw else None, "source": "nvml" if self.nvml is not None else "nvidia-smi"}


class ClockLog:
    """One NVML sampling SUBPROCESS for the whole run (10 ms period, rows stamped with time.time()).  The thread sampler above is
    starved while this process's main thread queues launches (it holds the GIL for the whole 0.2 s timed region: the driver-run
    line of round 2 carried one sample); a separate process is not.  region() brackets a timed region by wall clock; its summary
    keeps the rows stamped inside it."""
    SRC = r"""
import sys, time
import pynvml as n
n.nvmlInit()
h = n.nvmlDeviceGetHandleByIndex(int(sys.argv[1]))
f = open(sys.argv[2], "w", buffering=1)
B = [n.nvmlClocksThrottleReasonHwSlowdown, n.nvmlClocksThrottleReasonHwThermalSlowdown, n.nvmlClocksThrottleReasonSwThermalSlowdown, n.nvmlClocksThrottleReasonSwPowerCap]
while True:
    try:
        r = n.nvmlDeviceGetCurrentClocksThrottleReasons(h)
        f.write("%.4f %d %d %.1f %s\n" % (time.time(), n.nvmlDeviceGetClockInfo(h, n.NVML_CLOCK_SM), n.nvmlDeviceGetMaxClockInfo(h, n.NVML_CLOCK_SM),
                                          n.nvmlDeviceGetPowerUsage(h) / 1000.0, " ".join("1" if r & b else "0" for b in B)))
    except Exception:
        pass
    time.sleep(0.01)
"""

    def __init__(self, index: int):
        import tempfile
        self.index, self.proc = index, None
        self.path = os.path.join(tempfile.gettempdir(), f"saf3r_clocks_{os.getpid()}_{index}.log")
        try:
            self.proc = subprocess.Popen([sys.executable, "-c", self.SRC, str(index), self.path], stdout=subprocess.DEVNULL, stderr=subprocess.DEVNULL)
        except Exception:
            self.proc = None

    def rows(self, t0: float, t1: float):
        out = []
        try:
            for line in open(self.path):
                p = line.split()
                if len(p) == 8 and t0 <= float(p[0]) <= t1:
                    out.append(p)
        except Exception:
            pass
        return out

    def region(self):
        return _ClockRegion(self)

    def close(self):
        if self.proc is not None:
            self.proc.terminate()
            try:
                self.proc.wait(timeout=3)
            except Exception:
                self.proc.kill()
            self.proc = None
        try:
            os.remove(self.path)
        except OSError:
            pass


class _ClockRegion:
    """with log.region() as r: <timed region>;  r.summary() -> the `clocks` object of the JSON line.  Falls back to the in-process
    thread sampler when the subprocess gave nothing (no pynvml in a child, say)."""

    def __init__(self, log: ClockLog):
        self.log, self.t0, self.t1 = log, 0.0, 0.0
        self.fallback = ClockSampler(log.index)

    def __enter__(self):
        self.fallback.__enter__()
        self.t0 = time.time()
        return self

    def __exit__(self, *a):
        self.t1 = time.time()
        self.fallback.__exit__()

    def summary(self):
        time.sleep(0.03)                                          # let the sampler flush its last rows
        rows = self.log.rows(self.t0, self.t1)
        if len(rows) < 2:
            s = self.fallback.summary()
            s["source"] += " (in-process thread; the sampling subprocess returned %d rows)" % len(rows)
            return s
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        reasons = sorted({n for r in rows for n, v in zip(names, r[4:8]) if v == "1"})
        return {"sm_mhz": float(np.median([float(r[1]) for r in rows])), "sm_max_mhz": max(float(r[2]) for r in rows), "reasons": reasons,
                "samples": len(rows), "power_w_max": max(float(r[3]) for r in rows), "source": "nvml, sampling subprocess, 10 ms period",
                "region_s": round(self.t1 - self.t0, 4)}


def time_layer(sf, ctx, torch, stream, clocklog, peaks, sh, shape, qkv, out, cfgs, steps: int, warm: int):
    """select + sparse_attn of one resident layer with the rules `cfgs`, `steps` timed passes after `warm` untimed ones: CUDA events
    on the launching stream around every call, a clocks summary of the timed region.  Used for the side configurations of the
    default line (C2, the C4 sweep); the headline loop in run_ours does the same over rotating layers."""
    q, k, v = qkv
    entries, ws_bytes = sf.query_sizes(shape, cfgs)
    lists = sf.Lists(torch.empty(sh.H * sh.NB + 1, dtype=torch.int64, device=q.device), torch.empty(max(entries, 1), dtype=torch.int32, device=q.device))
    ws = torch.empty(ws_bytes, dtype=torch.uint8, device=q.device)
    for _ in range(warm):
        ctx.select(q, k, shape, cfgs, workspace=ws, lists=lists)
        ctx.sparse_attn(q, k, v, shape, lists, out=out)
    torch.cuda.synchronize()
    evs = [[torch.cuda.Event(enable_timing=True) for _ in range(3)] for _ in range(steps)]
    with clocklog.region() as clk:
        for e in evs:
            e[0].record(stream)
            ctx.select(q, k, shape, cfgs, workspace=ws, lists=lists)
            e[1].record(stream)
            ctx.sparse_attn(q, k, v, shape, lists, out=out)
            e[2].record(stream)
        torch.cuda.synchronize()
    sel = float(np.mean([e[0].elapsed_time(e[1]) for e in evs]))
    att = float(np.mean([e[1].elapsed_time(e[2]) for e in evs]))
    layer = evs[0][0].elapsed_time(evs[-1][2]) / steps
    need = sum((2 if c["type"] in (sy.HEAD_QUERY_PROBE_TOPK, sy.HEAD_BLOCK_TOPK) else 0) for c in cfgs)
    sel_gbs = need * sh.N * sh.D * 2 / (sel * 1e-3) / 1e9 if need else None
    tf = 4.0 * sh.B * sh.B * sh.D * entries / (att * 1e-3) / 1e12
    del lists, ws
    return {"layer_ms": layer, "select_ms": sel, "sparse_attn_ms": att, "select_fraction_of_layer": sel / layer,
            "select_frac_of_hbm_peak": (sel_gbs / peaks["hbm_gbs"]) if sel_gbs else None,
            "executed_tflops": tf, "frac_of_sustained_peak": tf / peaks["tflops_sustained"],
            "kept_pair_ratio": entries / (sh.H * sh.NB * sh.NB), "steps": steps, "warmup": warm, "clocks": clk.summary()}


def time_dense(ctx, torch, stream, sh, shape, qkv, out, reps: int):
    q, k, v = qkv
    ctx.dense_attn(q, k, v, shape, out=out)
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record(stream)
    for _ in range(reps):
        ctx.dense_attn(q, k, v, shape, out=out)
    e1.record(stream)
    torch.cuda.synchronize()
    ms = e0.elapsed_time(e1) / reps
    return ms, 4.0 * sh.N * sh.N * sh.D * sh.H / (ms * 1e-3) / 1e12


def side_configs(sf, ctx, torch, dev, stream, clocklog, peaks):
    """The other BASELINE.json configurations inside the default line (`configs` key), bounded so that the run stays within
    minutes: C2 (VGGT shape, one layer, the C2 head mix) and the C4 sparsity sweep at ALL five ratios {50, 25, 10, 5, 2} % for
    the same-position generator (16 BLOCK_TOPK heads, one resident layer, a few steps each; Q/K/V of 1.7 GB exceed L2) plus one
    dense pass of each.  C3 is the headline, C5 the `s500` key."""
    up = lambda x: torch.from_numpy(x.view(np.int16)).to(dev).view(torch.bfloat16)
    out = {}
    # ---- C2
    L = sy.config_c2()
    sh = L.shape
    shape = sf.make_shape(sh.S, sh.T, sh.H, sh.D, sh.B)
    qkv = (up(L.q), up(L.k), up(L.v))
    o = torch.empty_like(qkv[0])
    r = time_layer(sf, ctx, torch, stream, clocklog, peaks, sh, shape, qkv, o, L.cfgs, steps=200, warm=5)
    dms, dtf = time_dense(ctx, torch, stream, sh, shape, qkv, o, reps=4)
    r.update({"workload": workload_name("c2", sh), "dense_attn_ms": dms, "dense_tflops": dtf, "speedup_vs_own_dense": dms / r["layer_ms"],
              "l2": "one resident layer; its 270 MB of Q/K/V exceed the 126 MB L2"})
    out["c2"] = r
    del qkv, o, L
    # ---- C4 sweep
    sh = sy.shape_c4()
    shape = sf.make_shape(sh.S, sh.T, sh.H, sh.D, sh.B)
    gens, cfgs = sy.sweep_heads(sh, sy.GEN_SAME_POSITION, 0.5)
    L = sy.make_layer(sh, gens, cfgs, seed=4000, layer=0, threads=16)   # the data of a generator does not depend on the ratio
    qkv = (up(L.q), up(L.k), up(L.v))
    del L
    o = torch.empty_like(qkv[0])
    dms, dtf = time_dense(ctx, torch, stream, sh, shape, qkv, o, reps=1)
    sweep = []
    for ratio in (0.5, 0.25, 0.10, 0.05, 0.02):
        _, cfgs = sy.sweep_heads(sh, sy.GEN_SAME_POSITION, ratio)
        r = time_layer(sf, ctx, torch, stream, clocklog, peaks, sh, shape, qkv, o, cfgs, steps=3 if ratio > 0.2 else 6, warm=1)
        r.update({"ratio": ratio, "keep_blocks": cfgs[0]["keep_blocks"], "speedup_vs_own_dense": dms / r["layer_ms"]})
        sweep.append(r)
    out["c4"] = {"workload": workload_name("c4", sh, sy.GEN_SAME_POSITION, 0.5).replace(" at kept-block ratio 0.5", "") + ", kept-block ratios 50/25/10/5/2 %",
                 "dense_attn_ms": dms, "dense_tflops": dtf, "dense_reps": 1, "sweep": sweep,
                 "l2": "one resident layer; its 1.7 GB of Q/K/V exceed the 126 MB L2"}
    del qkv, o
    torch.cuda.empty_cache()
    return out


def cpu_sample_qblocks() -> int:
    """q-blocks sampled per head by the CPU-oracle legs: the oracle parallelises its attention over q-blocks (OpenMP, one
    q-block per thread at a time), so at least 2 per host core are needed to keep every core busy (>= 32)."""
    return max(32, 2 * (os.cpu_count() or 1))


def cpu_oracle_layer_ms(L: sy.Layer, nq: int | None = None):
    """The oracle as it stands on ALL host cores, on a bounded sample of the layer, extrapolated to the whole layer.  The one
    sampler both arms use (the GPU arm's cpu_baseline leg and --impl reference), so that their numbers agree:
      - one head of each head generator is run (the first of its kind): its full selection (timed, scaled by the number of heads
        of that kind) and its attention on `nq` sampled q-blocks (all cores busy: nq >= 2 x cores);
      - the attention time is scaled by listed (q-block, k-block) pairs: (pairs of ALL heads of that kind) / (pairs of the sampled
        q-blocks), since the oracle's attention time is proportional to the number of listed pairs.
    Returns (layer ms, select ms, cores, threads_busy, sample description)."""
    import oracle as orc
    sh = L.shape
    nq = min(sh.NB, nq or cpu_sample_qblocks())
    rng = np.random.default_rng(0)
    first = {}
    for h, g in enumerate(L.gens):
        first.setdefault(g, h)
    t_sel = t_att = 0.0
    for g, h in sorted(first.items(), key=lambda kv: kv[1]):
        same = [i for i, gg in enumerate(L.gens) if gg == g]
        t0 = time.perf_counter()
        hl = orc.select_head(L.q[h], L.k[h], sh.S, sh.T, sh.B, orc.make_cfg(**L.cfgs[h]))
        t1 = time.perf_counter()
        qb = np.sort(rng.choice(sh.NB, nq, replace=False)).astype(np.int64)
        orc.attn_lists(L.q[h], L.k[h], L.v[h], sh.B, hl.row_ptr, hl.col_idx, qb, want_lse=False)
        t2 = time.perf_counter()
        pairs_sampled = int(np.sum(hl.row_ptr[qb + 1] - hl.row_ptr[qb]))
        pairs_kind = 0
        for i in same:                                           # list lengths are closed forms of (shape, cfg): no data needed
            c = L.cfgs[i]
            if c == L.cfgs[h]:
                pairs_kind += int(hl.row_ptr[-1])
            else:
                pairs_kind += closed_form_pairs(sh, c, hl, L.cfgs[h])
        t_sel += len(same) * (t1 - t0)
        t_att += (t2 - t1) * pairs_kind / max(1, pairs_sampled)
    cores = orc.num_threads()
    sample = (f"one head per head generator ({len(first)} of {sh.H} heads): full select (scaled by heads of that kind) + attention on "
              f"{nq} sampled q-blocks of that head, scaled by listed block pairs of all heads of that kind / pairs sampled "
              f"(extrapolated to the layer)")
    return (t_sel + t_att) * 1e3, t_sel * 1e3, cores, min(cores, nq), sample


def closed_form_pairs(sh: sy.Shape, c: dict, hl_ref, c_ref: dict) -> int:
    """Listed pairs of a head with configuration c, given the oracle lists hl_ref of a head of the same kind with c_ref: list
    lengths depend only on (shape, cfg).  Top-n / stride-n heads: NB x n; per-row closed forms (frame-local): same as the reference."""
    if c["type"] in (sy.HEAD_QUERY_PROBE_TOPK, sy.HEAD_BLOCK_TOPK) and c.get("topk_scope", 0) == sy.SCOPE_GLOBAL:
        return sh.NB * min(sh.NB, c["keep_blocks"])
    if c["type"] == sy.HEAD_UNIFORM_STRIDE:
        n = c["keep_blocks"] if c["stride"] == 0 else -(-(sh.NB - c["offset"]) // c["stride"])
        return sh.NB * n
    assert c == c_ref, "per-row closed forms: heads of one kind share one configuration in the bench recipes"
    return int(hl_ref.row_ptr[-1])


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    sh = shape_for(args.config)
    layers = make_layers(args.config, 1)
    times = []
    for i in range(args.warmup + args.steps):
        ms, _, cores, busy, sample = cpu_oracle_layer_ms(layers[0])
        if i >= args.warmup:
            times.append(ms)
    v = float(np.mean(times))
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": v, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": v, "higher_is_better": False, "scaling": "weak", "vs_baseline": None,
        "dtype": "f64", "data": "synthetic",
        "config": {"workload": workload_name(args.config, sh), "note": "CPU oracle (oracle/), not tuned"},
        "cpu_baseline": {"value": v, "unit": UNIT, "cores": cores, "threads_busy": busy, "kind": "oracle", "sample": "per step: " + sample},
        "e2e": {"value": v, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
    }))


def workload_name(cfg: str, sh: sy.Shape, gen: str | None = None, ratio: float | None = None) -> str:
    base = f"{cfg.upper()}: one global-attention layer, S={sh.S} frames x T={sh.T} tokens, N={sh.N}, H={sh.H}, D={sh.D}, block {sh.B}, "
    if gen is not None:
        return base + f"all heads of generator '{gen}' at kept-block ratio {ratio:g}"
    return base + ("seeded per-layer mix of head types (uniform-stride / frame-local / same-position block top-k / "
                   "sink query-probe) and sparsity")


def run_ours(args):
    import torch
    import torch.distributed as dist
    import paper_2607_03612_b200 as sf

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device(f"cuda:{local}"))
    torch.cuda.set_device(local)
    dev = torch.device(f"cuda:{local}")
    clocklog = ClockLog(local)                                    # started early: the child needs ~0.5 s to import and initialise NVML
    peaks = load_peaks()
    sh = shape_for(args.config)
    n_res = min(args.resident_layers, args.steps)
    layers = make_layers(args.config, n_res, args.gen, args.ratio)
    ctx = sf.Context(local)
    shape = sf.make_shape(sh.S, sh.T, sh.H, sh.D, sh.B)
    stream = torch.cuda.current_stream()

    def up(x):
        return torch.from_numpy(x.view(np.int16)).to(dev).view(torch.bfloat16)

    dl = []
    for L in layers:
        q, k, v = up(L.q), up(L.k), up(L.v)
        entries, ws_bytes = sf.query_sizes(shape, L.cfgs)
        lists = sf.Lists(torch.empty(sh.H * sh.NB + 1, dtype=torch.int64, device=dev),
                         torch.empty(max(entries, 1), dtype=torch.int32, device=dev))
        ws = torch.empty(ws_bytes, dtype=torch.uint8, device=dev)
        out = torch.empty_like(q)
        dl.append(dict(q=q, k=k, v=v, lists=lists, ws=ws, out=out, cfgs=L.cfgs, entries=entries, ws_bytes=ws_bytes))

    def step(i, ev=None):
        d = dl[i % n_res]
        if ev:
            ev[0].record(stream)
        ctx.select(d["q"], d["k"], shape, d["cfgs"], workspace=d["ws"], lists=d["lists"])
        if ev:
            ev[1].record(stream)
        ctx.sparse_attn(d["q"], d["k"], d["v"], shape, d["lists"], out=d["out"])
        if ev:
            ev[2].record(stream)

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    for i in range(args.warmup):
        step(i)
    barrier()
    evs = [[torch.cuda.Event(enable_timing=True) for _ in range(3)] for _ in range(args.steps)]
    launches0 = ctx.launch_count()
    with clocklog.region() as clk:
        barrier()
        t_beg, t_end = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        t_beg.record(stream)
        for i in range(args.steps):
            step(i, evs[i])
        t_end.record(stream)
        barrier()
    launches = ctx.launch_count() - launches0
    total_ms = t_beg.elapsed_time(t_end)
    from paper_2607_03612_b200.sharding import max_over_ranks
    total_ms = max_over_ranks(total_ms, dev)                     # device timing, MAX over ranks
    sel_ms = [e[0].elapsed_time(e[1]) for e in evs]
    att_ms = [e[1].elapsed_time(e[2]) for e in evs]

    # work per step
    pairs = [d["entries"] for d in dl]
    exec_flop = [4.0 * sh.B * sh.B * sh.D * pairs[i % n_res] for i in range(args.steps)]
    dense_flop = 4.0 * sh.N * sh.N * sh.D * sh.H
    att_s = float(np.sum(att_ms)) * 1e-3
    exec_tflops = float(np.sum(exec_flop)) / att_s / 1e12
    ms_per_step = total_ms / args.steps
    value = total_ms / (args.steps * world)

    result = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": ms_per_step, "higher_is_better": False, "scaling": "weak", "vs_baseline": None, "dtype": "bf16",
        "data": "synthetic",
        "config": {"workload": workload_name(args.config, sh, args.gen, args.ratio), "resident_layers": n_res,
                   "resident_note": f"{n_res} seeded layers are resident and rotated (the C3 stack has 24; tests/test_gpu_parity.py checks exactly "
                                    "layers 0-3 against the oracle); --resident-layers 24 keeps all of them (27 GB)",
                   "l2": "inputs (844 MB of Q/K/V per layer at C3) exceed the 126 MB L2; layers rotate" if args.config != "c2"
                   else "inputs 270 MB/layer exceed L2; layers rotate",
                   "kept_pair_ratio": float(np.mean(pairs)) / (sh.H * sh.NB * sh.NB)},
        "gpu_launches": int(launches),
        "select_ms": float(np.mean(sel_ms)), "sparse_attn_ms": float(np.mean(att_ms)),
        "executed_tflops": exec_tflops, "dense_equiv_tflops": dense_flop * args.steps / (total_ms * 1e-3) / 1e12,
        "footprint_bytes": {"qkv_out": 4 * sh.H * sh.N * sh.D * 2, "lists": int(max(pairs)) * 4 + (sh.H * sh.NB + 1) * 8,
                            "select_workspace": int(dl[0]["ws_bytes"])},
    }

    if rank == 0:
        result["clocks"] = clk.summary()
        # roofline of the dominant kernel (block-sparse attention): executed FLOP per launch / mean launch duration
        traffic, traffic_note = None, "no ncu capture recorded (profiles/traffic.json)"
        tp = os.path.join(ROOT, "profiles", "traffic.json")
        if os.path.exists(tp):
            tj = json.load(open(tp))
            import hashlib
            sha = hashlib.sha256(open(os.path.join(ROOT, "paper_2607_03612_b200", "csrc", "attn_kernel.cuh"), "rb").read()).hexdigest()[:16]
            if tj.get("attn_kernel_sha16") == sha:               # the capture belongs to the kernel source that is running
                traffic = tj.get("saf3r_attn_kernel_bytes_per_launch")
                traffic_note = "ncu dram bytes read + written of the layer-0 launch (profiles/traffic.json, same attn_kernel.cuh); achieved is the mean over the resident layers"
            else:
                traffic_note = f"profiles/traffic.json was captured for another build of attn_kernel.cuh ({tj.get('attn_kernel_sha16')} != {sha}): dropped"
        result["roofline"] = {"bound": "tensor", "achieved": exec_tflops, "peak": peaks["tflops_sustained"], "unit": "TFLOP/s",
                              "frac": exec_tflops / peaks["tflops_sustained"], "traffic": traffic,
                              "traffic_note": traffic_note,
                              "kernel": "saf3r_attn_kernel", "peak_source": f"{peaks['source']} sustained bf16 (kernel timed inside a long step)",
                              "frac_of_burst": exec_tflops / peaks["tflops_burst"]}
        # selection pass against HBM: algorithmic bytes = Q and/or K of the heads whose rule reads them
        need = [sum((2 if c["type"] in (sy.HEAD_QUERY_PROBE_TOPK, sy.HEAD_BLOCK_TOPK) else 0) for c in d["cfgs"]) for d in dl]
        sel_bytes = [need[i % n_res] * sh.N * sh.D * 2 for i in range(args.steps)]
        sel_gbs = float(np.sum(sel_bytes)) / (float(np.sum(sel_ms)) * 1e-3) / 1e9
        result["select_roofline"] = {"bound": "hbm", "achieved": sel_gbs, "peak": peaks["hbm_gbs"], "unit": "GB/s",
                                     "frac": sel_gbs / peaks["hbm_gbs"], "note": "whole select call (pool+score+select) over the pool stage's algorithmic bytes"}
        # stage split of the select call (untimed extra pass with saf3r_set_stage_timing): pool launch vs score+select launch
        ctx.set_stage_timing(True)
        pool_ms, ssel_ms = [], []
        for i in range(2 * n_res):
            d = dl[i % n_res]
            torch.cuda._sleep(1_000_000)   # ~0.5 ms of GPU spin first, so that the host has queued the whole call before
                                           # its first kernel can start (otherwise the stage times include host submission)
            ctx.select(d["q"], d["k"], shape, d["cfgs"], workspace=d["ws"], lists=d["lists"])
            a, b = ctx.last_select_stage_ms()
            if i >= n_res:
                pool_ms.append(a)
                ssel_ms.append(b)
        ctx.set_stage_timing(False)
        pool_gbs = float(np.sum([need[i] * sh.N * sh.D * 2 for i in range(n_res)])) / (float(np.sum(pool_ms)) * 1e-3) / 1e9
        result["select_stages"] = {"pool_ms": float(np.mean(pool_ms)), "score_select_ms": float(np.mean(ssel_ms)),
                                   "pool_gbs": pool_gbs, "pool_frac_of_hbm_peak": pool_gbs / peaks["hbm_gbs"],
                                   "note": "pool launch = pooling + row_ptr + closed-form lists; score_select = probe + score + top-n + list copies; CUDA events inside saf3r_select"}

        if not args.skip_dense:
            d = dl[0]
            torch.cuda.synchronize()
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            ctx.dense_attn(d["q"], d["k"], d["v"], shape, out=d["out"])
            e0.record(stream)
            for _ in range(args.dense_reps):
                ctx.dense_attn(d["q"], d["k"], d["v"], shape, out=d["out"])
            e1.record(stream)
            torch.cuda.synchronize()
            dense_ms = e0.elapsed_time(e1) / args.dense_reps
            result["dense_attn_ms"] = dense_ms
            result["dense_tflops"] = dense_flop / (dense_ms * 1e-3) / 1e12
            result["speedup_vs_own_dense"] = dense_ms / ms_per_step
            result["speedup_vs_own_dense_s100"] = dense_ms / ms_per_step
            # quality of the sparse layer against the library's own dense output (Eq. 1 of the paper; reported,
            # not a gate): NMSE per head of layer 0, summarised by head generator.  d["out"] holds the dense output now.
            sp = torch.empty_like(d["out"])
            ctx.dense_attn(d["q"], d["k"], d["v"], shape, out=d["out"])
            ctx.select(d["q"], d["k"], shape, d["cfgs"], workspace=d["ws"], lists=d["lists"])
            ctx.sparse_attn(d["q"], d["k"], d["v"], shape, d["lists"], out=sp)
            nm = ctx.nmse(d["out"], sp, shape)                   # both sums of Eq. 1 in the library (saf3r_nmse_accumulate)
            by = {}
            for h, gname in enumerate(layers[0].gens):
                by.setdefault(gname, []).append(nm[h])
            bad = [h for h in range(sh.H) if not nm[h] < 1.0]
            result["quality_vs_own_dense"] = {
                "nmse_by_generator": {k2: float(np.mean(v2)) for k2, v2 in by.items()}, "nmse_max": float(max(nm)),
                "nmse_by_head": [float(x) for x in nm], "heads_with_nmse_ge_1": bad,
                "generators_with_nmse_ge_1": sorted({layers[0].gens[h] for h in bad}),
                "note": "layer 0; Eq. 1 (PAPER.md:L108) with O_full = dense mode, bf16 outputs.  Read speedup_vs_own_dense together with "
                        "this: it is the cost ratio at the SEEDED budgets of the synthetic recipe, not an iso-quality number.  Heads listed "
                        "under heads_with_nmse_ge_1 are no better than an all-zero output under Eq. 1 - an artefact of synthetic heads "
                        "whose full-attention output is a near-zero mean of V (tiny ||O_full||), not a property the paper's trained "
                        "heads have; c3_profiled_budgets quotes the speedup at the budgets the paper's own search (Eq. 2) settles for."}
            del sp

        # the layer with budgets chosen by the offline search (sigma = 0.85 as in L161) instead of the seeded
        # sigma of the C3 recipe: a speedup quoted at the NMSE the search settles for
        if not args.skip_profiled and args.config == "c3" and args.gen is None and not args.skip_dense:
            from paper_2607_03612_b200 import profiling
            d = dl[0]
            prof = profiling.profile_heads(ctx, [(d["q"], d["k"], d["v"])], shape, sigma=0.85)
            pcfgs = [p.cfg for p in prof]
            p_entries, _ = sf.query_sizes(shape, pcfgs)
            plists = sf.Lists(torch.empty(sh.H * sh.NB + 1, dtype=torch.int64, device=dev), torch.empty(max(p_entries, 1), dtype=torch.int32, device=dev))
            def pstep():
                ctx.select(d["q"], d["k"], shape, pcfgs, workspace=d["ws"], lists=plists)
                ctx.sparse_attn(d["q"], d["k"], d["v"], shape, plists, out=d["out"])
            for _ in range(2):
                pstep()
            torch.cuda.synchronize()
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record(stream)
            for _ in range(4):
                pstep()
            e1.record(stream)
            torch.cuda.synchronize()
            p_ms = e0.elapsed_time(e1) / 4
            by_n, by_b = {}, {}
            for h, gname in enumerate(layers[0].gens):
                by_n.setdefault(gname, []).append(prof[h].nmse)
                by_b.setdefault(gname, []).append(prof[h].nmse_base)
            kinds = {sy.HEAD_UNIFORM_STRIDE: "uniform_stride", sy.HEAD_STATIC: "static", sy.HEAD_QUERY_PROBE_TOPK: "query_probe_topk", sy.HEAD_BLOCK_TOPK: "block_topk"}
            result["c3_profiled_budgets"] = {
                "layer_ms": p_ms, "speedup_vs_own_dense": result["dense_attn_ms"] / p_ms,
                "kept_pair_ratio": p_entries / (sh.H * sh.NB * sh.NB),
                "kept_pair_ratio_baseline": sum(p.cost_base for p in prof) / (4.0 * sh.B * sh.B * sh.D) / (sh.H * sh.NB * sh.NB),
                "nmse_by_generator": {k2: float(np.mean(v2)) for k2, v2 in by_n.items()},
                "nmse_uniform_baseline_by_generator": {k2: float(np.mean(v2)) for k2, v2 in by_b.items()},
                "chosen_kernel_by_head": [kinds.get(p.cfg["type"], "?") for p in prof],
                "note": "layer 0; per-head kernel + setting chosen by paper_2607_03612_b200.profiling.profile_heads (Eq. 1 / Eq. 2, sigma = 0.85, "
                        "one calibration sample = the layer itself); NMSE on fp32 outputs"}
            del plists

        # the 500-frame point north_star asks for (C5: S = 500, N = 687 000, C2's head mix), bounded: 1 layer, 2 steps, 1 dense pass
        if not args.skip_s500 and args.config == "c3" and args.gen is None and not args.skip_dense:
            sh5 = sy.shape_c5()
            gens5, cfgs5 = sy.mixed_heads(sh5)
            L5 = sy.make_layer(sh5, gens5, cfgs5, seed=5000, layer=0, threads=16)
            shape5 = sf.make_shape(sh5.S, sh5.T, sh5.H, sh5.D, sh5.B)
            q5, k5, v5 = up(L5.q), up(L5.k), up(L5.v)
            del L5
            out5 = torch.empty_like(q5)
            ent5, ws5b = sf.query_sizes(shape5, cfgs5)
            lists5 = sf.Lists(torch.empty(sh5.H * sh5.NB + 1, dtype=torch.int64, device=dev), torch.empty(max(ent5, 1), dtype=torch.int32, device=dev))
            ws5 = torch.empty(ws5b, dtype=torch.uint8, device=dev)
            def step5():
                ctx.select(q5, k5, shape5, cfgs5, workspace=ws5, lists=lists5)
                ctx.sparse_attn(q5, k5, v5, shape5, lists5, out=out5)
            step5()
            torch.cuda.synchronize()
            e0, e1, e2 = (torch.cuda.Event(enable_timing=True) for _ in range(3))
            e0.record(stream)
            step5(); step5()
            e1.record(stream)
            ctx.dense_attn(q5, k5, v5, shape5, out=out5)
            e2.record(stream)
            torch.cuda.synchronize()
            l5, d5 = e0.elapsed_time(e1) / 2, e1.elapsed_time(e2)
            result["s500"] = {"workload": workload_name("c5", sh5), "layer_ms": l5, "dense_attn_ms": d5, "speedup_vs_own_dense": d5 / l5,
                              "executed_tflops_incl_select": 4.0 * sh5.B * sh5.B * sh5.D * ent5 / (l5 * 1e-3) / 1e12,
                              "dense_tflops": 4.0 * sh5.N * sh5.N * sh5.D * sh5.H / (d5 * 1e-3) / 1e12,
                              "kept_pair_ratio": ent5 / (sh5.H * sh5.NB * sh5.NB),
                              "footprint_bytes": {"qkv_out": 4 * sh5.H * sh5.N * sh5.D * 2, "lists": ent5 * 4 + (sh5.H * sh5.NB + 1) * 8, "select_workspace": ws5b},
                              "steps": 2, "dense_reps": 1}
            result["speedup_vs_own_dense_s500"] = d5 / l5
            result["layer_ms_s500"] = l5
            del q5, k5, v5, out5, lists5, ws5

        # the other BASELINE.json configurations (C2, the C4 sweep at all five ratios), bounded
        if not args.skip_configs and args.config == "c3" and args.gen is None and not args.skip_dense:
            result["configs"] = side_configs(sf, ctx, torch, dev, stream, clocklog, peaks)

        # e2e through the C ABI with HOST buffers (pinned), H2D + D2H inside the timed region
        if not args.skip_e2e:
            L = layers[0]
            qh, kh, vh = (torch.from_numpy(x.view(np.int16)).view(torch.bfloat16).pin_memory() for x in (L.q, L.k, L.v))
            oh = torch.empty_like(qh).pin_memory()
            scratch = torch.empty(ctx.layer_host_scratch_bytes(shape, L.cfgs), dtype=torch.uint8, device=dev)
            e_steps = max(2, min(args.steps, 6))
            for _ in range(2):
                ctx.layer_host(qh, kh, vh, shape, L.cfgs, scratch, oh)
            torch.cuda.synchronize()
            t0 = time.perf_counter()
            for _ in range(e_steps):
                ctx.layer_host(qh, kh, vh, shape, L.cfgs, scratch, oh)
                torch.cuda.synchronize()
            e_ms = (time.perf_counter() - t0) * 1e3 / e_steps
            nbytes = qh.numel() * 2
            result["e2e"] = {"value": e_ms, "unit": UNIT, "h2d_bytes_per_step": 3 * nbytes, "d2h_bytes_per_step": nbytes,
                             "steps": e_steps, "api": "saf3r_layer_host (pinned host q/k/v -> device, select + sparse_attn, out -> host; pipelined over 9 head groups)"}

        if world == 1 and not args.skip_cpu:
            ms, sel, cores, busy, sample = cpu_oracle_layer_ms(layers[0])
            result["cpu_baseline"] = {"value": ms, "unit": UNIT, "cores": cores, "threads_busy": busy, "kind": "oracle",
                                      "sample": "layer 0: " + sample, "select_ms": sel}
            result["vs_cpu_oracle"] = {"ratio": ms / ms_per_step, "note": "extrapolated, untuned CPU oracle / this run; reported, not a target"}
        print(json.dumps(result))
    clocklog.close()
    if world > 1:
        dist.destroy_process_group()


def run_head_parallel(args):
    """SURVEY 8(e), head-parallel split of ONE layer (strong scaling): the heads of C3 layer 0 are assigned to the N ranks by
    sharding.assign_heads (longest-processing-time first on the closed-form executed FLOP per head, "for each head
    h"); every rank holds only its heads' Q/K/V and runs select + sparse_attn on them.  No collective in the data path (an
    all-gather of O only if the consumer wants every head everywhere - not part of this path); the time of the layer is the MAX
    over ranks of the device time.  One JSON line, "scaling": "strong".  At N = 1 it is the whole layer on one GPU."""
    import torch
    import torch.distributed as dist
    import paper_2607_03612_b200 as sf
    from paper_2607_03612_b200 import sharding

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device(f"cuda:{local}"))
    torch.cuda.set_device(local)
    dev = torch.device(f"cuda:{local}")
    clocklog = ClockLog(local)
    peaks = load_peaks()
    sh = shape_for(args.config)
    L = make_layers(args.config, 1, args.gen, args.ratio)[0]
    full_shape = sf.make_shape(sh.S, sh.T, sh.H, sh.D, sh.B)
    costs = sharding.head_costs(full_shape, L.cfgs)              # closed form: every rank computes the same split, no communication
    parts = sharding.assign_heads(costs, world)
    mine = parts[rank]
    loads = [sum(costs[h] for h in p) for p in parts]
    ctx = sf.Context(local)
    stream = torch.cuda.current_stream()
    total_ms = 0.0
    launches = 0

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    step = None
    if mine:
        up = lambda x: torch.from_numpy(np.ascontiguousarray(x[mine]).view(np.int16)).to(dev).view(torch.bfloat16)
        q, k, v = up(L.q), up(L.k), up(L.v)
        cfgs = [L.cfgs[h] for h in mine]
        shape = sf.make_shape(sh.S, sh.T, len(mine), sh.D, sh.B)
        entries, ws_bytes = sf.query_sizes(shape, cfgs)
        lists = sf.Lists(torch.empty(len(mine) * sh.NB + 1, dtype=torch.int64, device=dev), torch.empty(max(entries, 1), dtype=torch.int32, device=dev))
        ws = torch.empty(ws_bytes, dtype=torch.uint8, device=dev)
        out = torch.empty_like(q)
        flush = torch.empty(256 << 20, dtype=torch.uint8, device=dev)   # one resident layer: flush the 126 MB L2 between steps

        def step():
            flush.zero_()
            ctx.select(q, k, shape, cfgs, workspace=ws, lists=lists)
            ctx.sparse_attn(q, k, v, shape, lists, out=out)
    for _ in range(args.warmup):
        if step:
            step()
    barrier()
    l0 = ctx.launch_count()
    with clocklog.region() as clk:
        barrier()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record(stream)
        for _ in range(args.steps):
            if step:
                step()
        e1.record(stream)
        barrier()
    launches = ctx.launch_count() - l0
    mine_ms = e0.elapsed_time(e1)
    if step:                                                      # the flush is not part of the layer: time it alone and subtract
        f0, f1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        f0.record(stream)
        for _ in range(args.steps):
            flush.zero_()
        f1.record(stream)
        torch.cuda.synchronize()
        mine_ms -= f0.elapsed_time(f1)
    total_ms = sharding.max_over_ranks(mine_ms, dev)
    if rank == 0:
        ms = total_ms / args.steps
        print(json.dumps({
            "metric": METRIC, "value": ms, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup, "ms_per_step": ms,
            "higher_is_better": False, "scaling": "strong", "vs_baseline": None, "dtype": "bf16", "data": "synthetic",
            "config": {"workload": workload_name(args.config, sh, args.gen, args.ratio), "parallelism": f"head-parallel x{world} (LPT by executed FLOP)",
                       "l2": "one resident layer per rank, 256 MB L2 flush between timed steps (its time measured alone and subtracted)"},
            "gpu_launches": int(launches), "heads_by_rank": parts, "executed_flop_by_rank": loads,
            "lpt_imbalance_max_over_mean": (max(loads) / (sum(loads) / world)) if sum(loads) else None,
            "executed_tflops_whole_job": sum(loads) / (ms * 1e-3) / 1e12,
            "roofline": {"bound": "tensor", "achieved": max(loads) / (ms * 1e-3) / 1e12, "peak": peaks["tflops_sustained"], "unit": "TFLOP/s",
                         "frac": max(loads) / (ms * 1e-3) / 1e12 / peaks["tflops_sustained"], "traffic": None,
                         "note": "the slowest rank's executed FLOP over the max-over-ranks layer time (includes its select)"},
            "clocks": clk.summary(),
            "note": "no data-path collective; the only communication is the barrier and the MAX all-reduce of the timing"}))
    clocklog.close()
    if world > 1:
        dist.destroy_process_group()


def run_stack(args):
    """the whole global-attention stack (default 24 layers) with the per-sequence index
    cache and as one CUDA graph.  Prints one JSON line (an extra, not the contract line)."""
    import torch
    import paper_2607_03612_b200 as sf
    from paper_2607_03612_b200.stack import GlobalStack, cached_cfgs
    dev = torch.device("cuda:0")
    torch.cuda.set_device(0)
    sh = shape_for(args.config)
    ctx = sf.Context(0)
    shape = sf.make_shape(sh.S, sh.T, sh.H, sh.D, sh.B)
    n_res = min(args.resident_layers, args.layers)
    res = [sy.config_c3_layer(l, sh=sh) for l in range(n_res)]          # resident Q/K/V sets (each >> L2), cycled
    up = lambda x: torch.from_numpy(x.view(np.int16)).to(dev).view(torch.bfloat16)
    qkv_res = [(up(L.q), up(L.k), up(L.v)) for L in res]
    out_res = [torch.empty_like(q) for q, _, _ in qkv_res]
    # per-layer rules: the C3 recipe; the stack with a cache turns the same-position heads into CACHED heads
    cache_cfgs = [sy.cfg(type=sy.HEAD_BLOCK_TOPK, topk_scope=sy.SCOPE_PER_FRAME, topk_per_frame=1, score_mode=sy.SCORE_COSINE),
                  sy.cfg(type=sy.HEAD_BLOCK_TOPK, topk_scope=sy.SCOPE_GLOBAL, keep_blocks=max(1, round(0.1 * sh.NB)),
                         score_mode=sy.SCORE_COSINE)]
    plain, cached = [], []
    for l in range(args.layers):
        gens = res[l % n_res].gens                                       # head types follow the resident data
        _, cfgs, _ = sy.stack_layer_heads(sh, l % n_res)
        plain.append(cfgs)
        cached.append(cached_cfgs(cfgs, cache_cfgs, {h: h % 2 for h, g in enumerate(gens) if g == sy.GEN_SAME_POSITION}))
    feat = up(np.stack([sy.make_features(sh, seed=77)] * 2))
    qkv = [qkv_res[l % n_res] for l in range(args.layers)]
    out = [out_res[l % n_res] for l in range(args.layers)]

    def timed(fn, reps):
        fn()
        torch.cuda.synchronize()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        for _ in range(reps):
            fn()
        e1.record()
        torch.cuda.synchronize()
        return e0.elapsed_time(e1) / reps

    def select_only_graph(st):
        """The stack's select calls alone, captured as a CUDA graph, so that the GPU time is measured and not the host time of
        24 back-to-back Python calls (select is far shorter than a host call sequence when no attention kernel hides it)."""
        n_cache = len(st.cache_cfgs) if st.cache_cfgs else 0
        side = torch.cuda.Stream()

        def go():
            for (q, k, v), cfgs, lists in zip(st.qkv, st.layer_cfgs, st.lists):
                ctx.select(q, k, shape, cfgs, workspace=st.ws, lists=lists, cache=st.cache, cache_heads=n_cache, stream=side)
        side.wait_stream(torch.cuda.current_stream())
        with torch.cuda.stream(side):
            go()
        torch.cuda.synchronize()
        g = torch.cuda.CUDAGraph()
        with torch.cuda.graph(g, stream=side):
            go()
        return g

    res_out = {}
    st0 = GlobalStack(ctx, shape, plain)
    st0.bind(qkv, out)
    res_out["eager_no_cache_ms"] = timed(st0.run, args.steps)
    g0 = select_only_graph(st0)
    res_out["select_no_cache_ms_per_layer"] = timed(g0.replay, args.steps) / args.layers
    pairs0 = sum(sf.query_sizes(shape, c)[0] for c in plain)
    del g0, st0
    st1 = GlobalStack(ctx, shape, cached, cache_cfgs)
    st1.bind(qkv, out)
    res_out["cache_build_ms"] = timed(lambda: st1.build_cache(feat), args.steps)
    res_out["eager_cached_ms"] = timed(st1.run, args.steps)
    g1 = select_only_graph(st1)
    res_out["select_cached_ms_per_layer"] = timed(g1.replay, args.steps) / args.layers
    st1.capture()
    res_out["graph_cached_ms"] = timed(st1.replay, args.steps)
    pairs1 = sum(sf.query_sizes(shape, c)[0] for c in cached)
    flop = lambda p: 4.0 * sh.B * sh.B * sh.D * p
    print(json.dumps({
        "metric": "global_attn_stack_ms", "unit": "ms/stack", "value": res_out["graph_cached_ms"], "n_gpus": 1, "steps": args.steps,
        "layers": args.layers, "data": "synthetic", "dtype": "bf16",
        "config": {"workload": f"{args.config.upper()} stack: {args.layers} global layers, S={sh.S}, N={sh.N}, H={sh.H}, block {sh.B}; "
                               f"{n_res} resident Q/K/V sets cycled; index cache = 2 rules (per-frame top-1, global 10 %) on synthetic features"},
        **res_out,
        "kept_pair_ratio_no_cache": pairs0 / (args.layers * sh.H * sh.NB * sh.NB),
        "kept_pair_ratio_cached": pairs1 / (args.layers * sh.H * sh.NB * sh.NB),
        "executed_tflops_no_cache_incl_select": flop(pairs0) / (res_out["eager_no_cache_ms"] * 1e-3) / 1e12,
        "executed_tflops_graph_cached_incl_select": flop(pairs1) / (res_out["graph_cached_ms"] * 1e-3) / 1e12,
    }))


def run_token(args):
    """the paper's token-level uniform stride and query-probe top-K kernels on one layer; one JSON line each
    (an extra, not the contract line)."""
    import torch
    import paper_2607_03612_b200 as sf
    dev = torch.device("cuda:0")
    sh = shape_for(args.config)
    ctx = sf.Context(0)
    shape = sf.make_shape(sh.S, sh.T, sh.H, sh.D, sh.B)
    L = sy.config_c3_layer(0, sh=sh)
    up = lambda x: torch.from_numpy(x.view(np.int16)).to(dev).view(torch.bfloat16)
    q, k, v = up(L.q), up(L.k), up(L.v)
    out = torch.empty_like(q)
    flush = torch.empty(256 << 20, dtype=torch.uint8, device=dev)

    def timed(fn, reps):
        fn()
        torch.cuda.synchronize()
        ts = []
        for _ in range(reps):
            flush.zero_()                                           # L2 flush between timed iterations
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record()
            fn()
            e1.record()
            torch.cuda.synchronize()
            ts.append(e0.elapsed_time(e1))
        return float(np.mean(ts))

    peaks = load_peaks()
    dense_ms = timed(lambda: ctx.dense_attn(q, k, v, shape, out=out), 2)
    lines = []
    for s in args.strides:
        n_kv = -(-sh.N // s)
        ms = timed(lambda: ctx.token_stride_attn(q, k, v, shape, s, 0, out=out), args.steps)
        tf = 4.0 * sh.N * (-(-n_kv // sh.B) * sh.B) * sh.D * sh.H / (ms * 1e-3) / 1e12
        lines.append({"variant": f"token stride s={s}", "kept_keys": n_kv / sh.N, "ms": ms, "executed_tflops": tf,
                      "frac_of_sustained_peak": tf / peaks["tflops_sustained"], "speedup_vs_own_dense": dense_ms / ms})
    for K in args.topks:
        sel_ws, att_ws = sf.token_query_sizes(shape, K)
        ws1 = torch.empty(sel_ws, dtype=torch.uint8, device=dev)
        ws2 = torch.empty(att_ws, dtype=torch.uint8, device=dev)
        idx = torch.empty((sh.H, K), dtype=torch.int32, device=dev)
        sel = timed(lambda: ctx.token_probe_select(q, k, shape, K, workspace=ws1, idx=idx), args.steps)
        att = timed(lambda: ctx.token_set_attn(q, k, v, shape, idx, workspace=ws2, out=out), args.steps)
        tf = 4.0 * sh.N * (-(-K // sh.B) * sh.B) * sh.D * sh.H / (att * 1e-3) / 1e12
        sel_gbs = 2.0 * sh.H * sh.N * sh.D * 2 / (sel * 1e-3) / 1e9  # Q once (qbar) + K once (probe)
        lines.append({"variant": f"token query-probe top-K K={K}", "kept_keys": K / sh.N, "select_ms": sel, "attn_ms": att,
                      "ms": sel + att, "executed_tflops": tf, "frac_of_sustained_peak": tf / peaks["tflops_sustained"],
                      "select_gbs": sel_gbs, "select_frac_of_hbm_peak": sel_gbs / peaks["hbm_gbs"],
                      "speedup_vs_own_dense": dense_ms / (sel + att)})
    print(json.dumps({"metric": "token_variant_layer_ms", "unit": "ms/layer", "data": "synthetic", "dtype": "bf16", "n_gpus": 1,
                      "steps": args.steps, "config": {"workload": workload_name(args.config, sh), "l2": "256 MB flush between timed iterations"},
                      "dense_attn_ms": dense_ms, "variants": lines}))


def run_tokenwise(args):
    """the paper's token-wise DINO Top-K kernel on one layer: per-sequence
    index computation (cosine similarity on the tensor cores + per-frame top-K), the per-q-tile union / mask structure, and the
    gathered, masked attention.  One JSON line (an extra, not the contract line)."""
    import torch
    import paper_2607_03612_b200 as sf
    dev = torch.device("cuda:0")
    sh = shape_for(args.config)
    ctx = sf.Context(0)
    shape = sf.make_shape(sh.S, sh.T, sh.H, sh.D, sh.B)
    gens, cfgs = sy.mixed_heads(sh)
    L = sy.make_layer(sh, gens, cfgs, seed=7000)
    up = lambda x: torch.from_numpy(x.view(np.int16)).to(dev).view(torch.bfloat16)
    q, k, v = up(L.q), up(L.k), up(L.v)
    feat = up(sy.make_features(sh, seed=7001))
    out = torch.empty_like(q)
    flush = torch.empty(256 << 20, dtype=torch.uint8, device=dev)
    peaks = load_peaks()

    def timed(fn, reps):
        fn()
        torch.cuda.synchronize()
        ts = []
        for _ in range(reps):
            flush.zero_()
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record()
            fn()
            e1.record()
            torch.cuda.synchronize()
            ts.append(e0.elapsed_time(e1))
        return float(np.mean(ts))

    dense_ms = timed(lambda: ctx.dense_attn(q, k, v, shape, out=out), 2)
    lines = []
    for K in args.topks:
        ws_bytes, _, _ = sf.token_topk_query_sizes(shape, K)
        ws = torch.empty(ws_bytes, dtype=torch.uint8, device=dev)
        idx = torch.empty((sh.N, sh.S, K), dtype=torch.int32, device=dev)
        sel_ms = timed(lambda: ctx.token_topk_select(feat, shape, K, workspace=ws, idx=idx), max(1, args.steps // 2))
        t0 = time.perf_counter()
        lists = ctx.token_lists_build(shape, idx)
        torch.cuda.synchronize()
        build_ms = (time.perf_counter() - t0) * 1e3
        att_ms = timed(lambda: ctx.token_lists_attn(q, k, v, shape, lists, out=out), args.steps)
        tf = 4.0 * sh.B * sh.B * sh.D * lists.tiles * sh.H / (att_ms * 1e-3) / 1e12
        lines.append({"K_per_frame": K, "kept_keys": K / sh.T, "index_select_ms_per_sequence": sel_ms, "lists_build_ms_per_sequence": build_ms,
                      "attn_ms": att_ms, "executed_tflops": tf, "frac_of_sustained_peak": tf / peaks["tflops_sustained"],
                      "union_tiles": lists.tiles, "union_tiles_over_dense_tiles": lists.tiles / (sh.NB * sh.NB),
                      "useful_pairs_over_executed": (sh.N * sh.S * K) / (lists.tiles * sh.B * sh.B),
                      "speedup_vs_own_dense": dense_ms / att_ms,
                      "index_bytes": int(idx.numel() * 4), "lists_bytes": int(lists.key_idx.numel() * 4 + lists.mask.numel() * 4)})
        del ws, idx, lists
    print(json.dumps({"metric": "tokenwise_topk_layer_ms", "unit": "ms/layer", "data": "synthetic", "dtype": "bf16", "n_gpus": 1,
                      "steps": args.steps, "config": {"workload": workload_name(args.config, sh) + "; every head attends per-query token lists (token-wise DINO Top-K, synthetic features)",
                                                      "l2": "256 MB flush between timed iterations"},
                      "dense_attn_ms": dense_ms, "variants": lines}))


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=24)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", default="c3", choices=["c2", "c3", "c4", "c5"])
    ap.add_argument("--resident-layers", type=int, default=4)
    ap.add_argument("--gen", default=None, choices=[sy.GEN_UNIFORM, sy.GEN_SAME_POSITION, sy.GEN_SINK],
                    help="sparsity sweep (C4): all heads of this generator type")
    ap.add_argument("--ratio", type=float, default=None, help="sparsity sweep: kept-block ratio, e.g. 0.10")
    ap.add_argument("--dense-reps", type=int, default=2)
    ap.add_argument("--skip-dense", action="store_true")
    ap.add_argument("--skip-e2e", action="store_true")
    ap.add_argument("--skip-cpu", action="store_true")
    ap.add_argument("--skip-s500", action="store_true", help="skip the bounded 500-frame (C5) point of the default run")
    ap.add_argument("--skip-configs", action="store_true", help="skip the C2 point and the C4 sweep of the default run (`configs` key)")
    ap.add_argument("--skip-profiled", action="store_true", help="skip the C3 point with budgets chosen by the offline search")
    ap.add_argument("--shard", default="layers", choices=["layers", "heads"],
                    help="N ranks: independent layers per rank (weak scaling, default) or the heads of ONE layer split over the ranks (strong)")
    ap.add_argument("--stack", action="store_true", help="time the whole stack with the index cache and as one CUDA graph")
    ap.add_argument("--layers", type=int, default=24)
    ap.add_argument("--token", action="store_true", help="time the token-granular variants (NEXT-2) on one layer")
    ap.add_argument("--strides", type=int, nargs="*", default=[8, 32, 64])
    ap.add_argument("--topks", type=int, nargs="*", default=None)
    ap.add_argument("--tokenwise", action="store_true", help="time the token-wise per-frame Top-K kernel (NEXT-2 iii) on one layer")
    args = ap.parse_args()
    if args.topks is None:
        args.topks = [16, 64] if args.tokenwise else [1024, 4096, 16384]
    if args.tokenwise:
        run_tokenwise(args)
    elif args.token:
        run_token(args)
    elif args.stack:
        run_stack(args)
    elif args.impl == "reference":
        run_reference(args)
    elif args.shard == "heads":
        run_head_parallel(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
