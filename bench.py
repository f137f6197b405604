#!/usr/bin/env python
"""bench.py -- routed-expert FFN tokens/s and % of roofline vs pruning budget on B200 (BASELINE.json metric).

    python bench.py [--gpus N] [--steps K] [--warmup W]              our arm (C-ABI library, CUDA kernels)
    python bench.py --impl reference [--steps K] [--warmup W]        the CPU oracle, timed on the host cores
    python bench.py --config C2 --T 4096 --r 704                     another workload (C2/C3/C4/C5, any T, any table)

A "step" is one fxm_moe_ffn call (route -> grouped GEMM-1 with the token gather, SwiGLU and
Y <- 0 fused -> grouped GEMM-2 with the router-weight scale and the scatter-add fused -> finalize) over one batch of
synthetic tokens.  Default workload = the largest single-GPU configuration of BASELINE.json: configs[3], the
Qwen2-57B-A14B-shaped layer (d=3584, E=64, top-8, I=2560), T=8192, 0 % pruned (uniform r_e=2560).  The same run adds
  "budget_sweep": 0/25/40/50/75 % pruned (uniform and heterogeneous nested tables) x T in {1, 64, 8192},
  "switch":       a short C5 loop (interleaved T=32 / T=4096 steps, a different nested table every step),
  "roofline", "cpu_baseline", "e2e", "clocks" as the contract asks.
N>1 = independent replicas of the layer, tokens sharded across ranks (weak scaling, no data-path collective; DESIGN.md
"Multi-GPU"); the sweep / switch / cpu_baseline legs run at N=1 only.  Prints ONE JSON line on rank 0.
"""
from __future__ import annotations

import argparse
import json
import os
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import numpy as np

METRIC = "routed_expert_ffn_tokens_per_s"
UNIT = "tokens/s"
FALLBACK_PEAKS = {"hbm_gbs": 6650.0, "bf16_tflops": 1590.0, "bf16_tflops_sustained": 1400.0}
DEFAULTS = {"config": "C4", "T": 8192, "r": "2560"}
SWEEP_T = (8192, 64, 1)
SWEEP_TABLES = [("U0", 2560), ("U25", 1920), ("U40", 1536), ("U50", 1280), ("U75", 640),
                ("H0", "hetero:0"), ("H25", "hetero:1"), ("H40", "hetero:2"), ("H50", "hetero:3"), ("H75", "hetero:4")]


def load_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    try:
        with open(p) as f:
            d = json.load(f)
        return {"hbm_gbs": float(d["hbm_gbs"]), "bf16_tflops": float(d["bf16_tflops"]),
                "bf16_tflops_sustained": float(d.get("bf16_tflops_sustained", d["bf16_tflops"])),
                "source": "measured (MEASURED_PEAKS.json)"}
    except Exception:
        return dict(FALLBACK_PEAKS, source="fallback (B200_PROFILING.md)")


# ------------------------------------------------------------------------------------------ ncu traffic of the dominant kernel
NCU_CAPTURES = {  # (config, T, table spec) -> committed extract of an `ncu --set full` capture of exactly that workload
    ("C4", 8192, "2560"): "profiles/r02d_ncu_full_pair_c4_T8192_r2560.csv",
}
NCU_KERNEL = {"gemm1_swiglu": "k_gemm_pair<1>", "gemm2_scatter_add": "k_gemm_pair<2>", "decode_fused": "k_decode"}


def ncu_traffic(cfg, T, spec, kernel):
    """dram__bytes_read.sum + dram__bytes_write.sum per launch of `kernel`, from the committed ncu extract of THIS workload
    (profiles/, the command that made it is in the README beside it); None when there is no capture of this workload."""
    path = NCU_CAPTURES.get((cfg, int(T), str(spec)))
    if not path or kernel not in NCU_KERNEL:
        return None, None
    try:
        import csv
        with open(os.path.join(ROOT, path)) as f:
            rows = list(csv.reader(f))
        hdr, units = rows[0], rows[1]
        scale = {"byte": 1.0, "Kbyte": 1e3, "Mbyte": 1e6, "Gbyte": 1e9}
        ir, iw = hdr.index("dram__bytes_read.sum"), hdr.index("dram__bytes_write.sum")
        for r in rows[2:]:
            if NCU_KERNEL[kernel] in r[0]:
                return float(r[ir]) * scale[units[ir]] + float(r[iw]) * scale[units[iw]], path
    except Exception:
        pass
    return None, None


# ------------------------------------------------------------------------------------------ work model
def work_model(ids: np.ndarray, r: np.ndarray, d: int, T: int, k: int):
    """Algorithmic work of one call, exactly SURVEY.md 8(d): S = sum_e n_e r_e, R_act = sum over experts with n_e > 0 of
    r_e.  FLOPs = 6 d S (gate 2 + up 2 + down 2 per token-channel-feature); bytes = every retained weight of an active
    expert once (6 d R_act) + x + y (4 T d) + ids/weights (8 A).  NOT counted (implementation traffic): the H round
    trip, the fp32 accumulator of y.  Per kernel: GEMM-1 = 4 d S flops, gate/up weights + x; GEMM-2 = 2 d S flops, down
    weights + y."""
    n = np.bincount(ids.ravel(), minlength=r.size).astype(np.int64)
    S = int((n * r.astype(np.int64)).sum())
    R_act = int(r.astype(np.int64)[n > 0].sum())
    A = T * k
    return {
        "S": S, "R_act": R_act,
        "flops": 6.0 * d * S, "bytes": 6.0 * d * R_act + 4.0 * T * d + 8.0 * A,
        "gemm1_flops": 4.0 * d * S, "gemm1_bytes": 4.0 * d * R_act + 2.0 * T * d + 4.0 * A,
        "gemm2_flops": 2.0 * d * S, "gemm2_bytes": 2.0 * d * R_act + 2.0 * T * d + 4.0 * A,
    }


def roof_time_s(flops, nbytes, peaks, tf_key="bf16_tflops"):
    """bound = the larger of the two floors"""
    t_tc = flops / (peaks[tf_key] * 1e12)
    t_hbm = nbytes / (peaks["hbm_gbs"] * 1e9)
    return (t_tc, "tensor") if t_tc >= t_hbm else (t_hbm, "hbm")


# ------------------------------------------------------------------------------------------ clocks
class ClockSampler:
    """Polls NVML (SM clock, power, clock-event reasons) from a thread while the timed regions run."""
    REASONS = {0x4: "sw_power_cap", 0x8: "hw_slowdown", 0x20: "sw_thermal_slowdown", 0x40: "hw_thermal_slowdown",
               0x80: "hw_power_brake_slowdown", 0x2: "applications_clocks_setting", 0x10: "sync_boost"}

    def __init__(self, index: int):
        self.samples = []
        self.max_mhz = None
        self._stop = threading.Event()
        self._thr = None
        self._h = None
        try:
            import pynvml
            pynvml.nvmlInit()
            vis = os.environ.get("CUDA_VISIBLE_DEVICES")
            phys = int(vis.split(",")[index]) if vis and vis.split(",")[index].isdigit() else index
            self._nv = pynvml
            self._h = pynvml.nvmlDeviceGetHandleByIndex(phys)
            self.max_mhz = int(pynvml.nvmlDeviceGetMaxClockInfo(self._h, pynvml.NVML_CLOCK_SM))
        except Exception:
            self._h = None

    def _poll(self):
        nv = self._nv
        while not self._stop.is_set():
            try:
                mhz = int(nv.nvmlDeviceGetClockInfo(self._h, nv.NVML_CLOCK_SM))
                try:
                    rs = int(nv.nvmlDeviceGetCurrentClocksEventReasons(self._h))
                except Exception:
                    rs = int(nv.nvmlDeviceGetCurrentClocksThrottleReasons(self._h))
                pw = nv.nvmlDeviceGetPowerUsage(self._h) / 1000.0
                self.samples.append((time.perf_counter(), mhz, rs, pw))
            except Exception:
                pass
            time.sleep(0.002)

    def start(self):
        if self._h is not None:
            self._thr = threading.Thread(target=self._poll, daemon=True)
            self._thr.start()

    def stop(self):
        self._stop.set()
        if self._thr is not None:
            self._thr.join()

    def summary(self, windows, brief=False):
        """windows: list of (t0, t1) perf_counter intervals during which the GPU was under load."""
        if self._h is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvml_unavailable"], "samples": 0}
        sel = [s for s in self.samples if any(a <= s[0] <= b for a, b in windows)]
        if not sel:          # region shorter than one poll: take the samples closest to it
            mid = sum(a + b for a, b in windows) / (2 * len(windows))
            sel = sorted(self.samples, key=lambda s: abs(s[0] - mid))[:3]
        bits = 0
        for s in sel:
            bits |= s[2]
        reasons = [n for b, n in self.REASONS.items() if bits & b]
        out = {"sm_mhz": float(np.median([s[1] for s in sel])) if sel else None, "sm_max_mhz": self.max_mhz,
               "reasons": reasons, "samples": len(sel)}
        if not brief:
            out["power_w_max"] = round(max(s[3] for s in sel), 1) if sel else None
        return out


# ------------------------------------------------------------------------------------------ workload
def make_table(gen, sh, spec, rng):
    """spec: an int width (uniform), 'full', 'hetero:<b>' (C4 nested-descent table b), 'fig6', 'mean60' (C3) or 'c1'."""
    if isinstance(spec, (int, np.integer)) or str(spec).isdigit():
        return gen.table_uniform(sh, int(spec))
    if spec == "full":
        return gen.table_uniform(sh, sh.I)
    if spec == "c1":
        return gen.table_c1(sh, rng)
    if spec == "mean60":
        return gen.table_mean_ratio(sh, rng, 0.6)
    if spec == "fig6":
        return gen.table_fig6_like(sh, rng)
    if str(spec).startswith("hetero:"):
        return gen.tables_nested_descent(sh, np.random.default_rng([0, 3]))[int(spec.split(":")[1])]
    raise SystemExit(f"unknown table spec {spec!r}")


def workload_string(cfg, sh, T, spec, r):
    """Identical for both arms (the driver compares the strings)."""
    return (f"{cfg} {sh.name}: d={sh.d} E={sh.E} top-{sh.k} I={sh.I} T={T} per GPU, table {spec} "
            f"(rho={1 - float(r.mean()) / sh.I:.3f} pruned)")


def rank_seed0(rank: int) -> int:
    """First batch seed of a rank: ranks are replicas of the layer that see disjoint seeded token batches."""
    return 1000 * rank


def aggregate(ms_list, T, steps, world, dist=None, device="cpu"):
    """Whole-job numbers from per-rank device times: every timed region takes the MAX over ranks (all_reduce MAX
    when `dist` is an initialised torch.distributed module), tokens are summed over ranks (weak scaling: T per rank).
    Returns (list of max times in ms, total tokens)."""
    if dist is not None and world > 1:
        import torch
        t = torch.tensor(list(ms_list), dtype=torch.float64, device=device)
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        ms_list = [float(v) for v in t]
    return list(ms_list), world * T * steps


def host_batches(gen, cfg, T, n, seed0):
    """n seeded batches (x, ids, w) of a named config; batch i uses seed seed0+i."""
    out = []
    for i in range(n):
        _, b, rng = gen.config(cfg, T=T, seed=seed0 + i, layer=False)
        out.append((b, rng))
    return out


def to_device(fx, torch, hb):
    return [(fx.bf16_from_bits(b.x), torch.from_numpy(b.topk_ids).cuda(), torch.from_numpy(b.topk_w).cuda()) for b, _ in hb]


# ------------------------------------------------------------------------------------------ budget sweep (N=1)
def sweep_point(torch, L, dev, y, iters, warm, flush_buf):
    """Median device time of one call (CUDA events on the launching stream around every call).  With flush_buf, a buffer
    larger than L2 is rewritten before every call so the weights never come from L2 (decode points)."""
    st = torch.cuda.current_stream()
    for i in range(warm):
        L.moe_ffn(*dev[i % len(dev)], out=y)
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(iters)]
    for i in range(iters):
        if flush_buf is not None:
            flush_buf.add_(1)
        ev[i][0].record(st)
        L.moe_ffn(*dev[i % len(dev)], out=y)
        ev[i][1].record(st)
    torch.cuda.synchronize()
    return np.array([a.elapsed_time(b) for a, b in ev])


def disjoint_decode_batches(torch, fx, gen, cfg, sh, seed):
    """T=1 batches for the back-to-back decode loop: batch i routes its token to experts perm[i*k:(i+1)*k] of a seeded
    permutation, so consecutive calls stream DIFFERENT experts' weights ("rotate over >= 8 routing
    batches that touch different experts"); x and the router weights come from the usual generator."""
    perm = np.random.default_rng([seed, 7]).permutation(sh.E)
    out = []
    for i in range(sh.E // sh.k):
        _, b, _ = gen.config(cfg, T=1, seed=seed + i, layer=False)
        ids = perm[i * sh.k:(i + 1) * sh.k].astype(np.int32).reshape(1, sh.k)
        out.append((ids, (fx.bf16_from_bits(b.x), torch.from_numpy(ids).cuda(), torch.from_numpy(b.topk_w).cuda())))
    return out


def pipelined_point(torch, L, dev, y, rounds):
    """Per-call time of `rounds` x len(dev) calls enqueued back to back (no flush, no event between calls): what a decode
    loop of a served model pays per layer -- launch latency and prologue of call i+1 overlap the tail of call i."""
    st = torch.cuda.current_stream()
    for d in dev:
        L.moe_ffn(*d, out=y)
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    torch.cuda.synchronize()
    e0.record(st)
    for _ in range(rounds):
        for d in dev:
            L.moe_ffn(*d, out=y)
    e1.record(st)
    torch.cuda.synchronize()
    return e0.elapsed_time(e1) / (rounds * len(dev))


def run_budget_sweep(torch, fx, gen, L, cfg, sh, peaks, sampler):
    """BASELINE.json metric "vs pruning budget": every budget of configs[3] x T in {8192, 64, 1}."""
    flush_buf = torch.zeros(512 << 20, dtype=torch.uint8, device="cuda")
    rows, base = [], {}
    for T in SWEEP_T:
        NB = 4 if T >= 1024 else 8
        hb = host_batches(gen, cfg, T, NB, 500)
        dev = to_device(fx, torch, hb)
        y = torch.empty((T, sh.d), dtype=torch.bfloat16, device="cuda")
        dj = disjoint_decode_batches(torch, fx, gen, cfg, sh, 700) if T == 1 else None
        for label, spec in SWEEP_TABLES:
            r = make_table(gen, sh, spec, None)
            L.set_budget(r)
            iters = 12 if T >= 1024 else 60
            if T >= 1024:
                time.sleep(0.4)      # every prefill point starts from an idle GPU: 12 calls fit before the 1 kW power cap bites
            w0 = time.perf_counter()
            ms = sweep_point(torch, L, dev, y, iters, 3, flush_buf if T <= 64 else None)
            w1 = time.perf_counter()
            wm = [work_model(b.topk_ids, r, sh.d, T, sh.k) for b, _ in hb]
            fl = float(np.mean([w["flops"] for w in wm]))
            by = float(np.mean([w["bytes"] for w in wm]))
            t_roof, bound = roof_time_s(fl, by, peaks)
            med = float(np.median(ms)) * 1e-3
            key = (T, label[0])
            if label in ("U0", "H0"):
                base[key] = med
            pipe = None
            if T <= 64:
                # back to back, no flush: T=64 streams every expert (0.9-3.5 GB per call, nothing survives in L2 until the
                # next call reaches it); T=1 rotates over E/k batches with disjoint expert sets
                pdev = [d for _, d in dj] if dj else dev
                pms = pipelined_point(torch, L, pdev, y, 8 if T == 1 else 4) * 1e-3
                pby = float(np.mean([work_model(i_, r, sh.d, T, sh.k)["bytes"] for i_, _ in dj])) if dj else by
                pipe = {"ms": round(pms * 1e3, 5), "tokens_per_s": round(T / pms, 1), "gbs": round(pby / pms / 1e9, 1),
                        "frac": round(pby / (peaks["hbm_gbs"] * 1e9) / pms, 4),
                        "how": ("calls enqueued back to back over %d batches with disjoint expert sets, no flush" % len(dj)) if dj
                               else "calls enqueued back to back over %d batches, no flush (every call streams all experts)" % len(dev)}
            rows.append({"T": T, "table": label, "rho": round(1 - float(r.mean()) / sh.I, 4), "back_to_back": pipe,
                         "ms": round(med * 1e3, 5), "tokens_per_s": round(T / med, 1),
                         "tflops": round(fl / med / 1e12, 2), "gbs": round(by / med / 1e9, 1), "bound": bound,
                         "t_roof_us": round(t_roof * 1e6, 2), "frac": round(t_roof / med, 4),
                         "speedup_vs_0pct": round(base[key] / med, 3) if key in base else None,
                         "launches": L.launches_per_ffn(),
                         "l2": "flushed before every call" if T <= 64 else "weights > L2",
                         "clocks": sampler.summary([(w0, w1)], brief=True)})
        del dev, y
    del flush_buf
    torch.cuda.empty_cache()
    return rows


# ------------------------------------------------------------------------------------------ C5: online budget switching (N=1)
def run_switch(torch, fx, gen, L, sh, steps, sampler):
    """BASELINE.json configs[4] in short: interleaved decode (T=32) / prefill (T=4096) steps on the resident layer, a
    different registered nested table every step (fxm_select_budget: host-only, no launch, no weight movement)."""
    tabs = gen.tables_nested_descent(sh, np.random.default_rng([0, 3]))
    L.register_budgets(tabs, require_nested=True)
    pools = {}
    for T in (32, 4096):
        pools[T] = to_device(fx, torch, host_batches(gen, "C5", T, 8, 0))
    ys = {T: torch.empty((T, sh.d), dtype=torch.bfloat16, device="cuda") for T in pools}
    L.workspace(4096, sh.k)
    rng = np.random.default_rng(5)
    seq, prev = [], -1
    for _ in range(steps):
        b = int(rng.integers(len(tabs)))
        while b == prev:
            b = int(rng.integers(len(tabs)))
        seq.append(b)
        prev = b
    st = torch.cuda.current_stream()

    def loop(switching):
        host_sel = 0.0
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        torch.cuda.synchronize()
        e0.record(st)
        for i, b in enumerate(seq):
            T = 32 if i % 2 == 0 else 4096
            if switching:
                t0 = time.perf_counter()
                L.select_budget(b)
                host_sel += time.perf_counter() - t0
            L.moe_ffn(*pools[T][(i // 2) % 8], out=ys[T])
        e1.record(st)
        torch.cuda.synchronize()
        return e0.elapsed_time(e1) * 1e-3, host_sel

    w0 = time.perf_counter()
    L.select_budget(2)
    loop(False)                                            # warm-up
    frozen = {}
    for b in range(len(tabs)):                             # the frozen-budget loops the switching loop is compared with
        L.select_budget(b)
        frozen[b] = loop(False)[0]
    t_sw, host_sel = loop(True)
    # what the switching loop should cost if a switch were free: every step at its own table's frozen per-step cost
    per_step = {}
    for b in range(len(tabs)):
        per_step[b] = frozen[b] / len(seq)
    expect = float(np.mean([frozen[b] for b in seq]))
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    torch.cuda.synchronize()
    t0 = time.perf_counter()
    e0.record(st)
    for b in seq:
        L.set_budget(tabs[b])
    e1.record(st)
    t_host_set = (time.perf_counter() - t0) / len(seq)
    torch.cuda.synchronize()
    w1 = time.perf_counter()
    t_dev_set = e0.elapsed_time(e1) * 1e-3 / len(seq)
    tokens = sum(32 if i % 2 == 0 else 4096 for i in range(len(seq)))
    return {"workload": f"C5: C4-shaped layer, {len(seq)} interleaved T=32 / T=4096 steps, 5 nested tables "
                        f"(rho={[round(1 - float(t.mean()) / sh.I, 3) for t in tabs]}), table switched every step",
            "sustained_tokens_per_s_switching": round(tokens / t_sw, 1),
            "loop_s_switching": round(t_sw, 5), "loop_s_expected_from_frozen_loops": round(expect, 5),
            "switch_cost_us_per_step_device": round((t_sw - expect) / len(seq) * 1e6, 3),
            "select_budget_host_us": round(host_sel / len(seq) * 1e6, 3),
            "set_budget_host_us": round(t_host_set * 1e6, 3), "set_budget_stream_us": round(t_dev_set * 1e6, 3),
            "frozen_loop_s": {str(b): round(v, 5) for b, v in frozen.items()},
            "weights_touched_by_switch_bytes": 0, "table_bytes": int(sh.E * 4),
            "clocks": sampler.summary([(w0, w1)], brief=True)}


# ------------------------------------------------------------------------------------------ SURVEY.md 8(f) rows (N=1)
def _median_ms(torch, fn, iters, warm=3):
    st = torch.cuda.current_stream()
    for _ in range(warm):
        fn()
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(iters)]
    for a_, b_ in ev:
        a_.record(st)
        fn()
        b_.record(st)
    torch.cuda.synchronize()
    return float(np.median([a_.elapsed_time(b_) for a_, b_ in ev]))


def run_next(torch, fx, gen, L, lay, cfg, sh, peaks):
    """The rows SURVEY.md 8(f) ranks after the hot path, timed on the same resident layer:
    offline clipping (export a fixed-budget blob, reload it, run the same kernels on it) against
    online clipping at the same budget; the router front end fused into the route launch (the router's
    output is the path's input); channel saliency + ranking (Eq. 2-3) as a streaming reduction."""
    out = {}
    hb = host_batches(gen, cfg, 8192, 2, 900)
    dev = to_device(fx, torch, hb)
    y = torch.empty((8192, sh.d), dtype=torch.bfloat16, device="cuda")
    hb64 = host_batches(gen, cfg, 64, 8, 910)
    dev64 = to_device(fx, torch, hb64)
    y64 = torch.empty((64, sh.d), dtype=torch.bfloat16, device="cuda")
    flush_buf = torch.zeros(512 << 20, dtype=torch.uint8, device="cuda")
    r = gen.table_uniform(sh, sh.I // 2)
    L.set_budget(r)
    it = [0]

    def call(layer, d_, y_, flush=False):
        def f():
            if flush:
                flush_buf.add_(1)
            layer.moe_ffn(*d_[it[0] % len(d_)], out=y_)
            it[0] += 1
        return f
    st = torch.cuda.current_stream()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    blob = L.export_clipped(r)                       # first call: the blob's cudaMalloc would sit between the two events
    torch.cuda.synchronize()
    del blob
    e0.record(st)
    blob = L.export_clipped(r)                       # same size: the block comes back from torch's caching allocator
    e1.record(st)
    torch.cuda.synchronize()
    C = fx.Layer.load_clipped(blob, sh.E, sh.d, sh.I, r)
    C.set_budget(r)
    time.sleep(0.4)
    on_p = _median_ms(torch, call(L, dev, y), 10)
    time.sleep(0.4)
    off_p = _median_ms(torch, call(C, dev, y), 10)
    # decode-sized calls: the flush kernel runs between the two events of a call, so time it alone and subtract
    fl = _median_ms(torch, lambda: flush_buf.add_(1), 20)
    on_d = _median_ms(torch, call(L, dev64, y64, True), 40) - fl
    off_d = _median_ms(torch, call(C, dev64, y64, True), 40) - fl
    out["offline_clipping"] = {
        "budget": f"uniform 50 % pruned (r_e = {sh.I // 2})", "blob_bytes": int(blob.numel()),
        "full_layer_bytes": int(fx.packed_bytes(sh.E, sh.d, sh.I)),
        "blob_over_full": round(blob.numel() / fx.packed_bytes(sh.E, sh.d, sh.I), 4),
        "export_ms": round(e0.elapsed_time(e1), 3),
        "export_gbs": round(2.0 * blob.numel() / (e0.elapsed_time(e1) * 1e-3) / 1e9, 1),   # blob read once + written once
        "T8192_ms": {"online": round(on_p, 4), "offline": round(off_p, 4)},
        "T64_ms_l2_flushed": {"online": round(on_d, 4), "offline": round(off_d, 4)},
        "note": "same kernels on both layouts (tiles are addressed through a per-expert block index); the paper's online path "
                "stays slower than its offline one because of slicing and dispatch (PAPER.md:239)"}
    del C, blob
    # router front end fused into the route launch
    L.set_budget(gen.table_uniform(sh, sh.I))
    logits = torch.from_numpy(np.random.default_rng(5).standard_normal((8192, sh.E)).astype(np.float32)).cuda()
    x0 = dev[0][0]
    time.sleep(0.4)
    t_ids = _median_ms(torch, call(L, dev, y), 10)
    time.sleep(0.4)
    t_log = _median_ms(torch, lambda: L.moe_ffn_router(x0, logits, sh.k, out=y), 10)
    out["router_front_end"] = {"T": 8192, "ms_with_given_topk": round(t_ids, 4), "ms_from_router_logits": round(t_log, 4),
                               "launches": L.launches_per_ffn()}
    del dev, dev64, y, y64, flush_buf, logits
    torch.cuda.empty_cache()
    # saliency + ranking on the C2-sized weight set (3 x 346 MB) with B = 2 synthetic gradient sets
    s2 = gen.SHAPES["C2"]
    B = 2
    g = torch.Generator(device="cuda")
    g.manual_seed(11)
    mk = lambda *shape: (torch.randn(*shape, device="cuda", dtype=torch.float32, generator=g) * 0.02).to(torch.bfloat16)
    Wg, Wu, Wd = mk(s2.E, s2.I, s2.d), mk(s2.E, s2.I, s2.d), mk(s2.E, s2.d, s2.I)
    Gg, Gu, Gd = mk(B, s2.E, s2.I, s2.d), mk(B, s2.E, s2.I, s2.d), mk(B, s2.E, s2.d, s2.I)
    t_sal = _median_ms(torch, lambda: fx.saliency(Wg, Wu, Wd, Gg, Gu, Gd), 10)
    sal = fx.saliency(Wg, Wu, Wd, Gg, Gu, Gd)
    t_rank = _median_ms(torch, lambda: fx.rank_channels(sal), 10)
    nbytes = (1 + B) * 6.0 * s2.E * s2.I * s2.d
    out["saliency_ranking"] = {"shape": "C2 weights (E=%d, I=%d, d=%d), B=%d gradient sets" % (s2.E, s2.I, s2.d, B),
                               "saliency_ms": round(t_sal, 4), "algorithmic_bytes": nbytes,
                               "gbs": round(nbytes / (t_sal * 1e-3) / 1e9, 1),
                               "frac_of_hbm_peak": round(nbytes / (t_sal * 1e-3) / 1e9 / peaks["hbm_gbs"], 4),
                               "rank_ms": round(t_rank, 4)}
    return out


# ------------------------------------------------------------------------------------------ our arm
def run_ours(args):
    import torch
    import torch.distributed as dist
    from paper_2606_27866_b200 import flexmoe as fx
    from paper_2606_27866_b200 import inputs as gen

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device (the product path has no CPU fallback)")
    torch.cuda.set_device(local)
    if world > 1:
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    fx.lib()                                        # fails loudly if libflexmoe.so is missing and cannot be built

    cfg, T = args.config.upper(), args.T
    sh = gen.SHAPES[cfg]
    peaks = load_peaks()
    NB = args.batches
    lay = gen.layer_for(cfg, 0)                      # same weights on every rank (replicas)
    hb = host_batches(gen, cfg, T, NB, rank_seed0(rank))  # each rank its own tokens
    r = make_table(gen, sh, args.r, hb[0][1])
    L = fx.Layer.pack(fx.bf16_from_bits(lay.W_gate), fx.bf16_from_bits(lay.W_up), fx.bf16_from_bits(lay.W_down),
                      lay.channel_rank)
    L.set_budget(r)
    torch.cuda.synchronize()
    if args.switch_only:
        # nothing but the C5 switching loop (for a profiler's launch list: which kernels and copies a budget switch costs)
        sampler = ClockSampler(local)
        sampler.start()
        out = {"switch": run_switch(torch, fx, gen, L, sh, args.switch_steps, sampler)}
        sampler.stop()
        assert L.device_flags() == 0
        print(json.dumps(out), flush=True)
        return
    if args.next_only:
        # nothing but the SURVEY.md 8(f) legs (for a profiler: the saliency / export / router kernels at bench size)
        out = {"next": run_next(torch, fx, gen, L, lay, cfg, sh, peaks)}
        assert L.device_flags() == 0
        print(json.dumps(out), flush=True)
        return
    dev = to_device(fx, torch, hb)
    y = torch.empty((T, sh.d), dtype=torch.bfloat16, device="cuda")
    stream = torch.cuda.current_stream()

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    # ---- warm-up (untimed)
    for i in range(args.warmup):
        L.moe_ffn(*dev[i % NB], out=y)
    barrier()
    flags = L.device_flags()
    assert flags == 0, f"device flags {flags:#x}"

    sampler = ClockSampler(local)
    sampler.start()
    # ---- timed region 1: EXACTLY K steps, inputs resident in HBM.  When a step streams more weight bytes than L2 holds
    #      twice over, nothing but the calls sits between the two events; a decode-sized step (its weights would stay in
    #      the 126 MB L2 between iterations) gets a buffer larger than L2 rewritten before every call and is timed
    #      call by call (CUDA events around every call, summed).
    wbytes = 6.0 * sh.d * float(np.mean([work_model(b.topk_ids, r, sh.d, T, sh.k)["R_act"] for b, _ in hb]))
    flush = wbytes < 2 * 126e6
    flush_buf = torch.zeros(512 << 20, dtype=torch.uint8, device="cuda") if flush else None
    barrier()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    w0 = time.perf_counter()
    if flush:
        evs = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(args.steps)]
        for i in range(args.steps):
            flush_buf.add_(1)
            evs[i][0].record(stream)
            L.moe_ffn(*dev[i % NB], out=y)
            evs[i][1].record(stream)
        barrier()
        ms_total = float(sum(a_.elapsed_time(b_) for a_, b_ in evs))
    else:
        e0.record(stream)
        for i in range(args.steps):
            L.moe_ffn(*dev[i % NB], out=y)
        e1.record(stream)
        barrier()
        ms_total = e0.elapsed_time(e1)
    w1 = time.perf_counter()
    del flush_buf
    launches = int(L.launches_per_ffn() * args.steps)
    # ---- the same K steps again with a CUDA event before every kernel (fxm_profile_begin/end): per-kernel device
    #      times for the roofline of the dominant kernel, measured live on the launching stream.  The events cost
    #      2-3 us each and serialise the programmatic dependent launches, which is why this pass is not the headline.
    L.profile_begin(args.steps)
    for i in range(args.steps):
        L.moe_ffn(*dev[i % NB], out=y)
    barrier()
    kern_ms, n_prof = L.profile_end()

    # ---- timed region 2: end to end through fxm_moe_ffn_host (pinned host buffers, H2D + D2H inside)
    hx = [(fx.bf16_from_bits(b.x, "cpu").pin_memory(), torch.from_numpy(b.topk_ids).pin_memory(),
           torch.from_numpy(b.topk_w).pin_memory()) for b, _ in hb]
    hys = [torch.empty((T, sh.d), dtype=torch.bfloat16).pin_memory() for _ in range(2)]
    for i in range(max(3, min(args.warmup, 5))):
        L.moe_ffn_host(*hx[i % NB], hys[i % 2], pipelined=True)
    L.host_flush()
    barrier()
    w2 = time.perf_counter()
    e0.record(stream)
    for i in range(args.steps):
        L.moe_ffn_host(*hx[i % NB], hys[i % 2], pipelined=True)
    L.host_flush()                                  # the stream waits for the y copies still in flight
    e1.record(stream)
    barrier()
    w3 = time.perf_counter()
    ms_e2e = e0.elapsed_time(e1)
    clocks = sampler.summary([(w0, w1), (w2, w3)])

    (ms_total, ms_e2e), tokens = aggregate([ms_total, ms_e2e], T, args.steps, world, dist if world > 1 else None, "cuda")
    value = tokens / (ms_total * 1e-3)
    e2e_value = tokens / (ms_e2e * 1e-3)
    wm = [work_model(b.topk_ids, r, sh.d, T, sh.k) for b, _ in hb]
    sel = [wm[i % NB] for i in range(args.steps)]
    mean = lambda key: float(np.mean([w[key] for w in sel]))

    # ---- roofline of the dominant kernel (largest share of the step) and of the whole step, SURVEY.md 8(d) work model
    per_launch_ms = {kname: v / max(n_prof, 1) for kname, v in kern_ms.items()}
    dom = max(per_launch_ms, key=per_launch_ms.get)
    kflops = {"gemm1_swiglu": mean("gemm1_flops"), "gemm2_scatter_add": mean("gemm2_flops"),
              "decode_fused": mean("flops")}.get(dom, 0.0)
    kbytes = {"gemm1_swiglu": mean("gemm1_bytes"), "gemm2_scatter_add": mean("gemm2_bytes")}.get(dom, mean("bytes"))
    t_roof, bound = roof_time_s(kflops, kbytes, peaks)
    dur = per_launch_ms[dom] * 1e-3
    if bound == "tensor":
        achieved, peak, unit = kflops / dur / 1e12, peaks["bf16_tflops"], "TFLOP/s"
    else:
        achieved, peak, unit = kbytes / dur / 1e9, peaks["hbm_gbs"], "GB/s"
    traffic, traffic_src = (args.traffic, "--traffic") if args.traffic is not None else ncu_traffic(cfg, T, args.r, dom)
    roofline = {"bound": bound, "achieved": round(achieved, 2), "peak": peak, "unit": unit,
                "frac": round(achieved / peak, 4),
                "traffic": traffic,                 # dram bytes per launch from an ncu --set full capture of THIS workload, else null
                "traffic_source": traffic_src,
                "kernel": dom, "kernel_ms": round(per_launch_ms[dom], 5),
                "kernel_share_of_step": round(per_launch_ms[dom] / max(sum(per_launch_ms.values()), 1e-12), 4),
                "peak_source": peaks["source"] + ", burst figure (the kernel is timed alone between CUDA events)",
                "frac_of_sustained": round(achieved / peaks["bf16_tflops_sustained"], 4) if bound == "tensor" else None,
                "algorithmic": {"flops": kflops, "bytes": kbytes,
                                "model": "SURVEY.md 8(d): weights of the kernel once + x (GEMM-1) or y (GEMM-2) + ids; no H, no accumulator traffic"}}
    step_roof, step_bound = roof_time_s(mean("flops"), mean("bytes"), peaks)
    step_s = ms_total * 1e-3 / args.steps
    roofline_step = {"bound": step_bound, "t_roof_us": round(step_roof * 1e6, 2), "t_step_us": round(step_s * 1e6, 2),
                     "frac": round(step_roof / step_s, 4),
                     "frac_of_sustained": round(roof_time_s(mean("flops"), mean("bytes"), peaks, "bf16_tflops_sustained")[0] / step_s, 4),
                     "tflops": round(mean("flops") / step_s / 1e12, 2), "gbs": round(mean("bytes") / step_s / 1e9, 1),
                     "kernel_ms_per_step": {kname: round(v, 5) for kname, v in per_launch_ms.items()}}

    out = {
        "metric": METRIC, "value": round(value, 1), "unit": UNIT, "n_gpus": world, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": round(ms_total / args.steps, 5), "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "bf16", "data": "synthetic",
        "config": {"workload": workload_string(cfg, sh, T, args.r, r),
                   "l2": (f"L2 flushed before every call (a 512 MB buffer is rewritten; the step streams only "
                          f"{wbytes / 1e6:.0f} MB of weights), each call timed with its own CUDA events" if flush else
                          f"inputs larger than L2: {wbytes / 1e6:.0f} MB of retained weights of active experts streamed "
                          f"per step, {NB} rotating token batches"),
                   "parallelism": f"replicas x{world}, tokens sharded, no data-path collective"},
        "e2e": {"value": round(e2e_value, 1), "unit": UNIT,
                "h2d_bytes_per_step": int(T * sh.d * 2 + 2 * T * sh.k * 4), "d2h_bytes_per_step": int(T * sh.d * 2),
                "ms_per_step": round(ms_e2e / args.steps, 5),
                "api": "fxm_moe_ffn_host_pipelined + fxm_host_flush (pinned host buffers; every step copies its x, ids, w in "
                       "and its y out inside the timed region; the input copy of step i+1 and the output copy of step i-1 "
                       "run on the library's side streams while step i computes; the flush is inside the region)"},
        "gpu_launches": launches,
        "clocks": clocks, "roofline": roofline, "roofline_step": roofline_step,
    }
    single = rank == 0 and world == 1
    if single and not args.no_sweep and cfg in ("C4", "C5"):
        out["budget_sweep"] = run_budget_sweep(torch, fx, gen, L, cfg, sh, peaks, sampler)
        out["switch"] = run_switch(torch, fx, gen, L, sh, args.switch_steps, sampler)
        out["next"] = run_next(torch, fx, gen, L, lay, cfg, sh, peaks)
        L.set_budget(r)
        assert L.device_flags() == 0
    sampler.stop()
    if single and not args.no_cpu_baseline:
        out["cpu_baseline"], out["parity_sample"] = cpu_baseline(gen, fx, lay, hb[0][0], r, L, dev[0], y, args.cpu_seconds)
    if world > 1:
        dist.barrier()
        dist.destroy_process_group()
    if rank == 0:
        print(json.dumps(out), flush=True)


# ------------------------------------------------------------------------------------------ CPU oracle legs
def _oracle_sample_rows(T, n, seed=7):
    return np.sort(np.random.default_rng(seed).choice(T, size=min(n, T), replace=False)).astype(np.int32)


def _time_oracle(oracle, b, packed, r, rows):
    t0 = time.perf_counter()
    ref = oracle.moe_ffn(b.x, *packed, r, b.topk_ids, b.topk_w, rows=rows)
    return time.perf_counter() - t0, ref


def _sample_size(T, cores, t_cal, n0, seconds, floor=512):
    """tokens of the bounded sample: about `seconds` of CPU work, at least `floor` (>= 512), at most T"""
    n = int((seconds / max(t_cal, 1e-6)) * n0)
    n = max(n, floor)
    n = min(T, max(cores, n // cores * cores))
    return n


def cpu_baseline(gen, fx, lay, b, r, L, dev0, y, seconds):
    """The oracle as it stands (oracle/oracle.c, fp64, OpenMP over tokens, gcc -O3 -march=native) timed on this box's
    host cores on a bounded token sample of the SAME workload; the same rows of the GPU output are compared with it."""
    import torch
    import oracle
    cores = oracle.threads()
    T = b.x.shape[0]
    packed = oracle.pack(lay.W_gate, lay.W_up, lay.W_down, lay.channel_rank)
    n0 = min(T, cores)
    t_cal, _ = _time_oracle(oracle, b, packed, r, _oracle_sample_rows(T, n0))
    n = _sample_size(T, cores, t_cal, n0, seconds)
    rows = _oracle_sample_rows(T, n)
    dt, ref = _time_oracle(oracle, b, packed, r, rows)
    L.moe_ffn(*dev0, out=y)
    torch.cuda.synchronize()
    yv = gen.bf16_bits_to_f32(fx.bf16_to_bits(y[torch.from_numpy(rows.astype(np.int64)).cuda()])).astype(np.float64)
    scale = float(np.abs(ref).max())
    parity = {"rows": int(rows.size), "max_err_over_max_ref": float(np.abs(yv - ref).max() / scale),
              "rel_l2": float(np.linalg.norm(yv - ref) / np.linalg.norm(ref)), "tol": {"max": 1e-2, "l2": 5e-3}}
    how = "all" if rows.size == T else "seeded random rows"
    return ({"value": round(rows.size / dt, 2), "unit": UNIT, "cores": cores, "kind": "oracle",
             "sample": f"{rows.size} of {T} tokens ({how}, full k and r_e), {dt:.1f} s wall, fp64, OpenMP over "
                       f"tokens, gcc -O3 -march=native"}, parity)


def run_reference(args):
    """--impl reference: the CPU oracle on the same config/metric; each step = a bounded token sample."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    import oracle
    from paper_2606_27866_b200 import inputs as gen
    cfg, T = args.config.upper(), args.T
    sh = gen.SHAPES[cfg]
    lay, b, rng = gen.config(cfg, T=T, seed=0)
    r = make_table(gen, sh, args.r, rng)
    cores = oracle.threads()
    packed = oracle.pack(lay.W_gate, lay.W_up, lay.W_down, lay.channel_rank)
    n0 = min(T, cores)
    t_cal, _ = _time_oracle(oracle, b, packed, r, _oracle_sample_rows(T, n0))
    budget_s = args.cpu_seconds * 6.0                      # whole run (warm-up + steps) ~ 1.5 min by default
    per_step = budget_s / (args.steps + args.warmup)
    n = _sample_size(T, cores, t_cal, n0, per_step, floor=cores)
    for i in range(args.warmup):
        _time_oracle(oracle, b, packed, r, _oracle_sample_rows(T, n, seed=100 + i))
    total = 0.0
    for i in range(args.steps):
        dt, _ = _time_oracle(oracle, b, packed, r, _oracle_sample_rows(T, n, seed=200 + i))
        total += dt
    value = n * args.steps / total
    sample = f"{n} of {T} tokens per step (seeded random rows), fp64, OpenMP over tokens, gcc -O3 -march=native"
    out = {"impl": "reference", "metric": METRIC, "value": round(value, 2), "unit": UNIT, "n_gpus": args.gpus,
           "steps": args.steps, "warmup": args.warmup, "ms_per_step": round(total / args.steps * 1e3, 3),
           "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
           "config": {"workload": workload_string(cfg, sh, T, args.r, r), "l2": "n/a (CPU)",
                      "parallelism": "host cores, rank 0 only"},
           "cpu_baseline": {"value": round(value, 2), "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
           "e2e": {"value": round(value, 2), "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
           "gpu_launches": 0}
    print(json.dumps(out), flush=True)


# ------------------------------------------------------------------------------------------ main
def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=50)
    ap.add_argument("--warmup", type=int, default=10)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", default=DEFAULTS["config"])
    ap.add_argument("--T", type=int, default=DEFAULTS["T"])
    ap.add_argument("--r", default=str(DEFAULTS["r"]), help="uniform width, 'full', 'hetero:<b>', 'fig6', 'mean60', 'c1'")
    ap.add_argument("--batches", type=int, default=4, help="rotating pre-generated token batches")
    ap.add_argument("--cpu-seconds", type=float, default=15.0, help="CPU work of the cpu_baseline sample")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-sweep", action="store_true", help="skip the budget_sweep and switch legs")
    ap.add_argument("--switch-steps", type=int, default=200)
    ap.add_argument("--switch-only", action="store_true", help="run only the C5 switching loop (N=1) and print its record")
    ap.add_argument("--next-only", action="store_true", help="run only the SURVEY.md 8(f) legs (N=1) and print their record")
    ap.add_argument("--traffic", type=float, default=None,
                    help="dram bytes per launch of the dominant kernel from an ncu --set full capture of this config (else null)")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3) if args.impl == "ours" else args.warmup
    if args.impl == "reference":
        return run_reference(args)
    return run_ours(args)


if __name__ == "__main__":
    main()
