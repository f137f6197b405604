"""Seeded synthetic inputs for the FlexMoE routed-expert FFN hot path.

This module is the ONLY code shared by the CPU oracle's tests and the CUDA path's
tests/bench.  It holds none of the method's arithmetic: it draws tensors, rounds
them to bf16 bit patterns, plays the (external, frozen) router, and builds width
tables.  Recipes follow SURVEY.md section 8(d) / DESIGN.md "Input recipe"; the
configs C1..C5 are BASELINE.json `configs` in order.  The paper's own workloads
(pretrained Mixtral / Phi-3.5-MoE / Qwen2-57B-A14B served on synthetic requests,
PAPER.md:165, 220) are not available; these inputs take their SHAPES only.

bf16 tensors are carried as numpy uint16 bit patterns (numpy has no bf16).
Streams per config: weights (W_gate, W_up, W_down, channel_rank in that order) from
default_rng([seed, 1]); x, router logits, then budget tables from default_rng([seed, 2, T]).
"""
from __future__ import annotations

from dataclasses import dataclass, field
import numpy as np

# --------------------------------------------------------------------------- bf16 plumbing


def f32_to_bf16_bits(a: np.ndarray) -> np.ndarray:
    """Round-to-nearest-even fp32 -> bf16, returned as uint16 bit patterns (finite inputs)."""
    u = np.ascontiguousarray(a, dtype=np.float32).view(np.uint32)
    rnd = ((u >> np.uint32(16)) & np.uint32(1)) + np.uint32(0x7FFF)
    return ((u + rnd) >> np.uint32(16)).astype(np.uint16)


def bf16_bits_to_f32(b: np.ndarray) -> np.ndarray:
    """Exact widening of bf16 bit patterns to fp32."""
    return (np.ascontiguousarray(b, dtype=np.uint16).astype(np.uint32) << np.uint32(16)).view(np.float32)


def _normal_bf16(rng: np.random.Generator, shape, std: float, chunk: int = 1 << 24) -> np.ndarray:
    """N(0, std) drawn in fp32 and rounded to bf16 bits; chunked so C4-size tensors fit in RAM."""
    n = int(np.prod(shape))
    out = np.empty(n, dtype=np.uint16)
    for s in range(0, n, chunk):
        m = min(chunk, n - s)
        v = rng.standard_normal(m, dtype=np.float32)
        if std != 1.0:
            v *= np.float32(std)
        out[s:s + m] = f32_to_bf16_bits(v)
    return out.reshape(shape)


# --------------------------------------------------------------------------- shapes


@dataclass(frozen=True)
class Shape:
    name: str
    d: int       # model width (paper's H)
    E: int       # routed experts
    k: int       # experts per token
    I: int       # intermediate width I_max (paper's d_ff / I)


SHAPES = {
    "C1": Shape("tiny", 256, 8, 2, 512),
    "C2": Shape("qwen1.5-moe-a2.7b-shaped", 2048, 60, 4, 1408),
    "C3": Shape("deepseek-v2-lite-shaped", 2048, 64, 6, 1408),
    "C4": Shape("qwen2-57b-a14b-shaped", 3584, 64, 8, 2560),
}
SHAPES["C5"] = SHAPES["C4"]

RATIO_EIGHTHS = (8, 7, 6, 5, 4, 3, 2)          # {1, .875, .75, .625, .5, .375, .25} as n/8
C4_LEVELS = (2560, 2048, 1536, 1280, 1024, 640, 256)
C4_PRUNED = (0.0, 0.25, 0.40, 0.50, 0.75)


@dataclass
class Layer:
    shape: Shape
    W_gate: np.ndarray          # [E, I, d] bf16 bits, ORIGINAL channel order
    W_up: np.ndarray            # [E, I, d]
    W_down: np.ndarray          # [E, d, I]
    channel_rank: np.ndarray    # [E, I] int32; channel_rank[e][p] = original index of p-th ranked channel


@dataclass
class Batch:
    x: np.ndarray               # [T, d] bf16 bits
    topk_ids: np.ndarray        # [T, k] int32
    topk_w: np.ndarray          # [T, k] float32
    logits: np.ndarray | None = field(default=None, repr=False)


# --------------------------------------------------------------------------- generators


def make_layer(shape: Shape, rng: np.random.Generator, w_std: float = 0.02,
               identity_rank: bool = False) -> Layer:
    E, I, d = shape.E, shape.I, shape.d
    Wg = _normal_bf16(rng, (E, I, d), w_std)
    Wu = _normal_bf16(rng, (E, I, d), w_std)
    Wd = _normal_bf16(rng, (E, d, I), w_std)
    if identity_rank:
        rank = np.tile(np.arange(I, dtype=np.int32), (E, 1))
    else:
        rank = np.stack([rng.permutation(I).astype(np.int32) for _ in range(E)])
    return Layer(shape, Wg, Wu, Wd, rank)


def make_x(T: int, d: int, rng: np.random.Generator) -> np.ndarray:
    return _normal_bf16(rng, (T, d), 1.0)


def route(logits: np.ndarray, k: int):
    """The frozen external router (reading #10): fp32 softmax over E, top-k with the lower
    expert id winning ties, renormalise the k weights to sum 1.  Returns (ids int32, w fp32)."""
    lg = np.asarray(logits, dtype=np.float32)
    z = lg - lg.max(axis=1, keepdims=True)
    p = np.exp(z, dtype=np.float32)
    p /= p.sum(axis=1, keepdims=True, dtype=np.float32)
    # stable argsort of -p: equal probabilities keep ascending id order
    order = np.argsort(-p, axis=1, kind="stable")[:, :k]
    w = np.take_along_axis(p, order, axis=1).astype(np.float32)
    w /= w.sum(axis=1, keepdims=True, dtype=np.float32)
    return order.astype(np.int32), w.astype(np.float32)


def make_logits(T: int, E: int, rng: np.random.Generator, std: float = 1.0,
                expert_bias_std: float = 0.0) -> np.ndarray:
    """i.i.d. N(0,std) logits; with expert_bias_std>0 adds a per-expert mean mu_e ~ N(0,bias^2)
    drawn once (the C3 'skewed load' reading: logit = mu_e + eps, eps ~ N(0,1))."""
    if expert_bias_std > 0.0:
        mu = rng.standard_normal(E, dtype=np.float32) * np.float32(expert_bias_std)
        return mu[None, :] + rng.standard_normal((T, E), dtype=np.float32) * np.float32(std)
    return rng.standard_normal((T, E), dtype=np.float32) * np.float32(std)


def make_batch(shape: Shape, T: int, rng: np.random.Generator, logit_std: float = 1.0,
               expert_bias_std: float = 0.0, keep_logits: bool = False) -> Batch:
    x = make_x(T, shape.d, rng)
    lg = make_logits(T, shape.E, rng, logit_std, expert_bias_std)
    ids, w = route(lg, shape.k)
    return Batch(x, ids, w, lg if keep_logits else None)


# --------------------------------------------------------------------------- width tables


def widths_from_eighths(I: int, eighths: np.ndarray) -> np.ndarray:
    """r_e = I * n/8 in exact integer arithmetic (all config I are multiples of 8)."""
    assert I % 8 == 0
    return (I // 8 * np.asarray(eighths, dtype=np.int64)).astype(np.int32)


def table_c1(shape: Shape, rng: np.random.Generator) -> np.ndarray:
    """C1: ratio drawn per expert uniformly from {1,.875,...,.25}."""
    n = rng.choice(np.array(RATIO_EIGHTHS), size=shape.E)
    return widths_from_eighths(shape.I, n)


def table_uniform(shape: Shape, r: int) -> np.ndarray:
    return np.full(shape.E, r, dtype=np.int32)


def table_mean_ratio(shape: Shape, rng: np.random.Generator, keep: float) -> np.ndarray:
    """C3: per-expert r_e in I*{1,.875,...,.25}; sum r_e = the multiple of I/8 nearest to
    keep*E*I.  Start from a uniform random draw, then move random experts one level up/down
    until the sum matches."""
    E, I = shape.E, shape.I
    unit = I // 8
    target = int(round(keep * E * I / unit))
    lv = rng.choice(np.array(RATIO_EIGHTHS), size=E).astype(np.int64)
    lo, hi = min(RATIO_EIGHTHS), max(RATIO_EIGHTHS)
    guard = 0
    while lv.sum() != target:
        e = int(rng.integers(E))
        if lv.sum() > target and lv[e] > lo:
            lv[e] -= 1
        elif lv.sum() < target and lv[e] < hi:
            lv[e] += 1
        guard += 1
        assert guard < 1_000_000
    return (lv * unit).astype(np.int32)


def tables_nested_descent(shape: Shape, rng: np.random.Generator,
                          pruned=C4_PRUNED, levels=C4_LEVELS) -> np.ndarray:
    """C4/C5 (H): heterogeneous NESTED tables.  Start all-I; for each next budget step a
    seeded-random expert down one level until sum r_e <= E*I*(1-rho); the last step may pick
    any lower level that lands exactly, else the nearest below.  Returns [B, E] int32,
    monotone non-increasing along B (reading #14)."""
    E, I = shape.E, shape.I
    lv = list(levels)
    assert lv[0] == I
    idx = np.zeros(E, dtype=np.int64)          # level index per expert
    cur = np.array([lv[i] for i in idx], dtype=np.int64)
    out = []
    for rho in pruned:
        target = int(round(E * I * (1.0 - rho)))
        while cur.sum() > target:
            e = int(rng.integers(E))
            if idx[e] + 1 >= len(lv):
                continue
            need = cur.sum() - target
            step = cur[e] - lv[idx[e] + 1]
            if step > need:
                # try to land exactly with some expert/level; otherwise overshoot with this step
                done = False
                for e2 in rng.permutation(E):
                    for j in range(idx[e2] + 1, len(lv)):
                        if cur[e2] - lv[j] == need:
                            idx[e2] = j
                            cur[e2] = lv[j]
                            done = True
                            break
                    if done:
                        break
                if done:
                    break
            idx[e] += 1
            cur[e] = lv[idx[e]]
        out.append(cur.copy())
    return np.array(out, dtype=np.int32)


def table_fig6_like(shape: Shape, rng: np.random.Generator) -> np.ndarray:
    """Bimodal table with the action histogram of the paper's printed 40 % mask
    (117x100 %, 26x70 %, 21x40 %, 92x10 % of 256 cells), widths snapped to
    multiples of 128 so that 0.1*I -> 256 for I=2560."""
    E, I = shape.E, shape.I
    frac = np.array([117, 26, 21, 92], dtype=np.float64) / 256.0
    widths = [I, (I * 7 // 10) // 128 * 128, (I * 4 // 10) // 128 * 128, max(128, (I // 10) // 128 * 128)]
    cnt = np.floor(frac * E).astype(int)
    cnt[0] += E - cnt.sum()
    r = np.concatenate([np.full(c, w) for c, w in zip(cnt, widths)])
    rng.shuffle(r)
    return r.astype(np.int32)


# --------------------------------------------------------------------------- named configs


_LAYER_CACHE: dict = {}


def layer_for(name: str, seed: int = 0) -> Layer:
    """The weights of a named config: one independent generator stream default_rng([seed, 1]), so the layer does
    not depend on T and can be cached across the T values of a config (C4 is 3.5 GB of bf16)."""
    key = (name.upper(), seed)
    if key not in _LAYER_CACHE:
        _LAYER_CACHE.clear()                    # keep at most one big layer alive
        _LAYER_CACHE[key] = make_layer(SHAPES[key[0]], np.random.default_rng([seed, 1]))
    return _LAYER_CACHE[key]


def config(name: str, T: int | None = None, seed: int = 0, layer: bool = True):
    """Returns (Layer|None, Batch, rng) for a named config.  Streams: weights + channel_rank from
    default_rng([seed, 1]) (see layer_for); x then router logits from default_rng([seed, 2, T]); the returned
    rng is that second stream, from which the caller draws budget tables."""
    name = name.upper()
    sh = SHAPES[name]
    default_T = {"C1": 64, "C2": 4096, "C3": 8192, "C4": 8192, "C5": 4096}[name]
    T = default_T if T is None else T
    lay = layer_for(name, seed) if layer else None
    rng = np.random.default_rng([seed, 2, T])
    x = make_x(T, sh.d, rng)
    if name == "C3":
        lg = make_logits(T, sh.E, rng, 1.0, 1.5)
    else:
        lg = make_logits(T, sh.E, rng, 1.0, 0.0)
    ids, w = route(lg, sh.k)
    return lay, Batch(x, ids, w), rng
