"""Pins for the CPU oracle (oracle/oracle.c) against what the paper and the mathematics fix.

Each test names the pin (P1..P10 of SURVEY.md section 8(c) / DESIGN.md) and the passage.  None of
them re-types the oracle's loop: they use a library routine with a different formulation (torch
fp64 einsum over ALL experts then gather), algebraic invariants the paper states, a numpy brute
force with a different loop nest, a CPU emulation of the paper's OTHER description of the same
function (Alg. 2), and values the paper prints (tests/golden/).
"""
import os

import numpy as np
import pytest
import torch

import oracle
from paper_2606_27866_b200 import inputs as gen

GOLD = os.path.join(os.path.dirname(__file__), "golden")


def small(seed=0, T=12, d=32, E=4, k=2, I=48, identity_rank=False):
    sh = gen.Shape("t", d, E, k, I)
    rng = np.random.default_rng(seed)
    lay = gen.make_layer(sh, rng, w_std=0.3, identity_rank=identity_rank)   # larger std: silu is exercised off-linear
    b = gen.make_batch(sh, T, rng)
    return sh, lay, b, rng


def f64(bits):
    return gen.bf16_bits_to_f32(bits).astype(np.float64)


def dense_torch(lay, b, Wg=None, Wu=None, Wd=None):
    """Textbook dense SwiGLU MoE (Eq. 1) via library routines: every expert on every
    token with einsum, then gather the routed ones."""
    Wg = torch.from_numpy(f64(lay.W_gate if Wg is None else Wg))
    Wu = torch.from_numpy(f64(lay.W_up if Wu is None else Wu))
    Wd = torch.from_numpy(f64(lay.W_down if Wd is None else Wd))
    x = torch.from_numpy(f64(b.x))
    g = torch.einsum("td,ecd->tec", x, Wg)
    u = torch.einsum("td,ecd->tec", x, Wu)
    h = torch.nn.functional.silu(g) * u
    o = torch.einsum("tec,edc->ted", h, Wd)                       # [T,E,d]
    ids = torch.from_numpy(b.topk_ids.astype(np.int64))
    w = torch.from_numpy(b.topk_w.astype(np.float64))
    sel = torch.gather(o, 1, ids[:, :, None].expand(-1, -1, o.shape[2]))
    return (sel * w[:, :, None]).sum(1).numpy()


def test_P1_dense_equality_vs_torch_einsum():
    """Eq. 4 with m = 1 is Eq. 1: r_e = I for all e equals the dense MoE."""
    sh, lay, b, _ = small(identity_rank=True)
    Gt, Ut, Dt = oracle.pack(lay.W_gate, lay.W_up, lay.W_down, None)
    y = oracle.moe_ffn(b.x, Gt, Ut, Dt, np.full(sh.E, sh.I), b.topk_ids, b.topk_w)
    ref = dense_torch(lay, b)
    assert np.abs(y - ref).max() <= 1e-12 * np.abs(ref).max()


def test_P1b_pack_then_full_width_equals_dense_on_original_weights():
    """Permutation invariance + Eq. 3: ranking must not change the full expert."""
    sh, lay, b, _ = small(seed=1)
    Gt, Ut, Dt = oracle.pack(lay.W_gate, lay.W_up, lay.W_down, lay.channel_rank)
    y = oracle.moe_ffn(b.x, Gt, Ut, Dt, np.full(sh.E, sh.I), b.topk_ids, b.topk_w)
    ref = dense_torch(lay, b)                                     # ORIGINAL, unranked weights
    assert np.abs(y - ref).max() <= 1e-12 * np.abs(ref).max()
    # and a mis-applied permutation (down columns not permuted) must FAIL this pin
    y_bad = oracle.moe_ffn(b.x, Gt, Ut, lay.W_down, np.full(sh.E, sh.I), b.topk_ids, b.topk_w)
    assert np.abs(y_bad - ref).max() > 1e-3 * np.abs(ref).max()


def test_P2_slice_equals_mask():
    """slicing the first r_e channels == zeroing channels r_e..I-1 of the full expert."""
    sh, lay, b, rng = small(seed=2)
    Gt, Ut, Dt = oracle.pack(lay.W_gate, lay.W_up, lay.W_down, lay.channel_rank)
    r = rng.integers(0, sh.I + 1, size=sh.E).astype(np.int32)
    r[0] = 0
    r[1] = sh.I
    y = oracle.moe_ffn(b.x, Gt, Ut, Dt, r, b.topk_ids, b.topk_w)
    Gm, Um, Dm = Gt.copy(), Ut.copy(), Dt.copy()
    for e in range(sh.E):
        Gm[e, r[e]:, :] = 0
        Um[e, r[e]:, :] = 0
        Dm[e, :, r[e]:] = 0
    y_mask = oracle.moe_ffn(b.x, Gm, Um, Dm, np.full(sh.E, sh.I), b.topk_ids, b.topk_w)
    assert np.array_equal(y, y_mask)                              # added terms are exactly +0
    # library cross-check of the masked model
    lay_m = gen.Layer(sh, Gm, Um, Dm, lay.channel_rank)
    ref = dense_torch(lay_m, b)
    assert np.abs(y - ref).max() <= 1e-12 * max(np.abs(ref).max(), 1e-30)


def test_P3_permutation_invariance_and_pack_direction():
    """PAPER.md:75, 82-84.  channel_rank = argsort-descending output (gather semantics, reading R3):
    after pack, the saliency of ranked channel p is s[rank[p]] and is non-increasing; W~ = P W with
    P[p, rank[p]] = 1."""
    sh, lay, b, rng = small(seed=3)
    s = rng.random((sh.E, sh.I))
    rank = np.argsort(-s, axis=1, kind="stable").astype(np.int32)
    Gt, Ut, Dt = oracle.pack(lay.W_gate, lay.W_up, lay.W_down, rank)
    for e in range(sh.E):
        assert (np.diff(s[e][rank[e]]) <= 0).all()
        P = np.zeros((sh.I, sh.I))
        P[np.arange(sh.I), rank[e]] = 1.0
        assert np.array_equal(f64(Gt[e]), P @ f64(lay.W_gate[e]))         # W~gate = P W_gate
        assert np.array_equal(f64(Ut[e]), P @ f64(lay.W_up[e]))
        assert np.array_equal(f64(Dt[e]), f64(lay.W_down[e]) @ P.T)       # W~down = W_down P^T
    y_perm = oracle.moe_ffn(b.x, Gt, Ut, Dt, np.full(sh.E, sh.I), b.topk_ids, b.topk_w)
    G0, U0, D0 = oracle.pack(lay.W_gate, lay.W_up, lay.W_down, None)
    y_id = oracle.moe_ffn(b.x, G0, U0, D0, np.full(sh.E, sh.I), b.topk_ids, b.topk_w)
    assert np.abs(y_perm - y_id).max() <= 1e-12 * np.abs(y_id).max()


def test_P4_channel_additivity_and_nesting():
    """Eq. 4 is a sum of rank-1 channel terms; budgets are nested prefixes."""
    sh, lay, b, rng = small(seed=4, T=6, k=1)
    Gt, Ut, Dt = oracle.pack(lay.W_gate, lay.W_up, lay.W_down, lay.channel_rank)
    r_lo = rng.integers(1, sh.I // 2, size=sh.E).astype(np.int32)
    r_hi = (r_lo + rng.integers(1, sh.I // 2, size=sh.E)).astype(np.int32)
    y_lo = oracle.moe_ffn(b.x, Gt, Ut, Dt, r_lo, b.topk_ids, b.topk_w)
    y_hi = oracle.moe_ffn(b.x, Gt, Ut, Dt, r_hi, b.topk_ids, b.topk_w)
    X = f64(b.x)
    for t in range(b.x.shape[0]):
        e = int(b.topk_ids[t, 0])
        cs = np.arange(r_lo[e], r_hi[e])
        g = f64(Gt[e][cs]) @ X[t]
        u = f64(Ut[e][cs]) @ X[t]
        h = g / (1.0 + np.exp(-g)) * u
        delta = float(b.topk_w[t, 0]) * (f64(Dt[e][:, cs]) @ h)
        assert np.abs((y_hi[t] - y_lo[t]) - delta).max() <= 1e-11 * max(np.abs(y_hi[t]).max(), 1e-30)
    # prefix masks nested: m(r) subset of m(r') for r < r'
    for e in range(sh.E):
        m_lo = np.arange(sh.I) < r_lo[e]
        m_hi = np.arange(sh.I) < r_hi[e]
        assert (m_lo <= m_hi).all()


def test_P5_linearity_in_router_weights_and_expert_additivity():
    """Form of Alg. 1 l.19: y is linear in topk_w and additive over experts."""
    sh, lay, b, rng = small(seed=5, k=3)
    Gt, Ut, Dt = oracle.pack(lay.W_gate, lay.W_up, lay.W_down, lay.channel_rank)
    r = gen.table_c1(gen.Shape("t", sh.d, sh.E, sh.k, sh.I), rng)
    y = oracle.moe_ffn(b.x, Gt, Ut, Dt, r, b.topk_ids, b.topk_w)
    y2 = oracle.moe_ffn(b.x, Gt, Ut, Dt, r, b.topk_ids, (2.0 * b.topk_w).astype(np.float32))
    assert np.abs(y2 - 2.0 * y).max() <= 1e-12 * np.abs(y).max()
    acc = np.zeros_like(y)
    for e in range(sh.E):
        w_e = np.where(b.topk_ids == e, b.topk_w, 0.0).astype(np.float32)
        acc += oracle.moe_ffn(b.x, Gt, Ut, Dt, r, b.topk_ids, w_e)
    assert np.abs(acc - y).max() <= 1e-12 * np.abs(y).max()


def brute(x, Gt, Ut, Dt, r, ids, w):
    """Independent numpy brute force: loops (expert, channel) outermost and scatters into tokens --
    a different nest and accumulation order from oracle.c's per-token loop."""
    T, d = x.shape
    E, I, _ = Gt.shape
    X = f64(x)
    y = np.zeros((T, d))
    for e in range(E):
        for c in range(int(r[e])):
            gc, uc, dc = f64(Gt[e, c]), f64(Ut[e, c]), f64(Dt[e, :, c])
            for t in range(T):
                for j in range(ids.shape[1]):
                    if ids[t, j] == e:
                        g = float(gc @ X[t])
                        u = float(uc @ X[t])
                        y[t] += float(w[t, j]) * (g / (1.0 + np.exp(-g)) * u) * dc
    return y


@pytest.mark.parametrize("seed", [6, 7])
def test_P6_brute_force_tiny(seed):
    sh, lay, b, rng = small(seed=seed, T=7, d=16, E=3, k=2, I=24)
    Gt, Ut, Dt = oracle.pack(lay.W_gate, lay.W_up, lay.W_down, lay.channel_rank)
    r = rng.integers(0, sh.I + 1, size=sh.E).astype(np.int32)
    y = oracle.moe_ffn(b.x, Gt, Ut, Dt, r, b.topk_ids, b.topk_w)
    ref = brute(b.x, Gt, Ut, Dt, r, b.topk_ids, b.topk_w)
    assert np.abs(y - ref).max() <= 1e-12 * max(np.abs(ref).max(), 1e-30)
    # duplicate ids inside a token simply add twice (reading R13)
    ids2 = b.topk_ids.copy()
    ids2[:, 1] = ids2[:, 0]
    y_dup = oracle.moe_ffn(b.x, Gt, Ut, Dt, r, ids2, b.topk_w)
    ref_dup = brute(b.x, Gt, Ut, Dt, r, ids2, b.topk_w)
    assert np.abs(y_dup - ref_dup).max() <= 1e-12 * max(np.abs(ref_dup).max(), 1e-30)


def alg2_emulation(x, Gt, Ut, Dt, r, ids, w, k_align):
    """CPU emulation of the paper's Alg. 2 data movement: interleaved gate-up
    layout [g0,u0,g1,u1,...] and transposed down, BucketByRetI, AlignUp, gather,
    Sort(eid), grouped GEMM, de-interleave 0::2 / 1::2, SiLU*U, zero pad cols [k,k_eff), grouped
    GEMM, scale by alpha, ScatterAdd."""
    T, d = x.shape
    E, I, _ = Gt.shape
    X = f64(x)
    Wgu = np.empty((E, 2 * I, d))
    Wgu[:, 0::2, :] = f64(Gt)
    Wgu[:, 1::2, :] = f64(Ut)
    WdT = np.transpose(f64(Dt), (0, 2, 1))                              # [E, I, H]
    Y = np.zeros((T, d))
    flat_e = ids.reshape(-1)
    flat_t = np.repeat(np.arange(T), ids.shape[1])
    flat_a = w.reshape(-1).astype(np.float64)
    active = np.unique(flat_e)
    buckets = {}
    for e in active:
        buckets.setdefault(int(r[e]), []).append(int(e))
    for kk, Ek in buckets.items():
        k_eff = min(I, -(-kk // k_align) * k_align)                     # AlignUp, clamped to I (reading R7)
        sel = np.isin(flat_e, Ek)
        Xk, ek, ak, tk = X[flat_t[sel]], flat_e[sel], flat_a[sel], flat_t[sel]
        pi = np.argsort(ek, kind="stable")
        Xk, ek, ak, tk = Xk[pi], ek[pi], ak[pi], tk[pi]
        Zd = np.zeros((Xk.shape[0], d))
        for e in Ek:
            seg = np.nonzero(ek == e)[0]
            if seg.size == 0:
                continue
            Zgu = Xk[seg] @ Wgu[e, 0:2 * k_eff, :].T
            G, U = Zgu[:, 0::2], Zgu[:, 1::2]
            Hh = G / (1.0 + np.exp(-G)) * U
            Hh[:, kk:k_eff] = 0.0
            Zd[seg] = Hh @ WdT[e, 0:k_eff, :]
        Zd *= ak[:, None]
        np.add.at(Y, tk, Zd)
    return Y


@pytest.mark.parametrize("k_align", [1, 16, 64])
def test_P7_alg1_equals_alg2(k_align):
    """Two descriptions of one function: pins the pad-zero rule and the
    interleave indexing g_j -> 2j, u_j -> 2j+1."""
    sh, lay, b, rng = small(seed=8, T=20, d=32, E=5, k=2, I=80)
    Gt, Ut, Dt = oracle.pack(lay.W_gate, lay.W_up, lay.W_down, lay.channel_rank)
    r = rng.choice([8, 24, 56, 80, 13], size=sh.E).astype(np.int32)
    y = oracle.moe_ffn(b.x, Gt, Ut, Dt, r, b.topk_ids, b.topk_w)
    ref = alg2_emulation(b.x, Gt, Ut, Dt, r, b.topk_ids, b.topk_w, k_align)
    assert np.abs(y - ref).max() <= 1e-12 * np.abs(ref).max()


@pytest.mark.parametrize("T,k,E,seed", [(1, 1, 1, 0), (5, 2, 3, 1), (64, 2, 8, 2), (257, 4, 60, 3), (1000, 8, 64, 4)])
def test_P8_grouping_vs_numpy(T, k, E, seed):
    rng = np.random.default_rng(seed)
    ids = rng.integers(0, E, size=(T, k)).astype(np.int32)
    if E > 2:
        ids[ids == 1] = 0                                               # force an empty expert
    counts, offsets, perm, inv = oracle.route(ids, E)
    flat = ids.reshape(-1)
    assert np.array_equal(counts, np.bincount(flat, minlength=E))
    assert np.array_equal(offsets, np.concatenate([[0], np.cumsum(counts)]))
    assert np.array_equal(perm, np.argsort(flat, kind="stable"))
    assert np.array_equal(perm[inv], np.arange(T * k))
    assert np.array_equal(inv[perm], np.arange(T * k))
    for e in range(E):
        seg = perm[offsets[e]:offsets[e + 1]]
        assert (flat[seg] == e).all() and (np.diff(seg) > 0).all()


def test_P8b_route_rejects_out_of_range():
    with pytest.raises(ValueError):
        oracle.route(np.array([[0, 4]], np.int32), 4)


def _fig6():
    rows = [l.split() for l in open(os.path.join(GOLD, "fig6_mask_40pct.txt")) if not l.startswith("#")]
    m = np.array([[int(v) for v in row[1:]] for row in rows])
    assert m.shape == (32, 8)
    return m


def test_P9_fig6_budget_formula():
    """Fig. 6 is captioned '40 % budget'; Eq. 12 is the UNWEIGHTED
    mean over experts -> rho = 0.4031."""
    m = _fig6()
    vals, cnt = np.unique(m, return_counts=True)
    assert dict(zip(vals.tolist(), cnt.tolist())) == {10: 92, 40: 21, 70: 26, 100: 117}
    I = 1000                                                            # ratios exact in thousandths
    r = (m * 10).astype(np.int32)
    rho = oracle.budget_rho(r, I)
    assert abs(rho - 0.403125) < 1e-12
    assert round(rho, 2) == 0.40
    # with k = ceil(r * d_ff) on a 14336-wide expert: 0.40311
    I2 = 14336
    r2 = np.array([[oracle.ratio_to_width(I2, int(v), 100) for v in row] for row in m], np.int32)
    assert oracle.ratio_to_width(I2, 10, 100) == 1434 and oracle.ratio_to_width(I2, 70, 100) == 10036
    assert abs(oracle.budget_rho(r2, I2) - 0.40311) < 5e-6


def test_ratio_to_width_is_integer_ceil():
    """Reading R2: float ceil(0.7*10) would give 8; the integer form gives 7."""
    assert oracle.ratio_to_width(10, 7, 10) == 7
    assert oracle.ratio_to_width(1408, 1, 2) == 704
    assert oracle.ratio_to_width(7, 1, 2) == 4
    assert oracle.ratio_to_width(2560, 1, 1) == 2560


def test_P10_table2_bytes_linear_in_retained_fraction():
    """Table 2: ckpt size = fixed + (1-rho) * routed-expert bytes, i.e. linear in rho.
    Fit on the end points of each model, check the interior points within the table's rounding."""
    rows = np.array([[float(v) for v in l.split()] for l in open(os.path.join(GOLD, "table2_ckpt_sizes.txt"))
                     if not l.startswith("#")])
    rho = rows[:, 0] / 100.0
    # all three models: strictly decreasing and close to a straight line in rho (least squares;
    # Mixtral within 0.15 GB, Qwen2 0.8 GB, Phi-3.5 1.5 GB of the fitted line)
    for col, tol in ((1, 0.2), (2, 1.5), (3, 0.8)):
        s = rows[:, col]
        assert (np.diff(s) < 0).all()
        A = np.stack([np.ones_like(rho), rho], 1)
        coef, *_ = np.linalg.lstsq(A, s, rcond=None)
        assert np.abs(A @ coef - s).max() <= tol
    # Mixtral: 32 layers x 8 experts x 3 x 4096 x 14336 bf16 params = 84.0 GiB of routed experts
    routed_gib = 32 * 8 * 3 * 4096 * 14336 * 2 / 2**30
    assert abs(routed_gib - 84.0) < 0.01
    pred = 87.0 - rho * routed_gib
    assert np.abs(pred - rows[:, 1]).max() <= 0.5


def test_f32_oracle_error_is_far_below_tolerance():
    """north_star's 'plain fp32 oracle' vs the fp64 default: ~1e-6, tolerance is 5e-3."""
    sh, lay, b, rng = small(seed=9, T=16, d=64, E=4, k=2, I=96)
    Gt, Ut, Dt = oracle.pack(lay.W_gate, lay.W_up, lay.W_down, lay.channel_rank)
    r = np.full(sh.E, sh.I, np.int32)
    y64 = oracle.moe_ffn(b.x, Gt, Ut, Dt, r, b.topk_ids, b.topk_w)
    y32 = oracle.moe_ffn(b.x, Gt, Ut, Dt, r, b.topk_ids, b.topk_w, precision="f32")
    rel = np.linalg.norm(y32 - y64) / np.linalg.norm(y64)
    assert rel < 1e-5


def test_rows_subset_is_exact():
    sh, lay, b, rng = small(seed=10)
    Gt, Ut, Dt = oracle.pack(lay.W_gate, lay.W_up, lay.W_down, lay.channel_rank)
    r = gen.table_c1(sh, rng)
    y = oracle.moe_ffn(b.x, Gt, Ut, Dt, r, b.topk_ids, b.topk_w)
    rows = np.array([3, 0, 11], np.int32)
    ys = oracle.moe_ffn(b.x, Gt, Ut, Dt, r, b.topk_ids, b.topk_w, rows=rows)
    assert np.array_equal(ys, y[rows])


def test_r_zero_expert_contributes_nothing():
    """Reading R12."""
    sh, lay, b, rng = small(seed=11, k=1)
    Gt, Ut, Dt = oracle.pack(lay.W_gate, lay.W_up, lay.W_down, lay.channel_rank)
    r = np.zeros(sh.E, np.int32)
    y = oracle.moe_ffn(b.x, Gt, Ut, Dt, r, b.topk_ids, b.topk_w)
    assert (y == 0).all()


# ------------------------------------------------------------------ P11: saliency (Eq. 2)
def _sal_inputs(seed=0, B=3, E=3, I=20, d=12):
    rng = np.random.default_rng(seed)
    mk = lambda *sh: gen.f32_to_bf16_bits(rng.standard_normal(sh).astype(np.float32) * 0.5)
    return (mk(E, I, d), mk(E, I, d), mk(E, d, I)), (mk(B, E, I, d), mk(B, E, I, d), mk(B, E, d, I))


def test_P11_saliency_constant_gradient_closed_form():
    """g = c everywhere  =>  s_j = c^2 * sum_{theta in Theta_j} theta^2: row norms of gate/up plus the COLUMN norm of
    down (Theta_j = row j of W_gate, row j of W_up, column j of W_down), via numpy's own sum of squares."""
    (Wg, Wu, Wd), (Gg, Gu, Gd) = _sal_inputs(1)
    c = 0.75
    cb = gen.f32_to_bf16_bits(np.full(1, c, np.float32))[0]
    s = oracle.saliency(Wg, Wu, Wd, np.full_like(Gg, cb), np.full_like(Gu, cb), np.full_like(Gd, cb))
    expect = c * c * ((f64(Wg) ** 2).sum(2) + (f64(Wu) ** 2).sum(2) + (f64(Wd) ** 2).sum(1))
    assert np.allclose(s, expect, rtol=1e-12, atol=0)
    # a transposed down operand (row instead of column) would give sum over axis 2 of Wd: must differ
    wrong = c * c * ((f64(Wg) ** 2).sum(2) + (f64(Wu) ** 2).sum(2))
    assert not np.allclose(s[:, :Wd.shape[1]], wrong[:, :Wd.shape[1]], rtol=1e-3)


def test_P11_saliency_invariants():
    """a^2 scaling in g, equivariance under a consistent channel permutation, additivity over the three matrices, the
    mean over batches (duplicating the ranking set changes nothing), non-negativity."""
    (Wg, Wu, Wd), (Gg, Gu, Gd) = _sal_inputs(2)
    s = oracle.saliency(Wg, Wu, Wd, Gg, Gu, Gd)
    assert (s >= 0).all() and s.shape == (3, 20)
    two = lambda g: gen.f32_to_bf16_bits(gen.bf16_bits_to_f32(g) * np.float32(2.0))      # exact in bf16
    assert np.allclose(oracle.saliency(Wg, Wu, Wd, two(Gg), two(Gu), two(Gd)), 4.0 * s, rtol=1e-12)
    zero = lambda g: np.zeros_like(g)
    parts = (oracle.saliency(Wg, Wu, Wd, Gg, zero(Gu), zero(Gd)) + oracle.saliency(Wg, Wu, Wd, zero(Gg), Gu, zero(Gd)) +
             oracle.saliency(Wg, Wu, Wd, zero(Gg), zero(Gu), Gd))
    assert np.allclose(parts, s, rtol=1e-12)
    dup = lambda g: np.concatenate([g, g])
    assert np.allclose(oracle.saliency(Wg, Wu, Wd, dup(Gg), dup(Gu), dup(Gd)), s, rtol=1e-12)
    rng = np.random.default_rng(5)
    pi = rng.permutation(20)
    sp = oracle.saliency(Wg[:, pi], Wu[:, pi], Wd[:, :, pi], Gg[:, :, pi], Gu[:, :, pi], Gd[:, :, :, pi])
    assert np.allclose(sp, s[:, pi], rtol=1e-12)
    # only batch 0 differs from the mean over batches: B matters as a divisor
    s0 = oracle.saliency(Wg, Wu, Wd, Gg[:1], Gu[:1], Gd[:1])
    assert not np.allclose(s0, s, rtol=1e-3)


def test_P11_saliency_brute_force_tiny():
    """pure-python triple loop over (batch, parameter) on a tiny case, grouping parameters by channel through an
    explicit membership list Theta_j built from index tuples."""
    (Wg, Wu, Wd), (Gg, Gu, Gd) = _sal_inputs(3, B=2, E=2, I=4, d=3)
    s = oracle.saliency(Wg, Wu, Wd, Gg, Gu, Gd)
    W = {"g": f64(Wg), "u": f64(Wu), "d": f64(Wd)}
    G = {"g": f64(Gg), "u": f64(Gu), "d": f64(Gd)}
    for e in range(2):
        for j in range(4):
            theta = [("g", (e, j, i)) for i in range(3)] + [("u", (e, j, i)) for i in range(3)] + [("d", (e, i, j)) for i in range(3)]
            tot = 0.0
            for b in range(2):
                sb = 0.0
                for m, idx in theta:
                    sb += (W[m][idx] * G[m][(b,) + idx]) ** 2
                tot += sb
            assert abs(s[e, j] - tot / 2) <= 1e-12 * max(1.0, tot)


# ------------------------------------------------------------------ P12: rank (Eq. 3's pi; reading R4)
def test_P12_rank_vs_numpy_stable_argsort_and_ties():
    rng = np.random.default_rng(0)
    s = rng.random((5, 257))
    s[1, 10:20] = s[1, 3]                     # a run of exact ties
    s[2, :] = 1.0                             # all equal -> identity
    s[3, ::2] = 0.0
    got = oracle.rank(s)
    for e in range(5):
        assert np.array_equal(got[e], np.argsort(-s[e], kind="stable"))
        assert sorted(got[e].tolist()) == list(range(257))
        assert (np.diff(s[e][got[e]]) <= 0).all()
    assert np.array_equal(got[2], np.arange(257))


def test_P12_rank_recovers_a_planted_importance_order_through_saliency_and_pack():
    """Plant the importance: channel c of expert e gets weight scale proportional to a planted score, gradients all
    one -> Eq. 2 orders the channels by the planted score -> rank returns the planted order, and packing with it puts the
    channels in that order (reading R3: rank[p] = ORIGINAL index of the p-th most important channel)."""
    rng = np.random.default_rng(7)
    E, I, d = 2, 16, 8
    order = np.stack([rng.permutation(I) for _ in range(E)])           # order[e][p] = channel with the p-th largest score
    scale = np.empty((E, I), np.float32)
    for e in range(E):
        scale[e, order[e]] = 2.0 ** (-np.arange(I) / 2.0).astype(np.float32)
    one = np.ones((E, I, d), np.float32)
    Wg = gen.f32_to_bf16_bits(one * scale[:, :, None])
    Wu = gen.f32_to_bf16_bits(one * scale[:, :, None])
    Wd = gen.f32_to_bf16_bits(np.ones((E, d, I), np.float32) * scale[:, None, :])
    ones = lambda sh: gen.f32_to_bf16_bits(np.ones(sh, np.float32))
    s = oracle.saliency(Wg, Wu, Wd, ones((1, E, I, d)), ones((1, E, I, d)), ones((1, E, d, I)))
    rk = oracle.rank(s)
    assert np.array_equal(rk, order)
    Gt, _, Dt = oracle.pack(Wg, Wu, Wd, rk)
    assert (np.diff(f64(Gt)[:, :, 0], axis=1) < 0).all() and (np.diff(f64(Dt)[:, 0, :], axis=1) < 0).all()


# ------------------------------------------------------------------ P13: router front end (reading R10)
def test_P13_router_topk_vs_generator_and_torch():
    """The generator plays the same router with the OTHER formulation (softmax over all E, top-k, renormalise);
    torch.topk / torch.softmax are a third.  ids equal (generic logits), weights within fp32 rounding."""
    rng = np.random.default_rng(0)
    lg = gen.make_logits(300, 24, rng)
    ids, w = oracle.router_topk(lg, 5)
    gi, gw = gen.route(lg, 5)
    assert np.array_equal(ids, gi) and np.allclose(w, gw, rtol=0, atol=3e-7)
    tv, ti = torch.topk(torch.from_numpy(lg).double(), 5, dim=1)
    assert np.array_equal(ids, ti.numpy().astype(np.int32))
    assert np.allclose(w, torch.softmax(tv, dim=1).numpy(), atol=1e-7)
    assert np.allclose(w.sum(1), 1.0, atol=1e-6) and (np.diff(w, axis=1) <= 0).all()


def test_P13_router_closed_forms():
    ids, w = oracle.router_topk(np.zeros((3, 8), np.float32), 3)               # all ties: lowest ids, equal weights
    assert (ids == np.array([0, 1, 2])).all() and np.allclose(w, 1 / 3, atol=1e-7)
    lg = np.array([[0.0, np.log(3.0), -50.0, np.log(3.0)]], np.float32)
    ids, w = oracle.router_topk(lg, 3)
    assert ids.tolist() == [[1, 3, 0]] and np.allclose(w, [[3 / 7, 3 / 7, 1 / 7]], atol=1e-7)
    rng = np.random.default_rng(1)
    lg = rng.standard_normal((50, 12)).astype(np.float32)
    i1, w1 = oracle.router_topk(lg, 4)
    i2, w2 = oracle.router_topk(lg + np.float32(8.0), 4)                       # shift invariance (8.0 keeps fp32 sums exact enough)
    assert np.array_equal(i1, i2) and np.allclose(w1, w2, atol=2e-6)
    iE, wE = oracle.router_topk(lg, 12)                                          # k = E: plain softmax, sorted
    sm = torch.softmax(torch.from_numpy(lg).double(), 1).numpy()
    assert np.allclose(np.take_along_axis(sm, iE.astype(np.int64), 1), wE, atol=1e-7)


# ------------------------------------------------------------------ P14: actions (Eq. 6-7, 10-11)
def test_P14_noise_free_argmax_reproduces_the_printed_mask():
    """Eq. 11: hardened action = argmax_k p_k.  Build logits whose argmax is the printed action of every
    cell of Fig. 6; with zero noise the sampled ratios must be the printed ones and Eq. 12 gives the
    printed budget 0.4031."""
    mask = _fig6() / 100.0                     # the golden file holds percent
    assert mask.shape == (32, 8)
    ratios = np.array([0.1, 0.4, 0.7, 1.0])
    num, den = np.array([1, 4, 7, 10], np.int32), 10
    act_true = np.array([[int(np.argmin(np.abs(ratios - v))) for v in row] for row in mask])
    rng = np.random.default_rng(0)
    alpha = rng.standard_normal((256, 4)).astype(np.float32)
    alpha[np.arange(256), act_true.ravel()] += 10.0
    action, width = oracle.sample_actions(alpha, np.zeros_like(alpha), num, den, 14336)
    assert np.array_equal(action, act_true.ravel())
    assert width.tolist().count(1434) == 92 and width.tolist().count(14336) == 117      # ceil(0.1 * 14336) = 1434
    assert abs(oracle.budget_rho(width, 14336) - 0.40311) < 1e-4


def test_P14_gumbel_argmax_properties_and_cost_closed_forms():
    rng = np.random.default_rng(3)
    E, K = 40, 4
    alpha = rng.standard_normal((E, K)).astype(np.float32)
    g = -np.log(-np.log(rng.random((E, K)))).astype(np.float32)
    num, den = np.array([1, 4, 7, 10], np.int32), 10
    a1, w1 = oracle.sample_actions(alpha, g, num, den, 2560)
    # Eq. 6 with any temperature: argmax of softmax((alpha+g)/tau) == argmax of alpha+g (fp32 sum)
    for tau in (0.1, 1.0, 5.0):
        z = torch.softmax(torch.from_numpy((alpha + g).astype(np.float64)) / tau, 1).numpy()
        assert np.array_equal(a1, z.argmax(1))
    assert np.array_equal(w1, np.array([256, 1024, 1792, 2560])[a1])
    # Eq. 10: uniform p (alpha = 0) -> C = mean(r) regardless of the load; one-hot p -> C = sum_e q_e r_{k(e)}
    counts = rng.integers(0, 100, E).astype(np.int32)
    assert abs(oracle.action_cost(np.zeros((E, K), np.float32), num, den, counts) - 0.55) < 1e-12
    hot = np.full((E, K), -1e4, np.float32)
    hot[np.arange(E), a1] = 0.0
    q = counts / counts.sum()
    assert abs(oracle.action_cost(hot, num, den, counts) - float((q * (num[a1] / den)).sum())) < 1e-12
    # initialisation at the thickest action: cost = 1
    thick = np.full((E, K), -1e4, np.float32)
    thick[:, K - 1] = 0.0
    assert abs(oracle.action_cost(thick, num, den, counts) - 1.0) < 1e-12
