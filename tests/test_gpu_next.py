"""GPU parity tests of the rows SURVEY.md 8(f) lists as NEXT: NEXT-2 channel saliency + ranking (Eq. 2-3), NEXT-3 the
router front end fused into the route kernel, NEXT-4 device-side action sampling and cost (Eq. 6-7, 10).  Everything goes
through the C ABI and is compared with the CPU oracle on the same seeded inputs; where floating point decides an index
(rank, top-k, argmax) both sides decide on the same fp32 numbers and the comparison is bit-exact."""
import numpy as np
import pytest

import oracle
from paper_2606_27866_b200 import inputs as gen

pytestmark = pytest.mark.gpu


def _fx():
    from paper_2606_27866_b200 import flexmoe as fx
    return fx


def _bf16(rng, shape, std):
    return gen.f32_to_bf16_bits(rng.standard_normal(shape, dtype=np.float32) * np.float32(std))


# ------------------------------------------------------------------------------ NEXT-2: saliency + ranking
@pytest.mark.parametrize("E,d,I,B", [(3, 64, 16, 1), (5, 192, 80, 3), (8, 256, 512, 2), (60, 512, 1408, 2), (2, 128, 4112, 1),
                                     (100, 64, 48, 3), (7, 192, 272, 5), (200, 64, 16, 2)])
def test_saliency_matches_oracle_and_rank_is_exact_on_the_same_keys(E, d, I, B):
    """The last three shapes: row chunks of W_down that are not a multiple of the kernel's four-row step (E=100, d=64:
    12 chunks of 5 or 6 rows; E=200: 6 chunks of 10 or 11), column groups with idle lanes (I=272: 34 chunks = one full
    group + 2 lanes) and an odd number of gradient sets beyond the two loaded at a time.
    Eq. 2 in fp32 (fixed summation order) vs the fp64 oracle: every s within 1e-5 relative.  The ranking is index
    work: on the SAME keys (the kernel's own fp32 s) it must equal the oracle's rank bit for bit (ties -> lower index),
    and where the oracle's own saliencies are separated by more than the fp32 error the two ranks agree."""
    import torch
    import gpu_util as gu
    fx = _fx()
    rng = np.random.default_rng(E * 1000 + I)
    Wg, Wu, Wd = _bf16(rng, (E, I, d), 0.05), _bf16(rng, (E, I, d), 0.05), _bf16(rng, (E, d, I), 0.05)
    Gg, Gu, Gd = _bf16(rng, (B, E, I, d), 1.0), _bf16(rng, (B, E, I, d), 1.0), _bf16(rng, (B, E, d, I), 1.0)
    # make a few channels exactly tie (duplicate their parameters and gradients) to exercise the tie rule
    if I >= 32:
        for (a, b_) in ((3, 17), (5, 6)):
            Wg[:, b_] = Wg[:, a]; Wu[:, b_] = Wu[:, a]; Wd[:, :, b_] = Wd[:, :, a]
            Gg[:, :, b_] = Gg[:, :, a]; Gu[:, :, b_] = Gu[:, :, a]; Gd[:, :, :, b_] = Gd[:, :, :, a]
    s = fx.saliency(gu.to_dev(Wg), gu.to_dev(Wu), gu.to_dev(Wd), gu.to_dev(Gg), gu.to_dev(Gu), gu.to_dev(Gd))
    rk = fx.rank_channels(s)
    torch.cuda.synchronize()
    s_gpu = s.cpu().numpy()
    ref = oracle.saliency(Wg, Wu, Wd, Gg, Gu, Gd)
    assert np.abs(s_gpu - ref).max() <= 1e-5 * np.abs(ref).max()
    assert np.abs(s_gpu / ref - 1).max() <= 2e-5
    rk_gpu = rk.cpu().numpy()
    assert np.array_equal(rk_gpu, oracle.rank(s_gpu.astype(np.float64))), "rank differs from the oracle on the same keys"
    if I >= 32:
        assert np.array_equal(s_gpu[:, 3], s_gpu[:, 17])          # the planted ties are exact ties in fp32 too
        pos = np.argsort(rk_gpu, axis=1)                           # position of every channel
        assert (pos[:, 3] + 1 == pos[:, 17]).all() and (pos[:, 5] + 1 == pos[:, 6]).all()
    # against the oracle's own ranking: compare where neighbouring oracle saliencies are well separated
    rk_ref = oracle.rank(ref)
    for e in range(E):
        sv = ref[e][rk_ref[e]]
        gap_ok = np.ones(I, bool)
        close = np.abs(np.diff(sv)) <= 4e-5 * sv[:-1]
        gap_ok[:-1] &= ~close
        gap_ok[1:] &= ~close
        assert np.array_equal(rk_gpu[e][gap_ok], rk_ref[e][gap_ok])


def test_saliency_at_bench_size_sampled_experts():
    """The launch configuration bench.py times (C2-sized weights, E=60, I=1408, d=2048, B=2: 3.1 GB, 720 column blocks +
    2640 row blocks in one grid, generated on the device as bench.py does) against the oracle on sampled experts:
    every channel of experts 0, 17, 31 and 59, both through fxm_saliency and through fxm_saliency_static."""
    import torch
    fx = _fx()
    E, I, d, B = 60, 1408, 2048, 2
    g = torch.Generator(device="cuda")
    g.manual_seed(11)
    mk = lambda *shape: (torch.randn(*shape, device="cuda", dtype=torch.float32, generator=g) * 0.02).to(torch.bfloat16)
    Wg, Wu, Wd = mk(E, I, d), mk(E, I, d), mk(E, d, I)
    Gg, Gu, Gd = mk(B, E, I, d), mk(B, E, I, d), mk(B, E, d, I)
    s = fx.saliency(Wg, Wu, Wd, Gg, Gu, Gd)
    s2 = torch.empty_like(s)
    fx.saliency_static(Wg, Wu, Wd, Gg, Gu, Gd, s2)
    torch.cuda.synchronize()
    assert torch.equal(s, s2)
    s_gpu = s.cpu().numpy()
    assert np.isfinite(s_gpu).all() and (s_gpu > 0).all()
    bits = fx.bf16_to_bits
    for e in (0, 17, 31, 59):
        ref = oracle.saliency(bits(Wg[e:e + 1]), bits(Wu[e:e + 1]), bits(Wd[e:e + 1]),
                              bits(Gg[:, e:e + 1]), bits(Gu[:, e:e + 1]), bits(Gd[:, e:e + 1]))[0]
        assert np.abs(s_gpu[e] / ref - 1).max() <= 2e-5, (e, np.abs(s_gpu[e] / ref - 1).max())


def test_ranked_pack_orders_channels_by_importance_and_keeps_the_function():
    """The whole offline front: saliency -> rank -> pack.  With the device ranking, (1) the packed prefix holds the
    channels in descending saliency, (2) at full width the FFN equals the unranked dense layer (permutation invariance,
    PAPER.md:75), (3) the forward on a prefix equals the oracle packed with the same ranking."""
    import torch
    import gpu_util as gu
    fx = _fx()
    sh = gen.Shape("t", 128, 4, 2, 96)
    rng = np.random.default_rng(11)
    lay = gen.make_layer(sh, rng, w_std=0.08, identity_rank=True)
    B = 2
    Gg, Gu, Gd = _bf16(rng, (B, 4, 96, 128), 1.0), _bf16(rng, (B, 4, 96, 128), 1.0), _bf16(rng, (B, 4, 128, 96), 1.0)
    s = fx.saliency(gu.to_dev(lay.W_gate), gu.to_dev(lay.W_up), gu.to_dev(lay.W_down), gu.to_dev(Gg), gu.to_dev(Gu), gu.to_dev(Gd))
    rk = fx.rank_channels(s).cpu().numpy()
    torch.cuda.synchronize()
    s_h = s.cpu().numpy()
    for e in range(4):
        assert (np.diff(s_h[e][rk[e]]) <= 0).all() and sorted(rk[e].tolist()) == list(range(96))
    lay.channel_rank = rk
    L = gu.pack_layer(lay)
    b = gen.make_batch(sh, 40, rng)
    full = np.full(4, 96, np.int32)
    lay_id = gen.Layer(sh, lay.W_gate, lay.W_up, lay.W_down, np.tile(np.arange(96, dtype=np.int32), (4, 1)))
    gu.check_close(gu.run_ffn(L, b, full), gu.oracle_ffn(lay_id, b, full), "ranked pack at full width == unranked layer")
    r = np.array([48, 16, 96, 33], np.int32)
    gu.check_close(gu.run_ffn(L, b, r), gu.oracle_ffn(lay, b, r), "ranked pack, prefix widths")


# ------------------------------------------------------------------------------ NEXT-3: router front end
@pytest.mark.parametrize("T,E,k,decode", [(64, 8, 2, False), (64, 8, 2, True), (1, 60, 4, True), (700, 64, 8, False),
                                          (333, 256, 16, False), (37, 7, 3, True), (4096, 60, 4, False)])
def test_router_front_end_fused_into_route(T, E, k, decode):
    """fxm_moe_ffn_router: ids bit-exact vs the oracle's router (top-k on fp32 logits, ties -> lower id), weights within
    fp32 rounding, and the FFN output equal to the forward fed with the oracle's routing."""
    import torch
    import gpu_util as gu
    fx = _fx()
    d, I = (256, 512) if E == 8 else (128, 64)
    sh = gen.Shape("t", d, E, k, I)
    rng = np.random.default_rng(T + E)
    lay = gen.make_layer(sh, rng, w_std=0.08)
    lg = gen.make_logits(T, E, rng, 1.0, 1.0)
    if T >= 8:
        lg[3, :] = 0.0                                            # all ties: ids 0..k-1, equal weights
        lg[5, 1] = lg[5, 0]                                       # a tie between two experts
    x = gen.make_x(T, d, rng)
    r = (rng.integers(1, I // 16 + 1, size=E) * 16).astype(np.int32)
    L = gu.pack_layer(lay)
    L.set_budget(r)
    L.set_decode(1024 if decode else 0)
    y, ids, w = L.moe_ffn_router(gu.to_dev(x), torch.from_numpy(lg).cuda(), k, return_routing=True)
    torch.cuda.synchronize()
    assert L.device_flags() == 0
    assert L.launches_per_ffn() == (2 if (decode and T * k <= 1024) else 4)
    ids_ref, w_ref = oracle.router_topk(lg, k)
    assert np.array_equal(ids.cpu().numpy(), ids_ref)
    assert np.abs(w.cpu().numpy() - w_ref).max() <= 2e-6
    b = gen.Batch(x, ids_ref, w_ref)
    rows = None if T <= 1024 else np.sort(rng.choice(T, 256, replace=False)).astype(np.int32)
    yv = gen.bf16_bits_to_f32(fx.bf16_to_bits(y)).astype(np.float64)
    gu.check_close(yv if rows is None else yv[rows], gu.oracle_ffn(lay, b, r, rows=rows), f"router front end T={T} E={E} k={k}")
    # the routing it returns is what the grouping used: route() on those ids reproduces the oracle's grouping
    got = [t.cpu().numpy() for t in L.route(ids)]
    for g, rr in zip(got, oracle.route(ids_ref, E)):
        assert np.array_equal(g, rr)


# ------------------------------------------------------------------------------ NEXT-4: action sampling + cost
def test_sample_budget_and_cost_on_device_then_masked_forward():
    """Eq. 6-7: hard actions from alpha + Gumbel noise (noise passed in), widths written into the layer's table on the
    device, forward run on them with no host round trip; Eq. 10 cost from the device counts.  Actions and widths
    bit-exact vs the oracle, cost within fp32 rounding, FFN within tolerance at the sampled table."""
    import torch
    import gpu_util as gu
    fx = _fx()
    sh, rng = gen.SHAPES["C1"], np.random.default_rng(4)
    lay, b, _ = gen.config("C1")
    K = 4
    num, den = np.array([1, 4, 7, 10], np.int32), 10
    L = gu.pack_layer(lay)
    x, ids, w = gu.to_dev(b.x), torch.from_numpy(b.topk_ids).cuda(), torch.from_numpy(b.topk_w).cuda()
    counts = L.route(ids)[0]
    for trial in range(4):
        alpha = rng.standard_normal((sh.E, K)).astype(np.float32)
        g = (-np.log(-np.log(rng.random((sh.E, K))))).astype(np.float32) if trial else None
        if trial == 2:
            alpha[:, 1] = alpha[:, 0]; g[:, 1] = g[:, 0]          # exact ties -> lower k
        act = L.sample_budget(torch.from_numpy(alpha).cuda(), torch.from_numpy(g).cuda() if g is not None else None, num, den,
                              return_actions=True)
        y = L.moe_ffn(x, ids, w)                                  # Eq. 4 with the sampled mask, straight after
        cost = L.action_cost(torch.from_numpy(alpha).cuda(), num, den, counts)
        torch.cuda.synchronize()
        assert L.device_flags() == 0
        a_ref, w_ref = oracle.sample_actions(alpha, g if g is not None else np.zeros_like(alpha), num, den, sh.I)
        assert np.array_equal(act.cpu().numpy(), a_ref)
        gu.check_close(gen.bf16_bits_to_f32(fx.bf16_to_bits(y)).astype(np.float64), gu.oracle_ffn(lay, b, w_ref), f"sampled table {trial}")
        c_ref = oracle.action_cost(alpha, num, den, counts.cpu().numpy())
        assert abs(float(cost.item()) - c_ref) <= 2e-6
    # K and ratio validation
    with pytest.raises(fx.FxmError):
        L.sample_budget(torch.zeros((sh.E, 2), device="cuda"), None, np.array([3, 11], np.int32), 10)
