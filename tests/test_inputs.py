"""Host-side checks of the seeded input generators (paper_2606_27866_b200/inputs.py)."""
import numpy as np

from paper_2606_27866_b200 import inputs as gen


def test_bf16_roundtrip_and_rne():
    a = np.array([1.0, -2.5, 0.02, 1.00390625, 1.01171875, 3.1415926], np.float32)
    b = gen.f32_to_bf16_bits(a)
    back = gen.bf16_bits_to_f32(b)
    assert np.array_equal(gen.f32_to_bf16_bits(back), b)
    assert np.abs(back - a).max() <= np.abs(a).max() * 2.0 ** -8
    # ties to even: 1 + 2^-8 is exactly between 1.0 and 1 + 2^-7 -> rounds to 1.0 (even mantissa)
    assert gen.bf16_bits_to_f32(gen.f32_to_bf16_bits(np.array([1.00390625], np.float32)))[0] == 1.0
    assert gen.bf16_bits_to_f32(gen.f32_to_bf16_bits(np.array([1.01171875], np.float32)))[0] == 1.015625


def test_router_topk_distinct_sorted_normalised():
    rng = np.random.default_rng(0)
    lg = gen.make_logits(100, 16, rng)
    ids, w = gen.route(lg, 4)
    assert ids.dtype == np.int32 and w.dtype == np.float32
    assert all(len(set(row)) == 4 for row in ids.tolist())
    assert np.allclose(w.sum(1), 1.0, atol=1e-6)
    assert (np.diff(w, axis=1) <= 0).all()
    # ties -> lower id first
    ids2, _ = gen.route(np.zeros((3, 8), np.float32), 3)
    assert (ids2 == np.array([0, 1, 2])).all()


def test_c3_bias_reading_gives_skew():
    rng = np.random.default_rng(0)
    sh = gen.SHAPES["C3"]
    ids_iid, _ = gen.route(gen.make_logits(8192, sh.E, rng, 1.5, 0.0), sh.k)
    ids_skew, _ = gen.route(gen.make_logits(8192, sh.E, rng, 1.0, 1.5), sh.k)
    c_iid = np.bincount(ids_iid.ravel(), minlength=sh.E)
    c_skew = np.bincount(ids_skew.ravel(), minlength=sh.E)
    assert c_iid.max() / c_iid.mean() < 1.2          # i.i.d. logits give uniform load for any sigma
    assert c_skew.max() / c_skew.mean() > 3.0


def test_tables():
    rng = np.random.default_rng(0)
    sh1, sh3, sh4 = gen.SHAPES["C1"], gen.SHAPES["C3"], gen.SHAPES["C4"]
    r1 = gen.table_c1(sh1, rng)
    assert set(r1.tolist()) <= {512 * n // 8 for n in gen.RATIO_EIGHTHS}
    r3 = gen.table_mean_ratio(sh3, rng, 0.6)
    assert (r3 % 176 == 0).all() and abs(r3.sum() / (sh3.E * sh3.I) - 0.6) < 176 / (sh3.E * sh3.I)
    tabs = gen.tables_nested_descent(sh4, rng)
    assert tabs.shape == (5, 64) and (tabs[0] == 2560).all()
    assert (np.diff(tabs.astype(np.int64), axis=0) <= 0).all()              # nested / monotone
    assert set(np.unique(tabs).tolist()) <= set(gen.C4_LEVELS)
    for rho, t in zip(gen.C4_PRUNED, tabs):
        assert abs(1.0 - t.sum() / (64 * 2560) - rho) < 0.01
    r6 = gen.table_fig6_like(sh4, rng)
    assert r6.shape == (64,) and (r6 % 128 == 0).all() and r6.min() == 256 and r6.max() == 2560


def test_config_seeded():
    _, b1, _ = gen.config("C1", seed=0, layer=False)
    _, b2, _ = gen.config("C1", seed=0, layer=False)
    assert np.array_equal(b1.x, b2.x) and np.array_equal(b1.topk_ids, b2.topk_ids)
    lay, b, _ = gen.config("C1", seed=0)
    assert lay.W_gate.shape == (8, 512, 256) and lay.W_down.shape == (8, 256, 512) and b.x.shape == (64, 256)
    for e in range(8):
        assert np.array_equal(np.sort(lay.channel_rank[e]), np.arange(512))
