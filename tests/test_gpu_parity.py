"""GPU parity tests proper: the CUDA path (through the C ABI) against the CPU oracle, element by element,
on the same seeded inputs.  Indices bit-exact; FFN output within north_star's tolerance (gpu_util.TOL_*).
Run on the B200 box:  python -m pytest tests -m gpu -x -q"""
import numpy as np
import pytest

import oracle
from paper_2606_27866_b200 import inputs as gen

pytestmark = pytest.mark.gpu


def _fx():
    from paper_2606_27866_b200 import flexmoe as fx
    return fx


def _small_layer(seed, d, E, k, I, w_std=0.05):
    sh = gen.Shape("t", d, E, k, I)
    rng = np.random.default_rng(seed)
    return sh, gen.make_layer(sh, rng, w_std=w_std), rng


# ------------------------------------------------------------------------------------------------ pack
@pytest.mark.parametrize("d,E,I", [(64, 2, 16), (256, 8, 512), (192, 3, 80), (128, 5, 1408)])
def test_pack_unpack_roundtrip_bitexact(d, E, I):
    """Eq. 3: unpack_prefix(pack(W, rank), r) == oracle.pack(W, rank)[:r] bit for bit."""
    import torch
    import gpu_util as gu
    fx = _fx()
    sh, lay, rng = _small_layer(1, d, E, min(2, E), I)
    L = gu.pack_layer(lay)
    Gt, Ut, Dt = oracle.pack(lay.W_gate, lay.W_up, lay.W_down, lay.channel_rank)
    for e in range(E):
        for r in sorted({I, 0, 16, I // 2 // 16 * 16 + 16 if I > 32 else 16}):
            r = min(r, I)
            Wg, Wu, Wd = L.unpack_prefix(e, r)
            torch.cuda.synchronize()
            assert np.array_equal(fx.bf16_to_bits(Wg), Gt[e, :r]) if r else True
            assert np.array_equal(fx.bf16_to_bits(Wu), Ut[e, :r]) if r else True
            assert np.array_equal(fx.bf16_to_bits(Wd), Dt[e, :, :r]) if r else True


@pytest.mark.parametrize("d,E,I", [(192, 3, 80), (128, 2, 1408)])
def test_pack_with_w_down_two_byte_aligned_only(d, E, I):
    """fxm_pack asks only 2-byte alignment of W_down (include/flexmoe.h).  A 16-byte aligned W_down is packed by the
    kernel that stages whole rows in shared memory, any other one by the gather kernel: both must give the oracle's
    W~down bit for bit (Eq. 3)."""
    import torch
    fx = _fx()
    sh, lay, rng = _small_layer(3, d, E, min(2, E), I)
    buf = torch.zeros(E * d * I + 8, dtype=torch.bfloat16, device="cuda")
    Wd = buf[1:1 + E * d * I].view(E, d, I)                       # data_ptr 2 bytes past a 16-byte boundary
    Wd.copy_(fx.bf16_from_bits(lay.W_down, "cuda"))
    assert Wd.data_ptr() % 16 == 2 and Wd.is_contiguous()
    L = fx.Layer.pack(fx.bf16_from_bits(lay.W_gate, "cuda"), fx.bf16_from_bits(lay.W_up, "cuda"), Wd, lay.channel_rank)
    torch.cuda.synchronize()
    Gt, Ut, Dt = oracle.pack(lay.W_gate, lay.W_up, lay.W_down, lay.channel_rank)
    for e in range(E):
        Wg_, Wu_, Wd_ = L.unpack_prefix(e, I)
        torch.cuda.synchronize()
        assert np.array_equal(fx.bf16_to_bits(Wd_), Dt[e])
        assert np.array_equal(fx.bf16_to_bits(Wg_), Gt[e])


def test_pack_rejects_non_permutation():
    import gpu_util as gu
    fx = _fx()
    sh, lay, rng = _small_layer(2, 64, 2, 1, 32)
    lay.channel_rank[1, 3] = lay.channel_rank[1, 4]
    with pytest.raises(fx.FxmError) as ei:
        gu.pack_layer(lay)
    assert ei.value.name == "FXM_EPERM"


# ----------------------------------------------------------------------------------------------- route
@pytest.mark.parametrize("T,k,E,seed", [(0, 2, 8, 0), (1, 1, 4, 1), (1, 4, 60, 2), (64, 2, 8, 0), (16, 4, 60, 3),
                                        (37, 3, 7, 4), (1000, 6, 64, 5), (4096, 4, 60, 6), (8192, 8, 64, 7),
                                        (8192, 6, 64, 8), (333, 16, 256, 9)])
def test_route_bitexact(T, k, E, seed):
    """Alg. 2 l.4-6, reading R5: stable grouping; all four index arrays bit-exact."""
    import torch
    import gpu_util as gu
    sh, lay, rng = _small_layer(seed, 64, E, k, 32)
    L = gu.pack_layer(lay, identity=True)
    bias = 1.5 if seed == 8 else 0.0                      # C3-style skew: some experts empty, some huge
    ids, _ = gen.route(gen.make_logits(T, E, rng, 1.0, bias), k)
    c, o, p, ip = [t.cpu().numpy() for t in L.route(torch.from_numpy(ids).cuda().reshape(T, k))]
    rc, ro, rp, rip = oracle.route(ids.reshape(T, k), E)
    assert np.array_equal(c, rc) and np.array_equal(o, ro)
    assert np.array_equal(p, rp) and np.array_equal(ip, rip)
    assert L.device_flags() == 0


def test_route_duplicate_and_single_expert():
    """Degenerate routings: every assignment to one expert; duplicate ids inside a token (reading R13)."""
    import torch
    import gpu_util as gu
    sh, lay, rng = _small_layer(0, 64, 8, 2, 32)
    L = gu.pack_layer(lay, identity=True)
    for ids in (np.full((300, 2), 5, np.int32), np.repeat(rng.integers(0, 8, (129, 1)), 2, 1).astype(np.int32)):
        got = [t.cpu().numpy() for t in L.route(torch.from_numpy(ids).cuda())]
        ref = oracle.route(ids, 8)
        for g, r in zip(got, ref):
            assert np.array_equal(g, r)


# ------------------------------------------------------------------------------------------ FFN, small
def _c1():
    lay, b, rng = gen.config("C1")
    return gen.SHAPES["C1"], lay, b, rng


# impl: 1 = SIMT debug path, 0 = CTA-pair tcgen05 kernels (the product; general four-launch path forced),
# "dec" = fused decode kernel
IMPLS = [1, 0, "dec"]
GENERAL_LAUNCHES = {0: 4, 1: 4}


def _run(gu, L, b, r, impl, **kw):
    if impl == "dec":
        y = gu.run_ffn(L, b, r, impl=0, decode=True, **kw)
        assert L.launches_per_ffn() == 1, "the fused decode kernel was not taken"
        return y
    y = gu.run_ffn(L, b, r, impl=impl, decode=False, **kw)
    assert L.launches_per_ffn() == GENERAL_LAUNCHES[impl]
    return y


@pytest.mark.parametrize("impl", IMPLS)
@pytest.mark.parametrize("table", ["full", "c1", "all128", "ragged", "zeros_some"])
def test_c1_tiny_all_budgets(impl, table):
    """C1 (BASELINE.json configs[0]): d=256, E=8, top-2, I=512, T=64, every element vs the oracle."""
    import gpu_util as gu
    sh, lay, b, rng = _c1()
    r = {"full": np.full(sh.E, sh.I), "c1": gen.table_c1(sh, rng), "all128": np.full(sh.E, 128),
         "ragged": np.array([512, 16, 100 // 16 * 16 + 4 * 0 + 48, 336, 64, 80, 496, 272]),
         "zeros_some": np.array([0, 512, 0, 256, 64, 0, 128, 384])}[table].astype(np.int32)
    L = gu.pack_layer(lay)
    y = _run(gu, L, b, r, impl)
    gu.check_close(y, gu.oracle_ffn(lay, b, r), f"C1 {table} impl={impl}")


@pytest.mark.parametrize("impl", IMPLS)
def test_widths_not_multiple_of_64_and_padded_dims(impl):
    """I % 64 != 0 (padded channel block), d % 128 == 64 (padded down rows), r_e any multiple of 1."""
    import gpu_util as gu
    sh, lay, rng = _small_layer(3, 192, 6, 3, 80, w_std=0.1)
    b = gen.make_batch(sh, 50, rng)
    L = gu.pack_layer(lay)
    for r in ([80] * 6, [1, 7, 33, 64, 65, 79], [0, 0, 0, 0, 0, 5]):
        r = np.array(r, np.int32)
        gu.check_close(_run(gu, L, b, r, impl), gu.oracle_ffn(lay, b, r), f"r={r.tolist()} impl={impl}")


@pytest.mark.parametrize("impl,tile_n", [(1, 128), (0, 128), (0, 256), (0, 0)])
def test_multi_tile_ragged_segments(impl, tile_n):
    """Expert segments that span several token tiles plus a ragged tail, heavy skew, empty experts.
    impl 0 = CTA-pair kernels (token tiles up to 128 / 256 / 512 rows; above 256 = two sub-tiles), impl 1 = SIMT debug."""
    import gpu_util as gu
    sh, lay, rng = _small_layer(4, 128, 6, 2, 192, w_std=0.08)
    T = 900
    lg = gen.make_logits(T, sh.E, rng, 1.0, 2.0)
    lg[:, 4] = -1e9                                        # expert 4 never routed
    ids, w = gen.route(lg, sh.k)
    b = gen.Batch(gen.make_x(T, sh.d, rng), ids, w)
    r = np.array([192, 128, 64, 176, 192, 16], np.int32)
    L = gu.pack_layer(lay)
    gu.check_close(gu.run_ffn(L, b, r, impl=impl, tile_n=tile_n), gu.oracle_ffn(lay, b, r), f"impl={impl} tile_n={tile_n}")


@pytest.mark.parametrize("T", [130, 273, 300, 512, 520, 1024, 1100, 2048, 4001])
def test_pair_subtile_boundaries(T):
    """CTA-pair path: one expert receives every token, so its segment is T rows: <=256 (one sub-tile), 257..512
    (two sub-tiles sharing the weight operand), >512 (several token tiles); odd retained-block counts give the
    second CTA of a pair a pruned block that must be skipped."""
    import gpu_util as gu
    sh, lay, rng = _small_layer(5, 192, 3, 2, 320, w_std=0.08)
    ids = np.tile(np.array([[1, 2]], np.int32), (T, 1))
    ids[::7, 1] = 0
    w = rng.random((T, 2)).astype(np.float32)
    b = gen.Batch(gen.make_x(T, sh.d, rng), ids, w)
    L = gu.pack_layer(lay)
    for r in ([320, 320, 320], [192, 64, 304], [16, 130, 65]):
        r = np.array(r, np.int32)
        gu.check_close(gu.run_ffn(L, b, r, decode=False), gu.oracle_ffn(lay, b, r), f"T={T} r={r.tolist()}")


def _check_shape_case(d, E, k, I, T, seed):
    import gpu_util as gu
    sh, lay, rng = _small_layer(1000 + seed, d, E, k, I, w_std=0.08)
    lg = gen.make_logits(T, E, rng, 1.0, 1.5)
    ids, w = gen.route(lg, k)
    b = gen.Batch(gen.make_x(T, d, rng), ids, w)
    L = gu.pack_layer(lay)
    r = rng.integers(0, I + 1, size=E).astype(np.int32)
    r[int(rng.integers(E))] = I
    ref = gu.oracle_ffn(lay, b, r)
    if np.abs(ref).max() == 0:
        r[:] = I
        ref = gu.oracle_ffn(lay, b, r)
    gu.check_close(gu.run_ffn(L, b, r, decode=False), ref, f"general d={d} E={E} k={k} I={I} T={T} r={r.tolist()[:8]}")
    if T * k <= 1024 and d <= 3840:
        y = gu.run_ffn(L, b, r, decode=True)
        assert L.launches_per_ffn() == 1
        gu.check_close(y, ref, f"decode d={d} E={E} k={k} I={I} T={T}")


@pytest.mark.parametrize("d,E,k,I,T", [(64, 1, 1, 16, 1), (64, 1, 1, 16, 40), (128, 256, 16, 32, 33), (64, 2, 2, 1040, 17),
                                       (3584, 3, 2, 64, 70)])
def test_extreme_small_shapes_product_path_and_decode(d, E, k, I, T):
    """The corners of the supported set (d = 64, E = 1 and 256, k = 1 and 16, I = 16, ragged I, d = 3584): random widths
    in [0, I] (any multiple of 1), skewed routing; product path and fused decode kernel, every element vs the oracle."""
    _check_shape_case(d, E, k, I, T, d + E + T)


def test_property_sweep_random_shapes():
    """a hypothesis sweep over (d, E, k, I, T, seed) -- empty experts, widths in {0..I} that are not
    multiples of 16 or 64, duplicate-free skewed routing, ragged token counts; every element against the oracle on the
    product path and, where T*k <= 1024, on the fused decode kernel."""
    from hypothesis import given, settings, strategies as st, HealthCheck

    @settings(max_examples=30, deadline=None, derandomize=True, suppress_health_check=list(HealthCheck))
    @given(d64=st.integers(1, 8), E=st.integers(1, 24), kk=st.integers(1, 6), I16=st.integers(1, 20),
           T=st.sampled_from([1, 2, 7, 31, 64, 129, 300, 700]), seed=st.integers(0, 10_000))
    def run(d64, E, kk, I16, T, seed):
        _check_shape_case(d64 * 64, E, min(kk, E), I16 * 16, T, seed)

    run()


# ------------------------------------------------------------------------------------- fused decode kernel (a6)
@pytest.mark.parametrize("T,k,E,bias", [(1, 1, 4, 0.0), (3, 2, 5, 0.0), (40, 4, 6, 2.0), (200, 2, 6, 2.5), (64, 16, 16, 0.0),
                                        (128, 8, 256, 1.0), (1024, 1, 7, 1.0)])
def test_decode_groups_runs_and_skew(T, k, E, bias):
    """a6: experts with more than 16 tokens (several token groups re-streaming the weights), experts with none,
    width-0 experts, ragged widths, A up to the kernel's limit of 1024 assignments; every element vs the oracle."""
    import gpu_util as gu
    sh, lay, rng = _small_layer(21 + T, 192, E, k, 208, w_std=0.08)
    lg = gen.make_logits(T, E, rng, 1.0, bias)
    if E > 3:
        lg[:, 2] = -1e9                                    # expert 2 never routed
    ids, w = gen.route(lg, k)
    b = gen.Batch(gen.make_x(T, sh.d, rng), ids, w)
    L = gu.pack_layer(lay)
    r = rng.integers(0, 208 // 16 + 1, size=E).astype(np.int32) * 16
    r[0] = 208
    r[E - 1] = 0
    for rt in (np.full(E, 208, np.int32), r, (r // 3).astype(np.int32)):
        y = gu.run_ffn(L, b, rt, decode=True)
        assert L.launches_per_ffn() == 1
        gu.check_close(y, gu.oracle_ffn(lay, b, rt), f"decode T={T} k={k} E={E} r={rt.tolist()[:8]}")


def test_decode_repeated_calls_and_interleaving_with_general_path():
    """The decode kernel's grid-wide synchronisation lives across calls (ever-growing arrival counters in the layer's state,
    per-item readiness counters that every call hands back zeroed): many calls in a row (no host sync), alternating with
    general-path calls and with budget switches, must all be right."""
    import torch
    import gpu_util as gu
    fx = _fx()
    sh, lay, b, rng = _c1()
    tabs = np.array([[512] * 8, [512, 384, 512, 256, 512, 128, 512, 64], [256, 128, 192, 64, 512, 64, 128, 0]], np.int32)
    L = gu.pack_layer(lay)
    L.register_budgets(tabs, require_nested=True)
    x, ids, w = gu.to_dev(b.x), torch.from_numpy(b.topk_ids).cuda(), torch.from_numpy(b.topk_w).cuda()
    refs = [gu.oracle_ffn(lay, b, t) for t in tabs]
    outs = []
    for i in range(24):
        bi = (i * 7) % 3
        L.select_budget(bi)
        L.set_decode(0 if i % 5 == 4 else 1024)
        outs.append((bi, L.moe_ffn(x, ids, w)))
    torch.cuda.synchronize()
    assert L.device_flags() == 0
    for bi, y in outs:
        gu.check_close(gen.bf16_bits_to_f32(fx.bf16_to_bits(y)).astype(np.float64), refs[bi], f"call with budget {bi}")


def test_decode_out_of_range_id_is_flagged_and_dropped():
    import torch
    import gpu_util as gu
    fx = _fx()
    sh, lay, b, rng = _c1()
    r = np.full(sh.E, sh.I, np.int32)
    L = gu.pack_layer(lay)
    L.set_budget(r)
    L.set_decode(1024)
    ids = b.topk_ids.copy()
    ids[3, 1] = 99
    w = b.topk_w.copy()
    y = L.moe_ffn(gu.to_dev(b.x), torch.from_numpy(ids).cuda(), torch.from_numpy(w).cuda())
    torch.cuda.synchronize()
    assert L.device_flags() & 1
    w[3, 1] = 0.0                                          # dropping the assignment == giving it weight 0
    ids[3, 1] = 0
    ref = oracle.moe_ffn(b.x, *gu.oracle_packed(lay), r, ids, w)
    gu.check_close(gen.bf16_bits_to_f32(fx.bf16_to_bits(y)).astype(np.float64), ref, "dropped assignment")


def test_h_intermediate_matches_definition():
    """Step a4 alone: H = silu(G) (.) U in sorted order, channels >= r_e exactly 0 (pad-zero rule).
    The RAW read (no reader-side mask) shows what the GEMM-1 epilogue itself wrote: the columns [r_e, ceil64(r_e)) of
    the last retained block must be exact zeros."""
    import torch
    import gpu_util as gu
    fx = _fx()
    sh, lay, b, rng = _c1()
    r = np.array([512, 100, 37, 336, 65, 1, 496, 250], np.int32)        # ragged: the last block of most experts is partial
    L = gu.pack_layer(lay)
    gu.run_ffn(L, b, r, decode=False)                       # the H panels exist only on the general path
    ids = torch.from_numpy(b.topk_ids).cuda()
    Hraw = fx.bf16_to_bits(L.debug_read_h(ids, raw=True))
    _, _, perm0, _ = oracle.route(b.topk_ids, sh.E)
    n_pad = 0
    for s_ in range(perm0.size):
        e = b.topk_ids.ravel()[perm0[s_]]
        lim = -(-int(r[e]) // 64) * 64
        assert np.all(Hraw[s_, r[e]:lim] == 0), f"pad columns of sorted row {s_} (expert {e}) are not zero"
        assert np.any(Hraw[s_, :r[e]] != 0)
        n_pad += lim - int(r[e])
    assert n_pad > 0
    H = gen.bf16_bits_to_f32(fx.bf16_to_bits(L.debug_read_h(ids))).astype(np.float64)
    Gt, Ut, _ = oracle.pack(lay.W_gate, lay.W_up, lay.W_down, lay.channel_rank)
    x = gen.bf16_bits_to_f32(b.x).astype(np.float64)
    _, _, perm, _ = oracle.route(b.topk_ids, sh.E)
    for s in range(0, perm.size, 7):
        f = perm[s]
        t, e = f // sh.k, b.topk_ids.ravel()[f]
        g = gen.bf16_bits_to_f32(Gt[e]).astype(np.float64) @ x[t]
        u = gen.bf16_bits_to_f32(Ut[e]).astype(np.float64) @ x[t]
        h = g / (1 + np.exp(-g)) * u
        h[r[e]:] = 0
        assert np.all(H[s, r[e]:] == 0)
        assert np.abs(H[s] - h).max() <= 2.0 ** -7 * max(np.abs(h).max(), 1e-6)


def test_budget_switch_select_and_nested_check():
    """a1: registered tables + host-only select; nestedness check (reading R14)."""
    import torch
    import gpu_util as gu
    fx = _fx()
    sh, lay, b, rng = _c1()
    tabs = np.array([[512] * 8, [512, 384, 512, 256, 512, 128, 512, 64], [256, 128, 192, 64, 512, 64, 128, 0]], np.int32)
    L = gu.pack_layer(lay)
    with pytest.raises(fx.FxmError) as ei:
        L.register_budgets(tabs[::-1].copy(), require_nested=True)
    assert ei.value.name == "FXM_ENOTNESTED"
    L.register_budgets(tabs, require_nested=True)
    x, ids, w = gu.to_dev(b.x), torch.from_numpy(b.topk_ids).cuda(), torch.from_numpy(b.topk_w).cuda()
    before = L.packed.clone()
    for bi in (2, 0, 1, 2, 1):
        L.select_budget(bi)
        y = gen.bf16_bits_to_f32(fx.bf16_to_bits(L.moe_ffn(x, ids, w))).astype(np.float64)
        gu.check_close(y, gu.oracle_ffn(lay, b, tabs[bi]), f"budget {bi}")
    E, d, I = sh.E, sh.d, sh.I
    nw = 3 * E * ((I + 63) // 64 * 64) * d * 2
    assert torch.equal(before[:nw], L.packed[:nw]), "a budget switch must not touch the weights"
    with pytest.raises(fx.FxmError):
        L.select_budget(3)


@pytest.mark.parametrize("decode", [False, True])
def test_cuda_graph_capture_and_replay(decode):
    """include/flexmoe.h: grid sizes do not depend on the routing or the budget, nothing synchronises -> a call is
    CUDA-graph capturable.  Capture one fxm_moe_ffn, then replay it on NEW token data and a NEW budget table written
    into the same buffers (the graph holds no routing- or budget-dependent launch shape)."""
    import torch
    import gpu_util as gu
    fx = _fx()
    sh, lay, b, rng = _c1()
    tabs = np.array([[512] * 8, [256, 128, 192, 64, 512, 64, 128, 0]], np.int32)
    L = gu.pack_layer(lay)
    L.set_decode(1024 if decode else 0)
    L.set_budget(tabs[0])
    x, ids, w = gu.to_dev(b.x), torch.from_numpy(b.topk_ids).cuda(), torch.from_numpy(b.topk_w).cuda()
    y = torch.empty((b.x.shape[0], sh.d), dtype=torch.bfloat16, device="cuda")
    L.moe_ffn(x, ids, w, out=y)                               # warm-up outside the capture (workspace allocation)
    torch.cuda.synchronize()
    g = torch.cuda.CUDAGraph()
    side = torch.cuda.Stream()
    with torch.cuda.stream(side):
        with torch.cuda.graph(g, stream=side):
            L.moe_ffn(x, ids, w, out=y)
    g.replay()
    torch.cuda.synchronize()
    gu.check_close(gen.bf16_bits_to_f32(fx.bf16_to_bits(y)).astype(np.float64), gu.oracle_ffn(lay, b, tabs[0]), "replay 1")
    b2 = gen.make_batch(sh, b.x.shape[0], np.random.default_rng(77))
    x.copy_(gu.to_dev(b2.x)); ids.copy_(torch.from_numpy(b2.topk_ids).cuda()); w.copy_(torch.from_numpy(b2.topk_w).cuda())
    L.set_budget(tabs[1])                                     # same device table slot, new widths
    g.replay()
    torch.cuda.synchronize()
    assert L.device_flags() == 0
    gu.check_close(gen.bf16_bits_to_f32(fx.bf16_to_bits(y)).astype(np.float64), gu.oracle_ffn(lay, b2, tabs[1]), "replay 2")


def test_host_buffer_entry_point_pipelined_calls():
    """fxm_moe_ffn_host: six back-to-back calls with different pinned inputs and no host synchronisation in between
    (the input copy of call i+1 runs on the library's side stream while call i computes; the two staging sets
    alternate), decode-sized and general path; every output against the oracle."""
    import torch
    import gpu_util as gu
    fx = _fx()
    sh, lay, b0, rng = _c1()
    r = gen.table_c1(sh, rng)
    L = gu.pack_layer(lay)
    L.set_budget(r)
    for max_a in (1024, 0):
        L.set_decode(max_a)
        batches = [gen.make_batch(sh, 64, np.random.default_rng(300 + i)) for i in range(6)]
        hx = [(fx.bf16_from_bits(b.x, "cpu").pin_memory(), torch.from_numpy(b.topk_ids).pin_memory(),
               torch.from_numpy(b.topk_w).pin_memory()) for b in batches]
        hy = [torch.empty((64, sh.d), dtype=torch.bfloat16).pin_memory() for _ in batches]
        for i in range(6):
            L.moe_ffn_host(*hx[i], hy[i])
        torch.cuda.synchronize()
        assert L.device_flags() == 0
        for i, b in enumerate(batches):
            y = gen.bf16_bits_to_f32(hy[i].view(torch.int16).numpy().view(np.uint16)).astype(np.float64)
            gu.check_close(y, gu.oracle_ffn(lay, b, r), f"host call {i} decode_max={max_a}")


def test_errors_and_state():
    import torch
    import gpu_util as gu
    fx = _fx()
    sh, lay, b, rng = _c1()
    L = gu.pack_layer(lay)
    x, ids, w = gu.to_dev(b.x), torch.from_numpy(b.topk_ids).cuda(), torch.from_numpy(b.topk_w).cuda()
    with pytest.raises(fx.FxmError) as ei:
        L.moe_ffn(x, ids, w)
    assert ei.value.name == "FXM_ESTATE"
    with pytest.raises(fx.FxmError) as ei:
        L.set_budget(np.full(sh.E, sh.I + 1, np.int32))
    assert ei.value.name == "FXM_EBUDGET"
    L.set_budget(np.full(sh.E, sh.I, np.int32))
    small_ws = torch.empty(4096, dtype=torch.uint8, device="cuda")
    off = (-small_ws.data_ptr()) % 1024
    with pytest.raises(fx.FxmError) as ei:
        L.moe_ffn(x, ids, w, workspace=small_ws[off:off + 2048])
    assert ei.value.name == "FXM_EWORKSPACE"
    bad = ids.clone()
    bad[3, 1] = 99
    L.moe_ffn(x, bad, w)
    torch.cuda.synchronize()
    assert L.device_flags() & 1
    # T = 0 is a no-op
    L.moe_ffn(x[:0], ids[:0], w[:0])


# ------------------------------------------------------------------------------- FFN, paper-shaped sizes
N_SAMPLE = 512            # prefill shapes are checked on >= 512 sampled token rows (rows of y are independent)


def _rows_sample(T, n, seed):
    return np.sort(np.random.default_rng(seed).choice(T, size=min(n, T), replace=False)).astype(np.int32)


@pytest.mark.parametrize("T,decode", [(1, True), (16, True), (1, False), (16, False), (4096, None)])
@pytest.mark.parametrize("r", [704, 1408])
def test_c2_qwen15_shaped(T, r, decode):
    """C2 (BASELINE.json configs[1]): d=2048, E=60, top-4, I=1408, uniform r_e.
    T<=16: every row; T=4096: grouping indices in full + 512 sampled rows (rows of y are independent)."""
    import torch
    import gpu_util as gu
    lay, b, rng = gen.config("C2", T=T)
    sh = gen.SHAPES["C2"]
    rt = gen.table_uniform(sh, r)
    L = gu.pack_layer(lay)
    y = gu.run_ffn(L, b, rt, decode=decode)
    assert L.launches_per_ffn() == (1 if decode else 4)
    rows = None if T <= 16 else _rows_sample(T, N_SAMPLE, 11)
    ref = gu.oracle_ffn(lay, b, rt, rows=rows)
    gu.check_close(y if rows is None else y[rows], ref, f"C2 T={T} r={r}")
    got = [t.cpu().numpy() for t in L.route(torch.from_numpy(b.topk_ids).cuda())]
    for g, rr in zip(got, oracle.route(b.topk_ids, sh.E)):
        assert np.array_equal(g, rr)


def test_c3_deepseek_shaped_skewed_heterogeneous():
    """C3: d=2048, E=64, top-6, I=1408, T=8192, skewed load (mu_e + eps reading), per-expert r_e with mean 60 %;
    512 sampled rows and the grouping indices in full."""
    import torch
    import gpu_util as gu
    lay, b, rng = gen.config("C3")
    sh = gen.SHAPES["C3"]
    r = gen.table_mean_ratio(sh, rng, 0.6)
    L = gu.pack_layer(lay)
    y = gu.run_ffn(L, b, r)
    rows = _rows_sample(8192, N_SAMPLE, 12)
    gu.check_close(y[rows], gu.oracle_ffn(lay, b, r, rows=rows), "C3")
    got = [t.cpu().numpy() for t in L.route(torch.from_numpy(b.topk_ids).cuda())]
    for g, rr in zip(got, oracle.route(b.topk_ids, sh.E)):
        assert np.array_equal(g, rr)


def _c4_tables(sh, rng):
    """Every budget table BASELINE.json configs[3] names: uniform 0/25/40/50/75 %, the heterogeneous nested-descent
    tables at the same budgets, and the Fig. 6-like bimodal table."""
    tabs = [(f"U{int(round(100 * (1 - w / sh.I)))}", gen.table_uniform(sh, w)) for w in (2560, 1920, 1536, 1280, 640)]
    het = gen.tables_nested_descent(sh, rng)
    tabs += [(f"H{int(round(100 * p))}", t) for p, t in zip(gen.C4_PRUNED, het)]
    tabs.append(("fig6", gen.table_fig6_like(sh, rng)))
    return tabs


@pytest.mark.parametrize("T,decode", [(1, None), (64, None), (64, False), (8192, None)])
def test_c4_qwen2_57b_shaped_budget_sweep(T, decode):
    """C4: d=3584, E=64, top-8, I=2560 at ALL budgets of the contract: uniform and heterogeneous nested tables at
    0/25/40/50/75 % pruned plus the Fig. 6-like table.  T=1 and T=64: every row; T=8192: 512 sampled rows."""
    import gpu_util as gu
    lay, b, rng = gen.config("C4", T=T)
    sh = gen.SHAPES["C4"]
    L = gu.pack_layer(lay)
    rows = None if T <= 64 else _rows_sample(T, N_SAMPLE, 13)
    for name, tab in _c4_tables(sh, rng):
        y = gu.run_ffn(L, b, tab, decode=decode)
        assert L.launches_per_ffn() == (4 if (decode is False or T > 64) else 1)
        ref = gu.oracle_ffn(lay, b, tab, rows=rows)
        gu.check_close(y if rows is None else y[rows], ref, f"C4 T={T} table {name}")


def test_c5_switching_interleaved_decode_prefill_on_c4_layer():
    """C5 (BASELINE.json configs[4]) in miniature: 40 interleaved decode (T=32) / prefill (T=4096) calls on the C4-shaped
    layer, a different registered nested table selected before EVERY call (fxm_select_budget: host-only), no host
    synchronisation in between, one shared workspace sized for the larger T.  Sampled rows of every output against
    the oracle at the table that call used."""
    import torch
    import gpu_util as gu
    fx = _fx()
    sh = gen.SHAPES["C5"]
    lay = gen.layer_for("C5", 0)
    tabs = gen.tables_nested_descent(sh, np.random.default_rng([0, 3]))
    L = gu.pack_layer(lay)
    L.register_budgets(tabs, require_nested=True)
    L.set_decode()                                               # library default: T=32 -> fused decode kernel, T=4096 -> general path
    pools = {}
    for T in (32, 4096):
        pools[T] = []
        for i in range(2):
            _, bt, _ = gen.config("C5", T=T, seed=40 + i, layer=False)
            pools[T].append((bt, gu.to_dev(bt.x), torch.from_numpy(bt.topk_ids).cuda(), torch.from_numpy(bt.topk_w).cuda()))
    L.workspace(4096, sh.k)
    rng = np.random.default_rng(9)
    calls, prev = [], -1
    for i in range(40):
        bi = int(rng.integers(len(tabs)))
        while bi == prev:
            bi = int(rng.integers(len(tabs)))
        prev = bi
        T = 32 if i % 2 == 0 else 4096
        bt, x, ids, w = pools[T][(i // 2) % 2]
        L.select_budget(bi)
        y = L.moe_ffn(x, ids, w)
        assert L.launches_per_ffn() == (1 if T == 32 else 4)
        calls.append((i, T, bi, bt, y))
    torch.cuda.synchronize()
    assert L.device_flags() == 0
    for i, T, bi, bt, y in calls:
        rows = _rows_sample(T, 32 if T == 32 else 12, 100 + i)
        yv = gen.bf16_bits_to_f32(fx.bf16_to_bits(y[torch.from_numpy(rows.astype(np.int64)).cuda()])).astype(np.float64)
        gu.check_close(yv, gu.oracle_ffn(lay, bt, tabs[bi], rows=rows), f"C5 call {i} T={T} budget {bi}")


# ------------------------------------------------------------------------------------ robustness items
def test_host_entry_point_interleaved_sizes_share_one_workspace():
    """fxm_moe_ffn_host with T=4096 and T=32 calls back to back on ONE workspace sized for the larger T and no host
    synchronisation: the staging area of a call must never land on memory the previous call still uses."""
    import torch
    import gpu_util as gu
    fx = _fx()
    lay, _, rng = gen.config("C2", T=32)
    sh = gen.SHAPES["C2"]
    r = gen.table_uniform(sh, 704)
    L = gu.pack_layer(lay)
    L.set_budget(r)
    L.workspace_host(4096, sh.k)
    seq = [4096, 32, 32, 4096, 4096, 32, 4096, 32]
    batches, hx, hy = [], [], []
    for i, T in enumerate(seq):
        _, b, _ = gen.config("C2", T=T, seed=70 + i, layer=False)
        batches.append(b)
        hx.append((fx.bf16_from_bits(b.x, "cpu").pin_memory(), torch.from_numpy(b.topk_ids).pin_memory(),
                   torch.from_numpy(b.topk_w).pin_memory()))
        hy.append(torch.empty((T, sh.d), dtype=torch.bfloat16).pin_memory())
    for i in range(len(seq)):
        L.moe_ffn_host(*hx[i], hy[i])
    torch.cuda.synchronize()
    assert L.device_flags() == 0
    for i, (T, b) in enumerate(zip(seq, batches)):
        rows = _rows_sample(T, 32, 200 + i)
        y = gen.bf16_bits_to_f32(hy[i].view(torch.int16).numpy().view(np.uint16)[rows]).astype(np.float64)
        gu.check_close(y, gu.oracle_ffn(lay, b, r, rows=rows), f"host call {i} T={T}")


def test_graph_replay_keeps_the_captured_table_slot():
    """include/flexmoe.h: a captured call is bound to the table SLOT that was current at capture time;
    fxm_select_budget afterwards does not change a replay, fxm_set_budget (which rewrites the captured slot) does."""
    import torch
    import gpu_util as gu
    fx = _fx()
    sh, lay, b, rng = _c1()
    tabs = np.array([[512] * 8, [256, 128, 192, 64, 512, 64, 128, 0], [128, 64, 64, 64, 256, 0, 64, 0]], np.int32)
    L = gu.pack_layer(lay)
    L.set_decode(0)
    L.register_budgets(tabs, require_nested=True)
    x, ids, w = gu.to_dev(b.x), torch.from_numpy(b.topk_ids).cuda(), torch.from_numpy(b.topk_w).cuda()
    y = torch.empty((b.x.shape[0], sh.d), dtype=torch.bfloat16, device="cuda")
    L.select_budget(1)
    L.moe_ffn(x, ids, w, out=y)
    torch.cuda.synchronize()
    g = torch.cuda.CUDAGraph()
    side = torch.cuda.Stream()
    with torch.cuda.stream(side):
        with torch.cuda.graph(g, stream=side):
            L.moe_ffn(x, ids, w, out=y)
    L.select_budget(2)                                           # host-only: the graph still reads registered table 1
    g.replay()
    torch.cuda.synchronize()
    gu.check_close(gen.bf16_bits_to_f32(fx.bf16_to_bits(y)).astype(np.float64), gu.oracle_ffn(lay, b, tabs[1]), "replay after select")
    y2 = L.moe_ffn(x, ids, w)                                    # an eager call does read table 2
    torch.cuda.synchronize()
    gu.check_close(gen.bf16_bits_to_f32(fx.bf16_to_bits(y2)).astype(np.float64), gu.oracle_ffn(lay, b, tabs[2]), "eager after select")


def test_misaligned_y_is_rejected_not_faulted():
    """y is written with 16-byte stores: an 8-byte-aligned y must come back as FXM_EINVAL, never as a misaligned-address fault."""
    import torch
    import gpu_util as gu
    fx = _fx()
    sh, lay, b, rng = _c1()
    L = gu.pack_layer(lay)
    L.set_budget(np.full(sh.E, sh.I, np.int32))
    x, ids, w = gu.to_dev(b.x), torch.from_numpy(b.topk_ids).cuda(), torch.from_numpy(b.topk_w).cuda()
    buf = torch.empty(b.x.shape[0] * sh.d + 8, dtype=torch.bfloat16, device="cuda")
    assert buf.data_ptr() % 16 == 0
    y_bad = buf[4:4 + b.x.shape[0] * sh.d].view(b.x.shape[0], sh.d)      # 8-byte aligned only
    for dec in (0, 1024):
        L.set_decode(dec)
        with pytest.raises(fx.FxmError) as ei:
            L.moe_ffn(x, ids, w, out=y_bad)
        assert ei.value.name == "FXM_EINVAL"
    torch.cuda.synchronize()
    assert L.device_flags() == 0


# ------------------------------------------------------------------------------ NEXT-1: offline clipping
@pytest.mark.parametrize("d,E,k,I,T", [(256, 8, 2, 512, 64), (192, 5, 3, 208, 300)])
def test_offline_clipped_export_reload_and_forward(d, E, k, I, T):
    """Export a fixed-budget blob (retained prefix tiles only), move it through HOST memory (as a checkpoint file
    would), reload it and run the forward with static widths:
    (1) the blob's weights are bit-exact: unpack_prefix on the reloaded layer == oracle.pack()[:r_e];
    (2) its size is the linear law of Table 2: 6 d bytes per retained 64-channel block + a constant;
    (3) the forward on it equals the oracle (and the online layer at the same table) within tolerance, on both the
        general path and the decode kernel; (4) nested sub-budgets of the clipped checkpoint work, wider ones are refused."""
    import torch
    import gpu_util as gu
    fx = _fx()
    sh, lay, rng = _small_layer(31 + d, d, E, k, I, w_std=0.08)
    b = gen.make_batch(sh, T, rng, expert_bias_std=1.0)
    L = gu.pack_layer(lay)
    r = (rng.integers(0, I // 16 + 1, size=E) * 16).astype(np.int32)
    r[0] = I
    r[E - 1] = 0
    r[1] = 40 if I >= 48 else 16                                  # a width that is not a multiple of 64
    blob = L.export_clipped(r)
    torch.cuda.synchronize()
    host = blob.cpu()                                            # "write the checkpoint"
    E2, d2, I2, r2 = fx.Layer.parse_clipped_header(host.numpy().tobytes()[:2048])
    assert (E2, d2, I2) == (E, d, I) and np.array_equal(r2, r)
    nblk = int(sum(-(-int(x) // 64) for x in r))
    gu_b = nblk * (d // 64) * 16384
    dn_b = nblk * (-(-d // 128)) * 16384
    assert 2048 + gu_b + dn_b <= blob.numel() <= 2048 + gu_b + dn_b + 32 * 1024
    raw = torch.empty(host.numel() + 1024, dtype=torch.uint8, device="cuda")
    off = (-raw.data_ptr()) % 1024
    dev = raw[off:off + host.numel()]
    dev.copy_(host)                                              # "load the checkpoint"
    Lc = fx.Layer.load_clipped(dev, E2, d2, I2, r2)
    Gt, Ut, Dt = oracle.pack(lay.W_gate, lay.W_up, lay.W_down, lay.channel_rank)
    for e in range(E):
        if r[e] == 0:
            continue
        Wg, Wu, Wd = Lc.unpack_prefix(e, int(r[e]))
        torch.cuda.synchronize()
        assert np.array_equal(fx.bf16_to_bits(Wg), Gt[e, :r[e]])
        assert np.array_equal(fx.bf16_to_bits(Wu), Ut[e, :r[e]])
        assert np.array_equal(fx.bf16_to_bits(Wd), Dt[e, :, :r[e]])
    with pytest.raises(fx.FxmError) as ei:
        Lc.unpack_prefix(1, int(r[1]) + 16)
    assert ei.value.name == "FXM_EBUDGET"
    x, ids, w = gu.to_dev(b.x), torch.from_numpy(b.topk_ids).cuda(), torch.from_numpy(b.topk_w).cuda()
    ref = gu.oracle_ffn(lay, b, r)
    for dec in (0, 1024):
        if dec and T * k > 1024:
            continue
        Lc.set_decode(dec)
        y = Lc.moe_ffn(x, ids, w)                                # static widths: usable right after the load
        torch.cuda.synchronize()
        assert Lc.device_flags() == 0
        gu.check_close(gen.bf16_bits_to_f32(fx.bf16_to_bits(y)).astype(np.float64), ref, f"clipped layer decode_max={dec}")
        L.set_decode(dec)
        L.set_budget(r)
        yo = L.moe_ffn(x, ids, w)
        torch.cuda.synchronize()
        # same kernels on the same tiles; what may differ is the ORDER in which a token's k expert contributions reach the
        # fp32 accumulator (scatter-add with atomics), i.e. the last bit before the one rounding to bf16
        yf, yof = y.float(), yo.float()
        assert (yf - yof).abs().max().item() <= 2.0 ** -7 * yof.abs().max().item()
        assert (y != yo).float().mean().item() < 0.02
    sub = (r // 2 // 16 * 16).astype(np.int32)                   # a nested sub-budget of the checkpoint
    Lc.set_decode(0)
    Lc.set_budget(sub)
    y = Lc.moe_ffn(x, ids, w)
    torch.cuda.synchronize()
    gu.check_close(gen.bf16_bits_to_f32(fx.bf16_to_bits(y)).astype(np.float64), gu.oracle_ffn(lay, b, sub), "nested sub-budget")
    wider = r.copy()
    wider[E - 1] = 16
    with pytest.raises(fx.FxmError) as ei:
        Lc.set_budget(wider)
    assert ei.value.name == "FXM_EBUDGET"


def test_offline_clipped_c2_shape_sampled_rows():
    """NEXT-1 at a paper-shaped size: C2 layer exported at r=704 (50 %), forward at T=4096 on the reloaded blob,
    512 sampled rows vs the oracle; blob bytes = half of the retained-weight bytes of the full layer + constants."""
    import torch
    import gpu_util as gu
    fx = _fx()
    lay, b, rng = gen.config("C2", T=4096)
    sh = gen.SHAPES["C2"]
    r = gen.table_uniform(sh, 704)
    L = gu.pack_layer(lay)
    blob = L.export_clipped(r)
    torch.cuda.synchronize()
    full_w = 3 * sh.E * sh.I * sh.d * 2
    assert abs(blob.numel() - full_w // 2) < 64 * 1024
    del L
    Lc = fx.Layer.load_clipped(blob, sh.E, sh.d, sh.I, r)
    y = Lc.moe_ffn(gu.to_dev(b.x), torch.from_numpy(b.topk_ids).cuda(), torch.from_numpy(b.topk_w).cuda())
    torch.cuda.synchronize()
    assert Lc.device_flags() == 0
    rows = _rows_sample(4096, N_SAMPLE, 21)
    yv = gen.bf16_bits_to_f32(fx.bf16_to_bits(y[torch.from_numpy(rows.astype(np.int64)).cuda()])).astype(np.float64)
    gu.check_close(yv, gu.oracle_ffn(lay, b, r, rows=rows), "C2 clipped r=704")


# ------------------------------------------------------------ NEXT-3 (part): shared-expert add
@pytest.mark.parametrize("decode", [False, True])
def test_shared_expert_output_is_added_before_the_rounding(decode):
    """y = bf16( routed(x) + y_shared ): the add happens in fp32 on the accumulator, so the result has ONE rounding."""
    import torch
    import gpu_util as gu
    fx = _fx()
    sh, lay, b, rng = _c1()
    r = gen.table_c1(sh, rng)
    L = gu.pack_layer(lay)
    L.set_budget(r)
    L.set_decode(1024 if decode else 0)
    ys_bits = gen.f32_to_bf16_bits(rng.standard_normal((b.x.shape[0], sh.d)).astype(np.float32) * 0.05)
    y = L.moe_ffn(gu.to_dev(b.x), torch.from_numpy(b.topk_ids).cuda(), torch.from_numpy(b.topk_w).cuda(),
                  y_shared=gu.to_dev(ys_bits))
    torch.cuda.synchronize()
    assert L.device_flags() == 0 and L.launches_per_ffn() == (1 if decode else 4)
    ref = gu.oracle_ffn(lay, b, r) + gen.bf16_bits_to_f32(ys_bits).astype(np.float64)
    got = gen.bf16_bits_to_f32(fx.bf16_to_bits(y)).astype(np.float64)
    gu.check_close(got, ref, "routed + shared")
    # one rounding: |y - ref| <= half an ulp of bf16 at ref (2^-9 relative) plus the H rounding's contribution
    assert np.abs(got - ref).max() <= 2.0 ** -8 * np.abs(ref).max()


def test_general_path_small_T_many_calls_on_c4_layer():
    """Regression (round 2): at decode-sized T on the C4-shaped layer the token tiles are 16-32 rows, so some of GEMM-1's
    six gather warps have no 4-row group to bring.  They used to poll the stage barriers anyway; a warp that only polls takes
    part in no handshake, the pipeline lapped it, its parity wait aliased and the call ended in the wait time-out (about one
    call in 100: "unspecified launch failure", device flag bit 1).  300 calls of the four-launch path at T=32 / 64, a buffer
    larger than L2 rewritten between calls, every output compared on the device with the oracle's rows of that batch."""
    import torch
    import gpu_util as gu
    fx = _fx()
    sh = gen.SHAPES["C4"]
    lay = gen.layer_for("C4", 0)
    L = gu.pack_layer(lay)
    r = gen.table_uniform(sh, 640)
    L.set_budget(r)
    L.set_decode(0)                                              # never the fused decode kernel
    flush = torch.zeros(256 << 20, dtype=torch.uint8, device="cuda")
    cases = []
    for T, seed in ((32, 61), (64, 62)):
        _, b, _ = gen.config("C4", T=T, seed=seed, layer=False)
        ref = torch.from_numpy(gu.oracle_ffn(lay, b, r)).cuda()
        cases.append((gu.to_dev(b.x), torch.from_numpy(b.topk_ids).cuda(), torch.from_numpy(b.topk_w).cuda(), ref,
                      float(ref.abs().max())))
    for i in range(300):
        x, ids, w, ref, scale = cases[i % 2]
        flush.add_(1)
        y = L.moe_ffn(x, ids, w)
        assert L.launches_per_ffn() == 4
        err = float((y.double() - ref).abs().max())
        assert err <= gu.TOL_MAX * scale, f"call {i}: max err {err:.3e} > {gu.TOL_MAX}*{scale:.3e}"
    torch.cuda.synchronize()
    assert L.device_flags() == 0


def test_host_entry_point_with_deferred_output_copies():
    """fxm_moe_ffn_host_pipelined + fxm_host_flush: y of call i travels back on the library's second stream under the
    kernels of call i+1.  Ten calls of alternating sizes (T=64 / T=300: the staging layout changes), every third one through
    the in-stream entry point, no host synchronisation before the flush; every output against the oracle."""
    import torch
    import gpu_util as gu
    fx = _fx()
    sh, lay, b0, rng = _c1()
    r = gen.table_c1(sh, rng)
    L = gu.pack_layer(lay)
    L.set_budget(r)
    L.set_decode()
    sizes = [64, 64, 64, 300, 300, 64, 300, 300, 300, 64]
    batches = [gen.make_batch(sh, T, np.random.default_rng(500 + i)) for i, T in enumerate(sizes)]
    hx = [(fx.bf16_from_bits(b.x, "cpu").pin_memory(), torch.from_numpy(b.topk_ids).pin_memory(),
           torch.from_numpy(b.topk_w).pin_memory()) for b in batches]
    hy = [torch.zeros((T, sh.d), dtype=torch.bfloat16).pin_memory() for T in sizes]
    L.workspace_host(300, sh.k)                                  # one workspace for both sizes
    for i in range(len(sizes)):
        L.moe_ffn_host(*hx[i], hy[i], pipelined=(i % 3 != 2))
    L.host_flush()
    torch.cuda.synchronize()
    assert L.device_flags() == 0
    for i, b in enumerate(batches):
        y = gen.bf16_bits_to_f32(hy[i].view(torch.int16).numpy().view(np.uint16)).astype(np.float64)
        gu.check_close(y, gu.oracle_ffn(lay, b, r), f"host call {i} T={sizes[i]}")
