"""Helpers shared by the GPU parity tests: move seeded inputs to the device, call the C ABI through the
binding, and compare with the CPU oracle under north_star's tolerances.  Test infrastructure only."""
import numpy as np

import oracle
from paper_2606_27866_b200 import flexmoe as fx
from paper_2606_27866_b200 import inputs as gen

# north_star: bf16 inputs, fp32 accumulate
TOL_MAX = 1e-2      # max|y - ref| <= TOL_MAX * max|ref|
TOL_L2 = 5e-3       # ||y - ref||_2 / ||ref||_2 <= TOL_L2


def to_dev(bits):
    return fx.bf16_from_bits(bits, "cuda")


def pack_layer(lay, identity=False):
    import torch
    L = fx.Layer.pack(to_dev(lay.W_gate), to_dev(lay.W_up), to_dev(lay.W_down),
                      None if identity else lay.channel_rank)
    torch.cuda.synchronize()
    return L


def run_ffn(L, batch, r, impl=fx.IMPL_TCGEN05, tile_n=0, decode=None):
    """decode: None = the library's default choice, False = never the fused decode kernel (general six-launch
    path even for tiny T), True = the fused decode kernel whenever T*k <= 1024."""
    import torch
    L.set_impl(impl)
    L.set_tile_n(tile_n)
    if decode is None:
        L.set_decode()
    else:
        L.set_decode(1024 if decode else 0)
    L.set_budget(r)
    x = to_dev(batch.x)
    ids = torch.from_numpy(batch.topk_ids).cuda()
    w = torch.from_numpy(batch.topk_w).cuda()
    y = L.moe_ffn(x, ids, w)
    torch.cuda.synchronize()
    flags = L.device_flags()
    assert flags == 0, f"device flags {flags:#x}"
    return gen.bf16_bits_to_f32(fx.bf16_to_bits(y)).astype(np.float64)


_PACK_CACHE = {}


def oracle_packed(lay):
    """oracle.pack of a layer, memoised on the layer object (the 3.5 GB C4 layer takes a while)."""
    key = id(lay)
    if key not in _PACK_CACHE:
        _PACK_CACHE.clear()
        _PACK_CACHE[key] = (lay, oracle.pack(lay.W_gate, lay.W_up, lay.W_down, lay.channel_rank))
    return _PACK_CACHE[key][1]


def oracle_ffn(lay, batch, r, rows=None):
    Gt, Ut, Dt = oracle_packed(lay)
    return oracle.moe_ffn(batch.x, Gt, Ut, Dt, r, batch.topk_ids, batch.topk_w, rows=rows)


def check_close(y, ref, what=""):
    scale = np.abs(ref).max()
    err = np.abs(y - ref).max()
    l2 = np.linalg.norm(y - ref) / max(np.linalg.norm(ref), 1e-300)
    assert np.isfinite(y).all(), f"{what}: non-finite output"
    assert err <= TOL_MAX * scale, f"{what}: max err {err:.3e} > {TOL_MAX}*{scale:.3e}"
    assert l2 <= TOL_L2, f"{what}: rel L2 {l2:.3e} > {TOL_L2}"
    return err / max(scale, 1e-300), l2
