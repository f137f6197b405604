"""fxm_saliency_static, the entry point that allocates nothing (its scratch is a fixed 8 MB device array inside the library):
checked against the existing fxm_saliency path (caller-provided workspace) on the same inputs.  This file is named so that
pytest collects it LAST: the suite runs with `pytest -x`, and a failure here must not hide any other test."""
import ctypes

import numpy as np
import pytest

from paper_2606_27866_b200 import inputs as gen

pytestmark = pytest.mark.gpu


def _bf16_dev(rng, shape, std):
    from paper_2606_27866_b200 import flexmoe as fx
    return fx.bf16_from_bits(gen.f32_to_bf16_bits(rng.standard_normal(shape, dtype=np.float32) * np.float32(std)), "cuda")


def _inputs(E, d, I, B, seed):
    rng = np.random.default_rng(seed)
    W = [_bf16_dev(rng, (E, I, d), 0.05), _bf16_dev(rng, (E, I, d), 0.05), _bf16_dev(rng, (E, d, I), 0.05)]
    G = [_bf16_dev(rng, (B, E, I, d), 1.0), _bf16_dev(rng, (B, E, I, d), 1.0), _bf16_dev(rng, (B, E, d, I), 1.0)]
    return W + G


def test_saliency_static_matches_the_workspace_path_on_two_calls_in_a_row():
    """Two calls in a row on one stream, the second on a SMALLER and different problem, so the shared scratch still holds the
    first call's partial sums when it starts (nothing may depend on the array's old contents).  Each output is compared with
    fxm_saliency on the same inputs: same kernels, same fixed summation order, so the tolerance of the saliency parity test
    (1e-5 of max|ref|) is met with room -- and in fact bit for bit.  The second call must not change the free device memory."""
    import torch
    from paper_2606_27866_b200 import flexmoe as fx
    cases = [(60, 512, 1408, 2, 71), (5, 192, 80, 3, 72)]        # 5.7 MB of the 8 MB scratch, then 27 KB of it
    ins = [_inputs(*c) for c in cases]
    outs = [torch.full((c[0], c[2]), float("nan"), dtype=torch.float32, device="cuda") for c in cases]
    refs = [fx.saliency(*a) for a in ins]                        # the existing path (torch-allocated workspace)
    torch.cuda.synchronize()
    fx.saliency_static(*ins[0], out=outs[0])                     # first call: also looks the array's device address up
    torch.cuda.synchronize()
    free0 = torch.cuda.mem_get_info()[0]
    fx.saliency_static(*ins[1], out=outs[1])                     # second call, straight after, stale scratch
    fx.saliency_static(*ins[0], out=outs[0])                     # and the first problem again over the second's leftovers
    torch.cuda.synchronize()
    assert torch.cuda.mem_get_info()[0] >= free0, "the no-allocation entry point changed the free device memory"
    for o, r, c in zip(outs, refs, cases):
        o, r = o.cpu().numpy(), r.cpu().numpy()
        assert np.isfinite(o).all() and (r > 0).all()
        assert np.abs(o - r).max() <= 1e-5 * np.abs(r).max(), f"case {c}"
        assert np.array_equal(o, r), f"case {c}: same kernels and summation order, expected identical bits"


def test_saliency_static_rejects_problems_beyond_its_scratch_and_bad_arguments():
    """C4-shaped weights (E=64, I=2560) need 11.1 MB of partial sums > 8 MB: FXM_ELIMIT, decided from the shape alone (before
    any pointer is touched or anything is launched)."""
    import torch
    from paper_2606_27866_b200 import flexmoe as fx
    L = fx.lib()
    n = ctypes.c_size_t()
    assert L.fxm_saliency_workspace_bytes(64, 3584, 2560, ctypes.byref(n)) == 0 and n.value > fx.SALIENCY_STATIC_BYTES
    assert L.fxm_saliency_workspace_bytes(60, 2048, 1408, ctypes.byref(n)) == 0 and n.value <= fx.SALIENCY_STATIC_BYTES
    buf = torch.zeros(4096, dtype=torch.uint8, device="cuda")
    p = buf.data_ptr()
    assert L.fxm_saliency_static(64, 3584, 2560, p, p, p, p, p, p, 1, p, None) == 10          # FXM_ELIMIT
    assert L.fxm_status_string(10).decode().startswith("FXM_ELIMIT")
    assert L.fxm_saliency_static(8, 256, 512, p, p, p, p, p, p, 0, p, None) == 1              # B < 1: FXM_EINVAL
    assert L.fxm_saliency_static(8, 256, 512, None, p, p, p, p, p, 1, p, None) == 1           # NULL: FXM_EINVAL
    assert L.fxm_saliency_static(8, 100, 512, p, p, p, p, p, p, 1, p, None) == 2              # d % 64 != 0: FXM_ESHAPE
    torch.cuda.synchronize()
