"""Host logic of bench.py (no GPU): the algorithmic work model of SURVEY.md 8(d), the roofline arithmetic, and the reader of
the committed ncu extract that supplies `roofline.traffic`."""
import os
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import bench


def test_work_model_matches_the_survey_table_for_c4():
    """SURVEY.md 8(d), row "C4 0 %, T=8192": 3607.8 GFLOP, 3523.2 MB of weights; 75 %: a quarter of both."""
    d, E, k, I, T = 3584, 64, 8, 2560, 8192
    ids = (np.arange(T * k, dtype=np.int64).reshape(T, k) % E).astype(np.int32)      # every expert gets T*k/E assignments
    for r_w, gflop, wmb in ((2560, 3607.8, 3523.2), (640, 901.9, 880.8)):
        w = bench.work_model(ids, np.full(E, r_w, np.int32), d, T, k)
        assert abs(w["flops"] / 1e9 - gflop) < 0.1
        assert abs(6.0 * d * w["R_act"] / 1e6 - wmb) < 0.1
        assert w["bytes"] == 6.0 * d * w["R_act"] + 4.0 * T * d + 8.0 * T * k       # weights once + x + y + ids / weights
        assert w["gemm1_flops"] + w["gemm2_flops"] == w["flops"]
        assert w["S"] == T * k * r_w


def test_work_model_counts_only_active_experts_and_their_widths():
    d, E, k, T = 256, 8, 2, 4
    ids = np.array([[0, 1], [0, 1], [1, 5], [5, 0]], np.int32)
    r = np.array([512, 128, 512, 512, 512, 64, 512, 512], np.int32)
    w = bench.work_model(ids, r, d, T, k)
    assert w["R_act"] == 512 + 128 + 64                         # experts 0, 1, 5 are active
    assert w["S"] == 3 * 512 + 3 * 128 + 2 * 64                 # n_e * r_e


def test_roofline_takes_the_larger_floor():
    peaks = {"hbm_gbs": 6500.0, "bf16_tflops": 1600.0, "bf16_tflops_sustained": 1400.0}
    t, bound = bench.roof_time_s(1.6e12, 1e6, peaks)
    assert bound == "tensor" and abs(t - 1e-3) < 1e-12
    t, bound = bench.roof_time_s(1e6, 6.5e9, peaks)
    assert bound == "hbm" and abs(t - 1e-3) < 1e-12
    t, _ = bench.roof_time_s(1.4e12, 1.0, peaks, "bf16_tflops_sustained")
    assert abs(t - 1e-3) < 1e-12


def test_ncu_traffic_reads_the_committed_extract_of_the_headline_workload_only():
    v, src = bench.ncu_traffic("C4", 8192, "2560", "gemm1_swiglu")
    path = os.path.join(ROOT, "profiles", "r02d_ncu_full_pair_c4_T8192_r2560.csv")
    if os.path.exists(path):
        assert src == "profiles/r02d_ncu_full_pair_c4_T8192_r2560.csv"
        assert 2.4e9 < v < 8e9                                  # gate/up weights once is 2.35 GB; the capture has ~4.7 GB
    else:
        assert v is None
    assert bench.ncu_traffic("C2", 4096, "704", "gemm1_swiglu") == (None, None)      # no capture of that workload: null
    assert bench.ncu_traffic("C4", 8192, "2560", "route") == (None, None)
