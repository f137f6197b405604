"""N>1 path of bench.py on CPU: world_size-2 gloo processes (replicas of the layer, tokens
sharded, no data-path collective; the only collective is the MAX over ranks of the timed regions).

Checked: (1) ranks draw disjoint token batches but identical layer weights, (2) rows of y are independent, so the
concatenation of the per-rank oracle outputs equals the oracle on the concatenated tokens bit for bit, (3)
bench.aggregate takes the max over ranks and sums tokens, (4) bench.py --impl reference prints on rank 0 only."""
import json
import os
import subprocess
import sys

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _worker(rank, world, port, out_dir):
    sys.path.insert(0, ROOT)
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    import torch
    import torch.distributed as dist
    import bench
    import oracle
    from paper_2606_27866_b200 import inputs as gen
    dist.init_process_group("gloo", rank=rank, world_size=world)
    T = 16
    sh = gen.SHAPES["C1"]
    lay = gen.layer_for("C1", 0)                               # same weights on every rank
    (b, rng), = bench.host_batches(gen, "C1", T, 1, bench.rank_seed0(rank))
    r = gen.table_uniform(sh, 384)
    packed = oracle.pack(lay.W_gate, lay.W_up, lay.W_down, lay.channel_rank)
    y = oracle.moe_ffn(b.x, *packed, r, b.topk_ids, b.topk_w)
    # gather every rank's inputs and outputs on every rank (test plumbing only; the data path has no collective)
    def gather(a):
        t = torch.from_numpy(np.ascontiguousarray(a))
        parts = [torch.empty_like(t) for _ in range(world)]
        dist.all_gather(parts, t)
        return [p.numpy() for p in parts]
    xs, ids, ws, ys = gather(b.x.view(np.int32)), gather(b.topk_ids), gather(b.topk_w), gather(y)
    wsum = gather(np.array([int(lay.W_gate.astype(np.int64).sum())], np.int64))
    ms, tokens = bench.aggregate([10.0 + rank, 5.0 - rank], T, 7, world, dist)
    if rank == 0:
        x_all = np.concatenate(xs).view(np.uint16)
        y_all = oracle.moe_ffn(x_all, *packed, r, np.concatenate(ids), np.concatenate(ws))
        res = {"weights_equal": bool(wsum[0][0] == wsum[1][0]),
               "tokens_differ": bool(not np.array_equal(xs[0], xs[1])),
               "sharded_equals_whole": bool(np.array_equal(y_all, np.concatenate(ys))),
               "ms": ms, "tokens": tokens}
        with open(os.path.join(out_dir, "res.json"), "w") as f:
            json.dump(res, f)
    dist.barrier()
    dist.destroy_process_group()


def test_two_rank_gloo_sharding_and_max_over_ranks(tmp_path):
    import torch.multiprocessing as mp
    port = 29500 + os.getpid() % 2000
    mp.spawn(_worker, args=(2, port, str(tmp_path)), nprocs=2, join=True)
    res = json.load(open(tmp_path / "res.json"))
    assert res["weights_equal"] and res["tokens_differ"] and res["sharded_equals_whole"]
    assert res["ms"] == [11.0, 5.0]                            # max over ranks of each timed region
    assert res["tokens"] == 2 * 16 * 7                         # whole-job tokens: summed over ranks


def test_reference_arm_prints_on_rank_zero_only():
    env = dict(os.environ, RANK="1", WORLD_SIZE="2", LOCAL_RANK="1")
    out = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2"],
                         capture_output=True, text=True, env=env, timeout=120)
    assert out.returncode == 0 and out.stdout.strip() == ""
