"""Host-side multi-GPU plumbing on CPU: world_size-2 `gloo` processes.

The path shards over independent (batch, kv head) units with no data-path collective; the only
cross-rank traffic is the barrier and the max-over-ranks of the device time that bench.py reports.
Checked here: the unit split is a partition, every rank's shard -- its OWN kv heads or its own batch
element, evicted on its own with head_offset / batch_offset -- equals the corresponding slice of the
unsharded result (the oracle stands in for the device work: these processes have no GPU; the same
split on a GPU through nacl_evict_ex is tests/test_gpu_parity.py::test_shards_draw_what_the_unsharded_call_draws),
and the reductions bench.py uses agree across ranks.
"""
from __future__ import annotations

import os
import socket

import numpy as np
import pytest
import torch
import torch.multiprocessing as mp

from paper_2408_03675_b200 import CONFIGS
from paper_2408_03675_b200 import dist as nacl_dist
from paper_2408_03675_b200.inputs import make_layer_inputs


def test_shard_units_is_a_balanced_partition():
    for n in (0, 1, 4, 7, 32, 33):
        for world in (1, 2, 3, 8):
            parts = [nacl_dist.shard_units(n, r, world) for r in range(world)]
            flat = [u for p in parts for u in p]
            assert flat == list(range(n))
            sizes = [len(p) for p in parts]
            assert max(sizes) - min(sizes) <= 1


def _free_port() -> int:
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank: int, world: int, port: int, out_dir: str):
    import oracle

    os.environ.update(RANK=str(rank), LOCAL_RANK=str(rank), WORLD_SIZE=str(world), MASTER_ADDR="127.0.0.1",
                      MASTER_PORT=str(port))
    r, lr, w = nacl_dist.init(backend="gloo")
    assert (r, lr, w) == (rank, rank, world)
    cfg = CONFIGS[1].scaled(batch=1, Hq=8, Hkv=4)  # 4 independent (batch, kv head) units, G = 2
    K, V, Q, _ = make_layer_inputs(cfg, layer=0)
    Bp, Br = cfg.budgets()
    units = nacl_dist.shard_units(cfg.Hkv, rank, world)  # this rank's kv heads
    G = cfg.G
    hk = slice(units.start, units.stop)
    hq = slice(units.start * G, units.stop * G)
    # head shard (tensor parallel): the rank evicts ITS OWN kv heads and their query heads, told where they start
    # (head_offset): the Philox counter carries the global kv-head index (R10)
    Ks, Vs, Qs = K[:, hk].contiguous(), V[:, hk].contiguous(), Q[:, hq].contiguous()
    idx_sh = oracle.evict(Ks, Vs, Qs, Bp, Br, cfg.n_sink, cfg.n_recent, cfg.layer_seed(0), 0, head_offset=units.start)[2]
    np.save(os.path.join(out_dir, f"idx_{rank}.npy"), idx_sh)
    idx_no = oracle.evict(Ks, Vs, Qs, Bp, Br, cfg.n_sink, cfg.n_recent, cfg.layer_seed(0), 0)[2]
    np.save(os.path.join(out_dir, f"idxno_{rank}.npy"), idx_no)
    # batch shard (data parallel): each rank evicts its own batch element of ONE batch-2 problem, with batch_offset
    cfgb = CONFIGS[1].scaled(batch=2)
    Kb, Vb, Qb, _ = make_layer_inputs(cfgb, layer=0)
    b = nacl_dist.shard_units(cfgb.batch, rank, world)
    sl = slice(b.start, b.stop)
    idx_b = oracle.evict(Kb[sl].contiguous(), Vb[sl].contiguous(), Qb[sl].contiguous(), Bp, Br, cfgb.n_sink, cfgb.n_recent,
                         cfgb.layer_seed(0), 0, batch_offset=b.start)[2]
    np.save(os.path.join(out_dir, f"idxb_{rank}.npy"), idx_b)
    # the reductions of bench.py
    nacl_dist.barrier()
    assert nacl_dist.max_over_ranks(10.0 + rank) == 10.0 + world - 1
    assert nacl_dist.sum_over_ranks(1.0 + rank) == sum(1.0 + i for i in range(world))
    nacl_dist.barrier()
    nacl_dist.finalize()


@pytest.mark.timeout(300)
def test_two_rank_gloo_shards_match_the_unsharded_result(tmp_path):
    import oracle

    world = 2
    mp.spawn(_worker, args=(world, _free_port(), str(tmp_path)), nprocs=world, join=True)
    cfg = CONFIGS[1].scaled(batch=1, Hq=8, Hkv=4)
    K, V, Q, _ = make_layer_inputs(cfg, layer=0)
    Bp, Br = cfg.budgets()
    idx_full = oracle.evict(K, V, Q, Bp, Br, cfg.n_sink, cfg.n_recent, cfg.layer_seed(0), 0)[2]
    got = np.concatenate([np.load(tmp_path / f"idx_{r}.npy") for r in range(world)], axis=1)
    np.testing.assert_array_equal(got, idx_full)
    # without head_offset the second rank numbers its heads from 0 and draws a different sample: the offsets matter
    assert not np.array_equal(np.load(tmp_path / "idxno_1.npy"), idx_full[:, 2:])
    np.testing.assert_array_equal(np.load(tmp_path / "idxno_0.npy"), idx_full[:, :2])
    # batch shards of one batch-2 problem
    cfgb = CONFIGS[1].scaled(batch=2)
    Kb, Vb, Qb, _ = make_layer_inputs(cfgb, layer=0)
    idx_bfull = oracle.evict(Kb, Vb, Qb, Bp, Br, cfgb.n_sink, cfgb.n_recent, cfgb.layer_seed(0), 0)[2]
    gotb = np.concatenate([np.load(tmp_path / f"idxb_{r}.npy") for r in range(world)], axis=0)
    np.testing.assert_array_equal(gotb, idx_bfull)


@pytest.mark.timeout(600)
def test_bench_gpus_flag_spawns_the_ranks_itself():
    """`python bench.py --gpus 2` with no torchrun environment launches two ranks (torch.distributed.run on 127.0.0.1).
    On a box without GPUs the CUDA arm must fail loudly instead of running one rank; the oracle arm (rank 0 works, the other
    rank exits 0) runs anywhere and reports n_gpus = 2."""
    import json
    import subprocess
    import sys

    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    env = {k: v for k, v in os.environ.items() if k not in ("RANK", "LOCAL_RANK", "WORLD_SIZE", "MASTER_ADDR", "MASTER_PORT")}
    r = subprocess.run([sys.executable, os.path.join(root, "bench.py"), "--gpus", "2", "--impl", "reference", "--config", "1",
                        "--steps", "1", "--warmup", "0"], capture_output=True, text=True, env=env, timeout=500)
    assert r.returncode == 0, r.stderr[-2000:]
    lines = [l for l in r.stdout.splitlines() if l.startswith("{")]
    assert len(lines) == 1, r.stdout
    rec = json.loads(lines[0])
    assert rec["impl"] == "reference" and rec["n_gpus"] == 2 and rec["cpu_baseline"]["cores"] >= 1
    if not torch.cuda.is_available() or torch.cuda.device_count() < 2:
        r = subprocess.run([sys.executable, os.path.join(root, "bench.py"), "--gpus", "2", "--steps", "1"], capture_output=True,
                           text=True, env=env, timeout=300)
        assert r.returncode != 0 and "needs 2 CUDA devices" in (r.stderr + r.stdout)
