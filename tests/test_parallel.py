"""Host-side logic of the N > 1 path on CPU: bin sharding and the trigger gather over gloo, world_size 2.
No GPU, no kernels: the per-rank filtering is covered by the GPU parity tests; this covers what is added when
bins are sharded across ranks (paper_2410_16416_b200/parallel.py)."""
import os
import socket

import numpy as np
import pytest

from paper_2410_16416_b200 import parallel as par
from paper_2410_16416_b200 import workloads as wl

TRIGGER_DTYPE = np.dtype([("bin", "<i4"), ("detector", "<i4"), ("template_idx", "<i4"), ("reserved", "<i4"),
                          ("sample", "<i8"), ("snr_re", "<f4"), ("snr_im", "<f4")])


def test_shard_bins_is_a_balanced_partition():
    costs = [5.0, 1.0, 4.0, 4.0, 2.0, 9.0, 1.0]
    for world in (1, 2, 3, 4, 8):
        shards = par.shard_bins(costs, world)
        assert len(shards) == world
        assert sorted(b for s in shards for b in s) == list(range(len(costs)))
        loads = [sum(costs[b] for b in s) for s in shards]
        assert max(loads) <= sum(costs) / world + max(costs)          # LPT bound
    assert par.shard_bins(costs, 2) == par.shard_bins(costs, 2)       # deterministic
    with pytest.raises(ValueError):
        par.shard_bins(costs, 0)


def test_bin_cost_orders_config3_shape_classes():
    w = wl.config3(n_bins=6, n_templates=8, seconds=1, n_detectors=1, n_basis=4)
    w.bins = [w.bins[0], w.bins[3], w.bins[5]]   # one bin of each shape class
    c = [par.bin_cost(b) for b in w.bins]
    assert len({b.template_len for b in w.bins}) == 3
    assert c[0] >= c[1] > c[2] > 0         # 8 s, 4 s, 2 s templates (8 s and 4 s classes differ only in taps)
    b = w.bins[0]
    assert c[0] == sum(s.n_basis * s.rate * (s.n_taps + 2 * b.n_templates) for s in b.slices)


def _fake_triggers(rank, shard, n):
    rng = np.random.Generator(np.random.PCG64(100 + rank))
    t = np.zeros(n, dtype=TRIGGER_DTYPE)
    t["bin"] = rng.integers(0, max(1, len(shard)), n)
    t["detector"] = rng.integers(0, 2, n)
    t["template_idx"] = rng.integers(0, 500, n)
    t["sample"] = rng.integers(0, 1 << 40, n)
    t["snr_re"] = rng.standard_normal(n)
    t["snr_im"] = rng.standard_normal(n)
    return t


def _worker(rank, world, port, shards, counts, out_dir):
    import torch.distributed as dist
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        local = par.to_global_bins(_fake_triggers(rank, shards[rank], counts[rank]), shards[rank])
        got = par.gather_triggers(local)
        np.save(os.path.join(out_dir, f"rank{rank}.npy"), got)
    finally:
        dist.destroy_process_group()


@pytest.mark.parametrize("counts", [(7, 3), (0, 5), (0, 0)])
def test_gather_triggers_gloo_world2(tmp_path, counts):
    import torch.multiprocessing as mp
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    port = s.getsockname()[1]
    s.close()
    costs = [3.0, 1.0, 2.0, 2.0, 1.0]
    shards = par.shard_bins(costs, 2)
    mp.spawn(_worker, args=(2, port, shards, counts, str(tmp_path)), nprocs=2, join=True)
    expect = np.concatenate([par.to_global_bins(_fake_triggers(r, shards[r], counts[r]), shards[r]) for r in range(2)])
    for r in range(2):
        got = np.load(tmp_path / f"rank{r}.npy")
        assert got.dtype == TRIGGER_DTYPE and len(got) == sum(counts)
        assert got.tobytes() == expect.tobytes()
    if sum(counts):
        assert set(expect["bin"][:counts[0]]) <= set(shards[0])       # global bin ids of rank 0's shard
