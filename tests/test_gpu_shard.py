"""The N > 1 path on the GPU, world_size 2: every rank builds a Bank over its own shard of the bins
(parallel.shard_bins), filters the same strain through lloid_filter, rewrites its local bin indices
(parallel.to_global_bins) and gathers the triggers (parallel.gather_triggers).  The union must be, record for record,
what one rank computes for the whole bank.  No rank's kernel waits on another rank (the data path has no
collective: SURVEY.md §8(e)), so the two ranks may share one GPU: with two or more GPUs visible each rank takes its
own and the gather runs over nccl, with one GPU both use cuda:0 and the gather runs over gloo."""
import os
import socket

import numpy as np
import pytest

pytestmark = pytest.mark.gpu

from paper_2410_16416_b200 import binding as lb          # noqa: E402
from paper_2410_16416_b200 import parallel as par        # noqa: E402
from paper_2410_16416_b200 import workloads as wl        # noqa: E402


def _workload():
    # three shape classes (8 s / 4 s / 2 s templates), two bins each with its own content
    return wl.config3(n_bins=6, n_templates=96, seconds=24, n_detectors=2, n_basis=32, distinct_per_class=2)


def _filter(w, precision, device, bins=None):
    import torch
    torch.cuda.set_device(device)
    bank = lb.Bank(w, precision, device=device, bins=bins)
    try:
        ids = bank.bin_ids
        cap = sum(w.bins[b].n_templates for b in ids) * w.n_detectors * (w.n_samples // w.peak_window + 1)
        strain = torch.from_numpy(w.strain).cuda()
        trig = torch.zeros(cap * 32, dtype=torch.uint8, device="cuda")
        cnt = torch.zeros(1, dtype=torch.int64, device="cuda")
        bank.filter(strain, trig, cnt)
        torch.cuda.synchronize()
        n = int(cnt.item())
        assert n <= cap
        assert lb.lloid_last_launch_count(bank.handle) > 0
        return trig.cpu().numpy().view(lb.TRIGGER_DTYPE)[:n].copy()
    finally:
        bank.close()


def _canon(t):
    order = np.lexsort((t["sample"], t["template_idx"], t["detector"], t["bin"]))
    return t[order]


def _worker(rank, world, port, precision, out_dir):
    import torch
    import torch.distributed as dist
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    own_gpu = torch.cuda.device_count() >= world
    device = rank if own_gpu else 0
    torch.cuda.set_device(device)
    dist.init_process_group("nccl" if own_gpu else "gloo", rank=rank, world_size=world)
    try:
        w = _workload()
        shards = par.shard_bins([par.bin_cost(b) for b in w.bins], world)
        local = _filter(w, precision, device, bins=shards[rank])
        assert len(local) and local["bin"].max() < len(shards[rank])
        got = par.gather_triggers(par.to_global_bins(local, shards[rank]), device="cuda" if own_gpu else None)
        np.save(os.path.join(out_dir, f"rank{rank}.npy"), got)
        np.save(os.path.join(out_dir, f"shard{rank}.npy"), np.asarray(shards[rank]))
    finally:
        dist.destroy_process_group()


@pytest.mark.parametrize("precision", [pytest.param(lb.LLOID_F32, id="fp32"), pytest.param(lb.LLOID_F16, id="fp16")])
def test_two_ranks_sharded_bins_equal_one_rank(tmp_path, precision):
    import torch.multiprocessing as mp
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    port = s.getsockname()[1]
    s.close()
    mp.spawn(_worker, args=(2, port, precision, str(tmp_path)), nprocs=2, join=True)
    w = _workload()
    whole = _canon(_filter(w, precision, 0))
    got = [np.load(tmp_path / f"rank{r}.npy") for r in range(2)]
    assert got[0].tobytes() == got[1].tobytes()               # every rank holds the same gathered list
    shards = [set(np.load(tmp_path / f"shard{r}.npy").tolist()) for r in range(2)]
    assert shards[0] and shards[1] and not (shards[0] & shards[1]) and shards[0] | shards[1] == set(range(6))
    merged = _canon(got[0])
    assert len(merged) == len(whole)
    # the same bin gives bit-identical triggers whether it is filtered alone, in a shard or in the whole bank
    assert merged.tobytes() == whole.tobytes()
