"""Multi-GPU host logic on CPU: world_size-2 gloo.  The path shards by independent units (frames /
GoPs) with no data-path collective; what crosses ranks is the timing reduction
bench.py does (max over ranks) and a gather of per-unit results.  Each rank stands in for its
GPU work with the float64 oracle on a tiny frame, so that the gathered results can be checked
against a single-process run."""
import os
import socket

import numpy as np
import pytest

torch = pytest.importorskip("torch")
import torch.distributed as dist  # noqa: E402
import torch.multiprocessing as mp  # noqa: E402


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _unit_psnr(unit):
    import oracle
    import workloads as wl
    frame, _ = wl.talking_head_frame(wl.SPEC_TINY, unit)
    g = wl.tiny_gaussians(64)
    p = oracle.Params.from_f32(g)
    return oracle.fit(64, 64, p, frame, 3, lr=1e-2).psnr


def _worker(rank, world, port, n_units, out_dir):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    import paper_2505_09324_b200 as gs
    mine = gs.shard_units(n_units, rank, world)
    res = torch.full((n_units,), -1.0, dtype=torch.float64)
    for u in mine:
        res[u] = _unit_psnr(u)
    # the reductions bench.py performs: max of the per-rank times, sum of the units processed
    t = torch.tensor([10.0 + rank], dtype=torch.float64)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    cnt = torch.tensor([len(mine)], dtype=torch.int64)
    dist.all_reduce(cnt, op=dist.ReduceOp.SUM)
    dist.all_reduce(res, op=dist.ReduceOp.MAX)      # gather: every unit was written by exactly one rank
    dist.barrier()
    if rank == 0:
        np.save(os.path.join(out_dir, "res.npy"), np.concatenate([res.numpy(), t.numpy(), cnt.numpy().astype(np.float64)]))
    dist.destroy_process_group()


def test_shard_units_partition():
    import paper_2505_09324_b200 as gs
    for n in (0, 1, 5, 8, 30, 31):
        for w in (1, 2, 3, 8):
            parts = [gs.shard_units(n, r, w) for r in range(w)]
            assert sorted(u for p in parts for u in p) == list(range(n))
            assert max(len(p) for p in parts) - min(len(p) for p in parts) <= 1
    with pytest.raises(ValueError):
        gs.shard_units(4, 2, 2)


def test_two_ranks_gloo_shard_and_gather(tmp_path):
    n_units, world = 5, 2
    port = _free_port()
    mp.spawn(_worker, args=(world, port, n_units, str(tmp_path)), nprocs=world, join=True)
    out = np.load(tmp_path / "res.npy")
    res, tmax, cnt = out[:n_units], out[n_units], out[n_units + 1]
    assert tmax == 11.0 and cnt == n_units
    ref = np.array([_unit_psnr(u) for u in range(n_units)])
    assert np.allclose(res, ref, rtol=0, atol=1e-9)
