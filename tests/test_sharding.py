"""The N > 1 path of bench.py under gloo, world_size 2 (CPU): samples are independent
(PAPER.md:337), so the batch is sharded over ranks with replicated parameters and Hamiltonian and
NO data-path collective; the only communication is the barrier and the max-over-ranks of the
timing.  This test runs the shard plan and that reduction in two real processes."""
import os
import socket
import sys

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, out_dir):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    sys.path.insert(0, ROOT)
    import torch
    import torch.distributed as dist

    import bench

    dist.init_process_group("gloo", rank=rank, world_size=world)
    plan = bench.shard_plan(world, rank, 2)
    w = bench.make_rank_workload(plan)
    # what every rank must agree on (replicated) and what must differ (its own samples)
    par = np.concatenate([w.a.view(np.float32), w.b.view(np.float32), w.W.view(np.float32).ravel()])
    digest = torch.tensor([float(np.float64(par).sum()), float(w.ham.coeffs.real.sum()), float(w.ham.T)],
                          dtype=torch.float64)
    gathered = [torch.zeros_like(digest) for _ in range(world)]
    dist.all_gather(gathered, digest)
    spin_digest = torch.tensor([float(w.spins[:64].astype(np.int64).sum()), float(w.spins.shape[0])],
                               dtype=torch.float64)
    sg = [torch.zeros_like(spin_digest) for _ in range(world)]
    dist.all_gather(sg, spin_digest)
    # the timing reduction bench.py uses: MAX over ranks
    t = torch.tensor([10.0 + rank], dtype=torch.float64)
    dist.barrier()
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    np.save(os.path.join(out_dir, f"r{rank}.npy"),
            np.array([plan["global_batch"], plan["B"], t.item(), plan["spin_seed"][-1],
                      float(all(torch.equal(g, gathered[0]) for g in gathered)),
                      float(not torch.equal(sg[0], sg[1])), sg[rank][1].item()]))
    np.save(os.path.join(out_dir, f"spins{rank}.npy"), w.spins[:16])
    dist.barrier()
    dist.destroy_process_group()


@pytest.mark.timeout(300)
def test_shard_plan_two_ranks_gloo(tmp_path):
    import torch.multiprocessing as mp

    world, port = 2, _free_port()
    mp.spawn(_worker, args=(world, port, str(tmp_path)), nprocs=world, join=True)
    r = [np.load(tmp_path / f"r{k}.npy") for k in range(world)]
    import workloads as wl

    B = wl.config_spec(2)["B"]
    for k in range(world):
        assert r[k][0] == world * B and r[k][1] == B      # weak scaling: per-rank work fixed
        assert r[k][2] == 10.0 + (world - 1)              # max over ranks reached everyone
        assert r[k][3] == k                               # rank-specific spin stream
        assert r[k][4] == 1.0                             # parameters + Hamiltonian replicated
        assert r[k][5] == 1.0                             # spins differ between ranks
        assert r[k][6] == B
    s0, s1 = np.load(tmp_path / "spins0.npy"), np.load(tmp_path / "spins1.npy")
    assert not np.array_equal(s0, s1)
    # rank 0 of a multi-rank run sees exactly the single-GPU workload
    assert np.array_equal(s0, wl.make_config(2).spins[:16])


def test_shard_plan_is_pure():
    import bench

    p0, p1 = bench.shard_plan(4, 0, 5), bench.shard_plan(4, 3, 5)
    assert p0["global_batch"] == p1["global_batch"] == 4 * 65536
    assert p0["spin_seed"] == [5, 1, 0] and p1["spin_seed"] == [5, 1, 3]
