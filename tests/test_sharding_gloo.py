"""Host-side logic of the N>1 path (bench.py --gpus N): the linear triplet index is cut into N contiguous
ranges (tc_triplet_partition), every rank reduces its own range and the only exchange is one all-reduce of the FP64 partial
energy (paper: independent tile batches per GPU, partial energies summed).
Run on CPU with the gloo backend, world_size 2 and 3; the per-range partial energies come from the CPU oracle
(the per-range CUDA call is covered by test_gpu_parity.py::test_cfg0_full)."""
import os
import sys

import numpy as np
import pytest

torch = pytest.importorskip("torch")
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _worker(rank, world, port, q):
    sys.path.insert(0, ROOT)
    sys.path.insert(0, os.path.join(ROOT, "tests"))
    import harness
    import oracle
    from paper_2512_01055_b200 import binding
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    p = harness.make_problem(5, 6, 7, seed=3, sigma_B=0.3, blocks=True)
    n = oracle.triplet_count(p.o)
    first, count = binding.triplet_partition(p.o, world, rank)     # the library's own partition (C-ABI, host only)
    E_part, _ = oracle.triples_energy(p, first, count) if count else (0.0, None)
    t = torch.tensor([E_part, float(count)], dtype=torch.float64)
    dist.all_reduce(t, op=dist.ReduceOp.SUM)
    tmax = torch.tensor([float(rank + 1)], dtype=torch.float64)   # stands for the per-rank device time
    dist.all_reduce(tmax, op=dist.ReduceOp.MAX)
    if rank == 0:
        E_full, _ = oracle.triples_energy(p)
        q.put((float(t[0]), float(t[1]), E_full, n, float(tmax[0])))
    dist.barrier()
    dist.destroy_process_group()


@pytest.mark.parametrize("world", [2, 3])
def test_partition_and_allreduce(world):
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = 29500 + (os.getpid() % 2000) + world
    procs = [ctx.Process(target=_worker, args=(r, world, port, q)) for r in range(world)]
    for pr in procs:
        pr.start()
    E_sum, n_sum, E_full, n, tmax = q.get(timeout=120)
    for pr in procs:
        pr.join(timeout=60)
        assert pr.exitcode == 0
    assert n_sum == n                       # the ranges tile [0, N_trip)
    assert abs(E_sum - E_full) <= 1e-12 * abs(E_full)
    assert tmax == world                    # max over ranks
