"""CPU-only: the workload generator is seeded and well-formed; the lambda sharding of the multi-GPU path
partitions exactly and gathers in order (world_size-2 gloo run on CPU)."""
import os
import socket
import sys

import numpy as np
import pytest

from workloads import CONFIGS, make_workload

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_generator_is_seeded_and_well_formed():
    a, b = make_workload("tiny"), make_workload("tiny")
    for k in ("dL", "m1d", "m2d", "ln_prior", "z_grid", "p_gal", "lam", "inj_dL", "inj_ln_pdraw"):
        assert np.array_equal(getattr(a, k), getattr(b, k)), k
    assert a.seed == 20250402 and make_workload("o5_spec", catalog=2, n_events=2, n_samples=10, n_lambda=2, n_det=50).seed == 20250402 + 1002
    assert np.all(a.m1d >= a.m2d) and np.all(a.dL > 0) and np.all(a.p_gal >= 0)
    z = a.z_grid.reshape(a.n_events, -1)
    assert np.all(np.diff(z, axis=1) > 0)
    assert a.n_det <= a.n_inj_total == 10_000
    assert np.allclose(a.ln_prior, 2 * np.log(a.dL))
    assert set(CONFIGS) == {"tiny", "o5_spec", "o5_photo", "full_pop", "sel_heavy"}


def test_lambda_batch_box():
    w = make_workload("o5_spec", n_events=2, n_samples=10, n_lambda=500, n_det=50)
    lam = w.lam
    assert np.array_equal(lam[0], w.fiducial)
    for c, (lo, hi) in {0: (60, 80), 1: (0.2, 0.4), 2: (0.5, 2.0), 3: (0.5, 3.0)}.items():
        assert lam[1:, c].min() >= lo and lam[1:, c].max() <= hi
    r = lam[1:, 4:] / w.fiducial[4:]
    assert r.min() >= 0.9 and r.max() <= 1.1


def test_shard_lambda_partitions_exactly():
    from paper_2504_02034_b200.sharding import shard_lambda
    for n in (0, 1, 7, 1024, 4097):
        for world in (1, 2, 3, 8):
            spans = [shard_lambda(n, r, world) for r in range(world)]
            assert spans[0][0] == 0 and spans[-1][1] == n
            assert all(a[1] == b[0] for a, b in zip(spans[:-1], spans[1:]))
            sizes = [hi - lo for lo, hi in spans]
            assert max(sizes) - min(sizes) <= 1
    with pytest.raises(ValueError):
        shard_lambda(10, 2, 2)


def _worker(rank, world, port, n_lambda, q):
    import torch
    import torch.distributed as dist
    sys.path.insert(0, ROOT)
    from paper_2504_02034_b200.sharding import gather_lambda_results, shard_lambda
    os.environ["MASTER_ADDR"], os.environ["MASTER_PORT"] = "127.0.0.1", str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    lo, hi = shard_lambda(n_lambda, rank, world)
    # stand-in for the per-rank GPU result: a deterministic function of the global lambda index
    local = torch.arange(lo, hi, dtype=torch.float64) ** 2 - 3.0
    full = gather_lambda_results(local, n_lambda)
    if rank == 0:
        q.put(full.numpy())
    dist.barrier()
    dist.destroy_process_group()


@pytest.mark.parametrize("n_lambda", [7, 1024])
def test_two_rank_gloo_gather(n_lambda):
    import torch.multiprocessing as mp
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    port = s.getsockname()[1]
    s.close()
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    ps = [ctx.Process(target=_worker, args=(r, 2, port, n_lambda, q)) for r in range(2)]
    [p.start() for p in ps]
    full = q.get(timeout=120)
    [p.join(60) for p in ps]
    assert all(p.exitcode == 0 for p in ps)
    assert np.array_equal(full, np.arange(n_lambda, dtype=np.float64) ** 2 - 3.0)
