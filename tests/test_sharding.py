"""Multi-GPU path: sharding by disorder sample.  CPU part: world_size-2 gloo processes, each
running ITS shard (here through the oracle, which takes the same sample_offset as the C ABI), gather their
per-sample observables and must reproduce the single-process run bit for bit.  GPU part (-m gpu): two hsg
contexts with sample offsets reproduce one context holding all samples."""
import os
import socket

import numpy as np
import pytest

import hsg_inputs
from paper_1204_6192_b200 import sharding

L, D_ALL, O, T, SEED = 4, 3, 2, 3, 17


def test_shard_bounds_cover_every_sample_once():
    for n in (0, 1, 3, 8, 64, 65):
        for w in (1, 2, 3, 8):
            b = sharding.shard_bounds(n, w)
            assert len(b) == w and sum(c for _, c in b) == n
            assert all(b[i][0] + b[i][1] == b[i + 1][0] for i in range(w - 1)) and b[0][0] == 0
            assert max(c for _, c in b) - min(c for _, c in b) <= 1
            for d in range(n):
                r, loc = sharding.owner_of_sample(n, w, d)
                assert b[r][0] + loc == d and loc < b[r][1]
    assert sharding.shard_of_rank(64, 8, 3) == (24, 8)
    with pytest.raises(ValueError):
        sharding.shard_of_rank(4, 2, 2)


def _run_shard(off, cnt):
    import oracle
    temps = hsg_inputs.geometric_ladder(0.1, 0.3, T)
    sim = oracle.Oracle(L, cnt, O, temps, SEED, precision=32, sample_offset=off)
    sim.set_disorder(hsg_inputs.couplings(L, cnt, SEED, off), hsg_inputs.gaussian_field(L, cnt, 0.1, SEED, off))
    sim.init_spins()
    accs = []
    for _ in range(3):
        sim.sweep(2, 1)
        accs.append(sim.pt_swap())
    E, M, q0, qk = sim.measure()
    return E, q0, np.stack(accs, axis=1)


def _worker(rank, world, port, q):
    import torch
    import torch.distributed as dist
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        off, cnt = sharding.shard_of_rank(D_ALL, world, rank)
        E, q0, acc = _run_shard(off, cnt)
        E_all = sharding.gather_by_sample(torch.from_numpy(E), D_ALL)
        q_all = sharding.gather_by_sample(torch.from_numpy(q0), D_ALL)
        a_all = sharding.gather_by_sample(torch.from_numpy(acc), D_ALL)
        tmax = sharding.max_over_ranks([float(rank), 1.0])
        if rank == 0:
            q.put((E_all.numpy(), q_all.numpy(), a_all.numpy(), tmax))
        dist.barrier()
    finally:
        dist.destroy_process_group()


def test_two_gloo_ranks_reproduce_the_single_process_run():
    import torch.multiprocessing as mp
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        port = s.getsockname()[1]
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    E_all, q_all, a_all, tmax = q.get(timeout=180)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    E1, q1, a1 = _run_shard(0, D_ALL)
    assert E_all.shape == (D_ALL, O, T)
    assert np.array_equal(E_all, E1) and np.array_equal(q_all, q1) and np.array_equal(a_all, a1)
    assert tmax == [1.0, 1.0]


def test_gather_without_process_group_is_the_identity():
    import torch
    x = torch.arange(6.0).reshape(3, 2)
    assert sharding.gather_by_sample(x, 3) is x
    with pytest.raises(ValueError):
        sharding.gather_by_sample(x, 4)
    assert sharding.max_over_ranks([1.5, 2.0]) == [1.5, 2.0]


@pytest.mark.gpu
@pytest.mark.parametrize("kernel", ["generic", "zmarch"])
def test_two_contexts_with_sample_offsets_reproduce_one_context(kernel):
    import paper_1204_6192_b200 as hsg
    Lg, D, Tg = 8, 3, 4
    temps = hsg_inputs.geometric_ladder(0.08, 0.3, Tg)

    def run(off, cnt):
        eng = hsg.hsg_create(Lg, cnt, O, temps, SEED, sample_offset=off, kernel=kernel)
        eng.set_disorder(hsg_inputs.couplings(Lg, cnt, SEED, off), hsg_inputs.gaussian_field(Lg, cnt, 0.1, SEED, off))
        eng.init_spins()
        for _ in range(3):
            eng.sweep(2, 1)
            eng.pt_swap()
        E, M, q0, qk = (x.cpu().numpy() for x in eng.measure())
        return E, q0, eng.get_spins().cpu().numpy()

    full = run(0, D)
    parts = [run(off, cnt) for off, cnt in sharding.shard_bounds(D, 2)]
    for k in range(3):
        assert np.array_equal(np.concatenate([p[k] for p in parts], axis=0), full[k])


def _run_gpu_shard(off, cnt, Lg=8, Tg=4):
    """One rank's work on the GPU through the C ABI: its shard of samples, three steps, observables + spins (CPU tensors)."""
    import paper_1204_6192_b200 as hsg
    temps = hsg_inputs.geometric_ladder(0.08, 0.3, Tg)
    eng = hsg.hsg_create(Lg, cnt, O, temps, SEED, sample_offset=off)
    eng.set_disorder(hsg_inputs.couplings(Lg, cnt, SEED, off), hsg_inputs.gaussian_field(Lg, cnt, 0.1, SEED, off))
    eng.init_spins()
    accs = []
    for _ in range(3):
        eng.sweep(2, 1)
        accs.append(eng.pt_swap().cpu())
    E, M, q0, qk = (x.cpu() for x in eng.measure())
    import torch
    return E, q0, torch.stack(accs, dim=1), eng.get_spins().cpu()


def _gpu_worker(rank, world, port, q, n_all):
    import torch
    import torch.distributed as dist
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    torch.cuda.set_device(rank % torch.cuda.device_count())     # two ranks may share one device (the driver's box has one)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        off, cnt = sharding.shard_of_rank(n_all, world, rank)
        parts = _run_gpu_shard(off, cnt)
        gathered = [sharding.gather_by_sample(x, n_all) for x in parts]
        if rank == 0:
            q.put([g.numpy() for g in gathered])
        dist.barrier()
    finally:
        dist.destroy_process_group()


@pytest.mark.gpu
def test_two_gpu_processes_gathered_over_gloo_reproduce_one_context():
    """The multi-GPU path as bench.py --gpus N runs it, with the real engine: two PROCESSES (one hsg context each, their own
    shard of the disorder samples via sample_offset), per-sample observables and spins gathered with
    sharding.gather_by_sample over gloo, must equal the single-context run of all samples bit for bit."""
    import torch.multiprocessing as mp
    n_all = 3
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        port = s.getsockname()[1]
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    procs = [ctx.Process(target=_gpu_worker, args=(r, 2, port, q, n_all)) for r in range(2)]
    for p in procs:
        p.start()
    got, waited = None, 0
    while got is None:                       # fail at once if a rank dies, not after the queue's time-out
        try:
            got = q.get(timeout=5)
        except Exception:
            waited += 5
            assert all(p.exitcode in (None, 0) for p in procs), [p.exitcode for p in procs]
            assert waited < 600, "ranks still running after 600 s"
    for p in procs:
        p.join(timeout=120)
        assert p.exitcode == 0
    full = [x.numpy() for x in _run_gpu_shard(0, n_all)]
    assert got[0].shape == (n_all, O, 4)
    for a, b in zip(got, full):
        assert np.array_equal(a, b)
