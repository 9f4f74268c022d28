"""The N>1 path on CPU: index arithmetic of the energy partition (Fig. 1)
and a world_size-2 gloo run in which every rank forms its share and rank 0 reassembles the whole."""
import os
import socket

import numpy as np
import pytest

from paper_1909_07321_b200 import shard


@pytest.mark.parametrize("world", [1, 2, 3, 4, 8])
@pytest.mark.parametrize("n_E", [0, 1, 7, 8, 9, 256, 1000])
def test_partition_is_a_disjoint_cover(world, n_E):
    for p in range(5):
        parts = [shard.energy_indices(n_E, p, r, world) for r in range(world)]
        allidx = np.concatenate(parts)
        assert np.array_equal(np.sort(allidx), np.arange(n_E))           # every energy exactly once
        for part in parts:
            assert np.all(np.diff(part) > 0)
            # whole kernel energy blocks only (the last block of the mesh may be short)
            blocks = np.unique(part // shard.ENERGY_BLOCK)
            assert part.size == sum(min(shard.ENERGY_BLOCK, n_E - b * shard.ENERGY_BLOCK) for b in blocks)


def test_rotation_over_waves():
    world, n_E = 4, 256
    for r in range(world):
        sets = [shard.energy_set_of_rank(p, r, world) for p in range(world)]
        assert sorted(sets) == list(range(world))           # over `world` waves a rank meets every energy set once
        first = [int(shard.energy_indices(n_E, p, r, world)[0]) for p in range(world)]
        assert len(set(first)) == world
    # "never consecutive energies for the same partial wave" beyond one kernel block (world > 1)
    idx = shard.energy_indices(n_E, 0, 1, world)
    gaps = np.diff(idx)
    assert set(gaps.tolist()) == {1, (world - 1) * shard.ENERGY_BLOCK + 1}


def test_balance_and_wave_order():
    n_E = [512] * 32
    c = shard.counts(n_E, 8)
    assert c.sum() == 512 * 32 and c.min() == c.max() == 64
    c = shard.counts([1000, 37, 8, 0], 3)
    assert np.array_equal(c.sum(axis=0), [1000, 37, 8, 0])
    assert c[:, 0].max() - c[:, 0].min() <= shard.ENERGY_BLOCK
    assert shard.wave_order(5, 2, 4) == [2, 3, 4, 0, 1]
    assert shard.wave_order(0, 0, 2) == []
    starts = {shard.wave_order(8, r, 8)[0] for r in range(8)}
    assert len(starts) == 8                                   # every rank starts on a different wave
    pl = shard.plan([16, 24], 1, 2)
    assert [p for p, _ in pl] == [1, 0]
    assert np.array_equal(pl[0][1], np.r_[0:8, 16:24])         # wave 1 (24 energies), rank 1 -> set 0: blocks 0 and 2
    assert np.array_equal(pl[1][1], np.arange(8, 16))          # wave 0, rank 1 -> set 1


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, ret):
    import torch
    import torch.distributed as dist
    from oracle import rmat_oracle
    from paper_1909_07321_b200 import inputs
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        waves = [inputs.make_wave(31, 12, 40, 37), inputs.make_wave(32, 5, 9, 16), inputs.make_wave(33, 9, 18, 3)]
        mine = {}
        for p, idx in shard.plan([w.n_E for w in waves], rank, world):
            w = waves[p]
            mine[p] = (idx, rmat_oracle.rmat_form(w.W, w.E_k, w.energies[idx], w.a))
        gathered = [None] * world
        dist.all_gather_object(gathered, mine)                # the optional gather; no collective on the data path
        slow = shard.max_over_ranks(10.0 + rank)
        if rank == 0:
            ok = slow == 10.0 + world - 1
            for p, w in enumerate(waves):
                full = np.full((w.n_E, w.n_chan, w.n_chan), np.nan)
                for g in gathered:
                    shard.scatter_into(full, *g[p])
                ok = ok and np.array_equal(full, rmat_oracle.rmat_form(w.W, w.E_k, w.energies, w.a))
            ret.put(bool(ok))
    finally:
        dist.destroy_process_group()


def test_two_ranks_gloo_reassemble_the_whole_mesh():
    torch = pytest.importorskip("torch")
    import torch.multiprocessing as mp
    from oracle import rmat_oracle
    rmat_oracle.build()
    ctx = mp.get_context("spawn")
    ret = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, ret)) for r in range(2)]
    for pr in procs:
        pr.start()
    for pr in procs:
        pr.join(120)
        assert pr.exitcode == 0
    assert ret.get(timeout=10) is True


@pytest.mark.parametrize("scaling,world", [("weak", 2), ("weak", 4), ("strong", 2), ("strong", 8)])
def test_bench_job_is_partitioned_exactly(scaling, world):
    """bench.py --gpus N: the ranks' shares (shard.plan over the job's meshes) are a disjoint cover of the job --
    weak scaling multiplies the mesh by N, strong scaling keeps the configuration's own mesh -- so that
    value = job energies / max-over-ranks time counts every energy once."""
    import argparse
    import bench
    args = argparse.Namespace(config=1, n_E=0, scaling=scaling)
    job = bench.job_workload(args, world)
    base = bench.job_workload(args, 1)
    assert job.n_energies() == (world if scaling == "weak" else 1) * base.n_energies()
    for p, w in enumerate(job.waves):
        seen = np.zeros(w.n_E, dtype=int)
        for r in range(world):
            for q, idx in shard.plan([x.n_E for x in job.waves], r, world):
                if q == p:
                    seen[idx] += 1
        assert np.all(seen == 1)
    assert bench.workload_description(1, job) == bench.workload_description(1, bench.job_workload(args, world))
