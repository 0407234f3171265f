"""`-m "not gpu"`: the N > 1 path on CPU -- world_size 2, `gloo`.

Simulations are independent units: the sim axis is sharded over ranks with
`workloads.shard_sims`, every rank runs its shard with the GLOBAL simulation ids as the `sim` field of
the random-number key, and one all-gather of the per-sim scores hands them to the GA's rank.  There is
no GPU here, so the per-rank compute is the CPU oracle (tests may call it); what is under test is the
host logic: the shards partition the batch, explicit sim ids reproduce the same fires as the full
batch, and the gathered score vector is in batch order.
"""
import os
import socket
import sys
from pathlib import Path

import numpy as np
import pytest

ROOT = Path(__file__).resolve().parent.parent


def _free_port() -> int:
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _rank_main(rank: int, world: int, port: int, out_dir: str) -> None:
    sys.path.insert(0, str(ROOT))
    import torch
    import torch.distributed as dist

    from oracle import fire_oracle as orc
    from paper_1701_03549_b200 import workloads as wl

    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    w = wl.load_workload(1)
    ls = w.landscape
    Lo = orc.Landscape(ls["veg"], ls["slope"], ls["aspect"], ls["wind"])
    ref = orc.simulate(Lo, w.ref_beta, w.ref_ignition, w.ref_seed, sim=0)["burned"]
    sl = wl.shard_sims(w.S, rank, world)
    ids = np.arange(w.S, dtype=np.int32)[sl]
    r = orc.simulate_batch(Lo, w.betas, w.ignitions[sl], w.sim_param[sl], w.seeds[sl], sim_index=ids, nthreads=1)
    _, score, _ = orc.fitness(ref, r["burned"], Lo.W, w.metric)
    # equal-size shards are required by all_gather_into_tensor: pad to the largest shard
    per = (w.S + world - 1) // world
    mine = torch.full((per,), float("nan"), dtype=torch.float32)
    mine[: len(score)] = torch.from_numpy(score)
    gathered = torch.empty((world * per,), dtype=torch.float32)
    dist.all_gather_into_tensor(gathered, mine)
    trials = torch.tensor([int(r["trials"].sum())], dtype=torch.int64)
    dist.all_reduce(trials, op=dist.ReduceOp.SUM)
    t = torch.tensor([float(rank + 1)], dtype=torch.float64)           # "max over ranks" timing reduction
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    # ---- the same generation partitioned BY PARAMETER VECTOR: every rank holds only its P / world vectors
    sh = wl.shard_by_param(w, rank, world)
    assert sh.betas.shape[0] == w.P // world and sh.sim_param.max() < sh.betas.shape[0]
    rp = orc.simulate_batch(Lo, sh.betas, sh.ignitions, sh.sim_param, sh.seeds, sim_index=sh.sim_ids, nthreads=1)
    _, score_p, _ = orc.fitness(ref, rp["burned"], Lo.W, w.metric)
    mine_p = torch.full((per,), float("nan"), dtype=torch.float32)
    mine_p[: len(score_p)] = torch.from_numpy(score_p)
    gathered_p = torch.empty((world * per,), dtype=torch.float32)
    dist.all_gather_into_tensor(gathered_p, mine_p)
    if rank == 0:
        shards = [wl.shard_by_param(w, k, world) for k in range(world)]
        vals = [gathered_p[k * per: k * per + len(shards[k].index)].numpy() for k in range(world)]
        np.save(os.path.join(out_dir, "scores_by_param.npy"), wl.merge_param_shards(shards, vals, w.S))
    if rank == 0:
        parts = [gathered[k * per: k * per + (wl.shard_sims(w.S, k, world).stop - wl.shard_sims(w.S, k, world).start)]
                 for k in range(world)]
        np.save(os.path.join(out_dir, "scores.npy"), torch.cat(parts).numpy())
        np.save(os.path.join(out_dir, "trials.npy"), trials.numpy())
        np.save(os.path.join(out_dir, "tmax.npy"), t.numpy())
    dist.barrier()
    dist.destroy_process_group()


@pytest.mark.timeout(300)
def test_two_rank_sharding_reproduces_the_full_batch(orc, tmp_path):
    import torch.multiprocessing as mp
    from paper_1701_03549_b200 import workloads as wl

    world = 2
    mp.spawn(_rank_main, args=(world, _free_port(), str(tmp_path)), nprocs=world, join=True)
    w = wl.load_workload(1)
    ls = w.landscape
    Lo = orc.Landscape(ls["veg"], ls["slope"], ls["aspect"], ls["wind"])
    ref = orc.simulate(Lo, w.ref_beta, w.ref_ignition, w.ref_seed, sim=0)["burned"]
    full = orc.simulate_batch(Lo, w.betas, w.ignitions, w.sim_param, w.seeds)
    _, score, _ = orc.fitness(ref, full["burned"], Lo.W, w.metric)
    got = np.load(tmp_path / "scores.npy")
    assert got.shape == (w.S,)
    assert np.array_equal(got.view(np.uint32), score.view(np.uint32))
    assert int(np.load(tmp_path / "trials.npy")[0]) == int(full["trials"].sum())
    assert float(np.load(tmp_path / "tmax.npy")[0]) == float(world)
    got_p = np.load(tmp_path / "scores_by_param.npy")
    assert np.array_equal(got_p.view(np.uint32), score.view(np.uint32))          # batch order, bit for bit


def test_param_shards_partition_vectors_and_sims():
    from paper_1701_03549_b200 import workloads as wl
    for cfg in (1, 2):
        w = wl.load_workload(cfg)
        for world in (1, 2, 3, 8):
            shards = [wl.shard_by_param(w, r, world) for r in range(world)]
            assert shards[0].p_lo == 0 and shards[-1].p_hi == w.P
            assert all(a.p_hi == b.p_lo for a, b in zip(shards, shards[1:]))
            assert max(s.betas.shape[0] for s in shards) - min(s.betas.shape[0] for s in shards) <= 1
            allidx = np.concatenate([s.index for s in shards])
            assert np.array_equal(np.sort(allidx), np.arange(w.S))
            for s in shards:
                assert np.array_equal(w.betas[s.p_lo + s.sim_param], w.betas[w.sim_param[s.index]])   # same vector, re-based index
                assert np.array_equal(s.sim_ids, s.index.astype(np.int32))
            back = wl.merge_param_shards(shards, [w.seeds[s.index] for s in shards], w.S)
            assert np.array_equal(back, w.seeds)
    # an out-of-range vector index stays invalid on rank 0
    w = wl.load_workload(1)
    w.sim_param = w.sim_param.copy(); w.sim_param[5] = -3; w.sim_param[9] = w.P + 7
    sh0 = wl.shard_by_param(w, 0, 2)
    assert 5 in sh0.index and 9 in sh0.index
    assert (sh0.sim_param[np.isin(sh0.index, [5, 9])] == sh0.betas.shape[0]).all()


def test_shards_are_contiguous_and_cover_the_batch():
    from paper_1701_03549_b200 import workloads as wl
    for S in (1, 7, 64, 2048, 16384):
        for world in (1, 2, 3, 8):
            parts = [wl.shard_sims(S, r, world) for r in range(world)]
            assert parts[0].start == 0 and parts[-1].stop == S
            assert all(a.stop == b.start for a, b in zip(parts, parts[1:]))
            sizes = [p.stop - p.start for p in parts]
            assert max(sizes) - min(sizes) <= 1
