"""World-size-2 CPU test (gloo) of the bench's multi-rank host logic: disjoint history ranges that cover
the job, max-over-ranks timing, and rank-independent results (the oracle stands in for the kernels)."""
import os
import socket
import sys

import numpy as np
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _worker(rank, world, port, n_per_rank, out_dir):
    sys.path.insert(0, ROOT)
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    from oracle import gpet_oracle as O
    from paper_2603_07327_b200 import sharding, workloads as W
    first, n = sharding.history_range(rank, world, n_per_rank)
    r = W.config_runs("C0")[0]
    res = O.simulate(r.geometry, W.tables(), r.source, n, r.seed, first_history=first, want_hash=True)
    t = sharding.max_over_ranks(1.0 + rank)            # the slowest rank defines the job's time
    tot = sharding.sum_over_ranks(float(len(res.hits)))
    np.savez(os.path.join(out_dir, f"rank{rank}.npz"), first=first, n=n, hash=res.outcome_hash, hist=res.hits.history, t=t, tot=tot)
    dist.barrier()
    dist.destroy_process_group()


def test_two_ranks_partition_the_histories(tmp_path):
    world, n_per_rank = 2, 20_000
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0)); port = s.getsockname()[1]
    mp.spawn(_worker, args=(world, port, n_per_rank, str(tmp_path)), nprocs=world, join=True)
    parts = [np.load(tmp_path / f"rank{r}.npz") for r in range(world)]
    assert [int(p["first"]) for p in parts] == [0, n_per_rank] and all(int(p["n"]) == n_per_rank for p in parts)
    assert all(float(p["t"]) == 2.0 for p in parts)                       # max over ranks, same on every rank
    assert all(float(p["tot"]) == sum(len(q["hist"]) for q in parts) for p in parts)
    sys.path.insert(0, ROOT)
    from oracle import gpet_oracle as O
    from paper_2603_07327_b200 import sharding, workloads as W
    r = W.config_runs("C0")[0]
    whole = O.simulate(r.geometry, W.tables(), r.source, sharding.total_pairs(world, n_per_rank), r.seed, want_hash=True)
    assert np.array_equal(np.concatenate([p["hash"] for p in parts]), whole.outcome_hash)
    assert np.array_equal(np.concatenate([p["hist"] for p in parts]), whole.hits.history)


def _worker_coinc(rank, world, port, n_per_rank, out_dir):
    sys.path.insert(0, ROOT)
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    from dataclasses import replace
    from oracle import gpet_oracle as O
    from paper_2603_07327_b200 import sharding, workloads as W
    first, n = sharding.history_range(rank, world, n_per_rank)
    r = W.config_runs("C1", n_per_rank)[0]
    src = replace(r.source, pairs_per_time_slice=n_per_rank)          # as bench.py: one time slice per rank and batch [R16]
    res = O.simulate(r.geometry, W.tables(), src, n, r.seed, first_history=first, threads=2)
    _, co, _ = O.digitize(src, r.seed, sharding.total_pairs(world, n_per_rank), res.hits, r.digitizer)
    n_co = sharding.sum_over_ranks(float(len(co.ids_a)))
    np.savez(os.path.join(out_dir, f"coinc{rank}.npz"), ids_a=co.ids_a, ids_b=co.ids_b, history_a=co.history_a, history_b=co.history_b,
             t_s=co.t_s, dt_ns=co.dt_ns, e_a=co.e_a, e_b=co.e_b, n_co=n_co)
    dist.barrier()
    dist.destroy_process_group()


def test_two_ranks_give_the_single_process_coincidence_list(tmp_path):
    """ADVICE r1 / VERDICT r2: bench.py --gpus N gives every rank its own time slice of one acquisition, so that no
    coincidence window straddles two ranks.  Then the ranks' list-mode outputs, put one after the other, must BE the list
    of the same run digitized in one process (the oracle stands in for the kernels: this is host logic)."""
    world, n_per_rank = 2, 30_000
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0)); port = s.getsockname()[1]
    mp.spawn(_worker_coinc, args=(world, port, n_per_rank, str(tmp_path)), nprocs=world, join=True)
    parts = [np.load(tmp_path / f"coinc{r}.npz") for r in range(world)]
    sys.path.insert(0, ROOT)
    from dataclasses import replace
    from oracle import gpet_oracle as O
    from paper_2603_07327_b200 import sharding, workloads as W
    r = W.config_runs("C1", n_per_rank)[0]
    src = replace(r.source, pairs_per_time_slice=n_per_rank)
    n_total = sharding.total_pairs(world, n_per_rank)
    whole = O.simulate(r.geometry, W.tables(), src, n_total, r.seed, threads=4)
    _, co, _ = O.digitize(src, r.seed, n_total, whole.hits, r.digitizer)
    assert len(co.ids_a) > 2000 and all(len(p["ids_a"]) > 800 for p in parts)
    assert all(float(p["n_co"]) == len(co.ids_a) for p in parts)
    for k in ("ids_a", "ids_b", "history_a", "history_b", "t_s", "dt_ns", "e_a", "e_b"):
        assert np.array_equal(np.concatenate([p[k] for p in parts]), getattr(co, k)), k
    assert parts[0]["t_s"].max() < parts[1]["t_s"].min()                 # rank 1's slice starts after rank 0's ends


def test_history_range_rejects_bad_ranks():
    sys.path.insert(0, ROOT)
    from paper_2603_07327_b200 import sharding
    import pytest
    with pytest.raises(ValueError):
        sharding.history_range(2, 2, 10)
    assert sharding.history_range(3, 8, 1000) == (3000, 1000)
    assert sharding.max_over_ranks(3.5) == 3.5                            # no process group: identity
