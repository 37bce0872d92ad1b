"""The N > 1 path on CPU: two processes, gloo backend (realizations sharded over ranks, no
data-path collective).  Each rank advances ITS shard with the oracle standing in for the device path; the
checks are about the host logic of paper_2501_06377_b200/ensemble.py:

  * the shards partition the weak-scaled ensemble (rank 0 owns exactly the 1-GPU workload),
  * every rank ends up with the same dt and STS stage count (all_reduce MIN of the limits),
  * the gathered diagnostics are in global realization order and equal a single-process run of the whole
    ensemble (realizations are independent, so this is exact),
  * the bench timing reduction is the max over ranks.
"""
import os
import socket

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from oracle import sft_oracle as orc
from paper_2501_06377_b200 import ensemble as ens
from paper_2501_06377_b200 import workloads as wl

NT, NP, NR = 24, 48, 3          # per-rank shard of the scaled-down configuration 3


def small_shard(rank, world):
    w = ens.shard(3, "f64", rank, world)
    g0 = int(w.extra.get("first_global_realization", 0))
    # scale the grid down, keep realizations [g0, g0 + NR) of the 64 this rank owns
    q = wl.scaled(w, NT, NP, n_real=NR, t_end_hours=6.0)
    q.extra["first_global_realization"] = g0
    return q


def run_shard(w, dt=None, n=None):
    o = orc.Oracle(w.n_theta, w.n_phi, w.params)
    maps = ens.shard_maps(w)
    for r in range(w.n_real):
        o.set_map(r, maps[r].numpy())
    lim = o.stable_dt()
    return o, lim


def free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def worker(rank, world, port, out_dir):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        w = small_shard(rank, world)
        o, lim = run_shard(w)
        glim = ens.global_limits(*lim)
        dt, n, _ = wl.plan(w, *glim)
        # one stage count for the whole ensemble: from the ensemble-wide Euler limit (reading U9)
        s_local = o.sts_stage_count(dt)
        s = int(ens.max_over_ranks(float(s_local)))
        o.step(n, dt, sts_stages=s)
        diag = ens.gather_diagnostics(o.diagnostics())
        tmax = ens.max_over_ranks(10.0 + rank)
        np.savez(os.path.join(out_dir, f"rank{rank}.npz"), lim=np.array(lim), glim=np.array(glim), dt=dt, n=n, s=s,
                 diag=diag, tmax=tmax, params=w.params, maps=np.stack([o.get_full(r) for r in range(w.n_real)]))
    finally:
        dist.destroy_process_group()


@pytest.mark.timeout(600)
def test_two_ranks_gloo(tmp_path):
    world = 2
    mp.spawn(worker, args=(world, free_port(), str(tmp_path)), nprocs=world, join=True)
    res = [np.load(tmp_path / f"rank{r}.npz") for r in range(world)]
    # same clock on every rank, and it is the minimum of the local limits
    assert res[0]["dt"] == res[1]["dt"] and res[0]["n"] == res[1]["n"] and res[0]["s"] == res[1]["s"]
    assert np.array_equal(res[0]["glim"], np.minimum(res[0]["lim"], res[1]["lim"]))
    assert np.array_equal(res[0]["glim"], res[1]["glim"])
    assert res[0]["tmax"] == 11.0 and res[1]["tmax"] == 11.0
    assert np.array_equal(res[0]["diag"], res[1]["diag"]) and res[0]["diag"].shape == (world * NR, 4)
    # single-process run of the whole (scaled) ensemble with the same clock
    params = np.concatenate([res[r]["params"] for r in range(world)])
    o = orc.Oracle(NT, NP, params)
    k = 0
    for r in range(world):
        w = small_shard(r, world)
        maps = ens.shard_maps(w)
        for i in range(NR):
            o.set_map(k, maps[i].numpy())
            k += 1
    assert np.array_equal(np.array(o.stable_dt()), res[0]["glim"])
    o.step(int(res[0]["n"]), float(res[0]["dt"]), sts_stages=int(res[0]["s"]))
    full = np.stack([o.get_full(r) for r in range(world * NR)])
    assert np.array_equal(full, np.concatenate([res[r]["maps"] for r in range(world)]))
    assert np.array_equal(o.diagnostics(), res[0]["diag"])


def test_shards_partition_the_ensemble():
    base = wl.config(3)
    one = ens.shard(3, "f64", 0, 1)
    assert np.array_equal(one.params, base.params)
    for world in (2, 4, 8):
        shards = [ens.shard(3, "f64", r, world) for r in range(world)]
        allp = np.concatenate([s.params for s in shards])
        assert allp.shape == (64 * world, 7)
        assert np.array_equal(shards[0].params, base.params)                  # rank 0 = the 1-GPU workload
        assert np.array_equal(allp, wl.ensemble_params(3, 64 * world))
        assert len({tuple(row) for row in allp}) == 64 * world                 # all realizations distinct
        assert [s.extra["first_global_realization"] for s in shards] == [64 * r for r in range(world)]
    # per-realization maps follow the global index: realization 1 of rank 1 is global realization 65
    a = small_shard(1, 2)
    m = ens.shard_maps(a)
    ref = wl.bipolar_map(NT, NP, a.n_pairs, a.map_seed + 1000 * (64 + 1 + 1))
    assert torch.equal(m[1], ref)
    # without a process group the reductions are identities
    assert ens.global_limits(1.5, 2.5) == (1.5, 2.5) and ens.max_over_ranks(3.0) == 3.0
