"""Multi-GPU plumbing: realizations sharded over ranks, one process per GPU.

The paper distributes REALIZATIONS over MPI ranks and never splits the grid, so the time
step has no data-path collective.  What ranks do exchange, outside the timed path and in O(1) or O(R) doubles:

  * the two step-size limits (the run has one clock: dt and the STS stage count s are shared by all
    realizations of the ensemble) -> all_reduce(MIN) of 2 doubles at plan time;
  * the R x 4 flux diagnostics -> all_gather of each rank's block;
  * the timing of a bench run -> all_reduce(MAX) of one double.

Works with any torch.distributed backend (nccl on the GPUs, gloo in the CPU tests).  Holds none of the method's
arithmetic.
"""
import copy

import numpy as np
import torch

from . import workloads as wl


def shard(idx: int, dtype: str, rank: int, world: int) -> wl.Workload:
    """Rank `rank`'s shard of the weak-scaled ensemble of configuration idx: the global ensemble has
    world x n_real realizations, global index g = rank * n_real + r; realization g has the same parameters
    and the same initial map whatever the world size (so rank 0 of any run owns exactly the 1-GPU workload)."""
    base = wl.config(idx, dtype)
    if world == 1:
        return base
    assert 0 <= rank < world
    w = copy.deepcopy(base)
    w.params = wl.ensemble_params(idx, base.n_real * world)[rank * base.n_real:(rank + 1) * base.n_real].copy()
    w.extra["first_global_realization"] = rank * base.n_real
    w.name = f"{base.name}_rank{rank}of{world}"
    return w


def shard_maps(w: wl.Workload, device="cpu"):
    """Initial maps of a shard: per-realization maps are seeded by the GLOBAL realization index."""
    g0 = int(w.extra.get("first_global_realization", 0))
    if not w.per_real_maps:
        return wl.initial_maps(w, device=device)
    return torch.stack([wl.bipolar_map(w.n_theta, w.n_phi, w.n_pairs, w.map_seed + 1000 * (g0 + r + 1),
                                       background_g=w.background_g, device=device) for r in range(w.n_real)])


def _dist():
    import torch.distributed as dist
    return dist if (dist.is_available() and dist.is_initialized()) else None


def _dev():
    dist = _dist()
    return torch.device("cuda", torch.cuda.current_device()) if (dist and dist.get_backend() == "nccl") else torch.device("cpu")


def global_limits(dt_adv_limit: float, dt_diff_expl: float):
    """Ensemble-wide step-size limits: the minimum over ranks of each rank's limits (inf stays inf)."""
    dist = _dist()
    if dist is None:
        return dt_adv_limit, dt_diff_expl
    t = torch.tensor([dt_adv_limit, dt_diff_expl], dtype=torch.float64, device=_dev())
    dist.all_reduce(t, op=dist.ReduceOp.MIN)
    return float(t[0]), float(t[1])


def max_over_ranks(x: float) -> float:
    dist = _dist()
    if dist is None:
        return x
    t = torch.tensor([x], dtype=torch.float64, device=_dev())
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t[0])


def gather_diagnostics(diag: np.ndarray) -> np.ndarray:
    """[n_real][4] per rank -> [world * n_real][4] on every rank, in global realization order."""
    dist = _dist()
    if dist is None:
        return np.asarray(diag)
    t = torch.from_numpy(np.ascontiguousarray(diag, dtype=np.float64)).to(_dev())
    out = [torch.empty_like(t) for _ in range(dist.get_world_size())]
    dist.all_gather(out, t)
    return torch.cat(out).cpu().numpy()
