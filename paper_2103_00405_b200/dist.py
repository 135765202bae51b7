"""Multi-GPU use of the ensemble path: trajectories are independent and keyed by trajectory id
(SURVEY.md 8(e)), so rank g simply takes a contiguous block of ids.  There is NO data-path
collective; one all_gather of the per-rank results at the end.  A single large-M trajectory
does not shard ("replicas only")."""
import numpy as np


def shard_range(n_traj, rank, world):
    """Contiguous block [first, first+count) of rank `rank`: sizes differ by at most one."""
    base, extra = divmod(int(n_traj), int(world))
    first = rank * base + min(rank, extra)
    return first, base + (1 if rank < extra else 0)


def ensemble_sharded(run_local, n_species, traj_first, n_traj, group=None):
    """run_local(first, count) -> dict(x[count,N], t, firings, stop, status) for this rank's block
    (normally Model.ensemble on this rank's GPU).  Returns the full ensemble on every rank, rows
    in trajectory order -- bit-identical to a single-GPU run by the determinism contract."""
    import torch
    import torch.distributed as dist
    rank, world = dist.get_rank(group), dist.get_world_size(group)
    first, count = shard_range(n_traj, rank, world)
    out = run_local(traj_first + first, count)
    gathered = [None] * world
    keys = [k for k in ("x", "t", "firings", "stop", "status") if out.get(k) is not None]
    dist.all_gather_object(gathered, {k: np.asarray(out[k]) for k in keys}, group=group)
    return {k: np.concatenate([g[k] for g in gathered], axis=0) for k in keys}
