"""Multi-GPU sharding of a batch: batch entries are independent, so rank k
of P owns the paper's contiguous slice [floor(k B / P), floor((k+1) B / P)) (L201), holds only the data sets it
references, runs its own Context on its own GPU and the results are concatenated in rank order.  There is no
collective on the data path; the gather below moves results only (nll, grad: a few MB at most).

Host logic only: nothing here touches CUDA, so it is covered by world-size-2 gloo tests on CPU."""
import numpy as np


def batch_slice(rank: int, world: int, batch: int):
    """[start, end) of rank's entries: i_start = floor(k N / P), i_end = floor((k+1) N / P)."""
    if not (0 <= rank < world) or batch < 0:
        raise ValueError("bad rank/world/batch")
    return (rank * batch) // world, ((rank + 1) * batch) // world


def shard_batch(cfg_of, data_of, rank: int, world: int):
    """Rank-local view of a batch.  Returns dict with
    start, end   : the global entry range of this rank
    cfg_of       : int32 [n_local]  (configuration ids are global: cluster maps are small and replicated)
    data_of      : int32 [n_local]  local data-set indices into `data_ids`
    data_ids     : int64 [n_data_local] global ids of the data sets this rank must hold, ascending
    """
    cfg_of = np.asarray(cfg_of, dtype=np.int32)
    data_of = np.asarray(data_of, dtype=np.int32)
    a, b = batch_slice(rank, world, int(cfg_of.shape[0]))
    ids, local = np.unique(data_of[a:b], return_inverse=True)
    return {"start": a, "end": b, "cfg_of": cfg_of[a:b].copy(), "data_of": local.astype(np.int32),
            "data_ids": ids.astype(np.int64)}


def param_slice(param_off, rank: int, world: int):
    """[start, end) of rank's parameters in the global parameter / gradient vector (param_off: int64 [B+1])."""
    a, b = batch_slice(rank, world, len(param_off) - 1)
    return int(param_off[a]), int(param_off[b])


def gather_concat(local: np.ndarray, dist=None):
    """Concatenation over ranks (rank order) of a 1-D or [n_local, ...] array whose first dimension differs per
    rank.  `dist` is an initialised torch.distributed module (any backend); None = single process."""
    local = np.ascontiguousarray(local)
    if dist is None or not dist.is_initialized() or dist.get_world_size() == 1:
        return local
    parts = [None] * dist.get_world_size()
    dist.all_gather_object(parts, local)
    return np.concatenate(parts, axis=0)
