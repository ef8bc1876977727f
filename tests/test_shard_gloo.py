"""Multi-GPU host logic on CPU: the paper's contiguous batch slices, the
rank-local view of a batch and the result gather, with torch.distributed / gloo at world size 2.  Each rank
evaluates its slice with the oracle (the CUDA library needs a GPU); the gathered result must equal the
single-process evaluation of the whole batch bit for bit."""
import os
import socket

import numpy as np
import pytest

import gen
import oracle
from paper_2604_08463_b200 import shard


def test_batch_slices_are_the_papers_formula():
    for B in (0, 1, 5, 64, 1000, 6400):
        for P in (1, 2, 3, 8, 64):
            prev = 0
            for k in range(P):
                a, b = shard.batch_slice(k, P, B)
                assert a == (k * B) // P and b == ((k + 1) * B) // P
                assert a == prev and b >= a
                prev = b
            assert prev == B
            sizes = [shard.batch_slice(k, P, B)[1] - shard.batch_slice(k, P, B)[0] for k in range(P)]
            assert max(sizes) - min(sizes) <= 1
    with pytest.raises(ValueError):
        shard.batch_slice(2, 2, 10)


def test_shard_batch_holds_only_referenced_data():
    w = gen.make_config(3, nside=8, batch=10, ndata=3)
    seen = []
    for k in range(3):
        s = shard.shard_batch(w.cfg_of, w.data_of, k, 3)
        assert np.array_equal(s["data_ids"][s["data_of"]], w.data_of[s["start"]:s["end"]])
        assert np.array_equal(s["cfg_of"], w.cfg_of[s["start"]:s["end"]])
        assert len(set(s["data_ids"].tolist())) == len(s["data_ids"])
        seen += list(range(s["start"], s["end"]))
    assert seen == list(range(w.batch))


def _entry(w, params, off, e, data):
    c = int(w.cfg_of[e])
    return oracle.nll_grad(oracle.Model(w.freqs), data, w.ninv, w.maps[w.cfg_maps[c]], w.K_of_cfg(c),
                           params[off[e]:off[e + 1]], region=w.region_idx, nregion=w.nregion)


def _worker(rank, world, port, out):
    import torch.distributed as dist
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        w = gen.make_config(3, nside=8, batch=7, ndata=3)
        params = w.params_jittered(seed=31)
        off = w.param_offsets()
        s = shard.shard_batch(w.cfg_of, w.data_of, rank, world)
        # the rank synthesises only the noise realisations it references
        local_data = gen.synthesize(w.truth, w.freqs, w.sigma, tuple(int(i) for i in s["data_ids"]))
        nll, grad = [], []
        for j, e in enumerate(range(s["start"], s["end"])):
            r = _entry(w, params, off, e, local_data[s["data_of"][j]])
            nll.append(r["nll"])
            grad.append(r["grad"])
        nll = np.stack(nll) if nll else np.zeros((0, w.nregion))
        grad = np.concatenate(grad) if grad else np.zeros(0)
        pa, pb = shard.param_slice(off, rank, world)
        assert grad.shape[0] == pb - pa
        nll_all = shard.gather_concat(nll, dist)
        grad_all = shard.gather_concat(grad, dist)
        dist.barrier()
        if rank == 0:
            np.savez(out, nll=nll_all, grad=grad_all)
    finally:
        dist.destroy_process_group()


def test_two_ranks_gloo_equal_single_process(tmp_path):
    import torch.multiprocessing as mp
    with socket.socket() as sk:
        sk.bind(("127.0.0.1", 0))
        port = sk.getsockname()[1]
    out = str(tmp_path / "gathered.npz")
    mp.spawn(_worker, args=(2, port, out), nprocs=2, join=True)
    got = np.load(out)
    w = gen.make_config(3, nside=8, batch=7, ndata=3)
    params = w.params_jittered(seed=31)
    off = w.param_offsets()
    ref = [_entry(w, params, off, e, w.data()[int(w.data_of[e])]) for e in range(w.batch)]
    assert np.array_equal(got["nll"], np.stack([r["nll"] for r in ref]))
    assert np.array_equal(got["grad"], np.concatenate([r["grad"] for r in ref]))
