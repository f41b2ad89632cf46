"""N > 1 host logic on CPU: world_size-2 gloo.  Each rank owns a slice of the charges, all-gathers the full
array (the one exchange of a time step), evaluates its target slice -- here with the
oracle standing in for the GPU -- and the concatenation must equal the unsharded evaluation."""
import os
import socket

import numpy as np
import pytest

from paper_2110_09214_b200.sharding import shard_range


def test_shard_range_covers_exactly_once():
    for n in (0, 1, 7, 4096, 1048576, 1048577):
        for world in (1, 2, 3, 8):
            nxt = 0
            for r in range(world):
                first, count = shard_range(n, world, r)
                assert first == nxt and count >= 0
                nxt = first + count
            assert nxt == n
            sizes = [shard_range(n, world, r)[1] for r in range(world)]
            assert max(sizes) - min(sizes) <= 1
    with pytest.raises(ValueError):
        shard_range(10, 2, 2)


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def _worker(rank, world, port, n, ret):
    import torch
    import torch.distributed as dist
    from oracle import ref
    from paper_2110_09214_b200 import workloads as W
    from paper_2110_09214_b200.sharding import all_gather_charges, all_gather_rows, shard_range as sr
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        wl = W.make_workload(1)
        xyzq = wl.xyzq[:n].copy()
        first, count = sr(n, world, rank)
        mine = torch.from_numpy(xyzq[first:first + count].copy())
        full = all_gather_charges(mine, n).numpy()
        assert np.array_equal(full, xyzq)                      # the exchange reproduces the global array
        tg = full[first:first + count]
        on, op = ref.eval_field(xyzq=full, verts=wl.verts, sigma=wl.sigma, targets=tg,
                                self_index=np.arange(first, first + count, dtype=np.int64), eps_pp=wl.eps_pp,
                                n_threads=1)
        part = torch.from_numpy(on + op)
        whole = all_gather_rows(part, n)
        if rank == 0:
            ret["sharded"] = whole.numpy()
            a, b = ref.eval_field(xyzq=xyzq, verts=wl.verts, sigma=wl.sigma, eps_pp=wl.eps_pp, n_threads=1)
            ret["whole"] = a + b
    finally:
        dist.destroy_process_group()


@pytest.mark.parametrize("n", [512, 341])          # equal slices (all_gather_into_tensor) and ragged (list gather)
def test_two_ranks_gloo_sharded_equals_whole(ref, n):
    import torch.multiprocessing as mp
    ref.build()
    world = 2
    port = _free_port()
    with mp.Manager() as mgr:
        ret = mgr.dict()
        mp.spawn(_worker, args=(world, port, n, ret), nprocs=world, join=True)
        sharded, whole = ret["sharded"], ret["whole"]
    assert sharded.shape == (n, 4)
    assert np.array_equal(sharded, whole)      # same arithmetic per target: bit-identical
