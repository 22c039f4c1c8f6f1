"""N > 1 path on CPU: world_size-2 gloo processes shard the material points exactly as bench.py / run_sharded do,
each rank computes its slab (with the oracle standing in for the GPU here) and the gathered result must equal the
single-rank result.  No collective touches the signature data itself."""
import os
import socket
import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_2009_00735_b200.parallel import shard_range, gather_counts


def test_shard_range_partitions():
    for M in (0, 1, 7, 1000, 175616):
        for world in (1, 2, 3, 8):
            cuts = [shard_range(M, r, world) for r in range(world)]
            assert cuts[0][0] == 0 and cuts[-1][1] == M
            assert all(cuts[i][1] == cuts[i + 1][0] for i in range(world - 1))
            sizes = [e - b for b, e in cuts]
            assert max(sizes) - min(sizes) <= 1
    with pytest.raises(ValueError):
        shard_range(10, 2, 2)


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, q):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    from oracle import oracle as O
    from workloads import make_config
    w = make_config(1)
    rng = np.random.default_rng(5)
    centres = (rng.random((7, 3)) - 0.5).astype(np.float32)          # 7 material points over 2 ranks: 4 + 3
    dirs = O.dirs_fibonacci(64)
    b, e = shard_range(len(centres), rank, world)
    sig, cnt = O.signatures(w.xyz, w.types, centres[b:e], dirs, w.R, w.B, k_lo=w.window[0], k_hi=w.window[1])
    allc = gather_counts(torch.from_numpy(cnt.astype(np.int64)), len(centres), rank, world)
    # signatures stay sharded; for the check only, rank 0 collects them as python objects
    parts = [None] * world
    dist.all_gather_object(parts, (b, e, sig))
    if rank == 0:
        q.put((allc.numpy(), parts))
    dist.barrier()
    dist.destroy_process_group()


def test_two_rank_gloo_matches_single_rank():
    from oracle import oracle as O
    from workloads import make_config
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    allc, parts = q.get(timeout=120)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    w = make_config(1)
    rng = np.random.default_rng(5)
    centres = (rng.random((7, 3)) - 0.5).astype(np.float32)
    dirs = O.dirs_fibonacci(64)
    sig, cnt = O.signatures(w.xyz, w.types, centres, dirs, w.R, w.B, k_lo=w.window[0], k_hi=w.window[1])
    assert (allc == cnt).all()
    got = np.concatenate([s for _, _, s in sorted(parts, key=lambda t: t[0])])
    assert [(b, e) for b, e, _ in sorted(parts, key=lambda t: t[0])] == [(0, 4), (4, 7)]
    assert np.array_equal(got, sig)
