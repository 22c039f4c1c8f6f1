"""N > 1 path on CPU: world_size-2 gloo processes run parallel.run_sharded -- the very function bench.py --gpus N calls --
on a stand-in plan object whose apx_run is served by the oracle (there is no GPU here): each rank computes its slab of
the centre list and the gathered result must equal the single-rank result.  No collective touches the signature data
itself."""
import os
import socket
import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_2009_00735_b200.parallel import shard_range, gather_counts, run_sharded


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


class _OraclePlan:
    """Stands in for binding.Plan on a box without a GPU: same apx_run signature, CPU tensors, the oracle inside.
    Records what run_sharded handed it."""

    def __init__(self, w, dirs):
        self.w, self.dirs, self.calls = w, dirs, []

    def apx_run(self, xyz, types, centres, sig, counts=None, stream=None):
        from oracle import oracle as O
        self.calls.append(tuple(centres.shape))
        s, c = O.signatures(xyz.numpy(), types.numpy(), centres.numpy(), self.dirs, self.w.R, self.w.B,
                            k_lo=self.w.window[0], k_hi=self.w.window[1])
        sig.copy_(torch.from_numpy(s))
        if counts is not None:
            counts.copy_(torch.from_numpy(c.astype(np.int64)))


def _worker(rank, world, port, q):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    from oracle import oracle as O
    from workloads import make_config
    w = make_config(1)
    rng = np.random.default_rng(5)
    centres = (rng.random((7, 3)) - 0.5).astype(np.float32)          # 7 material points over 2 ranks: 4 + 3
    dirs = O.dirs_fibonacci(64)
    b0, e0 = shard_range(len(centres), rank, world)
    plan = _OraclePlan(w, dirs)
    sig_t = torch.full((e0 - b0, len(dirs), 2), -7.0)
    cnt_t = torch.full((e0 - b0,), -1, dtype=torch.int64)
    b, e = run_sharded(plan, torch.from_numpy(w.xyz), torch.from_numpy(w.types), torch.from_numpy(centres), sig_t, cnt_t,
                       rank=rank, world=world)
    assert (b, e) == (b0, e0) and plan.calls == [(e0 - b0, 3)]        # one apx_run on exactly this rank's slab
    sig = sig_t.numpy()
    allc = gather_counts(cnt_t, len(centres), rank, world)
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
