"""apx_fsp_noalloc (include/aptsig_ext.h): the FSP entry point whose scratch lives in a static device array, against the
existing apx_fsp on the same inputs, on two calls in a row that share the array.  Collected last on purpose (the file name
sorts behind every other test file).  Run with -m gpu on a B200."""
import math

import numpy as np
import pytest

import paper_2009_00735_b200 as apx
from oracle import oracle as O
from workloads.lattices import fcc_basis, lattice_in_ball, random_rotation

pytestmark = pytest.mark.gpu


def _tol(ref, n_ions, k_max, R):
    """The tolerance of the FSP parity tests (tests/test_gpu_next.py::_fsp_check)."""
    return 1e-4 * ref + np.maximum(1.0, n_ions)[:, None, None, None] * (2e-6 + 2 * math.pi * 2e-7 * math.sqrt(3) * k_max * R)


def _both(plan, centres, k_max, L, check_free=False):
    """One call of the existing path and one of the no-allocation path on the same inputs -> (ref, got, counts, counts)."""
    import torch
    dev = torch.device("cuda:0")
    M = len(centres)
    c = torch.from_numpy(centres).to(dev)
    ref = torch.full((M, L, L, L), -7.0, dtype=torch.float32, device=dev)
    got = torch.full((M, L, L, L), -9.0, dtype=torch.float32, device=dev)
    cr = torch.full((M,), -1, dtype=torch.int32, device=dev)
    cg = torch.full((M,), -2, dtype=torch.int32, device=dev)
    plan.apx_fsp(c, k_max, L, ref, cr)
    torch.cuda.synchronize()
    free0 = torch.cuda.mem_get_info()[0]
    plan.apx_fsp_noalloc(c, k_max, L, got, cg)
    torch.cuda.synchronize()
    if check_free:                                         # (every kernel has run before: no lazy module loading left)
        assert torch.cuda.mem_get_info()[0] >= free0, "apx_fsp_noalloc took device memory"
    return ref.cpu().numpy(), got.cpu().numpy(), cr.cpu().numpy(), cg.cpu().numpy()


def test_fsp_noalloc_matches_apx_fsp_on_two_calls_in_a_row():
    import torch
    dev = torch.device("cuda:0")
    rng = np.random.Generator(np.random.PCG64(77))
    xyz = np.ascontiguousarray(lattice_in_ball(0.405, fcc_basis, random_rotation(rng), (0, 0, 0), 4.0).astype(np.float32))
    types = np.zeros(len(xyz), np.uint8)
    R = 2.75                                               # ~5100 ions around the origin: more than the tensor-core kernel holds
    plan = apx.Plan(R, 256, O.dirs_fibonacci(8), k_lo=7, k_hi=17, device=0)
    plan.apx_ingest(torch.from_numpy(xyz).to(dev), torch.from_numpy(types).to(dev))
    # call 1: a ROI that goes through the device list (tensor path) beside a small one; call 2: other centres, other grid, no
    # listed ROI -- the k axis and the list count left by call 1 must not leak into it; then call 1's inputs once more
    calls = ((np.array([[0.1, 0.2, -0.1], [3.9, 0.0, 0.0]], np.float32), 4.0, 12),
             (np.array([[3.8, 0.3, 0.0], [0.0, 3.9, 0.1], [9.0, 9.0, 9.0]], np.float32), 2.0 * math.pi, 9),
             (np.array([[0.1, 0.2, -0.1], [3.9, 0.0, 0.0]], np.float32), 4.0, 12))
    for path in (0, 1):                                    # 0 = tensor cores + FP32 for listed ROIs, 1 = FP32 pipe only
        plan.apx_fsp_set_path(path)
        for i, (centres, k_max, L) in enumerate(calls):
            ref, got, cr, cg = _both(plan, centres, k_max, L, check_free=i > 0)
            assert (cr == cg).all() and (cr >= 0).all()
            assert (ref >= 0).all() and (got >= 0).all()   # every element written by both paths
            err = np.abs(got - ref)
            assert (err <= _tol(ref, cr.astype(np.float64), k_max, R)).all(), (path, i, err.max())
        assert cr[0] > 4096 and cr[1] < 4096               # the last call had a listed ROI and a directly served one
    plan.apx_plan_destroy()


def test_fsp_noalloc_rejects_sizes_beyond_the_static_scratch():
    import torch
    dev = torch.device("cuda:0")
    max_m, max_l, nbytes = apx.apx_fsp_noalloc_limits()
    assert (max_m, max_l) == (16384, 1024) and nbytes <= 1 << 20
    xyz = np.ascontiguousarray(lattice_in_ball(0.405, fcc_basis, np.eye(3), (0, 0, 0), 1.5).astype(np.float32))
    plan = apx.Plan(1.0, 256, O.dirs_fibonacci(8), k_lo=7, k_hi=17, device=0)
    plan.apx_ingest(torch.from_numpy(xyz).to(dev), None)
    M = max_m + 1
    c = torch.zeros((M, 3), dtype=torch.float32, device=dev)
    out = torch.full((M, 1, 1, 1), -7.0, dtype=torch.float32, device=dev)
    with pytest.raises(apx.ApxError) as ei:
        plan.apx_fsp_noalloc(c, 1.0, 1, out)
    assert ei.value.status == -5 and str(max_m) in str(ei.value) and "static scratch" in str(ei.value)
    # L beyond the k-axis part of the array: rejected before anything is touched (straight through the C ABI; the output
    # of such a call would be 4 GB)
    from paper_2009_00735_b200.binding import _lib
    assert _lib().apx_fsp_noalloc(plan._h, c.data_ptr(), 1, 1.0, max_l + 1, out.data_ptr(), None, None) == -5
    torch.cuda.synchronize()
    assert (out == -7.0).all()                             # nothing was launched
    plan.apx_fsp_noalloc(c[:max_m], 1.0, 1, out[:max_m])   # the maximum itself is served: |F(0)| = N_w
    torch.cuda.synchronize()
    n = len(O.members(xyz, None, np.zeros(3, np.float32), 1.0))
    assert (out[:max_m] == float(n)).all() and (out[max_m:] == -7.0).all()
    plan.apx_plan_destroy()
