"""GPU parity: the CUDA path (through the C ABI) against the CPU oracle, element by element, on the
same seeded inputs.  Run with -m gpu on a B200."""
import numpy as np
import pytest

import paper_2009_00735_b200 as apx
from oracle import oracle as O
from workloads import make_config
from _parity import run_gpu, assert_parity

pytestmark = pytest.mark.gpu

PATHS = [pytest.param(apx.APX_FLAG_FORCE_FFT, id="fft"), pytest.param(0, id="auto")]


def _oracle(w, dirs, centres, window, accepted=None, pad=1):
    k_lo, k_hi = window if window else (0, 0)
    sig, cnt, win = O.signatures(w.xyz, w.types, centres, dirs, w.R, w.B, pad=pad, k_lo=k_lo, k_hi=k_hi,
                                 accepted=accepted, want_window=True)
    return sig, cnt, win, (k_lo if window else 1)


@pytest.mark.parametrize("flags", PATHS)
@pytest.mark.parametrize("window", ["bench", None], ids=["window", "full"])
def test_cfg1_exhaustive(flags, window):
    w = make_config(1)
    dirs = O.dirs_fibonacci(w.D)
    win = w.window if window == "bench" else None
    got, cnt, path = run_gpu(apx, w, dirs, w.centres, window=win, flags=flags)
    ref, rc, rwin, klo = _oracle(w, dirs, w.centres, win)
    assert_parity(got, cnt, ref, rc, rwin, klo)


@pytest.mark.parametrize("flags", PATHS)
def test_cfg2_sampled_points_all_directions(flags):
    w = make_config(2)
    dirs = O.dirs_fibonacci(w.D)
    idx = np.array([0, 9, 99, 455, 500, 555, 901, 999])       # corners, faces, interior
    got, cnt, path = run_gpu(apx, w, dirs, w.centres[idx], window=w.window, flags=flags, split=True)
    ref, rc, rwin, klo = _oracle(w, dirs, w.centres[idx], w.window)
    assert_parity(got, cnt, ref, rc, rwin, klo)


def test_cfg2_full_window_sample():
    w = make_config(2)
    dirs = O.dirs_fibonacci(w.D)[::20]
    idx = np.array([444, 555])
    got, cnt, _ = run_gpu(apx, w, dirs, w.centres[idx], window=None)
    ref, rc, rwin, klo = _oracle(w, dirs, w.centres[idx], None)
    assert_parity(got, cnt, ref, rc, rwin, klo)


def test_histograms_bit_exact_cfg2():
    import torch
    w = make_config(2)
    dirs = O.dirs_fibonacci(w.D)
    plan = apx.Plan(w.R, w.B, dirs, device=0)
    plan.apx_ingest(torch.from_numpy(w.xyz).cuda(), torch.from_numpy(w.types).cuda())
    for c in (w.centres[555], w.centres[0], np.array([19.5, 10.0, 0.3], np.float32)):
        out = torch.empty((512, w.B), dtype=torch.int32, device="cuda")
        plan.apx_debug_histograms(c, 1000, 512, out)
        torch.cuda.synchronize()
        ref, n = O.histograms(w.xyz, w.types, c, dirs, w.R, w.B, d0=1000, nd=512)
        assert (out.cpu().numpy().astype(np.uint32) == ref).all()
    plan.apx_plan_destroy()


@pytest.mark.parametrize("flags", PATHS)
@pytest.mark.parametrize("mask", [{0}, {1}])
def test_cfg3_type_filter_sample(flags, mask):
    w = make_config(3)
    dirs = O.dirs_geodesic(6)[::16]                       # 2561 of the 40 962 nodes
    g = w.centres.reshape(30, 30, 30, 3)
    centres = np.stack([g[14, 10, 10], g[15, 10, 10], g[0, 0, 0], g[29, 15, 3], g[3, 20, 20], g[25, 5, 17]])
    got, cnt, _ = run_gpu(apx, w, dirs, centres, accepted=mask, window=w.window, flags=flags)
    ref, rc, rwin, klo = _oracle(w, dirs, centres, w.window, accepted=mask)
    assert_parity(got, cnt, ref, rc, rwin, klo)


@pytest.mark.parametrize("flags", PATHS)
def test_cfg5_large_B_sample(flags):
    w = make_config(5, scale=0.3)
    dirs = O.dirs_geodesic(6)[::32]
    centres = w.centres[[0, 500, 865, 1727]]
    got, cnt, _ = run_gpu(apx, w, dirs, centres, accepted={0}, window=w.window, flags=flags)
    ref, rc, rwin, klo = _oracle(w, dirs, centres, w.window, accepted={0})
    assert_parity(got, cnt, ref, rc, rwin, klo)


@pytest.mark.parametrize("flags", PATHS)
def test_cfg4_sample(flags):
    w = make_config(4, scale=0.25)
    dirs = O.dirs_geodesic(6)[::32]
    centres = w.centres[::200]
    got, cnt, _ = run_gpu(apx, w, dirs, centres, window=w.window, flags=flags)
    ref, rc, rwin, klo = _oracle(w, dirs, centres, w.window)
    assert_parity(got, cnt, ref, rc, rwin, klo)


def _full_launch(w, dirs, accepted=None):
    """The whole config in ONE apx_run (the launch configuration bench.py times); results stay on the device."""
    import torch
    dev = torch.device("cuda:0")
    plan = apx.Plan(w.R, w.B, dirs, k_lo=w.window[0], k_hi=w.window[1], accepted_types=accepted, device=0)
    xyz = torch.from_numpy(w.xyz).to(dev)
    types = torch.from_numpy(w.types).to(dev)
    c = torch.from_numpy(w.centres).to(dev)
    M = c.shape[0]
    sig = torch.full((M, len(dirs), 2), -7.0, dtype=torch.float32, device=dev)
    counts = torch.full((M,), -1, dtype=torch.int32, device=dev)
    plan.apx_run(xyz, types, c, sig, counts)
    torch.cuda.synchronize()
    plan.apx_plan_destroy()
    return sig, counts


def _check_full(w, dirs, sig, counts, idx, accepted=None, count_all=True):
    import torch
    M = len(w.centres)
    cnt = counts.cpu().numpy().astype(np.uint32)
    if count_all:
        # every material point: ROI ion count against the oracle's brute force (one direction is enough for counts)
        _, rc_all = O.signatures(w.xyz, w.types, w.centres, dirs[:1], w.R, w.B, k_lo=w.window[0], k_hi=w.window[1],
                                 accepted=accepted)
        assert (cnt == rc_all).all()
    # properties that hold for every output: 0 <= A <= N_c (P4), k inside the window, nothing left unwritten
    amp, k = sig[..., 0], sig[..., 1]
    assert bool((amp >= 0).all()) and bool((amp <= counts.to(torch.float32)[:, None] * (1 + 1e-5) + 1e-3).all())
    assert bool((k >= w.window[0]).all()) and bool((k <= w.window[1]).all())
    # sampled material points x all directions, element by element
    got = sig[torch.from_numpy(idx).cuda()].cpu().numpy()
    ref, rc, rwin = O.signatures(w.xyz, w.types, w.centres[idx], dirs, w.R, w.B, k_lo=w.window[0], k_hi=w.window[1],
                                 accepted=accepted, want_window=True)
    assert_parity(got, cnt[idx], ref, rc, rwin, w.window[0])


def test_cfg2_full_size_bench_launch():
    w = make_config(2)
    dirs = O.dirs_fibonacci(w.D)
    sig, counts = _full_launch(w, dirs)
    _check_full(w, dirs, sig, counts, np.array([0, 99, 137, 455, 500, 555, 900, 999]))


def test_cfg3_full_size_al_filter():
    """Config 3 at full size (27 000 material points x 40 962 geodesic directions, 8.85 GB of signatures), Al filter."""
    w = make_config(3)
    dirs = O.dirs_geodesic(6)
    sig, counts = _full_launch(w, dirs, accepted={0})
    g = np.arange(27000).reshape(30, 30, 30)
    idx = np.array([g[14, 10, 10], g[15, 10, 10], g[0, 0, 0], g[29, 15, 3], g[3, 20, 20], g[7, 7, 29]])
    _check_full(w, dirs, sig, counts, idx, accepted={0})


def test_cfg4_full_size():
    """Config 4 at full size (175 616 material points x 40 962 directions, 57.5 GB of signatures, half-grid mode):
    properties on every output, sampled material points x all directions element by element (the brute-force count
    of every ROI would take the oracle minutes, so counts are checked on the sample)."""
    w = make_config(4)
    dirs = O.dirs_geodesic(6)
    sig, counts = _full_launch(w, dirs)
    rng = np.random.default_rng(4)
    idx = np.sort(np.concatenate([[0, len(w.centres) - 1], rng.choice(len(w.centres), 10, replace=False)]))
    _check_full(w, dirs, sig, counts, idx, count_all=False)


def test_cfg5_full_size_al_filter():
    """Config 5 at full size (64 000 x 40 962, B = 2048, Al filter) on the tensor-core kernel in half-grid mode."""
    w = make_config(5)
    dirs = O.dirs_geodesic(6)
    sig, counts = _full_launch(w, dirs, accepted={0})
    rng = np.random.default_rng(5)
    idx = np.sort(np.concatenate([[0, len(w.centres) - 1], rng.choice(len(w.centres), 6, replace=False)]))
    _check_full(w, dirs, sig, counts, idx, accepted={0}, count_all=False)
