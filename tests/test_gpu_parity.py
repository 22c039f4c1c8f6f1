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
