"""GPU parity on the edge cases of the path: empty inputs, ROIs that overflow the kernels' shared-memory ion
buffers (deferred list, streaming fallback, multi-pass binning), every B the ABI admits, pad = 0 with the bin
clamp active, non-unit directions, ragged direction counts.  Same comparator and tolerances as test_gpu_parity."""
from types import SimpleNamespace

import numpy as np
import pytest

import paper_2009_00735_b200 as apx
from oracle import oracle as O
from workloads.lattices import fcc_basis, lattice_in_ball, random_rotation, jitter_thin_shuffle
from workloads.configs import A_AL, window_for
from _parity import run_gpu, assert_parity

pytestmark = pytest.mark.gpu
PATHS = [pytest.param(apx.APX_FLAG_FORCE_FFT, id="fft"), pytest.param(0, id="auto")]


def _ball(R_cloud, eta=1.0, sigma=0.0, seed=7):
    rng = np.random.Generator(np.random.PCG64(seed))
    rot = random_rotation(rng)
    sites = lattice_in_ball(A_AL, fcc_basis, rot, (0, 0, 0), R_cloud)
    xyz, _, _, _ = jitter_thin_shuffle(sites, rng, eta, sigma)
    return xyz, np.zeros(len(xyz), np.uint8)


def _case(xyz, types, R, B):
    return SimpleNamespace(xyz=xyz, types=types, R=R, B=B)


def _check(w, dirs, centres, window, flags, pad=1):
    got, cnt, path = run_gpu(apx, w, dirs, centres, window=window, flags=flags, pad=pad)
    k_lo, k_hi = window if window else (0, 0)
    ref, rc, win = O.signatures(w.xyz, w.types, centres, dirs, w.R, w.B, pad=pad, k_lo=k_lo, k_hi=k_hi, want_window=True)
    assert_parity(got, cnt, ref, rc, win, k_lo if window else 1)
    return path, cnt


@pytest.mark.parametrize("flags", PATHS)
def test_empty_cloud_and_no_centres(flags):
    import torch
    dirs = O.dirs_fibonacci(100)
    plan = apx.Plan(1.0, 256, dirs, k_lo=7, k_hi=17, device=0, flags=flags)
    dev = torch.device("cuda:0")
    xyz = torch.zeros((0, 3), dtype=torch.float32, device=dev)
    centres = torch.tensor([[0.0, 0.0, 0.0], [1.0, 2.0, 3.0]], dtype=torch.float32, device=dev)
    sig = torch.full((2, 100, 2), -7.0, dtype=torch.float32, device=dev)
    counts = torch.full((2,), 9, dtype=torch.int32, device=dev)
    plan.apx_run(xyz, None, centres, sig, counts)                 # N = 0: every ROI empty
    plan.apx_query(centres[:0], sig[:0], counts[:0])              # M = 0 is valid
    torch.cuda.synchronize()
    assert (counts.cpu().numpy() == 0).all()
    s = sig.cpu().numpy()
    assert (s[..., 0] == 0.0).all() and (s[..., 1] == 7.0).all()   # empty ROI: (0, k_lo)
    plan.apx_plan_destroy()


@pytest.mark.parametrize("flags", PATHS)
def test_dense_roi_overflows_mma_ion_buffer(flags):
    """Noiseless full-density fcc Al, R = 2.2 nm: ~2700 ions per ROI > the MMA kernel's shared ion buffer at
    B = 1024, so the auto path defers these material points to the FFT kernel."""
    xyz, types = _ball(3.0)
    dirs = O.dirs_fibonacci(200)
    centres = np.array([[0, 0, 0], [0.3, -0.2, 0.1], [2.5, 0, 0]], np.float32)    # the last one is a partial ROI
    w = _case(xyz, types, 2.2, 1024)
    path, cnt = _check(w, dirs, centres, window_for(2.2, 1024), flags)
    assert cnt[0] > 2048


def test_multipass_binning_mma_b256():
    """B = 256 leaves room for 4096 ions in the MMA kernel: a ROI with more than 2048 ions is binned in two passes
    (u16 counters read as fp16 are exact up to 2048) that accumulate in TMEM."""
    xyz, types = _ball(3.0)
    dirs = O.dirs_fibonacci(96)
    centres = np.array([[0, 0, 0], [0.2, 0.1, -0.3]], np.float32)
    w = _case(xyz, types, 2.2, 256)
    path, cnt = _check(w, dirs, centres, window_for(2.2, 256), 0)
    assert path == 1 and cnt.min() > 2048


def test_streaming_fallback_fft():
    """ROI larger than the FFT kernel's shared ion buffer (~6900 ions at B = 1024): cell rows are streamed again
    for every direction group."""
    xyz, types = _ball(4.0)
    dirs = O.dirs_fibonacci(64)
    centres = np.array([[0, 0, 0]], np.float32)
    w = _case(xyz, types, 3.3, 1024)
    path, cnt = _check(w, dirs, centres, (20, 60), apx.APX_FLAG_FORCE_FFT)
    assert cnt[0] > 7500


@pytest.mark.parametrize("flags", PATHS)
@pytest.mark.parametrize("B", [256, 512, 1024, 2048, 4096])
def test_every_bin_count(flags, B):
    xyz, types = _ball(1.6, eta=0.6, sigma=0.04, seed=11)
    dirs = O.dirs_fibonacci(77)                                    # ragged: not a multiple of 32 / 16 / 8
    centres = np.array([[0, 0, 0], [0.4, 0.4, -0.2]], np.float32)
    w = _case(xyz, types, 1.2, B)
    _check(w, dirs, centres, window_for(1.2, B), flags)
    if B <= 512:
        _check(w, dirs[:40], centres, None, flags)                 # full window [1, B/2]


@pytest.mark.parametrize("B", [512, 2048])
@pytest.mark.parametrize("flags", PATHS)
def test_pad0_and_non_unit_directions_clamp(flags, B):
    """pad = 0 (north_star's [-R, R]) puts ions on the last bin edge, and directions 3 % longer than unit push
    projections past +-R: the bin clamp of Eq. 1 (reading #5) must act on both paths."""
    xyz, types = _ball(1.6, eta=0.7, sigma=0.03, seed=13)
    dirs = (O.dirs_fibonacci(64).astype(np.float64) * 1.03).astype(np.float32)
    centres = np.array([[0, 0, 0]], np.float32)
    w = _case(xyz, types, 1.2, B)
    _check(w, dirs, centres, (5, 20), flags, pad=0)
    _check(w, dirs, centres, (5, 20), flags, pad=1)


def test_run_host_matches_device_path():
    """apx_run_host (host pointers, slabbed and pipelined copies) returns exactly what apx_run leaves on the device."""
    import torch
    xyz, types = _ball(2.4, eta=0.5, sigma=0.05, seed=17)
    rng = np.random.default_rng(3)
    centres = ((rng.random((301, 3)) - 0.5) * 2.0).astype(np.float32)       # 301 points: four ragged slabs
    dirs = O.dirs_fibonacci(96)
    plan = apx.Plan(1.0, 256, dirs, k_lo=7, k_hi=17, device=0)
    dev = torch.device("cuda:0")
    sig_d = torch.empty((301, 96, 2), dtype=torch.float32, device=dev)
    cnt_d = torch.empty(301, dtype=torch.int32, device=dev)
    plan.apx_run(torch.from_numpy(xyz).to(dev), torch.from_numpy(types).to(dev), torch.from_numpy(centres).to(dev), sig_d, cnt_d)
    torch.cuda.synchronize()
    sig_h = torch.empty((301, 96, 2), dtype=torch.float32).pin_memory()
    cnt_h = torch.empty(301, dtype=torch.int32).pin_memory()
    plan.apx_run_host(torch.from_numpy(xyz), torch.from_numpy(types), torch.from_numpy(centres), sig_h, cnt_h)
    assert torch.equal(sig_h, sig_d.cpu()) and torch.equal(cnt_h, cnt_d.cpu())
    ref, rc = O.signatures(xyz, types, centres[:5], dirs, 1.0, 256, k_lo=7, k_hi=17)
    assert (cnt_h[:5].numpy().astype(np.uint32) == rc).all()
    plan.apx_plan_destroy()


@pytest.mark.parametrize("B", [1024, 2048])
@pytest.mark.parametrize("centre_ions", [False, True], ids=["fixups", "overflow"])
@pytest.mark.parametrize("flags", [pytest.param(0, id="half"), pytest.param(apx.APX_FLAG_NO_PAIRING, id="full")])
def test_half_grid_mode_with_exact_integer_projections(flags, centre_ions, B):
    """Half-grid mode on a symmetric grid: b(-n) = B-1-b(n) holds only while n'.d is not an integer
    (floor(-x) = -floor(x) - 1); for an exact integer b(-n) = B - b(n), and the kernel must redo -n on its own.
    R = (B/2-1)/(B/4) makes s = B/4 exactly, so ions on a 1/4 grid project to exact integers along the axis directions
    (+-x, +-y, +-z are vertices of the geodesic grid) and a random half of the cloud does not: using the mirrored
    histogram there would shift the grid ions against the rest by one bin and change the amplitudes.  With an ion
    exactly on each centre (x = +-0 for EVERY direction) the list of flagged pairs overflows and the material
    points are redone by the general kernel."""
    rng = np.random.Generator(np.random.PCG64(11))
    R = (B / 2 - 1) / (B / 4)
    c2 = np.array([0.25, 0.5, -0.25])
    g = np.arange(-10, 11) / 4.0
    grid = np.stack(np.meshgrid(g, g, g, indexing="ij"), -1).reshape(-1, 3)
    grid = grid[(grid ** 2).sum(1) <= 2.6 ** 2]
    on_centre = ((grid == 0).all(1)) | ((grid == c2).all(1))
    grid = grid[(rng.random(len(grid)) < 0.25) & ~on_centre]
    if centre_ions:
        grid = np.concatenate([grid, np.zeros((1, 3)), c2[None]])
    rnd = rng.uniform(-2.6, 2.6, size=(900, 3))
    xyz = np.concatenate([grid, rnd]).astype(np.float32)
    rng.shuffle(xyz)
    dirs = apx.apx_dirs_geodesic(3)
    assert any((np.abs(d) == (1, 0, 0)).all() for d in dirs)
    centres = np.array([[0, 0, 0], c2], np.float32)
    w = _case(xyz, np.zeros(len(xyz), np.uint8), R, B)
    plan = apx.Plan(R, B, dirs, k_lo=15, k_hi=34, device=0, flags=flags)
    assert plan.apx_plan_path() == 1 and plan.apx_plan_paired() == (0 if flags else 1)
    _, s, _ = plan.apx_plan_constants()
    assert s == B / 4
    plan.apx_plan_destroy()
    _check(w, dirs, centres, (15, 34), flags)


def test_half_grid_mode_is_off_for_asymmetric_grids():
    plan = apx.Plan(2.0, 1024, O.dirs_fibonacci(1000), k_lo=15, k_hi=34, device=0)
    assert plan.apx_plan_path() == 1 and plan.apx_plan_paired() == 0
    plan.apx_plan_destroy()


@pytest.mark.parametrize("flags", [pytest.param(0, id="half"), pytest.param(apx.APX_FLAG_NO_PAIRING, id="full")])
def test_b2048_tensor_path_multipass_and_deferred(flags):
    """B = 2048 on the tensor-core kernel (16 direction slots per group, one histogram buffer): a ROI of ~2700 ions is
    binned in two passes of <= 2048 ions, a ROI of more than 4096 ions is left to the general kernel, a partial ROI
    and an empty one ride along; whole symmetric grid, so the half-grid mode and its fix-up groups run as well."""
    xyz, types = _ball(3.4)
    dirs = apx.apx_dirs_geodesic(3)
    w = _case(xyz, types, 2.2, 2048)
    centres = np.array([[0, 0, 0], [0.3, -0.2, 0.1], [3.0, 0, 0], [9.0, 9.0, 9.0]], np.float32)
    plan = apx.Plan(2.2, 2048, dirs, k_lo=23, k_hi=51, device=0, flags=flags)
    assert plan.apx_plan_path() == 1 and plan.apx_plan_paired() == (0 if flags else 1)
    plan.apx_plan_destroy()
    path, cnt = _check(w, dirs, centres, (23, 51), flags)
    assert path == 1 and cnt[0] > 2048 and cnt[3] == 0
    w = _case(xyz, types, 2.7, 2048)
    path, cnt = _check(w, dirs, centres[:2], window_for(2.7, 2048), flags)
    assert path == 1 and cnt.min() > 4096
