"""GPU parity: the CUDA path (through the C ABI) against the CPU oracle, element by element, on the
same seeded inputs.  Run with -m gpu on a B200."""
import functools

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
    w = _config(2)
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


@functools.lru_cache(maxsize=2)
def _config(cfg):
    return make_config(cfg)


def _dirs_for(w):
    return O.dirs_geodesic(w.grid[1]) if w.grid[0] == "geodesic" else O.dirs_fibonacci(w.D)


def _hist_points(w, cfg, n=8):
    """Seeded material points for the histogram check: first / last centre (box corners), one off-grid point on a box
    face, and for config 3 the two grid planes next to the phase boundary."""
    M = len(w.centres)
    rng = np.random.default_rng(100 + cfg)
    pts = [w.centres[0], w.centres[M - 1]] if M > 1 else [w.centres[0]]
    if cfg == 3:
        g = w.centres.reshape(30, 30, 30, 3)
        pts += [g[14, 11, 7], g[15, 11, 7]]
    if M > 1:
        hi = w.centres.max(0)
        pts.append(np.array([hi[0] + 0.45, 0.5 * hi[1], 0.31 * hi[2]], np.float32))
        pts += [w.centres[i] for i in rng.choice(M, n - len(pts), replace=False)]
    return pts


@pytest.mark.parametrize("flags", PATHS)
@pytest.mark.parametrize("cfg", [1, 2, 3, 4, 5])
def test_histograms_bit_exact_production_kernels(cfg, flags):
    """north_star: histogram counts bit-exact.  apx_debug_histograms runs the plan's PRODUCTION kernel
    (k_signature_mma incl. half-grid mirroring / fix-ups, or k_signature_fft) with its export switched on: the
    shared-memory histogram the DFT reads, against the oracle's Eq. 1, 8 material points x 512 directions per config."""
    import torch
    w = _config(cfg)
    dirs = _dirs_for(w)
    accepted = {0} if cfg in (3, 5) else None
    plan = apx.Plan(w.R, w.B, dirs, k_lo=w.window[0], k_hi=w.window[1], accepted_types=accepted, device=0, flags=flags)
    if flags == 0:
        assert plan.apx_plan_path() == 1 and plan.apx_plan_paired() == (1 if w.grid[0] == "geodesic" else 0)
    plan.apx_ingest(torch.from_numpy(w.xyz).cuda(), torch.from_numpy(w.types).cuda())
    nd = min(512, len(dirs))
    for j, c in enumerate(_hist_points(w, cfg)):
        d0 = (j * 4999) % (len(dirs) - nd + 1)
        out = torch.full((nd, w.B), -1, dtype=torch.int32, device="cuda")
        plan.apx_debug_histograms(c, d0, nd, out)
        torch.cuda.synchronize()
        ref, n = O.histograms(w.xyz, w.types, c, dirs, w.R, w.B, accepted=accepted, d0=d0, nd=nd)
        got = out.cpu().numpy().astype(np.uint32)
        assert (got.sum(1) == n).all(), f"cfg {cfg} point {j}: histogram totals differ from N_c = {n}"
        assert (got == ref).all(), f"cfg {cfg} point {j}: {np.argwhere(got != ref)[:4]}"
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


def _full_launch(w, dirs, accepted=None, expect_paired=None):
    """The whole config in ONE apx_run (the launch configuration bench.py times); results stay on the device."""
    import torch
    dev = torch.device("cuda:0")
    plan = apx.Plan(w.R, w.B, dirs, k_lo=w.window[0], k_hi=w.window[1], accepted_types=accepted, device=0)
    assert plan.apx_plan_path() == 1
    if expect_paired is not None:
        assert plan.apx_plan_paired() == expect_paired            # half-grid mode is what runs on the geodesic grid
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
    cnt = counts.cpu().numpy().astype(np.uint32)
    # ROI ion counts against the oracle's brute force (one direction is enough for counts): every material point, or
    # -- where N x M makes that take the oracle an hour -- a seeded sample of 2048
    cidx = np.arange(len(cnt)) if count_all else np.sort(np.random.default_rng(len(cnt)).choice(len(cnt), 2048, replace=False))
    _, rc_all = O.signatures(w.xyz, w.types, w.centres[cidx], dirs[:1], w.R, w.B, k_lo=w.window[0], k_hi=w.window[1],
                             accepted=accepted)
    assert (cnt[cidx] == rc_all).all()
    # properties that hold for every output: 0 <= A <= N_c (P4), k inside the window, nothing left unwritten
    ok = torch.ones((), dtype=torch.bool, device=sig.device)
    for m0 in range(0, sig.shape[0], 8192):                                  # in slabs: no 57 GB temporaries
        blk, cb = sig[m0:m0 + 8192], counts[m0:m0 + 8192].to(torch.float32)[:, None]
        amp, k = blk[..., 0], blk[..., 1]
        ok &= (amp >= 0).all() & (amp <= cb * (1 + 1e-5) + 1e-3).all() & (k >= w.window[0]).all() & (k <= w.window[1]).all()
    assert bool(ok)
    # sampled material points x all directions, element by element
    idx = np.unique(np.asarray(idx))
    got = sig[torch.from_numpy(idx).cuda()].cpu().numpy()
    ref, rc, rwin = O.signatures(w.xyz, w.types, w.centres[idx], dirs, w.R, w.B, k_lo=w.window[0], k_hi=w.window[1],
                                 accepted=accepted, want_window=True)
    assert_parity(got, cnt[idx], ref, rc, rwin, w.window[0])


def _sample64(M, seed, extra=()):
    """64 seeded material points (SURVEY 8(c) parity protocol): the given special points plus random ones."""
    rng = np.random.default_rng(seed)
    extra = [int(e) for e in extra]
    return np.unique(np.concatenate([extra, rng.choice(M, 64 - len(extra), replace=False)]).astype(np.int64))


def test_cfg2_full_size_bench_launch():
    w = _config(2)
    dirs = O.dirs_fibonacci(w.D)
    sig, counts = _full_launch(w, dirs, expect_paired=0)
    _check_full(w, dirs, sig, counts, np.array([0, 99, 137, 455, 500, 555, 900, 999]))


@pytest.mark.parametrize("mask", [{0}, {1}], ids=["Al", "W"])
def test_cfg3_full_size_per_phase_filter(mask):
    """Config 3 at full size (27 000 material points x 40 962 geodesic directions, 8.85 GB of signatures), one run per
    phase filter; 64 sampled points include the box corners / faces and both grid planes next to the phase plane."""
    w = _config(3)
    dirs = O.dirs_geodesic(6)
    sig, counts = _full_launch(w, dirs, accepted=mask, expect_paired=1)
    g = np.arange(27000).reshape(30, 30, 30)
    special = [g[14, 10, 10], g[15, 10, 10], g[14, 0, 29], g[15, 29, 0], g[0, 0, 0], g[29, 29, 29], g[29, 15, 3],
               g[3, 20, 20], g[7, 7, 29], g[13, 13, 13], g[16, 16, 16]]
    _check_full(w, dirs, sig, counts, _sample64(27000, 3, special), accepted=mask)


def test_cfg4_full_size():
    """Config 4 at full size (175 616 material points x 40 962 directions, 57.5 GB of signatures, half-grid mode):
    properties on every output, ROI counts of 2048 sampled material points against the oracle's brute force, 64 sampled
    material points x all directions element by element (box corners / faces and the points nearest to grain
    boundaries -- smallest gap between the two nearest Voronoi seeds -- included)."""
    w = _config(4)
    dirs = O.dirs_geodesic(6)
    sig, counts = _full_launch(w, dirs, expect_paired=1)
    M = len(w.centres)
    seeds = w.meta["seeds"]
    dist = np.sort(np.linalg.norm(w.centres[:, None, :].astype(np.float64) - seeds[None], axis=2), axis=1)
    gb = np.argsort(dist[:, 1] - dist[:, 0])[:12]                           # on grain boundaries
    g = np.arange(M).reshape(56, 56, 56)
    special = [0, M - 1, g[0, 28, 28], g[55, 0, 31], g[28, 55, 55], *gb]
    _check_full(w, dirs, sig, counts, _sample64(M, 4, special), count_all=False)


def test_cfg5_full_size_al_filter():
    """Config 5 at full size (64 000 x 40 962, B = 2048, Al filter) on the tensor-core kernel in half-grid mode."""
    w = _config(5)
    dirs = O.dirs_geodesic(6)
    sig, counts = _full_launch(w, dirs, accepted={0}, expect_paired=1)
    M = len(w.centres)
    g = np.arange(M).reshape(40, 40, 40)
    special = [0, M - 1, g[0, 20, 20], g[39, 0, 17], g[20, 39, 39], g[20, 20, 20]]
    _check_full(w, dirs, sig, counts, _sample64(M, 5, special), accepted={0}, count_all=False)
