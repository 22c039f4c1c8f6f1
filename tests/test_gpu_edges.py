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
    B = 1024 (1152 ions), so on the auto path these ROIs spill into the second histogram buffer, run single-buffered
    and are binned in two passes of <= 2048 ions."""
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


@pytest.mark.parametrize("off", [0, 1, 2, 3])
def test_ingest_with_unaligned_inputs_and_ragged_tails(off):
    """Ingest reads four ions per thread with 16-byte loads when the caller's arrays allow it: views that start 12 * off bytes
    (coordinates) and off bytes (types) into an allocation, with ion counts of every residue mod 4, must give the same result
    through the scalar loads; an ion-type filter and a few non-finite ions ride along."""
    import torch
    dev = torch.device("cuda:0")
    rng = np.random.Generator(np.random.PCG64(3 + off))
    xyz, _ = _ball(2.6, eta=0.6, sigma=0.03)
    xyz = np.ascontiguousarray(xyz[: len(xyz) - off].astype(np.float32))
    types = (rng.random(len(xyz)) < 0.3).astype(np.uint8)
    xyz[5] = (np.nan, 0, 0); xyz[11] = (0, np.inf, 0)
    dirs = O.dirs_fibonacci(40)
    centres = np.array([[0, 0, 0], [1.0, -0.5, 0.3]], np.float32)
    xt = torch.from_numpy(xyz).to(dev); tt = torch.from_numpy(types).to(dev)
    plan = apx.Plan(1.5, 256, dirs, k_lo=7, k_hi=17, accepted_types={0}, device=0)
    xv, tv = xt[off:], tt[off:]                                   # contiguous views, data pointers moved by 12 * off / off bytes
    assert xv.data_ptr() % 16 == (12 * off) % 16 and xv.is_contiguous()
    sig = torch.full((2, len(dirs), 2), -7.0, dtype=torch.float32, device=dev)
    cnt = torch.full((2,), -1, dtype=torch.int32, device=dev)
    plan.apx_run(xv, tv, torch.from_numpy(centres).to(dev), sig, cnt)
    torch.cuda.synchronize()
    plan.apx_plan_destroy()
    with np.errstate(invalid="ignore"):
        ref, rc, win = O.signatures(xyz[off:], types[off:], centres, dirs, 1.5, 256, k_lo=7, k_hi=17, accepted={0}, want_window=True)
    assert_parity(sig.cpu().numpy(), cnt.cpu().numpy().astype(np.uint32), ref, rc, win, 7)
    assert rc[0] > 300


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


def test_run_host_against_oracle_and_device_path():
    """apx_run_host (host pointers, ring of two staging slabs, pipelined copies): every output element against the
    ORACLE, and bit for bit what apx_run leaves on the device."""
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
    sig_h = torch.full((301, 96, 2), -7.0, dtype=torch.float32).pin_memory()
    cnt_h = torch.full((301,), -1, dtype=torch.int32).pin_memory()
    plan.apx_run_host(torch.from_numpy(xyz), torch.from_numpy(types), torch.from_numpy(centres), sig_h, cnt_h)
    assert torch.equal(sig_h, sig_d.cpu()) and torch.equal(cnt_h, cnt_d.cpu())
    ref, rc, win = O.signatures(xyz, types, centres, dirs, 1.0, 256, k_lo=7, k_hi=17, want_window=True)
    assert_parity(sig_h.numpy(), cnt_h.numpy().astype(np.uint32), ref, rc, win, 7)
    # pageable numpy buffers, no counts, no types: same numbers
    sig_n = np.full((301, 96, 2), -7.0, np.float32)
    plan.apx_run_host(xyz, None, centres, sig_n, None)
    assert np.array_equal(sig_n, sig_h.numpy())
    plan.apx_plan_destroy()


def test_run_host_ring_reuses_two_slabs():
    """More slabs than staging buffers: D = 40 962 directions make a material point 328 KB, so 20 000 points are 6.5 GB of
    signatures = 7 slabs of <= 1 GiB through the two device staging buffers; sampled against the oracle."""
    import torch
    xyz, types = _ball(3.2, eta=0.3, sigma=0.05, seed=23)
    rng = np.random.default_rng(9)
    M = 20000
    centres = ((rng.random((M, 3)) - 0.5) * 3.0).astype(np.float32)
    dirs = O.dirs_geodesic(6)
    plan = apx.Plan(1.0, 256, dirs, k_lo=7, k_hi=17, device=0)
    sig_h = torch.full((M, len(dirs), 2), -7.0, dtype=torch.float32)
    cnt_h = torch.full((M,), -1, dtype=torch.int32)
    free0 = torch.cuda.mem_get_info()[0]
    plan.apx_run_host(xyz, types, centres, sig_h.numpy(), cnt_h.numpy())
    assert free0 - torch.cuda.mem_get_info()[0] < (3 << 30)              # two 1 GiB slabs, not 6.5 GB, live on the device
    idx = np.array([0, 3276, 3277, 6553, 9999, 13107, 16383, 19660, M - 1])       # around the slab seams
    ref, rc, win = O.signatures(xyz, types, centres[idx], dirs, 1.0, 256, k_lo=7, k_hi=17, want_window=True)
    assert_parity(sig_h.numpy()[idx], cnt_h.numpy().astype(np.uint32)[idx], ref, rc, win, 7)
    assert bool((sig_h[..., 1] >= 7).all())                               # nothing left unwritten
    plan.apx_plan_destroy()


def _hist_check(plan, w, dirs, centre, d0, nd, accepted=None, pad=1):
    import torch
    out = torch.full((nd, w.B), -1, dtype=torch.int32, device="cuda")
    plan.apx_debug_histograms(centre, d0, nd, out)
    torch.cuda.synchronize()
    ref, n = O.histograms(w.xyz, w.types, np.asarray(centre, np.float32), dirs, w.R, w.B, pad=pad, accepted=accepted, d0=d0, nd=nd)
    got = out.cpu().numpy().astype(np.uint32)
    assert (got == ref).all(), np.argwhere(got != ref)[:4]
    return n


@pytest.mark.parametrize("flags", PATHS)
def test_histograms_bit_exact_multipass_spill_deferred(flags):
    """The production kernels' histograms (export of apx_debug_histograms) against the oracle on the ROI sizes that take
    the special routes: B = 256 two-pass (> 2048 ions, partial counts added), B = 1024 spilled into the second buffer
    (1152 < n), B = 1024 beyond 8192 ions (deferred to the FFT kernel / streaming), B = 2048 two-pass single-buffered."""
    import torch
    xyz, types = _ball(4.0)
    X, T = torch.from_numpy(xyz).cuda(), torch.from_numpy(types).cuda()
    for R, B, window, lo in ((2.2, 256, window_for(2.2, 256), 2049), (2.2, 1024, window_for(2.2, 1024), 2049),
                             (3.3, 1024, (20, 39), 8193), (2.2, 2048, (23, 51), 2049)):
        dirs = O.dirs_fibonacci(200)
        w = _case(xyz, types, R, B)
        plan = apx.Plan(R, B, dirs, k_lo=window[0], k_hi=window[1], device=0, flags=flags)
        plan.apx_ingest(X, T)
        for c in ((0.0, 0.0, 0.0), (0.3, -0.2, 0.1)):
            n = _hist_check(plan, w, dirs, c, 3, 197)
            assert n >= lo
        plan.apx_plan_destroy()


@pytest.mark.parametrize("flags", PATHS)
def test_histograms_bit_exact_pad0_clamp(flags):
    xyz, types = _ball(1.6, eta=0.7, sigma=0.03, seed=13)
    dirs = (O.dirs_fibonacci(64).astype(np.float64) * 1.03).astype(np.float32)
    import torch
    for B in (512, 2048):
        w = _case(xyz, types, 1.2, B)
        plan = apx.Plan(1.2, B, dirs, pad=0, k_lo=5, k_hi=20, device=0, flags=flags)
        plan.apx_ingest(torch.from_numpy(xyz).cuda(), torch.from_numpy(types).cuda())
        _hist_check(plan, w, dirs, (0.0, 0.0, 0.0), 0, 64, pad=0)
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
    # bit-exact histograms of every direction: mirrored ones (reversed), flagged pairs (binned again on their own in the
    # fix-up groups) and, with an ion on the centre, the fix-list overflow that sends the point to the FFT kernel
    import torch
    plan.apx_ingest(torch.from_numpy(w.xyz).cuda(), torch.from_numpy(w.types).cuda())
    for c in centres:
        _hist_check(plan, w, dirs, c, 0, len(dirs))
    plan.apx_plan_destroy()
    _check(w, dirs, centres, (15, 34), flags)


@pytest.mark.parametrize("B", [1024, 4096])
@pytest.mark.parametrize("centre_ions", [False, True], ids=["some_flagged", "all_flagged"])
@pytest.mark.parametrize("flags", [pytest.param(apx.APX_FLAG_FORCE_FFT, id="half"),
                                   pytest.param(apx.APX_FLAG_FORCE_FFT | apx.APX_FLAG_NO_PAIRING, id="full")])
def test_general_kernel_half_grid_mode_with_exact_integer_projections(flags, centre_ions, B):
    """The same construction as above for the general (FFT) kernel, which has a half-grid mode of its own: one member of
    every pair (n, -n) is binned and transformed, the peak is written to both, pairs that met an exact-integer projection
    are flagged and their -n members are binned on their own in fix-up groups.  With an ion exactly on each centre EVERY
    pair is flagged (all of -n goes through fix-up groups); B = 4096 runs 8 directions per group.  A second pass with a
    wide window and the local-maximum peak mode covers the other epilogue."""
    rng = np.random.Generator(np.random.PCG64(12))
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
    dirs = apx.apx_dirs_geodesic(2 if B == 4096 else 3)
    centres = np.array([[0, 0, 0], c2], np.float32)
    w = _case(xyz, np.zeros(len(xyz), np.uint8), R, B)
    plan = apx.Plan(R, B, dirs, k_lo=15, k_hi=34, device=0, flags=flags)
    assert plan.apx_plan_path() == 0 and plan.apx_plan_paired() == (0 if flags & apx.APX_FLAG_NO_PAIRING else 1)
    # the histogram export runs the same kernel with the pairing switched off: every direction's own counters
    import torch
    plan.apx_ingest(torch.from_numpy(w.xyz).cuda(), torch.from_numpy(w.types).cuda())
    _hist_check(plan, w, dirs, centres[1], 0, min(len(dirs), 64))
    plan.apx_plan_destroy()
    _check(w, dirs, centres, (15, 34), flags)
    _check(w, dirs, centres, (1, B // 2), flags)


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


def test_single_pass_roi_with_a_counter_beyond_2048_is_caught_by_the_dc_column():
    """With a spare accumulator column (N > 4 W) the tensor-core kernel bins a ROI of more than 2048 ions in ONE pass and checks
    afterwards, through a "k = 0" twiddle column, that the counters the tensor core read sum to N_c -- they do unless some
    counter exceeded 2048, where a u16 bit pattern stops being the fp16 number of the same value.  Here 2600 ions sit within
    1e-4 nm of one point, so for almost every direction one bin holds more than 2048 of them: the material point must come
    out right all the same (it is handed to the general kernel).  The second centre is an ordinary two-pass-sized ROI that
    stays on the single-pass route."""
    rng = np.random.Generator(np.random.PCG64(5))
    xyz, types = _ball(3.0)
    blob = (np.array([0.31, -0.12, 0.2]) + rng.uniform(-1e-4, 1e-4, (2600, 3))).astype(np.float32)
    far = xyz[np.linalg.norm(xyz - np.array([0.31, -0.12, 0.2]), axis=1) > 1.2]      # thin the lattice around the blob
    xyz = np.ascontiguousarray(np.concatenate([far, blob]).astype(np.float32))
    rng.shuffle(xyz)
    types = np.zeros(len(xyz), np.uint8)
    for B, window, dirs in ((256, (12, 40), O.dirs_fibonacci(96)), (2048, (23, 51), apx.apx_dirs_geodesic(2))):
        w = _case(xyz, types, 2.2, B)
        centres = np.array([[0, 0, 0], [-0.6, 0.3, -0.2]], np.float32)
        plan = apx.Plan(2.2, B, dirs, k_lo=window[0], k_hi=window[1], device=0)
        assert plan.apx_plan_path() == 1
        plan.apx_plan_destroy()
        path, cnt = _check(w, dirs, centres, window, 0)
        assert path == 1 and cnt.min() > 2600


def test_large_roi_deferred_from_tensor_path_b1024():
    """B = 1024 on the auto path: more than 8192 ions exceed even the spill mode of the tensor-core kernel, the material
    point goes to the deferred list and the general kernel (streaming its cell rows) serves it in the same stream."""
    xyz, types = _ball(4.0)
    dirs = O.dirs_fibonacci(64)
    centres = np.array([[0, 0, 0], [3.9, 0, 0]], np.float32)             # the second one is a partial ROI on the tensor path
    w = _case(xyz, types, 3.3, 1024)
    path, cnt = _check(w, dirs, centres, (20, 39), 0)
    assert path == 1 and cnt[0] > 8192 and cnt[1] < 8192


def test_multipass_roi_run_to_run():
    """A ROI with more than 2048 ions is binned in passes of 2048 whose partial spectra accumulate in fp32 (TMEM).  Which
    ions fall into which pass depends on the order the counting sort's atomics and the gather's warp appends happen to
    take, so the last bits of the amplitude may differ from run to run.  Bound it: counts and peak
    bins identical (up to oracle-level ties), amplitudes within 4 fp32 ulps of N_c; single-pass ROIs are bit-identical."""
    import torch
    xyz, types = _ball(3.0)
    dirs = O.dirs_fibonacci(512)
    dev = torch.device("cuda:0")
    centres = torch.tensor([[0.0, 0.0, 0.0], [0.3, -0.2, 0.1], [2.6, 0.0, 0.0]], dtype=torch.float32, device=dev)
    plan = apx.Plan(2.2, 256, dirs, k_lo=12, k_hi=40, device=0)
    runs = []
    for _ in range(3):
        sig = torch.empty((3, 512, 2), dtype=torch.float32, device=dev)
        cnt = torch.empty(3, dtype=torch.int32, device=dev)
        plan.apx_run(torch.from_numpy(xyz).to(dev), torch.from_numpy(types).to(dev), centres, sig, cnt)
        torch.cuda.synchronize()
        runs.append((sig.cpu().numpy(), cnt.cpu().numpy()))
    n = runs[0][1].astype(np.float64)
    assert n[0] > 2048 and n[2] <= 2048
    for s, c in runs[1:]:
        assert (c == runs[0][1]).all()
        assert np.array_equal(s[2], runs[0][0][2])                              # single pass: bit-identical
        assert (np.abs(s[..., 0] - runs[0][0][..., 0]) <= 4 * 2.0 ** -23 * n[:, None]).all()
        assert (s[..., 1] == runs[0][0][..., 1]).mean() > 0.999
    plan.apx_plan_destroy()


def test_binding_rejects_wrong_dtype_shape_device():
    """The Python binding checks dtype, shape, contiguity and placement of every array before a raw pointer crosses the ABI."""
    import torch
    dev = torch.device("cuda:0")
    dirs = O.dirs_fibonacci(32)
    plan = apx.Plan(1.0, 256, dirs, k_lo=7, k_hi=17, device=0)
    xyz = torch.zeros((10, 3), dtype=torch.float32, device=dev)
    types = torch.zeros(10, dtype=torch.uint8, device=dev)
    centres = torch.zeros((2, 3), dtype=torch.float32, device=dev)
    sig = torch.zeros((2, 32, 2), dtype=torch.float32, device=dev)
    bad = [
        lambda: plan.apx_ingest(xyz.double(), types),                           # float64 coordinates
        lambda: plan.apx_ingest(xyz, types[:5]),                                # too few types
        lambda: plan.apx_ingest(xyz.cpu(), types),                              # host tensor where a device tensor is due
        lambda: plan.apx_ingest(xyz.t().contiguous().t(), types),               # not contiguous
        lambda: plan.apx_run(xyz, types, centres, sig[:1]),                     # signature buffer too small
        lambda: plan.apx_run(xyz, types, centres, sig, torch.zeros(1, dtype=torch.int32, device=dev)),   # counts too small
        lambda: plan.apx_run(xyz, types, centres, sig.half()),                  # wrong output dtype
        lambda: plan.apx_run_host(xyz, types, centres, sig),                    # device tensors into the host entry
    ]
    for f in bad:
        with pytest.raises(apx.ApxError) as ei:
            f()
        assert ei.value.status == apx.APX_EINVAL
    plan.apx_run(xyz, types, centres, sig)                                       # the well-formed call still works
    torch.cuda.synchronize()
    plan.apx_plan_destroy()


@pytest.mark.parametrize("flags", PATHS)
def test_half_grid_full_machine_runs_are_bitwise_repeatable(flags):
    """(Both kernels, each in its half-grid mode.)  Every SM busy with back-to-back groups (the regime where the warp-specialised pipeline of the tensor-core kernel runs
    furthest ahead of its epilogues): 1200 single-pass ROIs on the symmetric geodesic grid, five runs, bit-identical outputs
    (counts are integers and every ROI is binned in one pass, so nothing may differ), and a sample against the oracle."""
    import torch
    rng = np.random.Generator(np.random.PCG64(77))
    from workloads.lattices import lattice_in_box
    sites = lattice_in_box(A_AL, fcc_basis, random_rotation(rng), (0, 0, 0), (12, 12, 12))
    xyz, _, _, _ = jitter_thin_shuffle(sites, rng, 0.45, 0.05)
    types = np.zeros(len(xyz), np.uint8)
    dirs = apx.apx_dirs_geodesic(4)
    centres = rng.uniform(1.0, 11.0, (1200, 3)).astype(np.float32)
    dev = torch.device("cuda:0")
    plan = apx.Plan(2.0, 1024, dirs, k_lo=15, k_hi=34, device=0, flags=flags)
    assert plan.apx_plan_paired() == 1 and plan.apx_plan_path() == (0 if flags else 1)
    X, T, C_ = torch.from_numpy(xyz).to(dev), torch.from_numpy(types).to(dev), torch.from_numpy(centres).to(dev)
    ref_sig = None
    for _ in range(5):
        sig = torch.full((1200, len(dirs), 2), -7.0, dtype=torch.float32, device=dev)
        cnt = torch.full((1200,), -1, dtype=torch.int32, device=dev)
        plan.apx_run(X, T, C_, sig, cnt)
        torch.cuda.synchronize()
        if ref_sig is None:
            ref_sig, ref_cnt = sig, cnt
        else:
            assert torch.equal(sig, ref_sig) and torch.equal(cnt, ref_cnt)
    assert int(ref_cnt.max()) < 2048
    idx = np.array([0, 7, 599, 1199])
    ref, rc, win = O.signatures(xyz, types, centres[idx], dirs, 2.0, 1024, k_lo=15, k_hi=34, want_window=True)
    assert_parity(ref_sig[torch.from_numpy(idx).to(dev)].cpu().numpy(), ref_cnt.cpu().numpy().astype(np.uint32)[idx], ref, rc, win, 15)
    plan.apx_plan_destroy()
