"""GPU parity of the signature epilogues: several signatures (type masks x spectral windows) from one
ingest and one launch, normalised intensity A / N_c, local-maximum peak mode.  Every plane of a multi-signature plan must
equal the ORACLE's separate single-signature run."""
from types import SimpleNamespace

import numpy as np
import pytest

import paper_2009_00735_b200 as apx
from oracle import oracle as O
from oracle import next_oracle as X
from workloads.lattices import fcc_basis, bcc_basis, lattice_in_box, random_rotation
from _parity import assert_parity

pytestmark = pytest.mark.gpu
PATHS = [pytest.param(apx.APX_FLAG_FORCE_FFT, id="fft"), pytest.param(0, id="auto")]


def _rng(seed):
    return np.random.Generator(np.random.PCG64(seed))


def _bicrystal(L=9.0, seed=31, sigma=0.05, eta=0.6):
    """Small stand-in for config 3: fcc Al | bcc W split at x = L/2, types = phase with 10 % relabelled, plus type 2 ions."""
    rng = _rng(seed)
    a = lattice_in_box(0.405, fcc_basis, random_rotation(rng), (0, 0, 0), (L / 2, L, L))
    b = lattice_in_box(0.3165, bcc_basis, random_rotation(rng), (L / 2, 0, 0), (L, L, L))
    xyz = np.concatenate([a, b])
    types = np.concatenate([np.zeros(len(a), np.uint8), np.ones(len(b), np.uint8)])
    keep = rng.random(len(xyz)) < eta
    xyz, types = xyz[keep], types[keep]
    xyz = xyz + rng.standard_normal(xyz.shape) * sigma
    relabel = rng.random(len(types)) < 0.10
    types = np.where(relabel, rng.integers(0, 3, len(types)), types).astype(np.uint8)
    perm = rng.permutation(len(xyz))
    return np.ascontiguousarray(xyz[perm].astype(np.float32)), np.ascontiguousarray(types[perm])


def _run_multi(xyz, types, centres, dirs, R, B, specs, flags, host=False):
    import torch
    dev = torch.device("cuda:0")
    plan = apx.Plan(R, B, dirs, device=0, flags=flags, specs=specs)
    assert plan.apx_plan_num_signatures() == len(specs)
    M, S = len(centres), len(specs)
    if host:
        sig = np.full((S, M, len(dirs), 2), -7.0, np.float32)
        cnt = np.full((S, M), -1, np.int32)
        plan.apx_run_host(xyz, types, centres, sig, cnt)
    else:
        sig_d = torch.full((S, M, len(dirs), 2), -7.0, dtype=torch.float32, device=dev)
        cnt_d = torch.full((S, M), -1, dtype=torch.int32, device=dev)
        plan.apx_run(torch.from_numpy(xyz).to(dev), None if types is None else torch.from_numpy(types).to(dev),
                     torch.from_numpy(centres).to(dev), sig_d, cnt_d)
        torch.cuda.synchronize()
        sig, cnt = sig_d.cpu().numpy(), cnt_d.cpu().numpy()
    info = (plan.apx_plan_path(), plan.apx_plan_paired())
    plan.apx_plan_destroy()
    return sig, cnt.astype(np.uint32), info


def _check_planes(xyz, types, centres, dirs, R, B, specs, sig, cnt):
    for s, sp in enumerate(specs):
        ref, rc, win = O.signatures(xyz, types, centres, dirs, R, B, k_lo=sp["k_lo"], k_hi=sp["k_hi"],
                                    accepted=sp.get("accepted_types"), want_window=True)
        got = sig[s].copy()
        if sp.get("normalise"):
            nrm = X.normalised(ref[..., 0], rc)                                 # oracle's A / N_c
            assert np.allclose(got[..., 0], nrm, rtol=1e-4, atol=1e-6), f"spec {s}: normalised intensity"
            got[..., 0] = got[..., 0] * rc[:, None]                             # back to raw for the peak-bin comparison
        assert_parity(got, cnt[s], ref, rc, win, sp["k_lo"])


@pytest.mark.parametrize("flags", PATHS)
def test_two_phase_filters_one_launch(flags):
    """Config 3's "ion-type filter run per phase" as ONE plan: planes {0} and {1} (two classes = two gathers inside one
    launch, one ingest), on the symmetric geodesic grid (half-grid mode on the tensor path)."""
    xyz, types = _bicrystal()
    dirs = O.dirs_geodesic(3)
    rng = _rng(2)
    centres = np.concatenate([[[4.4, 4.5, 4.5], [4.6, 4.5, 4.5], [0.3, 0.3, 0.3]], rng.uniform(1.5, 7.5, (9, 3))]).astype(np.float32)
    specs = [dict(accepted_types={0}, k_lo=15, k_hi=34), dict(accepted_types={1}, k_lo=15, k_hi=34)]
    sig, cnt, (path, paired) = _run_multi(xyz, types, centres, dirs, 2.0, 1024, specs, flags)
    if flags == 0:
        assert path == 1 and paired == 1
    _check_planes(xyz, types, centres, dirs, 2.0, 1024, specs, sig, cnt)
    assert (cnt[0] != cnt[1]).any()


@pytest.mark.parametrize("flags", PATHS)
def test_three_plane_families_from_one_binning(flags):
    """L208: signatures for {002}, {220} and {111} of Al from ONE gather and ONE binning pass (same type mask = one class):
    sub-windows of the union window [16, 31] (+-10 % around k = 2(R+dR)/d, L416), one of them normalised; a fourth spec with
    another mask rides along as a second class."""
    xyz, types = _bicrystal(seed=37)
    dirs = O.dirs_fibonacci(700)
    centres = _rng(5).uniform(1.0, 4.0, (6, 3)).astype(np.float32)
    specs = [dict(accepted_types={0}, k_lo=18, k_hi=22), dict(accepted_types={0}, k_lo=26, k_hi=31, normalise=True),
             dict(accepted_types={0}, k_lo=16, k_hi=19), dict(accepted_types={0, 2}, k_lo=17, k_hi=30)]
    sig, cnt, (path, _) = _run_multi(xyz, types, centres, dirs, 2.0, 1024, specs, flags)
    if flags == 0:
        assert path == 1
    _check_planes(xyz, types, centres, dirs, 2.0, 1024, specs, sig, cnt)
    assert (cnt[0] == cnt[1]).all() and (cnt[0] == cnt[2]).all() and (cnt[3] >= cnt[0]).all()


def test_multi_plane_b2048_and_host_entry():
    """B = 2048 (single-buffered tensor path) with two classes, through apx_run_host (plane-wise copies out of the slab ring),
    and without a type array (no type information: every class accepts every ion)."""
    xyz, types = _bicrystal(L=8.0, seed=41)
    dirs = O.dirs_geodesic(3)
    centres = _rng(6).uniform(2.5, 5.5, (200, 3)).astype(np.float32)            # > 128 points: four slabs
    specs = [dict(accepted_types={0}, k_lo=23, k_hi=51), dict(accepted_types={1, 2}, k_lo=30, k_hi=45, normalise=True)]
    sig, cnt, (path, paired) = _run_multi(xyz, types, centres, dirs, 2.4, 2048, specs, 0, host=True)
    assert path == 1 and paired == 1
    idx = np.array([0, 49, 50, 99, 100, 150, 199])
    _check_planes(xyz, types, centres[idx], dirs, 2.4, 2048, specs, sig[:, idx], cnt[:, idx])
    sig2, cnt2, _ = _run_multi(xyz, None, centres[:8], dirs, 2.4, 2048, specs, 0)
    specs_all = [dict(s, accepted_types=None) for s in specs]
    _check_planes(xyz, None, centres[:8], dirs, 2.4, 2048, specs_all, sig2, cnt2)


def test_single_signature_flags_normalise():
    import torch
    xyz, types = _bicrystal(seed=43)
    dirs = O.dirs_fibonacci(300)
    centres = _rng(7).uniform(1.0, 8.0, (5, 3)).astype(np.float32)
    centres[4] = (50, 50, 50)                                                   # empty ROI: intensity 0, bin k_lo
    dev = torch.device("cuda:0")
    for flags in (apx.APX_FLAG_NORMALISE, apx.APX_FLAG_NORMALISE | apx.APX_FLAG_FORCE_FFT):
        plan = apx.Plan(2.0, 1024, dirs, k_lo=15, k_hi=34, accepted_types={0}, device=0, flags=flags)
        sig = torch.empty((5, 300, 2), dtype=torch.float32, device=dev)
        cnt = torch.empty(5, dtype=torch.int32, device=dev)
        plan.apx_run(torch.from_numpy(xyz).to(dev), torch.from_numpy(types).to(dev), torch.from_numpy(centres).to(dev), sig, cnt)
        torch.cuda.synchronize()
        _check_planes(xyz, types, centres, dirs, 2.0, 1024, [dict(accepted_types={0}, k_lo=15, k_hi=34, normalise=True)],
                      sig.cpu().numpy()[None], cnt.cpu().numpy().astype(np.uint32)[None])
        assert (sig[4, :, 0] == 0).all() and (sig[4, :, 1] == 15).all()
        plan.apx_plan_destroy()


def _check_local_max(got, win, k_first, k_lo, k_hi, B, nc):
    """Comparator for the local-maximum mode (reading #20).  The oracle decides in fp64, the kernel in fp32, so a bin whose
    neighbour is within 1e-4 relative may flip: the kernel's bin must be a local maximum of the ORACLE's spectrum up to that
    margin, at least as high as every local maximum the oracle finds robustly, with the oracle's amplitude at that bin."""
    eps = 1e-4
    nbad = 0
    for m in range(got.shape[0]):
        for d in range(got.shape[1]):
            A = win[m, d]
            a_ref, k_ref = X.local_max_peak(A, k_first, k_lo, k_hi, B)
            a, k = float(got[m, d, 0]), int(got[m, d, 1])
            tol = eps * max(a_ref, a) + 1e-6 * nc[m]
            if k == k_ref and abs(a - a_ref) <= tol:
                continue
            nbad += 1

            def amp(kk):
                kk = B - kk if kk > B // 2 else abs(kk)
                return A[kk - k_first]
            robust = [amp(kk) for kk in range(k_lo, k_hi + 1)
                      if amp(kk) > amp(kk - 1) * (1 + eps) + tol and amp(kk) > amp(kk + 1) * (1 + eps) + tol]
            if a == 0.0 and k == k_lo:                                          # the kernel found no local maximum
                assert not robust, (m, d, got[m, d], a_ref, k_ref)
                continue
            assert k_lo <= k <= k_hi and abs(a - amp(k)) <= tol, (m, d, got[m, d], amp(k))
            assert amp(k) >= amp(k - 1) * (1 - eps) - tol and amp(k) >= amp(k + 1) * (1 - eps) - tol, (m, d, got[m, d])
            assert not robust or a >= max(robust) * (1 - eps) - tol, (m, d, got[m, d], max(robust))
    return nbad


@pytest.mark.parametrize("window", [(1, 40), (15, 34), (100, 128)])
def test_local_maximum_mode(window):
    """APX_PEAK_LOCAL_MAX on the general kernel against the oracle's definition applied to the oracle's spectrum; wide
    window from k = 1 (DC as left neighbour, the ROI envelope must not be picked) and one that ends at Nyquist."""
    import torch
    B, R = 256, 2.0
    xyz, types = _bicrystal(seed=47, sigma=0.07)
    dirs = O.dirs_fibonacci(400)
    centres = np.concatenate([_rng(8).uniform(1.0, 4.0, (5, 3)), [[60, 60, 60]]]).astype(np.float32)
    k_lo, k_hi = window
    specs = [dict(accepted_types={0}, k_lo=k_lo, k_hi=k_hi, peak_mode=apx.APX_PEAK_LOCAL_MAX),
             dict(accepted_types={0}, k_lo=k_lo, k_hi=k_hi)]
    sig, cnt, (path, _) = _run_multi(xyz, types, centres, dirs, R, B, specs, 0)
    assert path == 0                                                            # local-maximum mode: general kernel
    kf, kl = max(k_lo - 1, 0), min(k_hi + 1, B // 2)
    ref, rc, win = O.signatures(xyz, types, centres, dirs, R, B, k_lo=kf, k_hi=kl, accepted={0}, want_window=True)
    assert (cnt[0] == rc).all()
    nbad = _check_local_max(sig[0], win, kf, k_lo, k_hi, B, rc.astype(np.float64))
    assert nbad < 0.01 * sig[0].shape[0] * sig[0].shape[1]
    assert (sig[0][5, :, 0] == 0).all() and (sig[0][5, :, 1] == k_lo).all()     # empty ROI
    _check_planes(xyz, types, centres, dirs, R, B, specs[1:], sig[1:], cnt[1:])
    if k_lo == 1:                                                               # the plain maximum sits on the envelope, the local one does not
        assert (sig[1][:5, :, 1] == 1).mean() > 0.5 and (sig[0][:5, :, 1] == 1).mean() < 0.2


def test_local_max_needs_the_general_kernel():
    dirs = O.dirs_fibonacci(64)
    with pytest.raises(apx.ApxError) as ei:
        apx.Plan(2.0, 1024, dirs, k_lo=15, k_hi=34, device=0, flags=apx.APX_FLAG_LOCAL_MAX | apx.APX_FLAG_FORCE_MMA)
    assert ei.value.status == apx.APX_EINVAL
    plan = apx.Plan(2.0, 1024, dirs, k_lo=15, k_hi=34, device=0, flags=apx.APX_FLAG_LOCAL_MAX)
    assert plan.apx_plan_path() == 0
    plan.apx_plan_destroy()
    with pytest.raises(apx.ApxError):
        apx.Plan(2.0, 1024, dirs, device=0, specs=[dict(k_lo=15, k_hi=34)] * 5)      # more than APX_MAX_SIGNATURES
