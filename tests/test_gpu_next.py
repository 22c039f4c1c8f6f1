"""GPU parity of the steps after the signature computation (include/aptsig_ext.h)
against oracle/next_oracle.py, through the C ABI.  Run with -m gpu on a B200."""
import math

import numpy as np
import pytest

import paper_2009_00735_b200 as apx
from oracle import oracle as O
from oracle import next_oracle as X
from workloads.lattices import fcc_basis, lattice_in_ball, lattice_in_box, random_rotation

pytestmark = pytest.mark.gpu


def _rng(seed):
    return np.random.Generator(np.random.PCG64(seed))


def _k0(R, B, d):
    return round(2 * (R + R / (B // 2 - 1)) / d)


# ---- NEXT-4 ------------------------------------------------------------------------------------------------------
def _pole_cloud():
    """A 12^3 nm box: noiseless fcc Al (strong poles) for x < 6, the same lattice jittered by 0.12 nm (no signal) beyond."""
    rng = _rng(41)
    rot = random_rotation(rng)
    a = lattice_in_box(0.405, fcc_basis, rot, (0, 0, 0), (6, 12, 12))
    b = lattice_in_box(0.405, fcc_basis, rot, (6, 0, 0), (12, 12, 12))
    b = b + rng.standard_normal(b.shape) * 0.12
    xyz = np.concatenate([a, b])
    keep = rng.random(len(xyz)) < 0.6
    xyz = xyz[keep]
    rng.shuffle(xyz)
    return np.ascontiguousarray(xyz.astype(np.float32)), rot


def test_refinement_chain_against_oracle():
    import torch
    from paper_2009_00735_b200.refine import coarse_grid, adaptive_scan
    xyz, rot = _pole_cloud()
    types = np.zeros(len(xyz), np.uint8)
    R, B, spacing, split, kappa = 1.5, 256, 2.0, 5, 0.75
    k0 = _k0(R, B, 0.405 / 2)
    dirs = np.concatenate([rot.T.astype(np.float32), -rot.T.astype(np.float32), O.dirs_fibonacci(500)])   # the six <100> poles + a grid
    centres_np = coarse_grid((1, 1, 1), (11, 11, 11), spacing)                                           # 5^3 coarse cells
    assert centres_np.shape == (125, 3)
    dev = torch.device("cuda:0")
    plan = apx.Plan(R, B, dirs, k_lo=k0 - 2, k_hi=k0 + 2, device=0)
    out = adaptive_scan(plan, torch.from_numpy(xyz).to(dev), torch.from_numpy(types).to(dev), torch.from_numpy(centres_np).to(dev),
                        spacing, kappa=kappa, split=split)
    torch.cuda.synchronize()
    sig, cnt = out["sig"].cpu().numpy(), out["counts"].cpu().numpy().astype(np.uint32)
    kmax = out["kappa_max"].cpu().numpy()
    # intensities: the kernel's maximum against the oracle's, from the oracle's own signatures (amplitude tolerance 1e-4)
    osig, ocnt = O.signatures(xyz, types, centres_np, dirs, R, B, k_lo=k0 - 2, k_hi=k0 + 2)
    assert (cnt == ocnt).all()
    okmax = X.intensity_max(osig[..., 0], ocnt)
    assert np.allclose(kmax, okmax, rtol=1e-4, atol=1e-6)
    # ... and exactly (one fp32 division) from the signatures the kernel was given
    assert np.allclose(kmax, X.intensity_max(sig[..., 0], cnt), rtol=2e-7, atol=0)
    # selection: the decision is taken in the kernel's precision (fp32 kappa_max >= fp32 kappa) on both sides; ordered
    sel = out["selected"].cpu().numpy().astype(np.int64)
    assert list(sel) == list(X.refine_select(kmax, np.float32(kappa)))
    assert 0 < len(sel) < 125 and (centres_np[sel, 0] < 6.5).all()             # the crystal half is refined, the noise is not
    unsure = np.abs(okmax - kappa) < 1e-3                                        # oracle-level decision, away from the threshold
    assert set(np.nonzero((okmax >= kappa) & ~unsure)[0]) <= set(sel) <= set(np.nonzero((okmax >= kappa) | unsure)[0])
    # new centres: bit-exact
    fine = out["fine_centres"].cpu().numpy()
    assert np.array_equal(fine, X.refine_centres(centres_np, sel, spacing, split))
    # second pass: signatures of a sample of the refined ROIs against the oracle
    idx = np.sort(_rng(2).choice(len(fine), 40, replace=False))
    rsig, rcnt, rwin = O.signatures(xyz, types, fine[idx], dirs, R, B, k_lo=k0 - 2, k_hi=k0 + 2, want_window=True)
    from _parity import assert_parity
    assert_parity(out["fine_sig"].cpu().numpy()[idx], out["fine_counts"].cpu().numpy().astype(np.uint32)[idx], rsig, rcnt, rwin, k0 - 2)
    plan.apx_plan_destroy()


def test_refine_select_and_centres_edge_cases():
    import torch
    dev = torch.device("cuda:0")
    plan = apx.Plan(1.0, 256, O.dirs_fibonacci(8), k_lo=7, k_hi=17, device=0)
    rng = _rng(5)
    M = 5000                                                                     # several 1024-point tiles + a ragged tail
    kmax_np = rng.random(M).astype(np.float32)
    kmax_np[[0, 1023, 1024, 4999]] = 0.75                                        # threshold is inclusive, tile seams
    kmax = torch.from_numpy(kmax_np).to(dev)
    sel = torch.full((M,), -1, dtype=torch.int32, device=dev)
    n = torch.zeros(1, dtype=torch.int32, device=dev)
    plan.apx_refine_select(kmax, 0.75, sel, n)
    ref = X.refine_select(kmax_np, np.float32(0.75))
    assert int(n.item()) == len(ref) and np.array_equal(sel.cpu().numpy()[:len(ref)], ref)
    plan.apx_refine_select(kmax, 2.0, sel, n)                                    # nothing selected
    assert int(n.item()) == 0
    centres_np = (rng.random((M, 3)) * 50).astype(np.float32)
    centres = torch.from_numpy(centres_np).to(dev)
    plan.apx_refine_select(kmax, 0.75, sel, n)
    for split, spacing in ((1, 2.0), (2, 1.0), (5, 2.0), (3, 0.7)):
        cap = 100                                                                # fewer slots than selected points: the rest is dropped
        out = torch.full((cap * split ** 3, 3), -7.0, dtype=torch.float32, device=dev)
        plan.apx_refine_centres(centres, sel, n, cap, spacing, split, out)
        torch.cuda.synchronize()
        assert np.array_equal(out.cpu().numpy(), X.refine_centres(centres_np, ref[:cap], spacing, split))
    plan.apx_plan_destroy()


# ---- NEXT-1 ------------------------------------------------------------------------------------------------------
def _al_ball(R, rot=np.eye(3), sigma=0.0, eta=1.0, seed=1):
    rng = _rng(seed)
    p = lattice_in_ball(0.405, fcc_basis, rot, (0, 0, 0), R)
    p = p[rng.random(len(p)) < eta] if eta < 1 else p
    if sigma:
        p = p + rng.standard_normal(p.shape) * sigma
    return np.ascontiguousarray(p.astype(np.float32))


def test_indexer_preprocessing_against_oracle():
    """Strongest nodes bit-exact; look-up table equal to the oracle's brute-force nearest node (a different node only when the
    oracle's own dot products tie to 1e-12)."""
    dirs = O.dirs_geodesic(4)                                                    # 2562 nodes
    G = apx.apx_so3_grid_cubic(7.5)
    R, B = 1.5, 256
    k0 = _k0(R, B, 0.405 / 2)
    sig, cnt = O.signatures(_al_ball(R + 0.5), None, np.zeros((1, 3), np.float32), dirs, R, B, k_lo=k0 - 1, k_hi=k0 + 1)
    ref = X.normalised(sig[..., 0], cnt)[0].astype(np.float32)
    n_hat = 100
    ix = apx.Indexer(dirs, G, ref, n_hat, device=0)
    nodes, vals = ix.apx_indexer_nodes()
    onodes = X.strongest_nodes(ref, n_hat)
    assert np.array_equal(nodes, onodes) and np.array_equal(vals, ref[onodes])
    gs = np.arange(0, len(G), 11)
    lut = np.stack([ix.apx_indexer_lut(g, 1)[0] for g in gs])
    olut = X.lookup_table(dirs, G[gs].astype(np.float64), onodes)
    d64 = dirs.astype(np.float64)
    for gi, v in np.argwhere(lut != olut):
        r = X.quat_to_matrix(G[gs[gi]].astype(np.float64)) @ d64[onodes[v]]
        assert abs(d64[lut[gi, v]] @ r - d64[olut[gi, v]] @ r) < 1e-12
    assert (lut != olut).mean() < 1e-3
    whole = ix.apx_indexer_lut(0, len(G))                                         # block copy = row copies
    assert np.array_equal(whole[gs], lut)
    ix.apx_indexer_destroy()


@pytest.mark.parametrize("K", [1, 4, 8])
def test_index_eq3_against_oracle(K):
    """Eq. 3 on the device against the oracle's plain loops, from the SAME inputs (signatures of the hot path, counts):
    image differences within fp32 summation error, the K best orientations identical up to oracle-level ties; and the best
    orientation of a rotated, noisy crystal is the true one within the resolution of mesh and orientation grid."""
    import torch
    dev = torch.device("cuda:0")
    dirs = O.dirs_geodesic(4)
    G = apx.apx_so3_grid_cubic(7.5)
    R, B = 1.5, 256
    k0 = _k0(R, B, 0.405 / 2)
    sig, cnt = O.signatures(_al_ball(R + 0.5), None, np.zeros((1, 3), np.float32), dirs, R, B, k_lo=k0 - 1, k_hi=k0 + 1)
    ref = X.normalised(sig[..., 0], cnt)[0].astype(np.float32)
    n_hat = 100
    ix = apx.Indexer(dirs, G, ref, n_hat, device=0)
    # measured: a crystal rotated by grid orientation g_true, thinned and jittered, 37 material points around the origin
    g_true = 300
    rot = X.quat_to_matrix(G[g_true].astype(np.float64))
    xyz = _al_ball(3.2, rot=rot, sigma=0.03, eta=0.7, seed=9)
    centres = (_rng(3).uniform(-1.0, 1.0, (37, 3))).astype(np.float32)
    plan = apx.Plan(R, B, dirs, k_lo=k0 - 1, k_hi=k0 + 1, device=0)
    sig_d = torch.empty((37, len(dirs), 2), dtype=torch.float32, device=dev)
    cnt_d = torch.empty(37, dtype=torch.int32, device=dev)
    plan.apx_run(torch.from_numpy(xyz).to(dev), None, torch.from_numpy(centres).to(dev), sig_d, cnt_d)
    bd = torch.full((37, K), -1.0, dtype=torch.float32, device=dev)
    bg = torch.full((37, K), -5, dtype=torch.int32, device=dev)
    ix.apx_index(sig_d, cnt_d, bd, bg)
    torch.cuda.synchronize()
    bd, bg = bd.cpu().numpy(), bg.cpu().numpy()
    img = X.normalised(sig_d.cpu().numpy()[..., 0], cnt_d.cpu().numpy())          # oracle normalisation of the same signatures
    onodes = X.strongest_nodes(ref, n_hat)
    olut = X.lookup_table(dirs, G.astype(np.float64), onodes)
    hits = 0
    for m in (0, 5, 17, 36):
        delta = X.index_delta(img[m], olut, ref[onodes])
        od, og = X.best_solutions(delta, K)
        assert np.allclose(bd[m], od, rtol=2e-5, atol=1e-6)
        for s in range(K):                                                       # tie rule: the device's pick is as good as the oracle's
            assert bg[m, s] == og[s] or abs(delta[bg[m, s]] - od[s]) <= 2e-5 * od[s] + 1e-6
        assert (np.diff(bd[m]) >= 0).all() and len(set(bg[m])) == K
        hits += X.quat_disorientation_deg_cubic(G[bg[m, 0]].astype(np.float64), G[g_true].astype(np.float64)) <= 10.0
    assert hits >= 3
    plan.apx_plan_destroy()
    ix.apx_indexer_destroy()


def test_index_many_points_chunks_and_prenormalised_input():
    """More material points than one chunk (8192) and a ragged last block of 32; counts = NULL takes the image as it is."""
    import torch
    dev = torch.device("cuda:0")
    rng = _rng(12)
    dirs = O.dirs_geodesic(2)                                                    # 162 nodes
    G = apx.apx_so3_grid_cubic(15.0)
    ref = rng.random(len(dirs)).astype(np.float32)
    ix = apx.Indexer(dirs, G, ref, 19, device=0)                                 # n_hat not a multiple of 8: padded rows
    M = 8192 + 777
    img = rng.random((M, len(dirs))).astype(np.float32)
    sig = np.zeros((M, len(dirs), 2), np.float32)
    sig[..., 0] = img
    bd = torch.empty((M, 2), dtype=torch.float32, device=dev)
    bg = torch.empty((M, 2), dtype=torch.int32, device=dev)
    ix.apx_index(torch.from_numpy(sig).to(dev), None, bd, bg)
    torch.cuda.synchronize()
    onodes = X.strongest_nodes(ref, 19)
    olut = X.lookup_table(dirs, G.astype(np.float64), onodes)
    # vectorised restatement for all M (the plain-loop oracle is checked on a sample below)
    dl = ((img[:, olut].astype(np.float64) - ref[onodes][None, None, :]) ** 2).sum(-1)      # [M, Ng]
    assert np.allclose(bd.cpu().numpy()[:, 0], dl.min(1), rtol=2e-5)
    for m in (0, 31, 32, 8191, 8192, M - 1):
        od, og = X.best_solutions(X.index_delta(img[m], olut, ref[onodes]), 2)
        assert np.allclose(bd[m].cpu().numpy(), od, rtol=2e-5) and list(bg[m].cpu().numpy()) == list(og)
    ix.apx_indexer_destroy()


# ---- NEXT-3 ------------------------------------------------------------------------------------------------------
def _fsp_check(plan, xyz, types, centres, R, k_max, L, accepted=None, path=0):
    """|F| of apx_fsp against Eq. 2 written out in fp64 (oracle), element by element.  Tolerance:
    the fp32 phase k.d carries <= 3 roundings of relative 6e-8 on |k.d| <= sqrt3 k_max R cycles, i.e. a phase error of
    about 2 pi * 2e-7 * sqrt3 k_max R per ion, and the sum over N_w ions at most N_w times that."""
    import torch
    dev = torch.device("cuda:0")
    M = len(centres)
    out = torch.full((M, L, L, L), -7.0, dtype=torch.float32, device=dev)
    cnt = torch.full((M,), -1, dtype=torch.int32, device=dev)
    plan.apx_fsp_set_path(path)                                                 # 0 = tensor cores (+ FP32 for big ROIs), 1 = FP32 pipe
    plan.apx_fsp(torch.from_numpy(centres).to(dev), k_max, L, out, cnt)
    torch.cuda.synchronize()
    got, gc = out.cpu().numpy(), cnt.cpu().numpy()
    for m in range(M):
        rel = O.members(xyz, types, centres[m], R, accepted=accepted)
        assert gc[m] == len(rel)
        ref = np.abs(X.fsp(rel, k_max, L))
        tol = 1e-4 * ref + max(1.0, len(rel)) * (2e-6 + 2 * math.pi * 2e-7 * math.sqrt(3) * k_max * R)
        assert (np.abs(got[m] - ref) <= tol).all(), (m, np.abs(got[m] - ref).max(), tol.min())
    return gc


def test_fsp_against_oracle_small_grids():
    import torch
    dev = torch.device("cuda:0")
    rng = _rng(21)
    rot = random_rotation(rng)
    xyz = lattice_in_ball(0.405, fcc_basis, rot, (0, 0, 0), 3.0)
    xyz = xyz[rng.random(len(xyz)) < 0.5] + rng.standard_normal((1, 3)) * 0.0
    xyz = np.ascontiguousarray((xyz + rng.standard_normal(xyz.shape) * 0.03).astype(np.float32))
    types = (rng.random(len(xyz)) < 0.2).astype(np.uint8)
    R = 1.5
    plan = apx.Plan(R, 256, O.dirs_fibonacci(8), k_lo=7, k_hi=17, device=0)
    plan.apx_ingest(torch.from_numpy(xyz).to(dev), torch.from_numpy(types).to(dev))
    centres = np.array([[0, 0, 0], [0.4, -0.3, 0.2], [2.6, 0, 0], [9, 9, 9]], np.float32)       # full, shifted, partial, empty
    for path in (0, 1):
        for L, k_max in ((9, 5.0), (16, 2.0 * math.pi), (33, 6.0), (1, 3.0), (6, 3.0), (7, 4.5)):      # every L mod 4: four z-slices per CTA
            gc = _fsp_check(plan, xyz, types, centres, R, k_max, L, path=path)
            assert gc[3] == 0 and gc[0] > 300
    plan.apx_plan_destroy()
    # with an ion-type filter (Eq. 2: "all atoms N_w of a selected atom type")
    plan = apx.Plan(R, 256, O.dirs_fibonacci(8), k_lo=7, k_hi=17, accepted_types={1}, device=0)
    plan.apx_ingest(torch.from_numpy(xyz).to(dev), torch.from_numpy(types).to(dev))
    for path in (0, 1):
        _fsp_check(plan, xyz, types, centres[:2], R, 5.0, 9, accepted={1}, path=path)
    plan.apx_plan_destroy()


def test_fsp_bragg_peak_and_multi_tile_grid():
    """L = 80 > one 64 x 64 tile (ragged second tile); noiseless fcc Al with its cube axes along x, y, z: the {200} reflection
    at |k| = 2/a sits on the grid and reaches |F| = N_w (every ion in phase); sampled z-slices against the oracle."""
    import torch
    dev = torch.device("cuda:0")
    a, R = 0.4, 1.6                                                              # 2/a = 5.0 = k_max: the last grid point
    xyz = np.ascontiguousarray(lattice_in_ball(a, fcc_basis, np.eye(3), (0, 0, 0), 2.5, shift=np.zeros(3)).astype(np.float32))
    plan = apx.Plan(R, 256, O.dirs_fibonacci(8), k_lo=7, k_hi=17, device=0)
    plan.apx_ingest(torch.from_numpy(xyz).to(dev), None)
    L, k_max = 81, 5.0
    rel = O.members(xyz, None, np.zeros(3, np.float32), R)
    ref = np.abs(X.fsp(rel, k_max, L))
    for path in (0, 1):
        out = torch.full((1, L, L, L), -7.0, dtype=torch.float32, device=dev)
        cnt = torch.empty(1, dtype=torch.int32, device=dev)
        plan.apx_fsp_set_path(path)
        plan.apx_fsp(torch.zeros((1, 3), dtype=torch.float32, device=dev), k_max, L, out, cnt)
        torch.cuda.synchronize()
        F, n = out.cpu().numpy()[0], int(cnt.item())
        c = L // 2
        assert F[c, c, c] == pytest.approx(n, rel=1e-6)                           # F(0) = N_w
        for idx in ((c, c, 0), (c, c, L - 1), (c, 0, c), (L - 1, c, c)):           # k = (+-2/a, 0, 0) etc.
            assert F[idx] == pytest.approx(n, rel=1e-4)
        tol = 1e-4 * ref + n * (2e-6 + 2 * math.pi * 2e-7 * math.sqrt(3) * k_max * R)
        assert (np.abs(F - ref) <= tol).all(), (path, np.abs(F - ref).max())
    plan.apx_plan_destroy()


def test_fsp_streams_rois_larger_than_the_shared_ion_buffer():
    import torch
    dev = torch.device("cuda:0")
    xyz = np.ascontiguousarray(lattice_in_ball(0.405, fcc_basis, random_rotation(_rng(4)), (0, 0, 0), 4.0).astype(np.float32))
    types = np.zeros(len(xyz), np.uint8)
    # ~9000 ions > 6144: the FP32 kernel streams the cell rows; ~5100 ions: more than the tensor-core kernel holds (4096) but
    # within the FP32 kernel's buffer; with a small ROI riding along so that the deferred list is shorter than M
    for R, lo, hi in ((3.3, 6144, 10 ** 6), (2.75, 4096, 6144)):
        plan = apx.Plan(R, 256, O.dirs_fibonacci(8), k_lo=7, k_hi=17, device=0)
        plan.apx_ingest(torch.from_numpy(xyz).to(dev), torch.from_numpy(types).to(dev))
        for path in (0, 1):
            gc = _fsp_check(plan, xyz, types, np.array([[0.1, 0.2, -0.1], [3.9, 0.0, 0.0]], np.float32), R, 4.0, 12, path=path)
            assert lo < gc[0] <= hi and gc[1] < 4096
        plan.apx_plan_destroy()
