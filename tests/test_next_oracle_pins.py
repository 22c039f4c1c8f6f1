"""Pins for oracle/next_oracle.py (SURVEY.md 8(f) rows NEXT-1..4): closed forms, invariants, special cases and tiny brute
force -- what the paper and the mathematics fix, not the oracle's formulas typed again.  CPU only."""
import cmath
import math

import numpy as np
import pytest

from oracle import oracle as O
from oracle import next_oracle as X
from workloads import fcc_basis, lattice_in_ball, random_rotation


def _rng(seed):
    return np.random.Generator(np.random.PCG64(seed))


def _uniform_ball(rng, n, R):
    p = rng.standard_normal((n, 3))
    p /= np.linalg.norm(p, axis=1, keepdims=True)
    return (p * (R * rng.random(n) ** (1 / 3))[:, None]).astype(np.float32)


def _al_ball(R, rot=np.eye(3), sigma=0.0, seed=1):
    p = lattice_in_ball(0.405, fcc_basis, rot, (0, 0, 0), R + 0.5)
    if sigma:
        p = p + _rng(seed).standard_normal(p.shape) * sigma
    return np.ascontiguousarray(p.astype(np.float32))


# ---- NEXT-2: normalised intensity (reading #19; L232, L424) -----------------------------------------------------
def test_normalised_single_ion_is_one_and_perfect_crystal_near_one():
    # L232 / L474: "few lithium atoms" -> intensity ~1.0: one ion gives A_k = 1 for every k, N_c = 1
    one = np.array([[0.3, -0.2, 0.1]], np.float32)
    sig, cnt = O.signatures(one, None, np.zeros((1, 3), np.float32), O.dirs_fibonacci(7), 2.0, 256, k_lo=5, k_hi=40)
    assert np.allclose(X.normalised(sig[..., 0], cnt), 1.0, atol=1e-6)
    # L424: perfect single crystal: peaks ~1.0 along <100>, background at least ten times lower along a generic direction
    xyz = _al_ball(2.0)
    dirs = np.array([[1, 0, 0], [0.5377, 0.2914, 0.7912]], np.float32)
    dirs /= np.linalg.norm(dirs, axis=1, keepdims=True)
    sig, cnt = O.signatures(xyz, None, np.zeros((1, 3), np.float32), dirs, 2.0, 256, k_lo=18, k_hi=22)
    nrm = X.normalised(sig[..., 0], cnt)
    assert nrm[0, 0] > 0.9 and nrm[0, 1] < 0.1 * nrm[0, 0]
    assert X.normalised(np.ones((1, 3)), np.zeros(1)).max() == 0.0            # empty ROI


# ---- NEXT-2: local-maximum peak mode (reading #20; L149-151) -----------------------------------------------------
def test_local_max_hand_sequences():
    B = 64
    amps = np.array([9, 5, 3, 4, 2, 2, 6, 6, 1], float)                        # A_0 .. A_8
    assert X.local_max_peak(amps, 0, 1, 7, B) == (6.0, 6)                        # plateau 6,6: the lower bin is the maximum
    assert X.local_max_peak(amps, 0, 1, 4, B) == (4.0, 3)
    assert X.local_max_peak(amps, 0, 1, 2, B) == (0.0, 1)                        # monotone decreasing: no local maximum
    full = np.concatenate([np.arange(33.0)])                                    # rising up to Nyquist: k = B/2 is a local max
    assert X.local_max_peak(full, 0, 20, 32, B) == (32.0, 32)                   # (A_{B/2+1} = A_{B/2-1} < A_{B/2})


def test_local_max_never_picks_the_ball_envelope():
    """P9: a uniform ball's spectrum falls monotonically over k = 1, 2, 3 (3(sin x - x cos x)/x^3), so the plain maximum
    of the window [1, 3] is the envelope at k = 1 while the local-maximum mode finds nothing there."""
    R, B, n = 2.0, 1024, 200_000
    xyz = _uniform_ball(_rng(11), n, R * 0.999999)
    h, nc = O.histograms(xyz, None, np.zeros(3, np.float32), O.dirs_fibonacci(3), R, B)
    for d in range(3):
        A = O.spectrum(h[d])
        assert A[1] > A[2] > A[3] > A[4]
        assert int(np.argmax(A[1:4])) + 1 == 1
        assert X.local_max_peak(A, 0, 1, 3, B) == (0.0, 1)


def test_local_max_finds_the_lattice_peak_under_the_envelope():
    """Jittered fcc Al along <100>: Debye-Waller damps the {200} peak (k0 = 2(R+dR)/d ~ 19.8 at B = 256, R = 2) below the
    ROI-shape envelope at k = 1, which wins a plain maximum over [1, 40]; the highest LOCAL maximum is the lattice peak."""
    R, B = 2.0, 256
    xyz = _al_ball(R, sigma=0.07, seed=3)
    d = np.array([[1, 0, 0]], np.float32)
    h, nc = O.histograms(xyz, None, np.zeros(3, np.float32), d, R, B)
    A = O.spectrum(h[0])
    assert int(np.argmax(A[1:41])) + 1 == 1
    a, k = X.local_max_peak(A, 0, 1, 40, B)
    assert abs(k - 2 * (R + R / (B // 2 - 1)) / (0.405 / 2)) <= 1 and a == A[k]


# ---- NEXT-4: refinement (reading #21; L210, L442-452) ------------------------------------------------------------
def test_refine_centres_tile_the_parent_cell():
    c = np.array([[10.0, 20.0, 30.0], [1.5, 2.5, 3.5], [7.0, 7.0, 7.0]], np.float32)
    sel = np.array([0, 2])
    out = X.refine_centres(c, sel, spacing=2.0, split=5)
    assert out.shape == (2 * 125, 3) and out.dtype == np.float32               # L210: 5^3 new ROIs per refined cell
    for s, m in enumerate(sel):
        blk = out[125 * s:125 * (s + 1)].astype(np.float64)
        assert np.allclose(blk.mean(0), c[m], atol=1e-6)
        for a in range(3):
            u = np.unique(np.round(blk[:, a], 5))
            assert len(u) == 5 and np.allclose(np.diff(u), 0.4, atol=1e-5)       # sub-cell edge = spacing / split
            assert u[0] == pytest.approx(c[m, a] - 0.8, abs=1e-5)                # outermost centres half a sub-cell inside
    assert np.allclose(out[1] - out[0], (0.4, 0, 0), atol=1e-6)                 # x fastest
    assert np.allclose(out[25] - out[0], (0, 0, 0.4), atol=1e-6)
    assert X.refine_centres(c, np.array([], np.int64), 2.0, 5).shape == (0, 3)


def test_intensity_threshold_selects_the_crystal_not_the_noise():
    """L210: ROIs whose maximum normalised intensity reaches kappa = 0.75 are refined: a perfect crystal reaches ~1 along
    its <100> poles, a random cloud stays near the Rayleigh floor 0.886/sqrt(N_c) (P10)."""
    R, B = 1.5, 256
    crystal = _al_ball(R)
    noise = _uniform_ball(_rng(2), len(crystal), R + 0.4) + np.float32(100.0)
    xyz = np.concatenate([crystal, noise])
    centres = np.array([[0, 0, 0], [100, 100, 100], [300, 0, 0]], np.float32)     # crystal, noise, empty
    dirs = np.concatenate([np.eye(3, dtype=np.float32), O.dirs_fibonacci(40)])
    k0 = round(2 * (R + R / (B // 2 - 1)) / (0.405 / 2))
    sig, cnt = O.signatures(xyz, None, centres, dirs, R, B, k_lo=k0 - 2, k_hi=k0 + 2)
    kmax = X.intensity_max(sig[..., 0], cnt)
    assert kmax[0] > 0.9 and kmax[1] < 0.3 and kmax[2] == 0.0
    assert list(X.refine_select(kmax, 0.75)) == [0]
    assert list(X.refine_select(np.array([0.75, 0.7499, 0.8]), 0.75)) == [0, 2]     # the threshold is inclusive (>=)


# ---- NEXT-1: rotations, orientation grid, look-up table, Eq. 3 ----------------------------------------------------
def test_quaternion_rotation_convention():
    s = math.sqrt(0.5)
    Rz = X.quat_to_matrix((s, 0, 0, s))                                        # 90 degrees about z, active: x -> y
    assert np.allclose(Rz @ [1, 0, 0], [0, 1, 0]) and np.allclose(Rz @ [0, 1, 0], [-1, 0, 0])
    q = _rng(1).standard_normal(4)
    q /= np.linalg.norm(q)
    M = X.quat_to_matrix(q)
    assert np.allclose(M @ M.T, np.eye(3), atol=1e-14) and np.linalg.det(M) == pytest.approx(1.0)
    ang = 2 * math.acos(abs(q[0]))
    assert np.trace(M) == pytest.approx(1 + 2 * math.cos(ang))                 # rotation angle from the trace
    assert np.allclose(M @ (q[1:] / np.linalg.norm(q[1:])), q[1:] / np.linalg.norm(q[1:]))   # the axis is fixed


def test_so3_grid_fills_the_cubic_fundamental_zone():
    spacing = 5.0
    G = X.so3_grid_cubic(spacing)
    assert np.allclose(np.linalg.norm(G, axis=1), 1.0) and (G[:, 0] > 0).all()
    assert (np.abs(G - [1, 0, 0, 0]).sum(1) < 1e-12).any()                      # the identity is a grid point
    r = G[:, 1:] / G[:, :1]
    lim = math.sqrt(2) - 1
    assert np.abs(r).max() <= lim + 1e-9 and np.abs(r).sum(1).max() <= 1 + 1e-9
    # volume of the truncated cube: (2 lim)^3 - 8 corner tetrahedra of leg 3 lim - 1
    vol = (2 * lim) ** 3 - 8 * (3 * lim - 1) ** 3 / 6
    assert len(G) == pytest.approx(vol / math.tan(math.radians(spacing) / 2) ** 3, rel=0.05)
    # quasi-equidistant: neighbours of a sample of grid points are 0.75 .. 1.0 spacings away, and any orientation has a grid
    # point within ~0.9 spacings (covering radius of a cubic lattice, sqrt3/2 lattice constants)
    rng = _rng(4)
    for i in rng.choice(len(G), 12, replace=False):
        others = np.delete(np.arange(len(G)), i)
        near = others[np.argsort(np.abs(G[others] @ G[i]))[-8:]]
        dmin = min(X.quat_disorientation_deg_cubic(G[i], G[j]) for j in near)
        assert 0.7 * spacing <= dmin <= 1.001 * spacing
    for _ in range(12):
        q = rng.standard_normal(4)
        q /= np.linalg.norm(q)
        cand = np.argsort(-np.max(np.abs(G @ _cubic_equivalents(q).T), axis=1))[:4]
        assert min(X.quat_disorientation_deg_cubic(q, G[j]) for j in cand) <= 0.9 * spacing


def _cubic_equivalents(q):
    """q * s for the 24 proper cubic symmetry rotations s (as rows)."""
    s = math.sqrt(0.5)
    syms = [(1, 0, 0, 0), (0, 1, 0, 0), (0, 0, 1, 0), (0, 0, 0, 1),
            (s, s, 0, 0), (s, -s, 0, 0), (s, 0, s, 0), (s, 0, -s, 0), (s, 0, 0, s), (s, 0, 0, -s),
            (0, s, s, 0), (0, s, -s, 0), (0, s, 0, s), (0, s, 0, -s), (0, 0, s, s), (0, 0, s, -s),
            (.5, .5, .5, .5), (.5, -.5, -.5, -.5), (.5, .5, -.5, -.5), (.5, -.5, .5, .5),
            (.5, .5, .5, -.5), (.5, -.5, -.5, .5), (.5, .5, -.5, .5), (.5, -.5, .5, -.5)]
    out = []
    for b in syms:
        a = q
        out.append([a[0] * b[0] - a[1] * b[1] - a[2] * b[2] - a[3] * b[3], a[0] * b[1] + a[1] * b[0] + a[2] * b[3] - a[3] * b[2],
                    a[0] * b[2] - a[1] * b[3] + a[2] * b[0] + a[3] * b[1], a[0] * b[3] + a[1] * b[2] - a[2] * b[1] + a[3] * b[0]])
    return np.array(out)


def test_lookup_table_identity_and_mesh_symmetry():
    dirs = O.dirs_geodesic(2)                                                   # 162 nodes
    nodes = np.array([0, 5, 17, 100, 161])
    ident = np.array([[1.0, 0, 0, 0]])
    assert (X.lookup_table(dirs, ident, nodes)[0] == nodes).all()              # unrotated: every node is its own neighbour
    # the geodesic mesh inherits the icosahedron's five-fold axis through base vertex 0: a rotation by 72 degrees about it
    # maps the node set onto itself, so the table is a permutation that reproduces the rotated nodes exactly
    ax = dirs[0].astype(np.float64)
    ax /= np.linalg.norm(ax)
    h = math.radians(72.0) / 2
    q = np.array([[math.cos(h), *(math.sin(h) * ax)]])
    allnodes = np.arange(len(dirs))
    lut = X.lookup_table(dirs, q, allnodes)[0]
    assert sorted(lut) == list(allnodes)
    assert np.allclose(dirs[lut], (X.quat_to_matrix(q[0]) @ dirs.astype(np.float64).T).T, atol=1e-6)
    assert X.nearest_node(dirs, dirs[42]) == 42


def test_strongest_nodes_and_best_solutions_order():
    img = np.array([0.1, 0.9, 0.5, 0.9, 0.2])
    assert list(X.strongest_nodes(img, 3)) == [1, 3, 2]                         # decreasing, lower index first among equals
    d, g = X.best_solutions(np.array([3.0, 1.0, 2.0, 1.0]), 3)
    assert list(g) == [1, 3, 2] and list(d) == [1.0, 1.0, 2.0]


def _cubic_image(dirs, rot):
    """A smooth test image with m-3m symmetry in the crystal frame `rot` (lab = rot @ crystal): peaks along <100>."""
    c = dirs.astype(np.float64) @ rot                                            # crystal-frame components
    return np.exp(-(1.0 - np.max(np.abs(c), axis=1)) / 0.02)


def test_eq3_recovers_a_known_rotation_of_the_reference():
    """Eq. 3 (L373): a measured image that IS the reference rotated by a grid orientation g0 has Delta ~ 0 at g0 (exactly 0
    for the identity), and the best solution is g0 up to cubic symmetry; Delta grows away from it."""
    dirs = O.dirs_geodesic(3)                                                   # 642 nodes, ~8 degrees apart
    G = X.so3_grid_cubic(10.0)
    ref = _cubic_image(dirs, np.eye(3))
    nodes = X.strongest_nodes(ref, 60)
    lut = X.lookup_table(dirs, G, nodes)
    g_id = int(np.argmin(np.abs(G - [1, 0, 0, 0]).sum(1)))
    assert X.index_delta(ref, lut, ref[nodes])[g_id] == 0.0                     # identical images: Delta = 0
    for g0 in (17, 240, len(G) - 5):
        msr = _cubic_image(dirs, X.quat_to_matrix(G[g0]))                       # the crystal rotated by G[g0]
        delta = X.index_delta(msr, lut, ref[nodes])
        d, g = X.best_solutions(delta, 3)
        assert X.quat_disorientation_deg_cubic(G[g[0]], G[g0]) <= 10.0
        assert d[0] < 0.25 * np.median(delta)


def test_indexing_end_to_end_on_hot_path_signatures():
    """The chain the paper describes (L92, L98): reference signature from an unrotated noiseless Al crystal, measured
    signature from the same crystal rotated by a known g0 (both through the hot-path oracle, {200} window), normalised
    A/N_c, N_hat strongest reference nodes, look-up table, Eq. 3: the best orientation is g0 within the resolution of the
    mesh (level 3: ~8 degrees between nodes) and of the orientation grid (10 degrees)."""
    R, B = 1.5, 256
    dirs = O.dirs_geodesic(3)
    k0 = round(2 * (R + R / (B // 2 - 1)) / (0.405 / 2))
    G = X.so3_grid_cubic(10.0)
    c0 = np.zeros((1, 3), np.float32)
    sig, cnt = O.signatures(_al_ball(R), None, c0, dirs, R, B, k_lo=k0 - 1, k_hi=k0 + 1)
    ref = X.normalised(sig[..., 0], cnt)[0]
    nodes = X.strongest_nodes(ref, 40)
    lut = X.lookup_table(dirs, G, nodes)
    for g0 in (33, 410):
        rot = X.quat_to_matrix(G[g0])
        sig, cnt = O.signatures(_al_ball(R, rot=rot), None, c0, dirs, R, B, k_lo=k0 - 1, k_hi=k0 + 1)
        delta = X.index_delta(X.normalised(sig[..., 0], cnt)[0], lut, ref[nodes])
        d, g = X.best_solutions(delta, 1)
        assert X.quat_disorientation_deg_cubic(G[g[0]], G[g0]) <= 12.0


# ---- NEXT-3: Eq. 2 ----------------------------------------------------------------------------------------------
def test_fsp_closed_forms():
    L, kmax = 9, 4.0
    k = X.fsp_kaxis(kmax, L)
    assert k[0] == -kmax and k[-1] == kmax and k[L // 2] == 0.0 and np.allclose(np.diff(k), 1.0)
    # one ion: |F| = 1 everywhere, phase -2 pi k.p; at the centre F = 1
    p = np.array([[0.13, -0.2, 0.31]])
    F = X.fsp(p, kmax, L)
    assert np.allclose(np.abs(F), 1.0)
    assert F[7, 2, 5] == pytest.approx(cmath.exp(-2j * math.pi * (k[5] * p[0, 0] + k[2] * p[0, 1] + k[7] * p[0, 2])))
    assert np.allclose(X.fsp(np.zeros((1, 3)), kmax, L), 1.0)
    # two ions: |F| = 2 |cos(pi k.(p1 - p2))|
    p2 = np.array([[0.1, 0.0, 0.0], [-0.15, 0.05, 0.2]])
    F = X.fsp(p2, kmax, L)
    dlt = p2[0] - p2[1]
    kk = np.stack(np.meshgrid(k, k, k, indexing="ij"), -1)                       # [iz, iy, ix] -> (kz, ky, kx)
    phase = kk[..., 2] * dlt[0] + kk[..., 1] * dlt[1] + kk[..., 0] * dlt[2]
    assert np.allclose(np.abs(F), 2 * np.abs(np.cos(math.pi * phase)), atol=1e-12)
    # F(0) = N_w; F(-k) = conj F(k)
    cloud = _rng(3).uniform(-1, 1, (50, 3))
    F = X.fsp(cloud, kmax, L)
    assert F[L // 2, L // 2, L // 2] == pytest.approx(50.0)
    assert np.allclose(F[::-1, ::-1, ::-1], np.conj(F))


def test_fsp_bragg_peaks_of_a_simple_cubic_lattice_and_brute_force():
    a, n = 0.5, 6
    g = (np.arange(n) - (n - 1) / 2) * a
    pts = np.stack(np.meshgrid(g, g, g, indexing="ij"), -1).reshape(-1, 3)
    L, kmax = 9, 4.0                                                            # k step 1.0: 1/a = 2.0 is on the grid
    F = np.abs(X.fsp(pts, kmax, L))
    k = X.fsp_kaxis(kmax, L)
    on = np.isclose(np.mod(k * a, 1.0), 0.0)                                    # reciprocal lattice points k a = integer
    assert np.allclose(F[np.ix_(on, on, on)], n ** 3)                           # every ion in phase: |F| = N_w
    assert F[L // 2, L // 2, L // 2 + 1] == pytest.approx(0.0, abs=1e-9)        # k a = 1/2: full cancellation along x
    # tiny brute force, written independently (Python complex numbers)
    cloud = _rng(8).uniform(-1, 1, (5, 3))
    Fc = X.fsp(cloud, 2.0, 3)
    kk = [-2.0, 0.0, 2.0]
    for iz in range(3):
        for iy in range(3):
            for ix in range(3):
                ref = sum(cmath.exp(-2j * math.pi * (kk[ix] * x + kk[iy] * y + kk[iz] * z)) for x, y, z in cloud)
                assert Fc[iz, iy, ix] == pytest.approx(ref, abs=1e-12)
