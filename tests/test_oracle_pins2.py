"""More oracle pins and pins of the oracle's direction grids. CPU only."""
import math

import numpy as np
import pytest

from oracle import oracle as O
from workloads import make_config, fcc_basis, random_rotation, lattice_in_ball


def _rng(seed):
    return np.random.Generator(np.random.PCG64(seed))


def _uniform_ball(rng, n, R):
    p = rng.standard_normal((n, 3))
    p /= np.linalg.norm(p, axis=1, keepdims=True)
    return (p * (R * rng.random(n) ** (1 / 3))[:, None]).astype(np.float32)


# ---- P9: ROI-shape envelope of a uniform ball (textbook: projection of a ball is a parabola) ----
def test_P9_uniform_ball_envelope():
    R, B, pad, n = 2.0, 1024, 1, 200_000
    xyz = _uniform_ball(_rng(11), n, R * 0.999999)
    dirs = O.dirs_fibonacci(3)
    h, nc = O.histograms(xyz, None, np.zeros(3, np.float32), dirs, R, B, pad)
    assert nc == n
    for d in range(3):
        A = O.spectrum(h[d])
        for k in (1, 2, 3):
            x = math.pi * k * (1 - 2.0 * pad / B)
            env = abs(3 * (math.sin(x) - x * math.cos(x)) / x ** 3)
            assert A[k] / n == pytest.approx(env, abs=5 / math.sqrt(n))


# ---- P10: noise floor (Rayleigh) and Debye-Waller damping (textbook) ---------------------------------
def test_P10_noise_floor_rayleigh():
    R, B = 2.0, 1024
    xyz = _uniform_ball(_rng(5), 1000, R * 0.999)
    dirs = O.dirs_fibonacci(200)
    sig, cnt, win = O.signatures(xyz, None, np.zeros((1, 3), np.float32), dirs, R, B,
                                 k_lo=40, k_hi=80, want_window=True)
    mean = win.mean() / math.sqrt(cnt[0])
    assert mean == pytest.approx(math.sqrt(math.pi) / 2, rel=0.05)      # 0.886 sqrt(N)


def test_P10_debye_waller():
    R, B, a, sigma = 2.0, 256, 0.405, 0.04
    rot = random_rotation(_rng(9))
    sites = lattice_in_ball(a, fcc_basis, rot, (0, 0, 0), R + 0.5)
    n = rot @ np.array([1.0, 0, 0])
    k0 = int(round(2 * (R + R / 127) / (a / 2)))
    ratios = []
    for seed in range(6):
        p = (sites + _rng(100 + seed).standard_normal(sites.shape) * sigma).astype(np.float32)
        s0, c0 = O.signatures(sites.astype(np.float32), None, np.zeros((1, 3), np.float32),
                              n[None].astype(np.float32), R, B, k_lo=k0 - 1, k_hi=k0 + 1)
        s1, c1 = O.signatures(p, None, np.zeros((1, 3), np.float32), n[None].astype(np.float32),
                              R, B, k_lo=k0 - 1, k_hi=k0 + 1)
        ratios.append((s1[0, 0, 0] / c1[0]) / (s0[0, 0, 0] / c0[0]))
    dw = math.exp(-2 * math.pi ** 2 * sigma ** 2 / (a / 2) ** 2)
    assert np.mean(ratios) == pytest.approx(dw, rel=0.2)


# ---- P11: library cross-check (numpy.fft.rfft; numpy floor in fp32) ---------------------------------------
def test_P11_rfft_and_numpy_bins():
    w = make_config(2)
    dirs = O.dirs_fibonacci(64)
    c = np.array([11.0, 9.0, 7.0], np.float32)
    h, n = O.histograms(w.xyz, w.types, c, dirs, w.R, w.B)
    for d in (0, 31, 63):
        np.testing.assert_allclose(O.spectrum(h[d]), np.abs(np.fft.rfft(h[d].astype(np.float64))),
                                   rtol=1e-10, atol=1e-9)
    # independent numpy evaluation of Eq. 1 in fp64 on the same member set: bins agree except
    # O(1e-5) of (ion, direction) pairs that sit within fp32 rounding of a bin edge
    rel = O.members(w.xyz, w.types, c, w.R).astype(np.float64)
    dR = w.R / (w.B // 2 - 1)
    t = rel @ dirs.astype(np.float64).T
    b = np.floor((t + w.R + dR) * w.B / (2 * dR + 2 * w.R)).astype(np.int64).clip(0, w.B - 1)
    hn = np.stack([np.bincount(b[:, d], minlength=w.B) for d in range(64)])
    assert np.abs(hn - h.astype(np.int64)).sum() <= 2 * max(4, int(2e-4 * b.size))
    sig, cnt = O.signatures(w.xyz, w.types, c[None], dirs, w.R, w.B, k_lo=15, k_hi=34)
    for d in (5, 40):
        A = np.abs(np.fft.rfft(h[d].astype(np.float64)))[15:35]
        assert int(sig[0, d, 1]) == 15 + int(np.argmax(A))
        assert sig[0, d, 0] == pytest.approx(A.max(), rel=1e-6)


# ---- P12: invariances of the definition ---------------------------------------------------------------------
def test_P12_exact_translation_invariance():
    rng = _rng(21)
    grid = (rng.integers(-2048, 2048, (4000, 3)) / 1024.0).astype(np.float32)     # multiples of 2^-10
    c = np.array([0.25, -0.5, 0.125], np.float32)
    t = np.array([8.0, -16.0, 4.0], np.float32)                                      # sums stay exact
    dirs = O.dirs_fibonacci(32)
    h0, n0 = O.histograms(grid, None, c, dirs, 1.5, 512)
    h1, n1 = O.histograms(grid + t, None, c + t, dirs, 1.5, 512)
    assert n0 == n1 and n0 > 500 and (h0 == h1).all()


def test_P12_rotation_covariance():
    w = make_config(1)
    rot = random_rotation(_rng(4))
    dirs = O.dirs_fibonacci(64).astype(np.float64)
    h0, n0 = O.histograms(w.xyz, None, w.centres[0], dirs.astype(np.float32), w.R, w.B)
    xr = (w.xyz.astype(np.float64) @ rot.T).astype(np.float32)
    dr = (dirs @ rot.T).astype(np.float32)
    h1, n1 = O.histograms(xr, None, w.centres[0], dr, w.R, w.B)
    assert abs(n0 - n1) <= 1
    assert np.abs(h0.astype(np.int64) - h1.astype(np.int64)).sum() <= 2 * (1 + int(1e-3 * n0 * 64))


def test_pad_flag_changes_only_the_scale():
    # pad=0: span [-R, R] (north_star literal); pad=1: paper Eq. 1. s differs by (B/2-1)/(B/2).
    _, s1 = O.constants(2.0, 256, 1)
    _, s0 = O.constants(2.0, 256, 0)
    assert float(s0) == 64.0 and float(s1) == 63.5
    xyz = np.array([[2.0, 0, 0], [-2.0, 0, 0], [0.01, 0, 0]], np.float32)
    d = np.array([[1.0, 0, 0]], np.float32)
    h0, _ = O.histograms(xyz, None, np.zeros(3, np.float32), d, 2.0, 256, pad=0)
    h1, _ = O.histograms(xyz, None, np.zeros(3, np.float32), d, 2.0, 256, pad=1)
    assert h0[0, 255] == 1 and h0[0, 0] == 1 and h0[0, 128] == 1       # +R clamps into B-1 (reading #5)
    assert h1[0, 255] == 1 and h1[0, 1] == 1 and h1[0, 128] == 1       # pad bin 0 stays empty at -R


# ---- direction grids of the oracle -----------------------------------------------------------------------------
def test_geodesic_grid_pins():
    for level, nv in [(0, 12), (1, 42), (2, 162), (3, 642)]:
        g = O.dirs_geodesic(level).astype(np.float64)
        assert len(g) == nv == 10 * 4 ** level + 2
        np.testing.assert_allclose(np.linalg.norm(g, axis=1), 1.0, atol=1e-7)
        # antipodally symmetric set; no duplicates
        key = {tuple(np.round(v, 5)) for v in g}
        assert len(key) == nv and all(tuple(np.round(-v, 5) + 0.0) in key or
                                      tuple(np.round(-v, 5)) in key for v in g)
    g6 = O.dirs_geodesic(6)
    assert len(g6) == 40962
    # near-uniform: nearest-neighbour angle spread stays within a factor ~1.4 (icosphere property)
    from scipy.spatial import cKDTree
    dd = cKDTree(g6).query(g6, k=2)[0][:, 1]
    assert dd.max() / dd.min() < 1.45


def test_fibonacci_grid_pins():
    D = 1000
    f = O.dirs_fibonacci(D).astype(np.float64)
    np.testing.assert_allclose(np.linalg.norm(f, axis=1), 1.0, atol=1e-7)
    np.testing.assert_allclose(f[:, 2], 1 - (2 * np.arange(D) + 1) / D, atol=1e-7)   # equal-area z
    ang = np.unwrap(np.arctan2(f[:, 1], f[:, 0]))
    np.testing.assert_allclose(np.diff(ang) % (2 * math.pi), (math.pi * (3 - math.sqrt(5))) % (2 * math.pi),
                               atol=1e-4)
    assert abs(f.mean(axis=0)).max() < 2e-3                                           # balanced


# ---- single-rounded fma order of the projection (reading #15) ---------------------
def _rn32(fr):
    """Fraction -> nearest binary32 (ties to even), exact integer arithmetic; normal range only."""
    from fractions import Fraction
    if fr == 0:
        return Fraction(0)
    sgn, a = (1 if fr > 0 else -1), abs(fr)
    e = 0
    while a >= 2 ** 24:
        a /= 2; e += 1
    while a < 2 ** 23:
        a *= 2; e -= 1
    q, r = divmod(a.numerator, a.denominator)
    twice = 2 * r
    if twice > a.denominator or (twice == a.denominator and (q & 1)):
        q += 1
    return sgn * Fraction(q) * (Fraction(2) ** e)


def test_projection_uses_single_rounded_fma_not_mul_add():
    """Eq. 1 in the contract's operation order: x = fma(n'z, dz, fma(n'y, dy, n'x*dx)), every fma ONE rounding.
    An oracle built with two-rounding a*b+c passes every pin whose inputs are dyadic; here (ion, direction) pairs are
    searched (seeded) whose bin differs between the two evaluation orders, in exact rational arithmetic, and the
    oracle must land on the fma bin for every one of them."""
    from fractions import Fraction
    rng = _rng(77)
    B, R = 1024, 2.0
    R2, s = O.constants(R, B, pad=1)
    found = 0
    for _ in range(400000):
        if found >= 6:
            break
        d = rng.standard_normal(3)
        d /= np.linalg.norm(d)
        n32 = d.astype(np.float32)
        npr = (n32 * np.float32(s)).astype(np.float32)                  # one fp32 multiply each (exact in numpy float32)
        # an ion whose projection sits within ~1e-5 of an integer: start from a random point and move it along n
        p = rng.uniform(-1.0, 1.0, 3)
        t = float(np.dot(npr.astype(np.float64), p))
        p = p + d * ((round(t) - t + rng.uniform(-3e-5, 3e-5)) / float(s))
        p32 = p.astype(np.float32)
        if float(np.dot(p32.astype(np.float64), p32.astype(np.float64))) > 3.9:
            continue
        F = [Fraction(float(v)) for v in npr]
        Dv = [Fraction(float(v)) for v in p32]                          # centre = origin: d = p exactly
        x_fma = _rn32(F[2] * Dv[2] + _rn32(F[1] * Dv[1] + _rn32(F[0] * Dv[0])))
        x_two = _rn32(_rn32(F[2] * Dv[2]) + _rn32(_rn32(F[1] * Dv[1]) + _rn32(F[0] * Dv[0])))
        b_fma, b_two = B // 2 + math.floor(x_fma), B // 2 + math.floor(x_two)
        if b_fma == b_two:
            continue
        found += 1
        h, n = O.histograms(p32[None, :], None, np.zeros(3, np.float32), n32[None, :], R, B)
        assert n == 1 and h[0, b_fma] == 1 and h[0, b_two] == 0, (b_fma, b_two, np.nonzero(h[0]))
    assert found >= 3, "search did not find pairs that separate fma from mul+add"
