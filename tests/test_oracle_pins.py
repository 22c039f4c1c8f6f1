"""Pins for the CPU oracle: what the paper and the mathematics fix, NOT the oracle's own formulas
re-typed.  Each test names the pin of SURVEY.md section 8(c) / DESIGN.md it implements.
CPU only (-m "not gpu")."""
import cmath
import math
import os
from fractions import Fraction

import numpy as np
import pytest

from oracle import oracle as O
from workloads import (fcc_basis, bcc_basis, random_rotation, lattice_in_ball, make_config)

GOLD = os.path.join(os.path.dirname(__file__), "golden", "paper_fig2_caption.txt")


def _gold():
    out = {}
    for line in open(GOLD):
        if line.startswith("#") or not line.strip():
            continue
        k, v = line.split()
        out[k] = float(v)
    return out


def _rng(seed):
    return np.random.Generator(np.random.PCG64(seed))


def _crystal(a, basis, rot, R, shift=(0.137, 0.259, 0.391)):
    p = lattice_in_ball(a, basis, rot, (0, 0, 0), R + 0.5, shift=np.array(shift))
    return np.ascontiguousarray(p.astype(np.float32))


# ---- P2: numbers printed in the paper -------------------------------------------------------
def test_P2_printed_values_fig2_caption():
    g = _gold()
    m, R = int(g["m"]), g["R_nm"]
    B = 2 ** m
    R2, s = O.constants(R, B, pad=1)
    # L436: (2^(m-1)-1)/R = 6.35 / Angstrom at R = 20 Angstrom  <=>  s = 63.5 / nm at R = 2 nm
    assert float(s) / 10.0 == pytest.approx(g["freq_resolution_per_angstrom"], abs=1e-6)
    assert (2 ** (m - 1) - 1) / g["R_angstrom"] == pytest.approx(g["freq_resolution_per_angstrom"])
    # L138: b = floor(f L / f_s), f = 1/(0.5 a), f_s = L/(2(R+dR)), dR = R/(2^(m-1)-1)
    dR = R / (2 ** (m - 1) - 1)
    fs = B / (2 * (R + dR))
    assert math.floor((1 / (0.5 * g["a_nm_matching_printed_bin"])) * B / fs) == int(g["printed_bin"])
    assert float(R2) == 4.0


# ---- P1: closed-form peak position on noiseless lattices (L122, L138; north_star (i)) ---------
@pytest.mark.parametrize("name,a,basis,hkl,dfac", [
    ("fcc100", 0.405, fcc_basis, (1, 0, 0), 1 / 2),
    ("fcc110", 0.405, fcc_basis, (1, 1, 0), 1 / (2 * math.sqrt(2))),
    ("fcc111", 0.405, fcc_basis, (1, 1, 1), 1 / math.sqrt(3)),
    ("bcc100", 0.316, bcc_basis, (1, 0, 0), 1 / 2),
    ("bcc110", 0.316, bcc_basis, (1, 1, 0), 1 / math.sqrt(2)),
    ("bcc111", 0.316, bcc_basis, (1, 1, 1), 1 / (2 * math.sqrt(3))),
])
@pytest.mark.parametrize("B,pad", [(256, 1), (1024, 1), (256, 0)])
def test_P1_closed_form_peak(name, a, basis, hkl, dfac, B, pad):
    R = 2.0
    rot = random_rotation(_rng(7))
    xyz = _crystal(a, basis, rot, R)
    n = rot @ (np.array(hkl, np.float64) / np.linalg.norm(hkl))
    dR = R / (B // 2 - 1) if pad else 0.0
    k0 = 2 * (R + dR) / (dfac * a)
    kr = int(round(k0))
    sig, cnt = O.signatures(xyz, None, np.zeros((1, 3), np.float32), n[None].astype(np.float32),
                            R, B, pad=pad, k_lo=kr - 2, k_hi=kr + 2)
    assert abs(int(sig[0, 0, 1]) - kr) <= 1
    # "perfect crystals give normalised peaks ~ 1.0" (L424): the plane comb is coherent
    assert sig[0, 0, 0] / cnt[0] > 0.6
    # a direction far from any low-index zone axis has no such peak
    off = rot @ (np.array([0.31, 0.79, 0.53]) / np.linalg.norm([0.31, 0.79, 0.53]))
    sig2, _ = O.signatures(xyz, None, np.zeros((1, 3), np.float32), off[None].astype(np.float32),
                           R, B, pad=pad, k_lo=kr - 2, k_hi=kr + 2)
    assert sig2[0, 0, 0] < 0.5 * sig[0, 0, 0]


# ---- P3/P4: counts and DC (north_star (ii); L122, L151) -----------------------------------------
def test_P3_P4_counts_and_dc():
    w = make_config(2)
    dirs = O.dirs_fibonacci(16)
    c = np.array([9.0, 11.0, 9.0], np.float32)
    h, n = O.histograms(w.xyz, w.types, c, dirs, w.R, w.B)
    d = w.xyz.astype(np.float64) - c.astype(np.float64)
    r2 = np.einsum("ij,ij->i", d, d)
    n_lo, n_hi = int((r2 <= 4.0 - 1e-5).sum()), int((r2 <= 4.0 + 1e-5).sum())
    assert n_lo <= n <= n_hi and n > 900
    assert (h.sum(axis=1) == n).all()
    amp = O.spectrum(h[3])
    assert amp[0] == pytest.approx(n, rel=1e-14)
    assert (amp <= n * (1 + 1e-12)).all()


def test_membership_type_filter_and_closed_ball():
    # points at exactly r = R are inside (closed ball, DESIGN reading #4); types filter by set
    xyz = np.array([[2, 0, 0], [0, -2, 0], [0, 0, 2.0000002], [1, 1, 1], [0.5, 0, 0]], np.float32)
    types = np.array([0, 1, 0, 2, 1], np.uint8)
    c = np.zeros(3, np.float32)
    assert len(O.members(xyz, types, c, 2.0)) == 4
    assert len(O.members(xyz, types, c, 2.0, accepted={1})) == 2
    assert len(O.members(xyz, types, c, 2.0, accepted={0, 2})) == 2
    assert len(O.members(xyz, None, c, 2.0)) == 4
    rel = O.members(xyz + np.float32(8.0), types, c + np.float32(8.0), 2.0, accepted={2})
    assert rel.tolist() == [[1.0, 1.0, 1.0]]


# ---- P5: antipodal mirror (north_star (iii)) ------------------------------------------------------
def test_P5_antipodal_mirror():
    w = make_config(1)
    dirs = O.dirs_fibonacci(50)
    both = np.concatenate([dirs, -dirs]).astype(np.float32)
    h, n = O.histograms(w.xyz, w.types, w.centres[0], both, w.R, w.B)
    hp, hm = h[:50], h[50:]
    assert (hm == hp[:, ::-1]).all()          # floor(-x) = -floor(x)-1 for non-integer x
    for i in (0, 17, 49):
        np.testing.assert_allclose(O.spectrum(hp[i]), O.spectrum(hm[i]), rtol=1e-11, atol=1e-9)


# ---- P6: Parseval (north_star (iv)) -----------------------------------------------------------------
@pytest.mark.parametrize("B", [256, 1024])
def test_P6_parseval(B):
    rng = _rng(3)
    h = rng.integers(0, 7, B).astype(np.uint32)
    h[rng.random(B) < 0.5] = 0
    A = O.spectrum(h)
    lhs = float((h.astype(np.float64) ** 2).sum())
    rhs = (A[0] ** 2 + 2 * (A[1:B // 2] ** 2).sum() + A[B // 2] ** 2) / B
    assert rhs == pytest.approx(lhs, rel=1e-12)


# ---- P7: one and two ions (L232, L474: "intensity ~ 1.0 for few-atom ROIs") ---------------------------
def test_P7_one_and_two_ions():
    B = 256
    h = np.zeros(B, np.uint32)
    h[77] = 1
    np.testing.assert_allclose(O.spectrum(h), 1.0, rtol=0, atol=1e-13)
    h[77 + 9] = 1
    k = np.arange(B // 2 + 1)
    np.testing.assert_allclose(O.spectrum(h), 2 * np.abs(np.cos(np.pi * k * 9 / B)), atol=1e-12)


def test_tie_rule_lowest_k_and_empty_roi():
    # one ion exactly at the centre: x = 0 -> bin B/2, |X_k| = 1 for every k -> lowest k wins
    xyz = np.zeros((1, 3), np.float32)
    dirs = O.dirs_fibonacci(4)
    sig, cnt = O.signatures(xyz, None, xyz, dirs, 1.0, 256, k_lo=5, k_hi=40)
    assert cnt[0] == 1 and (sig[0, :, 1] == 5).all() and (sig[0, :, 0] == 1.0).all()
    far = np.full((1, 3), 50.0, np.float32)                     # empty ROI: (0, k_lo), count 0
    sig, cnt = O.signatures(xyz, None, far, dirs, 1.0, 256, k_lo=5, k_hi=40)
    assert cnt[0] == 0 and (sig[0, :, 1] == 5).all() and (sig[0, :, 0] == 0.0).all()
    sig, cnt = O.signatures(xyz, None, far, dirs, 1.0, 256)     # default window [1, B/2]
    assert (sig[0, :, 1] == 1).all()


# ---- P8: brute force on tiny clouds with exact rational arithmetic (north_star (v)) ---------------------
def test_P8_bruteforce_exact_rational():
    """Dyadic coordinates / directions and s = 63.5: every fp32 operation of the contract is exact,
    so Eq. 1 evaluated with Python Fractions must give the same bins; DFT by cmath."""
    B, R, pad = 256, 2.0, 1
    pts = [(0.5, -0.25, 0.125), (-1.0, 0.75, 0.5), (0.0, 0.0, -1.5), (1.25, 0.5, -0.75),
           (-0.375, -1.5, 0.25), (1.0, 1.0, 1.0), (3.0, 0.0, 0.0), (-0.0625, 0.03125, 1.96875)]
    dirs = [(1.0, 0.0, 0.0), (0.0, -1.0, 0.0), (0.5, 0.5, -0.5), (-0.25, 0.75, 0.5)]   # need not be unit
    centre = (0.25, -0.5, 0.125)
    xyz = np.array(pts, np.float32) + np.array(centre, np.float32)
    h, n = O.histograms(xyz, None, np.array(centre, np.float32), np.array(dirs, np.float32), R, B, pad)
    dR = Fraction(2) / (B // 2 - 1)
    exp = np.zeros((len(dirs), B), np.int64)
    inside = [p for p in pts if sum(Fraction(v) ** 2 for v in p) <= 4]
    assert n == len(inside) == 7
    for di, nvec in enumerate(dirs):
        for p in inside:
            t = sum(Fraction(a) * Fraction(b) for a, b in zip(nvec, p))
            b = math.floor((t + 2 + dR) * B / (2 * dR + 4))          # Eq. 1 literally (L68)
            exp[di, min(max(b, 0), B - 1)] += 1
    assert (h.astype(np.int64) == exp).all()
    sig, _, win = O.signatures(xyz, None, np.array([centre], np.float32), np.array(dirs, np.float32),
                               R, B, pad, k_lo=3, k_hi=60, want_window=True)
    for di in range(len(dirs)):
        amps = [abs(sum(int(exp[di, j]) * cmath.exp(-2j * cmath.pi * j * k / B) for j in range(B)))
                for k in range(3, 61)]
        np.testing.assert_allclose(win[0, di], amps, rtol=1e-10, atol=1e-10)
        kb = 3 + int(np.argmax(np.array(amps) >= max(amps) * (1 - 1e-12)))
        assert int(sig[0, di, 1]) == kb
        assert sig[0, di, 0] == pytest.approx(max(amps), rel=1e-6)
