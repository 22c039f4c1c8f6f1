"""CPU ORACLE for the rows SURVEY.md 8(f) marks "next": signature epilogues (NEXT-2), indexing (NEXT-1, Eq. 3),
the reciprocal space method FSP (NEXT-3, Eq. 2) and the adaptive ROI-grid refinement (NEXT-4).

TEST INFRASTRUCTURE ONLY, like oracle/aptsig_oracle.c: importable from tests/, __graft_entry__.smoke() and bench.py's
cpu_baseline / --impl reference legs.  Plain numpy in fp64, one obvious loop or array expression per formula, in the
paper's order; nothing is shared with paper_2009_00735_b200/.  Citations are lines of /root/reference/PAPER.md.

Readings taken where the paper is silent (listed in DESIGN.md section 2):
  #19 "normalised intensity" = A / N_c, the amplitude over the DC amplitude = ion count (L122/L151: the strongest,
      unnormalised peak "gives only the total number of atoms"; L424: perfect crystals then give ~1.0; L232: few-atom
      ROIs give ~1.0; L210: the threshold kappa >= 0.75 is on that scale).  An empty ROI has intensity 0.
  #20 local-maximum peak mode (SURVEY reading R2, L149-151 "second strongest peak"): bin k of the window is a local
      maximum when A_k > A_{k-1} and A_k >= A_{k+1} (A_{B/2+1} = A_{B/2-1} by conjugate symmetry); the signature is the
      highest local maximum (lowest k on ties); a window without one gives (0, k_lo), like an empty ROI.
  #21 refinement (L210, L442-452): the grid cell (a cube of the grid spacing around the ROI centre) of every ROI
      whose maximum normalised intensity is >= kappa is split into split^3 sub-cells, a new ROI at each sub-cell centre:
      c' = fl32(c + fl32(((i + 0.5)/split - 0.5) * spacing)) per axis, i = 0..split-1, x fastest.
  #22 rotations are unit quaternions (w, x, y, z), acting actively: v' = q v q*; "closest neighbouring node" (L369) =
      the mesh node with the largest dot product with the rotated node, lowest index on ties.
  #23 the orientation set (L367: MTEX, 618 324 orientations, 1 degree, m-3m; not in the container) is replaced by a
      cubic lattice of Rodrigues vectors r = tan(w/2) n inside the m-3m fundamental zone
      (|r_i| <= sqrt2 - 1, |r_1|+|r_2|+|r_3| <= 1), lattice constant tan(spacing/2).
  #24 Eq. 3 as printed: Delta = sum_v (S_msr[p_v^g] - S_ref[v])^2 over the N_hat strongest reference nodes v (L369-373);
      the K best solutions are the K smallest Delta, lowest orientation index on ties (L416).
  #25 Eq. 2 as printed, exp(-2 pi i k.(p_w - p_c)); the k grid is L_D points per axis, uniformly spaced over
      [-k_max, +k_max] with both ends included (L389: "k in [-2pi, +2pi]^3", L_D = 64..512); the signature stores |F|.
"""
from __future__ import annotations
import math
import numpy as np


# ---------------------------------------------------------------------------------------------------------------
# NEXT-2: signature epilogues
# ---------------------------------------------------------------------------------------------------------------
def normalised(amplitude, counts):
    """Reading #19: A / N_c per material point (L424, L232); empty ROI -> 0.  amplitude [M, D], counts [M]."""
    a = np.asarray(amplitude, np.float64)
    n = np.asarray(counts, np.float64)[:, None]
    return np.where(n > 0, a / np.where(n > 0, n, 1.0), 0.0)


def local_max_peak(amps, k_first, k_lo, k_hi, B):
    """Reading #20.  `amps[j]` = A_k for k = k_first + j, covering at least [max(k_lo-1, 0), min(k_hi+1, B/2)].
    Returns (A*, k*)."""
    def A(k):
        if k > B // 2:
            k = B - k                       # conjugate symmetry of a real input: A_{B/2+1} = A_{B/2-1}
        if k < 0:
            k = -k
        return float(amps[k - k_first])
    best, kbest = 0.0, k_lo
    found = False
    for k in range(k_lo, k_hi + 1):
        if A(k) > A(k - 1) and A(k) >= A(k + 1):
            if not found or A(k) > best:
                best, kbest, found = A(k), k, True
    return (best, kbest) if found else (0.0, k_lo)


# ---------------------------------------------------------------------------------------------------------------
# NEXT-4: adaptive refinement of the ROI grid (L102, L210, L442-452)
# ---------------------------------------------------------------------------------------------------------------
def intensity_max(amplitude, counts):
    """Maximum normalised intensity per material point (L210 "maximum intensity per signature")."""
    nrm = normalised(amplitude, counts)
    return nrm.max(axis=1) if nrm.shape[1] else np.zeros(len(nrm))


def refine_select(kappa_max, kappa):
    """Indices of the material points whose maximum normalised intensity reaches the threshold (L210: kappa >= 0.75)."""
    return np.nonzero(np.asarray(kappa_max) >= kappa)[0]


def refine_centres(centres, selected, spacing, split):
    """Reading #21: split^3 new ROI centres per selected material point (L210: 5^3), float32 [len(selected)*split^3, 3],
    ordered by selected point, then z, y, x (x fastest)."""
    c = np.asarray(centres, np.float32)
    off = np.array([np.float32(((i + 0.5) / split - 0.5) * float(spacing)) for i in range(split)], np.float32)
    out = np.zeros((len(selected), split, split, split, 3), np.float32)
    for s, m in enumerate(selected):
        for iz in range(split):
            for iy in range(split):
                for ix in range(split):
                    out[s, iz, iy, ix, 0] = np.float32(c[m, 0] + off[ix])
                    out[s, iz, iy, ix, 1] = np.float32(c[m, 1] + off[iy])
                    out[s, iz, iy, ix, 2] = np.float32(c[m, 2] + off[iz])
    return out.reshape(-1, 3)


# ---------------------------------------------------------------------------------------------------------------
# NEXT-1: indexing (L98, L369-373, Eq. 3)
# ---------------------------------------------------------------------------------------------------------------
def quat_to_matrix(q):
    """Active rotation matrix of the unit quaternion (w, x, y, z): v' = q v q* (reading #22)."""
    w, x, y, z = [float(v) for v in q]
    return np.array([[1 - 2 * (y * y + z * z), 2 * (x * y - z * w), 2 * (x * z + y * w)],
                     [2 * (x * y + z * w), 1 - 2 * (x * x + z * z), 2 * (y * z - x * w)],
                     [2 * (x * z - y * w), 2 * (y * z + x * w), 1 - 2 * (x * x + y * y)]], np.float64)


def so3_grid_cubic(spacing_deg):
    """Reading #23: Rodrigues-vector lattice (lattice constant tan(spacing/2), origin included) cut to the m-3m
    fundamental zone; returns unit quaternions float64 [N_g, 4] with w > 0, ordered by lattice index (z, y, x)."""
    h = math.tan(math.radians(spacing_deg) / 2.0)
    lim = math.sqrt(2.0) - 1.0
    n = int(math.floor(lim / h + 1e-12))
    out = []
    for iz in range(-n, n + 1):
        for iy in range(-n, n + 1):
            for ix in range(-n, n + 1):
                r = np.array([ix * h, iy * h, iz * h])
                if np.abs(r).max() <= lim + 1e-12 and np.abs(r).sum() <= 1.0 + 1e-12:
                    w = 1.0 / math.sqrt(1.0 + float(r @ r))
                    out.append((w, r[0] * w, r[1] * w, r[2] * w))
    return np.array(out, np.float64)


def strongest_nodes(ref_image, n_hat):
    """The n_hat mesh nodes with the highest reference intensity, in decreasing order (L369 "pick those nodes for which
    the signal is strongest ... in decreasing order"), lower node index first among equals."""
    img = np.asarray(ref_image, np.float64)
    order = sorted(range(len(img)), key=lambda i: (-img[i], i))
    return np.array(order[:n_hat], np.int64)


def nearest_node(dirs, v):
    """Index of the mesh node closest to the unit vector v: largest dot product, lowest index on ties (reading #22)."""
    d = np.asarray(dirs, np.float64) @ np.asarray(v, np.float64)
    return int(np.argmax(d))


def lookup_table(dirs, quats, nodes):
    """L369-371: p[g][v] = mesh node closest to node `nodes[v]` rotated by quats[g].  int64 [N_g, N_hat]."""
    dirs64 = np.asarray(dirs, np.float64)
    out = np.zeros((len(quats), len(nodes)), np.int64)
    for g, q in enumerate(quats):
        Rm = quat_to_matrix(q)
        for v, node in enumerate(nodes):
            out[g, v] = nearest_node(dirs64, Rm @ dirs64[node])
    return out


def index_delta(image, lut, ref_values):
    """Eq. 3 for one measured image (normalised intensities, [D]) against every orientation: float64 [N_g]."""
    img = np.asarray(image, np.float64)
    ref = np.asarray(ref_values, np.float64)
    out = np.zeros(len(lut))
    for g in range(len(lut)):
        acc = 0.0
        for v in range(len(ref)):
            diff = img[lut[g, v]] - ref[v]
            acc += diff * diff
        out[g] = acc
    return out


def best_solutions(delta, K):
    """The K smallest image differences and their orientation indices, lowest index first among equals (L416)."""
    order = sorted(range(len(delta)), key=lambda g: (delta[g], g))[:K]
    return np.array([delta[g] for g in order]), np.array(order, np.int64)


def quat_disorientation_deg_cubic(q1, q2):
    """Smallest rotation angle (degrees) between two orientations under the 24 proper rotations of m-3m (L367);
    used only to check that indexing recovers a known orientation."""
    def mul(a, b):
        return np.array([a[0] * b[0] - a[1] * b[1] - a[2] * b[2] - a[3] * b[3],
                         a[0] * b[1] + a[1] * b[0] + a[2] * b[3] - a[3] * b[2],
                         a[0] * b[2] - a[1] * b[3] + a[2] * b[0] + a[3] * b[1],
                         a[0] * b[3] + a[1] * b[2] - a[2] * b[1] + a[3] * b[0]])
    s = math.sqrt(0.5)
    syms = [(1, 0, 0, 0), (0, 1, 0, 0), (0, 0, 1, 0), (0, 0, 0, 1),
            (s, s, 0, 0), (s, -s, 0, 0), (s, 0, s, 0), (s, 0, -s, 0), (s, 0, 0, s), (s, 0, 0, -s),
            (0, s, s, 0), (0, s, -s, 0), (0, s, 0, s), (0, s, 0, -s), (0, 0, s, s), (0, 0, s, -s),
            (.5, .5, .5, .5), (.5, -.5, -.5, -.5), (.5, .5, -.5, -.5), (.5, -.5, .5, .5),
            (.5, .5, .5, -.5), (.5, -.5, -.5, .5), (.5, .5, -.5, .5), (.5, -.5, .5, -.5)]
    q1c = np.array([q1[0], -q1[1], -q1[2], -q1[3]], np.float64)
    d = mul(q1c, np.asarray(q2, np.float64))          # misorientation in the crystal frame: g1^-1 g2, equivalents g1^-1 g2 s
    best = 0.0
    for sy in syms:
        w = abs(mul(d, np.array(sy, np.float64))[0])
        best = max(best, min(1.0, w))
    return math.degrees(2.0 * math.acos(best))


# ---------------------------------------------------------------------------------------------------------------
# NEXT-3: reciprocal space method, Eq. 2 (L79-84, L389-393)
# ---------------------------------------------------------------------------------------------------------------
def fsp_kaxis(k_max, L):
    """Reading #25: L points uniformly spaced over [-k_max, +k_max], both ends included."""
    if L == 1:
        return np.zeros(1)
    return -float(k_max) + np.arange(L) * (2.0 * float(k_max) / (L - 1))


def fsp(rel, k_max, L):
    """Eq. 2 for one ROI: F[iz, iy, ix] = sum_w exp(-2 pi i k.(p_w - p_c)), k = (kx[ix], ky[iy], kz[iz]);
    `rel` = p_w - p_c of the ROI's ions, [N_w, 3] (the oracle's membership, fp32 differences).  complex128 [L, L, L]."""
    rel = np.asarray(rel, np.float64).reshape(-1, 3)
    k = fsp_kaxis(k_max, L)
    F = np.zeros((L, L, L), np.complex128)
    for iz in range(L):
        for iy in range(L):
            phase = rel[:, 0][None, :] * k[:, None] + rel[:, 1][None, :] * k[iy] + rel[:, 2][None, :] * k[iz]   # [L, N_w]
            F[iz, iy, :] = np.exp(-2j * np.pi * phase).sum(axis=1)
    return F
