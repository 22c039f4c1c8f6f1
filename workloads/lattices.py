"""Lattice generators (numpy, fp64 internally, fp32 out). No method arithmetic lives here.

Recipe (stands in for paraprobe-synthetic):
lattice sites in the crystal frame (basis + fixed non-lattice shift) -> rotation into the lab frame
-> crop to box/ball -> Bernoulli(eta) thinning -> Gaussian jitter in the lab frame -> shuffle -> fp32.
"""
from __future__ import annotations
import numpy as np

fcc_basis = np.array([[0, 0, 0], [.5, .5, 0], [.5, 0, .5], [0, .5, .5]], dtype=np.float64)
bcc_basis = np.array([[0, 0, 0], [.5, .5, .5]], dtype=np.float64)

# fixed non-lattice offset (fractions of a) so that no site sits on a bin edge for zone-axis directions
DEFAULT_SHIFT = np.array([0.137, 0.259, 0.391], dtype=np.float64)


def random_rotation(rng: np.random.Generator) -> np.ndarray:
    """Uniform random rotation matrix from a normalised 4-Gaussian quaternion."""
    q = rng.standard_normal(4)
    q /= np.linalg.norm(q)
    w, x, y, z = q
    return np.array([
        [1 - 2 * (y * y + z * z), 2 * (x * y - z * w), 2 * (x * z + y * w)],
        [2 * (x * y + z * w), 1 - 2 * (x * x + z * z), 2 * (y * z - x * w)],
        [2 * (x * z - y * w), 2 * (y * z + x * w), 1 - 2 * (x * x + y * y)]], dtype=np.float64)


def _sites_bbox(a, basis, rot, lo, hi, shift, origin, chunk_cells=2_000_000):
    """Yield chunks of lab-frame sites rot @ (a*(ijk+basis+shift)) + origin that fall in [lo,hi]."""
    lo = np.asarray(lo, np.float64)
    hi = np.asarray(hi, np.float64)
    corners = np.array([[x, y, z] for x in (lo[0], hi[0]) for y in (lo[1], hi[1]) for z in (lo[2], hi[2])])
    cc = (corners - origin) @ rot / a          # crystal-frame coordinates in units of a (rot^T applied)
    imin = np.floor(cc.min(axis=0)).astype(np.int64) - 2
    imax = np.ceil(cc.max(axis=0)).astype(np.int64) + 2
    ny = int(imax[1] - imin[1] + 1)
    nz = int(imax[2] - imin[2] + 1)
    step = max(1, chunk_cells // (ny * nz))
    jj, kk = np.meshgrid(np.arange(imin[1], imax[1] + 1), np.arange(imin[2], imax[2] + 1), indexing="ij")
    jk = np.stack([jj.ravel(), kk.ravel()], axis=1).astype(np.float64)
    for i0 in range(int(imin[0]), int(imax[0]) + 1, step):
        ii = np.arange(i0, min(i0 + step, int(imax[0]) + 1), dtype=np.float64)
        cells = np.empty((ii.size, jk.shape[0], 3))
        cells[:, :, 0] = ii[:, None]
        cells[:, :, 1:] = jk[None, :, :]
        cells = cells.reshape(-1, 3)
        for b in basis:
            p = (cells + (b + shift)) * a
            p = p @ rot.T + origin
            keep = np.all((p >= lo) & (p < hi), axis=1)
            if keep.any():
                yield p[keep]


def lattice_in_box(a, basis, rot, lo, hi, shift=DEFAULT_SHIFT, origin=(0.0, 0.0, 0.0)) -> np.ndarray:
    """All lattice sites (fp64, lab frame) inside the half-open box [lo, hi)."""
    origin = np.asarray(origin, np.float64)
    parts = list(_sites_bbox(a, basis, rot, lo, hi, np.asarray(shift, np.float64), origin))
    if not parts:
        return np.zeros((0, 3))
    return np.concatenate(parts, axis=0)


def lattice_in_ball(a, basis, rot, centre, radius, shift=DEFAULT_SHIFT) -> np.ndarray:
    """All lattice sites (fp64, lab frame) within `radius` of `centre`."""
    centre = np.asarray(centre, np.float64)
    p = lattice_in_box(a, basis, rot, centre - radius, centre + radius, shift)
    d = p - centre
    return p[np.einsum("ij,ij->i", d, d) <= radius * radius]


def jitter_thin_shuffle(sites: np.ndarray, rng: np.random.Generator, eta: float, sigma_xyz,
                        extra: np.ndarray | None = None):
    """Bernoulli(eta) thinning, N(0, diag(sigma^2)) jitter in the lab frame, optional extra
    (background) points appended un-jittered, then a shuffle (APT order is not spatial).
    Returns (xyz float32 [N,3], perm-source index int64 [N]) where index >= len(kept) marks extras."""
    keep = rng.random(sites.shape[0]) < eta
    p = sites[keep]
    sig = np.broadcast_to(np.asarray(sigma_xyz, np.float64), (3,))
    p = p + rng.standard_normal(p.shape) * sig
    n_lattice = p.shape[0]
    if extra is not None and extra.shape[0]:
        p = np.concatenate([p, extra], axis=0)
    perm = rng.permutation(p.shape[0])
    return np.ascontiguousarray(p[perm].astype(np.float32)), perm, n_lattice, keep
