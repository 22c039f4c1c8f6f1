"""The five BASELINE.json configs as seeded synthetic workloads (SURVEY.md section 8(d) recipe).

Only inputs are built here: ion cloud, ion types, centres, and the scalar plan parameters.
Direction grids are NOT built here (they are a step of the hot path, built separately by the oracle
and by the CUDA library); a Workload only names which grid it wants.
"""
from __future__ import annotations
from dataclasses import dataclass, field
import math
import numpy as np
from .lattices import (fcc_basis, bcc_basis, random_rotation, lattice_in_box, lattice_in_ball,
                       jitter_thin_shuffle)

A_AL = 0.405     # nm, fcc Al
A_W = 0.3165     # nm, bcc W    (BASELINE.json config 3)
SEED0 = 200900735


@dataclass
class Workload:
    name: str
    xyz: np.ndarray            # float32 [N,3]
    types: np.ndarray          # uint8   [N]
    centres: np.ndarray        # float32 [M,3]
    R: float
    B: int
    grid: tuple                # ("fibonacci", D) or ("geodesic", level)
    D: int
    window: tuple              # (k_lo, k_hi) bench window
    masks: list = field(default_factory=lambda: [None])   # list of accepted-type sets (None = all)
    meta: dict = field(default_factory=dict)


def window_for(R: float, B: int, pad: int = 1, d_hi: float = 0.26, d_lo: float = 0.12):
    """Spectral-bin window covering plane spacings d_lo..d_hi nm: k = 2(R + pad*dR)/d."""
    dR = R / (B // 2 - 1) if pad else 0.0
    span = 2.0 * (R + dR)
    return int(math.floor(span / d_hi)), int(math.ceil(span / d_lo))


def _grid_centres(lo, hi, step):
    ax = np.arange(lo, hi + 1e-9, step)
    g = np.stack(np.meshgrid(ax, ax, ax, indexing="ij"), axis=-1).reshape(-1, 3)
    return np.ascontiguousarray(g.astype(np.float32))


def _cfg1(rng, scale):
    R, sigma = 1.0, 0.05
    rot = random_rotation(rng)
    sites = lattice_in_ball(A_AL, fcc_basis, rot, (0, 0, 0), R + 4 * sigma + 0.3)
    xyz, _, _, _ = jitter_thin_shuffle(sites, rng, 0.5, sigma)
    return Workload("cfg1_single_point", xyz, np.zeros(len(xyz), np.uint8),
                    np.zeros((1, 3), np.float32), R, 256, ("fibonacci", 1000), 1000,
                    window_for(R, 256), meta={"rot": rot})


def _cfg2(rng, scale):
    R = 2.0
    rot = random_rotation(rng)
    sites = lattice_in_box(A_AL, fcc_basis, rot, (0, 0, 0), (20, 20, 20))
    xyz, _, _, _ = jitter_thin_shuffle(sites, rng, 0.5, (0.05, 0.05, 0.02))
    centres = _grid_centres(1.0, 19.0, 2.0)
    return Workload("cfg2_single_crystal", xyz, np.zeros(len(xyz), np.uint8), centres, R, 1024,
                    ("fibonacci", 10000), 10000, window_for(R, 1024), meta={"rot": rot})


def _cfg3(rng, scale):
    R, L = 2.0, 30.0
    rot_al, rot_w = random_rotation(rng), random_rotation(rng)
    s_al = lattice_in_box(A_AL, fcc_basis, rot_al, (0, 0, 0), (L / 2, L, L))
    s_w = lattice_in_box(A_W, bcc_basis, rot_w, (L / 2, 0, 0), (L, L, L))
    sites = np.concatenate([s_al, s_w])
    phase = np.concatenate([np.zeros(len(s_al), np.uint8), np.ones(len(s_w), np.uint8)])
    xyz, perm, n_lat, keep = jitter_thin_shuffle(sites, rng, 0.5, 0.06)
    types = phase[keep][perm]
    relabel = rng.random(len(types)) < 0.10          # "optionally 10 % relabelled at random"
    types = np.where(relabel, rng.integers(0, 2, len(types)).astype(np.uint8), types).astype(np.uint8)
    centres = _grid_centres(0.5, L - 0.5, 1.0)
    return Workload("cfg3_bicrystal", xyz, types, centres, R, 1024, ("geodesic", 6), 40962,
                    window_for(R, 1024), masks=[{0}, {1}], meta={"rot_al": rot_al, "rot_w": rot_w})


def _cfg4(rng, scale):
    """64 Voronoi grains in a 60^3 box (scale < 1 shrinks the box edge, keeping the grain density)."""
    from scipy.spatial import cKDTree
    R = 2.0
    L = 60.0 * scale
    n_grains = max(2, int(round(64 * scale ** 3)))
    seeds = rng.random((n_grains, 3)) * L
    rots = [random_rotation(rng) for _ in range(n_grains)]
    tree = cKDTree(seeds)
    # per-grain bounding boxes from a coarse probe grid (+ margin), then exact nearest-seed assignment
    ax = np.arange(0.25, L, 0.5)
    probe = np.stack(np.meshgrid(ax, ax, ax, indexing="ij"), -1).reshape(-1, 3)
    owner = tree.query(probe)[1]
    parts = []
    for g in range(n_grains):
        pts = probe[owner == g]
        if len(pts) == 0:
            continue
        lo = np.maximum(pts.min(0) - 1.0, 0.0)
        hi = np.minimum(pts.max(0) + 1.0, L)
        s = lattice_in_box(A_AL, fcc_basis, rots[g], lo, hi, origin=seeds[g])
        s = s[rng.random(len(s)) < 0.37]              # thin early (memory); eta applied once here
        s = s[tree.query(s)[1] == g]
        parts.append(s)
    sites = np.concatenate(parts)
    xyz, _, _, _ = jitter_thin_shuffle(sites, rng, 1.1, 0.07)   # eta already applied above
    centres = _grid_centres(2.5, L - 2.5, 1.0)
    return Workload("cfg4_nanocrystal", xyz, np.zeros(len(xyz), np.uint8), centres, R, 1024,
                    ("geodesic", 6), 40962, window_for(R, 1024), meta={"seeds": seeds, "L": L})


def _cfg5(rng, scale):
    R = 3.0
    L = 40.0 * scale
    rot = random_rotation(rng)
    sites = lattice_in_box(A_AL, fcc_basis, rot, (0, 0, 0), (L, L, L))
    site_type = (rng.random(len(sites)) < 0.03).astype(np.uint8)      # 3 at% Sc on random sites
    n_bg = int(round(0.05 * 0.37 * len(sites)))
    bg = rng.random((n_bg, 3)) * L
    bg_type = (rng.random(n_bg) < 0.03).astype(np.uint8)
    xyz, perm, n_lat, keep = jitter_thin_shuffle(sites, rng, 0.37, 0.10, extra=bg)
    types = np.concatenate([site_type[keep], bg_type])[perm].astype(np.uint8)
    centres = _grid_centres(0.5, L - 0.5, 1.0)
    return Workload("cfg5_dilute_alloy", xyz, types, centres, R, 2048, ("geodesic", 6), 40962,
                    window_for(R, 2048), masks=[{0}], meta={"rot": rot, "L": L})


CONFIGS = {1: _cfg1, 2: _cfg2, 3: _cfg3, 4: _cfg4, 5: _cfg5}


def make_config(cfg: int, scale: float = 1.0) -> Workload:
    """Build config `cfg` (1..5) with seed 200900735+cfg. `scale` < 1 shrinks the box edge of
    configs 4 and 5 (same densities, noise, R, B, D) for parity tests; the bench uses scale = 1."""
    rng = np.random.Generator(np.random.PCG64(SEED0 + cfg))
    w = CONFIGS[cfg](rng, scale)
    w.meta["cfg"] = cfg
    w.meta["scale"] = scale
    return w
