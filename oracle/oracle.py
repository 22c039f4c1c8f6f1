"""ctypes front-end of the CPU oracle (oracle/aptsig_oracle.c) + the oracle's own direction grids.

TEST INFRASTRUCTURE ONLY (see the C file's header): importable from tests/, __graft_entry__.smoke()
and bench.py's cpu_baseline / --impl reference legs. Never import paper_2009_00735_b200 from here.
"""
from __future__ import annotations
import ctypes as C
import math
import os
import sys
import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, _HERE)
import build as _build  # noqa: E402  (oracle/build.py)
sys.path.pop(0)

_lib = None
_f32p = np.ctypeslib.ndpointer(np.float32, flags="C_CONTIGUOUS")
_u8p = np.ctypeslib.ndpointer(np.uint8, flags="C_CONTIGUOUS")
_u32p = np.ctypeslib.ndpointer(np.uint32, flags="C_CONTIGUOUS")
_f64p = np.ctypeslib.ndpointer(np.float64, flags="C_CONTIGUOUS")


def lib():
    global _lib
    if _lib is None:
        L = C.CDLL(_build.build())
        L.orc_constants.argtypes = [C.c_float, C.c_int, C.c_int, C.POINTER(C.c_float), C.POINTER(C.c_float)]
        L.orc_constants.restype = C.c_int
        L.orc_members.argtypes = [_f32p, C.c_void_p, C.c_int64, _f32p, C.c_float, _u8p, C.c_void_p, C.c_int64]
        L.orc_members.restype = C.c_int64
        L.orc_histograms.argtypes = [_f32p, C.c_void_p, C.c_int64, _f32p, _f32p, C.c_int, C.c_int,
                                     C.c_float, C.c_int, C.c_int, _u8p, _u32p]
        L.orc_histograms.restype = C.c_int64
        L.orc_hist_one.argtypes = [_f32p, C.c_int64, _f32p, C.c_int, _u32p]
        L.orc_hist_one.restype = None
        L.orc_scale_dirs.argtypes = [_f32p, C.c_int, C.c_float, _f32p]
        L.orc_scale_dirs.restype = None
        L.orc_amp_at.argtypes = [_u32p, C.c_int, C.c_int]
        L.orc_amp_at.restype = C.c_double
        L.orc_spectrum.argtypes = [_u32p, C.c_int, _f64p]
        L.orc_spectrum.restype = None
        L.orc_signatures.argtypes = [_f32p, C.c_void_p, C.c_int64, _f32p, C.c_int64, _f32p, C.c_int,
                                     C.c_float, C.c_int, C.c_int, C.c_int, C.c_int, _u8p,
                                     _f32p, C.c_void_p, C.c_void_p, C.c_int]
        L.orc_signatures.restype = C.c_int
        L.orc_num_threads.restype = C.c_int
        _lib = L
    return _lib


def type_mask(accepted=None) -> np.ndarray:
    """256-bit mask as uint8[32]; bit t set = ion type t accepted. None = all types."""
    m = np.zeros(32, np.uint8)
    if accepted is None:
        m[:] = 0xFF
    else:
        for t in accepted:
            m[t >> 3] |= np.uint8(1 << (t & 7))
    return m


def _types_ptr(types):
    if types is None:
        return None
    assert types.dtype == np.uint8 and types.flags.c_contiguous
    return types.ctypes.data


def constants(R, B, pad=1):
    r2, s = C.c_float(), C.c_float()
    rc = lib().orc_constants(R, B, pad, C.byref(r2), C.byref(s))
    if rc:
        raise ValueError("orc_constants: invalid R/B/pad")
    return np.float32(r2.value), np.float32(s.value)


def members(xyz, types, centre, R, accepted=None):
    """Relative positions d = p - c (float32 [N_c,3]) of accepted ions in the closed ball."""
    xyz = np.ascontiguousarray(xyz, np.float32)
    c = np.ascontiguousarray(centre, np.float32)
    R2 = np.float32(np.float32(R) * np.float32(R))
    m = type_mask(accepted)
    n = lib().orc_members(xyz, _types_ptr(types), len(xyz), c, R2, m, None, 0)
    rel = np.zeros((max(n, 1), 3), np.float32)
    lib().orc_members(xyz, _types_ptr(types), len(xyz), c, R2, m, rel.ctypes.data, n)
    return rel[:n]


def histograms(xyz, types, centre, dirs, R, B, pad=1, accepted=None, d0=0, nd=None):
    xyz = np.ascontiguousarray(xyz, np.float32)
    dirs = np.ascontiguousarray(dirs, np.float32)
    nd = len(dirs) - d0 if nd is None else nd
    out = np.zeros((nd, B), np.uint32)
    n = lib().orc_histograms(xyz, _types_ptr(types), len(xyz), np.ascontiguousarray(centre, np.float32),
                             dirs, d0, nd, R, B, pad, type_mask(accepted), out)
    if n < 0:
        raise ValueError(f"orc_histograms failed: {n}")
    return out, int(n)


def spectrum(h, B=None):
    h = np.ascontiguousarray(h, np.uint32)
    B = len(h) if B is None else B
    amp = np.zeros(B // 2 + 1, np.float64)
    lib().orc_spectrum(h, B, amp)
    return amp


def signatures(xyz, types, centres, dirs, R, B, pad=1, k_lo=0, k_hi=0, accepted=None,
               want_window=False, nthreads=0):
    """-> sig float32 [M,D,2], counts uint32 [M], (winamp float64 [M,D,W] if want_window)."""
    xyz = np.ascontiguousarray(xyz, np.float32)
    centres = np.ascontiguousarray(centres, np.float32).reshape(-1, 3)
    dirs = np.ascontiguousarray(dirs, np.float32)
    M, D = len(centres), len(dirs)
    sig = np.zeros((M, D, 2), np.float32)
    counts = np.zeros(M, np.uint32)
    klo, khi = (1, B // 2) if (k_lo == 0 and k_hi == 0) else (k_lo, k_hi)
    win = np.zeros((M, D, khi - klo + 1), np.float64) if want_window else None
    rc = lib().orc_signatures(xyz, _types_ptr(types), len(xyz), centres, M, dirs, D, R, B, pad,
                              k_lo, k_hi, type_mask(accepted), sig, counts.ctypes.data,
                              win.ctypes.data if want_window else None, nthreads)
    if rc:
        raise ValueError(f"orc_signatures failed: {rc}")
    return (sig, counts, win) if want_window else (sig, counts)


def num_threads() -> int:
    return int(lib().orc_num_threads())


# ---------------------------------------------------------------------------------------------
# Direction grids (step a3), the oracle's own construction in fp64 -> fp32.
# ---------------------------------------------------------------------------------------------
def dirs_fibonacci(D: int) -> np.ndarray:
    """Fibonacci sphere (BASELINE.json configs 1-2; reading #14):
    z_i = 1 - (2i+1)/D, phi_i = i*pi*(3-sqrt 5), n = (sqrt(1-z^2) cos phi, sqrt(1-z^2) sin phi, z)."""
    out = np.zeros((D, 3), np.float64)
    ga = math.pi * (3.0 - math.sqrt(5.0))
    for i in range(D):
        z = 1.0 - (2.0 * i + 1.0) / D
        r = math.sqrt(max(0.0, 1.0 - z * z))
        phi = i * ga
        out[i] = (r * math.cos(phi), r * math.sin(phi), z)
    return out.astype(np.float32)


def dirs_geodesic(level: int) -> np.ndarray:
    """Geodesic sphere (N_v = 40 962 = 10*4^6 + 2 at level 6; reading #13):
    icosahedron (0,+-1,+-phi)/norm and cyclic permutations, `level` rounds of edge-midpoint 4-way
    subdivision, midpoints re-normalised and de-duplicated; order = 12 base vertices, then midpoints
    in creation order (faces in order, edges (a,b),(b,c),(c,a))."""
    phi = (1.0 + math.sqrt(5.0)) / 2.0
    v = [(-1, phi, 0), (1, phi, 0), (-1, -phi, 0), (1, -phi, 0),
         (0, -1, phi), (0, 1, phi), (0, -1, -phi), (0, 1, -phi),
         (phi, 0, -1), (phi, 0, 1), (-phi, 0, -1), (-phi, 0, 1)]
    verts = [tuple(np.array(p, np.float64) / math.sqrt(1 + phi * phi)) for p in v]
    faces = [(0, 11, 5), (0, 5, 1), (0, 1, 7), (0, 7, 10), (0, 10, 11),
             (1, 5, 9), (5, 11, 4), (11, 10, 2), (10, 7, 6), (7, 1, 8),
             (3, 9, 4), (3, 4, 2), (3, 2, 6), (3, 6, 8), (3, 8, 9),
             (4, 9, 5), (2, 4, 11), (6, 2, 10), (8, 6, 7), (9, 8, 1)]
    for _ in range(level):
        cache = {}
        new_faces = []

        def mid(a, b):
            key = (a, b) if a < b else (b, a)
            if key not in cache:
                p = np.array(verts[a]) + np.array(verts[b])
                p /= np.linalg.norm(p)
                verts.append(tuple(p))
                cache[key] = len(verts) - 1
            return cache[key]

        for (a, b, c) in faces:
            ab, bc, ca = mid(a, b), mid(b, c), mid(c, a)
            new_faces += [(a, ab, ca), (b, bc, ab), (c, ca, bc), (ab, bc, ca)]
        faces = new_faces
    return np.array(verts, np.float64).astype(np.float32)
