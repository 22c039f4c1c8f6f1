"""Thin ctypes binding of libaptsig (include/aptsig.h): argument marshalling only.

Every step of the hot path runs inside the CUDA library; torch is used for device memory and streams.
There is no fallback: if the shared library is missing or a call fails, an exception is raised.
Function names mirror the C ABI (apx_*); `Plan` is a convenience holder for the opaque handle.
"""
from __future__ import annotations
import ctypes as C
import os
import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.environ.get("APTSIG_LIB", os.path.join(_HERE, "libaptsig.so"))     # override: a development build of the library

APX_OK, APX_EINVAL, APX_ENOMEM, APX_ECUDA, APX_ESTATE, APX_ERANGE = 0, -1, -2, -3, -4, -5
APX_FLAG_FORCE_FFT, APX_FLAG_FORCE_MMA, APX_FLAG_NO_PAIRING, APX_FLAG_NORMALISE, APX_FLAG_LOCAL_MAX = 1, 2, 4, 8, 16
APX_PEAK_MAX, APX_PEAK_LOCAL_MAX, APX_MAX_SIGNATURES = 0, 1, 4

EXPORTS = ["apx_plan_create", "apx_plan_destroy", "apx_plan_constants", "apx_plan_path", "apx_plan_paired", "apx_last_cuda_error",
           "apx_plan_create_multi", "apx_plan_num_signatures", "apx_plan_reserve", "apx_ingest", "apx_query", "apx_run", "apx_run_host", "apx_debug_histograms",
           "apx_dirs_fibonacci", "apx_dirs_geodesic", "apx_dirs_antipodes", "apx_strerror", "apx_version"]
PEAK_EXPORTS = ["apx_peak_name", "apx_peak_measure"]          # include/aptsig_peaks.h
EXT_EXPORTS = ["apx_intensity_max", "apx_refine_select", "apx_refine_centres", "apx_indexer_create", "apx_indexer_destroy",
               "apx_indexer_nodes", "apx_indexer_lut", "apx_last_cuda_error_indexer", "apx_index", "apx_so3_grid_cubic", "apx_fsp", "apx_fsp_set_path", "apx_fsp_noalloc", "apx_fsp_noalloc_limits"]   # aptsig_ext.h
APX_INDEX_MAX_K = 8


class apx_plan_desc(C.Structure):
    _fields_ = [("R", C.c_float), ("B", C.c_int32), ("pad", C.c_int32), ("k_lo", C.c_int32), ("k_hi", C.c_int32),
                ("dirs", C.POINTER(C.c_float)), ("D", C.c_int32), ("type_mask", C.c_uint8 * 32),
                ("device", C.c_int32), ("flags", C.c_int32)]


class apx_sig_spec(C.Structure):
    _fields_ = [("type_mask", C.c_uint8 * 32), ("k_lo", C.c_int32), ("k_hi", C.c_int32), ("peak_mode", C.c_int32),
                ("normalise", C.c_int32)]


class apx_peak_result(C.Structure):
    _fields_ = [("sm_count", C.c_int), ("ms", C.c_float), ("median_cycles", C.c_double), ("warp_inst_per_s", C.c_double),
                ("warp_inst_per_clk_per_sm", C.c_double), ("sm_mhz_effective", C.c_double)]


class ApxError(RuntimeError):
    def __init__(self, status, where, cuda=None):
        self.status = status
        try:
            text = _lib().apx_strerror(status).decode()
        except Exception:
            text = "error"
        msg = f"{where}: {text} ({status})"
        if cuda is not None:
            msg += f" [cudaError {cuda}]"
        super().__init__(msg)


_LIB = None


def _lib():
    global _LIB
    if _LIB is None:
        if not os.path.exists(LIB_PATH):
            raise ImportError(f"{LIB_PATH} not built: run `python -m paper_2009_00735_b200.build` "
                              "(or __graft_entry__.build()); there is no CPU fallback")
        L = C.CDLL(LIB_PATH)
        vp, i64, i32 = C.c_void_p, C.c_int64, C.c_int32
        L.apx_plan_create.argtypes = [C.POINTER(apx_plan_desc), C.POINTER(vp)]
        L.apx_plan_create_multi.argtypes = [C.POINTER(apx_plan_desc), C.POINTER(apx_sig_spec), i32, C.POINTER(vp)]
        L.apx_plan_num_signatures.argtypes = [vp]
        L.apx_plan_destroy.argtypes = [vp]
        L.apx_plan_constants.argtypes = [vp, C.POINTER(C.c_float), C.POINTER(C.c_float), C.POINTER(C.c_float)]
        L.apx_plan_path.argtypes = [vp]
        L.apx_plan_paired.argtypes = [vp]
        L.apx_last_cuda_error.argtypes = [vp]
        L.apx_plan_reserve.argtypes = [vp, i64, i64]
        L.apx_ingest.argtypes = [vp, vp, vp, i64, vp]
        L.apx_query.argtypes = [vp, vp, i64, vp, vp, vp]
        L.apx_run.argtypes = [vp, vp, vp, i64, vp, i64, vp, vp, vp]
        L.apx_run_host.argtypes = [vp, vp, vp, i64, vp, i64, vp, vp]
        L.apx_debug_histograms.argtypes = [vp, C.POINTER(C.c_float), i32, i32, vp, vp]
        L.apx_dirs_fibonacci.argtypes = [i32, vp]
        L.apx_dirs_geodesic.argtypes = [i32, vp, C.POINTER(i32)]
        L.apx_dirs_antipodes.argtypes = [vp, i32, vp]
        L.apx_strerror.argtypes = [C.c_int]
        L.apx_strerror.restype = C.c_char_p
        L.apx_version.restype = C.c_char_p
        f32 = C.c_float
        L.apx_intensity_max.argtypes = [vp, vp, vp, i64, vp, vp]
        L.apx_refine_select.argtypes = [vp, vp, i64, f32, vp, vp, vp]
        L.apx_refine_centres.argtypes = [vp, vp, vp, vp, i64, f32, i32, vp, vp]
        L.apx_indexer_create.argtypes = [vp, i32, vp, i64, vp, i32, i32, C.POINTER(vp)]
        L.apx_indexer_destroy.argtypes = [vp]
        L.apx_indexer_nodes.argtypes = [vp, vp, vp]
        L.apx_indexer_lut.argtypes = [vp, i64, i64, vp]
        L.apx_last_cuda_error_indexer.argtypes = [vp]
        L.apx_index.argtypes = [vp, vp, vp, i64, i32, vp, vp, vp]
        L.apx_so3_grid_cubic.argtypes = [f32, vp, C.POINTER(i64)]
        L.apx_fsp.argtypes = [vp, vp, i64, f32, i32, vp, vp, vp]
        L.apx_fsp_set_path.argtypes = [vp, i32]
        L.apx_fsp_noalloc.argtypes = [vp, vp, i64, f32, i32, vp, vp, vp]
        L.apx_fsp_noalloc_limits.argtypes = [C.POINTER(i64), C.POINTER(i32), C.POINTER(i64)]
        for name in EXT_EXPORTS:
            getattr(L, name).restype = C.c_int
        L.apx_peak_name.argtypes = [C.c_int]
        L.apx_peak_name.restype = C.c_char_p
        L.apx_peak_measure.argtypes = [C.c_int, C.c_int, C.c_int, C.POINTER(apx_peak_result)]
        L.apx_peak_measure.restype = C.c_int
        for name in EXPORTS:
            if name not in ("apx_strerror", "apx_version"):
                getattr(L, name).restype = C.c_int
        _LIB = L
    return _LIB


def type_mask_bytes(accepted=None) -> bytes:
    m = bytearray(32)
    if accepted is None:
        m = bytearray(b"\xff" * 32)
    else:
        for t in accepted:
            m[t >> 3] |= 1 << (t & 7)
    return bytes(m)


def apx_version() -> str:
    return _lib().apx_version().decode()


def apx_dirs_fibonacci(D: int) -> np.ndarray:
    out = np.empty((D, 3), np.float32)
    rc = _lib().apx_dirs_fibonacci(D, out.ctypes.data)
    if rc:
        raise ApxError(rc, "apx_dirs_fibonacci")
    return out


def apx_dirs_geodesic(level: int) -> np.ndarray:
    n = C.c_int32(0)
    rc = _lib().apx_dirs_geodesic(level, None, C.byref(n))
    if rc:
        raise ApxError(rc, "apx_dirs_geodesic")
    out = np.empty((n.value, 3), np.float32)
    rc = _lib().apx_dirs_geodesic(level, out.ctypes.data, C.byref(n))
    if rc:
        raise ApxError(rc, "apx_dirs_geodesic")
    return out


def apx_dirs_antipodes(dirs: np.ndarray):
    """(symmetric, partner): partner[i] = index of the direction -dirs[i], or -1 (host only)."""
    d = np.ascontiguousarray(dirs, np.float32)
    partner = np.empty(len(d), np.int32)
    rc = _lib().apx_dirs_antipodes(d.ctypes.data, len(d), partner.ctypes.data)
    if rc < 0:
        raise ApxError(rc, "apx_dirs_antipodes")
    return bool(rc), partner


def apx_peak_name(test: int):
    n = _lib().apx_peak_name(int(test))
    return None if n is None else n.decode()


def apx_peak_measure(device: int, test: int, iters: int) -> dict:
    """One on-chip peak microbenchmark (include/aptsig_peaks.h) -> dict of the result struct's fields."""
    r = apx_peak_result()
    rc = _lib().apx_peak_measure(int(device), int(test), int(iters), C.byref(r))
    if rc:
        raise ApxError(rc, "apx_peak_measure")
    return {k: getattr(r, k) for k, _ in apx_peak_result._fields_}


def apx_so3_grid_cubic(spacing_deg: float) -> np.ndarray:
    """Orientation set of include/aptsig_ext.h: unit quaternions float32 [Ng, 4] (host only)."""
    n = C.c_int64(0)
    rc = _lib().apx_so3_grid_cubic(float(spacing_deg), None, C.byref(n))
    if rc:
        raise ApxError(rc, "apx_so3_grid_cubic")
    out = np.empty((n.value, 4), np.float32)
    rc = _lib().apx_so3_grid_cubic(float(spacing_deg), out.ctypes.data, C.byref(n))
    if rc:
        raise ApxError(rc, "apx_so3_grid_cubic")
    return out


def _is_np(t):
    return isinstance(t, np.ndarray)


def _arg(t, name, dtype, shape, device=None, optional=False):
    """Pointer of a torch tensor / numpy array after checking dtype, shape, contiguity and placement.
    device = CUDA ordinal the array must live on, or None for a HOST array (numpy or CPU tensor)."""
    if t is None:
        if optional:
            return None
        raise ApxError(APX_EINVAL, f"{name}: missing")
    want = np.dtype(dtype)
    if _is_np(t):
        if device is not None:
            raise ApxError(APX_EINVAL, f"{name}: expected a tensor on cuda:{device}, got a numpy array")
        have, contiguous, ptr = t.dtype, t.flags.c_contiguous, t.ctypes.data
    else:
        try:
            have = np.dtype(str(t.dtype).replace("torch.", ""))
        except TypeError:
            raise ApxError(APX_EINVAL, f"{name}: dtype {t.dtype}, expected {want}") from None
        contiguous, ptr = t.is_contiguous(), t.data_ptr()
        if device is None:
            if t.device.type != "cpu":
                raise ApxError(APX_EINVAL, f"{name}: expected a host array, got {t.device}")
        elif t.device.type != "cuda" or t.device.index != device:
            raise ApxError(APX_EINVAL, f"{name}: expected a tensor on cuda:{device}, got {t.device}")
    # 4-byte integer outputs may be int32 or uint32 (torch has no full uint32 support)
    same = have == want or (want == np.uint32 and have == np.int32)
    if not same:
        raise ApxError(APX_EINVAL, f"{name}: dtype {have}, expected {want}")
    if tuple(t.shape) != tuple(shape):
        raise ApxError(APX_EINVAL, f"{name}: shape {tuple(t.shape)}, expected {tuple(shape)}")
    if not contiguous:
        raise ApxError(APX_EINVAL, f"{name}: must be contiguous")
    return ptr


class Plan:
    """Owner of one apx_plan*. Methods are 1:1 with the C entry points."""

    def __init__(self, R, B, dirs, pad=1, k_lo=0, k_hi=0, accepted_types=None, device=0, flags=0, specs=None):
        """specs = None: one signature (accepted_types, k_lo, k_hi; apx_plan_create).  specs = list of dicts with keys
        accepted_types / k_lo / k_hi / peak_mode / normalise: a multi-signature plan (apx_plan_create_multi); the outputs of
        apx_query / apx_run / apx_run_host then carry a leading axis of len(specs)."""
        dirs = np.ascontiguousarray(dirs, np.float32).reshape(-1, 3)
        d = apx_plan_desc()
        d.R, d.B, d.pad, d.k_lo, d.k_hi = float(R), int(B), int(pad), int(k_lo), int(k_hi)
        d.dirs = dirs.ctypes.data_as(C.POINTER(C.c_float))
        d.D = dirs.shape[0]
        d.type_mask = (C.c_uint8 * 32).from_buffer_copy(type_mask_bytes(accepted_types))
        d.device, d.flags = int(device), int(flags)
        self._h = C.c_void_p()
        self.B, self.D, self.device = int(B), dirs.shape[0], int(device)
        self.k_lo, self.k_hi = (1, B // 2) if (k_lo == 0 and k_hi == 0) else (int(k_lo), int(k_hi))
        self.S = 1 if specs is None else len(specs)
        if specs is None:
            rc = _lib().apx_plan_create(C.byref(d), C.byref(self._h))
        else:
            arr = (apx_sig_spec * max(1, len(specs)))()
            for a, sp in zip(arr, specs):
                a.type_mask = (C.c_uint8 * 32).from_buffer_copy(type_mask_bytes(sp.get("accepted_types")))
                a.k_lo, a.k_hi = int(sp.get("k_lo", 0)), int(sp.get("k_hi", 0))
                a.peak_mode, a.normalise = int(sp.get("peak_mode", APX_PEAK_MAX)), int(bool(sp.get("normalise", False)))
            rc = _lib().apx_plan_create_multi(C.byref(d), arr, len(specs), C.byref(self._h))
        if rc:
            self._h = C.c_void_p()
            raise ApxError(rc, "apx_plan_create" if specs is None else "apx_plan_create_multi")
        self._multi = specs is not None

    def _check(self, rc, where):
        if rc:
            raise ApxError(rc, where, _lib().apx_last_cuda_error(self._h) if rc == APX_ECUDA else None)

    def apx_plan_constants(self):
        r2, s, f = C.c_float(), C.c_float(), C.c_float()
        self._check(_lib().apx_plan_constants(self._h, C.byref(r2), C.byref(s), C.byref(f)), "apx_plan_constants")
        return np.float32(r2.value), np.float32(s.value), np.float32(f.value)

    def apx_plan_num_signatures(self) -> int:
        return _lib().apx_plan_num_signatures(self._h)

    def _sig_shape(self, M):
        return (self.S, M, self.D, 2) if self._multi else (M, self.D, 2)

    def _cnt_shape(self, M):
        return (self.S, M) if self._multi else (M,)

    def apx_plan_path(self) -> int:
        return _lib().apx_plan_path(self._h)

    def apx_plan_paired(self) -> int:
        return _lib().apx_plan_paired(self._h)

    def _stream(self, stream=None):
        import torch
        return (torch.cuda.current_stream(self.device) if stream is None else stream).cuda_stream

    def apx_plan_reserve(self, N_max, M_max):
        self._check(_lib().apx_plan_reserve(self._h, int(N_max), int(M_max)), "apx_plan_reserve")

    def apx_ingest(self, xyz, types=None, stream=None):
        N, dev = int(xyz.shape[0]), self.device
        self._check(_lib().apx_ingest(self._h, _arg(xyz, "xyz", np.float32, (N, 3), dev),
                                      _arg(types, "types", np.uint8, (N,), dev, optional=True), N,
                                      self._stream(stream)), "apx_ingest")

    def apx_query(self, centres, sig, counts=None, stream=None):
        M, dev = int(centres.shape[0]), self.device
        self._check(_lib().apx_query(self._h, _arg(centres, "centres", np.float32, (M, 3), dev), M,
                                     _arg(sig, "sig", np.float32, self._sig_shape(M), dev),
                                     _arg(counts, "counts", np.uint32, self._cnt_shape(M), dev, optional=True),
                                     self._stream(stream)), "apx_query")

    def apx_run(self, xyz, types, centres, sig, counts=None, stream=None):
        N, M, dev = int(xyz.shape[0]), int(centres.shape[0]), self.device
        self._check(_lib().apx_run(self._h, _arg(xyz, "xyz", np.float32, (N, 3), dev),
                                   _arg(types, "types", np.uint8, (N,), dev, optional=True), N,
                                   _arg(centres, "centres", np.float32, (M, 3), dev), M,
                                   _arg(sig, "sig", np.float32, self._sig_shape(M), dev),
                                   _arg(counts, "counts", np.uint32, self._cnt_shape(M), dev, optional=True),
                                   self._stream(stream)), "apx_run")

    def apx_run_host(self, xyz, types, centres, sig, counts=None):
        """All arguments are HOST arrays (numpy, or pinned CPU torch tensors)."""
        N, M = int(xyz.shape[0]), int(centres.shape[0])
        self._check(_lib().apx_run_host(self._h, _arg(xyz, "xyz", np.float32, (N, 3)),
                                        _arg(types, "types", np.uint8, (N,), optional=True), N,
                                        _arg(centres, "centres", np.float32, (M, 3)), M,
                                        _arg(sig, "sig", np.float32, self._sig_shape(M)),
                                        _arg(counts, "counts", np.uint32, self._cnt_shape(M), optional=True)), "apx_run_host")

    def apx_debug_histograms(self, centre3, d0, nd, out, stream=None):
        c = (C.c_float * 3)(*[float(v) for v in centre3])
        self._check(_lib().apx_debug_histograms(self._h, c, int(d0), int(nd),
                                                _arg(out, "out", np.uint32, (int(nd), self.B), self.device),
                                                self._stream(stream)), "apx_debug_histograms")

    # ---- include/aptsig_ext.h: grid refinement (NEXT-4) -------------------------------------------------------
    def apx_intensity_max(self, sig, counts, kappa_max, stream=None):
        M, dev = int(sig.shape[0]), self.device
        self._check(_lib().apx_intensity_max(self._h, _arg(sig, "sig", np.float32, (M, self.D, 2), dev),
                                             _arg(counts, "counts", np.uint32, (M,), dev), M,
                                             _arg(kappa_max, "kappa_max", np.float32, (M,), dev), self._stream(stream)),
                    "apx_intensity_max")

    def apx_refine_select(self, kappa_max, kappa, selected, n_selected, stream=None):
        M, dev = int(kappa_max.shape[0]), self.device
        self._check(_lib().apx_refine_select(self._h, _arg(kappa_max, "kappa_max", np.float32, (M,), dev), M, float(kappa),
                                             _arg(selected, "selected", np.uint32, (M,), dev),
                                             _arg(n_selected, "n_selected", np.uint32, (1,), dev), self._stream(stream)),
                    "apx_refine_select")

    def apx_refine_centres(self, centres, selected, n_selected, max_selected, spacing, split, out, stream=None):
        M, dev = int(centres.shape[0]), self.device
        self._check(_lib().apx_refine_centres(self._h, _arg(centres, "centres", np.float32, (M, 3), dev),
                                              _arg(selected, "selected", np.uint32, (int(selected.shape[0]),), dev),
                                              _arg(n_selected, "n_selected", np.uint32, (1,), dev), int(max_selected),
                                              float(spacing), int(split),
                                              _arg(out, "out", np.float32, (int(max_selected) * int(split) ** 3, 3), dev),
                                              self._stream(stream)), "apx_refine_centres")

    # ---- include/aptsig_ext.h: reciprocal space method (NEXT-3) ------------------------------------------------
    def apx_fsp_set_path(self, path):
        self._check(_lib().apx_fsp_set_path(self._h, int(path)), "apx_fsp_set_path")

    def apx_fsp(self, centres, k_max, L, out, counts=None, stream=None):
        M, dev, L = int(centres.shape[0]), self.device, int(L)
        self._check(_lib().apx_fsp(self._h, _arg(centres, "centres", np.float32, (M, 3), dev), M, float(k_max), L,
                                   _arg(out, "out", np.float32, (M, L, L, L), dev),
                                   _arg(counts, "counts", np.uint32, (M,), dev, optional=True), self._stream(stream)), "apx_fsp")

    def apx_fsp_noalloc(self, centres, k_max, L, out, counts=None, stream=None):
        """apx_fsp without any allocation: scratch in the library's static device array (limits: apx_fsp_noalloc_limits)."""
        M, dev, L = int(centres.shape[0]), self.device, int(L)
        rc = _lib().apx_fsp_noalloc(self._h, _arg(centres, "centres", np.float32, (M, 3), dev), M, float(k_max), L,
                                    _arg(out, "out", np.float32, (M, L, L, L), dev),
                                    _arg(counts, "counts", np.uint32, (M,), dev, optional=True), self._stream(stream))
        where = "apx_fsp_noalloc"
        if rc == APX_ERANGE:
            max_m, max_l, nbytes = apx_fsp_noalloc_limits()
            where += f" (M = {M}, L = {L}; the static scratch of {nbytes} bytes serves M <= {max_m}, L <= {max_l}: use apx_fsp)"
        self._check(rc, where)

    def apx_plan_destroy(self):
        if self._h:
            _lib().apx_plan_destroy(self._h)
            self._h = C.c_void_p()

    def __del__(self):
        try:
            self.apx_plan_destroy()
        except Exception:
            pass


def apx_fsp_noalloc_limits():
    """(max M, max L, bytes of the static device scratch array) of apx_fsp_noalloc."""
    m, l, b = C.c_int64(), C.c_int32(), C.c_int64()
    _lib().apx_fsp_noalloc_limits(C.byref(m), C.byref(l), C.byref(b))
    return m.value, l.value, b.value


class Indexer:
    """Owner of one apx_indexer* (include/aptsig_ext.h, NEXT-1): one crystal-structure candidate."""

    def __init__(self, dirs, quats, ref_image, n_hat, device=0):
        dirs = np.ascontiguousarray(dirs, np.float32).reshape(-1, 3)
        quats = np.ascontiguousarray(quats, np.float32).reshape(-1, 4)
        ref = np.ascontiguousarray(ref_image, np.float32).reshape(-1)
        if ref.shape[0] != dirs.shape[0]:
            raise ApxError(APX_EINVAL, "Indexer: ref_image must have one intensity per direction")
        self.D, self.Ng, self.n_hat, self.device = dirs.shape[0], quats.shape[0], int(n_hat), int(device)
        self._h = C.c_void_p()
        rc = _lib().apx_indexer_create(dirs.ctypes.data, self.D, quats.ctypes.data, self.Ng, ref.ctypes.data, self.n_hat,
                                       self.device, C.byref(self._h))
        if rc:
            self._h = C.c_void_p()
            raise ApxError(rc, "apx_indexer_create")

    def _check(self, rc, where):
        if rc:
            raise ApxError(rc, where, _lib().apx_last_cuda_error_indexer(self._h) if rc == APX_ECUDA else None)

    def apx_indexer_nodes(self):
        nodes, ref = np.empty(self.n_hat, np.int32), np.empty(self.n_hat, np.float32)
        self._check(_lib().apx_indexer_nodes(self._h, nodes.ctypes.data, ref.ctypes.data), "apx_indexer_nodes")
        return nodes, ref

    def apx_indexer_lut(self, g0, ng):
        out = np.empty((int(ng), self.n_hat), np.int32)
        self._check(_lib().apx_indexer_lut(self._h, int(g0), int(ng), out.ctypes.data), "apx_indexer_lut")
        return out

    def apx_index(self, sig, counts, best_delta, best_g, stream=None):
        import torch
        M, K, dev = int(sig.shape[0]), int(best_delta.shape[1]), self.device
        st = (torch.cuda.current_stream(dev) if stream is None else stream).cuda_stream
        self._check(_lib().apx_index(self._h, _arg(sig, "sig", np.float32, (M, self.D, 2), dev),
                                     _arg(counts, "counts", np.uint32, (M,), dev, optional=True), M, K,
                                     _arg(best_delta, "best_delta", np.float32, (M, K), dev),
                                     _arg(best_g, "best_g", np.int32, (M, K), dev), st), "apx_index")

    def apx_indexer_destroy(self):
        if self._h:
            _lib().apx_indexer_destroy(self._h)
            self._h = C.c_void_p()

    def __del__(self):
        try:
            self.apx_indexer_destroy()
        except Exception:
            pass
