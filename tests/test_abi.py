"""Host-side checks of the C ABI (no GPU): the library loads and exports every symbol declared in
include/aptsig.h; host-only entry points (direction grids, strerror) behave; and the library's
direction grids agree with the oracle's independent construction."""
import ctypes as C
import os
import re

import numpy as np
import pytest

import paper_2009_00735_b200 as apx
from paper_2009_00735_b200 import build as lib_build
from oracle import oracle as O

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    return C.CDLL(lib_build.build())


def test_every_declared_symbol_is_exported(lib):
    for header, exports in (("aptsig.h", apx.EXPORTS), ("aptsig_peaks.h", apx.PEAK_EXPORTS), ("aptsig_ext.h", apx.EXT_EXPORTS)):
        hdr = open(os.path.join(ROOT, "include", header)).read()
        hdr = re.sub(r"/\*.*?\*/", "", hdr, flags=re.S)
        declared = set(re.findall(r"\b(apx_[a-z_0-9]+)\s*\(", hdr))
        assert declared == set(exports), declared ^ set(exports)
        for name in declared:
            assert getattr(lib, name) is not None


def test_strerror_and_version():
    assert "aptsig" in apx.apx_version()
    from paper_2009_00735_b200.binding import _lib
    assert _lib().apx_strerror(0) == b"ok"
    assert b"invalid" in _lib().apx_strerror(apx.APX_EINVAL)


def test_fibonacci_matches_oracle_grid():
    for D in (1, 7, 1000):
        a, b = apx.apx_dirs_fibonacci(D), O.dirs_fibonacci(D)
        np.testing.assert_allclose(a, b, rtol=0, atol=2e-7)
    with pytest.raises(apx.ApxError):
        apx.apx_dirs_fibonacci(0)


def test_geodesic_matches_oracle_grid():
    for level in (0, 1, 3):
        a, b = apx.apx_dirs_geodesic(level), O.dirs_geodesic(level)
        assert a.shape == b.shape == (10 * 4 ** level + 2, 3)
        np.testing.assert_allclose(a, b, rtol=0, atol=2e-7)
    assert apx.apx_dirs_geodesic(6).shape == (40962, 3)
    with pytest.raises(apx.ApxError):
        apx.apx_dirs_geodesic(9)


def test_plan_create_rejects_bad_arguments_before_touching_cuda():
    d = np.array([[0, 0, 1]], np.float32)
    for kw in (dict(R=-1.0, B=256), dict(R=1.0, B=300), dict(R=1.0, B=128), dict(R=1.0, B=8192),
               dict(R=1.0, B=256, pad=2), dict(R=1.0, B=256, k_lo=5, k_hi=3), dict(R=1.0, B=256, k_lo=1, k_hi=129)):
        with pytest.raises(apx.ApxError) as ei:
            apx.Plan(dirs=d, **kw)
        assert ei.value.status == apx.APX_EINVAL


def test_antipodal_partners_of_direction_grids():
    """The geodesic grid (the paper's mesh, L60) is antipodally symmetric bit for bit -- what the half-grid mode of the
    tensor-core kernel relies on; a Fibonacci grid is not; duplicates and self-partners are rejected."""
    for level in (0, 1, 3):
        d = apx.apx_dirs_geodesic(level)
        sym, partner = apx.apx_dirs_antipodes(d)
        assert sym and (partner >= 0).all() and (partner[partner] == np.arange(len(d))).all()
        assert (d[partner] == -d).all()                       # numerically: -0.0 == +0.0
    sym, partner = apx.apx_dirs_antipodes(O.dirs_fibonacci(1000))
    assert not sym and (partner == -1).all()
    d = apx.apx_dirs_geodesic(1)
    sym, _ = apx.apx_dirs_antipodes(np.concatenate([d, d[:1]]))          # a duplicate
    assert not sym
    sym, partner = apx.apx_dirs_antipodes(np.array([[0, 0, 0], [1, 0, 0], [-1, 0, 0]], np.float32))
    assert not sym and partner[0] == -1 and partner[1] == 2 and partner[2] == 1
    # scaling by the plan's s (one fp32 multiply per component) keeps the pairs exact
    sym, _ = apx.apx_dirs_antipodes((apx.apx_dirs_geodesic(4) * np.float32(255.5)).astype(np.float32))
    assert sym


def test_binding_argument_checks_host_side():
    """binding._arg: dtype / shape / contiguity / placement checks (the host-array half runs without a GPU)."""
    from paper_2009_00735_b200.binding import _arg
    a = np.zeros((5, 3), np.float32)
    assert _arg(a, "xyz", np.float32, (5, 3)) == a.ctypes.data
    assert _arg(None, "types", np.uint8, (5,), optional=True) is None
    assert _arg(np.zeros(4, np.int32), "counts", np.uint32, (4,)) is not None      # int32 storage for uint32 counts
    for bad in (lambda: _arg(a.astype(np.float64), "xyz", np.float32, (5, 3)),
                lambda: _arg(a, "xyz", np.float32, (6, 3)),
                lambda: _arg(a[:, ::-1], "xyz", np.float32, (5, 3)),
                lambda: _arg(a, "xyz", np.float32, (5, 3), device=0),
                lambda: _arg(None, "xyz", np.float32, (5, 3))):
        with pytest.raises(apx.ApxError) as ei:
            bad()
        assert ei.value.status == apx.APX_EINVAL


def test_so3_grid_matches_oracle_grid():
    """The library's orientation set (host) against the oracle's own construction of reading #23."""
    from oracle import next_oracle as X
    for spacing in (10.0, 5.0):
        a, b = apx.apx_so3_grid_cubic(spacing), X.so3_grid_cubic(spacing)
        assert a.shape == b.shape
        np.testing.assert_allclose(a, b, rtol=0, atol=1e-7)
    with pytest.raises(apx.ApxError):
        apx.apx_so3_grid_cubic(0.0)
