"""Comparator shared by the GPU parity tests: north_star tolerances, written out.
  amplitudes : |A_gpu - A_or| <= 1e-4 * A_or + 1e-6 * N_c
  peak bin   : equal, or (tie rule, reading #9) the oracle's amplitude at the GPU's bin is
               within 1e-4 relative of the oracle's maximum
  counts     : bit-exact
"""
import numpy as np


def run_gpu(apx, w, dirs, centres, accepted=None, window=None, flags=0, pad=1, split=False):
    import torch
    dev = torch.device("cuda:0")
    k_lo, k_hi = window if window is not None else (0, 0)
    plan = apx.Plan(w.R, w.B, dirs, pad=pad, k_lo=k_lo, k_hi=k_hi, accepted_types=accepted, device=0, flags=flags)
    xyz = torch.from_numpy(np.ascontiguousarray(w.xyz)).to(dev)
    types = torch.from_numpy(np.ascontiguousarray(w.types)).to(dev)
    c = torch.from_numpy(np.ascontiguousarray(centres, np.float32)).to(dev)
    M = c.shape[0]
    sig = torch.full((M, len(dirs), 2), -7.0, dtype=torch.float32, device=dev)
    counts = torch.full((M,), -1, dtype=torch.int32, device=dev)
    if split:
        plan.apx_ingest(xyz, types)
        plan.apx_query(c, sig, counts)
    else:
        plan.apx_run(xyz, types, c, sig, counts)
    torch.cuda.synchronize()
    path = plan.apx_plan_path()
    plan.apx_plan_destroy()
    return sig.cpu().numpy(), counts.cpu().numpy().astype(np.uint32), path


def assert_parity(got_sig, got_counts, ref_sig, ref_counts, ref_win, k_lo):
    assert (got_counts == ref_counts).all(), "ROI ion counts differ"
    nc = ref_counts.astype(np.float64)[:, None]
    err = np.abs(got_sig[..., 0].astype(np.float64) - ref_sig[..., 0])
    tol = 1e-4 * ref_sig[..., 0] + 1e-6 * nc
    worst = np.unravel_index(np.argmax(err - tol), err.shape)
    assert (err <= tol).all(), f"amplitude off at {worst}: got {got_sig[worst]} ref {ref_sig[worst]}"
    bad = np.argwhere(got_sig[..., 1] != ref_sig[..., 1])
    for m, d in bad:
        k = int(got_sig[m, d, 1]) - k_lo
        assert 0 <= k < ref_win.shape[2], f"bin outside window at {(m, d)}: {got_sig[m, d]}"
        assert ref_win[m, d, k] >= ref_win[m, d].max() * (1 - 1e-4), \
            f"peak bin differs (no tie) at {(m, d)}: got {got_sig[m, d]} ref {ref_sig[m, d]}"
    return len(bad)
