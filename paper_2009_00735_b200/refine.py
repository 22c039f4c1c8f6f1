"""Adaptive refinement of the ROI grid: scan a coarse cubic ROI grid,
keep the grid cells whose maximum normalised signature intensity reaches kappa (L210: kappa >= 0.75), split each of them
into split^3 sub-cells (L210: 5^3) and scan those.

Host logic only: the grid of coarse centres is an input list built here; intensities, thresholding, compaction and the new
centres are computed by the library's kernels (include/aptsig_ext.h), the signatures by apx_query.  The one host read is
the number of selected cells (4 bytes), needed to size the second pass's output."""
from __future__ import annotations
import numpy as np


def coarse_grid(lo, hi, spacing) -> np.ndarray:
    """Centres of a cubic grid of edge `spacing` covering the box [lo, hi): float32 [M, 3], x fastest."""
    lo, hi = np.asarray(lo, np.float64), np.asarray(hi, np.float64)
    ax = [lo[a] + spacing * (np.arange(max(1, int(np.floor((hi[a] - lo[a]) / spacing + 1e-9)))) + 0.5) for a in range(3)]
    z, y, x = np.meshgrid(ax[2], ax[1], ax[0], indexing="ij")
    return np.ascontiguousarray(np.stack([x, y, z], -1).reshape(-1, 3).astype(np.float32))


def adaptive_scan(plan, xyz, types, centres, spacing, kappa=0.75, split=5, stream=None):
    """One coarse pass over `centres` (device float32 [M, 3], a grid of edge `spacing`) and one refined pass.
    Returns a dict of device tensors: coarse `sig`, `counts`, `kappa_max`, `selected` (indices into centres),
    `fine_centres`, `fine_sig`, `fine_counts`."""
    import torch
    dev = centres.device
    M = int(centres.shape[0])
    sig = torch.empty((M, plan.D, 2), dtype=torch.float32, device=dev)
    counts = torch.empty(M, dtype=torch.int32, device=dev)
    plan.apx_run(xyz, types, centres, sig, counts, stream=stream)
    kmax = torch.empty(M, dtype=torch.float32, device=dev)
    selected = torch.empty(M, dtype=torch.int32, device=dev)
    n_sel = torch.zeros(1, dtype=torch.int32, device=dev)
    plan.apx_intensity_max(sig, counts, kmax, stream=stream)
    plan.apx_refine_select(kmax, kappa, selected, n_sel, stream=stream)
    ns = int(n_sel.item())                                   # the one host read: sizes the second pass
    fine_centres = torch.empty((ns * split ** 3, 3), dtype=torch.float32, device=dev)
    fine_sig = torch.empty((ns * split ** 3, plan.D, 2), dtype=torch.float32, device=dev)
    fine_counts = torch.empty(ns * split ** 3, dtype=torch.int32, device=dev)
    if ns:
        plan.apx_refine_centres(centres, selected, n_sel, ns, spacing, split, fine_centres, stream=stream)
        plan.apx_query(fine_centres, fine_sig, fine_counts, stream=stream)
    return {"sig": sig, "counts": counts, "kappa_max": kmax, "selected": selected[:ns], "fine_centres": fine_centres,
            "fine_sig": fine_sig, "fine_counts": fine_counts}
