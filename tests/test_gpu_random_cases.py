"""Seeded random small cases, CUDA path against the oracle element by element (through the C ABI): every B, both kernels,
antipodally symmetric grids (shuffled, so that partners are far apart) and asymmetric ones, narrow windows with and without a
spare accumulator column, the full window, clouds on an exact quarter grid (exact-integer projections) or uniform, ROIs from
empty to several thousand ions, ion-type filter on and off.  Run with -m gpu on a B200."""
from types import SimpleNamespace

import numpy as np
import pytest

import paper_2009_00735_b200 as apx
from oracle import oracle as O
from _parity import run_gpu, assert_parity

pytestmark = pytest.mark.gpu


@pytest.mark.parametrize("seed", [1, 2, 3])
def test_random_cases_against_oracle(seed):
    rng = np.random.Generator(np.random.PCG64(seed))
    paths = set()
    for it in range(40):
        B = int(rng.choice([256, 512, 1024, 2048, 4096]))
        R = float(rng.uniform(0.8, 2.5))
        n_ions = int(rng.choice([0, 3, 40, 300, 1500, 2600, 5000]))
        box = R * rng.uniform(1.0, 1.6)
        xyz = rng.uniform(-box, box, (n_ions, 3)).astype(np.float32)
        if n_ions and rng.random() < 0.5:
            xyz = (np.round(xyz * 4) / 4).astype(np.float32)
        types = (rng.random(n_ions) < 0.3).astype(np.uint8)
        nd = int(rng.choice([1, 7, 33, 64, 150]))
        v = rng.standard_normal((nd, 3))
        v = (v / np.linalg.norm(v, axis=1)[:, None]).astype(np.float32)
        sym = rng.random() < 0.6
        dirs = np.concatenate([v, -v]) if sym else v
        if sym and rng.random() < 0.5:
            dirs = dirs[rng.permutation(len(dirs))]
        dirs = np.ascontiguousarray(dirs)
        k_lo = int(rng.integers(1, 40))
        W = int(rng.choice([1, 4, 20, 29, 32, 60]))
        window = (1, B // 2) if rng.random() < 0.3 else (k_lo, min(B // 2, k_lo + W - 1))
        flags = int(rng.choice([0, 0, apx.APX_FLAG_FORCE_FFT, apx.APX_FLAG_NO_PAIRING]))
        accepted = {0} if rng.random() < 0.4 else None
        M = int(rng.choice([1, 2, 5]))
        centres = rng.uniform(-0.5, 0.5, (M, 3)).astype(np.float32)
        if rng.random() < 0.3:
            centres[0] = 50.0                                                    # an empty ROI
        w = SimpleNamespace(xyz=xyz, types=types, R=R, B=B)
        what = f"case {it}: B={B} R={R:.3f} N={n_ions} D={len(dirs)} sym={sym} window={window} flags={flags} accepted={accepted} M={M}"
        got, cnt, path = run_gpu(apx, w, dirs, centres, accepted=accepted, window=window, flags=flags)
        ref, rc, win = O.signatures(xyz, types, centres, dirs, R, B, k_lo=window[0], k_hi=window[1], accepted=accepted,
                                    want_window=True)
        try:
            assert_parity(got, cnt, ref, rc, win, window[0])
        except AssertionError as e:
            raise AssertionError(what + ": " + str(e)) from e
        paths.add(path)
    assert paths == {0, 1}                                                       # both kernels were exercised


@pytest.mark.parametrize("seed", [1, 2])
def test_random_multi_signature_plans_against_oracle(seed):
    """Random plans of one to four signatures (type masks, windows, normalisation) on both kernels: every plane must equal the
    oracle's separate single-signature run (ROIs up to 4500 ions, so multi-pass, single-pass-with-DC-check and spilled ROIs
    occur with several signatures per class)."""
    import torch
    from oracle import next_oracle as X
    rng = np.random.Generator(np.random.PCG64(100 + seed))
    dev = torch.device("cuda:0")
    for it in range(25):
        B = int(rng.choice([256, 1024, 2048]))
        R = float(rng.uniform(1.0, 2.4))
        n_ions = int(rng.choice([50, 800, 2600, 4500]))
        box = R * rng.uniform(1.0, 1.4)
        xyz = rng.uniform(-box, box, (n_ions, 3)).astype(np.float32)
        if rng.random() < 0.5:
            xyz = (np.round(xyz * 4) / 4).astype(np.float32)
        types = rng.integers(0, 3, n_ions).astype(np.uint8)
        nd = int(rng.choice([9, 40, 100]))
        v = rng.standard_normal((nd, 3))
        v = (v / np.linalg.norm(v, axis=1)[:, None]).astype(np.float32)
        dirs = np.ascontiguousarray(np.concatenate([v, -v]) if rng.random() < 0.6 else v)
        specs = []
        for _ in range(int(rng.integers(1, 5))):
            k_lo = int(rng.integers(1, 30))
            sp = {"k_lo": k_lo, "k_hi": min(B // 2, k_lo + int(rng.choice([3, 12, 20, 29])) - 1)}
            if rng.random() < 0.6:
                sp["accepted_types"] = set(int(t) for t in rng.choice(3, size=int(rng.integers(1, 3)), replace=False))
            if rng.random() < 0.3:
                sp["normalise"] = 1
            specs.append(sp)
        flags = int(rng.choice([0, 0, apx.APX_FLAG_FORCE_FFT]))
        M = int(rng.choice([1, 3]))
        centres = rng.uniform(-0.4, 0.4, (M, 3)).astype(np.float32)
        what = f"case {it}: B={B} R={R:.2f} N={n_ions} D={len(dirs)} specs={specs} flags={flags}"
        plan = apx.Plan(R, B, dirs, device=0, flags=flags, specs=specs)
        sig = torch.full((len(specs), M, len(dirs), 2), -7.0, dtype=torch.float32, device=dev)
        cnt = torch.full((len(specs), M), -1, dtype=torch.int32, device=dev)
        plan.apx_run(torch.from_numpy(xyz).to(dev), torch.from_numpy(types).to(dev), torch.from_numpy(centres).to(dev), sig, cnt)
        torch.cuda.synchronize()
        plan.apx_plan_destroy()
        sig, cnt = sig.cpu().numpy(), cnt.cpu().numpy().astype(np.uint32)
        for s, sp in enumerate(specs):
            ref, rc, win = O.signatures(xyz, types, centres, dirs, R, B, k_lo=sp["k_lo"], k_hi=sp["k_hi"],
                                        accepted=sp.get("accepted_types"), want_window=True)
            got = sig[s].copy()
            try:
                if sp.get("normalise"):
                    assert np.allclose(got[..., 0], X.normalised(ref[..., 0], rc), rtol=1e-4, atol=1e-6), "normalised intensity"
                    got[..., 0] = got[..., 0] * rc[:, None]
                assert_parity(got, cnt[s], ref, rc, win, sp["k_lo"])
            except AssertionError as e:
                raise AssertionError(f"{what}, spec {s}: {e}") from e
