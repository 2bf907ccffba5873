"""Parity of the CUDA path with the CPU oracle at the FULL size of BASELINE.json configs[2..4] (run with -m gpu on a B200).

The oracle side is stored: tests/golden/oracle_<case>.npz, written by tests/golden/make_oracle_goldens.py, which calls only
oracle/ (2e8 histories for C2 and C3, 5e7 for each of five C4 fields incl. the smallest and the largest field size);
tests/test_oracle_goldens.py checks on the CPU that the files agree with the oracle as it stands.  The GPU runs the
config's own history count (C3: 1e9, in the launch configuration bench.py times) on a DISJOINT history range, so that the
two samples are independent.

Tolerances (BASELINE.json:north_star), all written out below:
  * >= 99 % of the EPID pixels above 20 % of the maximum within 3 combined sigma, on 3.1 mm (C2, C3, small C4 fields) or
    6.3 mm pixels (large C4 fields), >= 100 tested pixels; reading A20 (>= ~50 deposit events per tested pixel) is checked
    through the oracle's own relative error: (mean / sigma)^2 per history-count is printed as "effective events";
  * every channel of the energy budget within 0.5 % + 3 combined sigma, sigma from the per-history second moments;
  * phantom: >= 99 % of the voxel blocks above 20 % of the maximum within 3 combined sigma (blocks of 6 x 6 x 5 mm for
    C2 / C4, 8 x 8 x 10 mm for C3: the finest at which a block sees enough histories), z-score mean and width;
  * depth dose per slab within 1 % + 4 sigma of the spread over the oracle's K independent sub-runs;
  * energy ledger closed to 1e-6.
"""
import os

import numpy as np
import pytest

from gen import make_config

pytestmark = pytest.mark.gpu

HERE = os.path.dirname(os.path.abspath(__file__))
GPU_OFFSET = 1 << 40               # first history of the GPU run: disjoint from the oracle's [0, n)


def golden(case):
    import sys
    sys.path.insert(0, os.path.join(HERE, "golden"))
    from make_oracle_goldens import CASES, input_hash, depth_axes
    g = dict(np.load(os.path.join(HERE, "golden", "oracle_%s.npz" % case)))
    cname, field = CASES[case][0], CASES[case][1]
    cfg = make_config(cname, field=field)
    assert str(g["input_sha256"]) == input_hash(cfg), "the seeded inputs differ from those the golden file was made with"
    return g, cfg, depth_axes(cfg)


def gpu_rebinned(eng, r):
    b, nb = eng.read_batches()
    B = b.shape[0]
    rb = b.reshape(B, b.shape[1] // r, r, b.shape[2] // r, r).sum(axis=(2, 4)).astype(np.float64)
    N = nb.sum()
    mean = rb.sum(0) / N
    var = (nb[:, None, None] * (rb / nb[:, None, None] - mean) ** 2).sum(0) / ((B - 1) * N)
    return mean, np.sqrt(var)


@pytest.mark.parametrize("case,n_gpu", [("C2", 400_000_000), ("C3", 1_000_000_000), ("C4_00", 100_000_000), ("C4_04", 100_000_000),
                                        ("C4_07", 100_000_000), ("C4_17", 100_000_000), ("C4_21", 100_000_000)])
def test_full_size_tallies_match_the_oracle(case, n_gpu):
    from paper_2510_24154_b200 import Engine
    g, cfg, dd_ax = golden(case)
    n_or, rb = int(g["n"]), int(g["rb"])
    eng = Engine.for_config(cfg)
    eng.load_config(cfg)
    eng.set_history_offset(GPU_OFFSET)
    eng.simulate(n_gpu, int(g["seed"]))
    r = eng.read_tallies(sigma=False)                                   # raises AepidError INTERNAL if the kernel flagged anything
    L = r["ledger"]
    assert L[6] == n_gpu and L[7] == 0
    assert abs(L[1] + L[2] + L[3] + L[4] + L[5] - L[0]) <= 1e-6 * L[0]
    # ---- energy budget, channel by channel (per history); the per-history variance is the oracle's, used for both sides
    mo = g["ledger"] / n_or
    so = np.sqrt(np.maximum(g["ledger_sq"] / n_or - mo ** 2, 0.0))     # standard deviation over histories
    for k, name in ((0, "emitted"), (1, "dep_phantom"), (2, "dep_epid_scored"), (3, "dep_epid_other"), (4, "dep_air"), (5, "escaped")):
        sig = so[k] * np.sqrt(1.0 / n_or + 1.0 / n_gpu)
        d = L[k] / n_gpu - mo[k]
        print("%s %-16s gpu %.7f oracle %.7f rel %+.2e (sigma %.1e)" % (case, name, L[k] / n_gpu, mo[k], d / mo[k], sig / mo[k]))
        assert abs(d) <= 0.005 * mo[k] + 3.0 * sig, (name, d, sig)
        assert abs(d) <= 4.5 * sig + 3e-4 * mo[k], (name, d, sig)      # and no systematic offset beyond float32 table look-ups
    # ---- EPID image on re-binned pixels
    gm, gs = gpu_rebinned(eng, rb)
    om = g["rb_sum"] / n_or
    os_ = np.sqrt(np.maximum(g["rb_sq"] / n_or - om ** 2, 0.0) / (n_or - 1))
    k = om > 0.2 * om.max()
    z = (gm[k] - om[k]) / np.sqrt(gs[k] ** 2 + os_[k] ** 2)
    eff = (om[k] / os_[k]) ** 2
    print("%s EPID %.2f mm pixels: %d tested, within 3 sigma %.4f, z mean %+.3f std %.3f, effective oracle events per pixel min %.0f median %.0f"
          % (case, 10 * rb * cfg["epid"]["pitch"], k.sum(), np.mean(np.abs(z) < 3), z.mean(), z.std(), eff.min(), np.median(eff)))
    assert k.sum() >= 100 and eff.min() >= 50
    assert np.mean(np.abs(z) < 3) >= 0.99
    assert abs(z.mean()) < 4.0 / np.sqrt(k.sum()) + 0.05 and 0.85 < z.std() < 1.15
    # ---- phantom on voxel blocks (the GPU's own variance is n_or / n_gpu of the oracle's: same physics, more histories)
    bx, by, bz = (int(v) for v in g["pb"])
    pm = r["phantom_mean"].astype(np.float64)
    nz, ny, nx = pm.shape
    blk = pm.reshape(nz // bz, bz, ny // by, by, nx // bx, bx).sum(axis=(1, 3, 5)).ravel()[g["pc_idx"]]
    om = g["pc_sum"] / n_or
    os_ = np.sqrt(np.maximum(g["pc_sq"] / n_or - om ** 2, 0.0) / (n_or - 1))
    k = om > 0.2 * om.max()
    z = (blk[k] - om[k]) / (os_[k] * np.sqrt(1.0 + n_or / n_gpu))
    print("%s phantom blocks %dx%dx%d voxels: %d tested, within 3 sigma %.4f, z mean %+.3f std %.3f, max |rel diff| %.3e"
          % (case, bx, by, bz, k.sum(), np.mean(np.abs(z) < 3), z.mean(), z.std(), np.abs(blk[k] / om[k] - 1).max()))
    assert k.sum() >= 400                                                   # 501 for the 3 cm field, 2300 - 11500 for the others
    assert np.mean(np.abs(z) < 3) >= 0.99
    assert abs(z.mean()) < 0.1 and 0.9 < z.std() < 1.1
    # ---- depth dose: spread over the oracle's K independent sub-runs
    dd = g["dd_runs"]; K = dd.shape[0]
    do, sd = dd.mean(0), dd.std(0, ddof=1) / np.sqrt(K)
    dg = pm.sum(axis=dd_ax)
    k = do > 0.2 * do.max()
    sig = sd[k] * np.sqrt(1.0 + n_or / n_gpu)
    print("%s depth dose over %d slabs: max |gpu/oracle - 1| %.2e" % (case, k.sum(), np.abs(dg[k] / do[k] - 1).max()))
    assert np.all(np.abs(dg[k] - do[k]) <= 0.01 * do[k] + 4.0 * sig)
    eng.close()


def test_c4_response_post_pass_at_full_resolution():
    """K8 on the full 1024 x 768 image of a C4 field against the oracle's exact Siddon thickness map and bilinear look-up."""
    import oracle
    from paper_2510_24154_b200 import Engine
    cfg = make_config("C4", field=7)
    eng = Engine.for_config(cfg)
    eng.load_config(cfg)
    eng.simulate(20_000_000, cfg["seed"])
    dose = eng.read_tallies(phantom=False, sigma=False)["epid_mean"]
    lut = cfg["lut"]
    sig, tmap = eng.apply_response_lut(lut["lut"], lut["t_min"], lut["t_max"], lut["s_min"], lut["s_max"], -1.0, epid_in=dose)
    o = oracle.Oracle(cfg)
    s_o = o.field_size()
    assert eng.field_size() == pytest.approx(s_o, rel=1e-6)
    t_o = o.tmap()
    assert np.abs(tmap - t_o).max() <= 1e-4 * t_o.max()
    ref = o.apply_lut(lut, dose, t_o, s_o)
    assert np.abs(sig - ref).max() <= 2e-5 * np.abs(ref).max()
    eng.close()
