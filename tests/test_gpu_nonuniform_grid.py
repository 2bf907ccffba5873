"""The CUDA path on a photon energy grid that is not log-uniform (an irregular tabulation refined around an absorption edge,
`gen.tables.edge_resolving_tables`; SURVEY.md 8(f) NEXT-2 "drop-in NIST/DPM-format cross-section files").  The kernel finds the
table cell through a guide table and then interpolates as on a uniform grid; the oracle searches the grid (pinned by
tests/test_oracle_nonuniform_pins.py).  A cell taken on the wrong side of the edge changes the photoelectric coefficient by the
factor 5.2, a cell off by one elsewhere by per cent: both would fail the ledger comparison below."""
import numpy as np
import pytest

import oracle
from gen import make_config
from gen import tables as gt
from util import slab_cfg
from test_gpu_parity import engine_for, check_ledger, compare

pytestmark = pytest.mark.gpu


def test_thin_slab_either_side_of_the_edge():
    t = gt.edge_resolving_tables()
    n = 2_000_000
    for E in (0.0495, gt.GD_K_EDGE * (1 - 1e-5), gt.GD_K_EDGE * (1 + 1e-5), 0.060, 0.0117, 3.3):
        cfg = slab_cfg(n=(16, 16, 10), h=(1.0, 1.0, 0.05), rho=0.1, mat=gt.MAT_GOS, E=E, mode=0, t=t)
        eng = engine_for(cfg); eng.simulate(n, 9)
        L = eng.read_tallies()["ledger"]; check_ledger(L, n); eng.close()
        raw = oracle.run_sharded(cfg, n, 9, want_phantom_sq=False)
        Lo = raw["ledger"]
        for k in (1, 5):                                        # deposited in the slab, escaped: per history, 4 sigma + 0.1 %
            g, o = L[k] / n, Lo[k] / n
            spread = np.sqrt(max(raw["ledger_sq"][k] / n - o * o, 0.0))
            assert abs(g - o) <= 1e-3 * o + 4 * spread * np.sqrt(2.0 / n), (E, k, g, o)
        print("E = %.7f MeV: deposited in the slab gpu %.6f oracle %.6f MeV per history" % (E, L[1] / n, Lo[1] / n))


def test_whole_path_on_the_irregular_grid():
    cfg = make_config("C1", shrink=4, tables=gt.edge_resolving_tables())
    cfg["name"] = "C1-edge-grid"
    compare(cfg, 2_000_000, 1_000_000, rebin=8, seed=4, frac_ok=0.985, min_tested=20)


def test_grid_rules_at_the_boundary():
    from paper_2510_24154_b200.binding import AepidError
    t = gt.edge_resolving_tables()
    cfg = slab_cfg(t=t)
    eng = engine_for(cfg)
    bad = dict(t); bad["E_grid"] = t["E_grid"].copy(); bad["E_grid"][5] = bad["E_grid"][4]           # not strictly increasing
    with pytest.raises(AepidError):
        eng.init_materials(bad["E_grid"], t["mu_compton"], t["mu_pe"], t["mu_pair"], t["T_grid"], t["stop_pow"], t["rad_len"])
    Tg = t["T_grid"].copy(); Tg[7] *= 1.01                                                             # the electron grid stays log-uniform
    with pytest.raises(AepidError):
        eng.init_materials(t["E_grid"], t["mu_compton"], t["mu_pe"], t["mu_pair"], Tg, t["stop_pow"], t["rad_len"])
    eng.close()
