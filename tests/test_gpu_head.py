"""Parity of the collimation stage of the CUDA path against the oracle, through the C-ABI
(-m gpu).  The GPU follows the stage with analytic air gaps, a clear-passage test per slab and Woodcock flights only inside
slabs whose tungsten the ray may touch; the oracle tracks the whole stage by Woodcock flights: the same distribution, so the
comparison is statistical: Phase Space 2 yield and energy, energy absorbed in the head, then the usual tallies downstream."""
import numpy as np
import pytest

import oracle
from gen import head_config
from gen.configs import phase_space_1, _slab, HEAD_W, mono_spectrum
from gen.tables import MAT_W
from test_gpu_parity import compare, engine_for, check_ledger
from test_oracle_head_pins import head_cfg, pencil

pytestmark = pytest.mark.gpu


def head_stats_agree(cfg, n_gpu, n_or, seed=3):
    eng = engine_for(cfg)
    eng.simulate(n_gpu, seed)
    r = eng.read_tallies()
    check_ledger(r["ledger"], n_gpu)
    hg = eng.read_head()
    raw = oracle.run_sharded(cfg, n_or, seed, first=1 << 36, want_phantom_sq=False)
    ho = raw["head"]
    pg, po = hg[0] / n_gpu, ho[0] / n_or
    assert po > 0 and abs(pg - po) <= 4.5 * np.sqrt(po * (1 - po) * (1.0 / n_gpu + 1.0 / n_or)) + 1e-3 * po, (pg, po)   # Phase Space 2 yield
    Emax = float(cfg["ps1"]["records"][:, 5].max())
    for k in (1, 2):                                                     # energy through Phase Space 2, energy absorbed in the head (per history)
        g, o = hg[k] / n_gpu, ho[k] / n_or
        assert abs(g - o) <= 4.5 * Emax * np.sqrt(max(o / Emax, 1e-9) * (1.0 / n_gpu + 1.0 / n_or)) + 2e-3 * o, (k, g, o)
    assert hg[2] <= r["ledger"][4] * (1 + 1e-6)                           # booked in the ledger's air channel
    eng.close()
    return hg, ho


def test_closed_leaf_and_leaf_edge_on_the_gpu():
    E = 6.0
    closed = {"slabs": [_slab(HEAD_W["mlc"], 0, -5.0, 0.5, [0.0] * 20, [0.0] * 20)], "material": MAT_W, "density": 19.3, "w_ps2": HEAD_W["ps2"]}
    hg, ho = head_stats_agree(head_cfg(pencil(E, u=0.3, v=0.3), closed, E), 20_000_000, 4_000_000)
    assert hg[0] / 2e7 < 0.01                                            # 6.7 cm of tungsten
    ps1 = phase_space_1(seed=5, n=600_000, field_half_cm=4.0, spot_sigma_cm=0.0, spectrum=mono_spectrum(2.0))
    edge = {"slabs": [_slab(HEAD_W["mlc"], 0, -50.0, 100.0, [1.3], [60.0])], "material": MAT_W, "density": 19.3, "w_ps2": HEAD_W["ps2"]}
    head_stats_agree(head_cfg(ps1, edge, 2.0), 20_000_000, 4_000_000)


def test_phase_space_source_without_collimator():
    """Phase Space 1 handed straight to the patient stage (no slabs): the source sampler alone."""
    cfg = head_config(field=7, shrink=4, n_ps1=200_000)
    cfg["collimator"] = None
    compare(cfg, 20_000_000, 4_000_000, rebin=8, frac_ok=0.98, phantom_voxels=False, min_tested=30)


def test_c4_field_through_jaws_and_mlc():
    """One C4 field with the collimation stage in place of the fluence map: yield of the stage, then EPID image, energy budget
    and depth dose downstream, GPU against oracle."""
    cfg = head_config(field=7, shrink=2, n_ps1=1_000_000)
    head_stats_agree(cfg, 100_000_000, 20_000_000, seed=cfg["seed"])
    compare(cfg, 2_000_000_000, 200_000_000, rebin=4, frac_ok=0.98, phantom_voxels=False, min_tested=100)   # 3.1 mm pixels


def test_head_api_errors():
    from paper_2510_24154_b200 import AepidError
    cfg = head_config(field=7, shrink=8, n_ps1=1000)
    eng = engine_for(cfg)
    eng.load_phase_space_source(None, 0.0)
    with pytest.raises(AepidError, match="BAD_STATE"):
        eng.simulate(100, 1)                                             # a collimator without a phase-space source
    with pytest.raises(AepidError, match="NOMEM"):
        eng.load_phase_space_source(np.zeros((2000, 8), np.float32), 20.0)
    bad = dict(cfg["collimator"]); bad["slabs"] = list(reversed(bad["slabs"]))
    with pytest.raises(AepidError, match="BAD_ARG"):
        eng.load_collimator(bad)                                         # slabs must be sorted along w
    eng.load_collimator(None)
    eng.simulate(1000, 1)                                                # fluence-map source again
    r = eng.read_tallies(); check_ledger(r["ledger"], 1000)
    assert eng.read_head()[0] == 0
    eng.load_phase_space_source(cfg["ps1"]["records"], cfg["ps1"]["plane"]); eng.load_collimator(cfg["collimator"])
    eng.reset_tallies(); eng.simulate(100_000, 1)
    check_ledger(eng.read_tallies()["ledger"], 100_000)
    assert 0 < eng.read_head()[0] < 100_000
    eng.close()
