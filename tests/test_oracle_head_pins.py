"""Pins of the oracle's collimation stage (Phase Space 1 sampled, transported through
jaws and MLC, Phase Space 2 streamed to the patient stage).  No GPU.  Closed forms only: planar fluence of a point source,
Beer-Lambert transmission through a closed leaf, the geometric penumbra of a straight leaf edge, energy conservation."""
import numpy as np
import pytest
from scipy import stats as sst

import oracle
from gen import tables as gt
from gen.configs import phase_space_1, collimator_for_fluence, _slab, HEAD_W, mono_spectrum
from gen.tables import make_tables, TUNGSTEN, MAT_W
from util import slab_cfg

T9 = None


def head_cfg(ps1, col, E=2.0):
    global T9
    if T9 is None:
        T9 = make_tables(extra=(TUNGSTEN,))
    import copy
    cfg = slab_cfg(n=(8, 8, 4), h=(4.0, 4.0, 1.0), w0=100.0, rho=1e-6, E=E, mode=0, t=copy.deepcopy(T9))
    cfg["ps1"], cfg["collimator"] = ps1, col
    return cfg


def mu_lin(mat, rho, E):
    comp = (list(gt.MATERIALS) + [TUNGSTEN])[mat][1]
    return rho * float(gt.mu_compton(comp, E) + gt.mu_photoelectric(comp, E) + gt.mu_pair(comp, E))


def pencil(E, n=1, u=0.0, v=0.0, d=(0.0, 0.0, 1.0)):
    rec = np.zeros((n, 8), np.float32)
    rec[:, 0], rec[:, 1], rec[:, 2:5], rec[:, 5] = u, v, d, E
    return {"records": rec, "plane": HEAD_W["ps1"], "n": n}


def wide_open():
    big = 60.0
    return {"slabs": [_slab(HEAD_W["jaw_y"], 1, -100.0, 200.0, [-big], [big]), _slab(HEAD_W["jaw_x"], 0, -100.0, 200.0, [-big], [big]),
                      _slab(HEAD_W["mlc"], 0, -20.0, 0.25, [-big] * 160, [big] * 160)],
            "material": MAT_W, "density": 19.3, "w_ps2": HEAD_W["ps2"]}


def run(cfg, n, seed=3):
    o = oracle.Oracle(cfg)
    o.set_ps2(True); o.reset(); o.run(0, n, seed)
    return o, o.read(), o.read_ps2()


def test_open_collimator_hands_phase_space_1_through():
    """Without tungsten in the way Phase Space 2 is Phase Space 1 moved along its rays (minus the 0.2 % the air takes): the
    planar fluence on the isocentre plane is that of the fluence-map source of the same field (uniform), by chi-square; every
    record is used with equal probability; the spectrum is unchanged."""
    ps1 = phase_space_1(seed=11, n=20000, field_half_cm=5.0, spot_sigma_cm=0.0, spectrum=mono_spectrum(2.0))
    cfg = head_cfg(ps1, wide_open())
    n = 200_000
    o, r, ps2 = run(cfg, n)
    mu_a = mu_lin(gt.MAT_AIR, gt.RHO_AIR, 2.0)
    unc = ps2[ps2[:, 7] == 1]
    L = (HEAD_W["ps2"] - HEAD_W["ps1"])                                  # along w; obliquity <= 0.3 %
    p_exp = np.exp(-mu_a * L)
    assert abs(len(unc) / n - p_exp) < 4.5 * np.sqrt(p_exp * (1 - p_exp) / n) + 1e-5
    assert np.all(unc[:, 0] == np.float32(2.0))
    ui, vi = unc[:, 1] * 100.0 / HEAD_W["ps2"], unc[:, 2] * 100.0 / HEAD_W["ps2"]   # point source: straight lines through the origin
    assert np.abs(ui).max() <= 5.0 + 1e-4 and np.abs(vi).max() <= 5.0 + 1e-4
    h, _, _ = np.histogram2d(vi, ui, bins=10, range=[[-5, 5], [-5, 5]])
    # the table holds 20000 records drawn uniformly on the square; the histories draw from the table with replacement
    hr, _, _ = np.histogram2d(ps1["records"][:, 1] * 100 / 20.0, ps1["records"][:, 0] * 100 / 20.0, bins=10, range=[[-5, 5], [-5, 5]])
    exp = hr / hr.sum() * len(unc)
    assert sst.chi2.sf(((h - exp) ** 2 / exp).sum(), 99) > 1e-4                 # follows the table cell by cell
    # and it is the same planar fluence as the fluence-map source of a 10 x 10 cm open field
    s = oracle.Oracle(slab_cfg(field_cm=10.0)).sample_source(0, n, 5)
    hs, _, _ = np.histogram2d(s[:, 6], s[:, 5], bins=10, range=[[-5, 5], [-5, 5]])
    # a cell count of Phase Space 2 carries the noise of the 20000-record table as well: variance h (1 + n / N_table)
    f = len(unc) / n
    chi2 = (((h / f - hs) ** 2) / (h / f ** 2 * (1 + n / 20000.0) + hs)).sum()
    assert sst.chi2.sf(chi2, 99) > 1e-4
    # records are drawn uniformly: chi-square of how often each of the first 200 records was used is not possible from PS2 alone,
    # but the mean direction is that of the table
    assert np.abs(unc[:, 3:6].mean(0) - ps1["records"][:, 2:5].mean(0)).max() < 5e-4


def test_closed_leaf_transmission_is_beer_lambert():
    """A pencil beam onto a closed leaf pair: the uncollided fraction behind the stage is exp(-mu rho L) of 6.7 cm of tungsten
    (times the air).  Catches a wrong material / density in the slab, a slab thickness that is not w1 - w0, a closed pair read as open."""
    E = 6.0
    col = {"slabs": [_slab(HEAD_W["mlc"], 0, -5.0, 0.5, [0.0] * 20, [0.0] * 20)], "material": MAT_W, "density": 19.3, "w_ps2": HEAD_W["ps2"]}
    n = 1_000_000
    o, r, ps2 = run(head_cfg(pencil(E, u=0.3, v=0.3), col, E), n)
    Lw = HEAD_W["mlc"][1] - HEAD_W["mlc"][0]
    p_exp = np.exp(-mu_lin(MAT_W, 19.3, E) * Lw - mu_lin(gt.MAT_AIR, gt.RHO_AIR, E) * (HEAD_W["ps2"] - HEAD_W["ps1"] - Lw))
    k = (ps2[:, 7] == 1).sum()
    assert 500 < p_exp * n and abs(k - p_exp * n) < 4.5 * np.sqrt(p_exp * n)
    assert np.all(ps2[ps2[:, 7] == 1][:, 1] == np.float32(0.3))
    L = r["ledger"]
    assert abs(L[1] + L[2] + L[3] + L[4] + L[5] - L[0]) < 1e-12 * L[0] and L[0] == pytest.approx(n * E)
    assert r["head"][0] == len(ps2) and r["head"][2] > 0.8 * L[0]       # nearly all of the beam's energy stays in the leaf
    assert r["head"][2] <= L[4] + 1e-9


def test_leaf_edge_penumbra_of_a_straight_edge():
    """One leaf bank edge at x_e on the slab: seen from a point source the edge projects to the isocentre plane between
    100 x_e / w1 and 100 x_e / w0 (straight, unfocused edge), and a ray in between crosses (x_e / theta - w0) of tungsten."""
    E, xe = 2.0, 1.3
    w0, w1 = HEAD_W["mlc"]
    ps1 = phase_space_1(seed=5, n=600_000, field_half_cm=4.0, spot_sigma_cm=0.0, spectrum=mono_spectrum(E))
    col = {"slabs": [_slab(HEAD_W["mlc"], 0, -50.0, 100.0, [xe], [60.0])], "material": MAT_W, "density": 19.3, "w_ps2": HEAD_W["ps2"]}
    n = 600_000
    o, r, ps2 = run(head_cfg(ps1, col, E), n)
    unc = ps2[ps2[:, 7] == 1]
    ui = unc[:, 1] * 100.0 / HEAD_W["ps2"]
    edges = np.linspace(1.8, 3.2, 29)                                    # 0.5 mm bins across 100 xe / w1 = 2.37 ... 100 xe / w0 = 2.70
    obs, _ = np.histogram(ui, bins=edges)
    muw, mua = mu_lin(MAT_W, 19.3, E), mu_lin(gt.MAT_AIR, gt.RHO_AIR, E)
    def trans(u):                                                        # along the ray of slope theta = u / 100 (v = 0 plane: obliquity in v <= 1e-3)
        th = u / 100.0
        lw = np.clip(xe / th - w0, 0.0, w1 - w0)
        return np.exp(-muw * lw * np.sqrt(1 + th * th) - mua * (HEAD_W["ps2"] - HEAD_W["ps1"] - lw))
    # expected counts: records uniform in u on [-4, 4] (8 cm) and all v; integrate the transmission over each bin
    dens = n / 8.0
    exp = np.array([dens * np.mean(trans(np.linspace(a, b, 201))) * (b - a) for a, b in zip(edges[:-1], edges[1:])])
    k = exp > 20
    assert k.sum() >= 15
    chi2 = ((obs[k] - exp[k]) ** 2 / exp[k]).sum() / (1.0 + n / 600_000.0)   # histories draw from the 600000-record table with replacement
    assert sst.chi2.sf(chi2, k.sum()) > 1e-4, (obs, exp)
    assert obs[edges[1:] <= 100 * xe / w1 - 0.1].sum() < 0.02 * obs.sum()   # under the leaf: 0.5 % transmission
    assert abs(obs[edges[:-1] >= 100 * xe / w0].mean() / (dens * 0.05 * np.exp(-mua * 36.0)) - 1) < 0.05


def test_jaw_axes_and_row_lookup():
    """axis 1 (y-jaws) limits v, axis 0 (x-jaws, MLC) limits u; MLC rows are stacked along v.  An asymmetric opening in every
    slab: the photons that get through untouched lie exactly in the intersection of the projected openings."""
    ps1 = phase_space_1(seed=9, n=400_000, field_half_cm=10.0, spot_sigma_cm=0.0, spectrum=mono_spectrum(1.0))
    sc = lambda w: 0.5 * (w[0] + w[1]) / 100.0
    jy, jx, ml = HEAD_W["jaw_y"], HEAD_W["jaw_x"], HEAD_W["mlc"]
    lo, hi = np.zeros(40), np.zeros(40)
    lo[22:26], hi[22:26] = -1.0 * sc(ml), 3.0 * sc(ml)                  # leaf rows 22..25 of 0.5 cm: v in [1, 3] cm at the isocentre; u in [-1, 3]
    col = {"slabs": [_slab(jy, 1, -100.0, 200.0, [-2.0 * sc(jy)], [6.0 * sc(jy)]), _slab(jx, 0, -100.0, 200.0, [-4.0 * sc(jx)], [8.0 * sc(jx)]),
                     _slab(ml, 0, -10.0 * sc(ml), 0.5 * sc(ml), lo, hi)], "material": MAT_W, "density": 19.3, "w_ps2": HEAD_W["ps2"]}
    o, r, ps2 = run(head_cfg(ps1, col, 1.0), 400_000)
    unc = ps2[ps2[:, 7] == 1]
    ui, vi = unc[:, 1] * 100.0 / HEAD_W["ps2"], unc[:, 2] * 100.0 / HEAD_W["ps2"]
    core = (ui > -0.8) & (ui < 2.7) & (vi > 1.15) & (vi < 2.75)            # inside the umbra of every edge (penumbra <= 0.13 x |coordinate|)
    assert core.mean() > 0.7                                               # the rest lies in the penumbra of the straight edges
    inside = (ui > -1.0 - 0.2) & (ui < 3.0 + 0.45) & (vi > 1.0 - 0.2) & (vi < 3.0 + 0.45)
    assert inside.mean() > 0.98                                            # the rest leaked through 6.7 cm of tungsten (2e-4 per ray at 1 MeV)
    leak = unc[~inside]
    assert np.all((leak[:, 1] * 100 / HEAD_W["ps2"] > -4.3) & (leak[:, 1] * 100 / HEAD_W["ps2"] < 8.5))   # ... but not through leaves AND jaws
    frac = core.sum() / 400_000                                            # 5600 expected: 4.5 sigma incl. the noise of the table = 8.5 %
    assert frac == pytest.approx(3.5 * 1.6 / 400.0 * np.exp(-mu_lin(gt.MAT_AIR, gt.RHO_AIR, 1.0) * 36.0), rel=0.085)


def test_stage_ledger_and_scattered_photons():
    """Energy conservation through the stage with Compton scattering in the jaws: emitted = absorbed in the stage + escaped + what
    Phase Space 2 carries on; scattered photons are flagged, lose energy, and never travel upstream."""
    cfg = head_cfg(None, None, 2.0)
    from gen import head_config
    hc = head_config(field=7, shrink=8, n_ps1=50_000)
    o, r, ps2 = run(hc, 100_000)
    L = r["ledger"]
    assert abs(L[1] + L[2] + L[3] + L[4] + L[5] - L[0]) < 1e-12 * L[0] and L[6] == 100_000
    hd = r["head"]
    assert hd[0] == len(ps2) and hd[1] == pytest.approx(ps2[:, 0].sum(), rel=1e-12)
    assert 0.005 < hd[0] / 1e5 < 0.2                                     # a 4 cm field out of the 28 cm square of Phase Space 1
    sc = ps2[ps2[:, 7] == 0]
    assert len(sc) > 0 and np.all(sc[:, 5] > 0) and np.all(ps2[:, 5] > 0)
    assert 0 < len(sc) < 0.2 * len(ps2)
