"""Pins of the oracle's table look-up on a photon grid that is NOT log-uniform (the kind real tabulations come on: irregular
spacing, refined around an absorption edge that is carried as two grid points, "cross
sections").  `gen.tables.edge_resolving_tables` builds the input; what is checked is fixed by mathematics, not by the oracle:
a power law is reproduced exactly by log-log interpolation on any grid, node values are reproduced at the nodes, the edge is a
jump of the stated ratio, and the uncollided transmission through a slab is Beer-Lambert with the coefficient of its side."""
import numpy as np

import oracle
from gen import tables as gt
from util import slab_cfg


def edge_oracle():
    t = gt.edge_resolving_tables()
    o = oracle.Oracle(); o.init_materials(t)
    return t, o


def test_grid_is_irregular_and_carries_the_edge_as_two_points():
    t = gt.edge_resolving_tables()
    d = np.diff(np.log(t["E_grid"].astype(np.float64)))
    assert d.min() < 1e-5 and d.max() > 0.15 and d.max() / np.median(d) > 1.5          # not a log-uniform grid by any tolerance
    i = np.searchsorted(t["E_grid"], gt.GD_K_EDGE)
    assert abs(t["E_grid"][i - 1] / gt.GD_K_EDGE - 1) < 3e-6 and abs(t["E_grid"][i] / gt.GD_K_EDGE - 1) < 3e-6
    assert abs(t["mu_pe"][gt.MAT_GOS, i] / t["mu_pe"][gt.MAT_GOS, i - 1] - t["edge"]["jump"]) < 1e-3 * t["edge"]["jump"]


def test_power_law_is_reproduced_exactly_between_irregular_nodes():
    t, o = edge_oracle()
    rng = np.random.default_rng(3)
    E = np.exp(rng.uniform(np.log(1.2e-3), np.log(19.0), 400))
    for m in (gt.MAT_SOFT, gt.MAT_CU, gt.MAT_BONE):                  # photoelectric ~ E^-3: linear in (ln E, ln mu) on every cell
        comp = gt.MATERIALS[m][1]
        got = np.array([o.mu_partial(m, e)[0] for e in E])
        assert np.abs(got / gt.mu_photoelectric(comp, E) - 1).max() < 5e-7      # float32 storage of the node values
    # a wrong cell (off by one) or a fraction taken in E instead of ln E would miss by per cent on the 0.19-wide cells
    Eg = t["E_grid"].astype(np.float64)
    for m in (gt.MAT_SOFT, gt.MAT_GOS):
        for j in (0, 7, 40, len(Eg) - 1):                            # node values at the nodes, all three channels
            got = o.mu_partial(m, float(Eg[j]))
            want = (t["mu_pe"][m, j], t["mu_compton"][m, j], t["mu_pair"][m, j] if Eg[j] > 2 * gt.MEC2 else 0.0)
            assert np.allclose(got, want, rtol=1e-6, atol=1e-12)


def test_edge_is_a_jump_of_the_stated_ratio():
    t, o = edge_oracle()
    comp = gt.MATERIALS[gt.MAT_GOS][1]
    below, above = gt.GD_K_EDGE * (1 - 1e-5), gt.GD_K_EDGE * (1 + 1e-5)
    assert abs(o.mu_partial(gt.MAT_GOS, below)[0] / gt.mu_photoelectric(comp, below) - 1) < 1e-6
    assert abs(o.mu_partial(gt.MAT_GOS, above)[0] / (t["edge"]["jump"] * gt.mu_photoelectric(comp, above)) - 1) < 1e-6
    assert abs(o.mu_partial(gt.MAT_SOFT, above)[0] / o.mu_partial(gt.MAT_SOFT, below)[0] - (below / above) ** 3) < 1e-6   # no edge elsewhere


def test_transmission_through_a_slab_either_side_of_the_edge_is_beer_lambert():
    t = gt.edge_resolving_tables()
    comp = gt.MATERIALS[gt.MAT_GOS][1]
    for E in (0.0495, gt.GD_K_EDGE * (1 - 1e-5), gt.GD_K_EDGE * (1 + 1e-5), 0.060):
        cfg = slab_cfg(n=(16, 16, 10), h=(1.0, 1.0, 0.05), rho=0.1, mat=gt.MAT_GOS, E=E, mode=0, t=t)
        o = oracle.Oracle(cfg)
        o.set_fixed_primary(0, E, (0, 0, 0), (0, 0, 1))
        o.reset(); n = 100000; o.run(0, n, 5)
        r = o.read()
        mu = gt.mu_compton(comp, E) + gt.mu_photoelectric(comp, E) * (t["edge"]["jump"] if E > gt.GD_K_EDGE else 1.0)
        mu_air = sum(f(gt.MATERIALS[gt.MAT_AIR][1], E) for f in (gt.mu_compton, gt.mu_photoelectric))
        want = np.exp(-mu * 0.1 * 0.5) * np.exp(-mu_air * gt.RHO_AIR * (170.0 - 0.5))
        got = r["counters"][10] / n
        assert abs(got - want) < 4.5 * np.sqrt(want * (1 - want) / n) + 2e-3 * want, (E, got, want)
