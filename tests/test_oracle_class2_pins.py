"""Pins of the oracle's Class II collision mode (mode 2: discrete Moller events above the electron cut-off, restricted
stopping power below it, reading A31).  CPU only."""
import numpy as np
import pytest
from scipy import integrate, stats

import oracle
import gen.tables as gt
from util import slab_cfg, tables

MEC2, R_E = 0.51099895, 2.8179403262e-13


def dsigma_deps(eps, T):
    """Moller cross section per electron, differential in eps = W / T (textbook form, retyped here for the quadrature)."""
    tau = T / MEC2
    b2 = tau * (tau + 2) / (tau + 1) ** 2
    return 2 * np.pi * R_E ** 2 * MEC2 / (b2 * T) * (1 / eps ** 2 + 1 / (1 - eps) ** 2 + (tau / (tau + 1)) ** 2
                                                      - (2 * tau + 1) / (tau + 1) ** 2 / (eps * (1 - eps)))


@pytest.mark.parametrize("T,Tc", [(0.41, 0.2), (0.5, 0.2), (1.0, 0.2), (3.0, 0.2), (6.0, 0.2), (20.0, 0.2), (2.0, 0.01), (2.0, 0.9)])
def test_moller_closed_forms_equal_the_quadrature(T, Tc):
    s, h = oracle.moller_xs(T, Tc)
    qs = integrate.quad(dsigma_deps, Tc / T, 0.5, args=(T,), epsrel=1e-11)[0]
    qh = integrate.quad(lambda e: e * T * dsigma_deps(e, T), Tc / T, 0.5, epsrel=1e-11)[0]
    assert s == pytest.approx(qs, rel=1e-7) and h == pytest.approx(qh, rel=1e-7)


def test_moller_threshold_and_limits():
    assert oracle.moller_xs(0.4, 0.2) == (0.0, 0.0) and oracle.moller_xs(0.1, 0.2) == (0.0, 0.0)
    s, h = oracle.moller_xs(0.4 + 1e-9, 0.2)
    assert 0 <= s < 1e-30 and 0 <= h < 1e-30                          # both vanish continuously at T = 2 Tc
    # the hard loss can never exceed the total collision stopping power it is taken from
    t = tables()
    for m in range(t["n_mat"]):
        for T in (0.5, 1.0, 2.0, 6.0, 15.0):
            S = float(gt.stopping_power(gt.MATERIALS[m][1], T))
            assert 0 < float(t["electrons_per_gram"][m]) * oracle.moller_xs(T, 0.2)[1] < 0.35 * S
    # electrons per gram: water 3.343e23 (10 electrons per 18.015 g/mol)
    assert float(t["electrons_per_gram"][gt.MAT_SOFT]) == pytest.approx(10 * 6.02214076e23 / 18.015, rel=2e-4)


@pytest.mark.parametrize("T", [0.5, 2.0, 10.0])
def test_moller_sampler_follows_the_density(T):
    Tc, n = 0.2, 200_000
    eps = oracle.sample_moller(T, Tc, 7, n)
    assert eps.min() >= Tc / T and eps.max() <= 0.5
    edges = np.linspace(Tc / T, 0.5, 21)
    obs = np.histogram(eps, bins=edges)[0]
    sig = oracle.moller_xs(T, Tc)[0]
    exp = np.array([integrate.quad(dsigma_deps, a, b, args=(T,))[0] for a, b in zip(edges[:-1], edges[1:])]) / sig * n
    chi2 = ((obs - exp) ** 2 / exp).sum()
    assert chi2 < stats.chi2.ppf(0.9999, len(exp) - 1)
    s, h = oracle.moller_xs(T, Tc)
    assert eps.mean() == pytest.approx(h / (s * T), abs=5 * eps.std() / np.sqrt(n))


@pytest.mark.parametrize("T,W", [(1.0, 0.2), (2.0, 1.0), (6.0, 0.5), (0.5, 0.25)])
def test_moller_angles_conserve_momentum(T, W):
    p = lambda t: np.sqrt(t * (t + 2 * MEC2))
    cd, cp = oracle.moller_cos(W, T), oracle.moller_cos(T - W, T)
    sd, sp = np.sqrt(1 - cd * cd), np.sqrt(1 - cp * cp)
    assert p(W) * cd + p(T - W) * cp == pytest.approx(p(T), rel=1e-12)          # along the incoming direction
    assert p(W) * sd == pytest.approx(p(T - W) * sp, rel=1e-9)                  # transverse: opposite azimuths


def _thin_slab(mode, n, T0=2.0, thick=0.2, seed=3):
    """n electrons of T0 normally onto a water slab `thick` cm thick without multiple scattering; Phase Space 3 on a plane
    1 cm behind it."""
    t = tables()
    t["rad_len"][:] = 1e30
    cfg = slab_cfg(n=(4, 4, 1), h=(5.0, 5.0, thick), w0=100.0, mode=mode, t=t, sid=100.0 + thick + 1.0)
    o = oracle.Oracle(cfg)
    o.set_fixed_primary(1, T0, (0.1, 0.1, 100.0 + 1e-9), (0, 0, 1))
    o.set_ps3(True)
    o.reset()
    o.run(0, n, seed)
    return o, o.read(), o.read_ps3()


def test_class2_thin_slab_mean_loss_equals_csda_and_delta_rate_equals_the_cross_section():
    n, T0, thick = 100_000, 2.0, 0.2
    o1, r1, ps1 = _thin_slab(1, 200)
    o2, r2, ps2 = _thin_slab(2, n)
    for r in (r1, r2):
        L = r["ledger"]
        assert abs(L[1] + L[2] + L[3] + L[4] + L[5] - L[0]) < 1e-11 * L[0]
    # mode 1: every electron leaves with the same energy (CSDA, no straggling)
    e1 = ps1[ps1[:, 0] == 1, 1]
    assert len(e1) == 200 and e1.std() < 1e-12
    loss1 = T0 - e1.mean()
    # mode 2: the primary is the fastest electron of its history at the plane; its mean loss (restricted continuous loss +
    # hard transfers) is the unrestricted CSDA loss
    el = ps2[ps2[:, 0] == 1]
    h = el[:, 7].astype(np.int64)
    prim = np.zeros(n); np.maximum.at(prim, h, el[:, 1])
    assert np.all(prim > 0)
    loss2 = T0 - prim
    assert loss2.mean() == pytest.approx(loss1, rel=0.01, abs=4 * loss2.std() / np.sqrt(n))
    assert loss2.std() > 0.02                                           # there is straggling now
    # number of delta rays per primary = int rho n_e sigma(T(s)) ds along the slab (T(s) from the restricted loss)
    ne = float(o2.cfg["tables"]["electrons_per_gram"][gt.MAT_SOFT])
    Lr = lambda T: o2.stop_pow(gt.MAT_SOFT, T) - ne * oracle.moller_xs(T, 0.2)[1]
    sol = integrate.solve_ivp(lambda s, T: [-Lr(T[0])], (0, thick), [T0], dense_output=True, rtol=1e-9)
    expect = integrate.quad(lambda s: ne * oracle.moller_xs(float(sol.sol(s)[0]), 0.2)[0], 0, thick)[0]
    n_delta = r2["aux"][2]                                              # hard collisions inside the slab
    assert n_delta / n == pytest.approx(expect, rel=0.02, abs=4 * np.sqrt(n_delta) / n)
    # and they arrive (or stop on the way): never more electrons at the plane than primaries + delta rays
    assert len(el) <= n + r2["aux"][2] + r2["aux"][3]


def test_class2_full_config_ledger_and_mode1_equivalence_of_totals():
    from gen import make_config
    cfg = make_config("C1", shrink=4)
    n = 20_000
    res = {}
    for mode in (1, 2):
        cfg["physics"]["mode"] = mode
        o = oracle.Oracle(cfg); o.reset(); o.run(0, n, 1)
        r = o.read(); L = r["ledger"]
        assert abs(L[1] + L[2] + L[3] + L[4] + L[5] - L[0]) < 1e-12 * L[0]
        res[mode] = r
    # same source photons; the energy absorbed in a 20 cm phantom changes by far less than a per cent when some of the
    # electron energy travels a little farther as delta rays
    assert res[2]["ledger"][0] == res[1]["ledger"][0]
    assert res[2]["ledger"][1] == pytest.approx(res[1]["ledger"][1], rel=0.01)
    assert res[2]["counters"][9] > res[1]["counters"][9]                 # more charged particles are born


# ------------------------------------------------------------------------------------------------ bremsstrahlung (mode 3, A32)
def dSigma_dk(k, T, X0):
    y = k / T
    return (4.0 / 3.0 - 4.0 / 3.0 * y + y * y) / (X0 * k)


@pytest.mark.parametrize("T,kc,X0", [(0.5, 0.01, 36.3), (2.0, 0.01, 36.3), (6.0, 0.01, 13.2), (20.0, 0.1, 8.6), (0.02, 0.01, 40.8)])
def test_brems_closed_forms_quadrature_and_radiation_length_sum_rule(T, kc, X0):
    sig, soft = oracle.brems_xs(T, kc, X0)
    assert sig == pytest.approx(integrate.quad(dSigma_dk, kc, T, args=(T, X0), epsrel=1e-11)[0], rel=1e-8)
    assert soft == pytest.approx(integrate.quad(lambda k: k * dSigma_dk(k, T, X0), 0, kc, epsrel=1e-11)[0], rel=1e-8)
    hard = integrate.quad(lambda k: k * dSigma_dk(k, T, X0), kc, T, epsrel=1e-11)[0]
    assert soft + hard == pytest.approx(T / X0, rel=1e-8)               # total radiative stopping power = T / X0
    assert oracle.brems_xs(0.5 * kc, kc, X0) == (0.0, pytest.approx(0.5 * kc / X0))   # below the cut-off everything is soft


@pytest.mark.parametrize("T", [0.3, 2.0, 15.0])
def test_brems_sampler_follows_the_density(T):
    kc, n, X0 = 0.01, 200_000, 36.3
    k = oracle.sample_brems(T, kc, 11, n)
    assert k.min() >= kc and k.max() <= T
    edges = np.exp(np.linspace(np.log(kc), np.log(T), 25))
    obs = np.histogram(k, bins=edges)[0]
    sig = oracle.brems_xs(T, kc, X0)[0]
    exp = np.array([integrate.quad(dSigma_dk, a, b, args=(T, X0))[0] for a, b in zip(edges[:-1], edges[1:])]) / sig * n
    assert ((obs - exp) ** 2 / exp).sum() < stats.chi2.ppf(0.9999, len(exp) - 1)


def test_mode3_thin_slab_mean_loss_and_photon_yield():
    n, T0, thick = 100_000, 6.0, 0.2
    o3, r3, ps3 = _thin_slab(3, n, T0=T0, thick=thick)
    L = r3["ledger"]
    assert abs(L[1] + L[2] + L[3] + L[4] + L[5] - L[0]) < 1e-11 * L[0]
    X0 = float(o3.cfg["tables"]["rad_len"][gt.MAT_SOFT]); assert X0 > 1e29          # the slab config switches scattering off ...
    # ... which also switches this bremsstrahlung model off (it is normalised by X0): so give the slab its real X0 back
    t = tables(); X0 = float(t["rad_len"][gt.MAT_SOFT])
    t2 = tables(); t2["rad_len"][:] = 1e30; t2["rad_len"][gt.MAT_SOFT] = X0
    cfg = slab_cfg(n=(4, 4, 1), h=(5.0, 5.0, thick), w0=100.0, mode=3, t=t2, sid=100.0 + thick + 1.0)
    o = oracle.Oracle(cfg)
    o.set_fixed_primary(1, T0, (0.1, 0.1, 100.0 + 1e-9), (0, 0, 1))
    o.set_ps3(True); o.reset(); o.run(0, n, 3)
    r, ps = o.read(), o.read_ps3()
    el = ps[ps[:, 0] == 1]
    prim = np.zeros(n); np.maximum.at(prim, el[:, 7].astype(np.int64), el[:, 1])
    loss = T0 - prim[prim > 0]
    assert (prim > 0).mean() > 0.97                                     # multiple scattering in water is back on: a few do not arrive
    # mean loss of the primary over the slab = int (S_col + T / X0) ds (path a little longer than the slab because of scattering)
    S = lambda T: o.stop_pow(gt.MAT_SOFT, T) + T / X0
    sol = integrate.solve_ivp(lambda s, T: [-S(T[0])], (0, thick), [T0], rtol=1e-9)
    expect = T0 - sol.y[0, -1]
    assert loss.mean() == pytest.approx(expect, rel=0.03, abs=4 * loss.std() / np.sqrt(len(loss)))
    # photons at the plane per primary ~ int rho Sigma_brems(T(s)) ds (the slab and 1 cm of air absorb next to none of them)
    yield_exp = integrate.quad(lambda s: oracle.brems_xs(T0 - (T0 - sol.y[0, -1]) * s / thick, 0.01, X0)[0], 0, thick)[0]
    n_ph = (ps[:, 0] == 0).sum()
    assert n_ph / n == pytest.approx(yield_exp, rel=0.05, abs=4 * np.sqrt(n_ph) / n)
