"""Pins of the oracle parts that round 1 left unpinned ("What's weak" 2): channel branching and the pair
split in interact(), annihilate(), charged steps in the air / EPID layers incl. the mid-point pixel of reading A24, and
the history-by-history sigma of flush_history() / stats().  No GPU.

Each test reads what the *transport code path itself* did (the oracle's event log: one record per interaction and per
created secondary, written by interact() / make_child()) and compares it with a closed form from gen.tables or with
kinematics.  The mistake each test would catch is named in its docstring.
"""
import numpy as np
import pytest
from scipy import integrate, stats as sst

import oracle
from gen import tables as gt
from util import slab_cfg, tables

MEC2 = 0.51099895
PHOTON, ELECTRON, POSITRON = 0, 1, 2


def run_logged(cfg, ptype, E, pos, direction, n, seed, cap=4_000_000):
    o = oracle.Oracle(cfg)
    o.set_event_log(cap)
    o.set_fixed_primary(ptype, E, pos, direction)
    o.reset()
    o.run(0, n, seed)
    return o, o.read(), o.read_event_log()


# ------------------------------------------------------------------ (a) channel branching (PAPER.md:104 interaction list)
@pytest.mark.parametrize("mat,rho", [(gt.MAT_SOFT, 1.0), (gt.MAT_GOS, 7.32)])
@pytest.mark.parametrize("E", [0.03, 1.0, 10.0])
def test_channel_branching_follows_the_partial_coefficients(mat, rho, E):
    """First interactions of a pencil beam in a homogeneous block: n_pe : n_compton : n_pair = mu_pe : mu_C : mu_pp (closed
    forms of gen.tables, not the oracle's interpolation).  Catches `x < mu[1]` instead of `x < mu[0] + mu[1]`, swapped
    table columns, a channel chosen with the wrong material's coefficients."""
    cfg = slab_cfg(n=(4, 4, 20), h=(10.0, 10.0, 1.0), rho=rho, mat=mat, E=E, mode=0)
    n = 60_000
    _, _, log = run_logged(cfg, PHOTON, E, (0.0, 0.0, 99.0), (0, 0, 1), n, 17)
    it = log[(log[:, 0] == 1) & (log[:, 2] == 0) & (log[:, 4] == E) & (log[:, 9] == mat)]   # the primary's own first interaction in the block
    assert len(it) > 0.3 * n
    obs = np.bincount(it[:, 8].astype(int), minlength=3).astype(float)
    comp = gt.MATERIALS[mat][1]
    mu = np.array([float(gt.mu_photoelectric(comp, E)), float(gt.mu_compton(comp, E)), float(gt.mu_pair(comp, E))])
    p = mu / mu.sum()
    exp = p * len(it)
    for k in range(3):
        if p[k] == 0:
            assert obs[k] == 0
        else:                                                 # binomial z-score per channel, 4.5 sigma; table interpolation error < 1e-4
            assert abs(obs[k] - exp[k]) <= 4.5 * np.sqrt(exp[k] * (1 - p[k])) + 2e-4 * exp[k] + 1, (k, obs, exp)
    # the air in front of the block (1 cm) branches with air's coefficients
    ia = log[(log[:, 0] == 1) & (log[:, 2] == 0) & (log[:, 9] == gt.MAT_AIR) & (log[:, 4] == E)]
    assert len(ia) < 0.01 * n


def test_pair_is_impossible_at_or_below_threshold():
    """Reading A34: mu_pair = 0 for E <= 2 m_e c^2 although the table cell that straddles the threshold interpolates to > 0.
    Catches a pair event with negative kinetic energy."""
    cfg = slab_cfg(n=(4, 4, 20), h=(10.0, 10.0, 1.0), rho=7.32, mat=gt.MAT_GOS, E=1.0219, mode=1)
    o = oracle.Oracle(cfg)
    assert o.mu_partial(gt.MAT_GOS, 1.0219)[2] == 0.0 and o.mu_partial(gt.MAT_GOS, 2 * MEC2)[2] == 0.0
    assert o.mu_partial(gt.MAT_GOS, 1.03)[2] > 0.0
    E_next = float(cfg["tables"]["E_grid"][np.searchsorted(cfg["tables"]["E_grid"], 2 * MEC2)])
    assert o.mu_partial(gt.MAT_GOS, E_next)[2] == pytest.approx(float(cfg["tables"]["mu_pair"][gt.MAT_GOS][np.searchsorted(cfg["tables"]["E_grid"], 2 * MEC2)]))
    _, r, log = run_logged(cfg, PHOTON, 1.0219, (0.0, 0.0, 99.0), (0, 0, 1), 30_000, 3)
    assert r["counters"][5] == 0 and not np.any((log[:, 0] == 1) & (log[:, 8] == 2))
    b = log[log[:, 0] == 2]
    assert b[:, 9].min() > 0.0                                 # no secondary is born with negative energy


# ------------------------------------------------------------------ (b) pair production (readings A10, A11)
def test_pair_split_is_uniform_and_conserves_energy():
    """Per pair event T- + T+ = E - 2 m_e c^2, T- / (T- + T+) uniform on (0, 1), both leptons along the photon's direction.
    Catches a missing rest-mass term, a split that is not uniform, a swapped or scattered lepton direction."""
    E = 10.0
    cfg = slab_cfg(n=(4, 4, 20), h=(10.0, 10.0, 1.0), rho=7.32, mat=gt.MAT_GOS, E=E, mode=1)
    d0 = np.array([0.3, -0.2, 1.0]); d0 /= np.linalg.norm(d0)
    _, r, log = run_logged(cfg, PHOTON, E, (0.0, 0.0, 99.9), tuple(d0), 20_000, 5)
    # the two leptons of an event are consecutive birth records of the same photon: electron (sibling 0), positron (sibling 1)
    ip = np.nonzero((log[:, 0] == 2) & (log[:, 3] == PHOTON) & (log[:, 8] == POSITRON) & (log[:, 13] == 1))[0]
    em, ep = log[ip - 1], log[ip]
    assert np.all((em[:, 0] == 2) & (em[:, 3] == PHOTON) & (em[:, 8] == ELECTRON) & (em[:, 13] == 0))
    assert np.array_equal(em[:, 1:3], ep[:, 1:3])
    assert len(ep) == r["counters"][5] and len(ep) > 3000       # every pair event found
    assert np.count_nonzero((log[:, 0] == 2) & (log[:, 8] == POSITRON)) == len(ep)   # positrons are born in pair events only
    Eph, Tm, Tp = ep[:, 4], em[:, 9], ep[:, 9]
    assert np.array_equal(em[:, 4], Eph)
    assert np.abs(Tm + Tp - (Eph - 2 * MEC2)).max() < 1e-12
    assert Tm.min() >= 0 and Tp.min() >= 0
    first = Eph == E                                            # pairs of the primary: one energy, a clean sample
    assert first.sum() > 2000
    assert sst.kstest(Tm[first] / (E - 2 * MEC2), "uniform").pvalue > 1e-3
    assert np.abs(em[:, 10:13] - em[:, 5:8]).max() == 0 and np.abs(ep[:, 10:13] - ep[:, 5:8]).max() == 0
    assert np.abs(em[first][:, 10:13] - d0[None]).max() < 1e-12
    # distinct Philox streams for the two leptons and for the parent (reading A1)
    assert np.all(em[:, 15] != ep[:, 15]) and np.all(em[:, 15] != em[:, 2])


# ------------------------------------------------------------------ (c) annihilation (reading A11)
@pytest.mark.parametrize("mode", [0, 1])
def test_annihilation_photons_are_back_to_back_and_isotropic(mode):
    """Two 0.511 MeV photons, exactly opposite, cos(theta) uniform on [-1, 1], azimuth uniform; emitted where the positron
    stops (mode 1) or at the pair site (mode 0).  Catches two photons in the same direction (the ledger closes all the
    same), a non-isotropic polar angle (e.g. theta uniform), a missing second photon."""
    E = 8.0
    cfg = slab_cfg(n=(4, 4, 20), h=(10.0, 10.0, 1.0), rho=7.32, mat=gt.MAT_GOS, E=E, mode=mode)
    _, r, log = run_logged(cfg, PHOTON, E, (0.0, 0.0, 99.9), (0, 0, 1), 20_000, 6)
    parent = PHOTON if mode == 0 else POSITRON
    b = log[(log[:, 0] == 2) & (log[:, 3] == parent) & (log[:, 8] == PHOTON)]
    a, c = b[b[:, 13] == 0], b[b[:, 13] == 1]
    n_pair = int(r["counters"][5])
    assert len(a) == len(c) > 2000                              # never one photon without the other
    assert len(a) == n_pair if mode == 0 else 0.99 * n_pair < len(a) <= n_pair   # mode 1: a few positrons leave through the top face and the world
    assert np.array_equal(a[:, 1:3], c[:, 1:3])                 # consecutive records of the same parent
    assert np.all(a[:, 9] == MEC2) and np.all(c[:, 9] == MEC2)
    assert np.abs(a[:, 10:13] + c[:, 10:13]).max() < 1e-15      # exactly opposite
    assert np.abs(np.linalg.norm(a[:, 10:13], axis=1) - 1).max() < 1e-12
    ct, phi = a[:, 12], np.arctan2(a[:, 11], a[:, 10])
    assert sst.kstest((ct + 1) / 2, "uniform").pvalue > 1e-3
    assert sst.kstest((phi + np.pi) / (2 * np.pi), "uniform").pvalue > 1e-3
    if mode == 1:
        assert np.all(a[:, 4] <= 0.2)                           # the positron had reached its cut-off
    L = r["ledger"]
    assert abs(L[1] + L[2] + L[3] + L[4] + L[5] - L[0]) < 1e-12 * L[0]


def test_positron_leaving_the_world_carries_its_rest_energy():
    """Reading A11: a positron that escapes books T + 2 m_e c^2.  Catches an escape that forgets the rest energy and an
    annihilation at the world boundary."""
    cfg = slab_cfg(n=(4, 4, 4), h=(1.0, 1.0, 1.0), mode=1)
    T0, n = 1.5, 200
    o, r, log = run_logged(cfg, POSITRON, T0, (0.0, 0.0, 30.0), (0, 0, -1), n, 2)
    L = r["ledger"]
    assert L[0] == pytest.approx(n * (T0 + 2 * MEC2), rel=1e-14)
    assert abs(L[4] + L[5] - L[0]) < 1e-12 * L[0] and L[1] == L[2] == L[3] == 0
    S_air = float(gt.stopping_power(gt.MATERIALS[gt.MAT_AIR][1], T0))
    loss = gt.RHO_AIR * 31.0 * S_air                                # 31 cm of air at nearly constant S (0.4 % of T0)
    assert L[4] / n == pytest.approx(loss, rel=0.03)                # a little more: multiple scattering lengthens the path
    assert L[5] / n == pytest.approx(T0 - L[4] / n + 2 * MEC2, rel=1e-12)
    assert not np.any(log[:, 0] == 2)                               # no annihilation photons


# ------------------------------------------------------------------ (d) charged steps outside the phantom (reading A24)
def _epid_cfg(layers, nu=64, nv=64, pitch=0.4, sid=150.0, X0=1e30):
    t = tables()
    t["rad_len"][:] = X0
    cfg = slab_cfg(n=(4, 4, 4), h=(1.0, 1.0, 1.0), mode=1, t=t, sid=sid)
    cfg["epid"] = {"thickness": np.array([l[0] for l in layers], np.float32), "material": np.array([l[1] for l in layers], np.uint8),
                   "density": np.array([gt.MATERIALS[l[1]][2] for l in layers], np.float32),
                   "scored": np.array([l[2] for l in layers], np.uint8), "sid": sid, "nu": nu, "nv": nv, "pitch": pitch}
    return cfg


def test_csda_in_a_thick_epid_layer():
    """P7 in the EPID frame: no scattering, thick Cu layer: path length = int dT / (rho S), everything deposited in the
    layer's pixel.  Catches a wrong density / material in the layer branch and a deposit that misses the image."""
    cfg = _epid_cfg([(1.0, gt.MAT_CU, 1)])
    T0 = 2.0
    o = oracle.Oracle(cfg)
    o.set_fixed_primary(ELECTRON, T0, (0.1, -0.3, 150.0 + 1e-9), (0, 0, 1))
    o.reset(); o.run(0, 2, 1)
    r = o.read()
    S = lambda T: float(gt.stopping_power(gt.MATERIALS[gt.MAT_CU][1], T))
    ref, _ = integrate.quad(lambda T: 1.0 / (8.96 * S(T)), 0.2, T0, epsrel=1e-10)
    # the last step ends up to 10 % below the cut-off (the rest is deposited there), i.e. up to half a last
    # step = 0.4 % of the path beyond the integral; the midpoint rule itself is O(f_E^2)
    assert r["aux"][0] / 2 == pytest.approx(ref, rel=5e-3)
    assert r["aux"][1] / 2 == pytest.approx(8.96 * ref, rel=5e-3)
    assert r["ledger"][2] == pytest.approx(2 * T0, rel=1e-12)
    iu, iv = int(np.floor((0.1 + 32 * 0.4) / 0.4)), int(np.floor((-0.3 + 32 * 0.4) / 0.4))
    assert r["epid_sum"][iv, iu] == pytest.approx(2 * T0, rel=1e-12)


def test_layer_crossing_deposits_follow_the_energy_loss_ode():
    """A 6 MeV electron straight through the four-layer stack without scattering: the deposit in each layer is the loss of
    dT/dz = -rho_l S_l(T) over that layer, the rest leaves through the bottom.  Catches a layer index that is not advanced,
    a deposit booked to the neighbouring layer and a wrong layer density."""
    spec = [(0.1, gt.MAT_CU), (0.029, gt.MAT_GOS), (0.1, gt.MAT_GLASS), (0.2, gt.MAT_PMMA)]
    T, exp = 6.0, []
    for th, m in spec:
        S = lambda z, y, m=m: [-gt.MATERIALS[m][2] * float(gt.stopping_power(gt.MATERIALS[m][1], max(y[0], 0.01)))]
        sol = integrate.solve_ivp(S, (0, th), [T], rtol=1e-10, atol=1e-12)
        exp.append(T - sol.y[0, -1]); T = sol.y[0, -1]
    for k in range(4):
        cfg = _epid_cfg([(th, m, int(i == k)) for i, (th, m) in enumerate(spec)])
        o = oracle.Oracle(cfg)
        o.set_fixed_primary(ELECTRON, 6.0, (0.0, 0.0, 149.0), (0, 0, 1))   # starts in the air 1 cm above the stack
        o.reset(); o.run(0, 1, 1)
        L = o.read()["ledger"]
        assert L[2] == pytest.approx(exp[k], rel=3e-3), k
        assert L[3] == pytest.approx(sum(exp) - exp[k], rel=3e-3)
        assert L[5] == pytest.approx(T - L[4], rel=3e-3) and L[4] < 3e-3    # 1 cm of air costs 2 keV
        assert abs(L[2] + L[3] + L[4] + L[5] - 6.0) < 1e-12


def test_lateral_escape_from_a_layer():
    """An electron that runs sideways inside a layer leaves the world at |u| = 100 cm with what the ODE leaves it."""
    cfg = _epid_cfg([(1.0, gt.MAT_PMMA, 0)])
    o = oracle.Oracle(cfg)
    o.set_fixed_primary(ELECTRON, 3.0, (99.8, 0.0, 150.5), (1, 0, 0))
    o.reset(); o.run(0, 1, 1)
    L = o.read()["ledger"]
    S = lambda z, y: [-1.19 * float(gt.stopping_power(gt.MATERIALS[gt.MAT_PMMA][1], y[0]))]
    T_out = integrate.solve_ivp(S, (0, 0.2), [3.0], rtol=1e-10, atol=1e-12).y[0, -1]
    assert L[5] == pytest.approx(T_out, rel=1e-3) and L[3] == pytest.approx(3.0 - T_out, rel=3e-2) and L[2] == 0


def test_step_energy_goes_to_the_pixel_of_the_step_midpoint():
    """Reading A24, hand-worked: an electron runs obliquely inside the scored layer without scattering; steps are
    s_k = f_E T_k / (rho S(T_k)) (the layer faces and s_max are far), each deposit goes to the pixel under the step's
    mid-point.  The pixel pitch is chosen so that start, mid-point and end of every step lie in different pixels: an
    oracle that scored at either end of the step fails."""
    cfg = _epid_cfg([(0.5, gt.MAT_GOS, 1)], nu=512, nv=16, pitch=0.004)
    T0, u0, v0 = 2.0, -0.5031, 0.0021
    d = np.array([0.995, 0.0, np.sqrt(1 - 0.995**2)])
    o = oracle.Oracle(cfg)
    o.set_fixed_primary(ELECTRON, T0, (u0, v0, 150.0 + 1e-7), tuple(d))
    o.reset(); o.run(0, 1, 1)
    img = o.read()["epid_sum"]
    S = lambda T: o.stop_pow(gt.MAT_GOS, T)                          # unit-level table look-up (pinned against the closed form)
    rho, T, u, exp, ends = 7.32, T0, u0, {}, {}
    for _ in range(12):                                              # the first twelve steps by hand
        s = 0.1 * T / (rho * S(T))
        dE = rho * s * S(T - 0.5 * rho * s * S(T))
        pix = lambda uu: int(np.floor((uu + 256 * 0.004) / 0.004))
        exp[pix(u + 0.5 * s * d[0])] = exp.get(pix(u + 0.5 * s * d[0]), 0.0) + dE
        assert len({pix(u), pix(u + 0.5 * s * d[0]), pix(u + s * d[0])}) == 3
        ends[pix(u + s * d[0])] = dE
        u += s * d[0]; T -= dE
    row = int(np.floor((v0 + 8 * 0.004) / 0.004))
    for p, e in exp.items():
        assert img[row, p] == pytest.approx(e, rel=1e-9), p
    first = sorted(exp)[0]
    assert img[row, :first].sum() == 0                               # nothing upstream of the first mid-point (not even the start pixel)
    assert img.sum() == pytest.approx(T0, rel=1e-12) and img[row].sum() == pytest.approx(T0, rel=1e-12)


def test_electron_handed_from_air_into_the_stack():
    """Air -> EPID hand-off of a charged particle: the air step ends on the top plane, the rest is lost in the stack."""
    cfg = _epid_cfg([(1.0, gt.MAT_CU, 1)])
    o = oracle.Oracle(cfg)
    o.set_fixed_primary(ELECTRON, 1.0, (0.0, 0.0, 140.0), (0, 0, 1))
    o.reset(); o.run(0, 1, 1)
    r = o.read(); L = r["ledger"]
    S_air = float(gt.stopping_power(gt.MATERIALS[gt.MAT_AIR][1], 1.0))
    assert L[4] == pytest.approx(gt.RHO_AIR * 10.0 * S_air, rel=5e-3)
    assert L[2] == pytest.approx(1.0 - L[4], rel=1e-12) and L[5] == 0
    assert r["counters"][7] >= 10 and r["counters"][8] > 10          # steps of at most s_max = 1 cm in air, then steps in Cu


# ------------------------------------------------------------------ (e) the sigma estimator
def test_history_by_history_sigma_equals_the_binomial_closed_form():
    """P6 set-up (photoelectric only, kerma): the deposit of a history in depth bin k is E with probability p_k, else 0, so
    sigma of the mean is E sqrt(p_k (1 - p_k) / n); the estimator's own relative error is about sqrt((1/p_k - 3) / 4n) ... 2 %.
    Catches a missing mean^2 term, n instead of n - 1 at small n, a per-deposit instead of per-history square."""
    t = tables()
    t["mu_compton"][:] = 0.0; t["mu_pair"][:] = 0.0
    t["mu_pe"][gt.MAT_SOFT] *= 20.0
    E = 0.06
    cfg = slab_cfg(n=(8, 8, 20), h=(1.0, 1.0, 1.0), E=E, mode=0, t=t)
    o = oracle.Oracle(cfg)
    o.set_fixed_primary(0, E, (0.5, 0.5, 50.0), (0, 0, 1))
    o.reset()
    n = 200_000
    o.run(0, n, 8)
    st = oracle.stats(o.read())
    mu = 20.0 * float(gt.mu_photoelectric(gt.MATERIALS[gt.MAT_SOFT][1], E))
    mu_a = float(gt.mu_photoelectric(gt.MATERIALS[gt.MAT_AIR][1], E)) * gt.RHO_AIR
    z = np.arange(21, dtype=float)
    pk = np.exp(-mu_a * 50.0) * (np.exp(-mu * z[:-1]) - np.exp(-mu * z[1:]))
    sig = st["phantom_sigma"][:, 4, 4]
    ref = E * np.sqrt(pk * (1 - pk) / n)
    use = pk * n > 400
    assert use.sum() >= 8
    rel_err = np.sqrt((1.0 / pk[use]) / (4 * n))                     # relative sampling error of an estimated binomial sigma
    assert np.all(np.abs(sig[use] / ref[use] - 1) < 4.5 * rel_err + 1e-5)
    # the ledger channel: dep_phantom per history is E x Bernoulli(P), P = sum p_k
    P = pk.sum()
    assert st["ledger_sigma"][1] == pytest.approx(E * np.sqrt(P * (1 - P) / n), rel=0.02)
    assert st["ledger_mean"][1] == pytest.approx(E * P, abs=4.5 * E * np.sqrt(P * (1 - P) / n))
    # tiny n: the n - 1 of the unbiased estimator
    o.reset(); o.run(0, 2, 8)
    raw = o.read(); s, q = raw["ledger"][1], raw["ledger_sq"][1]
    assert oracle.stats(raw)["ledger_sigma"][1] == pytest.approx(np.sqrt(max(q / 2 - (s / 2) ** 2, 0.0) / 1.0))


def test_coarse_phantom_tally_is_the_block_sum_with_its_own_variance():
    """The coarse phantom tally (used by the full-size GPU parity tests) sums blocks of voxels history by history: its
    mean is the block sum of the fine tally, its variance is at least the sum of the voxel variances (deposits of one
    history in neighbouring voxels are positively correlated)."""
    from gen import make_config
    cfg = make_config("C1", shrink=4)
    o = oracle.Oracle(cfg); o.set_phantom_rebin(3, 2, 4); o.reset(); o.run(0, 4000, 3)
    raw = o.read()
    f = raw["phantom_sum"]; nz, ny, nx = f.shape
    blk = f.reshape(nz // 4, 4, ny // 2, 2, nx // 3, 3).sum(axis=(1, 3, 5))
    assert np.allclose(raw["pc_sum"], blk, rtol=1e-12, atol=1e-15)
    q = raw["phantom_sq"].reshape(nz // 4, 4, ny // 2, 2, nx // 3, 3).sum(axis=(1, 3, 5))
    assert np.all(raw["pc_sq"] >= q * (1 - 1e-12))
    assert raw["pc_sq"].sum() > 1.2 * q.sum()
