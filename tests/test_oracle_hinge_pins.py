"""Pins of the oracle's physics mode 4 (remainder: DPM-style multi-voxel condensed-history steps with a
random hinge; "developed based on DPM"; reading A38).  No GPU."""
import numpy as np
import pytest
from scipy import integrate

import oracle
from gen import tables as gt
from util import slab_cfg, tables

ELECTRON = 1


def S(mat, T):
    return float(gt.stopping_power(gt.MATERIALS[mat][1], T))


def test_csda_path_and_energy_without_scattering_equal_mode_1():
    """X0 -> infinity: the total path length from T0 to the cut-off is int dT / (rho S) and all of T0 is deposited, as in mode 1
    (pin P7); the number of steps is ln(T0 / T_cut) / -ln(1 - f_E), that of segments larger (voxel faces), and no step ends on a face."""
    t = tables(); t["rad_len"][:] = 1e30
    T0 = 2.0
    ref, _ = integrate.quad(lambda T: 1.0 / S(gt.MAT_SOFT, T), 0.2, T0, epsrel=1e-10)
    res = {}
    for mode in (1, 4):
        cfg = slab_cfg(n=(8, 8, 40), h=(0.25, 0.25, 0.25), mode=mode, t=t)
        o = oracle.Oracle(cfg)
        o.set_fixed_primary(ELECTRON, T0, (0.1, 0.1, 100.0 + 1e-9), (0, 0, 1))
        o.reset(); o.run(0, 3, 1)
        res[mode] = o.read()
        assert res[mode]["ledger"][1] == pytest.approx(3 * T0, rel=1e-12)
        assert res[mode]["aux"][0] / 3 == pytest.approx(ref, rel=5e-3)
    assert res[4]["aux"][0] == pytest.approx(res[1]["aux"][0], rel=5e-3)
    n_steps = res[4]["counters"][15] / 3
    assert n_steps == np.ceil(np.log(T0 / 0.2) / -np.log(0.9))           # 22 steps of 10 % each
    assert res[4]["counters"][6] / 3 > n_steps                             # plus the segments that end on a voxel face
    # depth profile = the energy-loss ODE, voxel by voxel (as P7)
    sol = integrate.solve_ivp(lambda z, T: [-S(gt.MAT_SOFT, max(T[0], 0.01))], (0, 0.95 * ref), [T0], dense_output=True, rtol=1e-10, atol=1e-12)
    col = res[4]["phantom_sum"][:, 4, 4] / 3
    for k in range(int(np.floor(0.95 * ref / 0.25))):
        assert col[k] == pytest.approx(sol.sol(0.25 * k)[0] - sol.sol(0.25 * (k + 1))[0], rel=3e-3)


def test_depth_profile_across_a_water_bone_lung_stack():
    """A step crosses voxels of different media: each voxel gets rho S of ITS medium.  Without scattering the deposit per voxel
    follows dT/dz = -rho(z) S_m(z)(T).  Catches a loss computed with the medium of the step's start."""
    t = tables(); t["rad_len"][:] = 1e30
    cfg = slab_cfg(n=(4, 4, 60), h=(1.0, 1.0, 0.05), mode=4, t=t)
    rho, mat = cfg["phantom"]["density"], cfg["phantom"]["material"]
    rho[8:14], mat[8:14] = 1.85, gt.MAT_BONE                              # 3 mm of bone behind 4 mm of water
    rho[14:40], mat[14:40] = 0.25, gt.MAT_LUNG                            # then lung
    T0 = 3.0
    o = oracle.Oracle(cfg)
    o.set_fixed_primary(ELECTRON, T0, (0.1, 0.1, 100.0 + 1e-9), (0, 0, 1))
    o.reset(); o.run(0, 1, 1)
    col = o.read()["phantom_sum"][:, 2, 2]
    rhs = lambda z, T: [-float(rho[min(int(z / 0.05), 59), 0, 0]) * S(int(mat[min(int(z / 0.05), 59), 0, 0]), max(T[0], 0.01))]
    T = T0
    for k in range(40):
        sol = integrate.solve_ivp(rhs, (0.05 * k + 1e-12, 0.05 * (k + 1) - 1e-12), [T], rtol=1e-10, atol=1e-12)
        T1 = sol.y[0, -1]
        if T1 < 0.25:
            break
        assert col[k] == pytest.approx(T - T1, rel=4e-3), k
        T = T1
    assert k > 30


def lateral_spread(mode, f_E, n, T0=2.0, depth=0.3):
    """<x^2 + y^2> of the electrons of a pencil beam where they cross the plane `depth` cm into water (the first crossing), from the
    voxel the energy lands in: voxels of 0.02 cm across the beam, one slab behind the plane."""
    cfg = slab_cfg(n=(200, 200, 2), h=(0.02, 0.02, depth), mode=mode)
    cfg["phantom"]["origin"][2] = 100.0
    cfg["physics"]["f_E"] = f_E
    o = oracle.Oracle(cfg)
    o.set_fixed_primary(ELECTRON, T0, (0.0, 0.0, 100.0 + 1e-9), (0, 0, 1))
    o.reset(); o.run(0, n, 5)
    img = o.read()["phantom_sum"][1]                                      # the slab behind the plane: where the electrons arrive
    c = (np.arange(200) + 0.5 - 100) * 0.02
    X, Y = np.meshgrid(c, c)
    return float((img * (X ** 2 + Y ** 2)).sum() / img.sum()), float(img.sum() / n)


def test_lateral_spread_of_a_pencil_beam_matches_fine_mode_1_steps():
    """The point of the hinge: with steps four times longer the lateral spread stays that of finely stepped mode 1 (f_E = 0.02,
    the reference), where mode 1 with the same long steps (deflection at the end of a step, no displacement within it) is too narrow."""
    ref, e_ref = lateral_spread(1, 0.02, 6000)
    m4, e4 = lateral_spread(4, 0.10, 6000)
    m4c, _ = lateral_spread(4, 0.25, 6000)
    m1c, _ = lateral_spread(1, 0.25, 6000)
    assert m4 == pytest.approx(ref, rel=0.10), (m4, ref)                  # energy-weighted second moment, 6000 tracks: about 3 % noise
    assert m4c == pytest.approx(ref, rel=0.20), (m4c, ref)
    assert abs(m4c / ref - 1) < abs(m1c / ref - 1), (m4c, m1c, ref)      # the hinge beats the end-of-step deflection at the same step size
    assert e4 == pytest.approx(e_ref, rel=0.05)                           # energy carried behind the plane


def test_mode_4_ledger_and_full_configuration():
    from gen import make_config
    cfg = make_config("C1", shrink=2)
    cfg["physics"]["mode"], cfg["physics"]["f_E"] = 4, 0.2
    o = oracle.Oracle(cfg); o.reset(); o.run(0, 20000, 1)
    r = o.read(); L = r["ledger"]
    assert abs(L[1] + L[2] + L[3] + L[4] + L[5] - L[0]) < 1e-12 * L[0]
    cfg["physics"]["mode"], cfg["physics"]["f_E"] = 1, 0.1
    o1 = oracle.Oracle(cfg); o1.reset(); o1.run(0, 20000, 1)
    L1 = o1.read()["ledger"]
    assert L[1] == pytest.approx(L1[1], rel=0.02)                         # the same photons, a different electron step structure
    c4, c1 = r["counters"], o1.read()["counters"]
    # steps of 20 %: half as many deflections as mode 1 has steps, and the air gap is crossed in a few segments instead of one per cm
    assert c4[15] < 0.55 * (c1[6] + c1[7] + c1[8]) and c4[7] < 0.2 * c1[7]
