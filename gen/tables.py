"""Parametric material tables (inputs of `aepid_init_materials`).

BASELINE.json:configs[0] prescribes parametric cross sections ("Klein-Nishina
per electron times electron density, photoelectric proportional to Z^4/E^3,
and a pair threshold formula, generated at 1 keV-20 MeV on a 500-point log
grid"); SURVEY.md 8(c) fixes every constant.  DPM/NIST data are not available
and are not recreated here.  The tables are evaluated in float64 and stored as
float32; how they are interpolated is the business of the consumer.

Units: MeV, cm, g.  Photon tables are mass coefficients [cm^2/g], stopping
power is mass collision stopping power [MeV cm^2/g], radiation length [g/cm^2].
"""
from __future__ import annotations

import numpy as np

R_E = 2.8179403262e-13        # classical electron radius, cm
MEC2 = 0.51099895             # electron rest energy, MeV
N_A = 6.02214076e23           # 1/mol
ALPHA = 7.2973525693e-3       # fine-structure constant
C_PE = 2.0e-32                # cm^2 MeV^3, photoelectric anchor
K_STOP = 2.0 * np.pi * R_E**2 * MEC2 * N_A   # 0.1535375 MeV cm^2/mol

# element -> (Z, A [g/mol], mean excitation energy I [eV])
ELEMENTS = {
    "H": (1, 1.008, 19.2), "C": (6, 12.011, 81.0), "N": (7, 14.007, 82.0),
    "O": (8, 15.999, 95.0), "Na": (11, 22.990, 149.0), "Mg": (12, 24.305, 156.0),
    "Si": (14, 28.085, 173.0), "P": (15, 30.974, 173.0), "S": (16, 32.06, 180.0),
    "Ar": (18, 39.948, 188.0), "Ca": (20, 40.078, 191.0), "Cu": (29, 63.546, 322.0),
    "Gd": (64, 157.25, 591.0), "W": (74, 183.84, 727.0),
}

_WATER = {"H": 0.111894, "O": 0.888106}
# index -> (name, mass fractions, nominal density g/cm^3)   (SURVEY 8(c) "Materials")
MATERIALS = [
    ("air", {"C": 0.000124, "N": 0.755268, "O": 0.231781, "Ar": 0.012827}, 1.205e-3),
    ("lung", _WATER, 0.25),
    ("soft", _WATER, 1.0),
    ("bone", {"H": 0.034, "C": 0.155, "N": 0.042, "O": 0.435, "Na": 0.001,
              "Mg": 0.002, "P": 0.103, "S": 0.003, "Ca": 0.225}, 1.85),
    ("Cu", {"Cu": 1.0}, 8.96),
    ("Gd2O2S", {"Gd": 0.830784, "O": 0.084526, "S": 0.084690}, 7.32),
    ("glass", {"Si": 0.467435, "O": 0.532565}, 2.40),
    ("PMMA", {"H": 0.080538, "C": 0.599848, "O": 0.319614}, 1.19),
]
MAT_AIR, MAT_LUNG, MAT_SOFT, MAT_BONE, MAT_CU, MAT_GOS, MAT_GLASS, MAT_PMMA = range(8)
RHO_AIR = 1.205e-3
# Jaws and MLC leaves of the collimation stage: tungsten.  Not part of MATERIALS, so that the tables of
# C0-C4 keep their eight materials; make_tables(extra=(TUNGSTEN,)) appends it as material 8.
TUNGSTEN = ("W", {"W": 1.0}, 19.3)
MAT_W = 8


def sigma_kn(E):
    """Total Klein-Nishina cross section per electron [cm^2] (closed form)."""
    k = np.asarray(E, dtype=np.float64) / MEC2
    a = (1 + k) / k**2 * (2 * (1 + k) / (1 + 2 * k) - np.log1p(2 * k) / k)
    b = np.log1p(2 * k) / (2 * k)
    c = (1 + 3 * k) / (1 + 2 * k) ** 2
    return 2 * np.pi * R_E**2 * (a + b - c)


def _fractions(comp):
    tot = sum(comp.values())
    return {el: w / tot for el, w in comp.items()}


def mu_compton(comp, E):
    ne = N_A * sum(w * ELEMENTS[el][0] / ELEMENTS[el][1] for el, w in _fractions(comp).items())
    return ne * sigma_kn(E)


def mu_photoelectric(comp, E):
    E = np.asarray(E, dtype=np.float64)
    s = sum(w / ELEMENTS[el][1] * ELEMENTS[el][0] ** 4 for el, w in _fractions(comp).items())
    return N_A * s * C_PE / E**3


def mu_pair(comp, E):
    E = np.asarray(E, dtype=np.float64)
    eth = 2 * MEC2
    s = sum(w / ELEMENTS[el][1] * ELEMENTS[el][0] ** 2 for el, w in _fractions(comp).items())
    x = np.maximum(E, eth)
    per_z2 = (28.0 / 9.0) * ALPHA * R_E**2 * np.log(x / eth) * (1 - eth / x) ** 2
    return np.where(E > eth, N_A * s * per_z2, 0.0)


def stopping_power(comp, T):
    """Collision mass stopping power for electrons, no density effect."""
    T = np.asarray(T, dtype=np.float64)
    fr = _fractions(comp)
    za = sum(w * ELEMENTS[el][0] / ELEMENTS[el][1] for el, w in fr.items())
    ln_i = sum(w * ELEMENTS[el][0] / ELEMENTS[el][1] * np.log(ELEMENTS[el][2] * 1e-6)
               for el, w in fr.items()) / za          # ln(I/MeV), Bragg additivity
    i_rel = np.exp(ln_i) / MEC2
    tau = T / MEC2
    beta2 = tau * (tau + 2) / (tau + 1) ** 2
    br = (np.log(tau**2 * (tau + 2) / (2 * i_rel**2)) + 1 - beta2
          + (tau**2 / 8 - (2 * tau + 1) * np.log(2)) / (tau + 1) ** 2)
    return K_STOP * za / beta2 * br


def radiation_length(comp):
    inv = 0.0
    for el, w in _fractions(comp).items():
        z, a, _ = ELEMENTS[el]
        x0 = 716.4 * a / (z * (z + 1) * np.log(287.0 / np.sqrt(z)))
        inv += w / x0
    return 1.0 / inv


def make_tables(n_E=500, E_min=1e-3, E_max=20.0, n_T=200, T_min=0.01, T_max=20.0, extra=(), E_grid=None):
    """All material tables, float32, in the layout of `aepid_init_materials`; `extra` appends materials to MATERIALS.
    `E_grid`: an explicit (increasing, not necessarily log-uniform) photon energy grid instead of the n_E-point log grid."""
    E = np.exp(np.linspace(np.log(E_min), np.log(E_max), n_E)) if E_grid is None else np.asarray(E_grid, dtype=np.float64)
    n_E = len(E)
    T = np.exp(np.linspace(np.log(T_min), np.log(T_max), n_T))
    mats = list(MATERIALS) + list(extra)
    n_mat = len(mats)
    mc = np.empty((n_mat, n_E)); mp = np.empty((n_mat, n_E)); mpp = np.empty((n_mat, n_E))
    sp = np.empty((n_mat, n_T)); x0 = np.empty(n_mat); ne = np.empty(n_mat)
    for m, (_, comp, _) in enumerate(mats):
        mc[m] = mu_compton(comp, E)
        mp[m] = mu_photoelectric(comp, E)
        mpp[m] = mu_pair(comp, E)
        sp[m] = stopping_power(comp, T)
        x0[m] = radiation_length(comp)
        ne[m] = N_A * sum(w * ELEMENTS[el][0] / ELEMENTS[el][1] for el, w in _fractions(comp).items())
    f32 = lambda a: np.ascontiguousarray(a, dtype=np.float32)
    return {
        "n_mat": n_mat, "names": [m[0] for m in mats],
        "E_grid": f32(E), "mu_compton": f32(mc), "mu_pe": f32(mp), "mu_pair": f32(mpp),
        "T_grid": f32(T), "stop_pow": f32(sp), "rad_len": f32(x0),
        "electrons_per_gram": f32(ne),      # N_A sum_i w_i Z_i / A_i: input of the Class II (Moller) mode
    }


GD_K_EDGE = 0.050239          # MeV, K absorption edge of gadolinium


def edge_resolving_tables(n_coarse=90, jump=5.2, seed=5):
    """Tables on a NON-UNIFORM photon grid of the kind real tabulations come on (SURVEY 8(f) NEXT-2 "drop-in NIST/DPM-format
    cross-section files"): a coarse, irregularly spaced grid (seeded jitter) that is refined around an absorption edge and
    carries the edge as two grid points a relative 2e-6 apart.  The edge itself is synthetic (the parametric Z^4/E^3
    photoelectric formula has none): the photoelectric coefficient of Gd2O2S is multiplied by `jump` at and above the Gd K edge.
    Inputs only: the consumer interpolates as it sees fit."""
    rng = np.random.default_rng(seed)
    ln = np.linspace(np.log(1e-3), np.log(20.0), n_coarse)
    ln[1:-1] += rng.uniform(-0.3, 0.3, n_coarse - 2) * (ln[1] - ln[0])
    E = np.exp(ln)
    near = GD_K_EDGE * np.exp(np.array([-0.2, -0.1, -0.05, -0.02, -0.005, 0.005, 0.02, 0.05, 0.1, 0.2]))
    E = np.sort(np.concatenate([E[np.abs(np.log(E / GD_K_EDGE)) > 0.25], near, [GD_K_EDGE * (1 - 1e-6), GD_K_EDGE * (1 + 1e-6)]]))
    t = make_tables(E_grid=E)
    Ef = t["E_grid"].astype(np.float64)
    assert np.all(np.diff(Ef) > 0)
    t["mu_pe"][MAT_GOS, Ef > GD_K_EDGE] *= np.float32(jump)
    t["edge"] = {"material": MAT_GOS, "E": GD_K_EDGE, "jump": jump}
    return t
