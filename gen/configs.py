"""Seeded synthetic workloads C0..C4 (BASELINE.json:configs[0..4]).

The paper's clinical plans, CT sets and the AS1200 layer specification are not
available (PAPER.md:127-141 only describes them); these inputs stand in for
them.  Every array is produced from a numpy `default_rng(seed)`; nothing is
read from disk.  Layouts follow `include/aepid.h`:
phantom [nz][ny][nx] (x fastest) in the phantom's own frame, fluence [fv][fu]
(u fastest), LUT [nt][ns].

World frame = phantom (CT) frame.  `beam_axes` rows are the unit vectors u, v,
w of the beam frame written in world coordinates; the source sits at `src_pos`
and the beam travels along +w (SURVEY 8(c) "Geometry", readings A2-A6).
"""
from __future__ import annotations

import numpy as np

from .tables import (make_tables, MATERIALS, MAT_AIR, MAT_LUNG, MAT_SOFT, MAT_BONE,
                     MAT_CU, MAT_GOS, MAT_GLASS, MAT_PMMA, TUNGSTEN, MAT_W)

CONFIG_NAMES = ("C0", "C1", "C2", "C3", "C4")

_IDENT = np.eye(3, dtype=np.float32)
# C2/C3: u = CT x, v = CT z, w = CT y (reading A5)
_AXES_Y = np.array([[1, 0, 0], [0, 0, 1], [0, 1, 0]], dtype=np.float32)


def default_physics(mode=1, n_batches=32):
    # PAPER.md:104 cutoffs 10 keV / 200 keV; SURVEY A13 step rule.
    return {"mode": int(mode), "photon_cut": 0.010, "electron_cut": 0.200,
            "f_E": 0.10, "s_max": 1.0, "n_batches": int(n_batches)}


def epid_stack(kind, nu, nv, pitch, sid):
    """EPID slab stacks of configs[0] and configs[1] (order along +w, reading A21)."""
    if kind == "C0":
        layers = [(0.1, MAT_CU, 0), (0.03, MAT_GOS, 1)]
    else:
        layers = [(0.1, MAT_CU, 0), (0.029, MAT_GOS, 1), (0.1, MAT_GLASS, 0), (0.2, MAT_PMMA, 0)]
    return {
        "thickness": np.array([l[0] for l in layers], dtype=np.float32),
        "material": np.array([l[1] for l in layers], dtype=np.uint8),
        "density": np.array([MATERIALS[l[1]][2] for l in layers], dtype=np.float32),
        "scored": np.array([l[2] for l in layers], dtype=np.uint8),
        "sid": float(sid), "nu": int(nu), "nv": int(nv), "pitch": float(pitch),
    }


def mono_spectrum(E):
    return (np.array([E, E], dtype=np.float32), np.array([1.0], dtype=np.float32))


def mv6_spectrum(n_bins=200, lo=0.1, hi=6.0):
    """Schiff-shaped 6 MV stand-in (configs[1]): p ~ (6/E - 1) exp(-0.8/E) at bin centres."""
    edges = np.linspace(lo, hi, n_bins + 1)
    c = 0.5 * (edges[:-1] + edges[1:])
    p = (hi / c - 1.0) * np.exp(-0.8 / c)
    p = np.maximum(p, 0.0)
    p /= p.sum()
    return edges.astype(np.float32), p.astype(np.float32)


def open_field(size_cm=10.0, pitch=0.1):
    n = int(round(size_cm / pitch))
    return np.ones((n, n), dtype=np.float32), pitch


def mlc_fluence(seed, n_rect=(8, 15), field_cm=None, n_px=200, pitch=0.1, leaf_px=5):
    """Seeded sum of rectangular MLC-style apertures (configs[2], configs[4]).

    Every rectangle spans an integer number of 5 mm leaves in v and a random
    interval in u, with a uniform(0.1, 1) weight.  `field_cm` confines all
    apertures to the central field_cm x field_cm square.
    """
    rng = np.random.default_rng(seed)
    f = np.zeros((n_px, n_px), dtype=np.float64)
    n_leaf = n_px // leaf_px
    k = int(rng.integers(n_rect[0], n_rect[1] + 1))
    if field_cm is None:
        lo_px, hi_px = 0, n_px
    else:
        half = int(round(0.5 * field_cm / pitch))
        lo_px, hi_px = n_px // 2 - half, n_px // 2 + half
    lo_leaf, hi_leaf = -(-lo_px // leaf_px), hi_px // leaf_px
    for _ in range(k):
        nl = int(rng.integers(1, max(2, (hi_leaf - lo_leaf) // 2 + 1)))
        l0 = int(rng.integers(lo_leaf, hi_leaf - nl + 1))
        wmin = min(10, hi_px - lo_px)
        wu = int(rng.integers(wmin, hi_px - lo_px + 1))
        u0 = int(rng.integers(lo_px, hi_px - wu + 1))
        f[l0 * leaf_px:(l0 + nl) * leaf_px, u0:u0 + wu] += rng.uniform(0.1, 1.0)
    return f.astype(np.float32), pitch


def hu_to_density_material(hu):
    """Piecewise-linear HU table (reading A22)."""
    rho = np.where(hu <= 0, np.maximum(0.0012, 1.0 + hu / 1000.0), 1.0 + 0.6 * hu / 1000.0)
    mat = np.full(hu.shape, MAT_BONE, dtype=np.uint8)
    mat[hu < 200] = MAT_SOFT
    mat[hu < -300] = MAT_LUNG
    mat[hu < -900] = MAT_AIR
    return rho.astype(np.float32), mat


def _grid_axes(n, h):
    return [(np.arange(n[a], dtype=np.float32) + 0.5) * h[a] - 0.5 * n[a] * h[a] for a in range(3)]


def phantom_water(n, h, origin, rho=1.0, mat=MAT_SOFT):
    nx, ny, nz = n
    return {"nx": nx, "ny": ny, "nz": nz,
            "spacing": np.array(h, dtype=np.float32), "origin": np.array(origin, dtype=np.float32),
            "density": np.full((nz, ny, nx), rho, dtype=np.float32),
            "material": np.full((nz, ny, nx), mat, dtype=np.uint8)}


def phantom_thorax_c2(seed=42, n=(256, 256, 128), h=(0.15, 0.15, 0.25)):
    """configs[2]: elliptic-cylinder body, two lungs, one bone cylinder; centred on the origin."""
    rng = np.random.default_rng(seed)
    x, y, z = _grid_axes(n, h)
    X = x[None, None, :]; Y = y[None, :, None]; Z = z[:, None, None]
    hu = np.full((n[2], n[1], n[0]), -1000.0, dtype=np.float32)
    body = (X / 17.0) ** 2 + (Y / 11.0) ** 2 <= 1.0
    body = np.broadcast_to(body, hu.shape)
    noise = rng.normal(0.0, 20.0, size=hu.shape).astype(np.float32)
    hu[body] = noise[body]
    for cx in (-8.5, 8.5):
        lung = ((X - cx) / 6.0) ** 2 + (Y / 7.5) ** 2 + (Z / 10.0) ** 2 <= 1.0
        hu[lung] = -750.0
    bone = np.broadcast_to(X ** 2 + (Y - 6.0) ** 2 <= 1.8 ** 2, hu.shape)
    hu[bone] = 900.0
    rho, mat = hu_to_density_material(hu)
    ext = np.array(n) * np.array(h)
    return {"nx": n[0], "ny": n[1], "nz": n[2], "spacing": np.array(h, dtype=np.float32),
            "origin": (-0.5 * ext).astype(np.float32), "density": rho, "material": mat}


def phantom_patient_c3(seed=44, n=(512, 512, 200), h=(0.1, 0.1, 0.25)):
    """configs[3]: nested ellipsoids (fat shell, muscle, lungs, spine, rib rings), noise sigma 15 HU."""
    rng = np.random.default_rng(seed)
    x, y, z = _grid_axes(n, h)
    X = x[None, None, :]; Y = y[None, :, None]
    rho = np.empty((n[2], n[1], n[0]), dtype=np.float32)
    mat = np.empty((n[2], n[1], n[0]), dtype=np.uint8)
    rib_z = -11.25 + 2.5 * np.arange(10)
    for k in range(n[2]):                       # slab by slab to bound memory
        zk = z[k]
        hu = np.full((n[1], n[0]), -1000.0, dtype=np.float32)
        e_out = (X[0] / 19.0) ** 2 + (Y[0] / 12.5) ** 2 + (zk / 40.0) ** 2
        e_in = (X[0] / 17.5) ** 2 + (Y[0] / 11.0) ** 2 + (zk / 38.5) ** 2
        hu[e_out <= 1.0] = -100.0
        hu[e_in <= 1.0] = 40.0
        for cx in (-8.0, 8.0):
            lung = ((X[0] - cx) / 5.5) ** 2 + (Y[0] / 7.0) ** 2 + (zk / 11.0) ** 2 <= 1.0
            hu[lung] = -800.0
        if np.min(np.abs(rib_z - zk)) <= 0.4:
            r_in = (X[0] / 15.5) ** 2 + (Y[0] / 9.5) ** 2
            r_out = (X[0] / 16.3) ** 2 + (Y[0] / 10.3) ** 2
            hu[(r_in > 1.0) & (r_out <= 1.0)] = 1000.0
        hu[X[0] ** 2 + (Y[0] - 7.0) ** 2 <= 1.8 ** 2] = 1000.0
        inside = e_out <= 1.0
        hu = np.where(inside, hu + rng.normal(0.0, 15.0, size=hu.shape).astype(np.float32), hu)
        rho[k], mat[k] = hu_to_density_material(hu)
    ext = np.array(n) * np.array(h)
    return {"nx": n[0], "ny": n[1], "nz": n[2], "spacing": np.array(h, dtype=np.float32),
            "origin": (-0.5 * ext).astype(np.float32), "density": rho, "material": mat}


def response_lut(seed=46, nt=64, ns=64, t_rng=(0.0, 40.0), s_rng=(2.0, 25.0)):
    """configs[4]: smooth seeded surface in [0.85, 1.15] over (thickness, field size)."""
    rng = np.random.default_rng(seed)
    t = np.linspace(t_rng[0], t_rng[1], nt)[:, None]
    s = np.linspace(s_rng[0], s_rng[1], ns)[None, :]
    g = np.zeros((nt, ns))
    for _ in range(3):
        a = rng.uniform(0.3, 1.0); ft = rng.uniform(0.2, 1.5); hs = rng.uniform(0.2, 1.5)
        ph = rng.uniform(0, 2 * np.pi)
        g += a * np.sin(2 * np.pi * (ft * t / t_rng[1] + hs * (s - s_rng[0]) / (s_rng[1] - s_rng[0])) + ph)
    k = 1.0 + 0.15 * g / np.abs(g).max()
    return {"lut": k.astype(np.float32), "nt": nt, "ns": ns,
            "t_min": t_rng[0], "t_max": t_rng[1], "s_min": s_rng[0], "s_max": s_rng[1]}


# PAPER.md:157-162, Table 1: rows = field size 5/10/15/20 cm, columns = thickness 0..20 cm.
PAPER_TABLE1_ROWS_S = np.array([
    [0.999, 0.974, 0.960, 0.949, 0.949],
    [1.001, 0.975, 0.967, 0.964, 0.953],
    [0.995, 0.982, 0.983, 0.996, 0.986],
    [0.991, 0.997, 1.015, 1.034, 1.043]], dtype=np.float32)


def paper_table1_lut():
    """Table 1 in the library's [nt][ns] order (reading A18)."""
    return {"lut": np.ascontiguousarray(PAPER_TABLE1_ROWS_S.T), "nt": 5, "ns": 4,
            "t_min": 0.0, "t_max": 20.0, "s_min": 5.0, "s_max": 20.0}


def _source(src_pos, axes, spectrum, fluence, pitch, plane=100.0):
    edges, pdf = spectrum
    return {"src_pos": np.array(src_pos, dtype=np.float32), "beam_axes": np.ascontiguousarray(axes, dtype=np.float32),
            "E_edges": edges, "E_pdf": pdf, "fu": int(fluence.shape[1]), "fv": int(fluence.shape[0]),
            "f_pitch": float(pitch), "f_plane_dist": float(plane), "fluence": np.ascontiguousarray(fluence)}


def calibration_config(t_cm, s_cm, tables=None):
    """One point of the k(t, s) calibration of PAPER.md:114 (section 2.2): a solid-water slab of thickness t_cm centred at the
    isocentre (30 x 30 cm, 0.5 cm voxels laterally, 1 cm along the beam), an open s_cm x s_cm field, the C1 EPID stack scored on
    the paper's 160 x 160 grid of 2.5 mm.  t_cm = 0 ("no phantom") is a 1 cm slab of density 1e-6."""
    t = tables if tables is not None else make_tables()
    nz = max(int(round(t_cm)), 1)
    ph = phantom_water((60, 60, nz), (0.5, 0.5, (t_cm if t_cm > 0 else 1.0) / nz), (-15.0, -15.0, 100.0 - 0.5 * (t_cm if t_cm > 0 else 1.0)),
                       rho=1.0 if t_cm > 0 else 1e-6)
    fl, p = open_field(float(s_cm))
    return {"name": "K_t%g_s%g" % (t_cm, s_cm), "tables": t, "lut": None, "phantom": ph,
            "epid": epid_stack("C1", 160, 160, 0.25, 150.0),
            "source": _source((0, 0, 0), _IDENT, mv6_spectrum(), fl, p),
            "physics": default_physics(mode=1), "n_histories": 10_000_000, "seed": 1}


# ---------------------------------------------------------------- collimation stage
# The paper samples a pre-computed, patient-independent Phase Space 1 of the Varian VitalBeam head and transports it through jaws
# and MLC built from the RTPLAN.  Neither the head model nor any plan is in the container and they are not recreated: the records
# below are SYNTHETIC (a Gaussian focal spot radiating into the maximum field with the Schiff-shaped stand-in spectrum), and the
# jaws / leaves are plain tungsten slabs with straight (unfocused) edges at invented but plausible distances from the target.
HEAD_W = {"ps1": 20.0, "jaw_y": (28.0, 35.8), "jaw_x": (36.7, 44.5), "mlc": (48.2, 54.9), "ps2": 56.0}   # cm from the source


def phase_space_1(seed=7, n=1_000_000, field_half_cm=14.0, spot_sigma_cm=0.05, plane=HEAD_W["ps1"], spectrum=None):
    """Synthetic Phase Space 1: n records [x, y, du, dv, dw, E, 0, 0] (float32, beam frame) on the plane w = `plane`.

    Each photon leaves a Gaussian focal spot on w = 0 towards a point drawn uniformly (planar fluence) in the square of
    half-size field_half_cm on the isocentre plane w = 100; its energy is drawn from the histogram spectrum.  The record is
    the crossing of the plane w = `plane`."""
    rng = np.random.default_rng(seed)
    edges, pdf = spectrum if spectrum is not None else mv6_spectrum()
    sx, sy = rng.normal(0.0, spot_sigma_cm, n), rng.normal(0.0, spot_sigma_cm, n)
    tx, ty = rng.uniform(-field_half_cm, field_half_cm, n), rng.uniform(-field_half_cm, field_half_cm, n)
    d = np.stack([tx - sx, ty - sy, np.full(n, 100.0)], axis=1)
    d /= np.linalg.norm(d, axis=1, keepdims=True)
    t = plane / d[:, 2]
    k = rng.choice(len(pdf), size=n, p=np.asarray(pdf, dtype=np.float64) / np.sum(pdf, dtype=np.float64))
    E = edges[k] + rng.uniform(0.0, 1.0, n) * (edges[k + 1] - edges[k])
    rec = np.zeros((n, 8), dtype=np.float32)
    rec[:, 0] = sx + t * d[:, 0]; rec[:, 1] = sy + t * d[:, 1]
    rec[:, 2:5] = d; rec[:, 5] = E
    return {"records": rec, "plane": float(plane), "n": int(n)}


def _slab(w, axis, row0, pitch, lo, hi):
    return {"w0": float(w[0]), "w1": float(w[1]), "axis": int(axis), "row0": float(row0), "pitch": float(pitch),
            "lo": np.asarray(lo, dtype=np.float32), "hi": np.asarray(hi, dtype=np.float32)}


def collimator_for_fluence(fluence, f_pitch=0.1, leaf_cm=0.5, margin_cm=0.5):
    """Jaws and MLC whose openings follow the envelope of a fluence map given on the isocentre plane (w = 100 cm).

    A slab opens, per row, the interval [lo, hi] of the coordinate across the rows; everything else inside its w-range is
    tungsten.  axis = 0: rows are stacked along v (leaf direction u, the MLC and the x-jaws), axis = 1: one row stacked along u
    (the y-jaws, opening in v).  Openings are given at the slab itself: isocentre size x (slab mid-plane / 100), straight edges.
    MLC: one leaf pair per leaf_cm at the isocentre; leaf row k opens from the first to the last non-zero fluence pixel of its
    rows (closed pairs park at lo = hi = 0 under the x-jaws); the jaws frame the bounding box plus margin_cm."""
    f = np.asarray(fluence)
    fv, fu = f.shape
    px = int(round(leaf_cm / f_pitch))
    n_leaf = fv // px
    u = (np.arange(fu + 1) - fu / 2) * f_pitch                     # pixel edges at the isocentre
    lo, hi = np.zeros(n_leaf), np.zeros(n_leaf)
    for k in range(n_leaf):
        cols = np.nonzero(f[k * px:(k + 1) * px].sum(axis=0) > 0)[0]
        if len(cols):
            lo[k], hi[k] = u[cols[0]], u[cols[-1] + 1]
    rows = np.nonzero(hi > lo)[0]
    v_lo, v_hi = (rows[0] * px - fv / 2) * f_pitch, ((rows[-1] + 1) * px - fv / 2) * f_pitch
    u_lo, u_hi = lo[rows].min(), hi[rows].max()
    sc = lambda w: 0.5 * (w[0] + w[1]) / 100.0
    jy, jx, ml = HEAD_W["jaw_y"], HEAD_W["jaw_x"], HEAD_W["mlc"]
    slabs = [_slab(jy, 1, -100.0, 200.0, [(v_lo - margin_cm) * sc(jy)], [(v_hi + margin_cm) * sc(jy)]),
             _slab(jx, 0, -100.0, 200.0, [(u_lo - margin_cm) * sc(jx)], [(u_hi + margin_cm) * sc(jx)]),
             _slab(ml, 0, -0.5 * n_leaf * leaf_cm * sc(ml), leaf_cm * sc(ml), lo * sc(ml), hi * sc(ml))]
    return {"slabs": slabs, "material": MAT_W, "density": float(TUNGSTEN[2]), "w_ps2": HEAD_W["ps2"]}


def head_config(field=0, shrink=1, n_ps1=1_000_000, seed_ps1=7):
    """C4 field `field` with the collimation stage in place of the fluence-map source: the same phantom, EPID, spectrum and
    aperture envelope, tables with tungsten as material 8, a synthetic Phase Space 1 and jaws / MLC from the field's map."""
    t = make_tables(extra=(TUNGSTEN,))
    cfg = make_config("C4", field=field, shrink=shrink, tables=t)
    cfg["name"] = "C4H"
    cfg["collimator"] = collimator_for_fluence(cfg["source"]["fluence"], cfg["source"]["f_pitch"])
    cfg["ps1"] = phase_space_1(seed_ps1, n_ps1)
    return cfg


def make_config(name, field=0, shrink=1, tables=None):
    """Build config `name` in {"C0".."C4"}.

    `field` selects one of C4's 25 fields.  `shrink` > 1 divides the phantom
    grid dimensions (same physical extent, coarser voxels) and the EPID pixel
    counts (coarser pixels, same area) for test-sized runs.
    """
    if name not in CONFIG_NAMES:
        raise ValueError(name)
    t = tables if tables is not None else make_tables()
    s = int(shrink)
    cfg = {"name": name, "tables": t, "lut": None}
    if name == "C0":
        n = (64 // s, 64 // s, 40 // s)
        h = (0.5 * s,) * 3
        cfg["phantom"] = phantom_water(n, h, (-16.0, -16.0, 100.0))
        cfg["epid"] = epid_stack("C0", 64 // s, 64 // s, 0.4 * s, 170.0)
        fl, p = open_field(10.0)
        cfg["source"] = _source((0, 0, 0), _IDENT, mono_spectrum(2.0), fl, p)
        cfg["physics"] = default_physics(mode=0)
        cfg["n_histories"], cfg["seed"] = 100_000, 1
    elif name == "C1":
        n = (120 // s, 120 // s, 80 // s)
        h = (0.25 * s,) * 3
        cfg["phantom"] = phantom_water(n, h, (-15.0, -15.0, 90.0))
        cfg["epid"] = epid_stack("C1", 512 // s, 384 // s, 0.0784 * s, 150.0)
        fl, p = open_field(10.0)
        cfg["source"] = _source((0, 0, 0), _IDENT, mv6_spectrum(), fl, p)
        cfg["physics"] = default_physics(mode=1)
        cfg["n_histories"], cfg["seed"] = 10_000_000, 1
    elif name in ("C2", "C4"):
        n = (256 // s, 256 // s, 128 // s)
        h = (0.15 * s, 0.15 * s, 0.25 * s)
        cfg["phantom"] = phantom_thorax_c2(42, n, h)
        cfg["epid"] = epid_stack("C1", 1024 // s, 768 // s, 0.0392 * s, 150.0)
        if name == "C2":
            fl, p = mlc_fluence(43, (8, 15))
            cfg["seed"] = 1
        else:
            rng = np.random.default_rng(1000 + field)          # reading A23
            fs = float(rng.uniform(3.0, 20.0))
            fl, p = mlc_fluence(1000 + field, (5, 20), field_cm=fs)
            cfg["seed"] = 2000 + field
            cfg["lut"] = response_lut(46)
            cfg["field"] = int(field)
        cfg["source"] = _source((0.0, -100.0, 0.0), _AXES_Y, mv6_spectrum(), fl, p)
        cfg["physics"] = default_physics(mode=1)
        cfg["n_histories"] = 100_000_000
    else:  # C3
        n = (512 // s, 512 // s, 200 // s)
        h = (0.1 * s, 0.1 * s, 0.25 * s)
        cfg["phantom"] = phantom_patient_c3(44, n, h)
        cfg["epid"] = epid_stack("C1", 1024 // s, 768 // s, 0.0392 * s, 150.0)
        fl, p = mlc_fluence(45, (9, 9))
        cfg["source"] = _source((0.0, -100.0, 0.0), _AXES_Y, mv6_spectrum(), fl, p)
        cfg["physics"] = default_physics(mode=1)
        cfg["n_histories"], cfg["seed"] = 1_000_000_000, 1
    return cfg
