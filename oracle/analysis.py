"""Oracle of the image-analysis chain (TEST INFRASTRUCTURE: only tests/, __graft_entry__.smoke() and bench.py's
cpu_baseline leg may import this; the product path never does).

Plain numpy, float64, the definitions written out; shares no code with the CUDA path.

PAPER.md:141 (section 2.3.3): "the lower-resolution simulated image was up-sampled to match the dimensions of the
measured image ... quantified using the Gamma Index ... global passing criteria of 3%/3 mm, 3%/2 mm, and 2%/2 mm, all
with a 10% low-dose threshold."  The paper names neither the interpolation nor the search; readings A28
(bilinear between pixel centres, edges clamped) and A29 (global gamma of Low et al., searched over the evaluated
grid points, reported up to a cap) are what both sides implement.
"""
from __future__ import annotations

import numpy as np


def upsample_bilinear(img, mv, mu):
    """Resample img [nv][nu] to [mv][mu] over the same physical area (reading A28).

    Output pixel (j, i) has its centre at x = (i + 0.5) nu/mu - 0.5, y = (j + 0.5) nv/mv - 0.5 in units of input
    pixels (input pixel centres at the integers); the value is the bilinear interpolant of the four surrounding
    input centres, with coordinates clamped to [0, n - 1] (no extrapolation beyond the outermost centres).
    """
    a = np.asarray(img, dtype=np.float64)
    nv, nu = a.shape
    out = np.empty((mv, mu), dtype=np.float64)
    for j in range(mv):
        y = min(max((j + 0.5) * nv / mv - 0.5, 0.0), nv - 1.0)
        j0 = min(int(np.floor(y)), max(nv - 2, 0))
        j1 = min(j0 + 1, nv - 1)
        fy = y - j0
        for i in range(mu):
            x = min(max((i + 0.5) * nu / mu - 0.5, 0.0), nu - 1.0)
            i0 = min(int(np.floor(x)), max(nu - 2, 0))
            i1 = min(i0 + 1, nu - 1)
            fx = x - i0
            out[j, i] = ((1 - fy) * ((1 - fx) * a[j0, i0] + fx * a[j0, i1])
                         + fy * ((1 - fx) * a[j1, i0] + fx * a[j1, i1]))
    return out


def gamma_index(ref, ev, pitch_cm, dose_frac, dta_cm, threshold_frac=0.10, cap=2.0):
    """Global 2-D gamma index of `ev` against `ref` (same grid [nv][nu], pixel pitch pitch_cm), reading A29.

    gamma(r) = min over evaluated grid points e of sqrt(|x_e - x_r|^2 / DTA^2 + (D_e - D_r)^2 / (dose_frac D_max)^2),
    D_max = max of the reference (global normalisation), reported as min(cap, gamma): grid points farther than
    cap * DTA cannot bring gamma below cap, so the search window is the disc of that radius.
    Reference pixels below threshold_frac * D_max are not tested and get gamma = -1; an all-zero reference tests nothing.
    Returns (gamma [nv][nu], stats) with stats = (n_tested, n_pass (gamma <= 1), mean gamma, max gamma) over tested pixels.
    """
    r = np.asarray(ref, dtype=np.float64)
    e = np.asarray(ev, dtype=np.float64)
    nv, nu = r.shape
    dmax = r.max()
    if not dmax > 0.0:
        return np.full((nv, nu), -1.0), (0, 0, 0.0, 0.0)
    dd = dose_frac * dmax
    w = int(np.floor(cap * dta_cm / pitch_cm + 1e-9))
    g2 = np.full((nv, nu), cap * cap, dtype=np.float64)
    for dj in range(-w, w + 1):
        for di in range(-w, w + 1):
            dist2 = (di * di + dj * dj) * pitch_cm * pitch_cm / (dta_cm * dta_cm)
            if dist2 > cap * cap:
                continue
            # evaluated point (j + dj, i + di) for every reference pixel (j, i) where it exists
            j0, j1 = max(0, -dj), min(nv, nv - dj)
            i0, i1 = max(0, -di), min(nu, nu - di)
            if j0 >= j1 or i0 >= i1:
                continue
            diff = e[j0 + dj:j1 + dj, i0 + di:i1 + di] - r[j0:j1, i0:i1]
            cand = dist2 + diff * diff / (dd * dd)
            np.minimum(g2[j0:j1, i0:i1], cand, out=g2[j0:j1, i0:i1])
    g = np.sqrt(g2)
    tested = r >= threshold_frac * dmax
    g[~tested] = -1.0
    n = int(tested.sum())
    gt = g[tested]
    stats = (n, int((gt <= 1.0).sum()), float(gt.mean()) if n else 0.0, float(gt.max()) if n else 0.0)
    return g, stats


def roi_mean(img, pitch_cm, roi_cm):
    """Mean of img [nv][nu] over the pixels whose centre lies in the central roi_cm x roi_cm square (Eq. 2:
    "the average ... within a 1 cm x 1 cm central region of the EPID image"; reading A33).  The image is centred on
    the beam axis: pixel (j, i) has its centre at u = (i + 0.5 - nu/2) pitch, v = (j + 0.5 - nv/2) pitch; the square is
    closed (|u|, |v| <= roi/2).  An ROI that holds no pixel centre gives nan."""
    a = np.asarray(img, dtype=np.float64)
    nv, nu = a.shape
    u = (np.arange(nu) + 0.5 - 0.5 * nu) * pitch_cm
    v = (np.arange(nv) + 0.5 - 0.5 * nv) * pitch_cm
    m = (np.abs(v)[:, None] <= 0.5 * roi_cm) & (np.abs(u)[None, :] <= 0.5 * roi_cm)
    return float(a[m].mean()) if m.any() else float("nan")


def response_factors(measured, simulated):
    """k(t, s) = M(t, s) / S(t, s) (Eq. 2) for arrays of ROI means of the measured signal and the simulated dose."""
    return np.asarray(measured, dtype=np.float64) / np.asarray(simulated, dtype=np.float64)
