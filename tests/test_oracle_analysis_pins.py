"""Pins of oracle/analysis.py (up-sampling and gamma index) against closed forms, hand-worked values and
a library routine.  CPU only."""
import numpy as np
import pytest

from oracle import analysis as A
from conftest import read_golden


# ------------------------------------------------------------------------------------------------ up-sampling (A28)
def test_upsample_identity_and_constant():
    rng = np.random.default_rng(3)
    a = rng.random((7, 5))
    assert np.allclose(A.upsample_bilinear(a, 7, 5), a, atol=1e-15)
    assert np.allclose(A.upsample_bilinear(np.full((4, 6), 2.5), 9, 13), 2.5, atol=1e-15)


def test_upsample_hand_worked_two_pixels():
    # centres of the 4 output pixels in input-pixel units: -0.25, 0.25, 0.75, 1.25 -> clamped 0, 0.25, 0.75, 1
    out = A.upsample_bilinear(np.array([[0.0, 1.0]]), 1, 4)
    assert np.allclose(out, [[0.0, 0.25, 0.75, 1.0]], atol=1e-15)
    # and along the other axis (a transposed operand would fail here)
    out = A.upsample_bilinear(np.array([[0.0], [1.0], [4.0]]), 6, 1)
    # centres: -0.25, 0.25, 0.75, 1.25, 1.75, 2.25 -> 0, .25, .75, 1+.25*3, 1+.75*3, 4
    assert np.allclose(out[:, 0], [0.0, 0.25, 0.75, 1.75, 3.25, 4.0], atol=1e-15)


def test_upsample_reproduces_a_linear_image_in_the_interior():
    nv, nu, mv, mu = 9, 12, 31, 50            # non-integer factors
    y, x = np.mgrid[0:nv, 0:nu]
    a = 0.3 * x - 0.7 * y + 2.0
    out = A.upsample_bilinear(a, mv, mu)
    xo = (np.arange(mu) + 0.5) * nu / mu - 0.5
    yo = (np.arange(mv) + 0.5) * nv / mv - 0.5
    inside = (yo[:, None] >= 0) & (yo[:, None] <= nv - 1) & (xo[None, :] >= 0) & (xo[None, :] <= nu - 1)
    exact = 0.3 * xo[None, :] - 0.7 * yo[:, None] + 2.0
    assert inside.sum() > 1000
    assert np.abs(out - exact)[inside].max() < 1e-12


def test_upsample_equals_scipy_map_coordinates():
    from scipy.ndimage import map_coordinates
    rng = np.random.default_rng(11)
    a = rng.random((16, 10))
    mv, mu = 119, 37
    yo = (np.arange(mv) + 0.5) * 16 / mv - 0.5
    xo = (np.arange(mu) + 0.5) * 10 / mu - 0.5
    yy, xx = np.meshgrid(yo, xo, indexing="ij")
    lib = map_coordinates(a, [yy, xx], order=1, mode="nearest")
    assert np.abs(A.upsample_bilinear(a, mv, mu) - lib).max() < 1e-12


# ------------------------------------------------------------------------------------------------ gamma index (A29)
def test_gamma_paper_criteria_fixture():
    rows = read_golden("paper_gamma_criteria.txt")
    crit = [(float(r[0]), float(r[1])) for r in rows if r[0] != "threshold"]
    assert crit == [(3.0, 3.0), (3.0, 2.0), (2.0, 2.0)]
    assert [float(r[1]) for r in rows if r[0] == "threshold"] == [10.0]


def test_gamma_identical_images_and_threshold():
    rng = np.random.default_rng(5)
    r = 0.9 * rng.random((20, 30)) + 0.01
    r[3, 4] = 10.0                                          # max 10 -> everything below 1.0 is under the 10 % threshold
    r[5, 6] = 1.0; r[7, 8] = 0.9999
    g, st = A.gamma_index(r, r, 0.1, 0.03, 0.3)
    tested = r >= 1.0
    assert st[0] == tested.sum() == 2 and st[1] == 2 and st[2] == 0.0
    assert np.all(g[tested] == 0.0) and np.all(g[~tested] == -1.0)


@pytest.mark.parametrize("eps,frac,expect", [(0.015, 0.03, 0.5), (0.03, 0.03, 1.0), (-0.02, 0.02, 1.0), (0.09, 0.03, 2.0)])
def test_gamma_uniform_dose_offset(eps, frac, expect):
    r = np.full((15, 11), 4.0)
    g, st = A.gamma_index(r, r * (1 + eps), 0.0784, frac, 0.3)      # expect min(cap, |eps| / frac)
    assert np.allclose(g, expect, atol=1e-12)
    assert st[0] == r.size
    if abs(expect - 1.0) > 1e-6:                            # exactly on the criterion the count depends on rounding
        assert st[1] == (r.size if expect < 1.0 else 0)


def test_gamma_shifted_ramp_closed_form():
    # D = g x on x = 0..10 cm (pitch 0.1), DTA 0.3, 3 % of D_max = g 10: distance and dose terms weigh the same per
    # pixel, so for a shift of s = 2 pixels the minimum over real offsets k of a k^2 + a (k - s)^2 sits at the integer
    # k = 1 and gamma = sqrt(2) pitch / DTA
    nu, nv, p, s = 101, 4, 0.1, 2
    x = np.arange(nu) * p
    r = np.tile(3.0 * x, (nv, 1))
    e = np.tile(3.0 * (x - s * p), (nv, 1))
    g, st = A.gamma_index(r, e, p, 0.03, 0.3)
    inner = g[:, 15:-5]                                     # tested (above 10 %) and away from the image edge
    assert np.allclose(inner, np.sqrt(2.0) * p / 0.3, atol=1e-9)
    # the same along v (transposed images): catches swapped axes
    gt, _ = A.gamma_index(r.T.copy(), e.T.copy(), p, 0.03, 0.3)
    assert np.allclose(gt, g.T, atol=1e-12)


def test_gamma_displaced_spike_and_cap():
    r = np.zeros((9, 21)); e = np.zeros((9, 21))
    r[4, 5] = 1.0; e[4, 8] = 1.0                            # same spike, 3 pixels away along u
    g, st = A.gamma_index(r, e, 0.05, 0.03, 0.3)
    assert st[0] == 1 and abs(g[4, 5] - 3 * 0.05 / 0.3) < 1e-12
    e2 = np.zeros((9, 21)); e2[7, 5] = 1.0                  # 3 pixels away along v
    g2, _ = A.gamma_index(r, e2, 0.05, 0.03, 0.3)
    assert abs(g2[4, 5] - 0.5) < 1e-12
    g3, st3 = A.gamma_index(r, np.zeros_like(r), 0.05, 0.03, 0.3)   # nothing to find: dose term 1/0.03 >> cap
    assert g3[4, 5] == 2.0 and st3[1] == 0
    # a spike farther away than cap * DTA is not seen
    e4 = np.zeros((9, 21)); e4[4, 18] = 1.0                 # 13 pixels = 0.65 cm > 2 * 0.3
    assert A.gamma_index(r, e4, 0.05, 0.03, 0.3)[0][4, 5] == 2.0


def test_gamma_brute_force_on_a_tiny_image():
    rng = np.random.default_rng(9)
    r = rng.random((6, 7)) + 0.5; e = r + 0.05 * rng.standard_normal((6, 7))
    p, frac, dta, cap = 0.2, 0.03, 0.3, 2.0
    g, _ = A.gamma_index(r, e, p, frac, dta, 0.1, cap)
    dd = frac * r.max()
    for j in range(6):
        for i in range(7):
            best = cap
            for jj in range(6):
                for ii in range(7):
                    d = np.hypot((ii - i) * p, (jj - j) * p) / dta
                    best = min(best, np.hypot(d, (e[jj, ii] - r[j, i]) / dd))
            assert abs(g[j, i] - best) < 1e-12


# ------------------------------------------------------------------------------------------------ ROI mean, Eq. 2 (A33)
def test_roi_mean_hand_worked_and_symmetry():
    a = np.arange(36, dtype=float).reshape(6, 6)            # pitch 1 cm: centres at -2.5 ... 2.5
    assert A.roi_mean(a, 1.0, 1.0) == pytest.approx(a[2:4, 2:4].mean())        # the four pixels around the axis (|centre| = 0.5 <= 0.5)
    assert A.roi_mean(a, 1.0, 0.9) != A.roi_mean(a, 1.0, 0.9)                 # no centre inside: nan
    assert A.roi_mean(a, 1.0, 3.0) == pytest.approx(a[1:5, 1:5].mean())
    assert A.roi_mean(a, 1.0, 100.0) == pytest.approx(a.mean())
    b = np.zeros((5, 7)); b[2, 3] = 9.0                     # odd sizes: the central pixel sits on the axis
    assert A.roi_mean(b, 0.4, 0.1) == 9.0
    assert A.roi_mean(b, 0.4, 0.8) == pytest.approx(9.0 / 9)
    # transposing the image changes nothing for a square ROI
    rng = np.random.default_rng(2); c = rng.random((12, 20))
    assert A.roi_mean(c, 0.25, 1.0) == pytest.approx(A.roi_mean(c.T.copy(), 0.25, 1.0))


def test_response_factors_reproduce_table1_from_its_own_products():
    from gen.configs import paper_table1_lut
    k = paper_table1_lut()["lut"].astype(np.float64)
    S = np.random.default_rng(4).uniform(0.5, 2.0, k.shape)
    assert np.allclose(A.response_factors(k * S, S), k, rtol=1e-14)
