"""Phase Space 3 (reading A30): pins of the oracle's recording (CPU) and GPU parity through the C-ABI."""
import numpy as np
import pytest

import oracle
from gen import make_config
from util import slab_cfg


def _oracle_ps3(cfg, n, seed=1, first=0):
    o = oracle.Oracle(cfg)
    o.set_ps3(True)
    o.reset()
    o.run(first, n, seed)
    return o, o.read_ps3(), o.read()


def _primaries(rec, src, cfg):
    """Records that are the history's own source photon, untouched: same energy and direction as the source sample
    (the sample's direction is in the world frame, the record's in the beam frame: rows u, v, w of beam_axes)."""
    h = rec[:, 7].astype(np.int64)
    s = src[h]
    d_beam = s[:, 1:4] @ np.asarray(cfg["source"]["beam_axes"], dtype=np.float64).reshape(3, 3).T
    return (rec[:, 0] == 0) & (np.abs(rec[:, 1] - s[:, 0]) <= 1e-6 * s[:, 0]) & (np.abs(rec[:, 4:7] - d_beam).max(axis=1) <= 1e-6)


# ------------------------------------------------------------------------------------------------ oracle pins (CPU)
def test_ps3_oracle_records_are_well_formed_and_primaries_lie_on_their_ray():
    cfg = make_config("C1", shrink=4)
    n = 20000
    o, rec, raw = _oracle_ps3(cfg, n)
    assert len(rec) > 0.2 * n
    assert np.all(np.isin(rec[:, 0], (0, 1, 2)))
    assert np.all(rec[:, 6] > 0)                                         # arrives from above
    assert np.abs(np.linalg.norm(rec[:, 4:7], axis=1) - 1).max() < 1e-12
    assert np.all(np.abs(rec[:, 2:4]) <= 100.0)
    assert np.all(rec[:, 1] <= cfg["source"]["E_edges"].max() + 1e-9)
    assert np.all(rec[rec[:, 0] == 0, 1] >= cfg["physics"]["photon_cut"]) and np.all(rec[rec[:, 0] > 0, 1] > cfg["physics"]["electron_cut"])
    assert np.all((rec[:, 7] >= 0) & (rec[:, 7] < n))
    # identity beam axes, source at the origin: an untouched source photon crosses the plane w = sid at sid * (du, dv) / dw
    src = oracle.Oracle(cfg).sample_source(0, n, 1)                      # {E, dx, dy, dz, pixel, u, v}
    prim = _primaries(rec, src, cfg)
    sid = cfg["epid"]["sid"]
    assert prim.sum() > 0.2 * n
    assert np.abs(rec[prim, 2] - sid * rec[prim, 4] / rec[prim, 6]).max() < 1e-9
    assert np.abs(rec[prim, 3] - sid * rec[prim, 5] / rec[prim, 6]).max() < 1e-9
    # and their number is the oracle's own uncollided tally (pinned to Beer-Lambert by test_oracle_pins P3)
    assert prim.sum() == raw["counters"][10]


def test_ps3_oracle_uncollided_fraction_is_beer_lambert():
    # 2 MeV pencil-like narrow field through 20 cm of water and the air: exp(-mu L) of SURVEY 8(c) P3 (0.37110 x 0.99731 for 50 cm of air,
    # here 150 cm of path in total of which 20 cm water)
    cfg = slab_cfg(n=(16, 16, 40), h=(0.5, 0.5, 0.5), w0=100.0, E=2.0, mode=0, field_cm=0.4)
    n = 40000
    o, rec, raw = _oracle_ps3(cfg, n)
    mu_w = o.mu_partial(2, 2.0).sum() * 1.0
    mu_a = o.mu_partial(0, 2.0).sum() * 1.205e-3
    expect = np.exp(-mu_w * 20.0 - mu_a * (170.0 - 20.0))
    src = oracle.Oracle(cfg).sample_source(0, n, 1)
    frac = _primaries(rec, src, cfg).sum() / n
    assert abs(frac - expect) < 4 * np.sqrt(expect * (1 - expect) / n) + 2e-4      # obliquity of a 0.4 cm field: < 1e-5


def test_ps3_oracle_off_by_default_and_cleared():
    cfg = make_config("C0")
    o = oracle.Oracle(cfg); o.reset(); o.run(0, 2000, 1)
    assert len(o.read_ps3()) == 0
    o.set_ps3(True); o.run(2000, 2000, 1)
    k = len(o.read_ps3()); assert k > 0
    o.set_ps3(True); assert len(o.read_ps3()) == 0


# ------------------------------------------------------------------------------------------------ GPU parity
def _hist(x, bins, w=None):
    return np.histogram(x, bins=bins, weights=w)[0].astype(np.float64)


@pytest.mark.gpu
@pytest.mark.parametrize("name,shrink,n,mode", [("C1", 1, 400_000, 1), ("C0", 1, 300_000, 0), ("C2", 2, 300_000, 1), ("C1", 1, 400_000, 2), ("C1", 1, 400_000, 3)])
def test_ps3_gpu_matches_oracle(name, shrink, n, mode):
    from paper_2510_24154_b200 import Engine
    cfg = make_config(name, shrink=shrink)
    cfg["physics"]["mode"] = mode                                        # 2: with Moller delta rays (reading A31)
    seed = cfg["seed"]
    eng = Engine.for_config(cfg); eng.load_config(cfg)
    eng.set_phase_space(n)                                               # at most ~0.5 arrivals per history
    eng.simulate(n, seed)
    g, n_arr = eng.read_phase_space()
    L = eng.read_tallies()["ledger"]
    assert L[7] == 0 and n_arr == len(g) and n_arr > 0.1 * n
    o, orc, _ = _oracle_ps3(cfg, n, seed)
    # well-formed
    assert np.all(np.isin(g[:, 0], (0, 1, 2))) and np.all(g[:, 6] > 0) and np.abs(np.linalg.norm(g[:, 4:7], axis=1) - 1).max() < 1e-5
    # (a) the untouched source photons: the same histories' source samples on both sides (K1 parity), so a history whose photon
    #     arrives untouched on both sides has the same record to float rounding
    src = oracle.Oracle(cfg).sample_source(0, n, seed)
    pg, po = _primaries(g, src, cfg), _primaries(orc, src, cfg)
    hg = dict(zip(g[pg, 7].astype(np.int64), np.flatnonzero(pg)))
    both = [(hg[h], k) for h, k in zip(orc[po, 7].astype(np.int64), np.flatnonzero(po)) if h in hg]
    assert len(both) > 0.5 * po.sum() * pg.sum() / n                      # the two sides draw the flights independently
    ig, io = np.array(both).T
    assert np.abs(g[ig, 2:4] - orc[io, 2:4]).max() < 2e-3               # cm on a plane 150-170 cm away: direction to 1e-5
    assert np.abs(g[ig, 1] - orc[io, 1]).max() < 1e-5
    #     and their number agrees (binomial; the two sides draw the flights independently)
    assert abs(pg.sum() - po.sum()) < 5 * np.sqrt(pg.sum() + po.sum()) + 5
    # (b) everything else statistically: counts per type, energy spectra, radial distribution (chi-square of two Poisson histograms)
    for t in (0, 1):
        a, b = g[(g[:, 0] == t) & ~pg], orc[(orc[:, 0] == t) & ~po]              # scattered photons, electrons
        assert abs(len(a) - len(b)) < 5 * np.sqrt(len(a) + len(b)) + 5, (t, len(a), len(b))
        if min(len(a), len(b)) < 2000:
            continue
        for x, y, bins in ((a[:, 1], b[:, 1], np.linspace(0, cfg["source"]["E_edges"].max(), 25)),
                           (np.hypot(a[:, 2], a[:, 3]), np.hypot(b[:, 2], b[:, 3]), np.linspace(0, 100, 21)),
                           (a[:, 6], b[:, 6], np.linspace(0, 1, 21))):
            ha, hb = _hist(x, bins), _hist(y, bins)
            k = (ha + hb) >= 20
            chi2 = ((ha[k] - hb[k]) ** 2 / (ha[k] + hb[k])).sum()
            dof = k.sum()
            assert chi2 < dof + 5 * np.sqrt(2 * dof) + 5, (t, chi2, dof)
    # energy carried through the plane per history
    eg, eo = g[:, 1].sum() / n, orc[:, 1].sum() / n
    assert abs(eg - eo) < 0.01 * eo
    eng.close()


@pytest.mark.gpu
def test_ps3_gpu_capacity_reset_and_errors():
    import torch
    from paper_2510_24154_b200 import Engine
    cfg = make_config("C0")
    eng = Engine.for_config(cfg); eng.load_config(cfg)
    eng.set_phase_space(1000)
    eng.simulate(50_000, 1)
    g, n_arr = eng.read_phase_space()
    assert len(g) == 1000 and n_arr > 10_000                             # counted beyond the capacity, stored up to it
    assert np.all(g[:, 6] > 0)
    eng.reset_tallies()
    assert eng.read_phase_space()[1] == 0
    eng.set_phase_space(0)                                               # off: nothing is counted
    eng.simulate(10_000, 1)
    n = __import__("ctypes").c_ulonglong(7)
    assert eng._lib.aepid_read_phase_space_count(eng._h, __import__("ctypes").byref(n)) == 0 and n.value == 0
    host = np.zeros((16, 8), dtype=np.float32)
    assert eng._lib.aepid_set_phase_space(eng._h, host.ctypes.data, 16) == -1           # host memory: BAD_ARG
    dev = torch.zeros(64, dtype=torch.float32, device=eng.device)
    assert eng._lib.aepid_set_phase_space(eng._h, dev.data_ptr() + 4, 1) == -1          # misaligned
    assert eng._lib.aepid_set_phase_space(eng._h, dev.data_ptr(), 0) == -1              # zero capacity
    eng.close()
