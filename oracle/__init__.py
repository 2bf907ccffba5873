"""ctypes binding of the CPU oracle (oracle/oracle.cpp).  TEST INFRASTRUCTURE ONLY.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl
reference legs import this package; the product (paper_2510_24154_b200) never
does.  It imports nothing from the product either.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "oracle.cpp")
_LIB = os.path.join(_HERE, "liboracle.so")
_lib = None

LEDGER_NAMES = ("emitted", "dep_phantom", "dep_epid_scored", "dep_epid_other", "dep_air", "escaped",
                "n_histories", "reserved")
COUNTER_NAMES = ("woodcock_flights", "air_flights", "epid_flights", "n_pe", "n_compton", "n_pair",
                 "esteps_phantom", "esteps_air", "esteps_epid", "n_secondaries", "uncollided_at_epid",
                 "max_stack", "kn_iterations", "photon_cutoffs", "e_tracks", "zero_steps")


def build(force=False):
    """Compile liboracle.so with g++ (plain -O2, never tuned)."""
    if not force and os.path.exists(_LIB) and os.path.getmtime(_LIB) >= os.path.getmtime(_SRC):
        return _LIB
    subprocess.check_call(["g++", "-O2", "-std=c++17", "-fPIC", "-shared", "-o", _LIB, _SRC])
    return _LIB


def lib():
    global _lib
    if _lib is None:
        _lib = C.CDLL(build())
        _lib.orc_create.restype = C.c_void_p
        _lib.orc_last_error.restype = C.c_char_p
        _lib.orc_ps3_count.restype = C.c_uint64
        _lib.orc_event_log_count.restype = C.c_uint64
        _lib.orc_ps2_count.restype = C.c_uint64
        _lib.orc_moller_cos.restype = C.c_double
        for f in ("orc_stop_pow", "orc_majorant", "orc_highland_theta0", "orc_field_size", "orc_lut_bilinear"):
            getattr(_lib, f).restype = C.c_double
    return _lib


def _p(a, t):
    return a.ctypes.data_as(C.POINTER(t)) if a is not None else None


def _f32(a):
    return np.ascontiguousarray(a, dtype=np.float32)


def _u8(a):
    return np.ascontiguousarray(a, dtype=np.uint8)


def philox(ctr, key):
    c = (C.c_uint32 * 4)(*ctr); k = (C.c_uint32 * 2)(*key); o = (C.c_uint32 * 4)()
    lib().orc_philox4x32_10(c, k, o)
    return [int(v) for v in o]


def sample_compton(E, seed, n):
    eps = np.empty(n); cost = np.empty(n)
    lib().orc_sample_compton(C.c_double(E), C.c_uint64(seed), C.c_uint64(n), _p(eps, C.c_double), _p(cost, C.c_double))
    return eps, cost


def compton_events(E, d0, seed, n):
    out = np.empty((n, 8)); d = np.ascontiguousarray(d0, dtype=np.float64)
    lib().orc_compton_events(C.c_double(E), _p(d, C.c_double), C.c_uint64(seed), C.c_uint64(n), _p(out, C.c_double))
    return out


def sample_deflection(d0, theta0, seed, n):
    out = np.empty((n, 3)); d = np.ascontiguousarray(d0, dtype=np.float64)
    lib().orc_sample_deflection(_p(d, C.c_double), C.c_double(theta0), C.c_uint64(seed), C.c_uint64(n), _p(out, C.c_double))
    return out


def moller_xs(T, Tc):
    """(cross section per electron [cm^2], integral of W d sigma [MeV cm^2]) for energy transfers above Tc (reading A31)."""
    o = (C.c_double * 2)()
    lib().orc_moller_xs(C.c_double(T), C.c_double(Tc), o)
    return o[0], o[1]


def sample_moller(T, Tc, seed, n):
    eps = np.empty(n)
    lib().orc_sample_moller(C.c_double(T), C.c_double(Tc), C.c_uint64(seed), C.c_uint64(n), _p(eps, C.c_double))
    return eps


def brems_xs(T, kc, X0):
    """(Sigma of photons above kc [cm^2/g], restricted radiative stopping power [MeV cm^2/g]) of the reading-A32 model."""
    o = (C.c_double * 2)()
    lib().orc_brems_xs(C.c_double(T), C.c_double(kc), C.c_double(X0), o)
    return o[0], o[1]


def sample_brems(T, kc, seed, n):
    k = np.empty(n)
    lib().orc_sample_brems(C.c_double(T), C.c_double(kc), C.c_uint64(seed), C.c_uint64(n), _p(k, C.c_double))
    return k


def moller_cos(T_out, T_in):
    return lib().orc_moller_cos(C.c_double(T_out), C.c_double(T_in))


def lut_bilinear(lut, t_min, t_max, s_min, s_max, t, s):
    a = np.ascontiguousarray(lut, dtype=np.float64)
    return lib().orc_lut_bilinear(_p(a, C.c_double), a.shape[0], a.shape[1], C.c_double(t_min), C.c_double(t_max),
                                  C.c_double(s_min), C.c_double(s_max), C.c_double(t), C.c_double(s))


class Oracle:
    """One oracle context loaded from a `gen.make_config` dictionary (or its pieces)."""

    def __init__(self, cfg=None):
        self._l = lib()
        self._h = C.c_void_p(self._l.orc_create())
        self.cfg = None
        if cfg is not None:
            self.load(cfg)

    def __del__(self):
        if getattr(self, "_h", None):
            self._l.orc_destroy(self._h); self._h = None

    def _chk(self, rc):
        if rc != 0:
            raise RuntimeError("oracle error %d: %s" % (rc, self._l.orc_last_error(self._h).decode()))

    # ---- loading (mirrors the C-ABI of include/aepid.h, independent code)
    def init_materials(self, t):
        E, T = _f32(t["E_grid"]), _f32(t["T_grid"])
        mc, mp, mpp, sp, x0 = (_f32(t[k]) for k in ("mu_compton", "mu_pe", "mu_pair", "stop_pow", "rad_len"))
        self.n_mat = int(mc.shape[0])
        if "electrons_per_gram" in t:                       # input of mode 2 (Class II collisions)
            ne = _f32(t["electrons_per_gram"])
            self._chk(self._l.orc_set_class2(self._h, len(ne), _p(ne, C.c_float)))
        self._chk(self._l.orc_init_materials(self._h, self.n_mat, len(E), _p(E, C.c_float), _p(mc, C.c_float), _p(mp, C.c_float),
                                             _p(mpp, C.c_float), len(T), _p(T, C.c_float), _p(sp, C.c_float), _p(x0, C.c_float)))

    def load_phantom(self, ph):
        rho, mat = _f32(ph["density"]), _u8(ph["material"])
        sp, org = _f32(ph["spacing"]), _f32(ph["origin"])
        self.nvox = (int(ph["nz"]), int(ph["ny"]), int(ph["nx"]))
        self._chk(self._l.orc_load_phantom(self._h, int(ph["nx"]), int(ph["ny"]), int(ph["nz"]), _p(sp, C.c_float), _p(org, C.c_float),
                                           _p(rho, C.c_float), _p(mat, C.c_uint8)))

    def load_epid_layers(self, ep):
        th, rho = _f32(ep["thickness"]), _f32(ep["density"])
        mat, sc = _u8(ep["material"]), _u8(ep["scored"])
        self.nu, self.nv = int(ep["nu"]), int(ep["nv"])
        self._chk(self._l.orc_load_epid_layers(self._h, len(th), _p(th, C.c_float), _p(mat, C.c_uint8), _p(rho, C.c_float), _p(sc, C.c_uint8),
                                               C.c_float(ep["sid"]), self.nu, self.nv, C.c_float(ep["pitch"])))

    def load_source(self, s):
        src, ax = _f32(s["src_pos"]), _f32(s["beam_axes"]).reshape(9)
        ed, pdf, fl = _f32(s["E_edges"]), _f32(s["E_pdf"]), _f32(s["fluence"])
        self._chk(self._l.orc_load_source(self._h, _p(src, C.c_float), _p(ax, C.c_float), len(pdf), _p(ed, C.c_float), _p(pdf, C.c_float),
                                          int(s["fu"]), int(s["fv"]), C.c_float(s["f_pitch"]), C.c_float(s["f_plane_dist"]), _p(fl, C.c_float)))

    def set_physics(self, ph):
        self._chk(self._l.orc_set_physics(self._h, int(ph["mode"]), C.c_double(ph["photon_cut"]), C.c_double(ph["electron_cut"]),
                                          C.c_double(ph["f_E"]), C.c_double(ph["s_max"])))

    def set_options(self, tracking=0, rebin=1, want_phantom_sq=True, fc_bins=0, fc_w0=0.0, fc_dw=1.0):
        self.rebin, self.fc_bins = int(rebin), int(fc_bins)
        self._chk(self._l.orc_set_options(self._h, int(tracking), int(rebin), int(bool(want_phantom_sq)), int(fc_bins),
                                          C.c_double(fc_w0), C.c_double(fc_dw)))
        self._want_sq = bool(want_phantom_sq)

    def set_phantom_rebin(self, rx=1, ry=1, rz=1):
        """Also tally the phantom on blocks of rx x ry x rz voxels, history by history (takes effect at reset)."""
        self.prb = (int(rx), int(ry), int(rz))
        self._chk(self._l.orc_set_phantom_rebin(self._h, *self.prb))

    def set_event_log(self, capacity):
        """Pins only: keep up to `capacity` interaction / birth records (see log_event in oracle.cpp)."""
        self._chk(self._l.orc_set_event_log(self._h, C.c_uint64(int(capacity))))

    def read_event_log(self):
        n = int(self._l.orc_event_log_count(self._h))
        out = np.empty((n, 16))
        self._chk(self._l.orc_read_event_log(self._h, _p(out, C.c_double)))
        return out

    def set_fixed_primary(self, ptype, E=0.0, pos=(0, 0, 0), direction=(0, 0, 1)):
        p = (C.c_double * 3)(*pos); d = (C.c_double * 3)(*direction)
        self._chk(self._l.orc_set_fixed_primary(self._h, int(ptype), C.c_double(E), p, d))

    # ---- collimation stage: Phase Space 1 source, jaws / MLC slabs, Phase Space 2 dump
    def load_phase_space_source(self, ps1):
        rec = _f32(ps1["records"]) if ps1 is not None else np.zeros((0, 8), np.float32)
        self._chk(self._l.orc_load_phase_space_source(self._h, C.c_uint64(len(rec)), _p(rec, C.c_float), C.c_double(ps1["plane"] if ps1 is not None else 0.0)))

    def load_collimator(self, col):
        if col is None:
            self._chk(self._l.orc_load_collimator(self._h, 0, None, None, None, None, None, None, None, None, 0, C.c_double(1.0), C.c_double(0.0)))
            return
        sl = col["slabs"]
        w0, w1 = _f32([s["w0"] for s in sl]), _f32([s["w1"] for s in sl])
        axis = np.ascontiguousarray([s["axis"] for s in sl], dtype=np.int32); nr = np.ascontiguousarray([len(s["lo"]) for s in sl], dtype=np.int32)
        row0, pitch = _f32([s["row0"] for s in sl]), _f32([s["pitch"] for s in sl])
        lo, hi = _f32(np.concatenate([s["lo"] for s in sl])), _f32(np.concatenate([s["hi"] for s in sl]))
        self._chk(self._l.orc_load_collimator(self._h, len(sl), _p(w0, C.c_float), _p(w1, C.c_float), _p(axis, C.c_int), _p(nr, C.c_int),
                                              _p(row0, C.c_float), _p(pitch, C.c_float), _p(lo, C.c_float), _p(hi, C.c_float),
                                              int(col["material"]), C.c_double(col["density"]), C.c_double(col["w_ps2"])))

    def set_ps2(self, on=True):
        self._chk(self._l.orc_set_ps2(self._h, int(bool(on))))

    def read_ps2(self):
        """Records [n][8] = {E, u, v, du, dv, dw, history, uncollided} of every photon that reached the Phase Space 2 plane."""
        n = int(self._l.orc_ps2_count(self._h))
        out = np.empty((n, 8))
        self._chk(self._l.orc_read_ps2(self._h, _p(out, C.c_double)))
        return out

    def read_head(self):
        """{PS2 particles, their energy, energy absorbed in the stage, interactions in the stage}."""
        out = np.zeros(4)
        self._chk(self._l.orc_read_head(self._h, _p(out, C.c_double)))
        return out

    def load(self, cfg):
        self.cfg = cfg
        self.init_materials(cfg["tables"])
        self.load_phantom(cfg["phantom"])
        self.load_epid_layers(cfg["epid"])
        self.load_source(cfg["source"])
        if cfg.get("ps1") is not None:
            self.load_phase_space_source(cfg["ps1"])
        if cfg.get("collimator") is not None:
            self.load_collimator(cfg["collimator"])
        self.set_physics(cfg["physics"])
        self.set_options()

    # ---- running
    def reset(self):
        self._chk(self._l.orc_reset(self._h))

    def run(self, first, n, seed):
        self._chk(self._l.orc_run(self._h, C.c_uint64(first), C.c_uint64(n), C.c_uint64(seed)))

    def read(self):
        """Raw accumulators: sums and sums of squares over histories (history-by-history estimator)."""
        nz, ny, nx = self.nvox
        r = getattr(self, "rebin", 1)
        out = {
            "epid_sum": np.zeros((self.nv, self.nu)), "epid_sq": np.zeros((self.nv, self.nu)),
            "rb_sum": np.zeros((self.nv // r, self.nu // r)), "rb_sq": np.zeros((self.nv // r, self.nu // r)),
            "phantom_sum": np.zeros((nz, ny, nx)),
            "phantom_sq": np.zeros((nz, ny, nx)) if getattr(self, "_want_sq", True) else None,
            "uncollided": np.zeros((self.nv, self.nu)),
            "ledger": np.zeros(8), "counters": np.zeros(16, dtype=np.uint64), "aux": np.zeros(4),
            "fc_hist": np.zeros(max(getattr(self, "fc_bins", 0), 1)),
        }
        self._chk(self._l.orc_read(self._h, _p(out["epid_sum"], C.c_double), _p(out["epid_sq"], C.c_double),
                                   _p(out["rb_sum"], C.c_double), _p(out["rb_sq"], C.c_double),
                                   _p(out["phantom_sum"], C.c_double), _p(out["phantom_sq"], C.c_double),
                                   _p(out["uncollided"], C.c_double), _p(out["ledger"], C.c_double),
                                   _p(out["counters"], C.c_uint64), _p(out["aux"], C.c_double), _p(out["fc_hist"], C.c_double)))
        rx, ry, rz = getattr(self, "prb", (1, 1, 1))
        coarse = rx * ry * rz > 1
        out["pc_sum"] = np.zeros((nz // rz, ny // ry, nx // rx)) if coarse else None
        out["pc_sq"] = np.zeros((nz // rz, ny // ry, nx // rx)) if coarse else None
        out["ledger_sq"] = np.zeros(8)
        self._chk(self._l.orc_read_extra(self._h, _p(out["pc_sum"], C.c_double), _p(out["pc_sq"], C.c_double), _p(out["ledger_sq"], C.c_double)))
        out["head"] = self.read_head()
        return out

    # ---- Phase Space 3 (reading A30)
    def set_ps3(self, on=True):
        self._chk(self._l.orc_set_ps3(self._h, int(bool(on))))

    def read_ps3(self):
        """Records [n][8] = {type, E, u, v, du, dv, dw, history} of every particle that arrived at the EPID top plane."""
        n = int(self._l.orc_ps3_count(self._h))
        out = np.empty((n, 8))
        self._chk(self._l.orc_read_ps3(self._h, _p(out, C.c_double)))
        return out

    # ---- unit-level entry points
    def mu_partial(self, m, E):
        o = (C.c_double * 3)(); self._l.orc_mu_partial(self._h, int(m), C.c_double(E), o); return np.array(o[:])

    def stop_pow(self, m, T):
        return self._l.orc_stop_pow(self._h, int(m), C.c_double(T))

    def majorant(self, E):
        return self._l.orc_majorant(self._h, C.c_double(E))

    def highland_theta0(self, m, rho_s, Tm):
        return self._l.orc_highland_theta0(self._h, int(m), C.c_double(rho_s), C.c_double(Tm))

    def sample_source(self, first, n, seed):
        out = np.empty((n, 7))
        self._chk(self._l.orc_sample_source(self._h, C.c_uint64(first), C.c_uint64(n), C.c_uint64(seed), _p(out, C.c_double)))
        return out

    def field_size(self, printed_form=False):
        return self._l.orc_field_size(self._h, int(bool(printed_form)))

    def tmap(self):
        out = np.empty((self.nv, self.nu))
        self._chk(self._l.orc_tmap(self._h, _p(out, C.c_double)))
        return out

    def apply_lut(self, lutd, dose, tmap, s_eff):
        a = np.ascontiguousarray(lutd["lut"], dtype=np.float64)
        d = np.ascontiguousarray(dose, dtype=np.float64); t = np.ascontiguousarray(tmap, dtype=np.float64)
        out = np.empty_like(d)
        self._l.orc_apply_lut(_p(a, C.c_double), a.shape[0], a.shape[1], C.c_double(lutd["t_min"]), C.c_double(lutd["t_max"]),
                              C.c_double(lutd["s_min"]), C.c_double(lutd["s_max"]), C.c_double(s_eff),
                              _p(d, C.c_double), _p(t, C.c_double), C.c_size_t(d.size), _p(out, C.c_double))
        return out


def stats(raw):
    """Mean per history and sigma of the mean from raw sums."""
    n = float(raw["ledger"][6])
    res = {"n": n}
    for k, ks, kq in (("epid", "epid_sum", "epid_sq"), ("rb", "rb_sum", "rb_sq"), ("phantom", "phantom_sum", "phantom_sq"),
                      ("pc", "pc_sum", "pc_sq"), ("ledger", "ledger", "ledger_sq")):
        s, q = raw.get(ks), raw.get(kq)
        if s is None:
            continue
        mean = s / n
        res[k + "_mean"] = mean
        if q is not None:
            var = np.maximum(q / n - mean * mean, 0.0) / max(n - 1.0, 1.0)
            res[k + "_sigma"] = np.sqrt(var)
    return res


_SHARED_CFG = None          # inherited by forked workers (copy-on-write): the config is not pickled per job


def _worker(args):
    cfg, first, n, seed, opts = args
    if cfg is None:
        cfg = _SHARED_CFG
    opts = dict(opts)
    prb = opts.pop("phantom_rebin", None)
    o = Oracle(cfg)
    o.set_options(**opts)
    if prb is not None:
        o.set_phantom_rebin(*prb)
    o.reset()
    o.run(first, n, seed)
    return o.read()


def run_sharded(cfg, n, seed, first=0, procs=None, **opts):
    """Run histories [first, first+n) split over `procs` processes (legal: the RNG is keyed by
    the global history index) and add the raw accumulators."""
    import multiprocessing as mp
    global _SHARED_CFG
    procs = procs or min(os.cpu_count() or 1, 32)
    procs = max(1, min(procs, int(n)))
    if procs == 1:
        return _worker((cfg, first, n, seed, opts))
    build()
    bounds = np.linspace(first, first + n, procs + 1).astype(np.uint64)
    jobs = [(None, int(bounds[i]), int(bounds[i + 1] - bounds[i]), seed, opts) for i in range(procs)]
    _SHARED_CFG = cfg
    try:
        with mp.get_context("fork").Pool(procs) as pool:
            tot = None
            for p in pool.imap_unordered(_worker, jobs):       # add as they arrive: one worker's arrays in flight at a time
                if tot is None:
                    tot = p
                    continue
                for k, v in p.items():
                    if v is None:
                        continue
                    if k == "counters":
                        mx = max(int(tot[k][11]), int(v[11]))
                        tot[k] = tot[k] + v; tot[k][11] = mx
                    else:
                        tot[k] += v
    finally:
        _SHARED_CFG = None
    return tot
