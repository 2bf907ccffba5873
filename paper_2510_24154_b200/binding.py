"""Thin ctypes binding of libaepid.so (include/aepid.h): argument marshalling only.

Every step of the path runs in the CUDA kernels behind the C-ABI.  PyTorch is used for the
device workspace, device tensors and the CUDA stream, nothing else.  There is no CPU fallback:
importing works anywhere, creating an Engine without the built library or a GPU raises.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
# AEPID_LIBRARY: another build of the same library (the checked build of build.build_checked, tests/test_gpu_checked_build.py)
LIB_PATH = os.environ.get("AEPID_LIBRARY") or os.path.join(_HERE, "libaepid.so")
_lib = None

STATUS = {0: "OK", -1: "BAD_ARG", -2: "BAD_STATE", -3: "GEOMETRY", -4: "CUDA", -5: "NOMEM", -6: "INTERNAL"}
LEDGER_NAMES = ("emitted", "dep_phantom", "dep_epid_scored", "dep_epid_other", "dep_air", "escaped",
                "n_histories", "overflow")
# the counter map of include/aepid.h (aepid_read_counters); tests/test_boundary.py checks the two against each other
COUNTER_NAMES = ("woodcock_flights", "air_flights", "epid_flights", "n_pe", "n_compton", "n_pair",
                 "esteps_phantom", "esteps_air", "esteps_epid", "n_secondaries", "unused10",
                 "unused11", "kn_iterations", "photon_cutoffs", "e_tracks", "zero_steps",
                 "iter_A", "iter_W", "iter_E", "iter_P", "iter_X",
                 "lanes_A", "lanes_W", "lanes_E", "lanes_P", "lanes_X",
                 "phases", "particles_stored", "particles_loaded", "particles_parked", "source_tasks", "majorant_violations")
EXPORTS = ("aepid_workspace_bytes", "aepid_create", "aepid_destroy", "aepid_last_error", "aepid_init_materials",
           "aepid_load_phantom", "aepid_load_epid_layers", "aepid_load_source", "aepid_set_physics",
           "aepid_reset_tallies", "aepid_simulate", "aepid_read_tallies", "aepid_read_batches",
           "aepid_set_counting", "aepid_read_counters", "aepid_sample_source", "aepid_field_size",
           "aepid_apply_response_lut", "aepid_synchronize", "aepid_set_history_offset", "aepid_read_moments",
           "aepid_finalize_moments", "aepid_upsample", "aepid_gamma_index",
           "aepid_set_phase_space", "aepid_read_phase_space_count", "aepid_set_live_limit", "aepid_set_class2", "aepid_roi_mean",
           "aepid_load_phase_space_source", "aepid_load_collimator", "aepid_read_head", "aepid_gamma_of_upsampled_static")
STATIC_MAX_PIXELS = 1280 * 1280            # AEPID_STATIC_MAX_PIXELS of include/aepid.h


class AepidError(RuntimeError):
    pass


class Dims(C.Structure):
    _fields_ = [(n, C.c_int) for n in ("n_mat", "n_E", "n_T", "nx", "ny", "nz", "n_layers", "nu", "nv",
                                       "n_bins", "fu", "fv", "n_batches", "n_ps1", "max_live_per_cta")]


def load_library():
    """dlopen libaepid.so; raise loudly if it has not been built (python -m paper_2510_24154_b200.build)."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise AepidError("libaepid.so is not built: run `python -m paper_2510_24154_b200.build` "
                         "(there is no CPU fallback)")
    lib = C.CDLL(LIB_PATH)
    lib.aepid_workspace_bytes.restype = C.c_size_t
    lib.aepid_workspace_bytes.argtypes = [C.POINTER(Dims)]
    lib.aepid_last_error.restype = C.c_char_p
    lib.aepid_last_error.argtypes = [C.c_void_p]
    lib.aepid_destroy.restype = None
    lib.aepid_destroy.argtypes = [C.c_void_p]
    lib.aepid_create.argtypes = [C.POINTER(C.c_void_p), C.c_int, C.c_void_p, C.POINTER(Dims), C.c_void_p, C.c_size_t]
    vp = C.c_void_p
    lib.aepid_init_materials.argtypes = [vp, C.c_int, C.c_int, vp, vp, vp, vp, C.c_int, vp, vp, vp]
    lib.aepid_load_phantom.argtypes = [vp, C.c_int, C.c_int, C.c_int, vp, vp, vp, vp]
    lib.aepid_load_epid_layers.argtypes = [vp, C.c_int, vp, vp, vp, vp, C.c_float, C.c_int, C.c_int, C.c_float]
    lib.aepid_load_source.argtypes = [vp, vp, vp, C.c_int, vp, vp, C.c_int, C.c_int, C.c_float, C.c_float, vp]
    lib.aepid_set_physics.argtypes = [vp, C.c_int, C.c_float, C.c_float, C.c_float, C.c_float]
    lib.aepid_reset_tallies.argtypes = [vp]
    lib.aepid_simulate.argtypes = [vp, C.c_ulonglong, C.c_ulonglong]
    lib.aepid_read_tallies.argtypes = [vp, vp, vp, vp, vp, vp]
    lib.aepid_read_batches.argtypes = [vp, vp, vp]
    lib.aepid_set_counting.argtypes = [vp, C.c_int]
    lib.aepid_read_counters.argtypes = [vp, vp]
    lib.aepid_sample_source.argtypes = [vp, C.c_ulonglong, C.c_ulonglong, C.c_ulonglong, vp]
    lib.aepid_field_size.argtypes = [vp, C.c_int, C.POINTER(C.c_float)]
    lib.aepid_apply_response_lut.argtypes = [vp, vp, C.c_int, C.c_int, C.c_float, C.c_float, C.c_float, C.c_float,
                                             C.c_float, vp, vp, vp]
    lib.aepid_synchronize.argtypes = [vp]
    lib.aepid_set_history_offset.argtypes = [vp, C.c_ulonglong]
    lib.aepid_read_moments.argtypes = [vp, vp, vp, vp, vp, vp]
    lib.aepid_finalize_moments.argtypes = [vp, vp, vp, C.c_size_t, C.c_double, C.c_double, vp, vp]
    lib.aepid_set_live_limit.argtypes = [vp, C.c_int]
    lib.aepid_set_class2.argtypes = [vp, vp]
    lib.aepid_set_phase_space.argtypes = [vp, vp, C.c_ulonglong]
    lib.aepid_read_phase_space_count.argtypes = [vp, vp]
    lib.aepid_roi_mean.argtypes = [vp, vp, C.c_int, C.c_int, C.c_float, C.c_float, vp]
    lib.aepid_load_phase_space_source.argtypes = [vp, C.c_ulonglong, vp, C.c_float]
    lib.aepid_load_collimator.argtypes = [vp, C.c_int, vp, vp, vp, vp, vp, vp, vp, vp, C.c_int, C.c_float, C.c_float]
    lib.aepid_read_head.argtypes = [vp, vp]
    lib.aepid_upsample.argtypes = [vp, vp, C.c_int, C.c_int, vp, C.c_int, C.c_int]
    lib.aepid_gamma_index.argtypes = [vp, vp, vp, C.c_int, C.c_int, C.c_float, C.c_float, C.c_float, C.c_float, C.c_float, vp, vp]
    _lib = lib
    return lib


def workspace_bytes(dims: Dims) -> int:
    return int(load_library().aepid_workspace_bytes(C.byref(dims)))


def _ptr(a, dtype=None):
    """Raw address of a numpy array (host) or a torch tensor (host or device); None -> NULL."""
    if a is None:
        return None
    if isinstance(a, np.ndarray):
        if dtype is not None and a.dtype != dtype:
            raise TypeError("expected %s, got %s" % (dtype, a.dtype))
        if not a.flags["C_CONTIGUOUS"]:
            raise ValueError("array must be C-contiguous")
        return a.ctypes.data
    if hasattr(a, "data_ptr"):
        if not a.is_contiguous():
            raise ValueError("tensor must be contiguous")
        return a.data_ptr()
    raise TypeError("expected a numpy array or a torch tensor")


def _host_f32(a):
    return np.ascontiguousarray(np.asarray(a, dtype=np.float32))


class Engine:
    """One aepid context on one GPU.  Method names follow the C-ABI: init_materials, load_phantom,
    load_epid_layers, load_source, set_physics, simulate, read_tallies, apply_response_lut."""

    def __init__(self, dims: Dims, device: int = 0, stream=None):
        import torch
        if not torch.cuda.is_available():
            raise AepidError("no CUDA device: the ARCHER-EPID path has no CPU fallback")
        self._lib = load_library()
        self._torch = torch
        self.device = torch.device("cuda", device)
        self.dims = dims
        nbytes = workspace_bytes(dims)
        if nbytes == 0:
            raise AepidError("invalid dims")
        with torch.cuda.device(self.device):
            self.workspace = torch.empty(nbytes, dtype=torch.uint8, device=self.device)   # device memory comes from torch
            self.stream = stream if stream is not None else torch.cuda.current_stream(self.device)
        self._h = C.c_void_p()
        rc = self._lib.aepid_create(C.byref(self._h), device, C.c_void_p(self.stream.cuda_stream), C.byref(dims),
                                    C.c_void_p(self.workspace.data_ptr()), nbytes)
        self._chk(rc)
        self.nu, self.nv = dims.nu, dims.nv
        self.nx, self.ny, self.nz = dims.nx, dims.ny, dims.nz
        self.n_batches = dims.n_batches

    @classmethod
    def for_config(cls, cfg, n_batches=None, device=0, stream=None, max_live_per_cta=None):
        """Engine sized for a gen.make_config dictionary (inputs are not loaded).  The class queues of the transport
        kernel are sized for the config's history count (aepid_dims.max_live_per_cta: a CTA never has more histories
        than n / 148 to start, times the two or three particles a history has alive at a time): up to 65536 particles alive
        per CTA (5 GB of queues) below 4e8 histories, 262144 (20 GB) from there on, where the longer phases pay (a 1e9-history
        launch of C3 runs 8 % faster; launches of 1e8 histories do not change)."""
        t, ph, ep, s = cfg["tables"], cfg["phantom"], cfg["epid"], cfg["source"]
        if max_live_per_cta is None:
            want = 4 * int(cfg.get("n_histories", 1 << 30)) // 128 + 1024
            max_live_per_cta = 65536 if want >= 65536 else 1 << (want - 1).bit_length()
            if int(cfg.get("n_histories", 0)) >= 400_000_000:
                max_live_per_cta = 262144
        d = Dims(n_mat=int(t["mu_compton"].shape[0]), n_E=len(t["E_grid"]), n_T=len(t["T_grid"]),
                 nx=int(ph["nx"]), ny=int(ph["ny"]), nz=int(ph["nz"]), n_layers=len(ep["thickness"]),
                 nu=int(ep["nu"]), nv=int(ep["nv"]), n_bins=len(s["E_pdf"]), fu=int(s["fu"]), fv=int(s["fv"]),
                 n_batches=int(n_batches if n_batches is not None else cfg["physics"]["n_batches"]),
                 n_ps1=int(cfg["ps1"]["n"]) if cfg.get("ps1") is not None else 0, max_live_per_cta=int(max_live_per_cta))
        return cls(d, device=device, stream=stream)

    def close(self):
        if getattr(self, "_h", None) and self._h.value:
            self._lib.aepid_destroy(self._h)
            self._h = C.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def _chk(self, rc):
        if rc != 0:
            msg = self._lib.aepid_last_error(self._h)
            raise AepidError("aepid %s: %s" % (STATUS.get(rc, rc), msg.decode() if msg else ""))

    # ---- loading: arrays may be numpy (host) or torch tensors (host or device)
    def init_materials(self, E_grid, mu_compton, mu_pe, mu_pair, T_grid, stop_pow, rad_len):
        n_mat, n_E = int(mu_compton.shape[0]), int(mu_compton.shape[1])
        self._chk(self._lib.aepid_init_materials(self._h, n_mat, n_E, _ptr(E_grid), _ptr(mu_compton), _ptr(mu_pe), _ptr(mu_pair),
                                                 int(stop_pow.shape[1]), _ptr(T_grid), _ptr(stop_pow), _ptr(rad_len)))

    def load_phantom(self, spacing, origin, density, material):
        nz, ny, nx = (int(v) for v in density.shape)
        sp, org = _host_f32(spacing), _host_f32(origin)
        self._chk(self._lib.aepid_load_phantom(self._h, nx, ny, nz, _ptr(sp), _ptr(org), _ptr(density), _ptr(material)))

    def load_epid_layers(self, thickness, material, density, scored, sid, nu, nv, pitch):
        th, rho = _host_f32(thickness), _host_f32(density)
        mat = np.ascontiguousarray(np.asarray(material, dtype=np.uint8)); sc = np.ascontiguousarray(np.asarray(scored, dtype=np.uint8))
        self._chk(self._lib.aepid_load_epid_layers(self._h, len(th), _ptr(th), _ptr(mat), _ptr(rho), _ptr(sc),
                                                   float(sid), int(nu), int(nv), float(pitch)))

    def load_source(self, src_pos, beam_axes, E_edges, E_pdf, f_pitch, f_plane_dist, fluence):
        src, ax = _host_f32(src_pos), _host_f32(beam_axes).reshape(9)
        fv, fu = (int(v) for v in fluence.shape)
        self._chk(self._lib.aepid_load_source(self._h, _ptr(src), _ptr(ax), int(E_pdf.shape[0]), _ptr(E_edges), _ptr(E_pdf),
                                              fu, fv, float(f_pitch), float(f_plane_dist), _ptr(fluence)))

    def set_physics(self, mode=1, photon_cut=0.010, electron_cut=0.200, f_E=0.10, s_max=1.0, **_):
        self._chk(self._lib.aepid_set_physics(self._h, int(mode), float(photon_cut), float(electron_cut), float(f_E), float(s_max)))

    def set_class2(self, electrons_per_gram):
        self._chk(self._lib.aepid_set_class2(self._h, _ptr(np.ascontiguousarray(electrons_per_gram, dtype=np.float32))))

    def load_config(self, cfg):
        """Host-array convenience: load everything of a gen.make_config dictionary."""
        t, ph, ep, s = cfg["tables"], cfg["phantom"], cfg["epid"], cfg["source"]
        self.init_materials(t["E_grid"], t["mu_compton"], t["mu_pe"], t["mu_pair"], t["T_grid"], t["stop_pow"], t["rad_len"])
        if "electrons_per_gram" in t:
            self.set_class2(t["electrons_per_gram"])
        self.load_phantom(ph["spacing"], ph["origin"], ph["density"], ph["material"])
        self.load_epid_layers(ep["thickness"], ep["material"], ep["density"], ep["scored"], ep["sid"], ep["nu"], ep["nv"], ep["pitch"])
        self.load_source(s["src_pos"], s["beam_axes"], s["E_edges"], s["E_pdf"], s["f_pitch"], s["f_plane_dist"], s["fluence"])
        if cfg.get("ps1") is not None:
            self.load_phase_space_source(cfg["ps1"]["records"], cfg["ps1"]["plane"])
        if cfg.get("collimator") is not None:
            self.load_collimator(cfg["collimator"])
        self.set_physics(**cfg["physics"])

    # ---- running
    def reset_tallies(self):
        self._chk(self._lib.aepid_reset_tallies(self._h))

    def simulate(self, n_histories, seed):
        self._chk(self._lib.aepid_simulate(self._h, int(n_histories), int(seed)))

    def synchronize(self):
        self._chk(self._lib.aepid_synchronize(self._h))

    def read_tallies(self, epid=True, phantom=True, sigma=True, out=None):
        """Returns a dict of numpy arrays (host).  `out` may supply preallocated numpy arrays or torch
        tensors (host or device) under the keys epid_mean / epid_sigma / phantom_mean / phantom_sigma."""
        out = dict(out or {})
        def buf(key, shape, want):
            if not want:
                return None
            if key not in out:
                out[key] = np.empty(shape, dtype=np.float32)
            return out[key]
        em = buf("epid_mean", (self.nv, self.nu), epid); es = buf("epid_sigma", (self.nv, self.nu), epid and sigma)
        pm = buf("phantom_mean", (self.nz, self.ny, self.nx), phantom); ps = buf("phantom_sigma", (self.nz, self.ny, self.nx), phantom and sigma)
        led = np.zeros(8, dtype=np.float64)
        self._chk(self._lib.aepid_read_tallies(self._h, _ptr(em), _ptr(es), _ptr(pm), _ptr(ps), _ptr(led)))
        out["ledger"] = led
        return out

    def set_history_offset(self, first_history):
        self._chk(self._lib.aepid_set_history_offset(self._h, int(first_history)))

    def read_moments(self, epid=True, phantom=True):
        """Device tensors s1 = sum_b x_b, s2 = sum_b x_b^2/n_b and totals [histories, batches]."""
        t = self._torch
        mk = lambda shape: t.empty(shape, dtype=t.float64, device=self.device)
        e1 = mk((self.nv, self.nu)) if epid else None; e2 = mk((self.nv, self.nu)) if epid else None
        p1 = mk((self.nz, self.ny, self.nx)) if phantom else None; p2 = mk((self.nz, self.ny, self.nx)) if phantom else None
        tot = np.zeros(2, dtype=np.float64)
        self._chk(self._lib.aepid_read_moments(self._h, _ptr(e1), _ptr(e2), _ptr(p1), _ptr(p2), _ptr(tot)))
        return {"epid_s1": e1, "epid_s2": e2, "phantom_s1": p1, "phantom_s2": p2, "totals": tot}

    def finalize_moments(self, s1, s2, n_histories, n_batches):
        t = self._torch
        mean = t.empty(s1.shape, dtype=t.float32, device=s1.device); sigma = t.empty(s1.shape, dtype=t.float32, device=s1.device)
        self._chk(self._lib.aepid_finalize_moments(self._h, _ptr(s1), _ptr(s2), s1.numel(), float(n_histories), float(n_batches),
                                                   _ptr(mean), _ptr(sigma)))
        return mean, sigma

    def read_batches(self):
        b = np.empty((self.n_batches, self.nv, self.nu), dtype=np.float32)
        n = np.zeros(self.n_batches, dtype=np.float64)
        self._chk(self._lib.aepid_read_batches(self._h, _ptr(b), _ptr(n)))
        return b, n

    def set_counting(self, on=True):
        self._chk(self._lib.aepid_set_counting(self._h, int(bool(on))))

    def read_counters(self):
        c = np.zeros(32, dtype=np.uint64)
        self._chk(self._lib.aepid_read_counters(self._h, _ptr(c)))
        return c

    def sample_source(self, first, n, seed):
        out = np.empty((int(n), 8), dtype=np.float32)
        self._chk(self._lib.aepid_sample_source(self._h, int(first), int(n), int(seed), _ptr(out)))
        return out

    def field_size(self, printed_form=False):
        s = C.c_float()
        self._chk(self._lib.aepid_field_size(self._h, int(bool(printed_form)), C.byref(s)))
        return float(s.value)

    # ---- collimation stage
    def load_phase_space_source(self, records, w_plane):
        """Phase Space 1 records [n][8] float32 (numpy or torch, host or device); None or empty: back to the fluence-map source."""
        n = 0 if records is None else int(records.shape[0])
        self._chk(self._lib.aepid_load_phase_space_source(self._h, n, _ptr(records) if n else None, float(w_plane)))

    def load_collimator(self, col):
        """col: {"slabs": [{w0, w1, axis, row0, pitch, lo[], hi[]}, ...], "material", "density", "w_ps2"} or None."""
        if col is None:
            self._chk(self._lib.aepid_load_collimator(self._h, 0, None, None, None, None, None, None, None, None, 0, 1.0, 0.0))
            return
        sl = col["slabs"]
        f = lambda k: _host_f32([s[k] for s in sl])
        i = lambda v: np.ascontiguousarray(v, dtype=np.int32)
        w0, w1, row0, pitch = f("w0"), f("w1"), f("row0"), f("pitch")
        axis, nr = i([s["axis"] for s in sl]), i([len(s["lo"]) for s in sl])
        lo, hi = _host_f32(np.concatenate([s["lo"] for s in sl])), _host_f32(np.concatenate([s["hi"] for s in sl]))
        self._chk(self._lib.aepid_load_collimator(self._h, len(sl), _ptr(w0), _ptr(w1), _ptr(axis), _ptr(nr), _ptr(row0), _ptr(pitch),
                                                  _ptr(lo), _ptr(hi), int(col["material"]), float(col["density"]), float(col["w_ps2"])))

    def read_head(self):
        """{Phase Space 2 particles, their energy, energy absorbed in the collimation stage, 0} since the last reset."""
        out = np.zeros(4, dtype=np.float64)
        self._chk(self._lib.aepid_read_head(self._h, _ptr(out)))
        return out

    def set_live_limit(self, max_live_per_cta=0):
        self._chk(self._lib.aepid_set_live_limit(self._h, int(max_live_per_cta)))

    def set_phase_space(self, capacity):
        """Record Phase Space 3 into a device buffer of `capacity` records (0: switch off)."""
        import torch
        if not capacity:
            self._ps3 = None
            self._chk(self._lib.aepid_set_phase_space(self._h, None, 0))
            return
        self._ps3 = torch.empty((int(capacity), 8), dtype=torch.float32, device=self.device)
        self._chk(self._lib.aepid_set_phase_space(self._h, _ptr(self._ps3), int(capacity)))

    def read_phase_space(self):
        """(records [n][8] float64 = {type, E, u, v, du, dv, dw, history}, arrivals): the stored records and the total count."""
        n = C.c_ulonglong(0)
        self._chk(self._lib.aepid_read_phase_space_count(self._h, C.byref(n)))
        k = min(int(n.value), int(self._ps3.shape[0]))
        raw = self._ps3[:k].cpu().numpy()
        bits = raw.view(np.uint32)
        out = np.empty((k, 8))
        out[:, 0] = bits[:, 6]; out[:, 1] = raw[:, 5]; out[:, 2:6] = raw[:, 0:4]; out[:, 6] = raw[:, 4]; out[:, 7] = bits[:, 7]
        return out, int(n.value)

    def _device_image(self, a):
        """float32 device tensor of a numpy array or tensor (marshalling: the C-ABI wants device pointers here)."""
        import torch
        if isinstance(a, np.ndarray):
            a = torch.from_numpy(np.ascontiguousarray(a, dtype=np.float32))
        return a.to(device=self.device, dtype=torch.float32).contiguous()

    def roi_mean(self, roi_cm=1.0, image=None, pitch_cm=None):
        """Eq. 2: mean of the current EPID image (or of `image` with its pitch) over the central ROI."""
        m = C.c_double(0.0)
        if image is None:
            self._chk(self._lib.aepid_roi_mean(self._h, None, 0, 0, 0.0, float(roi_cm), C.byref(m)))
        else:
            a = self._device_image(image)
            nv, nu = (int(v) for v in a.shape)
            self._chk(self._lib.aepid_roi_mean(self._h, _ptr(a), nu, nv, float(pitch_cm), float(roi_cm), C.byref(m)))
        return float(m.value)

    def upsample(self, image, mv, mu, out=None):
        """K9: bilinear up-sampling of image [nv][nu] to [mv][mu]; returns a device tensor."""
        import torch
        a = self._device_image(image)
        nv, nu = (int(v) for v in a.shape)
        if out is None:
            out = torch.empty((int(mv), int(mu)), dtype=torch.float32, device=self.device)
        self._chk(self._lib.aepid_upsample(self._h, _ptr(a), nu, nv, _ptr(out), int(mu), int(mv)))
        return out

    def gamma_index(self, ref, ev, pitch_cm, dose_frac=0.03, dta_cm=0.3, threshold_frac=0.10, cap=2.0, out=None):
        """K10: global gamma index of ev against ref (same grid); returns (gamma device tensor, stats dict)."""
        import torch
        r, e = self._device_image(ref), self._device_image(ev)
        if r.shape != e.shape or r.dim() != 2:
            raise ValueError("ref and ev must be 2-D images of the same shape")
        nv, nu = (int(v) for v in r.shape)
        if out is None:
            out = torch.empty((nv, nu), dtype=torch.float32, device=self.device)
        st = np.zeros(4, dtype=np.float64)
        self._chk(self._lib.aepid_gamma_index(self._h, _ptr(r), _ptr(e), nu, nv, float(pitch_cm), float(dose_frac), float(dta_cm),
                                              float(threshold_frac), float(cap), _ptr(out), _ptr(st)))
        n = int(st[0])
        return out, {"n_tested": n, "n_pass": int(st[1]), "pass_rate": (st[1] / st[0]) if n else float("nan"),
                     "mean_gamma": float(st[2]), "max_gamma": float(st[3])}

    def apply_response_lut(self, lut, t_min, t_max, s_min, s_max, s_eff=-1.0, epid_in=None, signal_out=None, tmap_out=None,
                           want_tmap=True):
        nt, ns = (int(v) for v in lut.shape)
        if signal_out is None:
            signal_out = np.empty((self.nv, self.nu), dtype=np.float32)
        if tmap_out is None and want_tmap:
            tmap_out = np.empty((self.nv, self.nu), dtype=np.float32)
        self._chk(self._lib.aepid_apply_response_lut(self._h, _ptr(lut), nt, ns, float(t_min), float(t_max), float(s_min), float(s_max),
                                                     float(s_eff), _ptr(epid_in), _ptr(signal_out), _ptr(tmap_out)))
        return signal_out, tmap_out


def gamma_of_upsampled_static(predicted, measured, pitch_cm, dose_frac=0.03, dta_cm=0.3, threshold_frac=0.10, cap=2.0,
                              out=None, stats_out=None, stream=None):
    """aepid_gamma_of_upsampled_static (include/aepid.h): K9 + K10 without a context or a workspace; the library's static device
    array is the scratch, nothing is allocated by the call.  predicted, measured: 2-D float32 CUDA tensors on the same device;
    out [mv][mu] float32 and stats_out [4] float64 are CUDA tensors of the caller (created here only if not given).  Returns
    (out, stats_out); asynchronous on `stream` (default: torch's current stream)."""
    import torch
    lib = load_library()
    if not (predicted.is_cuda and measured.is_cuda and predicted.dtype == torch.float32 and measured.dtype == torch.float32):
        raise ValueError("predicted and measured must be float32 CUDA tensors")
    predicted, measured = predicted.contiguous(), measured.contiguous()
    nv, nu = (int(v) for v in predicted.shape)
    mv, mu = (int(v) for v in measured.shape)
    dev = measured.device
    if out is None:
        out = torch.empty((mv, mu), dtype=torch.float32, device=dev)
    if stats_out is None:
        stats_out = torch.empty(4, dtype=torch.float64, device=dev)
    st = torch.cuda.current_stream(dev).cuda_stream if stream is None else int(stream)
    err = C.create_string_buffer(512)
    lib.aepid_gamma_of_upsampled_static.argtypes = [C.c_int, C.c_void_p, C.c_void_p, C.c_int, C.c_int, C.c_void_p, C.c_int, C.c_int,
                                                    C.c_float, C.c_float, C.c_float, C.c_float, C.c_float, C.c_void_p, C.c_void_p,
                                                    C.c_char_p, C.c_size_t]
    rc = lib.aepid_gamma_of_upsampled_static(dev.index or 0, C.c_void_p(st), C.c_void_p(predicted.data_ptr()), nu, nv,
                                             C.c_void_p(measured.data_ptr()), mu, mv, float(pitch_cm), float(dose_frac), float(dta_cm),
                                             float(threshold_frac), float(cap), C.c_void_p(out.data_ptr()), C.c_void_p(stats_out.data_ptr()),
                                             err, len(err))
    if rc != 0:
        raise AepidError("aepid %s: %s" % (STATUS.get(rc, rc), err.value.decode()))
    return out, stats_out
