"""Helpers shared by the tests: small seeded configs built from gen/ pieces (inputs only)."""
import copy

import numpy as np

from gen import make_tables
from gen.configs import (default_physics, epid_stack, mono_spectrum, mv6_spectrum, open_field, _source, _IDENT)
from gen.tables import MAT_SOFT

_TABLES = None


def tables():
    global _TABLES
    if _TABLES is None:
        _TABLES = make_tables()
    return copy.deepcopy(_TABLES)


def slab_cfg(n=(16, 16, 40), h=(0.5, 0.5, 0.5), w0=100.0, rho=1.0, mat=MAT_SOFT, E=2.0, mode=0,
             epid="C0", nu=64, nv=64, pitch=0.4, sid=170.0, field_cm=10.0, t=None, spectrum=None):
    """Homogeneous slab phantom centred on the beam axis, top face at w = w0, identity beam axes."""
    nx, ny, nz = n
    ph = {"nx": nx, "ny": ny, "nz": nz, "spacing": np.array(h, dtype=np.float32),
          "origin": np.array([-0.5 * nx * h[0], -0.5 * ny * h[1], w0], dtype=np.float32),
          "density": np.full((nz, ny, nx), rho, dtype=np.float32),
          "material": np.full((nz, ny, nx), mat, dtype=np.uint8)}
    fl, p = open_field(field_cm)
    spec = spectrum if spectrum is not None else mono_spectrum(E)
    return {"name": "slab", "tables": t if t is not None else tables(), "phantom": ph,
            "epid": epid_stack(epid, nu, nv, pitch, sid),
            "source": _source((0, 0, 0), _IDENT, spec, fl, p),
            "physics": default_physics(mode=mode), "n_histories": 100000, "seed": 1, "lut": None}


def rebin2d(a, r):
    a = np.asarray(a)
    return a.reshape(a.shape[0] // r, r, a.shape[1] // r, r).sum(axis=(1, 3))
