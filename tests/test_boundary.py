"""Host-side checks that need no GPU: the C-ABI library loads and exports every symbol include/aepid.h declares,
the binding fails loudly without a device, the product never touches the oracle, inputs are deterministic."""
import ctypes
import os
import re

import numpy as np
import pytest

import paper_2510_24154_b200 as pkg
from paper_2510_24154_b200 import build as pkg_build
from gen import make_config, make_tables

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    pkg_build.build()
    return pkg.load_library()


def test_library_exports_every_declared_symbol(lib):
    hdr = open(os.path.join(ROOT, "include", "aepid.h")).read()
    hdr = re.sub(r"/\*.*?\*/", "", hdr, flags=re.S)
    declared = set(re.findall(r"\b(aepid_[a-z_0-9]+)\s*\(", hdr))
    assert len(declared) >= 20
    for name in declared:
        assert hasattr(lib, name), name
    assert declared == set(pkg.EXPORTS)
    # the north_star call list is present
    for name in ("init_materials", "load_phantom", "load_epid_layers", "load_source", "simulate", "read_tallies", "apply_response_lut"):
        assert "aepid_" + name in declared


def test_counter_names_match_the_header():
    hdr = open(os.path.join(ROOT, "include", "aepid.h")).read()
    blk = hdr[hdr.index("Counter map, index name"):hdr.index("0-9, 12-15: events of the physics")]
    pairs = dict((int(i), n) for i, n in re.findall(r"\b(\d+) ([a-z][a-z_0-9A-Z]*)", blk))
    assert sorted(pairs) == list(range(32))
    assert tuple(pairs[i] for i in range(32)) == tuple(pkg.COUNTER_NAMES)
    # the oracle counts the same physics events under the same names (0-9, 12-15)
    import oracle
    for i in list(range(10)) + [12, 13, 14, 15]:
        assert oracle.COUNTER_NAMES[i] == pkg.COUNTER_NAMES[i], i
    assert "AEPID_ERR_INTERNAL = -6" in hdr and pkg.binding.STATUS[-6] == "INTERNAL"


def test_workspace_bytes_validates_dims(lib):
    d = pkg.Dims(n_mat=8, n_E=500, n_T=200, nx=120, ny=120, nz=80, n_layers=4, nu=512, nv=384, n_bins=200, fu=100, fv=100, n_batches=32)
    n = pkg.workspace_bytes(d)
    vox, pix = 120 * 120 * 80, 512 * 384
    assert n >= 4 * vox * (1 + 32 + 2) + 4 * pix * (32 + 2 + 3)
    pool = 160 * 5 * 131072 * 48                             # class queues of particle records of the transport kernel (params.h)
    assert n < 1.1 * (4 * vox * 35 + 4 * pix * 37) + pool + (2 << 20)
    # the class queues follow dims.max_live_per_cta: twice as many 48-byte records per class and CTA, rounded up to a power of two
    small = pkg.Dims.from_buffer_copy(d); small.max_live_per_cta = 1000
    assert n - pkg.workspace_bytes(small) == 160 * 5 * (131072 - 2048) * 48
    big = pkg.Dims.from_buffer_copy(d); big.max_live_per_cta = 262144          # the largest: what Engine.for_config takes from 4e8 histories on
    assert pkg.workspace_bytes(big) - n == 160 * 5 * (524288 - 131072) * 48
    for field, bad in (("n_batches", 1), ("n_batches", 256), ("nx", 0), ("nx", 2000), ("n_mat", 33), ("n_layers", 9), ("fu", 0),
                       ("max_live_per_cta", 63), ("max_live_per_cta", 262145)):
        e = pkg.Dims.from_buffer_copy(d)
        setattr(e, field, bad)
        assert pkg.workspace_bytes(e) == 0, field


def test_no_cpu_fallback_without_a_device(lib):
    import torch
    if torch.cuda.is_available():
        pytest.skip("has a GPU")
    d = pkg.Dims(n_mat=8, n_E=500, n_T=200, nx=8, ny=8, nz=8, n_layers=2, nu=8, nv=8, n_bins=1, fu=4, fv=4, n_batches=4)
    with pytest.raises(pkg.AepidError):
        pkg.Engine(d)
    # the raw C-ABI refuses as well
    h = ctypes.c_void_p()
    rc = lib.aepid_create(ctypes.byref(h), 0, None, ctypes.byref(d), ctypes.c_void_p(256), 1 << 30)
    assert rc == -4 and b"no CPU fallback" in lib.aepid_last_error(h)
    lib.aepid_destroy(h)


def test_product_is_independent_of_oracle_and_reference():
    pdir = os.path.join(ROOT, "paper_2510_24154_b200")
    for dp, _, files in os.walk(pdir):
        for f in files:
            if f.endswith((".py", ".cu", ".h", ".cuh")):
                src = open(os.path.join(dp, f)).read()
                assert not re.search(r"^\s*(from|import)\s+oracle", src, flags=re.M), f
                assert "liboracle" not in src and "/root/reference" not in src and "_work/" not in src, f
    ocpp = open(os.path.join(ROOT, "oracle", "oracle.cpp")).read()
    opy = open(os.path.join(ROOT, "oracle", "__init__.py")).read()
    assert not re.search(r"^\s*(from|import)\s+paper_2510_24154_b200", opy, flags=re.M) and "libaepid" not in opy
    includes = re.findall(r'#include\s*[<"]([^>"]+)[>"]', ocpp)
    assert includes and all("/" not in i and not i.endswith((".h", ".cuh")) for i in includes)   # standard library only
    for f in ("bench.py", "__graft_entry__.py"):
        assert "/root/reference" not in open(os.path.join(ROOT, f)).read()


def test_generators_are_seeded_and_shaped_like_the_configs():
    t = make_tables()
    assert t["mu_compton"].shape == (8, 500) and t["stop_pow"].shape == (8, 200)
    assert t["E_grid"][0] == pytest.approx(1e-3) and t["E_grid"][-1] == pytest.approx(20.0)
    c0, c1 = make_config("C0", tables=t), make_config("C1", tables=t)
    assert c0["phantom"]["density"].shape == (40, 64, 64) and c0["epid"]["nu"] == 64 and c0["physics"]["mode"] == 0
    assert c0["n_histories"] == 100_000 and c0["seed"] == 1 and c0["source"]["E_edges"][0] == 2.0
    assert c1["phantom"]["density"].shape == (80, 120, 120) and (c1["epid"]["nu"], c1["epid"]["nv"]) == (512, 384)
    assert c1["epid"]["pitch"] == pytest.approx(0.0784) and len(c1["epid"]["thickness"]) == 4 and c1["n_histories"] == 10_000_000
    e, p = c1["source"]["E_edges"].astype(float), c1["source"]["E_pdf"].astype(float)
    assert len(p) == 200 and abs((0.5 * (e[1:] + e[:-1]) * p).sum() / p.sum() - 1.8) < 0.05
    a, b = make_config("C2", shrink=4, tables=t), make_config("C2", shrink=4, tables=t)
    assert np.array_equal(a["phantom"]["density"], b["phantom"]["density"]) and np.array_equal(a["source"]["fluence"], b["source"]["fluence"])
    assert set(np.unique(a["phantom"]["material"])) == {0, 1, 2, 3}
    f0, f1 = make_config("C4", field=0, shrink=8, tables=t), make_config("C4", field=1, shrink=8, tables=t)
    assert not np.array_equal(f0["source"]["fluence"], f1["source"]["fluence"]) and (f0["seed"], f1["seed"]) == (2000, 2001)
    assert f0["lut"]["lut"].shape == (64, 64) and 0.85 <= f0["lut"]["lut"].min() and f0["lut"]["lut"].max() <= 1.15
    fl = make_config("C2", shrink=8, tables=t)["source"]["fluence"]
    rows = np.nonzero(fl.sum(axis=1))[0]
    assert rows.min() % 5 == 0 and (rows.max() + 1) % 5 == 0          # apertures span whole 5 mm leaves
