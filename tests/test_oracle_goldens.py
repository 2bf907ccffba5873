"""The stored oracle runs (tests/golden/oracle_<case>.npz, written by tests/golden/make_oracle_goldens.py from oracle/ alone)
still describe the oracle as it stands and the inputs as gen/ makes them today.  No GPU."""
import os
import sys

import numpy as np
import pytest

import oracle
from gen import make_config

HERE = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, os.path.join(HERE, "golden"))
from make_oracle_goldens import CASES, input_hash   # noqa: E402


@pytest.mark.parametrize("case", sorted(CASES))
def test_golden_file_matches_todays_inputs_and_oracle(case):
    path = os.path.join(HERE, "golden", "oracle_%s.npz" % case)
    assert os.path.exists(path), "run tests/golden/make_oracle_goldens.py --only %s" % case
    g = np.load(path)
    cname, field, n_decl, rb, pb = CASES[case]
    cfg = make_config(cname, field=field)
    assert str(g["input_sha256"]) == input_hash(cfg)
    n = int(g["n"])
    assert abs(n - n_decl) < 1e-3 * n_decl and int(g["rb"]) == rb and tuple(int(v) for v in g["pb"]) == pb and int(g["seed"]) == cfg["seed"]
    L = g["ledger"]
    assert L[6] == n and abs(L[1] + L[2] + L[3] + L[4] + L[5] - L[0]) < 1e-11 * L[0]
    assert g["rb_sum"].sum() == pytest.approx(L[2], rel=1e-10)
    assert g["dd_runs"].mean(0).sum() * n == pytest.approx(L[1], rel=1e-9)
    assert g["pc_sum"].sum() <= L[1] and g["pc_sum"].sum() > 0.3 * L[1]          # only the blocks above 2 % of the maximum are kept
    # a fresh, disjoint run of the oracle as it stands agrees channel by channel within its own statistics
    m = 8000 if cname == "C3" else 20000
    raw = oracle.run_sharded(cfg, m, cfg["seed"], first=n, procs=4, want_phantom_sq=False)
    mo = L / n
    so = np.sqrt(np.maximum(g["ledger_sq"] / n - mo ** 2, 0.0))
    for k in range(6):
        assert abs(raw["ledger"][k] / m - mo[k]) <= 4.5 * so[k] * np.sqrt(1.0 / m + 1.0 / n) + 1e-12, k
