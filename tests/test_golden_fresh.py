"""CPU-only: the cached oracle runs under tests/golden/ belong to the oracle as it stands.

The full-size GPU parity tests compare the CUDA path with values tests/golden/make_reference.py computed once (an hour of
oracle time).  Two things keep those files honest: every file records the sha256 of the oracle's sources it was written (or
re-stamped) with, compared here and in the GPU tests with the live sources; and a few (event, lambda) units per file are
recomputed here with the live oracle.  No value in the files or in this test comes from the CUDA path."""
import importlib.util
import os

import numpy as np
import pytest

from workloads import make_workload

GOLD = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden")
_spec = importlib.util.spec_from_file_location("make_reference", os.path.join(GOLD, "make_reference.py"))
MR = importlib.util.module_from_spec(_spec)
_spec.loader.exec_module(MR)


def test_every_cached_reference_names_the_live_oracle():
    live = MR.oracle_hash()
    for name in MR.SETS:
        g = np.load(os.path.join(GOLD, f"ref_{name}.npz"))
        assert "oracle_sha256" in g.files, name
        assert str(g["oracle_sha256"]) == live, (f"ref_{name}.npz was written with another version of oracle/: rerun "
                                                 "tests/golden/make_reference.py (or --stamp, which recomputes units first)")


# (the two sets whose inputs take seconds to draw; --stamp recomputes the same units on all six)
@pytest.mark.parametrize("name", ["o5_spec_cat0", "sel_heavy"])
def test_cached_units_recomputed_with_the_live_oracle(name):
    cfg, cat = MR.SETS[name][:2]
    w = make_workload(cfg, catalog=cat)
    g = np.load(os.path.join(GOLD, f"ref_{name}.npz"))
    assert MR.input_hash(w) == str(g["input_sha256"])
    for row, ev in MR.check_units(w):
        got, ref = MR.recompute_unit(w, g["lam"][row], ev), float(g["event_logI"][row, ev])
        assert np.isfinite(ref) == np.isfinite(got)
        if np.isfinite(ref):
            assert abs(got - ref) <= 1e-12 * abs(ref), (name, row, ev, got, ref)
