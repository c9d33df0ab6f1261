"""The oracle against its stored regression values (tests/golden/oracle_runs.json, written by
tests/golden/make_golden.py from oracle/ alone; PAPER.md prints no values to store instead)."""
import json
import os

import numpy as np
import pytest

import lgf_inputs as gi
import oracle

GOLDEN = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden", "oracle_runs.json")
CASES = {
    "config0_8x4_rough": lambda L: gi.make_config(L, gi.CONFIG_SEED + 0, 0.59),
    "config1_8x4_pure_gauge": lambda L: gi.make_config(L, gi.CONFIG_SEED + 1, kind="pure_gauge"),
    "mixed_radix_6x4x12x8_rough": lambda L: gi.make_config(L, gi.CONFIG_SEED + 3, 0.58),
}


@pytest.mark.parametrize("name", sorted(CASES))
def test_oracle_reproduces_golden_run(name):
    g = json.load(open(GOLDEN))[name]
    L = tuple(g["L"])
    _, n, theta, F, thh, Fh = oracle.fix(L, CASES[name](L), g["alpha"], g["theta_tol"], 5000)
    assert n == g["iterations"]
    assert abs(F - g["F"]) <= 1e-13
    # theta histories: relative 1e-9 while theta is above the cancellation floor
    ref = np.array(g["theta_history"])
    got = np.array(thh)
    big = ref > 1e-9
    assert np.all(np.abs(got[big] - ref[big]) <= 1e-9 * ref[big])
    assert np.all(np.abs(np.array(Fh) - np.array(g["F_history"])) <= 1e-12)
    # what the mathematics fixes, independent of the stored numbers: F never decreases, theta ends below tol
    assert np.all(np.diff(np.array(Fh)) >= -1e-15) and theta < g["theta_tol"]
    if "pure_gauge" in name:
        assert abs(1.0 - F) < 1e-13
