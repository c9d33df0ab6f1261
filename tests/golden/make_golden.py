#!/usr/bin/env python
"""Writes tests/golden/oracle_runs.json: theta / F histories and iteration counts of the ORACLE on the
seeded configs[0]-, configs[1]-shaped inputs (8^4 and a pure-gauge copy of the unit field).

PAPER.md prints no worked example and no intermediate values, so these are not the
paper's numbers: they are regression values of oracle/ alone (this script imports only `oracle` and the
input generator `lgf_inputs`; nothing from the CUDA path), checked by tests/test_golden.py so that a later
change of the oracle's arithmetic cannot pass unnoticed.  Run from the repo root:
    python tests/golden/make_golden.py
"""
import json
import os
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
sys.path.insert(0, ROOT)

import lgf_inputs as gi  # noqa: E402
import oracle  # noqa: E402

ALPHA = 0.08


def run(L, U, tol):
    _, n, theta, F, thh, Fh = oracle.fix(L, U, ALPHA, tol, 5000)
    return {"L": list(L), "alpha": ALPHA, "theta_tol": tol, "iterations": int(n), "theta": float(theta), "F": float(F),
            "theta_history": [float(v) for v in thh], "F_history": [float(v) for v in Fh]}


def main():
    out = {"_note": "oracle regression values (not from the paper); written by tests/golden/make_golden.py"}
    L = (8, 8, 8, 8)
    out["config0_8x4_rough"] = run(L, gi.make_config(L, gi.CONFIG_SEED + 0, 0.59), 1e-12)
    out["config1_8x4_pure_gauge"] = run(L, gi.make_config(L, gi.CONFIG_SEED + 1, kind="pure_gauge"), 1e-15)
    L2 = (6, 4, 12, 8)
    out["mixed_radix_6x4x12x8_rough"] = run(L2, gi.make_config(L2, gi.CONFIG_SEED + 3, 0.58), 1e-12)
    with open(os.path.join(os.path.dirname(os.path.abspath(__file__)), "oracle_runs.json"), "w") as f:
        json.dump(out, f, indent=1)
    for k, v in out.items():
        if isinstance(v, dict):
            print(k, v["iterations"], v["theta"], v["F"])


if __name__ == "__main__":
    main()
