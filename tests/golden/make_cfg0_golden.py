"""Writes tests/golden/cfg0_oracle_spectrum.txt: the ORACLE's spectrum of BASELINE.json
configs[0] (tiny helical check: 256 electrons, 128 steps, 8 directions x 64 linear
frequencies, raw scale = 1).  Calls only oracle/ and the seeded input generator.

The paper prints no values for this (or any) detector configuration, so this file is a
regression fixture for the oracle (it makes a silent change of the oracle's arithmetic
visible), NOT an external pin; the external pins are in tests/test_oracle_pins.py.

    python tests/golden/make_cfg0_golden.py
"""
import sys
from pathlib import Path

import numpy as np

ROOT = Path(__file__).resolve().parents[2]
sys.path.insert(0, str(ROOT))
from oracle import oracle  # noqa: E402
from paper_2501_03383_b200 import workloads as wl  # noqa: E402


def compute():
    w = wl.make_workload("0")
    o = oracle.Oracle(w.dirs, w.omega, w.dt, t0=w.t0, scale=1.0)
    for t, st in w.steps():
        o.accumulate_step(t, *st)
    return o.spectrum()


if __name__ == "__main__":
    S = compute()
    out = Path(__file__).with_name("cfg0_oracle_spectrum.txt")
    np.savetxt(out, S, fmt="%.17e",
               header="oracle spectrum, BASELINE.json configs[0], scale=1, rows=directions, "
                      "cols=frequencies; written by tests/golden/make_cfg0_golden.py")
    print("wrote", out, S.shape, S.max())
