"""Writes tests/golden/oracle_3d_digest.txt: SHA-256 digests of states produced by the ORACLE
(oracle/ only; nothing here touches the CUDA path) on a few small 3D cases with cubic cells.

Purpose: a regression pin.  The digests were written by the round-1 oracle (git 4b8e834, the
version pinned by P1-P12) BEFORE the oracle was extended to 1D / 2D runs and non-cubic cells
(readings R21-R24); the extended oracle must reproduce them bit for bit, i.e. the 3D
cubic-cell path is unchanged.  Re-running this script rewrites the file from the oracle as it
stands, so only run it to add cases.

    python tests/golden/make_oracle_digest.py
"""
import hashlib
import os
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
sys.path.insert(0, ROOT)

import numpy as np  # noqa: E402

import oracle  # noqa: E402
from paper_1812_07977_b200 import inputs  # noqa: E402

OUT, REF, PER = 0, 1, 2
CASES = [
    # name, shape, bc, gamma, cfl, theta, steps, generator
    ("sphere16_outflow", (16, 16, 16), (OUT,) * 6, 1.4, 0.7, 1.4, 6, lambda: inputs.sphere(16)),
    ("random_20x12x7_mixed", (20, 12, 7), (OUT, REF, PER, PER, REF, OUT), 1.4, 0.5, 2.0, 5,
     lambda: inputs.random_state(20, 12, 7, seed=42, vamp=0.4)),
    ("noise12_periodic", (12, 12, 12), (PER,) * 6, 5.0 / 3.0, 0.5, 1.0, 5,
     lambda: inputs.noise(12, seed=3)),
    ("sod_64x2x2", (64, 2, 2), (OUT, OUT, PER, PER, PER, PER), 1.4, 0.7, 1.4, 12,
     lambda: inputs.sod(64, 2, 2)),
]


def run(case):
    name, shape, bc, gamma, cfl, theta, steps, make = case
    h = oracle.OracleHydro(*shape, gamma, 1.0 / shape[0], bc)
    h.set_cfl(cfl)
    h.set_limiter_theta(theta)
    h.set_state(make())
    for _ in range(steps):
        h.step(h.cfl_dt())
    U = h.get_state()
    t, n = h.get_time()
    return hashlib.sha256(U.tobytes()).hexdigest(), t.hex(), n


def main():
    path = os.path.join(os.path.dirname(os.path.abspath(__file__)), "oracle_3d_digest.txt")
    with open(path, "w") as f:
        f.write("# written by tests/golden/make_oracle_digest.py from oracle/ (see its docstring)\n")
        f.write("# case  sha256(state bytes, float64 [5][nz][ny][nx])  t.hex()  steps\n")
        for c in CASES:
            d, t, n = run(c)
            f.write(f"{c[0]} {d} {t} {n}\n")
    print(open(path).read())


if __name__ == "__main__":
    main()
