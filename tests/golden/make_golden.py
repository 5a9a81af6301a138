#!/usr/bin/env python
"""Writes tests/golden/*.txt from the ORACLE alone (long-double build): regression fixtures of the oracle's answers on
small seeded cases.  The paper (arXiv 2103.15187) prints no worked example of the pressure projection,
so there is no paper value to store; the independent pins of the oracle are in tests/test_oracle_pins.py.  These
fixtures fix the oracle's output at sampled points so that a later change to its arithmetic is noticed, and give the
CUDA path a stored expected value that did not come from the CUDA path.

    python tests/golden/make_golden.py        # rewrites the fixtures; calls only oracle/ and the input generator
"""
import os
import sys

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, os.path.dirname(os.path.dirname(HERE)))

from oracle import Oracle                                  # noqa: E402
from paper_2103_15187_b200 import inputs                   # noqa: E402  (seeded inputs only: no method arithmetic)

CASES = {  # name: (config, shape or None, (bc_x, bc_y) or None, beta)
    "cfg1_32x32x32_PP": (1, None, None, 0.0),
    "cfg2_recipe_64x48x40_NN": (2, (64, 48, 40), (1, 1), 1e-4),
    "cfg4_recipe_96x32x24_PN": (4, (96, 32, 24), (0, 1), 0.0),
}
NSAMPLE = 24


def sample_points(case):
    rng = np.random.default_rng(12345)
    return [(int(rng.integers(case.nz)), int(rng.integers(case.ny)), int(rng.integers(case.nx))) for _ in range(NSAMPLE)]


def main():
    orc = Oracle("ld")
    for name, (cfg, shape, bc, beta) in CASES.items():
        case = inputs.make_case(cfg, shape=shape, bc=bc)
        u, v, w = case.u.copy(), case.v.copy(), case.w.copy()
        p = np.zeros_like(u)
        phi = orc.pressure_projection(case.grid, u, v, w, p, case.alpha_dt, beta)
        with open(os.path.join(HERE, name + ".txt"), "w") as f:
            f.write(f"# {name}: long-double oracle (oracle/fsei_oracle.c) on inputs.make_case({cfg}, shape={shape}, bc={bc}), "
                    f"beta={beta}\n# written by tests/golden/make_golden.py; columns: k j i phi u_new v_new w_new p_new (hex floats)\n")
            for (k, j, i) in sample_points(case):
                vals = [phi[k, j, i], u[k, j, i], v[k, j, i], w[k, j, i], p[k, j, i]]
                f.write(f"{k} {j} {i} " + " ".join(float(x).hex() for x in vals) + "\n")
        print("wrote", name)


if __name__ == "__main__":
    main()
