"""Stored expected values (tests/golden/*.txt, written by tests/golden/make_golden.py from the long-double oracle alone --
the paper prints no worked example of this path).  CPU: the oracle still reproduces them (a change to its arithmetic is
noticed); GPU: the CUDA path matches values that did not come from the CUDA path."""
import os

import numpy as np
import pytest

from paper_2103_15187_b200 import inputs
from tests.golden.make_golden import CASES
from tests.util import oracle_projection

GOLD = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden")


def _load(name):
    pts, vals = [], []
    with open(os.path.join(GOLD, name + ".txt")) as f:
        for line in f:
            if line.startswith("#"):
                continue
            c = line.split()
            pts.append(tuple(int(x) for x in c[:3]))
            vals.append([float.fromhex(x) for x in c[3:]])
    return pts, np.array(vals)


@pytest.mark.parametrize("name", sorted(CASES))
def test_oracle_reproduces_golden(oracle_ld, name):
    cfg, shape, bc, beta = CASES[name]
    case = inputs.make_case(cfg, shape=shape, bc=bc)
    u, v, w, p, phi = oracle_projection(oracle_ld, case, beta)
    pts, gold = _load(name)
    got = np.array([[phi[q], u[q], v[q], w[q], p[q]] for q in pts])
    assert np.array_equal(got, gold)                           # same oracle, same inputs: bit for bit


@pytest.mark.gpu
@pytest.mark.parametrize("name", sorted(CASES))
def test_gpu_matches_golden(name):
    from tests.util import gpu_projection
    cfg, shape, bc, beta = CASES[name]
    case = inputs.make_case(cfg, shape=shape, bc=bc)
    u, v, w, p, phi = gpu_projection(case, beta)
    pts, gold = _load(name)
    got = np.array([[phi[q], u[q], v[q], w[q], p[q]] for q in pts])
    scale = np.abs(gold).max(axis=0)
    assert (np.abs(got - gold).max(axis=0) <= 1e-11 * np.maximum(scale, 1.0)).all()
