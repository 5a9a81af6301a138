"""Host logic of libfsei (-m "not gpu"): the per-thread device phases of csrc/*.cuh stepped on the
host (tests/emu) against the long-double oracle, plus the plan's table/factorisation logic.
This checks the index arithmetic of the CUDA path without a GPU; the GPU parity tests proper are
in test_gpu_parity.py."""
import ctypes

import numpy as np
import pytest

from paper_2103_15187_b200 import inputs
from tests.util import emu_lib, emu_projection, oracle_projection, rel_l2

P, N = 0, 1


@pytest.mark.parametrize("bc", [(P, P), (N, N), (P, N), (N, P)])
@pytest.mark.parametrize("shape", [(8, 8, 8), (16, 12, 10), (48, 24, 20), (12, 36, 7), (64, 16, 5), (20, 10, 6), (40, 50, 5), (60, 30, 4)])
def test_stepped_phases_match_oracle(oracle_ld, bc, shape):
    for cfg, beta in ((1, 0.0), (2, 1e-4)):
        case = inputs.make_case(cfg, shape=shape, bc=bc)
        got = emu_projection(case, beta)
        ref = oracle_projection(oracle_ld, case, beta)
        assert rel_l2(got[4], ref[4]) < 1e-13
        for g, r in zip(got[:4], ref[:4]):
            assert np.abs(g - r).max() <= 1e-11 * max(1.0, np.abs(r).max())


def test_stepped_phases_config1_full(oracle_ld):
    case = inputs.make_case(1)
    got = emu_projection(case)
    ref = oracle_projection(oracle_ld, case)
    assert rel_l2(got[4], ref[4]) < 1e-13


@pytest.mark.parametrize("n,expect", [(16, [16]), (32, [8, 4]), (128, [16, 8]), (256, [16, 16]), (512, [8, 8, 8]),
                                      (1024, [16, 8, 8]), (384, [3, 16, 8]), (768, [3, 16, 16]), (6, [3, 2]), (2, [2]),
                                      (10, [5, 2]), (320, [5, 8, 8]), (60, [3, 5, 4]), (1250, [5, 5, 5, 5, 2])])
def test_radix_plan(n, expect):
    L = emu_lib()
    r = (ctypes.c_int * 8)()
    np_ = L.emu_plan_radices(n, r)
    got = list(r[:np_])
    assert got == expect and int(np.prod(got)) == n


def test_plan_argument_checks():
    L = emu_lib()
    zc = np.linspace(0, 1, 9)
    chk = lambda nx, ny, nz, Lx, Ly, z, bx, by: L.emu_plan_check(nx, ny, nz, Lx, Ly, z.ctypes.data_as(ctypes.POINTER(ctypes.c_double)), bx, by)
    assert chk(8, 8, 8, 1.0, 1.0, zc, 0, 0) == 0
    assert chk(28, 8, 8, 1.0, 1.0, zc, 0, 0) == 2          # 28 = 4*7
    assert chk(8, 14, 8, 1.0, 1.0, zc, 0, 0) == 2          # 14 = 2*7
    assert chk(20, 10, 8, 1.0, 1.0, zc, 0, 0) == 0         # radix 5
    assert chk(10, 8, 8, 1.0, 1.0, zc, 0, 0) == 2          # nx not a multiple of 4
    assert chk(6, 8, 8, 1.0, 1.0, zc, 0, 0) == 2           # nx not a multiple of 4
    assert chk(8, 8, 8, 0.0, 1.0, zc, 0, 0) == 3
    assert chk(8, 8, 8, 1.0, 1.0, zc[::-1].copy(), 0, 0) == 3
    assert chk(8, 8, 8, 1.0, 1.0, zc, 2, 0) == 1
    bad = zc.copy(); bad[3] = np.nan
    assert chk(8, 8, 8, 1.0, 1.0, bad, 0, 0) == 3
