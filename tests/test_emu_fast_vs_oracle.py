"""Host logic of the fast path (-m "not gpu"): the fast-path kernels of csrc/{xfast,yfast,zfast,stencil_fast}.cuh
compiled for the host (tests/emu/emu_fast.cpp, a CTA = a team of host threads with a barrier) against the long-double
oracle.  Checks the Stockham passes, padded tiles, Hermitian pair steps, split y-spectra and special z columns of every
line-length instantiation without a GPU; the GPU parity tests proper are in test_gpu_parity.py."""
import numpy as np
import pytest

from paper_2103_15187_b200 import inputs
from tests.util import emu_fast_lib, emu_fast_projection, oracle_projection, rel_l2

P, N = 0, 1


def _check(oracle_ld, shape, bc, split=False, cfg=2, beta=1e-4):
    case = inputs.make_case(cfg, shape=shape, bc=bc)
    got = emu_fast_projection(case, beta, split)
    ref = oracle_projection(oracle_ld, case, beta)
    assert rel_l2(got[4], ref[4]) < 1e-13
    for g, r in zip(got[:4], ref[:4]):
        assert np.abs(g - r).max() <= 1e-11 * max(1.0, np.abs(r).max())
    return got


@pytest.mark.parametrize("bc", [(P, P), (N, N), (P, N), (N, P)])
@pytest.mark.parametrize("shape", [(32, 32, 8), (64, 16, 5), (96, 48, 7), (128, 64, 3)])
def test_fast_kernels_match_oracle(oracle_ld, bc, shape):
    a = _check(oracle_ld, shape, bc, split=False)
    b = _check(oracle_ld, shape, bc, split=True)
    for x, y in zip(a, b):
        assert np.array_equal(x, y)                    # fused divergence == divergence kernel + x-forward


# every x line length (nx = 2 N) and every y column length with an instantiation, both transforms types
@pytest.mark.parametrize("nx", [32, 64, 96, 128, 192, 256, 384, 512, 768, 1024, 2048, 160, 320, 640, 1280, 480, 576, 960, 1152])
def test_every_x_length(oracle_ld, nx):
    for bc in ((P, P), (N, N)):
        _check(oracle_ld, (nx, 16, 2), bc)


@pytest.mark.parametrize("ny", [16, 32, 48, 64, 96, 128, 192, 256, 384, 512, 768, 1024, 80, 160, 320, 640, 1280, 240, 288, 480, 576, 960, 1152])
def test_every_y_length(oracle_ld, ny):
    for bc in ((P, P), (N, N), (N, P)):
        _check(oracle_ld, (32, ny, 2), bc)


@pytest.mark.parametrize("bc", [(P, P), (N, N), (P, N), (N, P)])
@pytest.mark.parametrize("shape", [(32, 16, 32), (32, 16, 7)])
def test_short_columns_pcr(oracle_ld, bc, shape):
    """nz <= 32: the warp-shuffle PCR kernel (lane = k) instead of the Thomas sweeps"""
    case = inputs.make_case(2, shape=shape, bc=bc)
    got = emu_fast_projection(case, 1e-4, 2)                     # split & 2: PCR z kernel
    ref = oracle_projection(oracle_ld, case, 1e-4)
    assert rel_l2(got[4], ref[4]) < 1e-13
    for g, r in zip(got[:4], ref[:4]):
        assert np.abs(g - r).max() <= 1e-11 * max(1.0, np.abs(r).max())


def test_fast_config1_full(oracle_ld):
    _check(oracle_ld, (32, 32, 32), (P, P), cfg=1, beta=0.0)


def test_fast_support_matrix():
    L = emu_fast_lib()
    assert L.emu_fast_supported(1024, 1024) and L.emu_fast_supported(768, 768) and L.emu_fast_supported(32, 32)
    assert not L.emu_fast_supported(12, 36) and not L.emu_fast_supported(8, 8)


# ---- fused path: blocked spectrum layout, Thomas sweeps riding on the z-marching y kernels (yzfused.cuh) ----------
# The short line lengths (nx = 32, 64, 96; ny = 16, 32, 48) are instantiated for tests; the plan picks the fused path
# on large grids only, and the GPU parity tests cover the production lengths.
def _check_fused(oracle_ld, shape, bc, cfg=2, beta=1e-4, mode=0):
    case = inputs.make_case(cfg, shape=shape, bc=bc)
    got = emu_fast_projection(case, beta, mode, fused=True)
    ref = oracle_projection(oracle_ld, case, beta)
    assert rel_l2(got[4], ref[4]) < 1e-13
    for g, r in zip(got[:4], ref[:4]):
        assert np.abs(g - r).max() <= 1e-11 * max(1.0, np.abs(r).max())
    return got


@pytest.mark.parametrize("bc", [(P, P), (N, N), (P, N), (N, P)])
@pytest.mark.parametrize("shape", [(32, 32, 5), (64, 16, 9), (96, 48, 4)])
def test_fused_kernels_match_oracle(oracle_ld, bc, shape):
    a = _check_fused(oracle_ld, shape, bc)
    b = _check_fused(oracle_ld, shape, bc, mode=1)               # divergence kernel + non-fused blocked x-forward
    for x, y in zip(a, b):
        assert np.array_equal(x, y)


@pytest.mark.parametrize("bc", [(P, P), (N, N), (P, N), (N, P)])
@pytest.mark.parametrize("shape", [(32, 32, 4), (64, 48, 7), (96, 16, 12), (32, 16, 5)])
def test_fused_twisted_factorisation(oracle_ld, bc, shape):
    """two CTAs per tile: planes [0, nz/2) eliminated upwards, planes [nz/2, nz) downwards, met in the middle"""
    a = _check_fused(oracle_ld, shape, bc, mode=4)               # mode & 4: twisted
    b = _check_fused(oracle_ld, shape, bc)
    assert rel_l2(a[4], b[4]) < 1e-13


# production lengths: one blocked x length and one z-marching y length per run (nz = 2 keeps the thread teams cheap)
@pytest.mark.parametrize("shape,bc", [((512, 384, 2), (P, P)), ((768, 512, 2), (N, N))])
def test_fused_production_lengths(oracle_ld, shape, bc):
    _check_fused(oracle_ld, shape, bc)


def test_fused_support_matrix():
    L = emu_fast_lib()
    assert L.emu_fused_supported(1024, 1024) and L.emu_fused_supported(768, 768) and L.emu_fused_supported(512, 384)
    assert L.emu_fused_supported(32, 32) and not L.emu_fused_supported(256, 256) and not L.emu_fused_supported(128, 64)
