"""Pins of the C2C oracle (oracle_c2c) against things other than itself: the O(N^6)
definition on tiny grids, closed forms, invariants, numpy.fft as a library cross-check, and the R2C oracle
(a real input's C2C spectrum restricted to kz <= Nz/2 is Eq. (4), its other half Eq. (3))."""
import numpy as np
import pytest


def rnd(shape, seed):
    g = np.random.Generator(np.random.PCG64(seed))
    return g.standard_normal(shape) + 1j * g.standard_normal(shape)


@pytest.mark.parametrize("shape", [(8, 8, 8), (4, 6, 10), (6, 5, 4), (3, 4, 7)])
def test_fast_matches_the_definition(oracle_mod, shape):
    f = rnd(shape, 1)
    for sign in (-1, +1):
        a = oracle_mod.c2c(f, sign)
        b = oracle_mod.dft3d_c2c_direct(f, sign)
        assert np.abs(a - b).max() <= 1e-12 * max(1.0, np.abs(b).max())


def test_delta_shift_and_sign(oracle_mod):
    shape = (6, 8, 10)
    j0 = (2, 5, 7)
    f = np.zeros(shape, dtype=np.complex128)
    f[j0] = 1.0
    F = oracle_mod.c2c(f, -1)
    k = np.meshgrid(*[np.arange(n) for n in shape], indexing="ij")
    phase = sum(k[d] * j0[d] / shape[d] for d in range(3))
    assert np.abs(F - np.exp(-2j * np.pi * phase)).max() <= 1e-13      # a flipped sign or swapped axes fail here
    G = oracle_mod.c2c(f, +1)
    assert np.abs(G - np.exp(+2j * np.pi * phase) / f.size).max() <= 1e-15


def test_single_mode_is_one_spike(oracle_mod):
    shape = (8, 12, 6)
    k0 = (3, 7, 5)
    j = np.meshgrid(*[np.arange(n) for n in shape], indexing="ij")
    f = np.exp(2j * np.pi * sum(j[d] * k0[d] / shape[d] for d in range(3)))
    F = oracle_mod.c2c(f, -1)
    assert abs(F[k0] - f.size) <= 1e-10
    F[k0] = 0
    assert np.abs(F).max() <= 1e-10


def test_round_trip_parseval_linearity(oracle_mod):
    shape = (12, 8, 10)
    f, g = rnd(shape, 2), rnd(shape, 3)
    F, G = oracle_mod.c2c(f, -1), oracle_mod.c2c(g, -1)
    assert np.abs(oracle_mod.c2c(F, +1) - f).max() <= 1e-13
    assert abs((np.abs(F) ** 2).sum() / f.size - (np.abs(f) ** 2).sum()) <= 1e-10 * (np.abs(f) ** 2).sum()
    a, b = 0.3 - 1.1j, 2.0 + 0.5j
    assert np.abs(oracle_mod.c2c(a * f + b * g, -1) - (a * F + b * G)).max() <= 1e-11


@pytest.mark.parametrize("shape", [(16, 16, 16), (12, 20, 18), (32, 24, 48)])
def test_numpy_cross_check(oracle_mod, shape):
    f = rnd(shape, 4)
    F = oracle_mod.c2c(f, -1)
    ref = np.fft.fftn(f)
    assert np.abs(F - ref).max() <= 1e-12 * np.abs(ref).max()
    b = oracle_mod.c2c(f, +1)
    ref = np.fft.ifftn(f)
    assert np.abs(b - ref).max() <= 1e-12 * np.abs(ref).max()


def test_agrees_with_r2c_oracle_and_eq3(oracle_mod):
    """Real input: kz <= Nz/2 is the R2C half spectrum (Eq. (4)), the rest is its Hermitian
    image (Eq. (3))."""
    shape = (8, 12, 10)
    g = np.random.Generator(np.random.PCG64(5))
    f = g.standard_normal(shape)
    F = oracle_mod.c2c(f.astype(np.complex128), -1)
    H = oracle_mod.r2c(f)
    Nz = shape[2]
    assert np.abs(F[:, :, : Nz // 2 + 1] - H).max() <= 1e-12
    for kz in range(Nz // 2 + 1, Nz):
        mirror = np.conj(H[(-np.arange(shape[0])) % shape[0]][:, (-np.arange(shape[1])) % shape[1], Nz - kz])
        assert np.abs(F[:, :, kz] - mirror).max() <= 1e-12
