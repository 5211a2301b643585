"""Pins for the fp64 CPU oracle (CPU only; `-m "not gpu"`).

The oracle is checked against what the paper and the mathematics fix, not against
itself: the O(N^6) definition (Eq. (1),(2),(3)), closed-form spectra
(delta, shifted delta, single cosine, the paper's worked example Eq. (5)),
Parseval, Hermitian symmetry (Eq. (3)), separable products, round trips, numpy.fft as a
library cross-check, and the paper's data-movement steps 2-4 executed literally.
"""
import math
import os

import numpy as np
import pytest

GOLDEN = os.path.join(os.path.dirname(__file__), "golden")


def rng_grid(shape, seed):
    return np.random.Generator(np.random.PCG64(seed)).uniform(-1.0, 1.0, size=shape)


# ---------------------------------------------------------------- 1D building block
@pytest.mark.parametrize("n", [1, 2, 3, 4, 5, 6, 7, 8, 9, 12, 16, 30, 49, 64, 96, 243, 1024, 1536])
@pytest.mark.parametrize("sign", [-1, +1])
def test_fft1d_matches_library(oracle_mod, n, sign):
    g = np.random.Generator(np.random.PCG64(n))
    x = g.standard_normal(n) + 1j * g.standard_normal(n)
    got = oracle_mod.fft1d(x, sign)
    ref = np.fft.fft(x) if sign < 0 else np.fft.ifft(x) * n
    assert np.linalg.norm(got - ref) <= 1e-13 * max(1.0, np.linalg.norm(ref)) * max(1, math.log2(n + 1))


def test_fft1d_shifted_delta_has_the_forward_sign(oracle_mod):
    # x = delta at j0 -> X[k] = exp(-2 pi i k j0 / n) for sign=-1 (Eq. (1) convention)
    n, j0 = 12, 5
    x = np.zeros(n, dtype=complex)
    x[j0] = 1.0
    k = np.arange(n)
    assert np.allclose(oracle_mod.fft1d(x, -1), np.exp(-2j * np.pi * k * j0 / n), atol=1e-15)
    assert np.allclose(oracle_mod.fft1d(x, +1), np.exp(+2j * np.pi * k * j0 / n), atol=1e-15)


# ---------------------------------------------------------------- the O(N^6) definition
def test_direct_dft_closed_forms(oracle_mod):
    shape = (4, 6, 8)
    f = np.zeros(shape)
    f[0, 0, 0] = 1.0
    F = oracle_mod.dft3d_direct(f)
    assert F.shape == (4, 6, 5)
    assert np.allclose(F, 1.0, atol=1e-15)                     # delta -> constant spectrum 1
    j0 = (1, 4, 3)
    f = np.zeros(shape)
    f[j0] = 2.5
    F = oracle_mod.dft3d_direct(f)
    kx, ky, kz = np.meshgrid(np.arange(4), np.arange(6), np.arange(5), indexing="ij")
    expect = 2.5 * np.exp(-2j * np.pi * (kx * j0[0] / 4 + ky * j0[1] / 6 + kz * j0[2] / 8))
    assert np.allclose(F, expect, atol=1e-14)                  # a flipped sign or swapped axis fails here


@pytest.mark.parametrize("shape", [(8, 8, 8), (12, 12, 12), (8, 12, 6)])
def test_fast_r2c_equals_direct_definition(oracle_mod, shape):
    f = rng_grid(shape, 1)
    Fd = oracle_mod.dft3d_direct(f)
    Ff = oracle_mod.r2c(f)
    assert np.abs(Ff - Fd).max() <= 1e-12
    # library cross-check of the definition itself
    assert np.abs(Fd - np.fft.rfftn(f)).max() <= 1e-12


@pytest.mark.parametrize("shape", [(8, 8, 8), (12, 12, 12), (8, 12, 6)])
def test_fast_c2r_equals_direct_definition_even_for_inconsistent_planes(oracle_mod, shape):
    # a random half spectrum is NOT Hermitian-consistent on kz=0 / kz=Nz/2: DESIGN.md reading R8
    g = np.random.Generator(np.random.PCG64(7))
    Nx, Ny, Nz = shape
    F = g.standard_normal((Nx, Ny, Nz // 2 + 1)) + 1j * g.standard_normal((Nx, Ny, Nz // 2 + 1))
    fd = oracle_mod.idft3d_direct(F, Nz)
    ff = oracle_mod.c2r(F, Nz)
    assert np.abs(ff - fd).max() <= 1e-13
    # sampled inverse in natural layout (p=1) and in the slab layout (p=2)
    pts = [(0, 0, 0), (1, 2, 3), (Nx - 1, Ny - 1, Nz - 1), (3, 5, 4)]
    jx, jy, jz = zip(*pts)
    for p in (1, 2):
        flat = oracle_mod.natural_to_slab(F, p)
        got = oracle_mod.c2r_points(flat, shape, p, jx, jy, jz)
        assert np.abs(got - np.array([fd[q] for q in pts])).max() <= 1e-13
    got32 = oracle_mod.c2r_points(oracle_mod.natural_to_slab(F, 2).astype(np.complex64), shape, 2, jx, jy, jz)
    assert np.abs(got32 - np.array([fd[q] for q in pts])).max() <= 1e-6


def test_inverse_is_scaled_by_one_over_n(oracle_mod):
    # DC-only spectrum F(0,0,0) = NxNyNz  ->  f == 1 everywhere (1/(NxNyNz) scale; BASELINE.json)
    shape = (6, 4, 10)
    F = np.zeros((6, 4, 6), dtype=complex)
    F[0, 0, 0] = 6 * 4 * 10
    assert np.allclose(oracle_mod.c2r(F, 10), 1.0, atol=1e-15)
    assert np.allclose(oracle_mod.idft3d_direct(F, 10), 1.0, atol=1e-15)


# ---------------------------------------------------------------- closed forms at FFT sizes
def test_single_cosine_gives_two_spikes(oracle_mod):
    N = 16
    k0 = (3, 14, 5)                                   # ky = 14 = -2 mod 16
    j = np.arange(N)
    jx, jy, jz = np.meshgrid(j, j, j, indexing="ij")
    f = np.cos(2 * np.pi * (k0[0] * jx + k0[1] * jy + k0[2] * jz) / N)
    F = oracle_mod.r2c(f)
    expect = np.zeros_like(F)
    expect[k0] = N ** 3 / 2                           # +k0 is in the stored half (kz=5 <= 8)
    # -k0 = (13, 2, 11) has kz = 11 > N/2: outside the stored half
    assert np.abs(F - expect).max() <= 1e-10
    # a mode on the kz = 0 plane shows both spikes
    f = np.cos(2 * np.pi * (3 * jx + 2 * jy) / N)
    F = oracle_mod.r2c(f)
    expect = np.zeros_like(F)
    expect[3, 2, 0] = N ** 3 / 2
    expect[13, 14, 0] = N ** 3 / 2
    assert np.abs(F - expect).max() <= 1e-10


def load_eq5_spikes():
    rows = []
    with open(os.path.join(GOLDEN, "eq5_spikes.txt")) as fh:
        for line in fh:
            line = line.strip()
            if not line or line.startswith("#"):
                continue
            kx, ky, kz, re, im = line.split()
            rows.append((int(kx), int(ky), int(kz), float(re), float(im)))
    assert len(rows) == 8
    return rows


def eq5_field(N):
    x = 2 * np.pi * np.arange(N) / N
    X, Y, Z = np.meshgrid(x, x, x, indexing="ij")
    return 8 * np.sin(X) * np.sin(2 * Y) * np.sin(3 * Z) + 8 * np.sin(4 * X) * np.sin(5 * Y) * np.sin(6 * Z)


@pytest.mark.parametrize("N", [16, 24, 32])
def test_paper_worked_example_eq5(oracle_mod, N):
    """PAPER.md:100 Eq. (5): exactly 8 non-zero half-spectrum entries, each +-i N^3; the fp64
    round trip recovers the field to ~1e-14."""
    f = eq5_field(N)
    F = oracle_mod.r2c(f)
    expect = np.zeros_like(F)
    for kx, ky, kz, re, im in load_eq5_spikes():
        expect[kx % N, ky % N, kz] = (re + 1j * im) * N ** 3
    assert np.abs(F - expect).max() <= 1e-12 * N ** 3
    back = oracle_mod.c2r(F, N)
    assert np.abs(back - f).max() <= 2e-14 * 16           # amplitude <= 16
    # inverse of the exact spikes returns Eq. (5)
    assert np.abs(oracle_mod.c2r(expect, N) - f).max() <= 1e-13


def test_separable_product_closed_form(oracle_mod):
    # f = a(x) b(y) c(z)  =>  F = A(kx) B(ky) C(kz), each 1D DFT summed directly here
    shape = (12, 16, 24)
    g = np.random.Generator(np.random.PCG64(3))
    a, b, c = (g.standard_normal(n) for n in shape)

    def dft(v):
        n = len(v)
        k = np.arange(n)
        return np.array([np.sum(v * np.exp(-2j * np.pi * k * kk / n)) for kk in range(n)])

    f = a[:, None, None] * b[None, :, None] * c[None, None, :]
    expect = dft(a)[:, None, None] * dft(b)[None, :, None] * dft(c)[None, None, : shape[2] // 2 + 1]
    assert np.abs(oracle_mod.r2c(f) - expect).max() <= 1e-11


# ---------------------------------------------------------------- invariants
@pytest.mark.parametrize("shape", [(16, 16, 16), (12, 24, 18), (32, 8, 64)])
def test_parseval_hermitian_roundtrip(oracle_mod, shape):
    Nx, Ny, Nz = shape
    f = rng_grid(shape, 11)
    F = oracle_mod.r2c(f)
    w = np.full(Nz // 2 + 1, 2.0)
    w[0] = 1.0
    w[Nz // 2] = 1.0
    lhs = np.sum(f * f)
    rhs = np.sum(w[None, None, :] * np.abs(F) ** 2) / (Nx * Ny * Nz)
    assert abs(lhs - rhs) <= 1e-12 * lhs
    # Eq. (3) on the two self-conjugate planes
    for kz in (0, Nz // 2):
        P = F[:, :, kz]
        M = np.conj(P[(-np.arange(Nx)) % Nx][:, (-np.arange(Ny)) % Ny])
        assert np.abs(P - M).max() <= 1e-11
    assert abs(F[0, 0, 0] - f.sum()) <= 1e-11                # DC entry = sum f
    assert np.abs(oracle_mod.c2r(F, Nz) - f).max() <= 1e-14 * math.log2(Nx * Ny * Nz) * 4


@pytest.mark.parametrize("shape", [(64, 64, 64), (48, 32, 96)])
def test_library_cross_check(oracle_mod, shape):
    f = rng_grid(shape, 5)
    F = oracle_mod.r2c(f)
    ref = np.fft.rfftn(f)
    assert np.linalg.norm(F - ref) <= 1e-13 * np.linalg.norm(ref)
    S = ref + 0.0
    back = oracle_mod.c2r(S, shape[2])
    assert np.abs(back - np.fft.irfftn(S, s=shape, axes=(0, 1, 2))).max() <= 1e-13
    # threads do not change the answer
    assert np.array_equal(oracle_mod.r2c(f, nthreads=1), F)


def test_pencil_oracle_matches_full_transform(oracle_mod):
    shape = (16, 12, 20)
    f = rng_grid(shape, 21)
    F = oracle_mod.r2c(f)
    kys = [0, 3, 11, 6]
    kzs = [0, 10, 4, 7]
    got = oracle_mod.r2c_pencils(f, kys, kzs)
    for c, (ky, kz) in enumerate(zip(kys, kzs)):
        assert np.abs(got[c] - F[:, ky, kz]).max() <= 1e-12
    got32 = oracle_mod.r2c_pencils(f.astype(np.float32), kys, kzs)
    F32 = oracle_mod.r2c(f.astype(np.float32).astype(np.float64))
    for c, (ky, kz) in enumerate(zip(kys, kzs)):
        assert np.abs(got32[c] - F32[:, ky, kz]).max() <= 1e-11


# ---------------------------------------------------------------- the slab permutation
@pytest.mark.parametrize("shape", [(8, 8, 8), (8, 16, 6), (16, 8, 10)])
@pytest.mark.parametrize("p", [1, 2, 4, 8])
def test_paper_steps_2_to_4_compose_to_slab_index(oracle_mod, shape, p):
    Nx, Ny, Nz = shape
    Nzh = Nz // 2 + 1
    # every element carries its own natural (kx,ky,kz) identity
    D2 = np.arange(Nx * Ny * Nzh, dtype=np.float64).reshape(Nx, Ny, Nzh)
    sim = oracle_mod.simulate_paper_steps_2_to_4(D2, p)
    assert np.array_equal(sim, oracle_mod.natural_to_slab(D2, p))
    kx, ky, kz = np.meshgrid(np.arange(Nx), np.arange(Ny), np.arange(Nzh), indexing="ij")
    off = oracle_mod.slab_index(p, Nx, Ny, Nz, kx, ky, kz)
    assert sorted(off.ravel().tolist()) == list(range(Nx * Ny * Nzh))       # a bijection
    assert np.array_equal(sim[off], D2)
    assert np.array_equal(oracle_mod.slab_to_natural(sim, shape, p), D2)
    # x-stride of step 5: Ny/p * (Nz/2+1)
    if Nx > 1:
        assert off[1, 0, 0] - off[0, 0, 0] == (Ny // p) * Nzh


# ---------------------------------------------------------------- the pencil layout (reading R17)
@pytest.mark.parametrize("shape", [(8, 8, 8), (8, 16, 12), (16, 8, 16)])
@pytest.mark.parametrize("px,py", [(1, 1), (2, 1), (1, 2), (2, 2), (4, 2), (2, 4), (8, 2)])
def test_pencil_transposes_compose_to_pencil_index(oracle_mod, shape, px, py):
    Nx, Ny, Nz = shape
    Nzh = Nz // 2 + 1
    if Nx % px or Ny % px or Ny % py or (Nz // 2) % py:
        pytest.skip("extents not divisible by the rank grid")
    D1 = np.arange(Nx * Ny * Nzh, dtype=np.float64).reshape(Nx, Ny, Nzh)     # every element carries its identity
    sim = oracle_mod.simulate_pencil_transposes(D1, px, py)
    kx, ky, kz = np.meshgrid(np.arange(Nx), np.arange(Ny), np.arange(Nzh), indexing="ij")
    off = oracle_mod.pencil_index(px, py, Nx, Ny, Nz, kx, ky, kz)
    assert sorted(off.ravel().tolist()) == list(range(Nx * Ny * Nzh))       # a bijection
    assert np.array_equal(sim[off], D1)
    assert np.array_equal(sim, oracle_mod.natural_to_pencil(D1, px, py))
    assert np.array_equal(oracle_mod.pencil_to_natural(sim, shape, px, py), D1)
    # py = 1 is the slab layout with p = px (the paper's own decomposition)
    if py == 1:
        assert np.array_equal(off, oracle_mod.slab_index(px, Nx, Ny, Nz, kx, ky, kz))
    # inside a rank x is the slowest index with stride (Ny/px) * cz_b, y next with stride cz_b
    cz0 = int(oracle_mod.pencil_cz(py, Nz, 0))
    assert off[1, 0, 0] - off[0, 0, 0] == (Ny // px) * cz0
    if Ny // px > 1:
        assert off[0, 1, 0] - off[0, 0, 0] == cz0
    # the last rank column also holds the Nyquist column
    assert int(oracle_mod.pencil_cz(py, Nz, py - 1)) == (Nz // 2) // py + 1
