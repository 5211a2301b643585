"""Seeded input generators: determinism, distributions, and closed-form content (CPU)."""
import math

import numpy as np
import torch

from paper_2202_12756_b200 import inputs


def test_uniform_is_deterministic_and_in_range():
    a = inputs.uniform_grid((8, 6, 10), torch.float64, seed=0)
    b = inputs.uniform_grid((8, 6, 10), torch.float64, seed=0)
    c = inputs.uniform_grid((8, 6, 10), torch.float64, seed=1)
    assert torch.equal(a, b) and not torch.equal(a, c)
    big = inputs.uniform_grid((64, 64, 64), torch.float64, seed=0)
    assert -1.0 <= big.min().item() and big.max().item() < 1.0
    assert abs(big.mean().item()) < 0.01 and abs(big.var().item() - 1.0 / 3.0) < 0.01
    # chunking does not change values
    flat = inputs._fill((1000,), torch.float64, "cpu",
                        lambda a_, b_: 2.0 * inputs._uniform01(a_, b_, 0, 0, "cpu") - 1.0, chunk=97)
    assert torch.equal(flat, inputs.uniform_grid((1000,), torch.float64, seed=0))


def test_normal_moments():
    g = inputs.normal_grid((64, 64, 64), torch.float64, seed=3)
    assert abs(g.mean().item()) < 0.01 and abs(g.std().item() - 1.0) < 0.01


def test_mode_sum_matches_pointwise_formula():
    shape = (12, 10, 16)
    g, modes = inputs.sinusoid_grid(shape, torch.float64, seed=4, n_modes=5, kmax=4, noise_var=0.0)
    jx, jy, jz = np.meshgrid(*(np.arange(n) for n in shape), indexing="ij")
    ref = np.zeros(shape)
    for (kx, ky, kz), amp, phi in modes:
        ref += amp * np.cos(2 * np.pi * (kx * jx / shape[0] + ky * jy / shape[1] + kz * jz / shape[2]) + phi)
    assert np.abs(g.numpy() - ref).max() < 1e-12


def test_turbulence_grid_unit_rms_and_shell():
    g, modes = inputs.turbulence_grid((48, 48, 48), torch.float64, seed=0, n_modes=32)
    assert abs(g.pow(2).mean().sqrt().item() - 1.0) < 1e-9
    for (kx, ky, kz), amp, _ in modes:
        k2 = kx * kx + ky * ky + kz * kz
        assert 1 <= k2 <= 16 * 16 and kz >= 0 and amp > 0
    assert len({m[0] for m in modes}) == len(modes)


def test_eq5_grid_formula():
    N = 16
    g = inputs.eq5_grid((N, N, N))
    x = 2 * np.pi * np.arange(N) / N
    X, Y, Z = np.meshgrid(x, x, x, indexing="ij")
    ref = 8 * np.sin(X) * np.sin(2 * Y) * np.sin(3 * Z) + 8 * np.sin(4 * X) * np.sin(5 * Y) * np.sin(6 * Z)
    assert np.abs(g.numpy() - ref).max() < 1e-13


def test_random_spectrum_shape_and_determinism():
    s = inputs.random_spectrum((8, 6, 10), torch.complex64, seed=2)
    assert s.shape == (8, 6, 6) and s.dtype == torch.complex64
    assert torch.equal(s, inputs.random_spectrum((8, 6, 10), torch.complex64, seed=2))
