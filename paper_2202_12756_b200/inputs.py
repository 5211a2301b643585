"""Seeded synthetic inputs shared by the tests, bench.py and smoke().

This module holds NONE of the method's arithmetic (no FFT, no DFT, no call into the
CUDA library or into oracle/): it only fills real grids and half spectra with seeded
values whose recipe is stated in DESIGN.md section 4.  Arrays are produced once and the
SAME array feeds both the CUDA path and the oracle (fp32 grids are rounded once; the
oracle promotes those fp32 values to fp64).

Generators work on any torch device: values come from a counter-based integer hash of
(seed, linear index) evaluated with wrap-around int64 arithmetic, so a grid generated on
``cuda`` and one generated on ``cpu`` hold the same uniform numbers.
"""
from __future__ import annotations

import math

import numpy as np
import torch

_M64 = (1 << 64) - 1


def _to_i64(u: int) -> int:
    u &= _M64
    return u - (1 << 64) if u >= (1 << 63) else u


_C1 = _to_i64(0xBF58476D1CE4E5B9)
_C2 = _to_i64(0x94D049BB133111EB)
_GOLD = 0x9E3779B97F4A7C15


def _lsr(x: torch.Tensor, s: int) -> torch.Tensor:
    """Logical shift right on int64 (torch's >> is arithmetic)."""
    return (x >> s) & ((1 << (64 - s)) - 1)


def _hash_u53(idx: torch.Tensor, seed: int, stream: int) -> torch.Tensor:
    """splitmix64 finaliser of (index, seed, stream) -> integers in [0, 2^53)."""
    x = idx + _to_i64((seed * 2 + 1) * _GOLD + stream * 0xD1B54A32D192ED03)
    x = (x ^ _lsr(x, 30)) * _C1
    x = (x ^ _lsr(x, 27)) * _C2
    x = x ^ _lsr(x, 31)
    return _lsr(x, 11)


def _uniform01(n0: int, n1: int, seed: int, stream: int, device) -> torch.Tensor:
    """fp64 uniform [0,1) for linear indices n0..n1-1."""
    idx = torch.arange(n0, n1, dtype=torch.int64, device=device)
    return _hash_u53(idx, seed, stream).to(torch.float64) * (1.0 / (1 << 53))


def _fill(shape, dtype, device, fn, chunk=1 << 24, x_range=None) -> torch.Tensor:
    """fn(a, b) = values for linear indices a..b-1 of the whole grid; x_range = (x0, x1) fills only the x-slab
    [x0, x1) of it (a rank's slab of a distributed field: the same values as in the whole grid)."""
    if x_range is not None:
        plane = int(np.prod(shape[1:]))
        shape = (x_range[1] - x_range[0],) + tuple(shape[1:])
        base = x_range[0] * plane
    else:
        base = 0
    n = int(np.prod(shape))
    out = torch.empty(n, dtype=dtype, device=device)
    for a in range(0, n, chunk):
        b = min(n, a + chunk)
        out[a:b] = fn(base + a, base + b).to(dtype)
    return out.reshape(shape)


def uniform_grid(shape, dtype=torch.float64, seed=0, device="cpu", x_range=None) -> torch.Tensor:
    """i.i.d. uniform[-1,1) (BASELINE.json configs[0] and configs[4])."""
    return _fill(shape, dtype, device, lambda a, b: 2.0 * _uniform01(a, b, seed, 0, device) - 1.0, x_range=x_range)


def _normal(a, b, seed, stream, device):
    u1 = _uniform01(a, b, seed, stream, device)
    u2 = _uniform01(a, b, seed, stream + 1, device)
    return torch.sqrt(-2.0 * torch.log1p(-u1)) * torch.cos(2.0 * math.pi * u2)


def normal_grid(shape, dtype=torch.float32, seed=0, device="cpu", sigma=1.0, x_range=None) -> torch.Tensor:
    """i.i.d. N(0, sigma^2) by Box-Muller on the hash uniforms (configs[3])."""
    return _fill(shape, dtype, device, lambda a, b: sigma * _normal(a, b, seed, 2, device), x_range=x_range)


def _mode_sum(shape, modes, dtype, device, xchunk=32, x_range=None) -> torch.Tensor:
    """f(j) = sum_m A_m cos(2 pi (kx jx/Nx + ky jy/Ny + kz jz/Nz) + phi_m), evaluated in
    fp64 as Re sum_m A_m e^{i phi_m} X_m[jx] Y_m[jy] Z_m[jz] (plain products, no transform)."""
    Nx, Ny, Nz = shape
    k = torch.tensor([m[0] for m in modes], dtype=torch.float64, device=device)   # (M,3)
    amp = torch.tensor([m[1] for m in modes], dtype=torch.float64, device=device)
    phi = torch.tensor([m[2] for m in modes], dtype=torch.float64, device=device)

    def phase(n, kcol):
        j = torch.arange(n, dtype=torch.float64, device=device)
        # reduce k*j mod n in integers first so the angle stays small
        kj = torch.remainder(kcol[:, None].to(torch.int64) * j[None, :].to(torch.int64), n)
        ang = 2.0 * math.pi * kj.to(torch.float64) / n
        return torch.complex(torch.cos(ang), torch.sin(ang))                      # (M,n)

    X, Y, Z = phase(Nx, k[:, 0]), phase(Ny, k[:, 1]), phase(Nz, k[:, 2])
    coef = torch.complex(amp * torch.cos(phi), amp * torch.sin(phi))
    YZ = (Y[:, :, None] * Z[:, None, :]).reshape(len(modes), Ny * Nz)              # (M,Ny*Nz)
    x0, x1 = x_range if x_range is not None else (0, Nx)
    out = torch.empty((x1 - x0, Ny * Nz), dtype=dtype, device=device)
    for a in range(x0, x1, xchunk):
        b = min(x1, a + xchunk)
        XA = (coef[:, None] * X[:, a:b]).transpose(0, 1)                           # (xc,M)
        # real part of a complex product-sum, written with real tensors
        re = XA.real.contiguous() @ YZ.real.contiguous() - XA.imag.contiguous() @ YZ.imag.contiguous()
        out[a - x0:b - x0] = re.to(dtype)
    return out.reshape(x1 - x0, Ny, Nz)


def sinusoid_grid(shape, dtype=torch.float32, seed=0, device="cpu", n_modes=16, kmax=20,
                  noise_var=0.01):
    """configs[1]: n_modes sinusoids with integer wavevector components in [-kmax,kmax],
    amplitudes N(0,1), phases uniform[0,2pi), plus N(0, noise_var) noise.
    Returns (grid, modes) with modes = [((kx,ky,kz), A, phi), ...]."""
    rng = np.random.Generator(np.random.PCG64(seed))
    modes = []
    for _ in range(n_modes):
        kv = tuple(int(v) for v in rng.integers(-kmax, kmax + 1, size=3))
        modes.append((kv, float(rng.standard_normal()), float(rng.uniform(0.0, 2.0 * math.pi))))
    g = _mode_sum(shape, modes, torch.float64, device)
    if noise_var > 0:
        g = g + normal_grid(shape, torch.float64, seed + 1000, device, sigma=math.sqrt(noise_var))
    return g.to(dtype), modes


def turbulence_grid(shape, dtype=torch.float32, seed=0, device="cpu", n_modes=128, kmax=None, x_range=None):
    """configs[2] stand-in (reading R16): a turbulence-like field built directly in
    physical space as n_modes random-phase Fourier modes, wavevectors drawn uniformly from the
    integer lattice shell 1 <= |k| <= kmax (kmax = N//3 = 341 at 1024^3) with kz >= 0, distinct
    up to sign, amplitudes A_m^2 proportional to |k|^(-5/3), scaled to unit rms.
    Returns (grid, modes)."""
    Nmin = min(shape)
    if kmax is None:
        kmax = max(1, Nmin // 3)
    rng = np.random.Generator(np.random.PCG64(seed))
    seen, modes = set(), []
    while len(modes) < n_modes:
        kv = [int(v) for v in rng.integers(-kmax, kmax + 1, size=3)]
        kv[2] = abs(kv[2])
        k2 = kv[0] ** 2 + kv[1] ** 2 + kv[2] ** 2
        if k2 < 1 or k2 > kmax * kmax:
            continue
        key = tuple(kv)
        neg = tuple(-v for v in kv)
        if key in seen or neg in seen:
            continue
        seen.add(key)
        amp = math.sqrt(k2) ** (-5.0 / 6.0)          # A^2 ~ |k|^(-5/3)
        modes.append((key, amp, float(rng.uniform(0.0, 2.0 * math.pi))))
        if len(seen) >= (2 * kmax + 1) ** 2 * (kmax + 1) // 2:
            break
    ms = sum(a * a for _, a, _ in modes) / 2.0        # mean square of a sum of distinct cosines
    s = 1.0 / math.sqrt(ms)
    modes = [(k, a * s, ph) for k, a, ph in modes]
    return _mode_sum(shape, modes, dtype, device, x_range=x_range), modes


def eq5_grid(shape, dtype=torch.float64, device="cpu") -> torch.Tensor:
    """The paper's own workload, Eq. (5), on x_j = 2 pi j / N:
    f = 8 sin x sin 2y sin 3z + 8 sin 4x sin 5y sin 6z."""
    Nx, Ny, Nz = shape

    def s(n, m):
        j = torch.arange(n, dtype=torch.int64, device=device)
        return torch.sin(2.0 * math.pi * torch.remainder(j * m, n).to(torch.float64) / n)

    a = s(Nx, 1)[:, None, None] * s(Ny, 2)[None, :, None] * s(Nz, 3)[None, None, :]
    b = s(Nx, 4)[:, None, None] * s(Ny, 5)[None, :, None] * s(Nz, 6)[None, None, :]
    return (8.0 * a + 8.0 * b).to(dtype)


def random_spectrum(shape, dtype=torch.complex64, seed=0, device="cpu") -> torch.Tensor:
    """i.i.d. complex half spectrum (Nx,Ny,Nz//2+1), re and im uniform[-1,1).  NOT
    Hermitian-consistent on the kz=0 and kz=Nz/2 planes on purpose (reading R8)."""
    Nx, Ny, Nz = shape
    n = Nx * Ny * (Nz // 2 + 1)
    rdt = torch.float32 if dtype == torch.complex64 else torch.float64
    flat = _fill((n, 2), rdt, device,
                 lambda a, b: 2.0 * _uniform01(a, b, seed, 7, device) - 1.0, chunk=1 << 24)
    return torch.view_as_complex(flat).reshape(Nx, Ny, Nz // 2 + 1)


def complex_grid(shape, dtype=torch.complex64, seed=0, device="cpu") -> torch.Tensor:
    """i.i.d. complex grid (Nx,Ny,Nz), re and im uniform[-1,1): input of the C2C transform."""
    Nx, Ny, Nz = shape
    rdt = torch.float32 if dtype == torch.complex64 else torch.float64
    flat = _fill((Nx * Ny * Nz, 2), rdt, device,
                 lambda a, b: 2.0 * _uniform01(a, b, seed, 9, device) - 1.0, chunk=1 << 24)
    return torch.view_as_complex(flat).reshape(Nx, Ny, Nz)
