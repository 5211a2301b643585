"""BASELINE.json configs[2] as it is written: "random-phase Fourier modes with |u(k)|^2 ~ k^-5/3 for 1 <= |k| <= N/3,
transformed to physical space by the oracle's recipe from seed".

Test-side helper (it calls the oracle, which the product package may not do; paper_2202_12756_b200/inputs.py therefore
carries a 128-mode stand-in for the bench, reading R16).  EVERY integer wavevector of the shell gets a mode:
amplitude |k|^(-5/6), phase uniform in [0, 2 pi) from a PCG64 stream of the seed, Hermitian-consistent on the plane
kz = 0 (the plane kz = N/2 lies outside the shell); the half spectrum goes through oracle.c2r (Eq. (2)+(3))
and the field is scaled to unit rms.  Returns (field fp64 (N,N,N), half spectrum of that field, complex128 (N,N,N/2+1))."""
import numpy as np


def literal_config2_field(N: int, seed: int, oracle_mod):
    kmax = N // 3
    k1 = np.fft.fftfreq(N, 1.0 / N).astype(np.int64)                 # 0, 1, ..., N/2-1, -N/2, ..., -1
    kx = k1[:, None, None]
    ky = k1[None, :, None]
    kz = np.arange(N // 2 + 1, dtype=np.int64)[None, None, :]
    k2 = kx * kx + ky * ky + kz * kz
    shell = (k2 >= 1) & (k2 <= kmax * kmax)
    rng = np.random.Generator(np.random.PCG64(seed))
    phase = rng.uniform(0.0, 2.0 * np.pi, size=shell.shape)
    amp = np.zeros(shell.shape)
    amp[shell] = k2[shell].astype(np.float64) ** (-5.0 / 12.0)       # |u|^2 ~ |k|^(-5/3)
    S = amp * np.exp(1j * phase)
    # plane kz = 0: u(-kx, -ky, 0) = conj u(kx, ky, 0); the half with kx > 0 (or kx = 0, ky > 0) decides
    P = S[:, :, 0]
    mirror = np.conj(P[(-np.arange(N)) % N][:, (-np.arange(N)) % N])
    upper = (k1[:, None] > 0) | ((k1[:, None] == 0) & (k1[None, :] > 0))
    S[:, :, 0] = np.where(upper, P, mirror)
    field = oracle_mod.c2r(np.ascontiguousarray(S), N)
    scale = 1.0 / np.sqrt(np.mean(field * field))
    return field * scale, S * scale            # r2c(c2r(S)) = S: the inverse carries the 1/N^3
