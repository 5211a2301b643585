"""Slab layout of the Fourier-space array -- TEST INFRASTRUCTURE, NOT THE PRODUCT.

The paper never writes the final layout as a formula (reading R5).  This file
holds (a) ``simulate_paper_steps_2_to_4``: the paper's data movement executed literally,
rank by rank, chunk by chunk (steps 2-4; Fig. 1(c)-(f) caption,
PAPER.md:94), and (b) ``slab_index``: the closed form it composes to,

    offset(kx,ky,kz) = ((q*Nx + kx)*(Ny/p) + ky_l)*Nzh + kz,   q = ky // (Ny/p), ky_l = ky % (Ny/p)

i.e. rank q ends up holding [Nx][Ny/p][Nzh] (x stride Ny/p * Nzh) and the
ranks are concatenated.  tests/test_oracle_pins.py checks (a) == (b) for p in {1,2,4,8}.
"""
from __future__ import annotations

import numpy as np


def slab_index(p: int, Nx: int, Ny: int, Nz: int, kx, ky, kz):
    """Element offset of F(kx,ky,kz) in the slab-layout output (works on arrays)."""
    L = Ny // p
    Nzh = Nz // 2 + 1
    kx = np.asarray(kx, dtype=np.int64)
    ky = np.asarray(ky, dtype=np.int64)
    kz = np.asarray(kz, dtype=np.int64)
    q = ky // L
    return ((q * Nx + kx) * L + (ky % L)) * Nzh + kz


def natural_to_slab(F_nat: np.ndarray, p: int) -> np.ndarray:
    """[Nx][Ny][Nzh] -> flat array in slab layout [p][Nx][Ny/p][Nzh]."""
    Nx, Ny, Nzh = F_nat.shape
    L = Ny // p
    return np.ascontiguousarray(F_nat.reshape(Nx, p, L, Nzh).transpose(1, 0, 2, 3)).reshape(-1)


def slab_to_natural(F_slab: np.ndarray, shape, p: int) -> np.ndarray:
    """Flat slab-layout array -> [Nx][Ny][Nzh]."""
    Nx, Ny, Nz = shape
    Nzh = Nz // 2 + 1
    L = Ny // p
    return np.ascontiguousarray(
        np.asarray(F_slab).reshape(p, Nx, L, Nzh).transpose(1, 0, 2, 3)).reshape(Nx, Ny, Nzh)


def simulate_paper_steps_2_to_4(D2_nat: np.ndarray, p: int) -> np.ndarray:
    """Run steps 2, 3, 4 of PAPER.md:70-76 on p simulated ranks with explicit loops.

    D2_nat is the array after step 1 in natural order [Nx][Ny][Nzh]; rank r holds the
    x-slab D2_nat[r*Nx/p:(r+1)*Nx/p].  Returns the concatenation over
    ranks of what each rank holds after step 4, flattened.
    """
    Nx, Ny, Nzh = D2_nat.shape
    assert Nx % p == 0 and Ny % p == 0
    Xl, L = Nx // p, Ny // p
    # step 2: local xy transpose, [Nx/p][Ny][Nzh] -> [Ny][Nx/p][Nzh]
    after2 = []
    for r in range(p):
        slab = D2_nat[r * Xl:(r + 1) * Xl]
        t = np.empty((Ny, Xl, Nzh), dtype=D2_nat.dtype)
        for xl in range(Xl):
            for y in range(Ny):
                t[y, xl, :] = slab[xl, y, :]
        after2.append(t)
    # step 3: all-to-all.  Rank r's send buffer is p chunks of
    # [Ny/p][Nx/p][Nzh]; chunk q goes to rank q; received chunks land in source-rank
    # order; the inside of a chunk is not touched ("remains unchanged").
    after3 = [np.empty((p, L, Xl, Nzh), dtype=D2_nat.dtype) for _ in range(p)]
    for r in range(p):                    # sender
        for q in range(p):                # receiver
            chunk = after2[r][q * L:(q + 1) * L]          # [Ny/p][Nx/p][Nzh], contiguous
            after3[q][r] = chunk
    # step 4: local xy transpose of every chunk, [Ny/p][Nx/p] -> [Nx/p][Ny/p]
    out = []
    for q in range(p):
        final = np.empty((p, Xl, L, Nzh), dtype=D2_nat.dtype)
        for r in range(p):
            for yl in range(L):
                for xl in range(Xl):
                    final[r, xl, yl, :] = after3[q][r, yl, xl, :]
        # [p][Nx/p][Ny/p][Nzh] read as [Nx][Ny/p][Nzh]: x = r*Nx/p + xl is now contiguous
        # in the slowest index, with stride Ny/p*Nzh -- the stride of step 5
        out.append(final.reshape(-1))
    return np.concatenate(out)
