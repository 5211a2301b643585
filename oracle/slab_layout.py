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


# ---------------------------------------------------------------------------------------------------
# Pencil decomposition (p = px x py ranks, each holding (Nx/px) x (Ny/py) x Nz real points; the
# paper describes it and refers to Pekurovsky / Chatterjee et al. for the algorithm, it does not build it).
# Reading taken (R17), the standard two-transpose scheme written in the paper's own conventions:
#   rank (a, b), a < px, b < py, starts with the z-pencil  f[x in a][y in b][all z];
#   1. z R2C locally                                          -> [Nx/px][Ny/py][Nzh]
#   2. exchange inside each ROW of the rank grid (fixed a): y is gathered, kz is scattered
#                                                             -> [Nx/px][Ny][cz_b]        then the y transform
#   3. exchange inside each COLUMN of the rank grid (fixed b): x is gathered, ky is scattered, and -- as in the
#      paper's step 4 -- x becomes the slowest index   -> [Nx][Ny/px][cz_b]  then the x transform
# kz = 0..Nz/2 is split into py ranges of Nz/(2 py) columns, the last rank also taking the Nyquist column kz = Nz/2:
# cz_b = Nz/(2 py) for b < py-1 and Nz/(2 py) + 1 for b = py-1.  Ranks are concatenated in row-major order r = a*py + b.
# For py = 1 this is exactly the slab layout with p = px.
# ---------------------------------------------------------------------------------------------------
def pencil_cz(py: int, Nz: int, b):
    """Number of kz columns rank column b holds (works on arrays)."""
    c = (Nz // 2) // py
    return np.where(np.asarray(b) == py - 1, c + 1, c)


def pencil_index(px: int, py: int, Nx: int, Ny: int, Nz: int, kx, ky, kz):
    """Element offset of F(kx,ky,kz) in the pencil-layout output (works on arrays)."""
    L = Ny // px
    c = (Nz // 2) // py
    Nzh = Nz // 2 + 1
    kx = np.asarray(kx, dtype=np.int64)
    ky = np.asarray(ky, dtype=np.int64)
    kz = np.asarray(kz, dtype=np.int64)
    a = ky // L
    b = np.minimum(kz // c, py - 1)
    cz = np.where(b == py - 1, c + 1, c)
    base = a * (Nx * L * Nzh) + b * (Nx * L * c)          # blocks [a][b], block (a, b) holds Nx*L*cz_b elements
    return base + (kx * L + (ky % L)) * cz + (kz - b * c)


def natural_to_pencil(F_nat: np.ndarray, px: int, py: int) -> np.ndarray:
    """[Nx][Ny][Nzh] -> flat array in the pencil layout (by the closed form)."""
    Nx, Ny, Nzh = F_nat.shape
    Nz = 2 * (Nzh - 1)
    kx, ky, kz = np.meshgrid(np.arange(Nx), np.arange(Ny), np.arange(Nzh), indexing="ij")
    out = np.empty(F_nat.size, dtype=F_nat.dtype)
    out[pencil_index(px, py, Nx, Ny, Nz, kx, ky, kz).ravel()] = F_nat.ravel()
    return out


def pencil_to_natural(F_pen: np.ndarray, shape, px: int, py: int) -> np.ndarray:
    Nx, Ny, Nz = shape
    Nzh = Nz // 2 + 1
    kx, ky, kz = np.meshgrid(np.arange(Nx), np.arange(Ny), np.arange(Nzh), indexing="ij")
    return np.asarray(F_pen).reshape(-1)[pencil_index(px, py, Nx, Ny, Nz, kx, ky, kz)]


def simulate_pencil_transposes(D1_nat: np.ndarray, px: int, py: int) -> np.ndarray:
    """The two exchanges of the pencil scheme executed literally, rank by rank, with explicit loops.

    D1_nat: the array after the z transform in natural order [Nx][Ny][Nzh] (only WHERE elements go is simulated, so the
    y and x transforms between the exchanges are left out: they act along axes that are complete on every rank).
    Returns the concatenation, in rank order r = a*py + b, of what each rank holds at the end, flattened.
    """
    Nx, Ny, Nzh = D1_nat.shape
    Nz = 2 * (Nzh - 1)
    assert Nx % px == 0 and Ny % px == 0 and Ny % py == 0 and (Nz // 2) % py == 0
    Xl, Yb, L, c = Nx // px, Ny // py, Ny // px, (Nz // 2) // py
    cz = [c + 1 if b == py - 1 else c for b in range(py)]
    z0 = [b * c for b in range(py)]
    # start: rank (a, b) holds [Nx/px][Ny/py][Nzh]
    start = {(a, b): D1_nat[a * Xl:(a + 1) * Xl, b * Yb:(b + 1) * Yb, :].copy() for a in range(px) for b in range(py)}
    # exchange 1, inside row a: rank (a, b) sends to (a, b2) its columns kz in range b2; the receiver stacks the
    # pieces in source order along y (standard all-to-all): [Nx/px][Ny][cz_b2]
    after1 = {}
    for a in range(px):
        for b2 in range(py):
            buf = np.empty((Xl, Ny, cz[b2]), dtype=D1_nat.dtype)
            for b in range(py):                                   # source, in order
                piece = start[(a, b)][:, :, z0[b2]:z0[b2] + cz[b2]]
                for xl in range(Xl):
                    for yl in range(Yb):
                        buf[xl, b * Yb + yl, :] = piece[xl, yl, :]
            after1[(a, b2)] = buf
    # exchange 2, inside column b: rank (a, b) sends to (a2, b) its rows ky in range a2; the receiver stacks the
    # pieces in source order along x, x slowest (PAPER.md:76-77 for slabs): [Nx][Ny/px][cz_b]
    out = []
    for a2 in range(px):
        for b in range(py):
            buf = np.empty((Nx, L, cz[b]), dtype=D1_nat.dtype)
            for a in range(px):                                   # source, in order
                piece = after1[(a, b)][:, a2 * L:(a2 + 1) * L, :]
                for xl in range(Xl):
                    for yl in range(L):
                        buf[a * Xl + xl, yl, :] = piece[xl, yl, :]
            out.append(buf.reshape(-1))
    return np.concatenate(out)
