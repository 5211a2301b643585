"""The N > 1 plumbing of the slab decomposition on CPU: two real processes, gloo.

paper_2202_12756_b200/dist.py::SlabFFT drives a rank's stages and the exchange between them.  Here its stage
provider is a numpy stand-in (test code: numpy.fft on the rank's data -- a library routine, not the CUDA path and
not the oracle), so that what is under test is the host logic the GPUs cannot check on a one-GPU box: chunk shapes and
order of the all-to-all, the all-gather of the plane parts for the packed column, which rank holds
the partner rows, and the descriptor hand-off of the UNIFIED exchange.  The result must equal the fp64 oracle's 3D
transform of the whole field.
"""
import os
import socket
import sys

import numpy as np
import pytest
import torch
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    port = s.getsockname()[1]
    s.close()
    return port


class NumpyStages:
    """The stage interface of dist.DistPlan on CPU tensors, each stage by its definition with numpy.fft."""

    def __init__(self, Nx, Ny, Nz, G, rank):
        self.shape, self.G, self.rank = (Nx, Ny, Nz), G, rank
        self.Nxl, self.L, self.M = Nx // G, Ny // G, Nz // 2
        self.complex_dtype = torch.complex128
        self.side = None

    def nbytes(self, which):
        raise NotImplementedError

    def empty_work(self, device):
        return torch.empty(1)

    def empty_plane_part(self, device):
        return torch.empty((2, self.shape[0], self.L), dtype=torch.complex128)

    def _pack(self, X):            # [..][M+1] -> [..][M] with (X[0], X[M]) packed in column 0
        P = X[..., : self.M].copy()
        P[..., 0] = X[..., 0] + 1j * X[..., self.M]
        return P

    def fwd_local(self, real_slab, xchg, layout, work):
        assert layout == 1
        Z = np.fft.rfft(real_slab.numpy(), axis=2)                       # step 1, z half: the two end columns are real
        P = Z[..., : self.M].copy()
        P[..., 0] = Z[..., 0].real + 1j * Z[..., self.M].real
        Y = np.fft.fft(P, axis=1)                                        # step 1, y half
        # steps 2-4 as addressing: chunk q = rows ky in [q L, (q+1) L), laid out [x_l][ky_l][kz]
        out = xchg.numpy()
        for q in range(self.G):
            out[q] = Y[:, q * self.L:(q + 1) * self.L, :]

    def fwd_x(self, slab_part, spec_part):
        S = np.asarray(slab_part).reshape(self.shape[0], self.L, self.M)
        X = np.fft.fft(S, axis=0)                                        # step 5
        out = spec_part.numpy()
        out[:, :, : self.M] = X
        out[:, :, self.M] = 0

    def fwd_col0(self, spec_part, plane_part):
        plane_part[0] = spec_part[:, :, 0]

    def _partner(self, planes, c):
        """C(-kx, -ky) for the own rows, from the gathered plane parts."""
        Nx, Ny, L = self.shape[0], self.shape[1], self.L
        full = np.concatenate([np.asarray(planes[q][c]) for q in range(self.G)], axis=1)      # [Nx][Ny]
        kx = (-np.arange(Nx)) % Nx
        ky = (-(self.rank * L + np.arange(L))) % Ny
        return full[np.ix_(kx, ky)]

    def fwd_unpack(self, spec_part, planes):
        c1 = np.asarray(planes[self.rank][0])
        c2 = self._partner(planes, 0)
        out = spec_part.numpy()
        out[:, :, 0] = 0.5 * (c1 + np.conj(c2))
        out[:, :, self.M] = (c1 - np.conj(c2)) / 2j

    def inv_planes(self, spec_part, plane_part):
        plane_part[0] = spec_part[:, :, 0]
        plane_part[1] = spec_part[:, :, self.M]

    def inv_pack(self, planes, work):
        a1, b1 = np.asarray(planes[self.rank][0]), np.asarray(planes[self.rank][1])
        As = 0.5 * (a1 + np.conj(self._partner(planes, 0)))
        Bs = 0.5 * (b1 + np.conj(self._partner(planes, 1)))
        self.side = As + 1j * Bs

    def inv_x(self, spec_part, slab_part, work):
        X = spec_part.numpy()[:, :, : self.M].copy()
        X[:, :, 0] = self.side
        S = np.fft.ifft(X, axis=0) * self.shape[0]
        np.asarray(slab_part).reshape(self.shape[0], self.L, self.M)[...] = S

    def inv_local(self, xchg, layout, real_slab, work):
        assert layout == 1
        Y = np.concatenate([xchg.numpy()[q] for q in range(self.G)], axis=1)                  # [Nxl][Ny][M]
        P = np.fft.ifft(Y, axis=1) * self.shape[1]
        Z = np.zeros(P.shape[:2] + (self.M + 1,), dtype=np.complex128)
        Z[..., : self.M] = P
        Z[..., 0] = P[..., 0].real
        Z[..., self.M] = P[..., 0].imag
        real_slab.numpy()[...] = np.fft.irfft(Z, n=self.shape[2], axis=2) / (self.shape[0] * self.shape[1])


def _worker(rank, world, port, shape, q):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), WORLD_SIZE=str(world), RANK=str(rank))
    sys.path.insert(0, ROOT)
    import torch.distributed as dist
    from paper_2202_12756_b200 import dist as D, inputs
    dist.init_process_group("gloo")
    Nx, Ny, Nz = shape
    f = inputs.uniform_grid(shape, torch.float64, seed=5)
    S = inputs.random_spectrum(shape, torch.complex128, seed=6)
    fft = D.SlabFFT(NumpyStages(Nx, Ny, Nz, world, rank), dist, "cpu", exchange="chunks")
    Nxl, L = Nx // world, Ny // world
    spec = torch.zeros((Nx, L, Nz // 2 + 1), dtype=torch.complex128)
    fft.forward(f[rank * Nxl:(rank + 1) * Nxl].contiguous(), spec)
    back = torch.zeros((Nxl, Ny, Nz), dtype=torch.float64)
    fft.inverse(S[:, rank * L:(rank + 1) * L, :].contiguous(), back)
    # descriptor hand-off of the UNIFIED exchange: each rank passes a pipe's read end to the other
    r_fd, w_fd = os.pipe()
    sockdir = D.private_socket_dir(dist)
    assert os.stat(sockdir).st_mode & 0o777 == 0o700
    fds = D.exchange_fds(rank, world, r_fd, sockdir, lambda: dist.barrier())
    D.remove_socket_dir(sockdir, rank)
    if rank == 0:                                          # a directory other users could enter is refused
        import tempfile
        loose = tempfile.mkdtemp()
        os.chmod(loose, 0o755)
        try:
            D.exchange_fds(rank, 1, r_fd, loose, lambda: None)
            raise AssertionError("exchange_fds accepted a world-accessible socket directory")
        except PermissionError:
            pass
        os.rmdir(loose)
    os.write(w_fd, (b"rank%d" % rank) * (world - 1))       # one 5-byte message for each peer that holds the read end
    got = [os.read(fd, 5).decode() if k != rank else None for k, fd in enumerate(fds)]
    dist.barrier()
    dist.destroy_process_group()
    q.put((rank, spec.numpy(), back.numpy(), got))


@pytest.mark.parametrize("shape,world", [((8, 12, 16), 2), ((12, 8, 6), 2), ((8, 8, 8), 4)])
def test_slab_fft_plumbing_matches_oracle(oracle_mod, shape, world):
    from paper_2202_12756_b200 import inputs
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, world, port, shape, q)) for r in range(world)]
    for p in procs:
        p.start()
    out = sorted((q.get(timeout=180) for _ in procs), key=lambda t: t[0])
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    Nx, Ny, Nz = shape
    L, Nxl = Ny // world, Nx // world
    F_ref = oracle_mod.r2c(inputs.uniform_grid(shape, torch.float64, seed=5).numpy())
    f_ref = oracle_mod.c2r(inputs.random_spectrum(shape, torch.complex128, seed=6).numpy(), Nz)
    for rank, spec, back, got in out:
        assert np.abs(spec - F_ref[:, rank * L:(rank + 1) * L, :]).max() <= 1e-11 * np.abs(F_ref).max()
        assert np.abs(back - f_ref[rank * Nxl:(rank + 1) * Nxl]).max() <= 1e-12 * max(1.0, np.abs(f_ref).max())
        assert got == [None if k == rank else "rank%d" % k for k in range(world)]


def test_layout_helpers():
    from paper_2202_12756_b200 import dist as D
    assert D.chunk_shape(1024, 1024, 1024, 8) == (128, 128, 512)            # 67 MB messages
    assert D.mirror_rank(0, 8) == [0, 7] and D.mirror_rank(3, 8) == [4, 5] and D.mirror_rank(0, 1) == [0]
    for G in (1, 2, 4, 8):
        L = 4
        for q in range(G):
            owners = {((-ky) % (G * L)) // L for ky in range(q * L, (q + 1) * L)}
            assert owners == set(D.mirror_rank(q, G))
