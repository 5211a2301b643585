"""Slab decomposition over G GPUs (one process per GPU) -- the paper's method itself.

Argument marshalling and plumbing only: every transform step runs in the kernels of ``libfft3d.so`` through the
stage entry points ``fft3d_dist_*`` (include/fft3d.h); ``torch.distributed`` supplies the process group, barriers
and -- for the CHUNKS exchange -- the all-to-all (NCCL grouped send/recv).

    DistPlan            ctypes wrapper of one rank's plan and its stage calls
    UnifiedExchange     the exchange array as ONE virtual range over all ranks' memory (CUDA VMM, descriptors passed
                        over Unix sockets): the forward y pass stores straight into the peers' HBM over NVLink
    SlabFFT             a rank's forward / inverse transform inside a process group, either exchange back-end
    EmulatedRanks       all G ranks on ONE device, one after the other, sharing one exchange array: the single-GPU
                        proof that the stage decomposition reproduces the monolithic transform bit for bit
"""
from __future__ import annotations

import ctypes
import os
import shutil
import socket
import stat
import tempfile

import torch

from . import binding as B

DIST_REAL, DIST_SLAB, DIST_SPEC, DIST_PLANES, DIST_WORK = 0, 1, 2, 3, 4
XCHG_UNIFIED, XCHG_CHUNKS = 0, 1


def _ptr(t):
    return ctypes.c_void_p(t if isinstance(t, int) else t.data_ptr())


class DistPlan:
    """fft3d_plan_dist(Nx, Ny, Nz, dtype, G, rank) and its stages, with torch tensors (or raw device addresses)."""

    def __init__(self, Nx, Ny, Nz, dtype=torch.float32, G=1, rank=0):
        lib = B.load_library()
        self._lib = lib
        self.shape = (int(Nx), int(Ny), int(Nz))
        self.G, self.rank = int(G), int(rank)
        self.dtype_code = {torch.float32: B.F32, torch.float64: B.F64}[dtype]
        self.real_dtype = dtype
        self.complex_dtype = {torch.float32: torch.complex64, torch.float64: torch.complex128}[dtype]
        h = ctypes.c_void_p()
        rc = lib.fft3d_plan_dist(ctypes.byref(h), Nx, Ny, Nz, self.dtype_code, self.G, self.rank)
        if rc != 0:
            raise B.Fft3dError(rc, "fft3d_plan_dist(%d,%d,%d,G=%d,rank=%d)" % (Nx, Ny, Nz, G, rank))
        self._h = h
        self.Nxl, self.L, self.M = Nx // G, Ny // G, Nz // 2

    def nbytes(self, which):
        return int(self._lib.fft3d_dist_bytes(self._h, which))

    # ---- buffers (shapes follow the layouts documented in include/fft3d.h) ----
    def empty_real_slab(self, device="cuda"):
        return torch.empty((self.Nxl, self.shape[1], self.shape[2]), dtype=self.real_dtype, device=device)

    def empty_slab_part(self, device="cuda"):
        return torch.empty((self.shape[0], self.L, self.M), dtype=self.complex_dtype, device=device)

    def empty_spec_part(self, device="cuda"):
        return torch.empty((self.shape[0], self.L, self.M + 1), dtype=self.complex_dtype, device=device)

    def empty_plane_part(self, device="cuda"):
        return torch.empty((2, self.shape[0], self.L), dtype=self.complex_dtype, device=device)

    def empty_work(self, device="cuda"):
        return torch.empty(self.nbytes(DIST_WORK), dtype=torch.uint8, device=device)

    def set_variant(self, v):
        rc = self._lib.fft3d_set_variant(self._h, int(v))
        if rc != 0:
            raise B.Fft3dError(rc, "fft3d_set_variant")

    def launch_impls(self, which):
        n = self._lib.fft3d_launches(self._h, which)
        return tuple(self._lib.fft3d_launch_impl(self._h, which, k).decode() for k in range(n))

    # ---- stages ----
    def _call(self, name, *args):
        rc = getattr(self._lib, name)(self._h, *args)
        if rc != 0:
            raise B.Fft3dError(rc, name)

    @staticmethod
    def _stream(stream):
        s = stream if stream is not None else torch.cuda.current_stream()
        return ctypes.c_void_p(s.cuda_stream)

    def _parts(self, parts):
        assert len(parts) == self.G
        return (ctypes.c_void_p * self.G)(*[_ptr(p) for p in parts])

    def fwd_local(self, real_slab, xchg, layout, work, stream=None):
        self._call("fft3d_dist_fwd_local", _ptr(real_slab), _ptr(xchg), int(layout), _ptr(work), self._stream(stream))

    def fwd_x(self, slab_part, spec_part, stream=None):
        self._call("fft3d_dist_fwd_x", _ptr(slab_part), _ptr(spec_part), self._stream(stream))

    def fwd_col0(self, spec_part, plane_part, stream=None):
        self._call("fft3d_dist_fwd_col0", _ptr(spec_part), _ptr(plane_part), self._stream(stream))

    def fwd_unpack(self, spec_part, plane_parts, stream=None):
        self._call("fft3d_dist_fwd_unpack", _ptr(spec_part), self._parts(plane_parts), self._stream(stream))

    def inv_planes(self, spec_part, plane_part, stream=None):
        self._call("fft3d_dist_inv_planes", _ptr(spec_part), _ptr(plane_part), self._stream(stream))

    def inv_pack(self, plane_parts, work, stream=None):
        self._call("fft3d_dist_inv_pack", self._parts(plane_parts), _ptr(work), self._stream(stream))

    def inv_x(self, spec_part, slab_part, work, stream=None):
        self._call("fft3d_dist_inv_x", _ptr(spec_part), _ptr(slab_part), _ptr(work), self._stream(stream))

    def inv_local(self, xchg, layout, real_slab, work, stream=None):
        self._call("fft3d_dist_inv_local", _ptr(xchg), int(layout), _ptr(real_slab), _ptr(work), self._stream(stream))

    def close(self):
        if getattr(self, "_h", None):
            self._lib.fft3d_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


# ------------------------------------------------------------------------------------------------------------------
# Layout arithmetic of the exchange (host side).  Pure index helpers, shared by the GPU path and by
# the CPU (gloo) tests of the N > 1 plumbing.
# ------------------------------------------------------------------------------------------------------------------
def chunk_shape(Nx, Ny, Nz, G):
    """One message of the all-to-all: Nx/G x Ny/G x Nz/2 packed complex (with the packed column)."""
    return (Nx // G, Ny // G, Nz // 2)


def mirror_rank(q, G):
    """Ranks whose rows hold ky' = -ky mod Ny for ky in rank q's rows [q*L, (q+1)*L): the partner planes of the
    Nyquist bookkeeping live there (row q*L itself maps to rank (G - q) % G, the others to rank G - 1 - q)."""
    return sorted({(G - q) % G, G - 1 - q})


def all_to_all_chunks(dist, send, recv, group=None):
    """send[q] (chunk for rank q) -> recv[r] (chunk from rank r); chunks land in source-rank order."""
    dist.all_to_all_single(torch.view_as_real(recv).reshape(-1), torch.view_as_real(send).reshape(-1), group=group)


def all_gather_parts(dist, part, gathered, group=None):
    """gathered[q] = rank q's `part` (the plane parts of the packed-column bookkeeping)."""
    dist.all_gather_into_tensor(torch.view_as_real(gathered).reshape(-1), torch.view_as_real(part).reshape(-1), group=group)


# ------------------------------------------------------------------------------------------------------------------
# UNIFIED exchange array over CUDA VMM
# ------------------------------------------------------------------------------------------------------------------
def private_socket_dir(dist, group=None):
    """A directory only this user can enter (mkdtemp: mode 0700, unpredictable name), made by rank 0 and announced to the
    group; also checks that every rank runs on rank 0's host -- descriptors travel over Unix sockets and the mapped
    memory over NVLink peer access: both are single-node mechanisms.  Rank 0 removes the directory after use
    (remove_socket_dir)."""
    rank = dist.get_rank(group)
    hosts = [None] * dist.get_world_size(group)
    dist.all_gather_object(hosts, socket.gethostname(), group=group)
    if len(set(hosts)) != 1:
        raise RuntimeError("the UNIFIED exchange maps peer memory of ONE node; ranks run on %s: use exchange='chunks'"
                           % sorted(set(hosts)))
    box = [tempfile.mkdtemp(prefix="fft3d_xchg_") if rank == 0 else None]
    dist.broadcast_object_list(box, src=dist.get_global_rank(group, 0) if group is not None else 0, group=group)
    return box[0]


def remove_socket_dir(path, rank):
    if rank == 0:
        shutil.rmtree(path, ignore_errors=True)


def exchange_fds(rank, world, fd, sockdir, barrier):
    """Every rank hands its file descriptor to every other rank over Unix sockets (SCM_RIGHTS).  Returns the list of
    descriptors in rank order (own entry = fd).  `barrier()` must synchronise the ranks.  The sockets live in `sockdir`,
    which must belong to this user and be closed to everybody else (private_socket_dir): whoever can reach a socket
    receives a handle to GPU memory, and whoever can replace one can inject a handle of its own."""
    st = os.stat(sockdir)
    if not stat.S_ISDIR(st.st_mode) or st.st_uid != os.geteuid() or (st.st_mode & 0o077) != 0:
        raise PermissionError("%s must be a directory owned by this user with mode 0700" % sockdir)
    path = os.path.join(sockdir, "rank_%d.sock")
    srv = socket.socket(socket.AF_UNIX, socket.SOCK_STREAM)
    srv.bind(path % rank)
    srv.listen(world)
    barrier()                                            # every server socket exists
    out = [None] * world
    out[rank] = fd
    # round r: connect to rank (rank + r) % world and fetch its fd, while serving whoever connects to us
    srv.settimeout(60.0)
    pending = world - 1
    clients = []
    for r in range(1, world):
        peer = (rank + r) % world
        c = socket.socket(socket.AF_UNIX, socket.SOCK_STREAM)
        c.settimeout(60.0)
        c.connect(path % peer)
        clients.append((peer, c))
    while pending:
        conn, _ = srv.accept()
        socket.send_fds(conn, [b"f"], [fd])
        conn.close()
        pending -= 1
    for peer, c in clients:
        _msg, fds, _flags, _addr = socket.recv_fds(c, 16, 1)
        out[peer] = fds[0]
        c.close()
    barrier()
    srv.close()
    try:
        os.unlink(path % rank)
    except FileNotFoundError:
        pass
    return out


class UnifiedExchange:
    """G device allocations mapped back to back into one virtual range: part q = rank q's memory.

    single-process form (tests, EmulatedRanks): UnifiedExchange.local(G, part_bytes) creates all G parts on the
    current device; multi-process form: UnifiedExchange.across(rank, world, part_bytes, dist, group) creates the own
    part, passes descriptors, imports the peers' parts."""

    def __init__(self, handles, part_bytes, own):
        lib = B.load_library()
        self._lib, self.handles, self.part_bytes, self._own = lib, handles, int(part_bytes), own
        arr = (ctypes.c_ulonglong * len(handles))(*handles)
        va = ctypes.c_void_p()
        rc = lib.fft3d_vmm_map(arr, len(handles), self.part_bytes, ctypes.byref(va))
        if rc != 0:
            raise B.Fft3dError(rc, "fft3d_vmm_map")
        self.base = int(va.value)

    @staticmethod
    def usable(part_bytes):
        g = int(B.load_library().fft3d_vmm_granularity())
        return g > 0 and part_bytes % g == 0

    @classmethod
    def local(cls, G, part_bytes):
        lib = B.load_library()
        hs = []
        for _ in range(G):
            h = ctypes.c_ulonglong()
            rc = lib.fft3d_vmm_create(part_bytes, ctypes.byref(h), None)
            if rc != 0:
                raise B.Fft3dError(rc, "fft3d_vmm_create")
            hs.append(h.value)
        return cls(hs, part_bytes, own=list(range(G)))

    @classmethod
    def across(cls, rank, world, part_bytes, dist, group=None):
        lib = B.load_library()
        sockdir = private_socket_dir(dist, group)        # also: all ranks on one host, or it raises
        h, fd = ctypes.c_ulonglong(), ctypes.c_int(-1)
        rc = lib.fft3d_vmm_create(part_bytes, ctypes.byref(h), ctypes.byref(fd))
        if rc != 0:
            raise B.Fft3dError(rc, "fft3d_vmm_create")
        try:
            fds = exchange_fds(rank, world, fd.value, sockdir, lambda: dist.barrier(group=group))
        finally:
            remove_socket_dir(sockdir, rank)
        hs = []
        for q in range(world):
            if q == rank:
                hs.append(h.value)
                continue
            hq = ctypes.c_ulonglong()
            rc = lib.fft3d_vmm_import(fds[q], ctypes.byref(hq))
            os.close(fds[q])
            if rc != 0:
                raise B.Fft3dError(rc, "fft3d_vmm_import")
            hs.append(hq.value)
        os.close(fd.value)
        return cls(hs, part_bytes, own=[rank])

    def part(self, q):
        return self.base + q * self.part_bytes

    def close(self):
        if self.base:
            self._lib.fft3d_vmm_unmap(ctypes.c_void_p(self.base), len(self.handles), self.part_bytes)
            for h in self.handles:
                self._lib.fft3d_vmm_release(h)
            self.base = 0

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


# ------------------------------------------------------------------------------------------------------------------
# one rank inside a process group
# ------------------------------------------------------------------------------------------------------------------
class SlabFFT:
    """A rank's 3D R2C / C2R over a torch.distributed group (NCCL, one process per GPU).

    exchange = "chunks": local chunk buffers + all_to_all_single (NCCL grouped send/recv) between the stages;
    exchange = "unified": the exchange array is one VMM range over all ranks' memory; the forward y pass pushes
    its rows into the peers' parts over NVLink, the inverse y pass pulls them; only barriers in between.
    The plane parts of the packed-column bookkeeping (one Nx x Ny/G plane per rank) are all-gathered.
    `times` accumulates device milliseconds per phase ("comp", "comm") when `timed` is set."""

    def __init__(self, plan, dist, device, exchange="chunks", group=None):
        """plan: a DistPlan (or, in the CPU tests of this plumbing, any object with its stage methods and buffer
        factories); dist: the torch.distributed module; device: this rank's device."""
        self.dist, self.group, self.device = dist, group, torch.device(device)
        self.G, self.rank = dist.get_world_size(group), dist.get_rank(group)
        assert (plan.G, plan.rank) == (self.G, self.rank)
        self.plan = p = plan
        Nx, Ny, Nz = p.shape
        self.work = p.empty_work(device)
        self.plane = p.empty_plane_part(device)
        self.planes = torch.empty((self.G,) + tuple(self.plane.shape), dtype=p.complex_dtype, device=device)
        self.exchange = exchange
        if exchange == "unified":
            part = p.nbytes(DIST_SLAB)
            if not UnifiedExchange.usable(part):
                raise ValueError("part size %d is not a multiple of the VMM granularity: use exchange='chunks'" % part)
            self.ux = UnifiedExchange.across(self.rank, self.G, part, dist, group)
        elif exchange == "chunks":
            self.send = torch.empty((self.G,) + chunk_shape(Nx, Ny, Nz, self.G), dtype=p.complex_dtype, device=device)
            self.recv = torch.empty_like(self.send)
        else:
            raise ValueError(exchange)
        self.timed = False
        self.times = {"comp": 0.0, "comm": 0.0}
        self._ev = []

    @classmethod
    def create(cls, Nx, Ny, Nz, dtype, dist, device, exchange="chunks", group=None, variant=0):
        plan = DistPlan(Nx, Ny, Nz, dtype, dist.get_world_size(group), dist.get_rank(group))
        plan.set_variant(variant)
        return cls(plan, dist, device, exchange, group)

    def _mark(self, kind):
        if self.timed and self.device.type == "cuda":
            e = torch.cuda.Event(enable_timing=True)
            e.record(torch.cuda.current_stream(self.device))
            self._ev.append((kind, e))

    def collect_times(self):
        """Sum the recorded phases (call after a synchronize)."""
        for (k0, e0), (_k1, e1) in zip(self._ev[:-1], self._ev[1:]):
            if k0 in self.times:
                self.times[k0] += e0.elapsed_time(e1)
        self._ev = []

    def _sync_ranks(self):
        """All ranks' enqueued work is complete: the point where peers' memory may be read / rewritten."""
        if self.device.type == "cuda":
            torch.cuda.current_stream(self.device).synchronize()
        self.dist.barrier(group=self.group)

    def forward(self, real_slab, spec_part):
        p, G = self.plan, self.G
        self._mark("comp")
        if self.exchange == "unified":
            p.fwd_local(real_slab, self.ux.base, XCHG_UNIFIED, self.work)
            self._mark("comm")
            self._sync_ranks()                           # every rank's rows have landed in my part
            self._mark("comp")
            p.fwd_x(self.ux.part(self.rank), spec_part)
        else:
            p.fwd_local(real_slab, self.send, XCHG_CHUNKS, self.work)
            self._mark("comm")
            all_to_all_chunks(self.dist, self.send, self.recv, self.group)
            self._mark("comp")
            p.fwd_x(self.recv, spec_part)
        p.fwd_col0(spec_part, self.plane)
        self._mark("comm")
        all_gather_parts(self.dist, self.plane, self.planes, self.group)
        self._mark("comp")
        p.fwd_unpack(spec_part, [self.planes[q] for q in range(G)])
        self._mark("end")
        return spec_part

    def inverse(self, spec_part, real_slab):
        p, G = self.plan, self.G
        self._mark("comp")
        p.inv_planes(spec_part, self.plane)
        self._mark("comm")
        all_gather_parts(self.dist, self.plane, self.planes, self.group)
        self._mark("comp")
        p.inv_pack([self.planes[q] for q in range(G)], self.work)
        if self.exchange == "unified":
            p.inv_x(spec_part, self.ux.part(self.rank), self.work)
            self._mark("comm")
            self._sync_ranks()                           # every rank's part is complete before anyone pulls from it
            self._mark("comp")
            p.inv_local(self.ux.base, XCHG_UNIFIED, real_slab, self.work)
            self._sync_ranks()                           # nobody overwrites a part that a peer is still reading
        else:
            p.inv_x(spec_part, self.send.reshape(p.shape[0], p.L, p.M), self.work)
            self._mark("comm")
            all_to_all_chunks(self.dist, self.send, self.recv, self.group)
            self._mark("comp")
            p.inv_local(self.recv, XCHG_CHUNKS, real_slab, self.work)
        self._mark("end")
        return real_slab

    def close(self):
        if self.exchange == "unified":
            self.ux.close()
        self.plan.close()


# ------------------------------------------------------------------------------------------------------------------
# all G ranks on one device (single-GPU proof of the stage decomposition)
# ------------------------------------------------------------------------------------------------------------------
class EmulatedRanks:
    """Runs the G ranks' stages one rank after the other on the current device.  The ranks do not wait on one
    another inside kernels (each stage is an ordinary launch), so running them in sequence on one stream IS a valid
    schedule of the distributed algorithm.  layout = XCHG_UNIFIED: one exchange array shared by all ranks (a plain
    buffer, or `vmm=True`: G separate allocations mapped into one range, as on a real node); XCHG_CHUNKS: per-rank
    send/recv chunk buffers and an explicit all-to-all done with copies."""

    def __init__(self, Nx, Ny, Nz, dtype, G, layout=XCHG_UNIFIED, vmm=False, variant=0, device="cuda"):
        self.G, self.layout, self.device = G, layout, device
        self.plans = [DistPlan(Nx, Ny, Nz, dtype, G, r) for r in range(G)]
        for p in self.plans:
            p.set_variant(variant)
        p0 = self.plans[0]
        self.work = p0.empty_work(device)                # the ranks run one after the other: one workspace serves all
        self.planes = torch.empty((G, 2, Nx, Ny // G), dtype=p0.complex_dtype, device=device)
        self.ux = None
        part = p0.nbytes(DIST_SLAB)
        if layout == XCHG_UNIFIED:
            if vmm:
                self.ux = UnifiedExchange.local(G, part)
                self.xbase = self.ux.base
            else:
                self.xbuf = torch.empty(G * part, dtype=torch.uint8, device=device)
                self.xbase = self.xbuf.data_ptr()
            self.part_bytes = part
        else:
            shp = (G, G) + chunk_shape(Nx, Ny, Nz, G)
            self.send = torch.empty(shp, dtype=p0.complex_dtype, device=device)
            self.recv = torch.empty(shp, dtype=p0.complex_dtype, device=device)

    def forward(self, real, spec):
        """real: [Nx][Ny][Nz] (rank r's slab = real[r*Nxl:(r+1)*Nxl]); spec: flat [G][Nx][L][M+1] (part q = rank q's)."""
        G, P = self.G, self.plans
        Nxl = P[0].Nxl
        parts = spec.reshape(G, -1)
        for r in range(G):
            if self.layout == XCHG_UNIFIED:
                P[r].fwd_local(real[r * Nxl:(r + 1) * Nxl], self.xbase, XCHG_UNIFIED, self.work)
            else:
                P[r].fwd_local(real[r * Nxl:(r + 1) * Nxl], self.send[r], XCHG_CHUNKS, self.work)
        if self.layout == XCHG_CHUNKS:
            self.recv.copy_(self.send.transpose(0, 1))   # the all-to-all: chunk q of rank r -> slot r of rank q
        for q in range(G):
            slab = self.xbase + q * self.part_bytes if self.layout == XCHG_UNIFIED else self.recv[q]
            P[q].fwd_x(slab, parts[q])
            P[q].fwd_col0(parts[q], self.planes[q])
        for q in range(G):
            P[q].fwd_unpack(parts[q], [self.planes[k] for k in range(G)])
        return spec

    def inverse(self, spec, real):
        G, P = self.G, self.plans
        Nxl = P[0].Nxl
        parts = spec.reshape(G, -1)
        for q in range(G):
            P[q].inv_planes(parts[q], self.planes[q])
        for q in range(G):
            P[q].inv_pack([self.planes[k] for k in range(G)], self.work)
            slab = self.xbase + q * self.part_bytes if self.layout == XCHG_UNIFIED else self.send[q]
            P[q].inv_x(parts[q], slab, self.work)
        if self.layout == XCHG_CHUNKS:
            self.recv.copy_(self.send.transpose(0, 1))
        for r in range(G):
            src = self.xbase if self.layout == XCHG_UNIFIED else self.recv[r]
            P[r].inv_local(src, self.layout, real[r * Nxl:(r + 1) * Nxl], self.work)
        return real

    def close(self):
        for p in self.plans:
            p.close()
        if self.ux is not None:
            self.ux.close()
