"""ctypes binding of include/fft3d.h -- argument marshalling only.

Every step of the transform runs in the kernels of ``libfft3d.so``; PyTorch supplies device
memory and the stream.  There is no fallback: if the library is missing or no CUDA device
is present the calls raise.
"""
from __future__ import annotations

import ctypes
import os

import torch

F32, F64 = 0, 1
OPT_FUSED_Z_SMS_FWD, OPT_FUSED_Z_SMS_INV, OPT_FUSED_RING_PLANES, OPT_FUSED_MIXED, OPT_FUSED_JITTER = 1, 2, 3, 4, 5
_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libfft3d.so")

EXPORTS = (
    "fft3d_plan", "fft3d_supported_length", "fft3d_workspace_bytes", "fft3d_real_bytes",
    "fft3d_complex_bytes", "fft3d_index", "fft3d_r2c", "fft3d_c2r", "fft3d_r2c_host",
    "fft3d_c2r_host", "fft3d_launches", "fft3d_launch_name", "fft3d_set_variant", "fft3d_destroy", "fft3d_strerror",
    "fft3d_timing_enable", "fft3d_timing_read", "fft3d_plan_c2c", "fft3d_c2c", "fft3d_c2c_host",
    "fft3d_launch_impl", "fft3d_set_option",
    "fft3d_plan_inplace", "fft3d_r2c_inplace", "fft3d_c2r_inplace", "fft3d_plan_pencil",
    "fft3d_plan_dist", "fft3d_dist_bytes", "fft3d_dist_fwd_local", "fft3d_dist_fwd_x", "fft3d_dist_fwd_col0",
    "fft3d_dist_fwd_unpack", "fft3d_dist_inv_planes", "fft3d_dist_inv_pack", "fft3d_dist_inv_x", "fft3d_dist_inv_local",
    "fft3d_r2c_static",
    "fft3d_vmm_granularity", "fft3d_vmm_create", "fft3d_vmm_import", "fft3d_vmm_map", "fft3d_vmm_unmap", "fft3d_vmm_release",
)

_lib = None


class Fft3dError(RuntimeError):
    def __init__(self, status: int, where: str):
        self.status = status
        super().__init__("%s: %s (status %d)" % (where, strerror(status), status))


def load_library() -> ctypes.CDLL:
    """Load libfft3d.so (built by ``__graft_entry__.build()`` / ``make -C csrc``)."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise ImportError(
            "%s is missing: build it with `python -c 'import __graft_entry__ as g; g.build()'` "
            "(there is no CPU or PyTorch fallback for the FFT path)" % LIB_PATH)
    lib = ctypes.CDLL(LIB_PATH)
    vp, ll, i, sz = ctypes.c_void_p, ctypes.c_longlong, ctypes.c_int, ctypes.c_size_t
    lib.fft3d_plan.argtypes = [ctypes.POINTER(vp), ll, ll, ll, i, i]
    lib.fft3d_plan.restype = i
    lib.fft3d_plan_c2c.argtypes = [ctypes.POINTER(vp), ll, ll, ll, i, i]
    lib.fft3d_plan_c2c.restype = i
    lib.fft3d_plan_pencil.argtypes = [ctypes.POINTER(vp), ll, ll, ll, i, i, i]
    lib.fft3d_plan_pencil.restype = i
    lib.fft3d_c2c.argtypes = [vp, vp, vp, vp, i, vp]
    lib.fft3d_c2c.restype = i
    lib.fft3d_c2c_host.argtypes = [vp, vp, vp, i]
    lib.fft3d_c2c_host.restype = i
    lib.fft3d_supported_length.argtypes = [ll]
    lib.fft3d_supported_length.restype = i
    for nm in ("fft3d_workspace_bytes", "fft3d_real_bytes", "fft3d_complex_bytes"):
        getattr(lib, nm).argtypes = [vp]
        getattr(lib, nm).restype = sz
    lib.fft3d_index.argtypes = [vp, ll, ll, ll]
    lib.fft3d_index.restype = ll
    for nm in ("fft3d_r2c", "fft3d_c2r"):
        getattr(lib, nm).argtypes = [vp, vp, vp, vp, vp]
        getattr(lib, nm).restype = i
    for nm in ("fft3d_r2c_host", "fft3d_c2r_host"):
        getattr(lib, nm).argtypes = [vp, vp, vp]
        getattr(lib, nm).restype = i
    lib.fft3d_r2c_static.argtypes = [ll, ll, ll, i, i, vp, vp, vp]
    lib.fft3d_r2c_static.restype = i
    lib.fft3d_launches.argtypes = [vp, i]
    lib.fft3d_launches.restype = i
    lib.fft3d_launch_name.argtypes = [vp, i, i]
    lib.fft3d_launch_name.restype = ctypes.c_char_p
    lib.fft3d_launch_impl.argtypes = [vp, i, i]
    lib.fft3d_launch_impl.restype = ctypes.c_char_p
    lib.fft3d_set_variant.argtypes = [vp, i]
    lib.fft3d_set_variant.restype = i
    ull = ctypes.c_ulonglong
    lib.fft3d_plan_inplace.argtypes = [ctypes.POINTER(vp), ll, ll, ll, i, i]
    lib.fft3d_plan_inplace.restype = i
    for nm in ("fft3d_r2c_inplace", "fft3d_c2r_inplace"):
        getattr(lib, nm).argtypes = [vp, vp, vp, vp]
        getattr(lib, nm).restype = i
    lib.fft3d_plan_dist.argtypes = [ctypes.POINTER(vp), ll, ll, ll, i, i, i]
    lib.fft3d_plan_dist.restype = i
    lib.fft3d_dist_bytes.argtypes = [vp, i]
    lib.fft3d_dist_bytes.restype = sz
    lib.fft3d_dist_fwd_local.argtypes = [vp, vp, vp, i, vp, vp]
    lib.fft3d_dist_inv_local.argtypes = [vp, vp, i, vp, vp, vp]
    lib.fft3d_dist_fwd_x.argtypes = [vp, vp, vp, vp]
    lib.fft3d_dist_inv_x.argtypes = [vp, vp, vp, vp, vp]
    lib.fft3d_dist_fwd_col0.argtypes = [vp, vp, vp, vp]
    lib.fft3d_dist_inv_planes.argtypes = [vp, vp, vp, vp]
    lib.fft3d_dist_fwd_unpack.argtypes = [vp, vp, ctypes.POINTER(vp), vp]
    lib.fft3d_dist_inv_pack.argtypes = [vp, ctypes.POINTER(vp), vp, vp]
    for nm in ("fft3d_dist_fwd_local", "fft3d_dist_inv_local", "fft3d_dist_fwd_x", "fft3d_dist_inv_x", "fft3d_dist_fwd_col0",
               "fft3d_dist_inv_planes", "fft3d_dist_fwd_unpack", "fft3d_dist_inv_pack"):
        getattr(lib, nm).restype = i
    lib.fft3d_vmm_granularity.argtypes = []
    lib.fft3d_vmm_granularity.restype = sz
    lib.fft3d_vmm_create.argtypes = [sz, ctypes.POINTER(ull), ctypes.POINTER(i)]
    lib.fft3d_vmm_import.argtypes = [i, ctypes.POINTER(ull)]
    lib.fft3d_vmm_map.argtypes = [ctypes.POINTER(ull), i, sz, ctypes.POINTER(vp)]
    lib.fft3d_vmm_unmap.argtypes = [vp, i, sz]
    lib.fft3d_vmm_release.argtypes = [ull]
    for nm in ("fft3d_vmm_create", "fft3d_vmm_import", "fft3d_vmm_map", "fft3d_vmm_unmap", "fft3d_vmm_release"):
        getattr(lib, nm).restype = i
    lib.fft3d_set_option.argtypes = [vp, i, ll]
    lib.fft3d_set_option.restype = i
    lib.fft3d_timing_enable.argtypes = [vp, i]
    lib.fft3d_timing_enable.restype = i
    lib.fft3d_timing_read.argtypes = [vp, i, ctypes.POINTER(ctypes.c_float), ctypes.POINTER(i)]
    lib.fft3d_timing_read.restype = i
    lib.fft3d_destroy.argtypes = [vp]
    lib.fft3d_destroy.restype = i
    lib.fft3d_strerror.argtypes = [i]
    lib.fft3d_strerror.restype = ctypes.c_char_p
    _lib = lib
    return lib


def strerror(status: int) -> str:
    return load_library().fft3d_strerror(int(status)).decode()


def supported_length(n: int) -> bool:
    return bool(load_library().fft3d_supported_length(int(n)))


_REAL = {F32: torch.float32, F64: torch.float64}
_CPLX = {F32: torch.complex64, F64: torch.complex128}

STATIC_SCRATCH_BYTES = 17 << 20


def r2c_static(real_in: torch.Tensor, cplx_out: torch.Tensor, virtual_slabs: int = 1, stream=None) -> torch.Tensor:
    """fft3d_r2c_static: forward R2C of ``real_in`` [Nx][Ny][Nz] into ``cplx_out`` (flat, Nx*Ny*(Nz/2+1) complex, slab
    layout) for callers that cannot allocate device memory -- code living inside someone else's memory pool, or inside a
    loop where cudaMalloc/cudaFree are off limits.  No plan and no workspace: the library's own 17 MiB built-in scratch
    array is used, so both tensors must be supplied by the caller (this wrapper allocates nothing either) and the grid
    must be small enough (Nx*Ny*Nz*sizeof(real) <= 16 MiB always fits; otherwise Fft3dError with status 5).  Calls on
    one stream are ordered; calls that can overlap on the GPU share the scratch and corrupt each other."""
    lib = load_library()
    if not (real_in.is_cuda and real_in.is_contiguous() and real_in.dim() == 3 and real_in.dtype in (torch.float32, torch.float64)):
        raise ValueError("real_in must be a contiguous 3-D CUDA tensor of float32 or float64")
    Nx, Ny, Nz = (int(v) for v in real_in.shape)
    code = F32 if real_in.dtype == torch.float32 else F64
    if not (cplx_out.is_cuda and cplx_out.is_contiguous() and cplx_out.device == real_in.device and
            cplx_out.dtype == _CPLX[code] and cplx_out.numel() == Nx * Ny * (Nz // 2 + 1)):
        raise ValueError("cplx_out must be a contiguous %s CUDA tensor of %d elements on %s"
                         % (_CPLX[code], Nx * Ny * (Nz // 2 + 1), real_in.device))
    s = stream if stream is not None else torch.cuda.current_stream(real_in.device)
    with torch.cuda.device(real_in.device):
        rc = lib.fft3d_r2c_static(Nx, Ny, Nz, code, int(virtual_slabs), real_in.data_ptr(), cplx_out.data_ptr(),
                                  ctypes.c_void_p(s.cuda_stream))
    if rc != 0:
        raise Fft3dError(rc, "fft3d_r2c_static(%d,%d,%d,p=%d)" % (Nx, Ny, Nz, virtual_slabs))
    return cplx_out


class Plan:
    """fft3d_plan(Nx, Ny, Nz, dtype, virtual_slabs) with torch tensors as buffers."""

    _PLAN_FN = "fft3d_plan"

    def __init__(self, Nx: int, Ny: int, Nz: int, dtype=torch.float32, virtual_slabs: int = 1):
        lib = load_library()
        self.dtype_code = {torch.float32: F32, torch.float64: F64}[dtype]
        self.shape = (int(Nx), int(Ny), int(Nz))
        self.p = int(virtual_slabs)
        h = ctypes.c_void_p()
        rc = getattr(lib, self._PLAN_FN)(ctypes.byref(h), Nx, Ny, Nz, self.dtype_code, self.p)
        if rc != 0:
            raise Fft3dError(rc, "%s(%d,%d,%d,p=%d)" % (self._PLAN_FN, Nx, Ny, Nz, self.p))
        self._h = h
        self._lib = lib
        self.real_dtype = _REAL[self.dtype_code]
        self.complex_dtype = _CPLX[self.dtype_code]
        self.real_bytes = lib.fft3d_real_bytes(h)
        self.complex_bytes = lib.fft3d_complex_bytes(h)
        self.workspace_bytes = lib.fft3d_workspace_bytes(h)
        self.n_complex = self.complex_bytes // (2 * (4 if self.dtype_code == F32 else 8))

    # ---- buffers -------------------------------------------------------------------------
    def empty_real(self, device="cuda"):
        return torch.empty(self.shape, dtype=self.real_dtype, device=device)

    def empty_complex(self, device="cuda"):
        """Flat complex buffer in the slab layout [p][Nx][Ny/p][Nz/2+1]."""
        return torch.empty(self.n_complex, dtype=self.complex_dtype, device=device)

    def empty_workspace(self, device="cuda"):
        return torch.empty(self.workspace_bytes, dtype=torch.uint8, device=device)

    def index(self, kx: int, ky: int, kz: int) -> int:
        return int(self._lib.fft3d_index(self._h, kx, ky, kz))

    def launches(self, which: int) -> int:
        return int(self._lib.fft3d_launches(self._h, which))

    def set_variant(self, v: int):
        rc = self._lib.fft3d_set_variant(self._h, int(v))
        if rc != 0:
            raise Fft3dError(rc, "fft3d_set_variant")

    def set_option(self, option: int, value: int):
        rc = self._lib.fft3d_set_option(self._h, int(option), int(value))
        if rc != 0:
            raise Fft3dError(rc, "fft3d_set_option(%d, %d)" % (option, value))

    def launch_names(self, which: int):
        return tuple(self._lib.fft3d_launch_name(self._h, which, k).decode() for k in range(self.launches(which)))

    def launch_impls(self, which: int):
        """Implementation of each launch ("tma", "fused_ring", "plain", ...), aligned with launch_names."""
        return tuple(self._lib.fft3d_launch_impl(self._h, which, k).decode() for k in range(self.launches(which)))

    def timing_enable(self, max_calls: int):
        rc = self._lib.fft3d_timing_enable(self._h, int(max_calls))
        if rc != 0:
            raise Fft3dError(rc, "fft3d_timing_enable")

    def timing_read(self, which: int):
        """-> (dict launch name -> summed ms, calls) for direction which (0 r2c, 1 c2r)."""
        ms = (ctypes.c_float * 8)()
        calls = ctypes.c_int(0)
        rc = self._lib.fft3d_timing_read(self._h, int(which), ms, ctypes.byref(calls))
        if rc != 0:
            raise Fft3dError(rc, "fft3d_timing_read")
        names = self.launch_names(which)
        n = len(names)
        return {names[k]: float(ms[k]) for k in range(n)}, calls.value

    # ---- device entry points -------------------------------------------------------------
    def _check(self, t: torch.Tensor, dtype, nbytes: int, name: str):
        if not (t.is_cuda and t.is_contiguous() and t.dtype == dtype and t.numel() * t.element_size() == nbytes):
            raise ValueError("%s must be a contiguous CUDA tensor of dtype %s and %d bytes" % (name, dtype, nbytes))

    def _check_work(self, work: torch.Tensor, ref: torch.Tensor):
        # the C side cannot see the size of a bare pointer: an undersized workspace would be an out-of-bounds write
        if not (work.is_cuda and work.is_contiguous() and work.device == ref.device and
                work.numel() * work.element_size() >= self.workspace_bytes):
            raise ValueError("work must be a contiguous CUDA tensor on %s of at least %d bytes"
                             % (ref.device, self.workspace_bytes))

    def _check_host(self, t: torch.Tensor, dtype, nbytes: int, name: str):
        if t.is_cuda or not t.is_contiguous() or t.dtype != dtype or t.numel() * t.element_size() != nbytes:
            raise ValueError("%s must be a contiguous host tensor of dtype %s and %d bytes" % (name, dtype, nbytes))

    def _stream(self, stream, ref: torch.Tensor, temporaries):
        """The stream to launch on; buffers allocated inside the call are tied to it so that the caching
        allocator does not hand them out again while the kernels are still queued."""
        s = stream if stream is not None else torch.cuda.current_stream(ref.device)
        for t in temporaries:
            t.record_stream(s)
        return s

    def r2c(self, real_in, cplx_out=None, work=None, stream=None):
        self._check(real_in, self.real_dtype, self.real_bytes, "real_in")
        tmp = []
        if cplx_out is None:
            cplx_out = self.empty_complex(real_in.device)
            tmp.append(cplx_out)
        if work is None:
            work = self.empty_workspace(real_in.device)
            tmp.append(work)
        self._check(cplx_out, self.complex_dtype, self.complex_bytes, "cplx_out")
        self._check_work(work, real_in)
        s = self._stream(stream, real_in, tmp)
        rc = self._lib.fft3d_r2c(self._h, real_in.data_ptr(), cplx_out.data_ptr(), work.data_ptr(),
                                 ctypes.c_void_p(s.cuda_stream))
        if rc != 0:
            raise Fft3dError(rc, "fft3d_r2c")
        return cplx_out

    def c2r(self, cplx_in, real_out=None, work=None, stream=None):
        self._check(cplx_in, self.complex_dtype, self.complex_bytes, "cplx_in")
        tmp = []
        if real_out is None:
            real_out = self.empty_real(cplx_in.device)
            tmp.append(real_out)
        if work is None:
            work = self.empty_workspace(cplx_in.device)
            tmp.append(work)
        self._check(real_out, self.real_dtype, self.real_bytes, "real_out")
        self._check_work(work, cplx_in)
        s = self._stream(stream, cplx_in, tmp)
        rc = self._lib.fft3d_c2r(self._h, cplx_in.data_ptr(), real_out.data_ptr(), work.data_ptr(),
                                 ctypes.c_void_p(s.cuda_stream))
        if rc != 0:
            raise Fft3dError(rc, "fft3d_c2r")
        return real_out

    # ---- host entry points (host tensors, copies inside the call) --------------------------
    def r2c_host(self, real_in: torch.Tensor, cplx_out: torch.Tensor):
        self._check_host(real_in, self.real_dtype, self.real_bytes, "real_in")
        self._check_host(cplx_out, self.complex_dtype, self.complex_bytes, "cplx_out")
        rc = self._lib.fft3d_r2c_host(self._h, real_in.data_ptr(), cplx_out.data_ptr())
        if rc != 0:
            raise Fft3dError(rc, "fft3d_r2c_host")
        return cplx_out

    def c2r_host(self, cplx_in: torch.Tensor, real_out: torch.Tensor):
        self._check_host(cplx_in, self.complex_dtype, self.complex_bytes, "cplx_in")
        self._check_host(real_out, self.real_dtype, self.real_bytes, "real_out")
        rc = self._lib.fft3d_c2r_host(self._h, cplx_in.data_ptr(), real_out.data_ptr())
        if rc != 0:
            raise Fft3dError(rc, "fft3d_c2r_host")
        return real_out

    # ---- layout helpers (index arithmetic only) --------------------------------------------
    def to_natural(self, cplx_flat: torch.Tensor) -> torch.Tensor:
        """View a slab-layout spectrum as [Nx][Ny][Nz/2+1] (a permuted copy)."""
        Nx, Ny, Nz = self.shape
        L = Ny // self.p
        return cplx_flat.reshape(self.p, Nx, L, Nz // 2 + 1).permute(1, 0, 2, 3).reshape(Nx, Ny, Nz // 2 + 1)

    def from_natural(self, cplx_nat: torch.Tensor) -> torch.Tensor:
        Nx, Ny, Nz = self.shape
        L = Ny // self.p
        return cplx_nat.reshape(Nx, self.p, L, Nz // 2 + 1).permute(1, 0, 2, 3).contiguous().reshape(-1)

    def close(self):
        if getattr(self, "_h", None) is not None and self._h:
            self._lib.fft3d_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


class PlanPencil(Plan):
    """fft3d_plan_pencil(Nx, Ny, Nz, dtype, px, py): the spectrum laid out as a px x py rank grid would hold it."""

    def __init__(self, Nx: int, Ny: int, Nz: int, dtype=torch.float32, px: int = 1, py: int = 1):
        lib = load_library()
        self.dtype_code = {torch.float32: F32, torch.float64: F64}[dtype]
        self.shape = (int(Nx), int(Ny), int(Nz))
        self.p, self.px, self.py = int(px), int(px), int(py)
        h = ctypes.c_void_p()
        rc = lib.fft3d_plan_pencil(ctypes.byref(h), Nx, Ny, Nz, self.dtype_code, self.px, self.py)
        if rc != 0:
            raise Fft3dError(rc, "fft3d_plan_pencil(%d,%d,%d,px=%d,py=%d)" % (Nx, Ny, Nz, px, py))
        self._h = h
        self._lib = lib
        self.real_dtype = _REAL[self.dtype_code]
        self.complex_dtype = _CPLX[self.dtype_code]
        self.real_bytes = lib.fft3d_real_bytes(h)
        self.complex_bytes = lib.fft3d_complex_bytes(h)
        self.workspace_bytes = lib.fft3d_workspace_bytes(h)
        self.n_complex = self.complex_bytes // (2 * (4 if self.dtype_code == F32 else 8))

    def _blocks(self):
        Nx, Ny, Nz = self.shape
        L, c = Ny // self.px, (Nz // 2) // self.py
        off = 0
        for a in range(self.px):
            for b in range(self.py):
                cz = c + 1 if b == self.py - 1 else c
                yield a, b, off, L, c, cz
                off += Nx * L * cz

    def to_natural(self, cplx_flat: torch.Tensor) -> torch.Tensor:
        """Pencil-layout spectrum -> [Nx][Ny][Nz/2+1] (a permuted copy; index arithmetic only)."""
        Nx, Ny, Nz = self.shape
        out = torch.empty((Nx, Ny, Nz // 2 + 1), dtype=cplx_flat.dtype, device=cplx_flat.device)
        for a, b, off, L, c, cz in self._blocks():
            out[:, a * L:(a + 1) * L, b * c:b * c + cz] = cplx_flat[off:off + Nx * L * cz].reshape(Nx, L, cz)
        return out

    def from_natural(self, cplx_nat: torch.Tensor) -> torch.Tensor:
        Nx, Ny, Nz = self.shape
        out = torch.empty(Nx * Ny * (Nz // 2 + 1), dtype=cplx_nat.dtype, device=cplx_nat.device)
        for a, b, off, L, c, cz in self._blocks():
            out[off:off + Nx * L * cz] = cplx_nat[:, a * L:(a + 1) * L, b * c:b * c + cz].reshape(-1)
        return out


class PlanInplace(Plan):
    """fft3d_plan_inplace: the padded in-place layout (rows of Nz+2 reals; the spectrum overwrites the field)."""

    _PLAN_FN = "fft3d_plan_inplace"

    def empty_data(self, device="cuda"):
        """The shared buffer, as a real tensor [Nx][Ny][Nz+2]."""
        Nx, Ny, Nz = self.shape
        return torch.empty((Nx, Ny, Nz + 2), dtype=self.real_dtype, device=device)

    def as_spectrum(self, data: torch.Tensor) -> torch.Tensor:
        """The same memory viewed as the flat slab-layout spectrum."""
        return torch.view_as_complex(data.reshape(-1, 2))

    def _run(self, name, data, work, stream):
        self._check(data, self.real_dtype, self.complex_bytes, "data")
        tmp = []
        if work is None:
            work = self.empty_workspace(data.device)
            tmp.append(work)
        self._check_work(work, data)
        s = self._stream(stream, data, tmp)
        rc = getattr(self._lib, name)(self._h, data.data_ptr(), work.data_ptr(), ctypes.c_void_p(s.cuda_stream))
        if rc != 0:
            raise Fft3dError(rc, name)
        return data

    def r2c_inplace(self, data, work=None, stream=None):
        return self._run("fft3d_r2c_inplace", data, work, stream)

    def c2r_inplace(self, data, work=None, stream=None):
        return self._run("fft3d_c2r_inplace", data, work, stream)


class PlanC2C(Plan):
    """fft3d_plan_c2c(Nx, Ny, Nz, dtype, virtual_slabs): 3D complex-to-complex transform (argument marshalling
    only).  Forward output / inverse input are flat complex buffers in the slab layout [p][Nx][Ny/p][Nz]."""

    _PLAN_FN = "fft3d_plan_c2c"

    def c2c(self, cplx_in, direction: int, cplx_out=None, work=None, stream=None):
        self._check(cplx_in, self.complex_dtype, self.complex_bytes, "cplx_in")
        tmp = []
        if cplx_out is None:
            cplx_out = self.empty_complex(cplx_in.device)
            tmp.append(cplx_out)
        if work is None:
            work = self.empty_workspace(cplx_in.device)
            tmp.append(work)
        self._check(cplx_out, self.complex_dtype, self.complex_bytes, "cplx_out")
        self._check_work(work, cplx_in)
        s = self._stream(stream, cplx_in, tmp)
        rc = self._lib.fft3d_c2c(self._h, cplx_in.data_ptr(), cplx_out.data_ptr(), work.data_ptr(), int(direction),
                                 ctypes.c_void_p(s.cuda_stream))
        if rc != 0:
            raise Fft3dError(rc, "fft3d_c2c")
        return cplx_out

    def c2c_host(self, cplx_in: torch.Tensor, cplx_out: torch.Tensor, direction: int):
        self._check_host(cplx_in, self.complex_dtype, self.complex_bytes, "cplx_in")
        self._check_host(cplx_out, self.complex_dtype, self.complex_bytes, "cplx_out")
        rc = self._lib.fft3d_c2c_host(self._h, cplx_in.data_ptr(), cplx_out.data_ptr(), int(direction))
        if rc != 0:
            raise Fft3dError(rc, "fft3d_c2c_host")
        return cplx_out

    def to_natural(self, cplx_flat: torch.Tensor) -> torch.Tensor:
        Nx, Ny, Nz = self.shape
        L = Ny // self.p
        return cplx_flat.reshape(self.p, Nx, L, Nz).permute(1, 0, 2, 3).reshape(Nx, Ny, Nz)

    def from_natural(self, cplx_nat: torch.Tensor) -> torch.Tensor:
        Nx, Ny, Nz = self.shape
        L = Ny // self.p
        return cplx_nat.reshape(Nx, self.p, L, Nz).permute(1, 0, 2, 3).contiguous().reshape(-1)

