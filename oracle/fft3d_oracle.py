"""ctypes binding of oracle/fft3d_oracle.c -- TEST INFRASTRUCTURE, NOT THE PRODUCT.

Everything is fp64, natural order, z fastest.  Half spectra are numpy
complex128 arrays of shape (Nx, Ny, Nz//2+1) (Eq. (4)).
"""
from __future__ import annotations

import ctypes
import os
import subprocess
import threading

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "fft3d_oracle.c")
_LIB = os.path.join(_HERE, "libfft3d_oracle.so")
_lock = threading.Lock()
_lib = None


def build_oracle(force: bool = False) -> str:
    """Compile the C oracle with gcc (building the checker is not using it)."""
    with _lock:
        stale = (not os.path.exists(_LIB)) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC)
        if force or stale:
            tmp = _LIB + ".tmp.%d" % os.getpid()
            cmd = ["gcc", "-O2", "-std=c11", "-fPIC", "-shared", "-fopenmp",
                   "-ffp-contract=off", "-o", tmp, _SRC, "-lm"]
            subprocess.run(cmd, check=True)
            os.replace(tmp, _LIB)
    return _LIB


def _load():
    global _lib
    if _lib is None:
        build_oracle()
        lib = ctypes.CDLL(_LIB)
        dp = ctypes.c_void_p
        L = ctypes.c_long
        I = ctypes.c_int
        lib.oracle_dft3d_direct.argtypes = [dp, I, I, I, dp]
        lib.oracle_idft3d_direct.argtypes = [dp, I, I, I, dp]
        lib.oracle_fft1d.argtypes = [dp, dp, L, I]
        lib.oracle_r2c.argtypes = [dp, L, L, L, dp, I]
        lib.oracle_c2r.argtypes = [dp, L, L, L, dp, I]
        for nm in ("oracle_r2c_pencils_f64", "oracle_r2c_pencils_f32"):
            getattr(lib, nm).argtypes = [dp, L, L, L, I, dp, dp, dp, I]
        for nm in ("oracle_c2r_points_f64", "oracle_c2r_points_f32"):
            getattr(lib, nm).argtypes = [dp, L, L, L, L, I, dp, dp, dp, dp, I]
        lib.oracle_dft3d_c2c_direct.argtypes = [dp, I, I, I, I, dp]
        lib.oracle_c2c.argtypes = [dp, L, L, L, I, dp, I]
        lib.oracle_max_threads.restype = I
        _lib = lib
    return _lib


def _ptr(a: np.ndarray):
    return ctypes.c_void_p(a.ctypes.data)


def _check(rc: int, what: str):
    if rc != 0:
        raise RuntimeError("oracle %s failed with code %d" % (what, rc))


def max_threads() -> int:
    """Threads the oracle will actually use when asked for 'all': min(OpenMP max,
    the cores this process may run on)."""
    n = _load().oracle_max_threads()
    try:
        n = min(n, len(os.sched_getaffinity(0)))
    except AttributeError:  # pragma: no cover
        pass
    return max(1, n)


def dft3d_direct(f: np.ndarray) -> np.ndarray:
    """Eq. (1) summed term by term, O(N^6); tiny grids only."""
    f = np.ascontiguousarray(f, dtype=np.float64)
    Nx, Ny, Nz = f.shape
    out = np.empty((Nx, Ny, Nz // 2 + 1), dtype=np.complex128)
    _check(_load().oracle_dft3d_direct(_ptr(f), Nx, Ny, Nz, _ptr(out)), "dft3d_direct")
    return out


def idft3d_direct(F: np.ndarray, Nz: int) -> np.ndarray:
    """Eq. (2) with the Eq. (3) extension, real part, 1/(NxNyNz)."""
    F = np.ascontiguousarray(F, dtype=np.complex128)
    Nx, Ny, Nzh = F.shape
    assert Nzh == Nz // 2 + 1
    out = np.empty((Nx, Ny, Nz), dtype=np.float64)
    _check(_load().oracle_idft3d_direct(_ptr(F), Nx, Ny, Nz, _ptr(out)), "idft3d_direct")
    return out


def fft1d(x: np.ndarray, sign: int) -> np.ndarray:
    """Unnormalised 1D DFT with exp(sign 2 pi i jk/n) by the recursive mixed-radix FFT."""
    x = np.ascontiguousarray(x, dtype=np.complex128)
    out = np.empty_like(x)
    _check(_load().oracle_fft1d(_ptr(x), _ptr(out), x.shape[0], int(sign)), "fft1d")
    return out


def r2c(f: np.ndarray, nthreads: int = 0) -> np.ndarray:
    """Forward 3D R2C, unnormalised, natural order (Nx, Ny, Nz//2+1)."""
    f = np.ascontiguousarray(f, dtype=np.float64)
    Nx, Ny, Nz = f.shape
    out = np.empty((Nx, Ny, Nz // 2 + 1), dtype=np.complex128)
    nt = nthreads if nthreads > 0 else max_threads()
    _check(_load().oracle_r2c(_ptr(f), Nx, Ny, Nz, _ptr(out), nt), "r2c")
    return out


def c2r(F: np.ndarray, Nz: int, nthreads: int = 0) -> np.ndarray:
    """Inverse 3D C2R scaled by 1/(NxNyNz); F in natural order (Nx, Ny, Nz//2+1)."""
    F = np.ascontiguousarray(F, dtype=np.complex128)
    Nx, Ny, Nzh = F.shape
    assert Nzh == Nz // 2 + 1
    out = np.empty((Nx, Ny, Nz), dtype=np.float64)
    nt = nthreads if nthreads > 0 else max_threads()
    _check(_load().oracle_c2r(_ptr(F), Nx, Ny, Nz, _ptr(out), nt), "c2r")
    return out


def r2c_pencils(f: np.ndarray, kys, kzs, nthreads: int = 0) -> np.ndarray:
    """F(:, ky_c, kz_c) for the given (ky, kz) pairs straight from Eq. (1); f may be
    float32 (promoted) or float64.  Returns complex128 (K, Nx)."""
    assert f.dtype in (np.float32, np.float64) and f.flags.c_contiguous
    Nx, Ny, Nz = f.shape
    kys = np.ascontiguousarray(kys, dtype=np.int64)
    kzs = np.ascontiguousarray(kzs, dtype=np.int64)
    K = kys.shape[0]
    out = np.empty((K, Nx), dtype=np.complex128)
    nt = nthreads if nthreads > 0 else max_threads()
    fn = _load().oracle_r2c_pencils_f32 if f.dtype == np.float32 else _load().oracle_r2c_pencils_f64
    _check(fn(_ptr(f), Nx, Ny, Nz, K, _ptr(kys), _ptr(kzs), _ptr(out), nt), "r2c_pencils")
    return out


def c2r_points(F_flat: np.ndarray, shape, p: int, jxs, jys, jzs, nthreads: int = 0) -> np.ndarray:
    """f(jx,jy,jz) at chosen points straight from Eq. (2)+(3), reading a half spectrum
    stored in the slab layout of ``slab_index`` with p virtual slabs (p=1: natural).
    F_flat: complex64 or complex128, Nx*Ny*(Nz//2+1) entries."""
    Nx, Ny, Nz = shape
    assert F_flat.dtype in (np.complex64, np.complex128) and F_flat.flags.c_contiguous
    assert F_flat.size == Nx * Ny * (Nz // 2 + 1)
    jxs = np.ascontiguousarray(jxs, dtype=np.int64)
    jys = np.ascontiguousarray(jys, dtype=np.int64)
    jzs = np.ascontiguousarray(jzs, dtype=np.int64)
    K = jxs.shape[0]
    out = np.empty((K,), dtype=np.float64)
    nt = nthreads if nthreads > 0 else max_threads()
    fn = _load().oracle_c2r_points_f32 if F_flat.dtype == np.complex64 else _load().oracle_c2r_points_f64
    _check(fn(_ptr(F_flat), Nx, Ny, Nz, int(p), K, _ptr(jxs), _ptr(jys), _ptr(jzs), _ptr(out), nt),
           "c2r_points")
    return out


def dft3d_c2c_direct(f: np.ndarray, sign: int) -> np.ndarray:
    """The complex 3D DFT summed term by term, O(N^6): sign -1 forward (unnormalised), +1 inverse
    (1/(NxNyNz)); tiny grids only."""
    f = np.ascontiguousarray(f, dtype=np.complex128)
    Nx, Ny, Nz = f.shape
    out = np.empty_like(f)
    _check(_load().oracle_dft3d_c2c_direct(_ptr(f), Nx, Ny, Nz, int(sign), _ptr(out)), "dft3d_c2c_direct")
    return out


def c2c(f: np.ndarray, sign: int, nthreads: int = 0) -> np.ndarray:
    """3D C2C, natural order (Nx, Ny, Nz): sign -1 forward (unnormalised), +1 inverse (1/(NxNyNz))."""
    f = np.ascontiguousarray(f, dtype=np.complex128)
    Nx, Ny, Nz = f.shape
    out = np.empty_like(f)
    nt = nthreads if nthreads > 0 else max_threads()
    _check(_load().oracle_c2c(_ptr(f), Nx, Ny, Nz, int(sign), _ptr(out), nt), "c2c")
    return out
