"""GPU parity: the CUDA path (through the C ABI) against the fp64 CPU oracle, element by element.

Tolerances are BASELINE.json's: relative L2 error <= 2e-6*log2(NxNyNz) in fp32 and
<= 1e-13*log2(NxNyNz) in fp64, over all stored entries; round-trip max-abs error / max|f|
within the same bound.
"""
import math

import numpy as np
import pytest
import torch

pytestmark = pytest.mark.gpu


def tol(shape, dtype):
    n = shape[0] * shape[1] * shape[2]
    return (2e-6 if dtype == torch.float32 else 1e-13) * math.log2(n)


def rel_l2(a, b):
    a = np.asarray(a)
    b = np.asarray(b)
    return float(np.linalg.norm((a - b).ravel()) / np.linalg.norm(b.ravel()))


@pytest.fixture(scope="module")
def fft():
    import paper_2202_12756_b200 as m
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    m.load_library()
    return m


def run_forward(fft, f_host, p, variant=0):
    """f_host: torch CPU real tensor.  Returns (natural-order spectrum as numpy c128, plan, flat device out)."""
    shape = tuple(f_host.shape)
    plan = fft.Plan(*shape, dtype=f_host.dtype, virtual_slabs=p)
    plan.set_variant(variant)
    d_in = f_host.cuda()
    keep = d_in.clone()
    out = plan.r2c(d_in)
    torch.cuda.synchronize()
    assert torch.equal(d_in, keep), "input must be preserved"
    nat = plan.to_natural(out).cpu().numpy().astype(np.complex128)
    return nat, plan, out


SMALL = [
    # shape, p
    ((64, 64, 64), 4),          # BASELINE.json configs[0] shape
    ((32, 16, 128), 2),
    ((16, 64, 8), 8),
    ((8, 4, 16), 1),
    ((48, 96, 24), 3),          # radix-3 on every axis (z half: 12)
    ((96, 48, 64), 6),
    ((24, 12, 192), 4),
    ((128, 256, 32), 16),
    ((4, 6, 8), 2),
    ((256, 128, 256), 2),       # several TMA boxes per tile on x, slab boxes spanning whole slabs on y
    ((64, 512, 64), 1),         # L = 512 > 256: slab boxes are parts of one slab
    ((384, 192, 48), 12),       # 3*2^a lengths through the TMA path
    ((1536, 8, 32), 4),         # Nx = 1536: x passes as two 768-point half tiles with the shifted windows of odd rows
    ((1536, 32, 64), 16),
    ((40, 80, 160), 4),         # 5*2^a lengths on every axis (radix-5 leaf; z half: 80)
    ((20, 20, 40), 1),
    ((320, 160, 80), 8),
    ((80, 40, 1280), 4),        # 640-point rows through the bulk z kernel
    ((56, 112, 224), 4),        # 7*2^a lengths on every axis (radix-7 leaf; z half: 112)
    ((28, 28, 56), 1),
    ((448, 224, 112), 8),
    ((112, 56, 1792), 4),       # 896-point rows
    ((1792, 16, 56), 4),        # Nx = 1792
    ((64, 192, 64), 32),        # L = 6: the two-class shifted windows (four classes need L % 4 == 0)
    ((2048, 8, 32), 2),         # Nx = 2048: inverse x pass as four 512-point quarter tiles + a radix-4 combine
    ((2048, 16, 64), 4),
    ((8, 2048, 16), 4),         # Ny = 2048: y passes as two half tiles + a radix-2 combine (fft_split2.cuh)
    ((128, 2048, 16), 128),     # ... with slab boxes spanning several virtual slabs (L = 16)
]


# Thin slabs that run the very FFT-1024 kernel instantiations bench.py times at 1024^3 (full oracle, < 1 s each):
# shape, p, variant, {launch name: implementation that must be selected}
BENCH_KERNELS = [
    # F3 with four row classes l % 4 and every thin tile (columns M-2, M-1 / M-1 / 0), I1 + the col0 launch
    ((1024, 16, 32), 4, 0, {"x_c2c_fwd": "tma", "x_c2c_inv": "tma", "x_c2c_inv_col0": "plain"}),
    ((1024, 32, 64), 2, 0, {"x_c2c_fwd": "tma", "x_c2c_inv": "tma"}),
    ((1024, 8, 32), 4, 0, {"x_c2c_fwd": "tma", "x_c2c_inv": "tma"}),       # L = 2: the two-class windows
    # FFT-1024 Y passes: slab boxes inside one slab (L = 1024) and spanning several (L = 64)
    ((16, 1024, 32), 1, 0, {"y_c2c_fwd": "tma", "y_c2c_inv": "tma"}),
    ((16, 1024, 32), 16, 0, {"y_c2c_fwd": "tma", "y_c2c_inv": "tma"}),
    # 512-point rows through the bulk z kernel next to 1024-point y lines, unfused
    ((8, 1024, 1024), 8, 2, {"z_r2c": "bulk", "y_c2c_fwd": "tma", "z_c2r": "bulk", "y_c2c_inv": "tma"}),
    # 1536 / 2048 on x and y at bench-like row lengths
    # (fp32 implementation, fp64 implementation) where they differ: fp64 whole tiles still leave room for a ring
    ((1536, 16, 32), 4, 0, {"x_c2c_fwd": ("tma_split2", "tma"), "x_c2c_inv": ("tma_split2", "tma")}),
    ((2048, 16, 32), 4, 0, {"x_c2c_inv": ("tma_split4", "tma")}),
    ((8, 2048, 32), 8, 0, {"y_c2c_fwd": "tma_split2", "y_c2c_inv": "tma_split2"}),
    ((16, 1536, 32), 16, 0, {"y_c2c_fwd": "tma", "y_c2c_inv": "tma"}),
]


@pytest.mark.parametrize("shape,p,variant,impls", BENCH_KERNELS)
@pytest.mark.parametrize("dtype", [torch.float32, torch.float64])
def test_bench_kernel_instantiations_match_full_oracle(fft, oracle_mod, shape, p, variant, impls, dtype):
    """Element-wise parity, against the FULL oracle, of the kernels that make up bench.py's step; the plan must
    select the implementation named (fft3d_launch_impl), so a silent fallback fails the test."""
    from paper_2202_12756_b200 import inputs
    f = inputs.uniform_grid(shape, dtype, seed=11)
    plan = fft.Plan(*shape, dtype=dtype, virtual_slabs=p)
    plan.set_variant(variant)
    got = dict(zip(plan.launch_names(0) + plan.launch_names(1), plan.launch_impls(0) + plan.launch_impls(1)))
    for name, impl in impls.items():
        if isinstance(impl, tuple):
            impl = impl[0] if dtype == torch.float32 else impl[1]
        assert got.get(name) == impl, (name, impl, got)
    d_in = f.cuda()
    d_out = plan.r2c(d_in)
    F_gpu = plan.to_natural(d_out).cpu().numpy().astype(np.complex128)
    F_ref = oracle_mod.r2c(f.double().numpy())
    assert rel_l2(F_gpu, F_ref) <= tol(shape, dtype)
    # worst single entry, relative to the rms of the spectrum (white-noise input: every entry is O(rms))
    rms = np.sqrt(np.mean(np.abs(F_ref) ** 2))
    assert np.abs(F_gpu - F_ref).max() <= 8 * tol(shape, dtype) * rms
    S = inputs.random_spectrum(shape, plan.complex_dtype, seed=12)
    f_ref = oracle_mod.c2r(S.to(torch.complex128).numpy(), shape[2])
    f_gpu = plan.c2r(plan.from_natural(S.cuda())).cpu().double().numpy()
    assert rel_l2(f_gpu, f_ref) <= tol(shape, dtype)
    assert np.abs(f_gpu - f_ref).max() <= 8 * tol(shape, dtype) * np.sqrt(np.mean(f_ref ** 2))
    back = plan.c2r(d_out)
    err = (back.cpu().double() - f.double()).abs().max().item() / f.double().abs().max().item()
    assert err <= tol(shape, dtype)
    plan.close()


@pytest.mark.parametrize("shape,p", SMALL)
@pytest.mark.parametrize("dtype", [torch.float64, torch.float32])
@pytest.mark.parametrize("variant", [0, 1])     # 0: TMA-pipelined strided passes where possible, 1: plain-load kernels
def test_r2c_and_c2r_match_oracle(fft, oracle_mod, shape, p, dtype, variant):
    from paper_2202_12756_b200 import inputs
    f = inputs.uniform_grid(shape, dtype, seed=0)
    F_ref = oracle_mod.r2c(f.double().numpy())
    F_gpu, plan, d_out = run_forward(fft, f, p, variant)
    assert rel_l2(F_gpu, F_ref) <= tol(shape, dtype)
    # no single entry off by more than a few bounds of the spectrum's rms (a norm alone would let one wrong entry through)
    assert np.abs(F_gpu - F_ref).max() <= 8 * tol(shape, dtype) * np.sqrt(np.mean(np.abs(F_ref) ** 2))
    # the slab layout agrees with fft3d_index on a sample of entries
    rng = np.random.Generator(np.random.PCG64(1))
    flat = d_out.cpu().numpy()
    for _ in range(64):
        kx, ky, kz = (int(rng.integers(0, n)) for n in (shape[0], shape[1], shape[2] // 2 + 1))
        off = plan.index(kx, ky, kz)
        assert off == int(oracle_mod.slab_index(p, *shape, kx, ky, kz))
        assert flat[off] == F_gpu[kx, ky, kz].astype(flat.dtype)
    assert plan.index(shape[0], 0, 0) == -1
    # inverse of a random, NOT Hermitian-consistent half spectrum (reading R8)
    S = inputs.random_spectrum(shape, plan.complex_dtype, seed=3)
    f_ref = oracle_mod.c2r(S.to(torch.complex128).numpy(), shape[2])
    d_S = plan.from_natural(S.cuda())
    keep = d_S.clone()
    f_gpu = plan.c2r(d_S)
    torch.cuda.synchronize()
    assert torch.equal(d_S, keep), "input must be preserved"
    assert rel_l2(f_gpu.cpu().double().numpy(), f_ref) <= tol(shape, dtype)
    assert np.abs(f_gpu.cpu().double().numpy() - f_ref).max() <= 8 * tol(shape, dtype) * np.sqrt(np.mean(f_ref ** 2))
    # round trip
    back = plan.c2r(d_out)
    err = (back.cpu().double() - f.double()).abs().max().item() / f.double().abs().max().item()
    assert err <= tol(shape, dtype)


def test_config0_64cubed_fp64_p4(fft, oracle_mod):
    """BASELINE.json configs[0]: 64^3 fp64 uniform[-1,1) seed 0, p=4, 64x64x33 half spectrum."""
    from paper_2202_12756_b200 import inputs
    shape = (64, 64, 64)
    f = inputs.uniform_grid(shape, torch.float64, seed=0)
    F_ref = oracle_mod.r2c(f.numpy())
    F_gpu, plan, d_out = run_forward(fft, f, 4)
    assert F_gpu.shape == (64, 64, 33)
    assert rel_l2(F_gpu, F_ref) <= 1e-13 * 18
    # Parseval with half-spectrum weights and Hermitian symmetry of the self-conjugate planes
    w = np.full(33, 2.0)
    w[0] = w[32] = 1.0
    assert abs((w * np.abs(F_gpu) ** 2).sum() / 64 ** 3 - (f.numpy() ** 2).sum()) <= 1e-11 * (f.numpy() ** 2).sum()
    for kz in (0, 32):
        P = F_gpu[:, :, kz]
        Mi = np.conj(P[(-np.arange(64)) % 64][:, (-np.arange(64)) % 64])
        assert np.abs(P - Mi).max() <= 1e-10
    back = plan.c2r(d_out).cpu()
    assert (back - f).abs().max().item() <= 1e-13 * 18


@pytest.mark.parametrize("dtype", [torch.float64, torch.float32])
def test_results_do_not_depend_on_virtual_slabs(fft, dtype):
    """Reading R12: after un-permuting, results are bit-identical across p."""
    from paper_2202_12756_b200 import inputs
    shape = (32, 64, 32)
    f = inputs.normal_grid(shape, dtype, seed=5)
    ref = None
    for variant in (0, 1):
        for p in (1, 2, 8, 32):
            F, plan, d_out = run_forward(fft, f, p, variant)
            back = plan.c2r(d_out).cpu()
            if ref is None:
                ref = (F, back)
            else:
                assert np.array_equal(F, ref[0]) and torch.equal(back, ref[1])
    # and run to run
    F2, _, _ = run_forward(fft, f, 1)
    assert np.array_equal(F2, ref[0])


@pytest.mark.parametrize("dtype", [torch.float64, torch.float32])
def test_paper_worked_example_eq5(fft, dtype):
    """PAPER.md:100 Eq. (5): 8 spikes of +-i N^3 (tests/golden/eq5_spikes.txt); the fp64 round
    trip recovers the field to ~1e-14 relative to its amplitude."""
    from paper_2202_12756_b200 import inputs
    from test_oracle_pins import load_eq5_spikes
    N = 64
    f = inputs.eq5_grid((N, N, N), dtype)
    F, plan, d_out = run_forward(fft, f, 8)
    expect = np.zeros_like(F)
    for kx, ky, kz, re, im in load_eq5_spikes():
        expect[kx % N, ky % N, kz] = (re + 1j * im) * N ** 3
    eps = 1e-6 if dtype == torch.float32 else 1e-14
    assert np.abs(F - expect).max() <= 40 * eps * N ** 3
    back = plan.c2r(d_out).cpu().double()
    assert (back - f.double()).abs().max().item() <= (1e-13 if dtype == torch.float64 else 2e-5)


@pytest.mark.parametrize("dtype", [torch.float32, torch.float64])
def test_config1_256cubed_sinusoids(fft, oracle_mod, dtype):
    """BASELINE.json configs[1]: 256^3, 16 sinusoids + noise, p=8, both precisions."""
    from paper_2202_12756_b200 import inputs
    shape = (256, 256, 256)
    f, modes = inputs.sinusoid_grid(shape, dtype, seed=0)
    F_ref = oracle_mod.r2c(f.double().numpy())
    F_gpu, plan, d_out = run_forward(fft, f, 8)
    assert rel_l2(F_gpu, F_ref) <= tol(shape, dtype)
    back = plan.c2r(d_out).cpu().double()
    assert (back - f.double()).abs().max().item() / f.double().abs().max().item() <= tol(shape, dtype)
    f_ref = oracle_mod.c2r(F_ref, 256)
    S = plan.from_natural(torch.from_numpy(F_ref).to(plan.complex_dtype).cuda())
    assert rel_l2(plan.c2r(S).cpu().double().numpy(), f_ref) <= tol(shape, dtype)


def test_host_entry_points(fft, oracle_mod):
    from paper_2202_12756_b200 import inputs
    shape = (32, 32, 64)
    f = inputs.uniform_grid(shape, torch.float32, seed=2)
    plan = fft.Plan(*shape, dtype=torch.float32, virtual_slabs=4)
    h_in = f.pin_memory()
    h_spec = torch.empty(plan.n_complex, dtype=torch.complex64).pin_memory()
    plan.r2c_host(h_in, h_spec)
    F_ref = oracle_mod.r2c(f.double().numpy())
    assert rel_l2(plan.to_natural(h_spec).numpy().astype(np.complex128), F_ref) <= tol(shape, torch.float32)
    h_back = torch.empty(shape, dtype=torch.float32).pin_memory()
    plan.c2r_host(h_spec, h_back)
    assert (h_back - f).abs().max().item() <= tol(shape, torch.float32)


def test_argument_errors(fft):
    with pytest.raises(fft.Fft3dError) as e:
        fft.Plan(64, 64, 63)
    assert e.value.status == 2
    with pytest.raises(fft.Fft3dError) as e:
        fft.Plan(64, 64, 64, virtual_slabs=3)
    assert e.value.status == 1
    with pytest.raises(fft.Fft3dError) as e:
        fft.Plan(44, 64, 64)                       # 44 = 11*4: no radix 11
    assert e.value.status == 2
    plan = fft.Plan(16, 16, 16, dtype=torch.float32)
    x = plan.empty_real()
    with pytest.raises(ValueError):
        plan.r2c(x.double())
    # aliasing is rejected
    import ctypes
    w = plan.empty_workspace()
    rc = plan._lib.fft3d_r2c(plan._h, x.data_ptr(), x.data_ptr(), w.data_ptr(), ctypes.c_void_p(0))
    assert rc == 1
