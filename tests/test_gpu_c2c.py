"""GPU parity of the 3D C2C transform (fft3d_plan_c2c / fft3d_c2c) against the fp64 CPU
oracle, through the C ABI.  Tolerances as for R2C/C2R: rel-L2 <= 2e-6*log2(NxNyNz) (fp32), 1e-13*log2 (fp64)."""
import math

import numpy as np
import pytest
import torch

pytestmark = pytest.mark.gpu


def tol(shape, dtype):
    n = shape[0] * shape[1] * shape[2]
    return (2e-6 if dtype == torch.float32 else 1e-13) * math.log2(n)


def rel_l2(a, b):
    return float(np.linalg.norm((np.asarray(a) - np.asarray(b)).ravel()) / np.linalg.norm(np.asarray(b).ravel()))


@pytest.fixture(scope="module")
def fft():
    import paper_2202_12756_b200 as m
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    m.load_library()
    return m


CASES = [
    ((64, 256, 256), 8),         # Nz == Ny: also runs fused (variant 3)
    ((48, 384, 384), 12),
    ((32, 32, 128), 4),
    ((16, 64, 256), 8),
    ((64, 16, 192), 2),          # radix-3 rows
    ((48, 96, 384), 3),
    ((128, 128, 128), 8),
    ((32, 256, 1024), 16),       # 64 KiB row tiles; y pass through the TMA kernels
    ((8, 64, 1536), 1),          # rows whose threads span two warps (no Hermitian step, so allowed)
    ((32, 32, 16), 2),           # rows shorter than 1 KiB: the plain-load row kernel
    ((16, 24, 64), 4),
    ((12, 20, 28), 2),           # radix 3, 5 and 7 lengths, Nz not a multiple of the bulk tile
    ((6, 20, 40), 2),
    ((64, 64, 96), 8),
    ((20, 6, 1024), 2),
    ((6, 6, 128), 2),            # rows of >= 1 KiB, but Nx*Ny = 36 rows are not whole 16- or 32-row tiles: plain-load rows
    ((6, 6, 256), 3),
]


PLAIN_ROWS = {(6, 6, 128), (6, 6, 256), (32, 32, 16), (12, 20, 28)}


@pytest.mark.parametrize("shape,p", CASES)
@pytest.mark.parametrize("dtype", [torch.float64, torch.float32])
@pytest.mark.parametrize("variant", [2, 3])     # 2: three passes per direction; 3: z+y fused wherever compiled (Nz == Ny)
def test_c2c_matches_oracle(fft, oracle_mod, shape, p, dtype, variant):
    from paper_2202_12756_b200 import inputs
    try:
        plan = fft.PlanC2C(*shape, dtype=dtype, virtual_slabs=p)
    except fft.Fft3dError as e:
        assert e.status == 2
        pytest.skip("no C2C row kernel for %s %s" % (shape, dtype))
    plan.set_variant(variant)
    fused = plan.launch_names(0)[0] == "zy_c2c_fused_fwd"
    if variant == 3 and not fused:
        plan.close()
        pytest.skip("no fused C2C kernels for %s %s" % (shape, dtype))
    assert fused == (variant == 3)
    if shape in PLAIN_ROWS:          # the path these cases were written for must be the one that runs
        assert plan.launch_impls(0)[0] == "plain" and plan.launch_impls(1)[2] == "plain", plan.launch_impls(0)
    cd = plan.complex_dtype
    f = inputs.complex_grid(shape, cd, seed=11)
    d_in = f.cuda().reshape(-1)
    keep = d_in.clone()
    out = plan.c2c(d_in, -1)
    torch.cuda.synchronize()
    assert torch.equal(torch.view_as_real(d_in), torch.view_as_real(keep)), "input must be preserved"
    F_gpu = plan.to_natural(out).cpu().numpy().astype(np.complex128)
    F_ref = oracle_mod.c2c(f.to(torch.complex128).numpy(), -1)
    assert rel_l2(F_gpu, F_ref) <= tol(shape, dtype)
    # slab layout == fft3d_index
    flat = out.cpu().numpy()
    rng = np.random.Generator(np.random.PCG64(2))
    for _ in range(32):
        kx, ky, kz = (int(rng.integers(0, n)) for n in shape)
        off = plan.index(kx, ky, kz)
        L = shape[1] // p
        assert off == (((ky // L) * shape[0] + kx) * L + ky % L) * shape[2] + kz
        assert flat[off] == F_gpu[kx, ky, kz].astype(flat.dtype)
    assert plan.index(0, 0, shape[2]) == -1
    # inverse of an unrelated field, then the round trip
    g = inputs.complex_grid(shape, cd, seed=12)
    g_ref = oracle_mod.c2c(g.to(torch.complex128).numpy(), +1)
    g_gpu = plan.c2c(plan.from_natural(g.cuda()), +1).reshape(shape).cpu().numpy().astype(np.complex128)
    assert rel_l2(g_gpu, g_ref) <= tol(shape, dtype)
    back = plan.c2c(out, +1).reshape(shape).cpu()
    err = (back - f).abs().max().item() / f.abs().max().item()
    assert err <= tol(shape, dtype)
    if fused:
        assert plan.launch_names(0) == ("zy_c2c_fused_fwd", "x_c2c_fwd")
        assert plan.launch_names(1) == ("x_c2c_inv", "yz_c2c_fused_inv")
    else:
        assert plan.launch_names(0) == ("z_c2c_fwd", "y_c2c_fwd", "x_c2c_fwd")
        assert plan.launch_names(1) == ("x_c2c_inv", "y_c2c_inv", "z_c2c_inv")
    plan.close()


def test_plan_kinds_do_not_mix(fft):
    c = fft.PlanC2C(32, 32, 128, dtype=torch.float32, virtual_slabs=2)
    r = fft.Plan(32, 32, 128, dtype=torch.float32, virtual_slabs=2)
    x = torch.zeros(32 * 32 * 128, dtype=torch.complex64, device="cuda")
    with pytest.raises(fft.Fft3dError):
        fft.PlanC2C.c2c(r, torch.zeros(r.n_complex, dtype=torch.complex64, device="cuda"), -1)
    lib = fft.load_library()
    w = c.empty_workspace("cuda")
    assert lib.fft3d_r2c(c._h, x.data_ptr(), x.data_ptr(), w.data_ptr(), None) == 1      # FFT3D_EINVAL
    assert lib.fft3d_c2c(c._h, x.data_ptr(), x.data_ptr(), w.data_ptr(), -1, None) == 1  # in == out rejected
    assert lib.fft3d_c2c(c._h, x.data_ptr(), w.data_ptr(), w.data_ptr(), 0, None) == 1   # bad direction
    with pytest.raises(fft.Fft3dError) as e:
        fft.PlanC2C(32, 32, 44, dtype=torch.float32, virtual_slabs=2)                     # 44 = 11*4: no kernel
    assert e.value.status == 2
    short = fft.PlanC2C(32, 32, 16, dtype=torch.float32, virtual_slabs=2)                 # short rows: plain-load rows
    assert short.launch_impls(0)[0] == "plain" and short.launch_impls(1)[-1] == "plain"
    assert c.launch_impls(0)[0] == "bulk"
    short.close()
    c.close(); r.close()


def test_c2c_512_full_oracle_and_1024_properties(fft, oracle_mod):
    """512^3 fp32 against the full fp64 oracle; 1024^3 fp32 (8 GiB per array) by properties that hold at any
    size: a sum of plane waves gives exactly those spikes (closed form), Parseval, round trip."""
    from paper_2202_12756_b200 import inputs
    shape, p = (512, 512, 512), 8
    plan = fft.PlanC2C(*shape, dtype=torch.float32, virtual_slabs=p)
    f = inputs.complex_grid(shape, torch.complex64, seed=21)
    out = plan.c2c(f.cuda().reshape(-1), -1)
    F_gpu = plan.to_natural(out).cpu().numpy()
    F_ref = oracle_mod.c2c(f.to(torch.complex128).numpy(), -1)
    num = np.linalg.norm((F_gpu - F_ref).ravel())
    assert num / np.linalg.norm(F_ref.ravel()) <= tol(shape, torch.float32)
    del F_ref, F_gpu, out
    plan.close()

    n = 1024
    shape = (n, n, n)
    plan = fft.PlanC2C(*shape, dtype=torch.float32, virtual_slabs=64)
    assert plan.launch_names(0)[0] == "zy_c2c_fused_fwd"      # the default at this size
    modes = [((3, 1000, 17), 1.5 - 0.5j), ((512, 0, 1023), -0.75 + 2.0j), ((77, 301, 640), 0.25 + 0.125j)]
    ax = torch.arange(n, device="cuda", dtype=torch.float64)
    f = torch.zeros(shape, dtype=torch.complex64, device="cuda")
    for (kx, ky, kz), amp in modes:                       # separable phases built in fp64, rounded once
        ex = torch.exp(2j * math.pi * ((ax * kx) % n) / n)
        ey = torch.exp(2j * math.pi * ((ax * ky) % n) / n)
        ez = torch.exp(2j * math.pi * ((ax * kz) % n) / n)
        for x0 in range(0, n, 128):
            blk = amp * ex[x0:x0 + 128, None, None] * ey[None, :, None] * ez[None, None, :]
            f[x0:x0 + 128] += blk.to(torch.complex64)
    work = plan.empty_workspace("cuda")
    out = plan.c2c(f.reshape(-1), -1, work=work)
    energy_in = sum((f[i].abs().double() ** 2).sum().item() for i in range(n))
    energy_out = sum((out[i * n * n:(i + 1) * n * n].abs().double() ** 2).sum().item() for i in range(n))
    assert abs(energy_out / n ** 3 - energy_in) <= 1e-5 * energy_in
    peak = 0.0
    for (kx, ky, kz), amp in modes:
        got = out[plan.index(kx, ky, kz)].item()
        assert abs(got - amp * n ** 3) <= 2e-5 * abs(amp) * n ** 3
        peak = max(peak, abs(amp) * n ** 3)
        out[plan.index(kx, ky, kz)] = 0
    rest = max(out[i * n * n:(i + 1) * n * n].abs().max().item() for i in range(n))
    assert rest <= 2e-5 * peak                             # everything else is rounding noise
    for (kx, ky, kz), amp in modes:
        out[plan.index(kx, ky, kz)] = amp * n ** 3
    back = plan.c2c(out, +1, work=work).reshape(shape)
    err = max((back[i] - f[i]).abs().max().item() for i in range(n))
    fmax = max(f[i].abs().max().item() for i in range(n))
    assert err / fmax <= tol(shape, torch.float32)         # round-trip max-abs error relative to max|f|
    plan.close()


def test_c2c_host_entry_point(fft, oracle_mod):
    from paper_2202_12756_b200 import inputs
    shape, p = (32, 64, 256), 4
    plan = fft.PlanC2C(*shape, dtype=torch.float64, virtual_slabs=p)
    f = inputs.complex_grid(shape, torch.complex128, seed=31)
    out = torch.empty(plan.n_complex, dtype=torch.complex128)
    plan.c2c_host(f.reshape(-1).contiguous(), out, -1)
    F_ref = oracle_mod.c2c(f.numpy(), -1)
    assert rel_l2(plan.to_natural(out).numpy(), F_ref) <= tol(shape, torch.float64)
    back = torch.empty_like(out)
    plan.c2c_host(out, back, +1)
    assert (back.reshape(shape) - f).abs().max().item() <= tol(shape, torch.float64) * 2
    plan.close()
