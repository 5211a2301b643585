"""GPU parity of the pencil layout (fft3d_plan_pencil, reading R17):
the transform's values against the fp64 CPU oracle and the position of every element against the oracle's literal
two-exchange simulation of a px x py rank grid (oracle/slab_layout.py), through the C ABI."""
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
    ((64, 64, 64), 4, 2),
    ((64, 64, 64), 1, 4),
    ((32, 48, 40), 2, 4),          # radix 3 and 5 extents, cz = 5 / 6
    ((16, 64, 256), 8, 8),
    ((128, 128, 128), 4, 4),
    ((64, 256, 256), 8, 2),        # runs the fused z+y kernels with variant 3
    ((56, 28, 112), 4, 7),         # radix-7 extents, py = 7
    ((64, 64, 64), 4, 1),          # py = 1: identical to the slab layout with p = px
]


@pytest.mark.parametrize("shape,px,py", CASES)
@pytest.mark.parametrize("dtype", [torch.float64, torch.float32])
def test_pencil_layout_matches_oracle(fft, oracle_mod, shape, px, py, dtype):
    from paper_2202_12756_b200 import inputs
    Nx, Ny, Nz = shape
    Nzh = Nz // 2 + 1
    f = inputs.uniform_grid(shape, dtype, seed=21)
    plan = fft.PlanPencil(*shape, dtype=dtype, px=px, py=py)
    assert plan.launch_names(0)[-1] == "pencil_split" and plan.launch_names(1)[0] == "pencil_merge"
    assert plan.workspace_bytes >= plan.complex_bytes
    d_in = f.cuda()
    out = plan.r2c(d_in)
    torch.cuda.synchronize()
    flat = out.cpu().numpy().astype(np.complex128)
    F_ref = oracle_mod.r2c(f.double().numpy())                         # natural order [Nx][Ny][Nzh]
    # (1) every element where the literal rank-by-rank simulation puts it
    expect = oracle_mod.simulate_pencil_transposes(F_ref, px, py) if Nx * Ny * Nzh <= 300000 else \
        oracle_mod.natural_to_pencil(F_ref, px, py)
    assert rel_l2(flat, expect) <= tol(shape, dtype)
    # (2) fft3d_index is the closed form
    rng = np.random.Generator(np.random.PCG64(5))
    for _ in range(64):
        kx, ky, kz = int(rng.integers(0, Nx)), int(rng.integers(0, Ny)), int(rng.integers(0, Nzh))
        assert plan.index(kx, ky, kz) == int(oracle_mod.pencil_index(px, py, Nx, Ny, Nz, kx, ky, kz))
    assert plan.index(0, 0, Nzh) == -1
    for kz in (0, Nz // 2):                                             # the two self-conjugate planes end up in b = 0 / py-1
        assert flat[plan.index(3, 5, kz)] == pytest.approx(F_ref[3, 5, kz], rel=0, abs=tol(shape, dtype) * np.abs(F_ref).max())
    # (3) bit-identical to the slab transform with p = px, element by element through the two index maps
    slab = fft.Plan(*shape, dtype=dtype, virtual_slabs=px)
    s_out = slab.r2c(d_in)
    assert torch.equal(torch.view_as_real(plan.to_natural(out)), torch.view_as_real(slab.to_natural(s_out)))
    # (4) inverse of an unrelated, not Hermitian-consistent spectrum (reading R8), and the round trip
    G = inputs.random_spectrum(shape, plan.complex_dtype, seed=22)
    g_ref = oracle_mod.c2r(G.to(torch.complex128).numpy(), Nz)
    g_gpu = plan.c2r(plan.from_natural(G.cuda())).cpu().numpy().astype(np.float64)
    assert rel_l2(g_gpu, g_ref) <= tol(shape, dtype)
    back = plan.c2r(out).cpu()
    assert (back - f).abs().max().item() / f.abs().max().item() <= tol(shape, dtype)
    plan.close(); slab.close()


def test_pencil_fused_variant_and_errors(fft, oracle_mod):
    from paper_2202_12756_b200 import inputs
    shape = (64, 256, 256)
    plan = fft.PlanPencil(*shape, dtype=torch.float32, px=8, py=4)
    plan.set_variant(3)
    assert plan.launch_names(0) == ("zy_r2c_fused", "x_c2c_fwd", "nyquist_unpack", "pencil_split")
    f = inputs.uniform_grid(shape, torch.float32, seed=23)
    out = plan.r2c(f.cuda())
    F_ref = oracle_mod.r2c(f.double().numpy())
    assert rel_l2(plan.to_natural(out).cpu().numpy().astype(np.complex128), F_ref) <= tol(shape, torch.float32)
    plan.close()
    for bad in ((64, 64, 64, 3, 2), (64, 64, 64, 4, 3), (64, 64, 64, 4, 0), (64, 64, 96, 4, 5)):
        with pytest.raises(fft.Fft3dError) as e:
            fft.PlanPencil(*bad[:3], dtype=torch.float32, px=bad[3], py=bad[4])
        assert e.value.status == 1
    with pytest.raises(fft.Fft3dError) as e:
        fft.PlanPencil(64, 64, 63, dtype=torch.float32, px=4, py=1)
    assert e.value.status == 2
