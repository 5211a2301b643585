"""The padded in-place layout (fft3d_plan_inplace): rows of Nz+2 reals, the half
spectrum overwrites the field.  Same oracle, inputs and outputs viewed through the padded pitch; tolerances are
BASELINE.json's.  The arithmetic is that of the out-of-place kernels, so the results must also be bit-identical to
an out-of-place plan's (unfused variants)."""
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
    ((64, 64, 64), 4),            # BASELINE.json configs[0] shape
    ((256, 256, 256), 8),         # configs[1] shape
    ((1024, 16, 32), 4),          # thin slab with FFT-1024 x passes (TMA) next to the padded rows
    ((16, 1024, 64), 1),          # natural order, 1024-point y lines read at the padded pitch
    ((8, 4, 16), 2),
    ((48, 96, 24), 3),            # radix 3; odd M + 1 = 13
    ((40, 20, 80), 4),            # radix 5
    ((32, 2048, 16), 2),
]


@pytest.mark.parametrize("shape,p", CASES)
@pytest.mark.parametrize("dtype", [torch.float32, torch.float64])
def test_inplace_matches_oracle_and_out_of_place(fft, oracle_mod, shape, p, dtype):
    from paper_2202_12756_b200 import inputs
    Nx, Ny, Nz = shape
    f = inputs.uniform_grid(shape, dtype, seed=31)
    plan = fft.PlanInplace(*shape, dtype=dtype, virtual_slabs=p)
    assert plan.launch_impls(0)[0] == "plain" and plan.launch_impls(0)[1] == "plain"
    assert plan.complex_bytes == Nx * Ny * (Nz + 2) * f.element_size()
    data = plan.empty_data("cuda")
    data.fill_(float("nan"))                              # the two pad reals of every row must never matter
    data[:, :, :Nz] = f.cuda()
    work = plan.empty_workspace("cuda")
    plan.r2c_inplace(data, work)
    spec = plan.as_spectrum(data)
    F_gpu = plan.to_natural(spec).cpu().numpy().astype(np.complex128)
    F_ref = oracle_mod.r2c(f.double().numpy())
    assert rel_l2(F_gpu, F_ref) <= tol(shape, dtype)
    # bit-identical to the out-of-place transform (plain-load variant: the same kernels, dense pitch)
    oop = fft.Plan(*shape, dtype=dtype, virtual_slabs=p)
    oop.set_variant(1)
    ref = oop.r2c(f.cuda())
    assert torch.equal(torch.view_as_real(spec), torch.view_as_real(ref))
    # round trip in place
    plan.c2r_inplace(data, work)
    back = data[:, :, :Nz].cpu().double()
    assert (back - f.double()).abs().max().item() / f.double().abs().max().item() <= tol(shape, dtype)
    # inverse of a random, NOT Hermitian-consistent spectrum (reading R8)
    S = inputs.random_spectrum(shape, plan.complex_dtype, seed=32)
    f_ref = oracle_mod.c2r(S.to(torch.complex128).numpy(), Nz)
    spec.copy_(plan.from_natural(S.cuda()))
    plan.c2r_inplace(data, work)
    assert rel_l2(data[:, :, :Nz].cpu().double().numpy(), f_ref) <= tol(shape, dtype)
    plan.close()
    oop.close()


def test_inplace_argument_errors(fft):
    plan = fft.PlanInplace(32, 32, 32, dtype=torch.float32, virtual_slabs=2)
    oop = fft.Plan(32, 32, 32, dtype=torch.float32, virtual_slabs=2)
    lib = fft.load_library()
    d, w = plan.empty_data("cuda"), plan.empty_workspace("cuda")
    assert lib.fft3d_r2c(plan._h, d.data_ptr(), w.data_ptr(), w.data_ptr(), None) == 1          # wrong entry point
    assert lib.fft3d_r2c_inplace(oop._h, d.data_ptr(), w.data_ptr(), None) == 1
    assert lib.fft3d_r2c_inplace(plan._h, d.data_ptr(), d.data_ptr(), None) == 1                # workspace aliases the data
    with pytest.raises(fft.Fft3dError):
        fft.PlanInplace(32, 32, 31)
    plan.close(); oop.close()
