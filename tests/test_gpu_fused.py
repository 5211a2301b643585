"""GPU parity of the fused z+y passes (csrc/fft_fused.cuh) against the fp64 CPU oracle.

variant 3 forces the fused kernels wherever they are compiled (cubic-like plans, N >= 128), so the
small shapes here run the very kernels that variant 0 picks by default at 1024^3 fp32
(tests/test_gpu_fullsize.py covers that size).  Tolerances are BASELINE.json's.
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


CASES = [
    # shape (Ny == Nz), p
    ((128, 128, 128), 4),       # no bulk z kernel for 64-point rows: skipped (the plan falls back to the unfused passes)
    ((64, 256, 256), 8),        # fewer planes than CTAs per role; ring deeper than a role's lead
    ((256, 256, 256), 8),       # BASELINE.json configs[1] shape
    ((96, 384, 384), 12),       # 3*2^a lengths (radix 3) through the fused kernels
    ((16, 512, 512), 2),        # Nx barely above the ring depth
    # the 512/1024 instantiation bench.py times at 1024^3 (default there), ring of 8 planes, on a thin slab
    ((16, 1024, 1024), 8),
    ((24, 1024, 1024), 1),
]


@pytest.mark.parametrize("shape,p", CASES)
@pytest.mark.parametrize("dtype", [torch.float64, torch.float32])
def test_fused_matches_oracle(fft, oracle_mod, shape, p, dtype):
    from paper_2202_12756_b200 import inputs
    f = inputs.uniform_grid(shape, dtype, seed=2)
    plan = fft.Plan(*shape, dtype=dtype, virtual_slabs=p)
    plan.set_variant(3)
    if "zy_r2c_fused" not in plan.launch_names(0):
        pytest.skip("fused kernels are not compiled for %s %s" % (shape, dtype))
    assert "yz_c2r_fused" in plan.launch_names(1)
    assert "z_r2c" not in plan.launch_names(0) and "z_c2r" not in plan.launch_names(1)
    assert plan.launch_impls(0)[0] == "fused_ring" and plan.launch_impls(1)[-1] == "fused_ring"
    d_in = f.cuda()
    keep = d_in.clone()
    work = plan.empty_workspace("cuda")
    d_out = plan.r2c(d_in, work=work)
    torch.cuda.synchronize()
    assert torch.equal(d_in, keep), "input must be preserved"
    F_gpu = plan.to_natural(d_out).cpu().numpy().astype(np.complex128)
    F_ref = oracle_mod.r2c(f.double().numpy())
    assert rel_l2(F_gpu, F_ref) <= tol(shape, dtype)
    # inverse of a random, NOT Hermitian-consistent half spectrum (reading R8)
    S = inputs.random_spectrum(shape, plan.complex_dtype, seed=4)
    f_ref = oracle_mod.c2r(S.to(torch.complex128).numpy(), shape[2])
    d_S = plan.from_natural(S.cuda())
    keep = d_S.clone()
    f_gpu = plan.c2r(d_S, work=work)
    torch.cuda.synchronize()
    assert torch.equal(d_S, keep), "input must be preserved"
    assert rel_l2(f_gpu.cpu().double().numpy(), f_ref) <= tol(shape, dtype)
    # round trip, reusing the same workspace (the counters are re-zeroed by every call)
    back = plan.c2r(d_out, work=work)
    err = (back.cpu().double() - f.double()).abs().max().item() / f.double().abs().max().item()
    assert err <= tol(shape, dtype)
    plan.close()


@pytest.mark.parametrize("dtype", [torch.float64, torch.float32])
def test_fused_is_deterministic_and_close_to_unfused(fft, dtype):
    """Run to run and across virtual_slabs the fused path is bit-identical (no atomics on data, reading
    R12); against the unfused kernels it may differ in the last bits only (separately compiled code)."""
    from paper_2202_12756_b200 import inputs
    shape = (128, 256, 256)
    f = inputs.normal_grid(shape, dtype, seed=6).cuda()
    ref = None
    for p in (1, 8, 32):
        for rep in range(2):
            plan = fft.Plan(*shape, dtype=dtype, virtual_slabs=p)
            plan.set_variant(3)
            assert "zy_r2c_fused" in plan.launch_names(0)
            out = plan.r2c(f)
            back = plan.c2r(out)
            nat = plan.to_natural(out).contiguous()
            if ref is None:
                ref = (nat.clone(), back.clone())
            else:
                assert torch.equal(torch.view_as_real(nat), torch.view_as_real(ref[0]))
                assert torch.equal(back, ref[1])
            plan.close()
    plan = fft.Plan(*shape, dtype=dtype, virtual_slabs=8)
    plan.set_variant(2)
    assert "z_r2c" in plan.launch_names(0)
    nat2 = plan.to_natural(plan.r2c(f))
    scale = ref[0].abs().max().item()
    eps = 1.2e-7 if dtype == torch.float32 else 2.3e-16
    assert (nat2 - ref[0]).abs().max().item() <= 64 * eps * scale
    plan.close()


def test_default_variant_picks_fused_only_where_it_wins(fft):
    small = fft.Plan(256, 256, 256, dtype=torch.float32, virtual_slabs=8)
    assert small.launch_names(0)[0] == "z_r2c"            # L2-sized problem: unfused passes
    small.set_variant(3)
    assert small.launch_names(0)[0] == "zy_r2c_fused"
    small.set_variant(1)
    assert small.launch_names(0)[0] == "z_r2c" and "x_c2c_inv_col0" not in small.launch_names(1)
    small.close()
    with pytest.raises(fft.binding.Fft3dError):
        bad = fft.Plan(64, 64, 64, dtype=torch.float32, virtual_slabs=4)
        bad.set_variant(4)


@pytest.mark.parametrize("variant", [3, 2])
def test_repeated_calls_are_bit_identical(fft, variant):
    """Race hunt by repetition: the persistent pipelines (mbarrier rings shared by two consumer groups, the
    per-plane counters of the fused kernels) must give the same bits on every call; one workspace reused."""
    from paper_2202_12756_b200 import inputs
    shape = (256, 256, 256)
    f = inputs.normal_grid(shape, torch.float32, seed=8).cuda()
    plan = fft.Plan(*shape, dtype=torch.float32, virtual_slabs=8)
    plan.set_variant(variant)
    work = plan.empty_workspace("cuda")
    out0 = plan.r2c(f, work=work).clone()
    back0 = plan.c2r(out0, work=work).clone()
    out, back = plan.empty_complex("cuda"), plan.empty_real("cuda")
    for _ in range(60):
        plan.r2c(f, out, work)
        plan.c2r(out, back, work)
        assert torch.equal(torch.view_as_real(out), torch.view_as_real(out0))
        assert torch.equal(back, back0)
    plan.close()


def test_fused_options_do_not_change_the_result(fft):
    """fft3d_set_option: any split of the SMs between the z and the y role and any ring depth gives the same bits
    (tiles are dealt dynamically: with 2 or 146 SMs in a role most CTAs of the other role find no tile at all and
    must leave through the end items), and out-of-range values are refused."""
    from paper_2202_12756_b200 import inputs
    B = fft.binding
    shape = (16, 512, 512)
    f = inputs.uniform_grid(shape, torch.float32, seed=31).cuda()
    plan = fft.Plan(*shape, dtype=torch.float32, virtual_slabs=2)
    plan.set_variant(3)
    assert plan.launch_names(0)[0] == "zy_r2c_fused"
    out0 = plan.r2c(f).clone()
    back0 = plan.c2r(out0).clone()
    for kz, ring in ((2, 8), (146, 8), (0, 8), (84, 2), (40, 3), (100, 5), (-1, 8), (-1, 2), (-1, 3)):
        plan.set_option(B.OPT_FUSED_MIXED, 1 if kz < 0 else 0)     # kz = -1: both roles in every CTA (the default)
        kz = max(kz, 0)
        plan.set_option(B.OPT_FUSED_Z_SMS_FWD, kz)
        plan.set_option(B.OPT_FUSED_Z_SMS_INV, kz)
        plan.set_option(B.OPT_FUSED_RING_PLANES, ring)
        out = plan.r2c(f)
        back = plan.c2r(out0)
        torch.cuda.synchronize()
        assert torch.equal(torch.view_as_real(out), torch.view_as_real(out0)), (kz, ring)
        assert torch.equal(back, back0), (kz, ring)
    for opt, val in ((B.OPT_FUSED_RING_PLANES, 1), (B.OPT_FUSED_RING_PLANES, 99), (B.OPT_FUSED_Z_SMS_FWD, 3), (B.OPT_FUSED_MIXED, 2), (99, 1)):
        with pytest.raises(B.Fft3dError):
            plan.set_option(opt, val)
    plan.close()


def test_fused_with_fewer_tiles_than_ctas(fft, oracle_mod):
    """Nx = 8 planes of 256 x 256: 128 z tiles and 128 y tiles for 148 CTAs -- some CTAs get one tile, some none."""
    from paper_2202_12756_b200 import inputs
    shape = (8, 256, 256)
    f = inputs.uniform_grid(shape, torch.float32, seed=32)
    plan = fft.Plan(*shape, dtype=torch.float32, virtual_slabs=1)
    plan.set_variant(3)
    if plan.launch_names(0)[0] != "zy_r2c_fused":
        plan.close()
        pytest.skip("no fused kernels for this shape")
    out = plan.r2c(f.cuda())
    back = plan.c2r(out)
    torch.cuda.synchronize()
    F_ref = oracle_mod.r2c(f.double().numpy())
    err = np.linalg.norm((plan.to_natural(out).cpu().numpy().astype(np.complex128) - F_ref).ravel()) / np.linalg.norm(F_ref.ravel())
    bound = 2e-6 * math.log2(shape[0] * shape[1] * shape[2])
    assert err <= bound
    assert (back.cpu() - f).abs().max().item() <= bound
    plan.close()


@pytest.mark.parametrize("shape", [(32, 1024, 1024), (24, 512, 512)])
def test_fused_pipeline_is_live_and_bit_identical_under_jitter(fft, shape):
    """Liveness of the dealt pipelines must not depend on timing.  FFT3D_OPT_FUSED_JITTER makes every load warp pause a
    pseudo-random time before each item, which scrambles the order in which the 148 CTAs draw and take their tiles (at
    1024 x 1024 planes, 128 phase-1 and 64 phase-2 tiles per plane on a 3-slot ring: the configuration in which a CTA could
    hold back the very phase-1 ticket its phase-2 ticket was waiting for).  A stall would end in the kernels' bounded spins
    (__trap, a CUDA error here); the result must stay the same to the bit, in both role modes and both directions."""
    from paper_2202_12756_b200 import inputs
    B = fft.binding
    f = inputs.uniform_grid(shape, torch.float32, seed=41).cuda()
    plan = fft.Plan(*shape, dtype=torch.float32, virtual_slabs=8)
    plan.set_variant(3)
    assert plan.launch_impls(0)[0] == "fused_ring" and plan.launch_impls(1)[-1] == "fused_ring"
    work = plan.empty_workspace("cuda")
    out0 = plan.r2c(f, work=work).clone()
    back0 = plan.c2r(out0, work=work).clone()
    out, back = plan.empty_complex("cuda"), plan.empty_real("cuda")
    for mixed in (1, 0):
        plan.set_option(B.OPT_FUSED_MIXED, mixed)
        for jitter in (300, 2000, 20000, 150000):
            plan.set_option(B.OPT_FUSED_JITTER, jitter)
            for _ in range(3):
                plan.r2c(f, out, work)
                plan.c2r(out0, back, work)
                torch.cuda.synchronize()
                assert torch.equal(torch.view_as_real(out), torch.view_as_real(out0)), (mixed, jitter)
                assert torch.equal(back, back0), (mixed, jitter)
    with pytest.raises(B.Fft3dError):
        plan.set_option(B.OPT_FUSED_JITTER, -1)
    plan.set_option(B.OPT_FUSED_JITTER, 0)
    plan.close()
