"""fft3d_r2c_static -- the entry point for callers that cannot allocate device memory -- against the planned path.

Why the entry point exists: fft3d_plan cudaMalloc's its twiddle tables and fft3d_r2c needs an array-sized workspace from
the caller.  A plug-in inside an application whose memory pool owns the whole card, the inner loop of a solver or server
where cudaMalloc/cudaFree are banned (they stall the device and can fail on a full card), a process on a fixed memory
budget: none of them can supply either.  fft3d_r2c_static takes only the input and the output and keeps its scratch in
a 17 MiB array that is part of the library image.

What is checked: its spectrum agrees with fft3d_plan + fft3d_r2c (default kernels) within the parity tolerance of
tests/test_gpu_parity.py, on consecutive calls that share the built-in scratch -- same shape twice (the second call
finds the first one's tables and stale intermediate data in the array), then other shapes and the other precision (the
tables must be replaced) -- and that a grid beyond the limit is refused with FFT3D_EWORKSPACE before anything runs.

This file is named so that pytest collects it last: with `-x` a failure here cannot hide another test.  It must pass
alone in a fresh process (its first call is then the first use of the library on the device) and after the whole suite.
"""
import math

import pytest
import torch

pytestmark = pytest.mark.gpu


def tol(shape, dtype):                      # the bound of tests/test_gpu_parity.py (BASELINE.json's)
    n = shape[0] * shape[1] * shape[2]
    return (2e-6 if dtype == torch.float32 else 1e-13) * math.log2(n)


@pytest.fixture(scope="module")
def fft():
    import paper_2202_12756_b200 as m
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    m.load_library()
    return m


def planned(fft, d_in, p, variant=0):
    """The existing path: a plan, a torch-allocated workspace, fft3d_r2c."""
    plan = fft.Plan(*d_in.shape, dtype=d_in.dtype, virtual_slabs=p)
    plan.set_variant(variant)
    out = plan.r2c(d_in)
    torch.cuda.synchronize()
    plan.close()
    return out


def check(fft, shape, p, dtype, seed):
    from paper_2202_12756_b200 import binding, inputs
    d_in = inputs.uniform_grid(shape, dtype, seed=seed).cuda()
    keep = d_in.clone()
    cdt = torch.complex64 if dtype == torch.float32 else torch.complex128
    # the caller owns the output; NaNs make sure every entry is really written
    out = torch.full((shape[0] * shape[1] * (shape[2] // 2 + 1),), float("nan"), dtype=cdt, device="cuda")
    binding.r2c_static(d_in, out, virtual_slabs=p)
    torch.cuda.synchronize()
    assert torch.equal(d_in, keep), "input must be preserved"
    ref = planned(fft, d_in, p)
    a, b = out.to(torch.complex128), ref.to(torch.complex128)
    assert bool(torch.isfinite(a.real).all()) and bool(torch.isfinite(a.imag).all())
    rel = (torch.linalg.vector_norm(a - b) / torch.linalg.vector_norm(b)).item()
    assert rel <= tol(shape, dtype), (shape, p, dtype, rel)
    # worst single entry, against the spectrum's rms (the bound the parity tests use for entries)
    rms = (torch.linalg.vector_norm(b) / math.sqrt(b.numel())).item()
    worst = (a - b).abs().max().item()
    assert worst <= 8 * tol(shape, dtype) * rms, (shape, p, dtype, worst, rms)
    # same kernels and same tables as the plain-load variant of the planned path: identical bits
    assert torch.equal(out, planned(fft, d_in, p, variant=1))
    return out


def test_two_calls_in_a_row_match_the_planned_path(fft):
    shape, p = (64, 64, 64), 4                                   # BASELINE.json configs[0] shape
    first = check(fft, shape, p, torch.float64, seed=0)
    second = check(fft, shape, p, torch.float64, seed=1)         # scratch still holds call 1's tables and intermediate
    assert not torch.equal(first, second)
    # and once more with the first input: leftovers of call 2 in the scratch must not show
    assert torch.equal(check(fft, shape, p, torch.float64, seed=0), first)


def test_changing_shape_and_precision_between_calls(fft):
    seq = [((48, 96, 24), 3, torch.float32),                     # radix 3
           ((64, 64, 64), 4, torch.float32),
           ((40, 80, 160), 4, torch.float64),                    # radix 5, larger tables than the call before
           ((8, 4, 16), 1, torch.float32),                       # tiny: most of the scratch keeps the previous call's data
           ((128, 128, 256), 8, torch.float32),                  # exactly 16 MiB of intermediate array: the documented maximum
           ((64, 64, 64), 4, torch.float64)]
    for k, (shape, p, dtype) in enumerate(seq):
        check(fft, shape, p, dtype, seed=10 + k)


def test_calls_do_not_allocate_device_memory(fft):
    from paper_2202_12756_b200 import binding, inputs
    shape = (64, 64, 64)
    d_in = inputs.uniform_grid(shape, torch.float32, seed=5).cuda()
    out = torch.empty(64 * 64 * 33, dtype=torch.complex64, device="cuda")
    binding.r2c_static(d_in, out, virtual_slabs=2)               # first use on this device may load the library's code
    torch.cuda.synchronize()
    free0, _ = torch.cuda.mem_get_info()
    for _ in range(3):
        binding.r2c_static(d_in, out, virtual_slabs=2)
    torch.cuda.synchronize()
    free1, _ = torch.cuda.mem_get_info()
    assert free1 == free0, "device memory in use changed across fft3d_r2c_static calls: %d -> %d" % (free0, free1)


def test_too_large_and_bad_arguments_are_refused(fft):
    from paper_2202_12756_b200 import binding
    lib = fft.load_library()
    assert binding.STATIC_SCRATCH_BYTES == 17 << 20
    big = torch.zeros((256, 256, 256), dtype=torch.float32, device="cuda")        # needs 64 MiB of scratch
    out = torch.full((256 * 256 * 129,), 7.0, dtype=torch.complex64, device="cuda")
    with pytest.raises(fft.Fft3dError) as e:
        binding.r2c_static(big, out)
    assert e.value.status == 5 and "workspace" in str(e.value)
    torch.cuda.synchronize()
    assert bool((out == 7.0).all()), "a refused call must not touch the output"
    # one step over the limit in fp64: 128 x 128 x 130 is unsupported (65 has no kernel), 128 x 160 x 128 is 20 MiB
    x = torch.zeros((128, 160, 128), dtype=torch.float64, device="cuda")
    o = torch.empty(128 * 160 * 65, dtype=torch.complex128, device="cuda")
    with pytest.raises(fft.Fft3dError) as e:
        binding.r2c_static(x, o)
    assert e.value.status == 5
    # the argument rules of fft3d_plan / fft3d_r2c
    a = torch.zeros((64, 64, 64), dtype=torch.float32, device="cuda")
    b = torch.empty(64 * 64 * 33, dtype=torch.complex64, device="cuda")
    st = torch.cuda.current_stream().cuda_stream
    assert lib.fft3d_r2c_static(64, 64, 64, 0, 3, a.data_ptr(), b.data_ptr(), st) == 1      # p does not divide
    assert lib.fft3d_r2c_static(64, 64, 63, 0, 1, a.data_ptr(), b.data_ptr(), st) == 2      # odd Nz
    assert lib.fft3d_r2c_static(64, 64, 64, 0, 1, None, b.data_ptr(), st) == 1              # null input
    assert lib.fft3d_r2c_static(64, 64, 64, 0, 1, a.data_ptr() + 4, b.data_ptr(), st) == 1  # misaligned
    assert lib.fft3d_r2c_static(64, 64, 64, 0, 1, a.data_ptr(), a.data_ptr(), st) == 1      # in == out
    assert lib.fft3d_r2c_static(64, 64, 64, 7, 1, a.data_ptr(), b.data_ptr(), st) == 1      # bad dtype
    torch.cuda.synchronize()
