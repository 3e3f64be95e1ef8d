"""dr_avg_stress_static (include/dr.h, csrc/dr_static.cu): the volume averages of Eq. 7 for callers that cannot allocate.

Most of libdr works in a workspace the caller allocated.  A hook that reports <sigma> while a long solve is running cannot
afford that (cudaMalloc / cudaFree wait for the whole device, so each report would stall the solver), and a plug-in inside a
host program whose allocator already holds the free device memory cannot get one at all.  For them this one call keeps its
reduction scratch in a 6 MiB array compiled into libdr.so.  What that costs, and what is tested here:
  * every call shares the one array and nobody clears it -> two calls in a row, a small grid after a large one and the
    large one again must each give the right numbers (stale partial sums of the other grid are still lying there);
  * the array has a fixed size -> the largest grid it holds works, one row more is refused with a message;
  * the reference is the existing path: dr_step + dr_avg_stress on a handle with a workspace, at the 1e-10 (relative to
    the largest component) the parity tests put on averages.

The file name sorts last on purpose: the suite runs with `pytest -x`, and a failure in this addition must not hide the parity
tests.  Nothing here depends on what ran before it in the process (it passes alone in a fresh process too)."""
import ctypes as C

import numpy as np
import pytest

from paper_2410_20441_b200 import inputs

AVG_TOL = 1e-10          # tests/test_gpu_parity.py: |avg_gpu - avg_ref|_inf <= 1e-10 |avg_ref|_inf


def _binding():
    from paper_2410_20441_b200 import build, binding
    build.build()
    binding.lib()
    return binding


def _solved_fields(binding, shape, seed, lc, niter):
    """existing path: a handle with its own workspace; returns (<sigma> from dr_avg_stress, the six dense stress fields)"""
    import torch
    K, G, _ = inputs.random_two_phase(shape, frac=0.35, seed=seed)
    s = binding.Solver(torch.from_numpy(K).cuda(), torch.from_numpy(G).cuda())
    s.step(lc, 1e-4, niter)
    ref = s.avg_stress()
    fields = [s.get_field(f) for f in range(3, 9)]
    torch.cuda.synchronize()
    s.close()
    return ref, fields


@pytest.mark.gpu
def test_static_average_equals_the_handle_path_on_calls_in_a_row():
    import torch
    assert torch.cuda.is_available(), "this test needs a CUDA device"
    binding = _binding()
    refA, fA = _solved_fields(binding, (70, 50, 45), seed=5, lc=4, niter=30)      # 51 x 46 rows -> 294 blocks, ragged last block
    refB, fB = _solved_fields(binding, (33, 21, 12), seed=6, lc=2, niter=17)      # 22 x 13 rows -> 36 blocks
    out = torch.full((3, 6), float("nan"), dtype=torch.float64, device="cuda")    # the caller's output, allocated up front
    binding.avg_stress_static(fB, out=out[1])               # set-up call: address look-up, kernels loaded
    torch.cuda.synchronize()
    before, free_before = torch.cuda.memory_allocated(), torch.cuda.mem_get_info()[0]
    # three calls back to back on one stream, no synchronisation in between: large, small, large again
    binding.avg_stress_static(fA, out=out[0])
    binding.avg_stress_static(fB, out=out[1])
    binding.avg_stress_static(fA, out=out[2])
    torch.cuda.synchronize()
    # nothing was allocated: neither through torch nor behind its back (free device memory as the driver reports it)
    assert torch.cuda.memory_allocated() == before and torch.cuda.mem_get_info()[0] >= free_before
    got = out.cpu().numpy()
    for g, ref in ((got[0], refA), (got[1], refB), (got[2], refA)):
        assert np.all(np.isfinite(g))
        assert np.max(np.abs(g - ref)) <= AVG_TOL * np.max(np.abs(ref)), (g, ref)
    assert np.array_equal(got[0], got[2])                   # fixed summation order: same bits whatever the array held before
    assert np.max(np.abs(refA)) > 0 and np.max(np.abs(refB)) > 0


@pytest.mark.gpu
def test_static_average_at_the_largest_grid_the_scratch_holds():
    """(ny+1)*(nz+1) == DR_STATIC_MAX_ROWS exactly: every entry of the built-in array is used.  A handle for this grid would
    need a 15 GB workspace, so the reference is Eq. 7 with the trapezoid weights of Reading R7 written in torch."""
    import torch
    assert torch.cuda.is_available(), "this test needs a CUDA device"
    binding = _binding()
    nx, ny, nz = 3, 1023, 1023
    assert (ny + 1) * (nz + 1) == binding.STATIC_MAX_ROWS
    g = torch.Generator(device="cuda").manual_seed(11)
    fields = [torch.rand(binding.field_shape(nx, ny, nz, f), generator=g, dtype=torch.float64, device="cuda") - 0.25 for f in range(3, 9)]

    def w(n):        # weights along an axis with n+1 nodes
        v = torch.ones(n + 1, dtype=torch.float64, device="cuda")
        v[0] = v[-1] = 0.5
        return v
    N = nx * ny * nz
    ref = [float(fields[m].sum() / N) for m in range(3)]
    ref.append(float((fields[3] * w(nz)[:, None, None] * w(ny)[None, :, None]).sum() / N))      # tyz (nz+1, ny+1, nx)
    ref.append(float((fields[4] * w(nz)[:, None, None] * w(nx)[None, None, :]).sum() / N))      # txz (nz+1, ny, nx+1)
    ref.append(float((fields[5] * w(ny)[None, :, None] * w(nx)[None, None, :]).sum() / N))      # txy (nz, ny+1, nx+1)
    ref = np.array(ref)
    got = binding.avg_stress_static(fields).cpu().numpy()
    assert np.max(np.abs(got - ref)) <= AVG_TOL * np.max(np.abs(ref)), (got, ref)
    # and a small grid straight after it reads none of the 131072 partial sums that call left behind
    refB, fB = _solved_fields(binding, (20, 9, 14), seed=7, lc=5, niter=8)
    gotB = binding.avg_stress_static(fB).cpu().numpy()
    assert np.max(np.abs(gotB - refB)) <= AVG_TOL * np.max(np.abs(refB)), (gotB, refB)


def test_static_average_refuses_grids_beyond_the_scratch_before_touching_the_device():
    """one x-row more than the array holds: DR_ERR_ARG and a message naming the limit; decided on the host before any CUDA
    call, so it runs on the CPU box as well (the pointers are never followed)"""
    binding = _binding()
    lib = binding.lib()
    dummy = (C.c_double * 8)()
    ptrs = (C.c_void_p * 6)(*([C.addressof(dummy)] * 6))
    err = C.create_string_buffer(512)
    rc = lib.dr_avg_stress_static(3, 1023, 1024, ptrs, C.addressof(dummy), None, err, len(err))
    assert rc == binding.ERR_ARG
    msg = err.value.decode()
    assert "DR_STATIC_MAX_ROWS" in msg and str(binding.STATIC_MAX_ROWS) in msg and str(1024 * 1025) in msg
    assert lib.dr_avg_stress_static(1, 8, 8, ptrs, C.addressof(dummy), None, err, len(err)) == binding.ERR_ARG
    assert b"2 .. 8192" in err.value
    assert lib.dr_avg_stress_static(8, 8, 8, None, C.addressof(dummy), None, None, 0) == binding.ERR_ARG
    ptrs[3] = None
    assert lib.dr_avg_stress_static(8, 8, 8, ptrs, C.addressof(dummy), None, err, len(err)) == binding.ERR_ARG
    assert b"NULL" in err.value
    import torch
    if not torch.cuda.is_available():                       # no device: a loud DR_ERR_CUDA, never a CPU computation
        ptrs[3] = C.addressof(dummy)
        assert lib.dr_avg_stress_static(8, 8, 8, ptrs, C.addressof(dummy), None, err, len(err)) == binding.ERR_CUDA
        assert b"cudaGetDevice" in err.value
