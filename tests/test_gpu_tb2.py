"""DR_KERNEL 3: two PT iterations per sweep on stencil-coded images (csrc/dr_kernels_tb2.cuh).
Parity against the oracle's dro_step(n) for even and odd n, every z chunking, boundary modes and void/fluid phases; the
same numbers, bit for bit, as the one-sweep kernel (the tables hold what that kernel computes on the fly); the pairing
of iterations around residual checks (odd ncheck); fallback on images that cannot be coded."""
import numpy as np
import pytest

from paper_2410_20441_b200 import inputs
from tests.test_gpu_parity import FIELD_TOL, C_TOL, field_errors, run_pair, to_dev, gpu, _quantised  # noqa: F401

pytestmark = pytest.mark.gpu


def _all_fields(s):
    return [s.get_field(f).clone() for f in range(9)]


@pytest.mark.parametrize("shape,levels,lc,niter,extra", [
    ((45, 33, 21), 7, 2, 6, {}), ((45, 33, 21), 7, 4, 7, {}), ((30, 30, 30), 2, 5, 11, dict(bc_mode=1)),
    ((61, 29, 33), 3, 3, 9, dict(gavg=1)), ((5, 64, 7), 3, 0, 5, {}), ((2, 2, 2), 2, 1, 4, {}), ((3, 2, 9), 2, 2, 3, {}),
    ((70, 50, 45), 4, 4, 12, dict(zchunk=7)), ((70, 50, 45), 4, 2, 11, dict(zchunk=1)), ((33, 40, 80), 3, 1, 8, dict(void_rel=0.2)),
    ((29, 11, 58), 5, 5, 10, dict(zchunk=2, bc_mode=1, gavg=1)), ((57, 21, 12), 6, 0, 1, {}), ((28, 10, 30), 2, 3, 2, dict(zchunk=64))])
def test_two_iteration_sweeps_vs_oracle_and_bitwise_vs_one_sweep_kernel(oracle_mod, gpu, shape, levels, lc, niter, extra):
    import torch
    K, G = _quantised(shape, levels, seed=sum(shape) + levels)
    errs, ro, rs, ao, as_ = run_pair(oracle_mod, gpu, K, G, lc, 1e-4, niter, h=0.7, kernel=3, **extra)
    assert max(errs) <= FIELD_TOL, errs
    assert abs(ro - rs) <= 1e-9 * ro
    # h = 1: the coded kernels fold 1/h into their constants, which is exact for h = 1 -> the same bits as kernel 0
    ref = gpu.Solver(to_dev(K), to_dev(G), kernel=0, **extra)
    ref.step(lc, 1e-4, niter)
    fr = _all_fields(ref)
    for kern in (3, 4):
        s = gpu.Solver(to_dev(K), to_dev(G), kernel=kern, **extra)
        s.step(lc, 1e-4, niter)
        assert s.active_kernel() == kern
        for a, b in zip(fr, _all_fields(s)):
            assert torch.equal(a, b), (kern,)
        assert s.info()[1] == ref.info()[1]


def test_pairing_around_residual_checks_and_maxiter(oracle_mod, gpu):
    """odd ncheck: a check iteration that would be the FIRST of a pair runs alone; same stopping iteration as the oracle;
    maxiter odd; dr_iterate with odd counts continues the same state"""
    import torch
    K, G, _ = inputs.config1_sphere(n=24, r=4.0)
    for ncheck in (7, 10, 1):
        o = oracle_mod.Oracle(K, G, ncheck=ncheck)
        s = gpu.Solver(to_dev(K), to_dev(G), ncheck=ncheck)
        assert s.solve(4, 1e-4, 1e-6, 1001) == o.solve(4, 1e-4, 1e-6, 1001) == 0
        assert s.info()[0] == o.info()[0], (ncheck, s.info(), o.info())
        assert abs(s.info()[1] - o.info()[1]) <= 1e-6 * o.info()[1]
        assert np.max(np.abs(s.avg_stress() - o.avg_stress())) <= 1e-9 * np.max(np.abs(o.avg_stress()))
    o = oracle_mod.Oracle(K, G, ncheck=50)
    s = gpu.Solver(to_dev(K), to_dev(G), ncheck=50)
    assert s.solve(1, 1e-4, 1e-30, 77) == gpu.MAXITER and o.solve(1, 1e-4, 1e-30, 77) == oracle_mod.MAXITER
    assert s.info()[0] == 77 and max(field_errors(o, s, K, G, 1e-4)) <= FIELD_TOL
    o.step(2, 1e-4, 3 + 5 + 8)
    s.step(2, 1e-4, 3); s.iterate(2, 1e-4, 5); s.iterate(2, 1e-4, 8)
    torch.cuda.synchronize()
    assert max(field_errors(o, s, K, G, 1e-4)) <= FIELD_TOL


def test_uncodable_images_fall_back_to_the_one_sweep_kernel(oracle_mod, gpu):
    K, G = inputs.random_smooth((20, 18, 16), seed=9)                 # every voxel different: no palette, no codes
    s = gpu.Solver(to_dev(K), to_dev(G))
    s.step(0, 1e-4, 4)
    assert s.active_kernel() == 0 and not s.uses_palette()
    K, G = _quantised((20, 18, 16), 40, seed=1)                       # 40 phases: palette yes, > 256 distinct edge means
    errs, ro, rs, _, _ = run_pair(oracle_mod, gpu, K, G, 3, 1e-4, 6)
    assert max(errs) <= FIELD_TOL
    s = gpu.Solver(to_dev(K), to_dev(G))
    s.step(0, 1e-4, 4)
    assert s.active_kernel() == 0 and s.uses_palette()
    K, G = _quantised((20, 18, 16), 3, seed=1)
    s = gpu.Solver(to_dev(K), to_dev(G))
    s.step(0, 1e-4, 4)
    assert s.active_kernel() == 3
    s.set_param("form", 1)                                            # displacement form: one-sweep kernel
    s.step(0, 1e-4, 4)
    assert s.active_kernel() == 0
    # codes follow DR_GAVG / DR_VOID_REL changes on a live handle (the oracle gets the same parameter history)
    s = gpu.Solver(to_dev(K), to_dev(G))
    cur = dict(gavg=0, void_rel=0.0)
    for params in (dict(gavg=1), dict(void_rel=0.3), dict(gavg=0), dict(void_rel=0.0)):
        cur.update(params)
        for k, v in params.items():
            s.set_param(k, v)
        s.step(5, 1e-4, 6)
        o = oracle_mod.Oracle(K, G, **cur)
        o.step(5, 1e-4, 6)
        assert s.active_kernel() == 3 and max(field_errors(o, s, K, G, 1e-4)) <= FIELD_TOL, cur


def test_solve_six_and_host_api_use_the_two_iteration_kernel(oracle_mod, gpu):
    K, G, _ = inputs.config1_sphere(n=20, r=3.0)
    C6, log6, solvers = gpu.solve_six(to_dev(K), to_dev(G), eps0=1e-4, tol=1e-8, maxiter=2000)
    assert all(sv.active_kernel() == 3 for sv in solvers)
    Ch, iters, st = gpu.solve_image_host(K, G, tol=1e-8, maxiter=2000, ncheck=50)
    o = oracle_mod.Oracle(K, G)
    Co, logo = o.solve_all(1e-4, 1e-8, 2000)
    assert [l[1] for l in log6] == [l[1] for l in logo] == iters
    assert np.max(np.abs(Co - C6)) <= C_TOL * np.max(np.abs(Co)) and np.array_equal(C6, Ch)


# ------------------------------------------------------------------------------------------------ dr_solve_all (S: 8(f) f2)
def test_solve_all_batched_equals_six_dr_solve_calls_and_the_oracle(oracle_mod, gpu):
    """six load cases per launch on one handle: bit-identical C, iteration counts and stop reasons to six dr_solve calls"""
    K, G, _ = inputs.config1_sphere()
    Kd, Gd = to_dev(K), to_dev(G)
    Cs, logs = gpu.Solver(Kd, Gd).solve_all(1e-4, 1e-8, 3200)
    b = gpu.Solver(Kd, Gd, six=True)
    Cb, logb = b.solve_all_batched(1e-4, 1e-8, 3200)
    assert b.active_kernel() == 3
    assert [l[1] for l in logb] == [l[1] for l in logs] and all(l[0] == 0 and l[3] == gpu.STOP_RESIDUAL for l in logb)
    assert np.array_equal(Cb, Cs)
    o = oracle_mod.Oracle(K, G)
    Co, logo = o.solve_all(1e-4, 1e-8, 3200)
    assert [l[1] for l in logo] == [l[1] for l in logb]
    assert np.max(np.abs(Co - Cb)) <= C_TOL * np.max(np.abs(Co))
    for lo, lb in zip(logo, logb):
        assert abs(lo[2] - lb[2]) <= 1e-6 * lo[2]
    # a second call on the same handle, other parameters: odd ncheck (single sweeps in between), maxiter not reached by all
    b.set_param("ncheck", 7); b.set_param("bc_mode", 1)
    Cb2, logb2 = b.solve_all_batched(1e-4, 1e-7, 301)
    s2 = gpu.Solver(Kd, Gd, ncheck=7, bc_mode=1)
    Cs2, logs2 = s2.solve_all(1e-4, 1e-7, 301)
    assert [(l[0], l[1]) for l in logb2] == [(l[0], l[1]) for l in logs2] and np.array_equal(Cb2, Cs2)


def test_solve_all_batched_ragged_stagnation_maxiter_and_fallbacks(oracle_mod, gpu):
    K, G, m = inputs.config3_random_spheres(n=48, npores=30, rmin=2.0, rmax=5.0, seed=7)       # plateaus: stagnation rule
    K = np.ascontiguousarray(K[:40, :45, :]); G = np.ascontiguousarray(G[:40, :45, :])           # 48 x 45 x 40
    Kd, Gd = to_dev(K), to_dev(G)
    b = gpu.Solver(Kd, Gd, six=True, ncheck=100)
    Cb, logb = b.solve_all_batched(1e-4, 1e-8, 4800)
    Cs, logs = gpu.Solver(Kd, Gd, ncheck=100).solve_all(1e-4, 1e-8, 4800)
    assert [l[1] for l in logb] == [l[1] for l in logs] and np.array_equal(Cb, Cs)
    assert all(l[0] == 0 and l[3] == gpu.STOP_STAGNATION for l in logb)
    o = oracle_mod.Oracle(K, G, ncheck=100)
    assert o.solve(4, 1e-4, 1e-8, 4800) == 0
    assert np.max(np.abs(o.avg_stress() / 1e-4 - Cb[:, 4])) <= C_TOL * np.max(np.abs(Cb))
    # soft maxiter
    Cm, logm = b.solve_all_batched(1e-4, 1e-30, 150)
    assert all(l[0] == gpu.MAXITER and l[1] == 150 and l[3] == gpu.STOP_MAXITER for l in logm)
    # images that cannot be coded, other kernels: same call, six plain solves behind it
    Kr, Gr = inputs.random_smooth((20, 18, 16), seed=9)
    br = gpu.Solver(to_dev(Kr), to_dev(Gr), six=True)
    Cr, logr = br.solve_all_batched(1e-4, 1e-8, 3000)
    Cq, logq = gpu.Solver(to_dev(Kr), to_dev(Gr)).solve_all(1e-4, 1e-8, 3000)
    assert br.active_kernel() == 0 and np.array_equal(Cr, Cq) and [l[1] for l in logr] == [l[1] for l in logq]
    # a single-solve workspace refuses the batch
    with pytest.raises(gpu.DrError) as e:
        gpu.Solver(Kd, Gd).solve_all_batched()
    assert e.value.status == gpu.ERR_WORKSPACE
    # the host-buffer call takes the batch when given the larger workspace
    Ch, iters, st = gpu.solve_image_host(K, G, tol=1e-8, maxiter=4800, ncheck=100, six=True)
    assert st == 0 and iters == [l[1] for l in logb] and np.array_equal(Ch, Cb)


def test_palette_toggle_rebuilds_the_stencil_codes(gpu):
    """DR_PALETTE 1 -> 0 -> 1 on one handle: the codes dropped at 0 are rebuilt at 1 (the cache key used to survive with
    has_codes false, which left the handle on the one-sweep kernel until gavg or void_rel changed)"""
    import torch
    K, G = _quantised((40, 30, 20), 3, seed=3)
    s = gpu.Solver(to_dev(K), to_dev(G))
    s.step(2, 1e-4, 6)
    assert s.active_kernel() == 3
    f3 = _all_fields(s)
    s.set_param("palette", 0)
    s.step(2, 1e-4, 6)
    assert s.active_kernel() == 0 and not s.uses_palette()
    s.set_param("palette", 1)
    s.step(2, 1e-4, 6)
    assert s.active_kernel() == 3
    for a, b in zip(f3, _all_fields(s)):
        assert torch.equal(a, b)


def test_solve_all_fallback_reports_every_load_case_after_a_hard_error(gpu):
    """dr_solve_all on its six-plain-solves path (DR_KERNEL 0) with a C~ far above the stability limit: load case 0 diverges,
    the call returns DR_ERR_DIVERGED, and the load cases that never ran say DR_ERR_STATE / 0 iterations / DR_STOP_NONE"""
    import ctypes as C
    K, G = _quantised((20, 18, 16), 3, seed=4)
    b = gpu.Solver(to_dev(K), to_dev(G), six=True, kernel=0, cfl=3.0, ncheck=20)
    stat = (C.c_int * 6)(*([-7] * 6))
    rc = gpu.lib().dr_solve_all(b._h, 1e-4, 1e-8, 4000, stat)
    assert rc == gpu.ERR_DIVERGED and list(stat) == [gpu.ERR_DIVERGED] + [gpu.ERR_STATE] * 5
    for lc in range(1, 6):
        it, r, sp = C.c_int(-1), C.c_double(-1.0), C.c_int(-1)
        gpu.lib().dr_info_lc(b._h, lc, C.byref(it), C.byref(r), C.byref(sp))
        assert it.value == 0 and sp.value == gpu.STOP_NONE and r.value == float("inf")


def test_run_to_run_bitwise_determinism_and_kernel_equality_at_191(gpu):
    """compute-sanitizer is closed on the GPU pool (profiles/r3_sanitizer.txt holds its output), so races in the shared-memory pipeline of the two-iteration
    kernel are hunted the other way: at 191^3 (560 CTAs of 512 threads, 4 waves, every tile shape) five runs of 60 iterations
    are identical bit for bit, and identical to the one-sweep kernel, whose staging, barriers and thread-to-node map differ."""
    import torch
    K, G, _ = inputs.config3_random_spheres()
    Kd, Gd = to_dev(K), to_dev(G)
    ref = None
    for rep in range(6):
        s = gpu.Solver(Kd, Gd, kernel=0 if rep == 5 else 3)
        s.step(4, 1e-4, 60)
        assert s.active_kernel() == (0 if rep == 5 else 3)
        f = _all_fields(s)
        if ref is None:
            ref = f
        else:
            for a, b in zip(ref, f):
                assert torch.equal(a, b), rep
        s.close()
