"""GPU parity: libdr (through the C ABI) against the CPU oracle on the same seeded inputs.
Bars (BASELINE.json north_star): per-field relative L-inf <= 1e-10 after a fixed iteration count,
C_ij relative <= 1e-6 at convergence."""
import numpy as np
import pytest

from paper_2410_20441_b200 import inputs

pytestmark = pytest.mark.gpu

FIELD_TOL = 1e-10
C_TOL = 1e-6


@pytest.fixture(scope="module")
def gpu():
    import torch
    assert torch.cuda.is_available(), "these tests need a CUDA device"
    from paper_2410_20441_b200 import binding
    binding.lib()
    return binding


def to_dev(a):
    import torch
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def field_errors(o, s, K, G, eps0, h=1.0):
    """err_f = |f_gpu - f_cpu|_inf / max(|f_cpu|_inf, 1e-6 S); S = eps0 L (velocities), max(K+4G/3) eps0 (stresses)"""
    L = h * max(K.shape)
    Sv = abs(eps0) * L
    Ss = abs(eps0) * float(np.max(K + 4 * G / 3))
    errs = []
    for f in range(9):
        a = o.get_field(f)
        b = s.get_field(f).cpu().numpy()
        assert a.shape == b.shape
        S = Sv if f < 3 else Ss
        errs.append(float(np.max(np.abs(a - b)) / max(np.max(np.abs(a)), 1e-6 * S)))
    return errs


def run_pair(oracle_mod, gpu, K, G, lc, eps0, niter, h=1.0, **params):
    o = oracle_mod.Oracle(K, G, h=h, **{k: v for k, v in params.items() if k not in ("kernel", "zchunk", "palette")})
    s = gpu.Solver(to_dev(K), to_dev(G), h=h, **params)
    o.step(lc, eps0, niter)
    s.step(lc, eps0, niter)
    errs = field_errors(o, s, K, G, eps0, h)
    ro, rs = o.info()[1], s.info()[1]
    ao, as_ = o.avg_stress(), s.avg_stress()
    return errs, ro, rs, ao, as_


@pytest.mark.parametrize("kernel", [0, 1, 2, 3, 4])
@pytest.mark.parametrize("lc", range(6))
def test_fields_config1_sphere_100_iterations(oracle_mod, gpu, kernel, lc):
    K, G, _ = inputs.config1_sphere()
    errs, ro, rs, ao, as_ = run_pair(oracle_mod, gpu, K, G, lc, 1e-4, 100, kernel=kernel)
    assert max(errs) <= FIELD_TOL, errs
    assert abs(ro - rs) <= 1e-9 * ro
    assert np.max(np.abs(ao - as_)) <= 1e-10 * np.max(np.abs(ao))


@pytest.mark.parametrize("kernel", [0, 1, 2])
@pytest.mark.parametrize("shape,h", [((37, 21, 19), 0.5), ((5, 64, 7), 1.0), ((2, 2, 2), 2.0), ((61, 29, 33), 1.0)])
def test_fields_ragged_noncubic_random_moduli(oracle_mod, gpu, kernel, shape, h):
    """several tiles with ragged tails in x, y and z; every voxel has different moduli"""
    K, G = inputs.random_smooth(shape, seed=sum(shape))
    for lc in (0, 3, 4, 5):
        errs, ro, rs, ao, as_ = run_pair(oracle_mod, gpu, K, G, lc, -2e-3, 25, h=h, kernel=kernel)
        assert max(errs) <= FIELD_TOL, (lc, errs)
        assert abs(ro - rs) <= 1e-9 * ro


@pytest.mark.parametrize("kernel", [0, 1, 2, 3, 4])
def test_fields_void_and_fluid_cells(oracle_mod, gpu, kernel):
    """degenerate moduli: exact void (K=G=0), fluid (G=0), 1e-6 contrast"""
    K, G, m = inputs.random_two_phase((40, 33, 20), frac=0.3, seed=4, matrix=(37.0, 44.0), incl=(2.2, 0.0))
    K[3:6, 10:20, 5:30] = 0.0
    G[3:6, 10:20, 5:30] = 0.0
    for lc in (1, 2, 4):
        errs, ro, rs, _, _ = run_pair(oracle_mod, gpu, K, G, lc, 1e-4, 30, kernel=kernel)
        assert max(errs) <= FIELD_TOL, (lc, errs)
        assert np.isfinite(rs) and abs(ro - rs) <= 1e-9 * ro


@pytest.mark.parametrize("kernel", [0, 1, 2, 3, 4])
@pytest.mark.parametrize("params", [dict(bc_mode=1), dict(gavg=1), dict(cfl=0.5, st_factor=0.7), dict(void_rel=1e-5)])
def test_fields_parameter_variants(oracle_mod, gpu, kernel, params):
    K, G, _ = inputs.config1_sphere(n=24, r=4.0)
    for lc in (0, 5):
        errs, ro, rs, _, _ = run_pair(oracle_mod, gpu, K, G, lc, 1e-4, 40, kernel=kernel, **params)
        assert max(errs) <= FIELD_TOL, (params, lc, errs)


def test_zero_iterations_is_the_initial_field(oracle_mod, gpu):
    K, G = inputs.random_smooth((9, 8, 7), seed=1)
    for lc in range(6):
        errs, _, _, ao, as_ = run_pair(oracle_mod, gpu, K, G, lc, 1e-3, 0, h=0.3)
        assert max(errs) <= 1e-14, errs
        assert np.max(np.abs(ao - as_)) <= 1e-13 * np.max(np.abs(ao))


@pytest.mark.parametrize("kernel", [0, 1, 2, 3])
def test_converged_C_config1(oracle_mod, gpu, kernel):
    """cfg 1 to tol 1e-8, same ncheck on both sides -> same iteration counts; C within 1e-6"""
    K, G, _ = inputs.config1_sphere()
    o = oracle_mod.Oracle(K, G)
    Co, logo = o.solve_all(1e-4, 1e-8, 3200)
    s = gpu.Solver(to_dev(K), to_dev(G), kernel=kernel)
    Cs, logs = s.solve_all(1e-4, 1e-8, 3200)
    assert [l[1] for l in logo] == [l[1] for l in logs]
    assert all(l[0] == 0 for l in logs)
    assert np.max(np.abs(Co - Cs)) <= C_TOL * np.max(np.abs(Co))
    for lo, ls in zip(logo, logs):
        assert abs(lo[2] - ls[2]) <= 1e-6 * lo[2]


def test_converged_C_two_phase_48(oracle_mod, gpu):
    K, G, _ = inputs.config4_grf(n=48, ell=6.0, seed=5)
    o = oracle_mod.Oracle(K, G, ncheck=100)
    Co, logo = o.solve_all(1e-4, 1e-8, 4800)
    s = gpu.Solver(to_dev(K), to_dev(G), ncheck=100)
    Cs, logs = s.solve_all(1e-4, 1e-8, 4800)
    assert [l[1] for l in logo] == [l[1] for l in logs]
    assert np.max(np.abs(Co - Cs)) <= C_TOL * np.max(np.abs(Co))


def test_host_api_end_to_end(oracle_mod, gpu):
    K, G, _ = inputs.config1_sphere(n=20, r=3.0)
    C, iters, st = gpu.solve_image_host(K, G, tol=1e-8, maxiter=2000, ncheck=50)
    o = oracle_mod.Oracle(K, G)
    Co, logo = o.solve_all(1e-4, 1e-8, 2000)
    assert st == 0 and iters == [l[1] for l in logo]
    assert np.max(np.abs(Co - C)) <= C_TOL * np.max(np.abs(Co))


def test_status_codes_and_errors(gpu):
    import torch
    K, G = inputs.homogeneous(8)
    s = gpu.Solver(to_dev(K), to_dev(G))
    with pytest.raises(gpu.DrError) as e:
        s.effective_C()
    assert e.value.status == gpu.ERR_STATE
    with pytest.raises(gpu.DrError):
        s.solve(7)
    with pytest.raises(gpu.DrError):
        s.solve(0, eps0=0.0)
    with pytest.raises(gpu.DrError):
        s.iterate(0, 1e-4, 3)                      # no fields yet
    assert s.solve(0, 1e-4, 1e-30, 7) == gpu.MAXITER
    assert s.info()[0] == 7
    Kb = K.copy(); Kb[1, 2, 3] = -1.0
    with pytest.raises(gpu.DrError) as e:
        gpu.Solver(to_dev(Kb), to_dev(G))
    assert e.value.status == gpu.ERR_ARG
    Kb[1, 2, 3] = np.nan
    with pytest.raises(gpu.DrError):
        gpu.Solver(to_dev(Kb), to_dev(G))
    small = torch.empty(1024, dtype=torch.uint8, device="cuda")
    with pytest.raises(gpu.DrError) as e:
        gpu.Solver(to_dev(K), to_dev(G), workspace=small)
    assert e.value.status == gpu.ERR_WORKSPACE


def test_homogeneous_block_on_gpu(gpu):
    K, G = inputs.homogeneous((33, 17, 40), 70.2, 29.0)
    s = gpu.Solver(to_dev(K), to_dev(G), ncheck=10)
    C, log = s.solve_all()
    assert all(l[0] == 0 and l[1] == 10 and l[2] < 1e-11 for l in log), log
    H = np.zeros((6, 6)); H[:3, :3] = 70.2 - 2 * 29 / 3
    H[np.arange(3), np.arange(3)] = 70.2 + 4 * 29 / 3; H[np.arange(3, 6), np.arange(3, 6)] = 29.0
    assert np.max(np.abs(C - H)) <= 1e-11 * 108.9


def test_iterate_continues_step(oracle_mod, gpu):
    K, G = inputs.random_smooth((20, 18, 16), seed=9)
    o = oracle_mod.Oracle(K, G)
    o.step(2, 1e-4, 30)
    s = gpu.Solver(to_dev(K), to_dev(G))
    s.step(2, 1e-4, 10)
    s.iterate(2, 1e-4, 20)
    import torch
    torch.cuda.synchronize()
    errs = field_errors(o, s, K, G, 1e-4)
    assert max(errs) <= FIELD_TOL, errs


# ---------------------------------------------------------------- BASELINE.json full sizes, bench launch configuration
def _host_gb():
    try:
        import psutil
        return psutil.virtual_memory().available / 1e9
    except Exception:
        return 0.0


def test_full_size_703_homogeneous_block(gpu):
    """cfg 5 size (703^3, the largest): a property that holds at any size (homogeneous block: Hooke, zero residual);
    the oracle comparison on the penny-crack image itself is in tests/test_gpu_configs.py"""
    import torch
    n = 703
    Kd = torch.full((n, n, n), 70.2, dtype=torch.float64, device="cuda")
    Gd = torch.full((n, n, n), 29.0, dtype=torch.float64, device="cuda")
    s = gpu.Solver(Kd, Gd, ncheck=5)
    for lc in (2, 3):
        assert s.solve(lc, 1e-4, 1e-8, 50) == 0
        it, r, _ = s.info()
        assert it == 5 and r < 1e-10
        col = s.avg_stress() / 1e-4
        want = np.zeros(6)
        if lc == 2:
            want[:3] = 70.2 - 2 * 29 / 3; want[2] = 70.2 + 4 * 29 / 3
        else:
            want[3] = 29.0
        assert np.max(np.abs(col - want)) <= 1e-10 * 108.9
    s.close(); del s, Kd, Gd
    torch.cuda.empty_cache()


# ---------------------------------------------------------------- displacement form (DR_FORM = 1, S: 8(f) f1)
@pytest.mark.parametrize("kernel", [0, 1])
@pytest.mark.parametrize("lc", range(6))
def test_displacement_form_fields_config1(oracle_mod, gpu, kernel, lc):
    K, G, _ = inputs.config1_sphere()
    errs, ro, rs, ao, as_ = run_pair(oracle_mod, gpu, K, G, lc, 1e-4, 100, kernel=kernel, form=1)
    assert max(errs) <= FIELD_TOL, errs
    assert abs(ro - rs) <= 1e-9 * ro
    assert np.max(np.abs(ao - as_)) <= 1e-10 * np.max(np.abs(ao))


@pytest.mark.parametrize("kernel", [0, 1])
def test_displacement_form_ragged_void_fluid_and_variants(oracle_mod, gpu, kernel):
    K, G = inputs.random_smooth((37, 21, 19), seed=77)
    K[3:6, 4:9, 5:30] = 0.0; G[3:6, 4:9, 5:30] = 0.0          # void
    G[10:12, 2:6, 3:9] = 0.0                                   # fluid
    for lc, extra in ((0, {}), (3, dict(bc_mode=1)), (4, dict(gavg=1)), (5, dict(cfl=0.5, st_factor=0.7))):
        errs, ro, rs, _, _ = run_pair(oracle_mod, gpu, K, G, lc, -2e-3, 30, h=0.5, kernel=kernel, form=1, **extra)
        assert max(errs) <= FIELD_TOL, (lc, errs)
        assert abs(ro - rs) <= 1e-9 * ro
    errs, _, _, ao, as_ = run_pair(oracle_mod, gpu, K, G, 2, 1e-3, 0, kernel=kernel, form=1)      # initial fields
    assert max(errs) <= 1e-13, errs


def test_displacement_form_converged_C_and_continue(oracle_mod, gpu):
    K, G, _ = inputs.config1_sphere()
    o = oracle_mod.Oracle(K, G, form=1)
    Co, logo = o.solve_all(1e-4, 1e-8, 3200)
    s = gpu.Solver(to_dev(K), to_dev(G), form=1)
    Cs, logs = s.solve_all(1e-4, 1e-8, 3200)
    assert [l[1] for l in logo] == [l[1] for l in logs] and all(l[0] == 0 for l in logs)
    assert np.max(np.abs(Co - Cs)) <= C_TOL * np.max(np.abs(Co))
    # same fixed point as the paper's stress-relaxation form
    s0 = gpu.Solver(to_dev(K), to_dev(G))
    C0, _ = s0.solve_all(1e-4, 1e-8, 3200)
    assert np.max(np.abs(C0 - Cs)) <= 1e-6 * np.max(np.abs(C0))
    # step + get_field (forms the stresses) + iterate continues from the same state
    o.step(2, 1e-4, 30)
    s.step(2, 1e-4, 10); s.get_field("sxx"); s.iterate(2, 1e-4, 20)
    import torch
    torch.cuda.synchronize()
    assert max(field_errors(o, s, K, G, 1e-4)) <= FIELD_TOL


def test_solve_six_on_streams_equals_sequential(oracle_mod, gpu):
    """row a7: six handles on six streams give the same iterates, iteration counts and C as six dr_solve calls"""
    K, G, _ = inputs.config1_sphere()
    Kd, Gd = to_dev(K), to_dev(G)
    Cs, logs = gpu.Solver(Kd, Gd).solve_all(1e-4, 1e-8, 3200)
    C6, log6, solvers = gpu.solve_six(Kd, Gd, eps0=1e-4, tol=1e-8, maxiter=3200)
    assert [l[1] for l in log6] == [l[1] for l in logs] and all(l[0] == 0 for l in log6)
    assert np.array_equal(C6, Cs)                                  # same kernels, same order: bit-identical
    o = oracle_mod.Oracle(K, G)
    Co, _ = o.solve_all(1e-4, 1e-8, 3200)
    assert np.max(np.abs(Co - C6)) <= C_TOL * np.max(np.abs(Co))
    # soft status and error paths
    C6b, log6b, _ = gpu.solve_six(Kd, Gd, eps0=1e-4, tol=1e-30, maxiter=120, ncheck=50)
    assert all(l[0] == gpu.MAXITER and l[1] == 120 for l in log6b)


@pytest.mark.parametrize("zchunk", [1, 2, 5, 13, 64])
def test_fields_do_not_depend_on_the_z_chunking(oracle_mod, gpu, zchunk):
    """DR_ZCHUNK only changes how the z-march is cut into CTAs (priming step at every chunk start): same results"""
    K, G = inputs.random_smooth((35, 31, 27), seed=123)
    for kernel in (0, 2):
        errs, ro, rs, _, _ = run_pair(oracle_mod, gpu, K, G, 4, 1e-4, 12, kernel=kernel, zchunk=zchunk)
        assert max(errs) <= FIELD_TOL, (kernel, errs)
        assert abs(ro - rs) <= 1e-9 * ro
    errs, _, _, _, _ = run_pair(oracle_mod, gpu, K, G, 1, 1e-4, 12, kernel=0, zchunk=zchunk, form=1)
    assert max(errs) <= FIELD_TOL, errs


@pytest.mark.parametrize("form", [0, 1])
def test_fields_191_default_chunking(oracle_mod, gpu, form):
    """191^3 (cfg 2/3 size) with the automatic z chunking (32 layers: ring slots are recycled many times per chunk)"""
    K, G, _ = inputs.config3_random_spheres()
    errs, ro, rs, ao, as_ = run_pair(oracle_mod, gpu, K, G, 4, 1e-4, 15, form=form)
    assert max(errs) <= FIELD_TOL, errs
    assert abs(ro - rs) <= 1e-9 * ro
    assert np.max(np.abs(ao - as_)) <= 1e-10 * np.max(np.abs(ao))


def _fuzz_case(rng):
    shape = tuple(int(v) for v in rng.integers(2, 70, size=3))
    kernel = int(rng.integers(0, 3))
    form = int(rng.integers(0, 2)) if kernel != 2 else 0
    params = dict(kernel=kernel, form=form, bc_mode=int(rng.integers(0, 2)), gavg=int(rng.integers(0, 2)))
    if kernel != 1 and rng.uniform() < 0.6:
        params["zchunk"] = int(rng.integers(1, 40))
    if rng.uniform() < 0.3:
        params["st_factor"] = float(rng.uniform(0.5, 0.9))
    return shape, params, int(rng.integers(0, 6)), float(rng.choice([1e-4, -3e-3])), int(rng.integers(1, 16)), float(rng.choice([1.0, 0.37, 2.5]))


@pytest.mark.parametrize("seed", range(24))
def test_fuzz_random_shapes_and_parameters(oracle_mod, gpu, seed):
    """seeded random shapes (2..69 per axis), kernels, forms, boundary modes, chunkings, void/fluid cells"""
    rng = np.random.default_rng(1000 + seed)
    shape, params, lc, eps0, niter, h = _fuzz_case(rng)
    if seed % 2:                                  # every other case: few distinct (K,G) pairs -> phase-id path
        K, G = _quantised(shape, int(rng.integers(2, 40)) if seed % 4 == 1 else int(rng.integers(2, 5)), seed)
        if params["kernel"] != 1 and params["form"] == 0:
            params["kernel"] = 3 if seed % 4 == 3 or params["kernel"] == 0 else 4       # coded kernels (fall back when > 256 edge values)
        if rng.uniform() < 0.3:
            params["void_rel"] = 0.1
    else:
        K, G = inputs.random_smooth(shape, seed=seed)
        m = rng.uniform(size=K.shape)
        K[m < 0.05] = 0.0; G[m < 0.05] = 0.0          # void
        G[(m > 0.05) & (m < 0.1)] = 0.0               # fluid
    if params.get("form") == 1:
        params.setdefault("st_factor", 0.5 if max(shape) < 12 else 1.0)      # keep theta well below 1 on tiny grids
        if max(shape) < 12:
            params["st_factor"] = 0.4
    errs, ro, rs, ao, as_ = run_pair(oracle_mod, gpu, K, G, lc, eps0, niter, h=h, **params)
    assert max(errs) <= FIELD_TOL, (shape, params, lc, niter, errs)
    assert np.isfinite(rs) and abs(ro - rs) <= 1e-9 * max(ro, 1e-300), (shape, params, ro, rs)


def _quantised(shape, levels, seed):
    """image with `levels` distinct (K,G) pairs: exercises the phase-id (palette) path of the fused kernel"""
    rng = np.random.default_rng(seed)
    sh = tuple(shape)[::-1]
    ph = rng.integers(0, levels, size=sh)
    Kt = rng.uniform(1.0, 70.0, size=levels); Gt = rng.uniform(0.5, 45.0, size=levels)
    if levels > 3:
        Kt[1] = Gt[1] = 0.0          # a void phase
        Gt[2] = 0.0                  # a fluid phase
    return np.ascontiguousarray(Kt[ph]), np.ascontiguousarray(Gt[ph])


@pytest.mark.parametrize("levels", [1, 2, 7, 256, 300])
@pytest.mark.parametrize("palette", [1, 0])
def test_palette_path_matches_oracle(oracle_mod, gpu, levels, palette):
    """<= 256 distinct pairs -> uint8 phase ids + table; 300 -> falls back to the fp64 fields.  Same values either way."""
    K, G = _quantised((45, 33, 21), levels, seed=levels)
    cases = ((2, {}), (5, dict(bc_mode=1, gavg=1)), (3, dict(form=1)), (0, dict(void_rel=0.2)))
    if levels == 1:
        cases = cases[:1]        # one phase: every other field is identically zero and only rounding noise is compared
    for lc, extra in cases:
        errs, ro, rs, _, _ = run_pair(oracle_mod, gpu, K, G, lc, 1e-4, 14, h=0.8, palette=palette, **extra)
        assert max(errs) <= FIELD_TOL, (levels, palette, lc, errs)
        assert abs(ro - rs) <= 1e-9 * ro + 1e-13          # a one-phase image has residual ~1e-16
    s = gpu.Solver(to_dev(K), to_dev(G), palette=palette)
    assert s.uses_palette() == (palette == 1 and levels <= 256)


def test_palette_path_is_bitwise_the_fp64_path(gpu):
    import torch
    K, G, _ = inputs.config3_random_spheres(n=96, npores=40)
    res = []
    for palette in (1, 0):
        s = gpu.Solver(to_dev(K), to_dev(G), palette=palette)
        s.step(4, 1e-4, 25)
        res.append([s.get_field(f).clone() for f in range(9)] + [torch.tensor(s.info()[1])])
    for a, b in zip(*res):
        assert torch.equal(a, b)


# ---------------------------------------------------------------- round-2 additions: stopping rule, parameter hygiene
def test_stagnation_rule_same_stop_as_oracle(oracle_mod, gpu):
    """Reading R9b: 48^3 pores at 1e-6 contrast plateau near 1e-5; both sides stop on <sigma> stagnation with DR_OK, the
    same C, at the same check (both sides evaluate Eq. 7 to working precision, reading R7b)."""
    K, G, m = inputs.config3_random_spheres(n=48, npores=30, rmin=2.0, rmax=5.0, seed=7)
    s = gpu.Solver(to_dev(K), to_dev(G), ncheck=100)
    o = oracle_mod.Oracle(K, G, ncheck=100)
    for lc in (0, 3):
        assert s.solve(lc, 1e-4, 1e-8, 4800) == 0 and o.solve(lc, 1e-4, 1e-8, 4800) == 0
        assert s.stop_reason() == gpu.STOP_STAGNATION and o.stop_reason() == oracle_mod.STOP_STAGNATION
        assert s.info()[0] == o.info()[0] and s.info()[0] < 4800, (s.info(), o.info())
        assert np.max(np.abs(s.avg_stress() - o.avg_stress())) <= C_TOL * np.max(np.abs(o.avg_stress()))
    # rule off -> soft DR_MAXITER, same column
    s0 = gpu.Solver(to_dev(K), to_dev(G), ncheck=100, stag_tol=0.0)
    assert s0.solve(3, 1e-4, 1e-8, 2500) == gpu.MAXITER and s0.stop_reason() == gpu.STOP_MAXITER
    assert np.max(np.abs(s0.avg_stress() - o.avg_stress())) <= C_TOL * np.max(np.abs(o.avg_stress()))
    # six load cases on streams take the same decisions as six dr_solve calls
    C6, log6, solvers = gpu.solve_six(to_dev(K), to_dev(G), eps0=1e-4, tol=1e-8, maxiter=4800, ncheck=100)
    Cs, logs = gpu.Solver(to_dev(K), to_dev(G), ncheck=100).solve_all(1e-4, 1e-8, 4800)
    assert [l[1] for l in log6] == [l[1] for l in logs] and np.array_equal(C6, Cs)
    assert all(sv.stop_reason() == gpu.STOP_STAGNATION for sv in solvers)


def test_negative_zero_moduli_are_plain_zero(oracle_mod, gpu):
    """-0.0 passes the >= 0 validation; it must behave as +0.0 (void / fluid), not poison hmax or the edge means"""
    K, G = inputs.random_smooth((12, 10, 9), seed=3)
    K[2:4, 3:6, 4:8] = 0.0; G[2:4, 3:6, 4:8] = 0.0
    G[6, 2:5, 1:7] = 0.0
    Kn, Gn = K.copy(), G.copy()
    Kn[K == 0.0] = -0.0; Gn[G == 0.0] = -0.0
    assert np.signbit(Kn).any() and np.signbit(Gn).any()
    for pal, Kq, Gq in ((0, K, G), (1, *_quantised((12, 10, 9), 9, 5))):
        Kq = Kq.copy(); Gq = Gq.copy()
        Km, Gm = Kq.copy(), Gq.copy()
        Km[Kq == 0.0] = -0.0; Gm[Gq == 0.0] = -0.0
        a = gpu.Solver(to_dev(Kq), to_dev(Gq), void_rel=1e-3)
        b = gpu.Solver(to_dev(Km), to_dev(Gm), void_rel=1e-3)
        for lc in (0, 4):
            a.step(lc, 1e-4, 12); b.step(lc, 1e-4, 12)
            import torch
            for f in range(9):
                assert torch.equal(a.get_field(f), b.get_field(f)), (pal, lc, f)
            assert np.isfinite(b.info()[1])
    errs, ro, rs, _, _ = run_pair(oracle_mod, gpu, Kn, Gn, 5, 1e-4, 12)
    assert max(errs) <= FIELD_TOL and np.isfinite(rs)


def test_set_param_discards_fields_built_under_old_parameters(gpu):
    K, G = inputs.random_smooth((10, 9, 8), seed=4)
    s = gpu.Solver(to_dev(K), to_dev(G))
    for name, v in (("kernel", 1), ("gavg", 1), ("bc_mode", 1), ("void_rel", 1e-3), ("cfl", 0.5), ("st_factor", 0.8), ("form", 1)):
        s.step(0, 1e-4, 3)
        s.iterate(0, 1e-4, 2)                       # fine: fields exist
        s.set_param(name, v)
        with pytest.raises(gpu.DrError) as e:
            s.iterate(0, 1e-4, 2)
        assert e.value.status == gpu.ERR_STATE, name
        with pytest.raises(gpu.DrError):
            s.get_field(0)
    s.step(0, 1e-4, 3)
    s.set_param("ncheck", 7); s.set_param("zchunk", 4); s.set_param("palette", 0); s.set_param("stag_tol", 0.0)
    s.iterate(0, 1e-4, 2)                           # these do not shape the iterate


# ------------------------------------------------------------------------------------------------ 7th direct test (App. A.3)
def test_triaxial_load_case_and_eq27_29_vs_oracle(oracle_mod, gpu):
    """load case 6 and dr_offdiag_direct (Eq. 24-29): fields after a fixed iteration count and the three
    off-diagonal components at convergence against the oracle; equal to the symmetrised columns of the six-test C"""
    K, G = _quantised((26, 22, 30), 3, seed=5)
    errs, ro, rs, ao, as_ = run_pair(oracle_mod, gpu, K, G, 6, 1e-4, 40)
    assert max(errs) <= FIELD_TOL, errs
    assert abs(ro - rs) <= 1e-9 * ro and np.max(np.abs(ao - as_)) <= 1e-10 * np.max(np.abs(ao))
    s = gpu.Solver(to_dev(K), to_dev(G))
    o = oracle_mod.Oracle(K, G)
    with pytest.raises(gpu.DrError) as e:
        s.offdiag_direct()
    assert e.value.status == gpu.ERR_STATE
    for lc in (0, 1, 2, 6):
        assert s.solve(lc, 1e-4, 1e-9, 20000) == 0 and o.solve(lc, 1e-4, 1e-9, 20000) == 0
        assert s.info()[0] == o.info()[0]
    d, do = s.offdiag_direct(), o.offdiag_direct()
    assert np.max(np.abs(d - do)) <= C_TOL * np.max(np.abs(do)), (d, do)
    for lc in (3, 4, 5):
        assert s.solve(lc, 1e-4, 1e-9, 20000) == 0
    C = s.effective_C()
    sym = np.array([0.5 * (C[0, 1] + C[1, 0]), 0.5 * (C[0, 2] + C[2, 0]), 0.5 * (C[1, 2] + C[2, 1])])
    assert np.max(np.abs(d - sym)) <= 1e-6 * C[0, 0]


# ------------------------------------------------------------------------------------------------ segmented images (phase ids + tables)
def test_segmented_create_is_bitwise_the_fp64_create(oracle_mod, gpu):
    """dr_create_segmented (uint8 phase ids + per-phase tables) builds the same handle as dr_create on the expanded arrays:
    identical fields after a fixed iteration count (hence the oracle parity of the fp64 path carries over), identical C from
    the host-buffer call; ids outside the table and bad table sizes are refused."""
    import torch
    rng = np.random.default_rng(11)
    shape = (23, 31, 40)                                  # (nz, ny, nx)
    Kt = np.array([37.0, 5.0, 0.0, 2.2, 70.2]); Gt = np.array([44.0, 2.0, 0.0, 0.0, 29.0])     # matrix, soft, void, fluid, calcite
    ph = rng.integers(0, 5, size=shape).astype(np.uint8)
    K, G = np.ascontiguousarray(Kt[ph]), np.ascontiguousarray(Gt[ph])
    a = gpu.Solver(to_dev(K), to_dev(G))
    b = gpu.Solver(Kt, Gt, phase=torch.from_numpy(ph).cuda())
    for lc, n in ((1, 7), (5, 10)):
        a.step(lc, 1e-4, n); b.step(lc, 1e-4, n)
        assert a.active_kernel() == b.active_kernel() == 3 and b.uses_palette()
        for f in range(9):
            assert torch.equal(a.get_field(f), b.get_field(f)), (lc, f)
        assert a.info()[1] == b.info()[1] and np.array_equal(a.avg_stress(), b.avg_stress())
    o = oracle_mod.Oracle(K, G)
    o.step(5, 1e-4, 10)
    assert max(field_errors(o, b, K, G, 1e-4)) <= FIELD_TOL
    # voxel noise with void and fluid cells: some load cases stop on a rule, others at maxiter -- the same way in all three calls
    Ca, ia, sa = gpu.solve_image_host(K, G, tol=1e-6, maxiter=1500, ncheck=50)
    Cb, ib, sb = gpu.solve_image_host_segmented(ph, Kt, Gt, tol=1e-6, maxiter=1500, ncheck=50)
    Cc, ic, sc = gpu.solve_image_host_segmented(ph, Kt, Gt, tol=1e-6, maxiter=1500, ncheck=50, six=True)
    assert sa == sb == sc and sa in (0, gpu.MAXITER) and ia == ib == ic and np.array_equal(Ca, Cb) and np.array_equal(Ca, Cc)
    with pytest.raises(gpu.DrError) as e:                 # an id beyond the table
        gpu.Solver(Kt[:4], Gt[:4], phase=torch.from_numpy(ph).cuda())
    assert e.value.status == gpu.ERR_ARG
    with pytest.raises(gpu.DrError) as e:                 # more than 256 phases
        gpu.Solver(np.ones(257), np.ones(257), phase=torch.from_numpy(ph).cuda())
    assert e.value.status == gpu.ERR_ARG
    with pytest.raises(gpu.DrError) as e:                 # negative modulus in the table
        gpu.Solver(np.array([1.0, -1.0, 1.0, 1.0, 1.0]), Gt, phase=torch.from_numpy(ph).cuda())
    assert e.value.status == gpu.ERR_ARG


# ------------------------------------------------------------------------------------------------ maximum extent per axis
@pytest.mark.parametrize("shape", [(8192, 2, 2), (2, 8192, 3), (3, 2, 8192)])
def test_maximum_extent_along_one_axis(oracle_mod, gpu, shape):
    """the largest size dr.h admits (8192) along x, y and z in turn, two or three nodes across: hundreds of tiles / z chunks
    of mostly halo; coded two-iteration kernel and the one-sweep kernel against the oracle, shear and normal load case"""
    K, G = _quantised(shape, 3, seed=shape[0] + 2 * shape[1])
    for kernel, lc, n in ((3, 2, 5), (3, 4, 4), (0, 5, 3)):
        errs, ro, rs, ao, as_ = run_pair(oracle_mod, gpu, K, G, lc, 1e-4, n, kernel=kernel)
        assert max(errs) <= FIELD_TOL, (kernel, lc, errs)
        assert abs(ro - rs) <= 1e-9 * ro
    assert gpu.workspace_bytes(8193, 2, 2) == 0
