"""GPU parity: libmg_b200 (through the C ABI) against the fp64 CPU oracle, element by element
on the same seeded inputs.  Tolerances are BASELINE.json's: per-sweep relative L2 <= 1e-5 (fp32),
<= 1e-12 (fp64); converged solutions within 1e-6 relative L2 of the oracle's."""
import numpy as np
import pytest

from workloads import configs, rng

pytestmark = pytest.mark.gpu

TOL = {"f32": 1e-5, "f64": 1e-12}
N, D, H0 = configs.BC_NEUMANN, configs.BC_DIRICHLET, configs.BC_DIRICHLET_HALO
BC_MIXES = [(D,) * 6, (N, N, N, N, N, D), (H0,) * 6, (N, D, H0, N, D, H0), (N,) * 6]


@pytest.fixture(scope="module")
def mg():
    import torch
    if not torch.cuda.is_available():
        pytest.fail("GPU tests need a CUDA device")
    import paper_2401_06755_b200 as m
    return m


from _parity import assert_close, rel_l2  # noqa: E402  (relative L2 AND max-abs bound on every comparison)


def to_dev(a, dt):
    import torch
    return torch.from_numpy(np.ascontiguousarray(a)).to(torch.float32 if dt == "f32" else torch.float64).cuda()


def as_f64(t):
    return t.detach().cpu().double().numpy()


def quantise(a, dt):
    """Round the fp64 input to the run precision so both sides see the very same numbers."""
    return np.ascontiguousarray(a, dtype=np.float32).astype(np.float64) if dt == "f32" else np.ascontiguousarray(a)


def make_problem(shape, dt, var, seed):
    n = int(np.prod(shape))
    x = quantise(rng.normal(seed, n).reshape(shape), dt)
    b = quantise(rng.uniform(seed + 1, n).reshape(shape), dt)
    k = None
    if var:  # strong contrast, like 1/rho with rho in [1, 1000]
        k = quantise(np.exp(-6.9 * rng.uniform01(seed + 2, n)).reshape(shape), dt)
    return x, b, k


def make_solver(mg, shape, h, levels, bc, dt, k=None, fused=1, **params):
    nz, ny, nx = shape
    hh = h if isinstance(h, tuple) else (h, h, h)
    s = mg.mg_create((nx, ny, nz, *hh), levels, bc, mg.MG_F32 if dt == "f32" else mg.MG_F64)
    # fused: 0 = one generic kernel per operation, 1 = streaming kernels, one stage per launch (sweeps_per_pass 1),
    #        T >= 2 = wave kernel, up to T dependent stages per launch (sweeps_per_pass T; wave_kernel.cuh)
    p = dict(nu_pre=2, nu_post=2, coarse_sweeps=50, sweeps_per_pass=max(fused, 1), omega=2.0 / 3.0, mixed_precision=1)
    p.update(params)
    mg.mg_set_params(s, **p)
    mg.mg_set_fused(s, 1 if fused else 0)
    if k is not None:
        mg.mg_set_coefficient(s, to_dev(k, dt))
    return s


SHAPES = [((32, 32, 32), 1.0 / 32), ((8, 24, 40), 1.0 / 40), ((70, 36, 132), 0.01), ((4, 4, 4), 0.25)]


@pytest.mark.parametrize("fused", [0, 1, 2, 3, 4])
@pytest.mark.parametrize("dt", ["f32", "f64"])
@pytest.mark.parametrize("var", [False, True])
@pytest.mark.parametrize("bc", BC_MIXES)
@pytest.mark.parametrize("shape,h", SHAPES)
def test_operator_residual_and_sweeps(mg, orc, shape, h, bc, var, dt, fused):
    import torch
    nz, ny, nx = shape
    g = orc.grid(nx, ny, nz, h)
    x, b, k = make_problem(shape, dt, var, 11)
    s = make_solver(mg, shape, h, 1, bc, dt, k, fused)
    dx, db = to_dev(x, dt), to_dev(b, dt)
    dy = torch.empty_like(dx)
    mg.mg_apply_operator(s, dx, dy)
    assert_close(as_f64(dy), orc.apply_operator(g, bc, k, x), TOL[dt])
    mg.mg_residual(s, dx, db, dy)
    assert_close(as_f64(dy), orc.residual(g, bc, k, x, b), TOL[dt])
    # per-sweep parity, every sweep restarted from the oracle's iterate
    xo = x
    for sweep in range(3):
        dxs = to_dev(xo, dt)
        mg.mg_smooth(s, dxs, db, 1)
        xo_next = orc.jacobi_sweep(g, bc, k, quantise(xo, dt), b, 2.0 / 3.0)
        assert_close(as_f64(dxs), xo_next, TOL[dt], "sweep %d" % sweep)
        xo = xo_next
    # several sweeps in one call (temporal fusion inside the library must not change the result)
    for sweeps in (2, 3, 4, 5):
        dxs = to_dev(x, dt)
        mg.mg_smooth(s, dxs, db, sweeps)
        assert_close(as_f64(dxs), orc.smooth(g, bc, k, x, b, 2.0 / 3.0, sweeps), sweeps * TOL[dt])
    mg.mg_destroy(s)


def test_anisotropic_spacing(mg, orc):
    """hx != hy != hz: all 27 weights differ and some off-diagonals are positive.
    The coefficient contrast is kept mild so that the Jacobi diagonal stays well away from 0
    (with positive off-diagonals and a random 1000:1 k it does not, and the sweep is ill-posed)."""
    import torch
    shape, bc, hh = (12, 20, 16), (N, D, H0, N, D, N), (0.1, 0.08, 0.125)
    g = orc.grid(16, 20, 12, *hh)
    for dt in ("f32", "f64"):
        x, b, _ = make_problem(shape, dt, False, 21)
        k = quantise(np.exp(-rng.uniform01(23, x.size)).reshape(shape), dt)
        diag = orc.diagonal(g, k)
        assert diag.min() > 0.2 * diag.max()
        s = make_solver(mg, shape, hh, 2, bc, dt, k)
        dx, db = to_dev(x, dt), to_dev(b, dt)
        dy = torch.empty_like(dx)
        mg.mg_apply_operator(s, dx, dy)
        assert_close(as_f64(dy), orc.apply_operator(g, bc, k, x), TOL[dt])
        mg.mg_smooth(s, dx, db, 2)
        assert_close(as_f64(dx), orc.smooth(g, bc, k, x, b, 2.0 / 3.0, 2), 2 * TOL[dt])
        dx = to_dev(x, dt)
        mg.mg_vcycle(s, dx, db)
        assert_close(as_f64(dx), orc.vcycle(g, bc, k, x, b, 2), 10 * TOL[dt])
        mg.mg_destroy(s)


@pytest.mark.parametrize("fused", [0, 1, 2, 3, 4])
@pytest.mark.parametrize("dt", ["f32", "f64"])
@pytest.mark.parametrize("var", [False, True])
@pytest.mark.parametrize("shape,h,levels,bc,nu", [
    ((32, 32, 32), 1.0 / 32, 4, (D,) * 6, (2, 2)),
    ((32, 32, 32), 1.0 / 32, 4, (N, N, N, N, N, D), (2, 2)),
    ((16, 48, 80), 1.0 / 80, 3, (N, D, H0, N, N, D), (1, 3)),
    ((64, 64, 64), 1.0 / 64, 5, (N, N, N, N, N, D), (2, 2)),
    ((64, 32, 96), 1.0 / 96, 4, (D, N, N, D, H0, D), (3, 1)),
    ((32, 32, 32), 1.0 / 32, 3, (D,) * 6, (0, 2)),
    ((8, 8, 8), 1.0 / 8, 2, (N, N, N, N, N, D), (2, 2)),
])
def test_vcycle_parity(mg, orc, shape, h, levels, bc, nu, var, dt, fused):
    nz, ny, nx = shape
    g = orc.grid(nx, ny, nz, h)
    x, b, k = make_problem(shape, dt, var, 31)
    s = make_solver(mg, shape, h, levels, bc, dt, k, fused, nu_pre=nu[0], nu_post=nu[1], coarse_sweeps=50)
    dx, db = to_dev(x, dt), to_dev(b, dt)
    xo = x
    for cycle in range(2):
        mg.mg_vcycle(s, dx, db)
        xo = orc.vcycle(g, bc, k, xo, b, levels, nu[0], nu[1], 50, 2.0 / 3.0)
        # growth allowance: a cycle is ~ (nu1 + nu2 + transfers) sweeps per level
        assert_close(as_f64(dx), xo, 10 * (cycle + 1) * TOL[dt], "cycle %d" % cycle)
    mg.mg_destroy(s)


@pytest.mark.parametrize("dt", ["f32", "f64"])
def test_config1_solve(mg, orc, dt):
    """BASELINE config 1: 32^3, constant coefficient, zero Dirichlet, 4 levels, V(2,2), tol 1e-8."""
    w = configs.config1()
    g = orc.grid(w.nx, w.ny, w.nz, w.h)
    b = quantise(w.fields["b"], dt)
    x_ref, n_ref, rel_ref, _ = orc.solve(g, w.bc, None, np.zeros(w.shape), b, w.levels, 1e-12, 100)
    assert rel_ref < 1e-12
    s = make_solver(mg, w.shape, w.h, w.levels, w.bc, dt)
    dx, db = to_dev(np.zeros(w.shape), dt), to_dev(b, dt)
    status, cycles, rel = mg.mg_solve(s, dx, db, w.tol, 100)
    assert status == mg.MG_OK and rel < w.tol
    hist = mg.mg_get_history(s)
    assert len(hist) == cycles and all(hist[i + 1] < hist[i] for i in range(len(hist) - 1))
    # the oracle needs the same number of cycles to reach the same tolerance
    _, n_tol, _, hist_o = orc.solve(g, w.bc, None, np.zeros(w.shape), b, w.levels, w.tol, 100)
    assert abs(cycles - n_tol) <= 1
    assert_close(as_f64(dx), x_ref, 1e-6)
    # residual of the GPU solution, evaluated by the oracle
    r = orc.residual(g, w.bc, None, as_f64(dx), b)
    assert np.linalg.norm(r) / np.linalg.norm(b) < (2e-7 if dt == "f32" else 1e-8)
    mg.mg_destroy(s)


@pytest.mark.parametrize("m", [2, 3])
def test_cycles_per_defect(mg, orc, m):
    """cycles_per_defect = m: m V-cycles on one correction equation between two fp64 defects.  In exact arithmetic the iterates
    are those of plain cycles, so the residual history (one entry per defect) must follow the oracle's at the cycles m, 2m, ...,
    the converged solution must be the oracle's, and a fixed cycle count that is not a multiple of m ends with a shorter round."""
    w = configs.config1()
    g = orc.grid(w.nx, w.ny, w.nz, w.h)
    b = quantise(w.fields["b"], "f32")
    x_ref, _, _, hist_o = orc.solve(g, w.bc, None, np.zeros(w.shape), b, w.levels, 1e-12, 100)
    s = make_solver(mg, w.shape, w.h, w.levels, w.bc, "f32", cycles_per_defect=m)
    assert mg.mg_get_params(s)["cycles_per_defect"] == m
    dx, db = to_dev(np.zeros(w.shape), "f32"), to_dev(b, "f32")
    status, cycles, rel = mg.mg_solve(s, dx, db, 1e-9, 100)
    hist = mg.mg_get_history(s)
    assert status == mg.MG_OK and rel < 1e-9 and cycles % m == 0 and len(hist) == cycles // m
    assert np.allclose(hist[:3], hist_o[m - 1::m][:3], rtol=1e-3), (hist, hist_o)
    assert_close(as_f64(dx), x_ref, 1e-6)
    # 7 fixed cycles: rounds of m, m, ... and a shorter last one; same iterate as with a defect after every cycle
    dx7 = to_dev(np.zeros(w.shape), "f32")
    status, cycles, rel = mg.mg_solve(s, dx7, db, 0.0, 7)
    assert cycles == 7 and len(mg.mg_get_history(s)) == -(-7 // m)
    x7, _, _, h7 = orc.solve(g, w.bc, None, np.zeros(w.shape), b, w.levels, 0.0, 7)
    assert abs(rel - h7[-1]) <= 1e-3 * h7[-1]
    assert_close(as_f64(dx7), x7, 1e-5)
    assert mg.mg_get_history_cycles(s) == [min(m * (i + 1), 7) for i in range(-(-7 // m))]
    with pytest.raises(mg.MgError):
        mg.mg_set_params(s, cycles_per_defect=9)
    mg.mg_destroy(s)


def test_adaptive_cycles_per_defect(mg, orc):
    """cycles_per_defect = 0: the solve loop picks the cycles of every round from the contraction it has seen.  Whatever it picks,
    each history entry must be the oracle's residual after the reported number of cycles, the solve must not run more than one
    round past the oracle's cycle count, and a fixed-count solve must do exactly the cycles asked for."""
    w = configs.config2(64, 5)
    g = orc.grid(w.nx, w.ny, w.nz, w.h)
    alpha = quantise(w.fields["alpha"], "f32")
    b = quantise(orc.pressure_rhs(g, w.fields["u"], w.fields["v"], w.fields["w"], 1.0), "f32")
    k = orc.k_from_vof(alpha, w.rho_l, w.rho_g)
    _, n_o, _, hist_o = orc.solve(g, w.bc, k, np.zeros(w.shape), b, w.levels, 1e-7, 200)
    s = make_solver(mg, w.shape, w.h, w.levels, w.bc, "f32", cycles_per_defect=0)
    mg.mg_set_coefficient_from_vof(s, to_dev(alpha, "f32"), w.rho_l, w.rho_g)
    assert mg.mg_get_params(s)["cycles_per_defect"] == 0
    dx, db = to_dev(np.zeros(w.shape), "f32"), to_dev(b, "f32")
    status, cycles, rel = mg.mg_solve(s, dx, db, 1e-7, 200)
    hist, at = mg.mg_get_history(s), mg.mg_get_history_cycles(s)
    assert status == mg.MG_OK and rel < 1e-7 and at[-1] == cycles and len(hist) == len(at)
    assert n_o <= cycles <= n_o + 3, (cycles, n_o, at)
    assert at[0] == 1 and all(b_ - a_ in (1, 2, 4, 8) for a_, b_ in zip(at, at[1:])) and len(at) < cycles      # fewer defects than cycles
    ho = orc.solve(g, w.bc, k, np.zeros(w.shape), b, w.levels, 0.0, cycles)[3]
    assert np.allclose(hist, [ho[c - 1] for c in at], rtol=2e-2), (hist, at, ho)
    # fixed count: rounds of 4 and a shorter last one
    dx.zero_()
    status, cycles, rel = mg.mg_solve(s, dx, db, 0.0, 10)
    assert cycles == 10 and mg.mg_get_history_cycles(s) == [4, 8, 10]        # rounds of 4, 4, 2
    x10 = orc.solve(g, w.bc, k, np.zeros(w.shape), b, w.levels, 0.0, 10)[0]
    assert_close(as_f64(dx), x10, 1e-4)
    mg.mg_destroy(s)


def test_pure_fp32_solve_stagnates_cleanly(mg, orc):
    w = configs.config1()
    b = quantise(w.fields["b"], "f32")
    s = make_solver(mg, w.shape, w.h, w.levels, w.bc, "f32", mixed_precision=0)
    dx, db = to_dev(np.zeros(w.shape), "f32"), to_dev(b, "f32")
    status, cycles, rel = mg.mg_solve(s, dx, db, 1e-10, 60)
    assert status in (mg.MG_STAGNATED, mg.MG_NOT_CONVERGED) and rel < 1e-5 and cycles <= 60
    mg.mg_destroy(s)


def test_sawtooth_nu0_reports_instead_of_looping(mg, orc):
    """V(0,1) with the C5 transfers and omega = 2/3 DIVERGES (SURVEY hard part 5: factor ~4 per cycle): mg_solve must say
    MG_STAGNATED once three cycles in a row have failed to reduce the residual, with a finite residual that equals the oracle's at the
    same cycles -- not loop, and not report success."""
    w = configs.config1()
    g = orc.grid(w.nx, w.ny, w.nz, w.h)
    b = quantise(w.fields["b"], "f32")
    s = make_solver(mg, w.shape, w.h, w.levels, w.bc, "f32", nu_pre=0, nu_post=1)
    dx, db = to_dev(np.zeros(w.shape), "f32"), to_dev(b, "f32")
    status, cycles, rel = mg.mg_solve(s, dx, db, 1e-8, 30)
    hist = mg.mg_get_history(s)
    _, _, _, hist_o = orc.solve(g, w.bc, None, np.zeros(w.shape), b, w.levels, 0.0, cycles, 0, 1)
    assert status == mg.MG_STAGNATED and 3 <= cycles <= 8, (status, cycles, rel)
    assert np.isfinite(rel) and rel > 1.0 and hist[-1] > hist[0]
    assert np.allclose(hist, hist_o, rtol=1e-3), (hist, hist_o)
    mg.mg_destroy(s)


def test_mg_solve_host_matches_the_oracle(mg, orc):
    """The end-to-end entry point bench.py times (`e2e`): host buffers in, host buffers out.  Config 1 (32^3), both a
    tolerance-driven solve and the paper's fixed cycle count (tol = 0)."""
    import torch
    w = configs.config1()
    g = orc.grid(w.nx, w.ny, w.nz, w.h)
    b = quantise(w.fields["b"], "f32")
    x_ref, _, rel_ref, _ = orc.solve(g, w.bc, None, np.zeros(w.shape), b, w.levels, 1e-12, 100)
    s = make_solver(mg, w.shape, w.h, w.levels, w.bc, "f32")
    hb = torch.from_numpy(b.astype(np.float32)).pin_memory()
    hx = torch.zeros(w.shape, dtype=torch.float32).pin_memory()
    status, cycles, rel = mg.mg_solve_host(s, hx, hb, 1e-9, 100)
    assert status == mg.MG_OK and rel < 1e-9
    assert_close(hx.double().numpy(), x_ref, 1e-6)
    assert np.array_equal(hb.numpy(), b.astype(np.float32))              # b is never modified
    hx.zero_()
    status, cycles, rel = mg.mg_solve_host(s, hx, hb, 0.0, 5)
    x5, _, _, hist_o = orc.solve(g, w.bc, None, np.zeros(w.shape), b, w.levels, 0.0, 5)
    assert cycles == 5 and np.allclose(mg.mg_get_history(s), hist_o, rtol=1e-3)
    assert_close(hx.double().numpy(), x5, 1e-5)
    # zero-guess entry point: the output buffer is not read (fill it with NaN), the iterates are the same bit for bit
    hz = torch.full(w.shape, float("nan"), dtype=torch.float32).pin_memory()
    status, cycles, rel = mg.mg_solve_host_zero(s, hz, hb, 0.0, 5)
    assert cycles == 5 and np.array_equal(hz.numpy(), hx.numpy())
    assert_close(hz.double().numpy(), x5, 1e-5)
    mg.mg_destroy(s)


def _config2_problem(orc, n, levels):
    w = configs.config2(n, levels)
    g = orc.grid(w.nx, w.ny, w.nz, w.h)
    alpha = quantise(w.fields["alpha"], "f32")
    b = quantise(orc.pressure_rhs(g, w.fields["u"], w.fields["v"], w.fields["w"], 1.0), "f32")
    return w, g, alpha, b


def test_config2_converged_solution(mg, orc):
    """BASELINE config 2 at its full size (128^3 water column, 6 levels): the oracle is driven to 1e-12, the GPU to 1e-9
    (error / residual amplification ~65 on this problem, reading C6-iii), and the converged solutions agree to 1e-6."""
    w, g, alpha, b = _config2_problem(orc, 128, 6)
    k = orc.k_from_vof(alpha, w.rho_l, w.rho_g)
    x_ref, _, rel_ref, _ = orc.solve(g, w.bc, k, np.zeros(w.shape), b, w.levels, 1e-12, 300)
    assert rel_ref < 1e-12
    s = make_solver(mg, w.shape, w.h, w.levels, w.bc, "f32")
    mg.mg_set_coefficient_from_vof(s, to_dev(alpha, "f32"), w.rho_l, w.rho_g)
    dx, db = to_dev(np.zeros(w.shape), "f32"), to_dev(b, "f32")
    status, cycles, rel = mg.mg_solve(s, dx, db, 1e-9, 300)
    assert status == mg.MG_OK, (status, cycles, rel)
    assert_close(as_f64(dx), x_ref, 1e-6)
    mg.mg_destroy(s)


def test_config2_full_size(mg, orc):
    """BASELINE config 2 at 128^3, 6 levels: solve to 1e-7, cycle count and per-cycle history
    against the oracle, and the residual of the GPU solution evaluated by the oracle."""
    w, g, alpha, b = _config2_problem(orc, 128, 6)
    k = orc.k_from_vof(alpha, w.rho_l, w.rho_g)
    s = make_solver(mg, w.shape, w.h, w.levels, w.bc, "f32")
    mg.mg_set_coefficient_from_vof(s, to_dev(alpha, "f32"), w.rho_l, w.rho_g)
    dx, db = to_dev(np.zeros(w.shape), "f32"), to_dev(b, "f32")
    status, cycles, rel = mg.mg_solve(s, dx, db, w.tol, 100)
    assert status == mg.MG_OK and rel < w.tol
    x_o, n_o, rel_o, hist_o = orc.solve(g, w.bc, k, np.zeros(w.shape), b, w.levels, w.tol, 100)
    hist = mg.mg_get_history(s)
    assert abs(cycles - n_o) <= 1
    m = min(len(hist), len(hist_o))
    assert np.allclose(hist[:m], hist_o[:m], rtol=2e-2)
    r = orc.residual(g, w.bc, k, as_f64(dx), b)
    assert np.linalg.norm(r) / np.linalg.norm(b) < 2 * w.tol
    # both stopped at the same residual level: solutions agree to the error/residual amplification
    assert_close(as_f64(dx), x_o, 1e-4)
    mg.mg_destroy(s)


def test_config3_full_size_cycle_parity(mg, orc):
    """BASELINE config 3 (256^3 bubble, 7 levels), the launch configuration bench.py times:
    one fused fp32 V-cycle against the oracle's, element by element."""
    w = configs.config3()
    g = orc.grid(w.nx, w.ny, w.nz, w.h)
    alpha = quantise(w.fields["alpha"], "f32")
    b = quantise(orc.pressure_rhs(g, w.fields["u"], w.fields["v"], w.fields["w"], 1.0), "f32")
    k = orc.k_from_vof(alpha, w.rho_l, w.rho_g)
    s = make_solver(mg, w.shape, w.h, w.levels, w.bc, "f32")
    mg.mg_set_coefficient_from_vof(s, to_dev(alpha, "f32"), w.rho_l, w.rho_g)
    dx, db = to_dev(np.zeros(w.shape), "f32"), to_dev(b, "f32")
    mg.mg_vcycle(s, dx, db)
    x_o = orc.vcycle(g, w.bc, k, np.zeros(w.shape), b, w.levels)
    assert_close(as_f64(dx), x_o, 1e-4)
    mg.mg_destroy(s)


def test_config3_twenty_cycle_solve_history(mg, orc):
    """BASELINE config 3 as the paper runs a pressure solve: a fixed 20 cycles, here through the mixed-precision
    loop (fp64 defect, fp32 correction cycles from the Jacobi seed) that bench.py's e2e leg and flow_time_step use.  The
    residual history must follow the fp64 oracle's cycle by cycle, and the iterate after 20 cycles must agree."""
    w = configs.config3()
    g = orc.grid(w.nx, w.ny, w.nz, w.h)
    alpha = quantise(w.fields["alpha"], "f32")
    b = quantise(orc.pressure_rhs(g, w.fields["u"], w.fields["v"], w.fields["w"], 1.0), "f32")
    k = orc.k_from_vof(alpha, w.rho_l, w.rho_g)
    s = make_solver(mg, w.shape, w.h, w.levels, w.bc, "f32")
    mg.mg_set_coefficient_from_vof(s, to_dev(alpha, "f32"), w.rho_l, w.rho_g)
    dx, db = to_dev(np.zeros(w.shape), "f32"), to_dev(b, "f32")
    status, cycles, rel = mg.mg_solve(s, dx, db, 0.0, 20)
    hist = mg.mg_get_history(s)
    x_o, n_o, rel_o, hist_o = orc.solve(g, w.bc, k, np.zeros(w.shape), b, w.levels, 0.0, 20)
    assert cycles == 20 and len(hist) == 20 and n_o == 20
    assert np.allclose(hist, hist_o, rtol=1e-2), (hist, hist_o)
    # 20 cycles of an iteration that contracts by ~0.95 per cycle here: rounding differences are not damped, allow 20 x the
    # one-cycle bound
    assert_close(as_f64(dx), x_o, 20 * 1e-5)
    mg.mg_destroy(s)


def test_argument_errors(mg):
    import torch
    with pytest.raises(mg.MgError) as e:
        mg.mg_create((30, 32, 32, 0.1), 3, (N,) * 6)
    assert e.value.code == mg.MG_ESHAPE
    with pytest.raises(mg.MgError) as e:
        mg.mg_create((32, 32, 32, 0.1), 6, (N,) * 6)       # coarsest dimension would be 1
    assert e.value.code == mg.MG_ESHAPE
    with pytest.raises(mg.MgError) as e:
        mg.mg_create((32, 32, 32, 0.1), 2, (N, N, N, N, N, 7))
    assert e.value.code == mg.MG_EINVAL
    s = mg.mg_create((32, 32, 32, 0.1), 2, (D,) * 6)
    x = torch.zeros(32, 32, 32, device="cuda")
    with pytest.raises(mg.MgError):
        mg.mg_apply_operator(s, x, x)                        # aliased
    with pytest.raises(ValueError):
        mg.mg_apply_operator(s, x, torch.zeros(16, 32, 32, device="cuda"))
    with pytest.raises(mg.MgError):
        mg.mg_set_params(s, omega=-1.0)
    for spp in (0, 5, 8):                                        # only 1 .. 4 stages per launch are implemented
        with pytest.raises(mg.MgError) as e:
            mg.mg_set_params(s, sweeps_per_pass=spp)
        assert e.value.code == mg.MG_EINVAL
    mg.mg_destroy(s)


def test_empty_cycles_and_zero_rhs(mg):
    import torch
    s = mg.mg_create((16, 16, 16, 1.0 / 16), 3, (D,) * 6)
    x = torch.zeros(16, 16, 16, device="cuda"); b = torch.zeros_like(x)
    status, cycles, rel = mg.mg_solve(s, x, b, 1e-8, 10)       # b = 0: converged at once, x stays 0
    assert status == mg.MG_OK and cycles == 0 and float(x.abs().max()) == 0.0
    b.fill_(1.0)
    status, cycles, rel = mg.mg_solve(s, x, b, 1e-8, 0)        # max_cycles = 0
    assert status == mg.MG_NOT_CONVERGED and cycles == 0
    mg.mg_smooth(s, x, b, 0)
    assert float(x.abs().max()) == 0.0
    mg.mg_destroy(s)


@pytest.mark.parametrize("var", [False, True])
@pytest.mark.parametrize("shape,levels,nu", [((64, 48, 96), 4, 2), ((32, 32, 32), 4, 1), ((16, 16, 16), 3, 2), ((40, 24, 48), 3, 0),
                                             ((32, 48, 64), 3, 3)])
def test_zero_guess_cycle_equals_cycle_from_cleared_x(mg, shape, levels, nu, var):
    """The correction cycles of mg_solve / mg_pcg_solve start from x = 0 without reading x (lean_kernel zero_x; cleared x
    where level 0 is not a lean_kernel level or nu_pre = 0); with nu_pre >= 2 mg_solve's cycles start from the seed y = r / D
    written by the defect kernel and do the first two sweeps in one pass.  One cycle of the mixed-precision solve from x = 0 is
    x = V(0, float(b)): it must equal the public mg_vcycle from a cleared x up to the fp64 -> fp32 rounding of the result."""
    dt = "f32"
    _, b, k = make_problem(shape, dt, var, 77)
    bc = (N, N, N, N, N, D)
    s = make_solver(mg, shape, 1.0 / shape[2], levels, bc, dt, k=k if var else None, nu_pre=nu, nu_post=max(nu, 1))
    db = to_dev(b, dt)
    x_cycle = to_dev(np.zeros(shape), dt)
    assert mg.mg_vcycle(s, x_cycle, db) == mg.MG_OK
    x_solve = to_dev(np.zeros(shape), dt)                  # the solver's correction buffer is uninitialised at this point
    st, cycles, rel = mg.mg_solve(s, x_solve, db, 0.0, 1)
    assert cycles == 1
    assert_close(as_f64(x_solve), as_f64(x_cycle), 2e-7)
    # a second solve reuses the (possibly dirty) correction buffer: same answer
    x2 = to_dev(np.zeros(shape), dt)
    mg.mg_solve(s, x2, db, 0.0, 1)
    assert rel_l2(as_f64(x2), as_f64(x_solve)) == 0.0
    mg.mg_destroy(s)


def test_recorded_cycle_survives_a_coefficient_change(mg, orc):
    """mg_vcycle replays a recorded CUDA graph; a new variable coefficient reuses the solver's buffers, so the recording is
    kept -- and must then use the NEW coefficient: cycle parity against the oracle before and after the change, and after
    going to a constant coefficient and back."""
    shape, levels, dt = (32, 32, 32), 4, "f32"
    bc = (N, N, N, N, N, D)
    g = orc.grid(32, 32, 32, 1.0 / 32)
    x0, b, k1 = make_problem(shape, dt, True, 5)
    _, _, k2 = make_problem(shape, dt, True, 9)
    s = make_solver(mg, shape, 1.0 / 32, levels, bc, dt, k=k1)
    db = to_dev(b, dt)
    for k in (k1, k2, k1, None, k2):
        if k is None:
            mg.mg_set_coefficient(s, None)
        else:
            mg.mg_set_coefficient(s, to_dev(k, dt))
        for rep in range(2):                                   # first call records (or reuses), second replays
            dx = to_dev(x0, dt)
            assert mg.mg_vcycle(s, dx, db) == mg.MG_OK
            ref = orc.vcycle(g, bc, k, x0, b, levels, 2, 2, 50, 2.0 / 3.0)
            assert_close(as_f64(dx), ref, 20 * TOL[dt])
    mg.mg_destroy(s)


@pytest.mark.parametrize("var", [False, True])
def test_tabulated_coarsest_solve_follows_parameters_and_coefficient(mg, orc, var):
    """On a 4^3 coarsest level the cluster tail applies the coarse_sweeps Jacobi sweeps as one tabulated matrix
    (ctail_kernel.cuh `cmat`).  The table must follow coarse_sweeps, omega and the coefficient: cycle parity against the
    oracle after each change, and with the table switched off by a coarsest level that is not 4^3."""
    dt, bc = "f32", (N, N, N, N, N, D)
    shape = (64, 64, 64)
    g = orc.grid(64, 64, 64, 1.0 / 64)
    x0, b, k1 = make_problem(shape, dt, var, 41)
    _, _, k2 = make_problem(shape, dt, var, 43)
    for levels in (5, 4):                                   # coarsest 4^3 (tabulated) and 8^3 (sweeps)
        s = make_solver(mg, shape, 1.0 / 64, levels, bc, dt, k=k1)
        db = to_dev(b, dt)
        for cs, omega, k in ((50, 2.0 / 3.0, k1), (7, 2.0 / 3.0, k1), (7, 0.8, k1), (7, 0.8, k2), (1, 0.8, k2), (50, 2.0 / 3.0, k2)):
            mg.mg_set_params(s, nu_pre=2, nu_post=2, coarse_sweeps=cs, sweeps_per_pass=1, omega=omega, mixed_precision=1)
            if var:
                mg.mg_set_coefficient(s, to_dev(k, dt))
            dx = to_dev(x0, dt)
            assert mg.mg_vcycle(s, dx, db) == mg.MG_OK
            ref = orc.vcycle(g, bc, k if var else None, x0, b, levels, 2, 2, cs, omega)
            assert_close(as_f64(dx), ref, 20 * TOL[dt], (levels, cs, omega))
        mg.mg_destroy(s)
