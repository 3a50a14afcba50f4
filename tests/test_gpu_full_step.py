"""GPU parity of SURVEY 8(f) next 3 -- free-slip wall halos, the forcing terms of Eq. 18 and the paper's four-stage
time step -- against the fp64 CPU oracle, through the C ABI."""
import numpy as np
import pytest

from workloads import configs, rng
from test_gpu_mg import TOL, as_f64, mg, quantise, to_dev  # noqa: F401
from _parity import assert_close  # noqa: E402

pytestmark = pytest.mark.gpu
N, D = configs.BC_NEUMANN, configs.BC_DIRICHLET
BCP = (N, N, N, N, N, D)
SHAPES = [((24, 24, 24), 1.0 / 24), ((10, 36, 68), 1.0 / 68), ((12, 10, 22), 0.05)]      # the last one: scalar (W = 1) kernels


def _fields(shape, dt, seed):
    n = int(np.prod(shape))
    nz, ny, nx = shape
    x, y, z = configs.centres(nx, ny, nz, 1.0)
    d = (0.6 * x / nx + 0.5 * y / ny + 0.62 * z / nz) - 0.8
    Cf = quantise(0.5 * (1 + np.tanh(d * 6.0)) + 0.0 * (x + y + z), dt)
    q = tuple(quantise(0.3 * rng.normal(seed + c, n).reshape(shape) + 0.2, dt) for c in range(3))
    return Cf, q


@pytest.mark.parametrize("dt", ["f32", "f64"])
@pytest.mark.parametrize("walls", [(1, 1, 1, 1, 1, 0), (0, 1, 1, 0, 0, 1)])
@pytest.mark.parametrize("shape,h", SHAPES)
def test_wall_halos_in_predictor_and_rhs(mg, orc, shape, h, walls, dt):
    import torch
    nz, ny, nx = shape
    g = orc.grid(nx, ny, nz, h)
    Cf, qh = _fields(shape, dt, 50)
    _, qn = _fields(shape, dt, 60)
    tstep = 0.1 * h
    vbc = orc.velocity_bc(walls)
    assert vbc == mg.velocity_bc(walls)
    qt_ref, qhn_ref = orc.mom_predictor(g, Cf, qh, qn, 1000.0, 1.0, 1e-3, 1e-5, tstep, vbc)
    dC = to_dev(Cf, dt)
    dqh, dqn = [to_dev(a, dt) for a in qh], [to_dev(a, dt) for a in qn]
    dqt, dqhn = [torch.empty_like(dC) for _ in range(3)], [torch.empty_like(dC) for _ in range(3)]
    mg.mom_predictor_bc(dC, dqh, dqn, vbc, h, 1000.0, 1.0, 1e-3, 1e-5, tstep, dqt, dqhn)
    for c in range(3):
        assert_close(as_f64(dqt[c]), qt_ref[c], TOL[dt])
        assert_close(as_f64(dqhn[c]), qhn_ref[c], TOL[dt])
    # the halo codes matter on this input (the copy-halo result is far outside the tolerance)
    qt_copy, _ = orc.mom_predictor(g, Cf, qh, qn, 1000.0, 1.0, 1e-3, 1e-5, tstep)
    assert max(np.abs(a - b).max() for a, b in zip(qt_copy, qt_ref)) > 1e-3 * max(np.abs(a).max() for a in qt_ref)
    db = torch.empty_like(dC)
    mg.pressure_rhs_bc(dqh[0], dqh[1], dqh[2], vbc, h, tstep, db)
    assert_close(as_f64(db), orc.pressure_rhs(g, qh[0], qh[1], qh[2], tstep, vbc), TOL[dt])


@pytest.mark.parametrize("dt", ["f32", "f64"])
@pytest.mark.parametrize("terms", ["all", "phs", "pnh", "force"])
@pytest.mark.parametrize("shape,h", SHAPES)
def test_mom_forcing_parity(mg, orc, shape, h, terms, dt):
    """q~ <- q~ - (dt / rho)(grad p_hs + grad p_nh + M F): every combination of present / absent terms, with and without the
    half-level output; p_hs sees the bottom extrapolation ghost, p_nh the halo factors given."""
    import torch
    nz, ny, nx = shape
    n = nx * ny * nz
    g = orc.grid(nx, ny, nz, h)
    Cf, qt0 = _fields(shape, dt, 80)
    _, qn = _fields(shape, dt, 90)
    grav, rho_l, rho_g, tstep = 9.81, 1000.0, 1.0, 0.1 * h
    rho = rho_l * Cf + rho_g * (1 - Cf)
    p_hs = quantise(1e3 * rng.normal(101, n).reshape(shape), dt) if terms in ("all", "phs") else None
    p_nh = quantise(1e3 * rng.normal(102, n).reshape(shape), dt) if terms in ("all", "pnh") else None
    F = tuple(quantise(1e3 * rng.normal(103 + c, n).reshape(shape), dt) for c in range(3)) if terms in ("all", "force") else None
    pbc = (N, D, N, N, N, D)
    # oracle side: sources s + s_t = -F, i.e. s_t = -F - (0, 0, -g rho); without a force field gravity enters only p_hs' ghost
    if F is not None:
        st = (-F[0], -F[1], -F[2] + grav * rho)
        ref = orc.mom_forcing(g, Cf, p_hs, p_nh, pbc, grav, st, rho_l, rho_g, tstep, qt0)
    else:
        z0 = np.zeros(shape)
        ref = orc.mom_forcing(g, Cf, p_hs, p_nh, pbc, grav, (z0, z0, grav * rho), rho_l, rho_g, tstep, qt0)
    dC = to_dev(Cf, dt)
    dev = lambda a: None if a is None else to_dev(a, dt)
    dq = [to_dev(a, dt) for a in qt0]
    dqn = [to_dev(a, dt) for a in qn]
    dqh = [torch.empty_like(dC) for _ in range(3)]
    mg.mom_forcing(dC, dev(p_hs), dev(p_nh), pbc, h, grav, None if F is None else [dev(a) for a in F], rho_l, rho_g, tstep, dq, dqn, dqh)
    scale = max(np.abs(r - a).max() for r, a in zip(ref, qt0))
    for c in range(3):
        # the increment is what is computed: bound its error relative to the increment, not to q~
        assert_close(as_f64(dq[c]) - qt0[c], ref[c] - qt0[c], (20 if dt == "f32" else 1e3) * TOL[dt])
        assert np.abs(as_f64(dqh[c]) - 0.5 * (qn[c] + ref[c])).max() <= (2e-6 if dt == "f32" else 1e-12) * max(scale, 1.0)
    dq2 = [to_dev(a, dt) for a in qt0]
    mg.mom_forcing(dC, dev(p_hs), dev(p_nh), pbc, h, grav, None if F is None else [dev(a) for a in F], rho_l, rho_g, tstep, dq2)
    for c in range(3):
        assert np.array_equal(as_f64(dq2[c]), as_f64(dq[c]))


@pytest.mark.parametrize("dt", ["f32", "f64"])
def test_hydrostatic_force_field(mg, orc, dt):
    """hydrostatic_rhs_force writes F = -(s + s_t) = (-s_tu, -s_tv, g rho - s_tw) next to b."""
    import torch
    n = 32
    h = 1.0 / n
    g = orc.grid(n, n, n, h)
    c = (np.arange(n) + 0.5) * h
    Z, Y, X = np.meshgrid(c, c, c, indexing="ij")
    r = np.sqrt((X - 0.5) ** 2 + (Y - 0.45) ** 2 + (Z - 0.65) ** 2)
    Cf = quantise(np.maximum(0.5 * (1 - np.tanh((r - 0.18) / (1.5 * h))), 0.5 * (1 + np.tanh((0.25 - Z) / (1.5 * h)))), dt)
    rho_l, rho_g, grav, sig = 1000.0, 1.0, 9.81, 0.0728
    b_ref, _, st = orc.hydrostatic_rhs(g, Cf, rho_l, rho_g, grav, sig)
    rho = rho_l * Cf + rho_g * (1 - Cf)
    dC = to_dev(Cf, dt)
    db = torch.empty_like(dC)
    dF = [torch.empty_like(dC) for _ in range(3)]
    mg.hydrostatic_rhs_force(dC, h, rho_l, rho_g, grav, sig, db, None, dF)
    assert_close(as_f64(db), b_ref, (5 * TOL[dt] if dt == "f32" else 1e-9))
    gx = np.gradient(Cf, h)
    band = np.sqrt(gx[0] ** 2 + gx[1] ** 2 + gx[2] ** 2) > 1.0
    for d, ref in enumerate((-st[0], -st[1], grav * rho - st[2])):
        # s_t = sigma kappa grad C; kappa is rounding-dominated where |grad C| is tiny (see the hydrostatic test): compare on the interface band
        assert_close(as_f64(dF[d])[band], ref[band], (2e-4 if dt == "f32" else 1e-9))


@pytest.mark.parametrize("dt", ["f32", "f64"])
def test_four_stage_step_parity(mg, orc, dt):
    """flow_time_step_full at 32^3 (4 levels): a collapsing water column under gravity with surface tension and free-slip
    walls, two steps from rest, every field against oracle.time_step_full."""
    import torch
    n, levels = 32, 4
    w = configs.config5(n, levels)
    g = orc.grid(n, n, n, w.h)
    Cf = quantise(w.fields["alpha"], dt)
    u, v, ww = (quantise(0.02 * w.fields[q], dt) for q in ("u", "v", "w"))
    grav, sig, tstep = 9.81, 0.0728, 0.05 * w.h
    code = mg.MG_F32 if dt == "f32" else mg.MG_F64
    s_hs = mg.mg_create((n, n, n, w.h), levels, BCP, code)
    s_nh = mg.mg_create((n, n, n, w.h), levels, BCP, code)
    dC, du, dv, dw = (to_dev(a, dt) for a in (Cf, u, v, ww))
    dphs, dpnh = torch.zeros_like(dC), torch.zeros_like(dC)
    p_nh = np.zeros(g.shape)
    tol = 1e-9
    for step in range(2):
        Cf, u, v, ww, p_hs, p_nh, cyc_o, rel_o = orc.time_step_full(g, Cf, u, v, ww, p_nh, levels, w.rho_l, w.rho_g, w.mu_l, w.mu_g,
                                                                    grav, sig, tstep, tol, 200, hs_tol=0.0, hs_cycles=20)
        status, cyc, rel = mg.flow_time_step_full(s_hs, s_nh, dC, du, dv, dw, dphs, dpnh, w.rho_l, w.rho_g, w.mu_l, w.mu_g, grav, sig,
                                                  tstep, tol, 200, 0.0, 20)
        assert status == mg.MG_OK and rel < tol and abs(cyc - cyc_o) <= 2
        lim = (step + 1) * (5e-5 if dt == "f32" else 1e-7)
        assert_close(as_f64(dphs), p_hs, 1e-4 if dt == "f32" else 1e-8)          # 20 fixed cycles on both sides
        assert_close(as_f64(dpnh), p_nh, lim * 5)
        assert_close(as_f64(dC), Cf, lim)
        vmax = max(np.abs(a).max() for a in (u, v, ww))
        for a, r in ((du, u), (dv, v), (dw, ww)):
            # a component can be much smaller than the velocity: bound its error by the velocity's magnitude
            assert np.linalg.norm(as_f64(a) - r) <= lim * np.sqrt(r.size) * vmax and np.abs(as_f64(a) - r).max() <= 10 * lim * vmax
    # the column has started to fall: the step is not a no-op
    assert np.abs(ww).max() > 0.5 * grav * tstep
    mg.mg_destroy(s_hs); mg.mg_destroy(s_nh)


@pytest.mark.parametrize("dt", ["f32", "f64"])
def test_material_mixtures_with_out_of_range_volume_fraction(mg, orc, dt):
    """Reading C7 (revised): rho and mu from C limited to [0, 1], everything else from C as it is.  C runs from -0.2 to 1.25 here
    (rho would be negative without the limit), through every entry point that forms a mixture."""
    import torch
    shape, h = (12, 16, 20), 0.05
    nz, ny, nx = shape
    n = nx * ny * nz
    g = orc.grid(nx, ny, nz, h)
    x, y, z = configs.centres(nx, ny, nz, 1.0)
    d = (0.7 * x / nx + 0.4 * y / ny + 0.6 * z / nz) - 0.8
    Cf = quantise(1.45 * (0.5 * (1 + np.tanh(d * 5.0)) + 0.0 * (x + y + z)) - 0.2 + 0.02 * rng.normal(3, n).reshape(shape), dt)
    assert Cf.min() < -0.1 and Cf.max() > 1.1
    q = tuple(quantise(0.3 * rng.normal(40 + c, n).reshape(shape) + 0.2, dt) for c in range(3))
    rho_l, rho_g, mu_l, mu_g, tstep, grav = 1000.0, 1.0, 1e-3, 1e-5, 0.1 * h, 9.81
    dC = to_dev(Cf, dt)
    dq = [to_dev(a, dt) for a in q]
    # k = 1 / rho in the solver: the operator built from it against the oracle's
    code = mg.MG_F32 if dt == "f32" else mg.MG_F64
    s = mg.mg_create((nx, ny, nz, h), 2, BCP, code)
    mg.mg_set_coefficient_from_vof(s, dC, rho_l, rho_g)
    dy = torch.empty_like(dC)
    mg.mg_apply_operator(s, dq[0], dy)
    assert_close(as_f64(dy), orc.apply_operator(g, BCP, orc.k_from_vof(Cf, rho_l, rho_g), q[0]), TOL[dt])
    mg.mg_destroy(s)
    # momentum predictor, forcing terms, hydrostatic right-hand side, the paper's stage-3 right-hand side
    vbc = orc.velocity_bc()
    qt_ref, qh_ref = orc.mom_predictor(g, Cf, q, q, rho_l, rho_g, mu_l, mu_g, tstep, vbc)
    dqt, dqh = [torch.empty_like(dC) for _ in range(3)], [torch.empty_like(dC) for _ in range(3)]
    mg.mom_predictor_bc(dC, dq, dq, vbc, h, rho_l, rho_g, mu_l, mu_g, tstep, dqt, dqh)
    for c in range(3):
        assert_close(as_f64(dqt[c]), qt_ref[c], TOL[dt])
        assert_close(as_f64(dqh[c]), qh_ref[c], TOL[dt])
    p_hs = quantise(1e3 * rng.normal(51, n).reshape(shape), dt)
    pbc = (N, D, N, N, N, D)
    rho = rho_l * np.clip(Cf, 0, 1) + rho_g * (1 - np.clip(Cf, 0, 1))
    z0 = np.zeros(shape)
    ref = orc.mom_forcing(g, Cf, p_hs, None, pbc, grav, (z0, z0, grav * rho), rho_l, rho_g, tstep, q)
    dq2 = [to_dev(a, dt) for a in q]
    mg.mom_forcing(dC, to_dev(p_hs, dt), None, pbc, h, grav, None, rho_l, rho_g, tstep, dq2)
    for c in range(3):
        assert_close(as_f64(dq2[c]) - q[c], ref[c] - q[c], (20 if dt == "f32" else 1e3) * TOL[dt])
    b_ref, _, _ = orc.hydrostatic_rhs(g, Cf, rho_l, rho_g, grav, 0.0)
    db = torch.empty_like(dC)
    mg.hydrostatic_rhs(dC, h, rho_l, rho_g, grav, 0.0, db)
    assert_close(as_f64(db), b_ref, 5 * TOL[dt] if dt == "f32" else 1e-9)
    mg.pressure_rhs_paper(dC, dq[0], dq[1], dq[2], h, rho_l, rho_g, tstep, db)
    assert_close(as_f64(db), orc.pressure_rhs_paper(g, Cf, q[0], q[1], q[2], rho_l, rho_g, tstep), 50 * TOL[dt])


def test_non_finite_right_hand_side_is_reported(mg):
    """A step that has blown up hands NaN to the solver: mg_solve and mg_pcg_solve must say MG_STAGNATED with a NaN residual, not
    MG_OK with residual 0 (||b|| = NaN fails every comparison)."""
    import torch
    n = 32
    for mixed in (1, 0):
        s = mg.mg_create((n, n, n, 1.0 / n), 3, BCP, mg.MG_F32)
        mg.mg_set_params(s, mixed_precision=mixed)
        b = torch.randn(n, n, n, device="cuda")
        b[3, 4, 5] = float("nan")
        x = torch.zeros_like(b)
        status, cycles, rel = mg.mg_solve(s, x, b, 1e-6, 10)
        assert status == mg.MG_STAGNATED and cycles == 0 and np.isnan(rel)
        status, its, rel = mg.mg_pcg_solve(s, x, b, 1e-6, 10)
        assert status == mg.MG_STAGNATED and its == 0 and np.isnan(rel)
        b[3, 4, 5] = float("inf")
        status, cycles, rel = mg.mg_solve(s, x, b, 0.0, 3)
        assert status == mg.MG_STAGNATED and np.isnan(rel)
        mg.mg_destroy(s)


@pytest.mark.parametrize("pressure_solver", [0, 1])
def test_collapsing_column_runs_and_behaves(mg, pressure_solver):
    """Qualitative check of the whole four-stage step ("a real collapsing-column run can be sanity-checked
    qualitatively"): a water column (width a = 0.25, height H = 0.5, 1000:1 density, free-slip box, 32^3) released from rest, 330
    steps to T* = t sqrt(2 g / a) = 3.  Not a parity test -- the oracle would need minutes -- but physics any correct
    implementation shows: the run stays finite (it does NOT without the limit of reading C7: rho < 0 at step 100), liquid volume
    is conserved to 0.1 %, the column height falls and the front advances monotonically, the front has crossed x = 3 a by
    T* = 3 at a speed between sqrt(g H) and Ritter's dam-break bound 2 sqrt(g H), and the liquid never moves faster than
    free fall from the column top allows, sqrt(2 g H), by more than 15 %.  Both stage-3 solvers (plain cycles, PCG) must do it."""
    import torch
    n, levels = 32, 4
    w = configs.config5(n, levels)
    h, grav, sig, a, H = w.h, 9.81, 0.0728, 0.25, 0.5
    s_hs = mg.mg_create((n, n, n, h), levels, BCP, mg.MG_F32)
    s_nh = mg.mg_create((n, n, n, h), levels, BCP, mg.MG_F32)
    for s in (s_hs, s_nh):
        mg.mg_set_params(s, cycles_per_defect=0)
    C = to_dev(w.fields["alpha"], "f32")
    u, v, ww = (torch.zeros_like(C) for _ in range(3))
    phs, pnh = torch.zeros_like(C), torch.zeros_like(C)
    tstep = 0.1 * h / 3.0
    vol0 = float(C.double().sum())
    xs = (np.arange(n) + 0.5) * h
    tstar = lambda t: t * np.sqrt(2 * grav / a)
    fronts, heights, t = [], [], 0.0
    while tstar(t) < 3.0:
        status, cyc, rel = mg.flow_time_step_full_ex(s_hs, s_nh, C, u, v, ww, phs, pnh, w.rho_l, w.rho_g, w.mu_l, w.mu_g, grav, sig, tstep,
                                                     1e-6, 100, 0.0, 20, (1, 1, 1, 1, 1, 0), pressure_solver)
        t += tstep
        assert status == mg.MG_OK and rel < 1e-6, (t, status, cyc, rel)
        if len(fronts) % 10 == 0 or tstar(t) >= 3.0:
            Cb, Cw = C[0, n // 2, :].cpu().numpy(), C[:, n // 2, 0].cpu().numpy()
            wet, col = np.where(Cb > 0.5)[0], np.where(Cw > 0.5)[0]
            assert wet.size and col.size
            speed = torch.sqrt(u * u + v * v + ww * ww)
            assert float((speed * (C > 0.5)).max()) <= 1.15 * np.sqrt(2 * grav * H)
            fronts.append((tstar(t), xs[wet.max()])); heights.append(xs[col.max()])
        else:
            fronts.append(None)
    fr = [f for f in fronts if f is not None]
    assert all(np.isfinite(float(q.abs().max())) for q in (C, u, v, ww))
    assert abs(float(C.double().sum()) / vol0 - 1) < 1e-3
    assert float(C.min()) > -0.15 and float(C.max()) < 1.15
    assert all(b[1] >= a_[1] - 1e-12 for a_, b in zip(fr, fr[1:])) and all(b <= a_ + 1e-12 for a_, b in zip(heights, heights[1:]))
    assert fr[-1][1] > 3.0 * a and heights[-1] < 0.6 * H
    # front speed over 1.2 <= T* <= 2.8 (after the initial acceleration, before the far wall)
    mid = [f for f in fr if 1.2 <= f[0] <= 2.8]
    vfront = (mid[-1][1] - mid[0][1]) / ((mid[-1][0] - mid[0][0]) / np.sqrt(2 * grav / a))
    assert np.sqrt(grav * H) < vfront < 2 * np.sqrt(grav * H), vfront
    mg.mg_destroy(s_hs); mg.mg_destroy(s_nh)


def test_full_step_argument_errors(mg):
    import torch
    n = 16
    s_hs = mg.mg_create((n, n, n, 1.0 / n), 2, BCP, mg.MG_F32)
    s_nh = mg.mg_create((n, n, n, 1.0 / n), 2, BCP, mg.MG_F32)
    f = [torch.zeros(n, n, n, device="cuda") for _ in range(6)]
    with pytest.raises(mg.MgError) as e:
        mg.flow_time_step_full_ex(s_hs, s_nh, *f, 1000.0, 1.0, 1e-3, 1e-5, 9.81, 0.07, 1e-3, 1e-6, 10, 0.0, 5, (1, 1, 1, 1, 1, 0), 2)
    assert e.value.code == mg.MG_EINVAL and "pressure_solver" in str(e.value)
    s_other = mg.mg_create((2 * n, n, n, 1.0 / n), 2, BCP, mg.MG_F32)
    with pytest.raises(mg.MgError) as e:
        mg.flow_time_step_full(s_other, s_nh, *f, 1000.0, 1.0, 1e-3, 1e-5, 9.81, 0.07, 1e-3, 1e-6, 10, 0.0, 5)
    assert e.value.code == mg.MG_EINVAL
    for s in (s_hs, s_nh, s_other):
        mg.mg_destroy(s)
