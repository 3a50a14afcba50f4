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
