"""GPU parity of the explicit stencil residuals (a8-a10) and of the config-5 time step against
the fp64 CPU oracle, through the C ABI.  Tolerances: relative L2 <= 1e-5 (fp32) / 1e-12 (fp64)
per kernel pass, as for the sweeps (BASELINE.json)."""
import numpy as np
import pytest

from workloads import configs, rng
from test_gpu_mg import TOL, as_f64, mg, quantise, rel_l2, to_dev  # noqa: F401
from _parity import assert_close  # noqa: E402

pytestmark = pytest.mark.gpu
N, D, H0 = configs.BC_NEUMANN, configs.BC_DIRICHLET, configs.BC_DIRICHLET_HALO


def flow_fields(n, dt, solenoidal=True):
    """Water-column alpha and a divergence-free velocity, the structure of config 5, at n^3."""
    w = configs.config5(n, 3)
    f = w.fields
    if not solenoidal:
        f["u"], f["v"], f["w"] = configs.random_velocity((71, 72, 73), w.shape)
    return w, tuple(quantise(f[q], dt) for q in ("alpha", "u", "v", "w"))


@pytest.mark.parametrize("dt", ["f32", "f64"])
@pytest.mark.parametrize("shape,h", [((24, 24, 24), 1.0 / 24), ((10, 36, 68), 1.0 / 68), ((40, 40, 40), (0.02, 0.025, 0.03))])
def test_vof_residual_parity(mg, orc, shape, h, dt):
    import torch
    nz, ny, nx = shape
    hh = h if isinstance(h, tuple) else (h, h, h)
    g = orc.grid(nx, ny, nz, *hh)
    # a smeared interface crossing the box obliquely, so every branch (override, w+, w-, clips) is taken
    x, y, z = configs.centres(nx, ny, nz, 1.0)
    d = (0.6 * x / nx + 0.5 * y / ny + 0.62 * z / nz) - 0.8
    Cf = quantise(0.5 * (1 + np.tanh(d * 6.0)) + 0.0 * (x + y + z), dt)
    n = Cf.size
    u, v, w = (quantise(0.3 * rng.normal(40 + c, n).reshape(shape) + 0.5, dt) for c in range(3))
    tstep = 0.1 * min(hh)
    s_ref, c_ref = orc.vof_residual(g, Cf, u, v, w, tstep)
    dC, du, dv, dw = (to_dev(a, dt) for a in (Cf, u, v, w))
    ds, dc = torch.empty_like(dC), torch.empty_like(dC)
    mg.vof_residual(dC, du, dv, dw, hh, tstep, ds, dc)
    assert_close(as_f64(ds), s_ref, 5 * TOL[dt])  # 3 chained passes (adv -> coefficients -> diffusion)
    assert_close(as_f64(dc), c_ref, TOL[dt])
    # outputs are optional one at a time
    dc2 = torch.empty_like(dC)
    mg.vof_residual(dC, du, dv, dw, hh, tstep, None, dc2)
    assert torch.equal(dc, dc2)


@pytest.mark.parametrize("dt", ["f32", "f64"])
def test_vof_trivial_inputs(mg, dt):
    import torch
    tdt = torch.float32 if dt == "f32" else torch.float64
    C_ = torch.full((16, 16, 16), 0.5, device="cuda", dtype=tdt)
    q = torch.ones_like(C_)
    s = torch.empty_like(C_)
    mg.vof_residual(C_, q, q, q, 1.0 / 16, 0.01, s, None)
    assert float(s.abs().max()) <= 1e-5 * 16                # uniform C: residual vanishes (to rounding of |q| C / h)
    Cg = torch.rand(16, 16, 16, device="cuda", dtype=tdt)
    z = torch.zeros_like(Cg)
    mg.vof_residual(Cg, z, z, z, 1.0 / 16, 0.01, s, None)
    assert float(s.abs().max()) == 0.0                      # q = 0: no advection, k_abs = k- = 0


@pytest.mark.parametrize("dt", ["f32", "f64"])
@pytest.mark.parametrize("n", [24, 40])
def test_momentum_rhs_projection_parity(mg, orc, n, dt):
    import torch
    w, (alpha, u, v, ww) = flow_fields(n, dt)
    g = orc.grid(n, n, n, w.h)
    bc = w.bc
    # momentum predictor, both outputs, half-level velocity different from level n
    qn = (u, v, ww)
    qh = tuple(quantise(0.9 * a + 0.05, dt) for a in qn)
    qt_ref, qhn_ref = orc.mom_predictor(g, alpha, qh, qn, w.rho_l, w.rho_g, w.mu_l, w.mu_g, w.dt)
    dC = to_dev(alpha, dt)
    dqn = [to_dev(a, dt) for a in qn]; dqh = [to_dev(a, dt) for a in qh]
    dqt = [torch.empty_like(dC) for _ in range(3)]; dqhn = [torch.empty_like(dC) for _ in range(3)]
    mg.mom_predictor(dC, dqh, dqn, w.h, w.rho_l, w.rho_g, w.mu_l, w.mu_g, w.dt, dqt, dqhn)
    for c in range(3):
        assert_close(as_f64(dqt[c]), qt_ref[c], TOL[dt])
        assert_close(as_f64(dqhn[c]), qhn_ref[c], TOL[dt])
    # pressure RHS
    b_ref = orc.pressure_rhs(g, u, v, ww, w.dt)
    db = torch.empty_like(dC)
    mg.pressure_rhs(dqn[0], dqn[1], dqn[2], w.h, w.dt, db)
    assert_close(as_f64(db), b_ref, TOL[dt] * (50 if dt == "f32" else 1e3))  # divergence of a solenoidal field: cancellation
    ur, vr, wr = (quantise(rng.normal(90 + c, alpha.size).reshape(alpha.shape), dt) for c in range(3))
    b_ref = orc.pressure_rhs(g, ur, vr, wr, w.dt)
    mg.pressure_rhs(to_dev(ur, dt), to_dev(vr, dt), to_dev(wr, dt), w.h, w.dt, db)
    assert_close(as_f64(db), b_ref, TOL[dt])
    # projection with the solver's BC factors on p
    p = quantise(rng.normal(95, alpha.size).reshape(alpha.shape), dt)
    k = quantise(orc.k_from_vof(alpha, w.rho_l, w.rho_g), dt)
    for bcs in (bc, (D, N, H0, D, N, H0)):
        u_ref, v_ref, w_ref = orc.project_velocity(g, bcs, p, k, w.dt, u, v, ww)
        du, dv, dw = to_dev(u, dt), to_dev(v, dt), to_dev(ww, dt)
        mg.project_velocity(to_dev(p, dt), to_dev(k, dt), w.h, bcs, w.dt, du, dv, dw)
        for a, r in ((du, u_ref), (dv, v_ref), (dw, w_ref)):
            assert_close(as_f64(a), r, TOL[dt])


@pytest.mark.parametrize("dt", ["f32", "f64"])
def test_time_step_parity(mg, orc, dt):
    """Config 5 at reduced size (32^3, 4 levels): two full time steps against the oracle."""
    n, levels = 32, 4
    w = configs.config5(n, levels)
    g = orc.grid(n, n, n, w.h)
    Cf, u, v, ww = (quantise(w.fields[q], dt) for q in ("alpha", "u", "v", "w"))
    s = mg.mg_create((n, n, n, w.h), levels, w.bc, mg.MG_F32 if dt == "f32" else mg.MG_F64)
    dC, du, dv, dw = (to_dev(a, dt) for a in (Cf, u, v, ww))
    import torch
    dp = torch.empty_like(dC)
    tol = 1e-9    # both sides driven well below config 5's 1e-6 so the comparison is of converged pressures
    for step in range(2):
        Cf, u, v, ww, p, cyc_o, rel_o = orc.time_step(g, w.bc, Cf, u, v, ww, levels, w.rho_l, w.rho_g, w.mu_l, w.mu_g,
                                                      w.dt, tol, 200)
        status, cyc, rel = mg.flow_time_step(s, dC, du, dv, dw, dp, w.rho_l, w.rho_g, w.mu_l, w.mu_g, w.dt, tol, 200)
        assert status == mg.MG_OK and rel < tol and abs(cyc - cyc_o) <= 2
        lim = (step + 1) * (2e-5 if dt == "f32" else 1e-7)
        assert_close(as_f64(dp), p, lim * 5)
        for a, r in ((dC, Cf), (du, u), (dv, v), (dw, ww)):
            assert_close(as_f64(a), r, lim)
    mg.mg_destroy(s)


@pytest.mark.parametrize("dt", ["f32", "f64"])
def test_time_step_pcg_parity(mg, orc, dt):
    """Config 5 at 32^3 with the pressure solved by V-cycle-preconditioned CG (flow_time_step_pcg): two steps."""
    import torch
    n, levels = 32, 4
    w = configs.config5(n, levels)
    g = orc.grid(n, n, n, w.h)
    Cf, u, v, ww = (quantise(w.fields[q], dt) for q in ("alpha", "u", "v", "w"))
    s = mg.mg_create((n, n, n, w.h), levels, w.bc, mg.MG_F32 if dt == "f32" else mg.MG_F64)
    dC, du, dv, dw = (to_dev(a, dt) for a in (Cf, u, v, ww))
    dp = torch.empty_like(dC)
    tol = 1e-9
    for step in range(2):
        Cf, u, v, ww, p, it_o, rel_o = orc.time_step(g, w.bc, Cf, u, v, ww, levels, w.rho_l, w.rho_g, w.mu_l, w.mu_g,
                                                     w.dt, tol, 200, solver="pcg")
        status, its, rel = mg.flow_time_step_pcg(s, dC, du, dv, dw, dp, w.rho_l, w.rho_g, w.mu_l, w.mu_g, w.dt, tol, 200)
        assert status == mg.MG_OK and rel < tol and abs(its - it_o) <= 2
        lim = (step + 1) * (2e-5 if dt == "f32" else 1e-7)
        assert_close(as_f64(dp), p, lim * 5)
        for a, r in ((dC, Cf), (du, u), (dv, v), (dw, ww)):
            assert_close(as_f64(a), r, lim)
    mg.mg_destroy(s)


# ---------------------------------------------------------------- the 5-point detectors of Eq. 34
@pytest.mark.parametrize("dt", ["f32", "f64"])
@pytest.mark.parametrize("shape,h", [((24, 24, 24), 1.0 / 24), ((10, 36, 68), 1.0 / 68), ((40, 40, 40), (0.02, 0.025, 0.03)),
                                     ((12, 10, 22), 0.05), ((3, 4, 6), 0.1)])
def test_vof_residual_five_point_detectors(mg, orc, shape, h, dt):
    """vof_residual_ex(detector = 5) against the oracle's: vector and scalar kernels, several z chunks, a ragged tail, and a
    grid thinner than the detector's reach (reflection lands two cells inside)."""
    import torch
    nz, ny, nx = shape
    hh = h if isinstance(h, tuple) else (h, h, h)
    g = orc.grid(nx, ny, nz, *hh)
    x, y, z = configs.centres(nx, ny, nz, 1.0)
    d = (0.6 * x / nx + 0.5 * y / ny + 0.62 * z / nz) - 0.8
    n = nx * ny * nz
    # smeared interface plus small wiggles: extrema next to monotone cells, where Eq. 34 and Eq. 33 disagree
    Cf = quantise(0.5 * (1 + np.tanh(d * 6.0)) + 0.03 * np.sin(1.7 * x + 2.3 * y + 1.1 * z), dt)
    u, v, w = (quantise(0.3 * rng.normal(40 + c, n).reshape(shape) + 0.5, dt) for c in range(3))
    tstep = 0.1 * min(hh)
    s_ref, c_ref = orc.vof_residual(g, Cf, u, v, w, tstep, detector=5)
    s3, _ = orc.vof_residual(g, Cf, u, v, w, tstep, detector=3)
    assert np.abs(s_ref - s3).max() > 1e-3 * np.abs(s3).max()                 # the option matters on this input
    dC, du, dv, dw = (to_dev(a, dt) for a in (Cf, u, v, w))
    ds, dc = torch.empty_like(dC), torch.empty_like(dC)
    mg.vof_residual_ex(dC, du, dv, dw, hh if isinstance(h, tuple) else h, tstep, 5, ds, dc)
    assert_close(as_f64(ds), s_ref, 5 * TOL[dt])
    assert_close(as_f64(dc), c_ref, TOL[dt])
    with pytest.raises(mg.MgError):
        mg.vof_residual_ex(dC, du, dv, dw, hh if isinstance(h, tuple) else h, tstep, 4, ds, dc)


# ---------------------------------------------------------------- the paper's own stage 3
@pytest.mark.parametrize("dt", ["f32", "f64"])
@pytest.mark.parametrize("shape,h", [((24, 24, 24), 1.0 / 24), ((10, 36, 68), (0.02, 0.025, 0.03))])
def test_pressure_rhs_paper_parity(mg, orc, shape, h, dt):
    import torch
    nz, ny, nx = shape
    hh = h if isinstance(h, tuple) else (h, h, h)
    g = orc.grid(nx, ny, nz, *hh)
    n = nx * ny * nz
    Cf = quantise(rng.uniform01(71, n).reshape(shape), dt)
    u, v, w = (quantise(rng.normal(72 + c, n).reshape(shape), dt) for c in range(3))
    b_ref = orc.pressure_rhs_paper(g, Cf, u, v, w, 1000.0, 1.0, 0.01)
    db = torch.empty(shape, device="cuda", dtype=torch.float32 if dt == "f32" else torch.float64)
    mg.pressure_rhs_paper(to_dev(Cf, dt), to_dev(u, dt), to_dev(v, dt), to_dev(w, dt), hh, 1000.0, 1.0, 0.01, db)
    # rho q - q rho cancels to rho div q: the same cancellation allowance as the divergence right-hand side
    assert_close(as_f64(db), b_ref, TOL[dt] * (50 if dt == "f32" else 1e3))


@pytest.mark.parametrize("dt", ["f32", "f64"])
def test_time_step_paper_parity(mg, orc, dt):
    """Config 5 at 32^3 with the paper's stage 3 (constant-coefficient Laplacian, 2 passes x 20 cycles): two steps."""
    import torch
    n, levels = 32, 4
    w = configs.config5(n, levels)
    g = orc.grid(n, n, n, w.h)
    Cf, u, v, ww = (quantise(w.fields[q], dt) for q in ("alpha", "u", "v", "w"))
    s = mg.mg_create((n, n, n, w.h), levels, w.bc, mg.MG_F32 if dt == "f32" else mg.MG_F64)
    dC, du, dv, dw = (to_dev(a, dt) for a in (Cf, u, v, ww))
    dp = torch.empty_like(dC)
    for step in range(2):
        Cf, u, v, ww, p, rel_o = orc.time_step_paper(g, w.bc, Cf, u, v, ww, levels, w.rho_l, w.rho_g, w.mu_l, w.mu_g, w.dt)
        rel = mg.flow_time_step_paper(s, dC, du, dv, dw, dp, w.rho_l, w.rho_g, w.mu_l, w.mu_g, w.dt, 20, 2)
        lim = (step + 1) * (1e-4 if dt == "f32" else 1e-7)
        assert abs(rel - rel_o) <= 0.05 * rel_o + 1e-12
        assert_close(as_f64(dp), p, lim * 5)
        for a, r in ((dC, Cf), (du, u), (dv, v), (dw, ww)):
            assert_close(as_f64(a), r, lim)
    mg.mg_destroy(s)


# ---------------------------------------------------------------- stage 1, hydrostatic + surface-tension pressure
@pytest.mark.parametrize("dt", ["f32", "f64"])
def test_hydrostatic_rhs_and_solve_parity(mg, orc, dt):
    """A drop (C = 1 inside) above a water layer: curvature, right-hand side of Eq. 44 with the bottom boundary fold, and the
    p_hs it gives after 20 constant-coefficient V-cycles (the paper's fixed count)."""
    import torch
    n, levels = 32, 4
    h = 1.0 / n
    g = orc.grid(n, n, n, h)
    c = (np.arange(n) + 0.5) * h
    Z, Y, X = np.meshgrid(c, c, c, indexing="ij")
    r = np.sqrt((X - 0.5) ** 2 + (Y - 0.45) ** 2 + (Z - 0.65) ** 2)
    Cf = np.maximum(0.5 * (1 - np.tanh((r - 0.18) / (1.5 * h))), 0.5 * (1 + np.tanh((0.25 - Z) / (1.5 * h))))
    Cf = quantise(Cf, dt)
    rho_l, rho_g, grav, sig = 1000.0, 1.0, 9.81, 0.0728
    b_ref, kap_ref, _ = orc.hydrostatic_rhs(g, Cf, rho_l, rho_g, grav, sig)
    dC = to_dev(Cf, dt)
    db, dk = torch.empty_like(dC), torch.empty_like(dC)
    mg.hydrostatic_rhs(dC, h, rho_l, rho_g, grav, sig, db, dk)
    # kappa divides by |grad C|, tiny away from the interfaces, where rounding decides it: compare where there is an interface
    gx = np.gradient(Cf, h)
    band = np.sqrt(gx[0] ** 2 + gx[1] ** 2 + gx[2] ** 2) > 1.0
    assert band.sum() > 1000
    assert_close(as_f64(dk)[band], kap_ref[band], (2e-4 if dt == "f32" else 1e-9))
    assert_close(as_f64(db), b_ref, (5 * TOL[dt] if dt == "f32" else 1e-9))
    bc = (N, N, N, N, N, D)
    s = mg.mg_create((n, n, n, h), levels, bc, mg.MG_F32 if dt == "f32" else mg.MG_F64)
    dp = torch.zeros_like(dC)
    mg.mg_solve(s, dp, db, 0.0, 20)
    p_ref, _, _, _ = orc.solve(g, bc, None, np.zeros(g.shape), b_ref, levels, 0.0, 20)
    assert_close(as_f64(dp), p_ref, (1e-4 if dt == "f32" else 1e-8))
    # physics of the result: hydrostatic at the bottom of the water layer, higher pressure inside the drop
    p = as_f64(dp)
    assert abs((p[0, 4, 4] - p[2, 4, 4]) / (2 * h) - rho_l * grav) <= 0.02 * rho_l * grav
    mg.mg_destroy(s)


# ---------------------------------------------------------------- pack widths of the marching kernels
def _offset_dev(a, dt):
    """Device copy of `a` whose first element sits 1 element past a 16-byte boundary (forces the scalar kernels)."""
    import torch
    t = to_dev(np.concatenate([[0.0], a.ravel()]), dt)
    return t[1:].view(a.shape)


@pytest.mark.parametrize("dt", ["f32", "f64"])
@pytest.mark.parametrize("shape,unaligned", [((9, 14, 30), False), ((7, 10, 15), False), ((6, 12, 260), False), ((8, 12, 32), True)])
def test_explicit_kernels_every_pack_width(mg, orc, shape, unaligned, dt):
    """The marching kernels own 4 (fp32) / 2 (fp64) x points per thread when nx allows it and every field is 16-byte aligned,
    and 1 otherwise: nx = 30 (fp32 scalar, fp64 pairs), nx = 15 (scalar), nx = 260 (a partial 128-wide block), and an
    aligned shape handed over in misaligned buffers (scalar).  Every explicit kernel against the oracle."""
    import torch
    nz, ny, nx = shape
    hh = (1.0 / nx, 1.0 / nx, 1.0 / nx)
    g = orc.grid(nx, ny, nz, *hh)
    n = nx * ny * nz
    dev = (lambda a: _offset_dev(a, dt)) if unaligned else (lambda a: to_dev(a, dt))
    out = (lambda: dev(np.zeros(shape)))
    x, y, z = configs.centres(nx, ny, nz, 1.0)
    Cf = quantise(0.5 * (1 + np.tanh(((0.6 * x / nx + 0.5 * y / ny + 0.62 * z / nz) - 0.8) * 6.0)), dt)
    u, v, w = (quantise(0.3 * rng.normal(140 + c, n).reshape(shape) + 0.5, dt) for c in range(3))
    tstep = 0.1 * hh[0]
    dC, du, dv, dw = (dev(a) for a in (Cf, u, v, w))
    # VoF residual
    s_ref, c_ref = orc.vof_residual(g, Cf, u, v, w, tstep)
    ds, dc = out(), out()
    mg.vof_residual(dC, du, dv, dw, hh, tstep, ds, dc)
    assert_close(as_f64(ds), s_ref, 5 * TOL[dt])
    assert_close(as_f64(dc), c_ref, TOL[dt])
    # momentum predictor
    qh = tuple(quantise(0.9 * a + 0.05, dt) for a in (u, v, w))
    qt_ref, qhn_ref = orc.mom_predictor(g, Cf, qh, (u, v, w), 1000.0, 1.0, 1e-3, 1.8e-5, tstep)
    dqt, dqhn = [out() for _ in range(3)], [out() for _ in range(3)]
    mg.mom_predictor(dC, [dev(a) for a in qh], [du, dv, dw], hh, 1000.0, 1.0, 1e-3, 1.8e-5, tstep, dqt, dqhn)
    for c in range(3):
        assert_close(as_f64(dqt[c]), qt_ref[c], TOL[dt])
        assert_close(as_f64(dqhn[c]), qhn_ref[c], TOL[dt])
    # pressure right-hand sides
    db = out()
    mg.pressure_rhs(du, dv, dw, hh, tstep, db)
    assert_close(as_f64(db), orc.pressure_rhs(g, u, v, w, tstep), TOL[dt])
    mg.pressure_rhs_paper(dC, du, dv, dw, hh, 1000.0, 1.0, tstep, db)
    # rho q - q rho cancels to rho div q: the cancellation allowance of test_pressure_rhs_paper_parity
    assert_close(as_f64(db), orc.pressure_rhs_paper(g, Cf, u, v, w, 1000.0, 1.0, tstep), TOL[dt] * (50 if dt == "f32" else 1e3))
    # projection with mixed halo factors
    p = quantise(rng.normal(195, n).reshape(shape), dt)
    k = quantise(orc.k_from_vof(Cf, 1000.0, 1.0), dt)
    bcs = (D, N, H0, D, N, H0)
    refs = orc.project_velocity(g, bcs, p, k, tstep, u, v, w)
    pu, pv, pw = dev(u), dev(v), dev(w)
    mg.project_velocity(dev(p), dev(k), hh, bcs, tstep, pu, pv, pw)
    for a, r in zip((pu, pv, pw), refs):
        assert_close(as_f64(a), r, TOL[dt])
    # stage 1
    b_ref, kap_ref, _ = orc.hydrostatic_rhs(g, Cf, 1000.0, 1.0, 9.81, 0.07)
    dk = out()
    mg.hydrostatic_rhs(dC, hh[0], 1000.0, 1.0, 9.81, 0.07, db, dk)
    # kappa divides by |grad C|, tiny away from the interface, where rounding decides it: compare where there is an interface
    gr = np.gradient(Cf, hh[0])
    band = np.sqrt(gr[0] ** 2 + gr[1] ** 2 + gr[2] ** 2) > 1.0
    assert band.sum() > 100
    assert_close(as_f64(dk)[band], kap_ref[band], (2e-4 if dt == "f32" else 1e-9))
    assert_close(as_f64(db), b_ref, (5 * TOL[dt] if dt == "f32" else 1e-9))
