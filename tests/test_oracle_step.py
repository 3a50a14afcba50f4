"""Pins of the ORDER in which the oracle composes one time step (oracle.time_step, oracle.time_step_paper;
PAPER.md:431-443 stage 2, 445-498 stage 3, 500-505 stage 4).  The stage functions themselves are pinned in
test_oracle_flow.py / test_oracle_multigrid.py; here the composition is pinned three ways:

  (a) against the stages chained by hand, in the paper's order, on inputs where a wrong order shows at O(1)
      (the hand side also evaluates the two plausible slips and asserts that they are far away);
  (b) by a property the mathematics fixes: a potential flow is removed by the projection, so stage 4 -- which
      advects with u^{n+1} (Eq. 16) -- leaves C almost unchanged, while advecting with the predictor
      velocity would not;
  (c) by the order of accuracy: two predictor iterations with the half-level velocity (Eqs. 45-46)
      are the midpoint rule, second order in dt; feeding q^n to the second iteration is forward Euler, first order.
"""
import numpy as np
import pytest

from workloads import configs

N, D = 0, 1
BC = (N, N, N, N, N, D)


def _rel(a, b):
    return float(np.linalg.norm(np.asarray(a) - np.asarray(b)) / max(np.linalg.norm(b), 1e-300))


def _case(n=16, levels=3, courant=0.6, div_amp=0.6):
    """Water column + swirl of config 5 at n^3 with a strongly divergent part added and a large time step, so that
    q~ differs from q^{n+1} and q^{n+1/2} from q^n at O(1)."""
    w = configs.config5(n, levels)
    x, y, z = configs.centres(n, n, n, w.h)
    u = w.fields["u"] + div_amp * np.sin(np.pi * x) * np.cos(np.pi * y) * np.cos(0.5 * np.pi * z)
    v = w.fields["v"] + div_amp * np.cos(np.pi * x) * np.sin(np.pi * y) * np.cos(0.5 * np.pi * z)
    ww = w.fields["w"] + div_amp * np.cos(np.pi * x) * np.cos(np.pi * y) * np.sin(0.5 * np.pi * z)
    w.dt = courant * w.h
    return w, np.ascontiguousarray(u), np.ascontiguousarray(v), np.ascontiguousarray(ww)


def _chain(orc, g, w, Cf, qn, levels, tol, max_cycles, second_pass_uses="half", advect_with="projected"):
    """Stages 2-4 written out in the paper's order from the pinned stage functions."""
    # stage 2: q^{n+1/2} = q^n for the first iteration; Eq. 45 gives q~, Eq. 46 the new half-level value;
    # "this process is repeated twice" with the updated q^{n+1/2}
    qt1, qhalf = orc.mom_predictor(g, Cf, qn, qn, w.rho_l, w.rho_g, w.mu_l, w.mu_g, w.dt)
    qt, _ = orc.mom_predictor(g, Cf, qhalf if second_pass_uses == "half" else qn, qn, w.rho_l, w.rho_g, w.mu_l, w.mu_g, w.dt)
    # stage 3 (reading C10): b = -(1/dt) D.q~, A(1/rho) p = b from p = 0, q^{n+1} = q~ - dt k G p (Eq. 54)
    k = orc.k_from_vof(Cf, w.rho_l, w.rho_g)
    b = orc.pressure_rhs(g, qt[0], qt[1], qt[2], w.dt)
    p, cycles, rel, _ = orc.solve(g, w.bc, k, np.zeros(g.shape), b, levels, tol, max_cycles)
    q1 = orc.project_velocity(g, w.bc, p, k, w.dt, qt[0], qt[1], qt[2])
    # stage 4: Eq. 55 with the residual of Eq. 16, which advects with u^{n+1}
    qa = q1 if advect_with == "projected" else qt
    _, Cn = orc.vof_residual(g, Cf, qa[0], qa[1], qa[2], w.dt)
    return Cn, q1, p, qt, qhalf


def test_time_step_equals_the_stages_chained_by_hand(orc):
    w, u, v, ww = _case()
    n, levels = w.nx, w.levels
    g = orc.grid(n, n, n, w.h)
    Cf = w.fields["alpha"]
    got = orc.time_step(g, w.bc, Cf, u, v, ww, levels, w.rho_l, w.rho_g, w.mu_l, w.mu_g, w.dt, 1e-10, 300)
    Cn, q1, p, qt, qhalf = _chain(orc, g, w, Cf, (u, v, ww), levels, 1e-10, 300)
    assert got[6] < 1e-10
    assert _rel(got[0], Cn) < 1e-13 and _rel(got[4], p) < 1e-13
    for a, b in zip(got[1:4], q1):
        assert _rel(a, b) < 1e-13
    # the inputs discriminate: the half-level velocity is not q^n, the projected velocity is not q~ ...
    assert _rel(np.stack(qhalf), np.stack((u, v, ww))) > 0.02
    assert _rel(np.stack(q1), np.stack(qt)) > 0.2
    # ... and each of the two slips moves the result far beyond the tolerance above
    Cn_a, _, _, _, _ = _chain(orc, g, w, Cf, (u, v, ww), levels, 1e-10, 300, advect_with="predictor")
    assert _rel(Cn_a - Cf, Cn - Cf) > 0.2
    Cn_b, q1_b, _, _, _ = _chain(orc, g, w, Cf, (u, v, ww), levels, 1e-10, 300, second_pass_uses="n")
    assert _rel(np.stack(q1_b), np.stack(q1)) > 1e-3 and _rel(Cn_b - Cf, Cn - Cf) > 1e-3


def test_time_step_paper_equals_the_stages_chained_by_hand(orc):
    """time_step_paper: stage 2 as above; stage 3 = Eqs. 52-54 carried out `passes` times, each pass a fixed
    number of constant-coefficient cycles from a zero guess on the CURRENT velocity, p_nh accumulating; stage 4
    with the final velocity."""
    w, u, v, ww = _case(courant=0.3, div_amp=0.3)
    n, levels = w.nx, w.levels
    g = orc.grid(n, n, n, w.h)
    Cf = w.fields["alpha"]
    qn = (u, v, ww)
    for passes, cycles in ((2, 6), (1, 4)):
        got = orc.time_step_paper(g, w.bc, Cf, u, v, ww, levels, w.rho_l, w.rho_g, w.mu_l, w.mu_g, w.dt, cycles, passes)
        _, qhalf = orc.mom_predictor(g, Cf, qn, qn, w.rho_l, w.rho_g, w.mu_l, w.mu_g, w.dt)
        qt, _ = orc.mom_predictor(g, Cf, qhalf, qn, w.rho_l, w.rho_g, w.mu_l, w.mu_g, w.dt)
        k = orc.k_from_vof(Cf, w.rho_l, w.rho_g)
        q = qt
        p = np.zeros(g.shape)
        for _ in range(passes):
            b = orc.pressure_rhs_paper(g, Cf, q[0], q[1], q[2], w.rho_l, w.rho_g, w.dt)
            dp, _, _, _ = orc.solve(g, w.bc, None, np.zeros(g.shape), b, levels, 0.0, cycles)
            q = orc.project_velocity(g, w.bc, dp, k, w.dt, q[0], q[1], q[2])      # Eq. 54: dq = -dt grad(dp) / rho
            p = p + dp
        _, Cn = orc.vof_residual(g, Cf, q[0], q[1], q[2], w.dt)
        assert _rel(got[0], Cn) < 1e-13 and _rel(got[4], p) < 1e-13
        for a, b in zip(got[1:4], q):
            assert _rel(a, b) < 1e-13
        # discriminating: the second pass changes the velocity, the slips change C
        _, Cn_a = orc.vof_residual(g, Cf, qt[0], qt[1], qt[2], w.dt)
        assert _rel(Cn_a - Cf, Cn - Cf) > 0.05
        qt_b, _ = orc.mom_predictor(g, Cf, qn, qn, w.rho_l, w.rho_g, w.mu_l, w.mu_g, w.dt)
        assert _rel(np.stack(qt_b), np.stack(qt)) > 1e-3


@pytest.mark.parametrize("step", ["time_step", "time_step_paper"])
def test_stage4_advects_with_the_projected_velocity(orc, step):
    """Eq. 16: the volume fraction is advected by u^{n+1}.  With equal densities (k constant) a potential
    flow q^n = grad(phi), phi obeying the pressure boundary conditions, is removed by the projection up to the
    O(h^2) mismatch between D.G and the compact Laplacian and the O(dt) change in the predictor: C barely moves.
    Advected with the predictor velocity q~ it would move by dt q~.grad C."""
    n, levels = 16, 3
    h = 1.0 / n
    g = orc.grid(n, n, n, h)
    x, y, z = configs.centres(n, n, n, h)
    amp = 1.0 / np.pi
    u = -amp * np.pi * np.sin(np.pi * x) * np.cos(np.pi * y) * np.cos(0.5 * np.pi * z)          # grad of
    v = -amp * np.pi * np.cos(np.pi * x) * np.sin(np.pi * y) * np.cos(0.5 * np.pi * z)          # amp cos cos cos(pi z / 2):
    w = -amp * 0.5 * np.pi * np.cos(np.pi * x) * np.cos(np.pi * y) * np.sin(0.5 * np.pi * z)    # d/dn = 0 on walls, 0 on top
    u, v, w = (np.ascontiguousarray(a + 0 * (x + y + z)) for a in (u, v, w))
    Cf = np.ascontiguousarray(0.5 * (1 + np.tanh((0.45 - x + 0.2 * y - 0.1 * z) / (2.5 * h))))
    rho, mu, dt = 3.0, 1e-4, 0.05 * h
    if step == "time_step":
        out = orc.time_step(g, BC, Cf, u, v, w, levels, rho, rho, mu, mu, dt, 1e-11, 300)
    else:
        out = orc.time_step_paper(g, BC, Cf, u, v, w, levels, rho, rho, mu, mu, dt, cycles=40, passes=2)
    Cn, u1, v1, w1 = out[:4]
    speed = np.sqrt(u * u + v * v + w * w).max()
    assert np.sqrt(u1 * u1 + v1 * v1 + w1 * w1).max() < 0.2 * speed                      # the projection removed it
    qn = (u, v, w)
    qt, qh = orc.mom_predictor(g, Cf, qn, qn, rho, rho, mu, mu, dt)
    qt, _ = orc.mom_predictor(g, Cf, qh, qn, rho, rho, mu, mu, dt)
    _, C_wrong = orc.vof_residual(g, Cf, qt[0], qt[1], qt[2], dt)
    assert np.linalg.norm(Cn - Cf) < 0.2 * np.linalg.norm(C_wrong - Cf)


def test_two_predictor_iterations_are_second_order_in_dt(orc):
    """Stage 2: iteration 1 evaluates the residual at q^n, iteration 2 at q^{n+1/2} = (q^n + q~)/2 -- the
    explicit midpoint rule for dq/dt = -s(q)/rho.  Its one-step error against a finely sub-stepped RK4 integration of
    the same semi-discrete system falls 8x when dt is halved; evaluating iteration 2 at q^n again (forward Euler) gives
    4x.  Measured through time_step itself: the projection that follows is linear in q~ and independent of dt."""
    n, levels = 12, 2
    w = configs.config5(n, levels)
    g = orc.grid(n, n, n, w.h)
    Cf = np.full(g.shape, 0.5)                    # uniform fluid: k constant, VoF stage inert; the momentum stage is what is tested
    rho_l = rho_g = 2.0
    mu_l = mu_g = 0.05                            # smooth regime: viscous term dominates the (non-smooth) PG coefficient
    qn = tuple(np.ascontiguousarray(w.fields[c]) for c in ("u", "v", "w"))

    def rhs(q):                                   # -s(q)/rho from the pinned stage function (Eq. 45 with q_half = q_n = q)
        qt, _ = orc.mom_predictor(g, Cf, q, q, rho_l, rho_g, mu_l, mu_g, 1.0)
        return tuple(a - b for a, b in zip(qt, q))

    def rk4(q, dt, sub):
        hh = dt / sub
        ax = lambda q, s, k: tuple(np.ascontiguousarray(a + s * b) for a, b in zip(q, k))
        for _ in range(sub):
            k1 = rhs(q); k2 = rhs(ax(q, hh / 2, k1)); k3 = rhs(ax(q, hh / 2, k2)); k4 = rhs(ax(q, hh, k3))
            q = tuple(np.ascontiguousarray(a + hh / 6 * (b + 2 * c + 2 * d + e)) for a, b, c, d, e in zip(q, k1, k2, k3, k4))
        return q

    k = orc.k_from_vof(Cf, rho_l, rho_g)

    def project(q, dt):
        b = orc.pressure_rhs(g, q[0], q[1], q[2], dt)
        p, _, rel, _ = orc.solve(g, BC, k, np.zeros(g.shape), b, levels, 1e-13, 400)
        assert rel < 1e-12
        return orc.project_velocity(g, BC, p, k, dt, q[0], q[1], q[2])

    errs = []
    for dt in (0.4 * w.h, 0.2 * w.h):
        got = orc.time_step(g, BC, Cf, qn[0], qn[1], qn[2], levels, rho_l, rho_g, mu_l, mu_g, dt, 1e-13, 400)
        ref = project(rk4(qn, dt, 8), dt)
        errs.append(np.linalg.norm(np.stack(got[1:4]) - np.stack(ref)))
    assert errs[0] / errs[1] > 6.5, errs          # 8 for the midpoint rule, 4 for forward Euler
