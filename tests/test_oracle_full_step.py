"""Pins of the oracle's four-stage time step: free-slip velocity halos
(P:538), the forcing terms of Eq. 18 and the composition oracle.time_step_full.  The paper has no worked
example for any of this; the pins are closed forms, hand reductions and physical invariants."""
import numpy as np
import pytest

from workloads import configs

N, D = 0, 1
BCP = (N, N, N, N, N, D)


def _xyz(g):
    x, y, z = configs.centres(g.nx, g.ny, g.nz, g.hx)
    o = np.zeros(g.shape)
    return x + o, y + o, z + o


def test_free_slip_halo_codes(orc):
    """Walls on the sides and the bottom, open top: the component normal to a wall is odd about it."""
    assert orc.velocity_bc() == orc.FREE_SLIP_OPEN_TOP
    assert orc.velocity_bc((0,) * 6) == (0,) * 18
    vbc = orc.velocity_bc((1, 0, 0, 1, 1, 1))
    assert vbc[0:6] == (1, 0, 0, 0, 0, 0) and vbc[6:12] == (0, 0, 0, 1, 0, 0) and vbc[12:18] == (0, 0, 0, 0, 1, 1)


def test_wall_divergence_of_a_linear_flow_is_exact(orc):
    """u = a x, v = b y, w = c z vanish on the walls x = 0, y = 0, z = 0 and are linear: with the odd halo the FE
    divergence is a + b + c in EVERY cell, wall cells included; with copy halos the wall cells see half a derivative."""
    n, h, dt = 8, 0.125, 0.02
    g = orc.grid(n, n, n, h)
    X, Y, Z = _xyz(g)
    a, b, c = 0.7, -0.3, 1.1
    vbc = orc.velocity_bc((1, 0, 1, 0, 1, 0))
    rhs = orc.pressure_rhs(g, a * X, b * Y, c * Z, dt, vbc)
    inner = (slice(0, -1),) * 3                                   # the open faces x+, y+, z+ copy: half a derivative there
    assert np.abs(rhs[inner] + (a + b + c) / dt).max() < 1e-11
    rhs_copy = orc.pressure_rhs(g, a * X, b * Y, c * Z, dt)
    assert abs(rhs_copy[3, 3, 0] + (0.5 * a + b + c) / dt) < 1e-11


def _mom_1d_wall(c, adv_vel, speed_sum, C, cn, h, dt, rho_l, rho_g, mu_l, mu_g, odd):
    """tests/test_oracle_flow.py::_mom_1d with a wall at both ends of the line: the advected component is odd about the
    walls when it is the wall-normal one (`odd`), every derived field keeps its copy halo (reading C9-iv)."""
    cp = np.concatenate(([-c[0] if odd else c[0]], c, [-c[-1] if odd else c[-1]]))
    cx = (cp[2:] - cp[:-2]) / (2 * h)
    adv = adv_vel * cx
    ap = np.pad(adv, 1, mode="edge")
    a = 2.0 * (ap[:-2] - 2 * adv + ap[2:]) / 6.0
    kabs = (1.0 / 16.0) * h * np.abs(a) / (1e-7 + np.abs(cx) / 3.0)
    rho = rho_l * C + rho_g * (1 - C); mu = mu_l * C + mu_g * (1 - C)
    kc = rho * np.minimum(h * speed_sum, kabs) + mu
    kp = np.pad(kc, 1, mode="edge")
    diff = (0.5 * (kc + kp[:-2]) * (c - cp[:-2]) + 0.5 * (kc + kp[2:]) * (c - cp[2:])) / (h * h)
    return cn - dt * (rho * adv + diff) / rho


@pytest.mark.parametrize("axis", [2, 1, 0])
def test_momentum_predictor_with_walls_one_dimensional(orc, axis):
    """Profiles along one axis between two walls: the wall-normal component takes the odd halo in its gradient and in its
    diffusion, the tangential ones the copy; against the hand-reduced scheme, wall cells included."""
    n, h, dt = 24, 0.05, 0.004
    rho_l, rho_g, mu_l, mu_g = 1000.0, 1.0, 0.5, 0.02
    i = np.arange(n)
    C = 0.5 * (1 + np.tanh((i - 11.2) / 2.5))
    prof = [0.25 * np.cos(0.9 * i + 0.3) + 0.15, 0.2 * np.cos(0.55 * i) - 0.13, 0.15 * np.sin(0.35 * i + 1.0) + 0.2]
    normal = 2 - axis                                             # the velocity component along `axis`
    shape = [4, 4, 4]; shape[axis] = n
    bshape = [1, 1, 1]; bshape[axis] = n
    g = orc.grid(shape[2], shape[1], shape[0], h)
    b3 = lambda a: np.broadcast_to(a.reshape(bshape), shape).copy()
    walls = [0] * 6; walls[2 * normal] = walls[2 * normal + 1] = 1
    vbc = orc.velocity_bc(walls)
    q = tuple(b3(p) for p in prof)
    qt, _ = orc.mom_predictor(g, b3(C), q, q, rho_l, rho_g, mu_l, mu_g, dt, vbc)
    qt_copy, _ = orc.mom_predictor(g, b3(C), q, q, rho_l, rho_g, mu_l, mu_g, dt)
    speed = sum(np.abs(p) for p in prof)
    for comp in range(3):
        ref = _mom_1d_wall(prof[comp], prof[normal], speed, C, prof[comp], h, dt, rho_l, rho_g, mu_l, mu_g, comp == normal)
        scale = np.abs(ref - prof[comp]).max()
        assert np.abs(qt[comp] - ref.reshape(bshape)).max() < 1e-11 * scale
    # the halo matters: the wall-normal component differs from the copy-halo result next to the walls (the stencil chain reaches three cells), and only there
    d = np.abs(qt[normal] - qt_copy[normal]).reshape(-1, n) if axis == 2 else np.moveaxis(np.abs(qt[normal] - qt_copy[normal]), axis, -1).reshape(-1, n)
    assert d[:, 0].max() > 1e-5 and d[:, -1].max() > 1e-5 and d[:, 3:-3].max() == 0.0


def test_forcing_balances_a_hydrostatic_column_exactly(orc):
    """One fluid at rest: p_hs = rho g (H - z) is linear, the bottom ghost (mirror + h g rho) and the top ghost (-mirror)
    continue it exactly, and M(-g rho) = -g rho: the forcing terms cancel in every cell, bottom and top rows included.
    Dropping the bottom extrapolation, or a wrong sign of either term, leaves -+ dt g there."""
    nx, ny, nz, h = 6, 5, 12, 0.05
    g = orc.grid(nx, ny, nz, h)
    rho, grav, dt = 1000.0, 9.81, 1e-3
    _, _, Z = _xyz(g)
    p_hs = rho * grav * (nz * h - Z)
    z0 = tuple(np.zeros(g.shape) for _ in range(3))
    qt = orc.mom_forcing(g, np.ones(g.shape), p_hs, None, BCP, grav, None, rho, 1.0, dt, z0)
    assert max(np.abs(a).max() for a in qt) < 1e-12 * grav * dt
    # gravity alone: free fall, w~ = -g dt everywhere
    qt = orc.mom_forcing(g, np.ones(g.shape), None, None, BCP, grav, None, rho, 1.0, dt, z0)
    assert np.abs(qt[2] + grav * dt).max() < 1e-13 and np.abs(qt[0]).max() == 0.0
    # pressure alone: w~ = +g dt (the gradient of p_hs is -rho g)
    qt = orc.mom_forcing(g, np.ones(g.shape), p_hs, None, BCP, 0.0, None, rho, 1.0, dt, z0)
    assert np.abs(qt[2][1:] - grav * dt).max() < 1e-12          # without g the bottom ghost is a plain copy: row 0 sees half


def test_forcing_terms_closed_forms(orc):
    """p_nh linear with its solver's halos; a uniform surface-tension force passes the mass filter unchanged; rho(C)
    divides."""
    n, h, dt = 8, 0.1, 0.01
    g = orc.grid(n, n, n, h)
    X, Y, Z = _xyz(g)
    Cf = np.full(g.shape, 0.25)
    rho = 1000.0 * 0.25 + 0.75
    z0 = tuple(np.zeros(g.shape) for _ in range(3))
    p = 2.0 * X - 1.5 * Y + 0.5 * Z
    qt = orc.mom_forcing(g, Cf, None, p, (N,) * 6, 0.0, None, 1000.0, 1.0, dt, z0)
    sl = (slice(1, -1),) * 3
    for a, gr in zip(qt, (2.0, -1.5, 0.5)):
        assert np.abs(a[sl] + dt * gr / rho).max() < 1e-13
    st = tuple(np.full(g.shape, s) for s in (3.0, -2.0, 0.5))
    qt = orc.mom_forcing(g, Cf, None, None, BCP, 0.0, st, 1000.0, 1.0, dt, z0)
    for a, s in zip(qt, (3.0, -2.0, 0.5)):
        assert np.abs(a - dt * s / rho).max() < 1e-14
    # the mass filter is applied to the source (Eq. 18: f(s; w_m)): a checkerboard source is damped by (1/3)^3
    cb = ((-1.0) ** (np.arange(n)[:, None, None] + np.arange(n)[None, :, None] + np.arange(n)[None, None, :]))
    qt = orc.mom_forcing(g, Cf, None, None, BCP, 0.0, (cb, 0 * cb, 0 * cb), 1000.0, 1.0, dt, z0)
    assert np.abs(qt[0][sl] - dt * cb[sl] / (27.0 * rho)).max() < 1e-15


def test_full_step_equals_the_stages_chained_by_hand(orc):
    """time_step_full against the four stages written out in the paper's order from the pinned stage functions."""
    n, levels = 16, 3
    w = configs.config5(n, levels)
    g = orc.grid(n, n, n, w.h)
    Cf = w.fields["alpha"]
    u, v, ww = (0.05 * w.fields[c] for c in ("u", "v", "w"))
    grav, sig, dt = 9.81, 0.0728, 0.02 * w.h
    p_old = 0.3 * np.cos(np.pi * configs.centres(n, n, n, w.h)[0]) + np.zeros(g.shape)
    got = orc.time_step_full(g, Cf, u, v, ww, p_old, levels, w.rho_l, w.rho_g, w.mu_l, w.mu_g, grav, sig, dt, 1e-10, 300, hs_cycles=20)
    vbc = orc.velocity_bc()
    b_hs, _, st = orc.hydrostatic_rhs(g, Cf, w.rho_l, w.rho_g, grav, sig)                       # stage 1
    p_hs, _, _, _ = orc.solve(g, BCP, None, np.zeros(g.shape), b_hs, levels, 0.0, 20)
    qn = (u, v, ww); qh = qn
    for _ in range(2):                                                                          # stage 2
        qt, _ = orc.mom_predictor(g, Cf, qh, qn, w.rho_l, w.rho_g, w.mu_l, w.mu_g, dt, vbc)
        qt = orc.mom_forcing(g, Cf, p_hs, p_old, BCP, grav, st, w.rho_l, w.rho_g, dt, qt)
        qh = tuple(0.5 * (a + b) for a, b in zip(qn, qt))
    k = orc.k_from_vof(Cf, w.rho_l, w.rho_g)                                                    # stage 3
    b = orc.pressure_rhs(g, qt[0], qt[1], qt[2], dt, vbc)
    dp, _, _, _ = orc.solve(g, BCP, k, np.zeros(g.shape), b, levels, 1e-10, 300)
    q1 = orc.project_velocity(g, BCP, dp, k, dt, qt[0], qt[1], qt[2])
    _, Cn = orc.vof_residual(g, Cf, q1[0], q1[1], q1[2], dt)                                   # stage 4
    rel = lambda a, r: np.linalg.norm(a - r) / max(np.linalg.norm(r), 1e-300)
    assert rel(got[0], Cn) < 1e-13 and rel(got[4], p_hs) < 1e-13 and rel(got[5], p_old + dp) < 1e-13
    for a, r in zip(got[1:4], q1):
        assert rel(a, r) < 1e-13
    # the forcing is not a spectator: without it the predicted velocity is far away
    qt0, _ = orc.mom_predictor(g, Cf, qn, qn, w.rho_l, w.rho_g, w.mu_l, w.mu_g, dt, vbc)
    assert rel(np.stack(qt0), np.stack(qt)) > 0.1


def test_two_layer_column_at_rest_stays_at_rest(orc):
    """Water under air, flat interface, no motion: stage 1 balances gravity, so after a full step the velocity is a small
    fraction of the free-fall gain g dt that the same step produces when p_hs is left out -- and C does not move."""
    n, levels = 16, 3
    h = 1.0 / n
    g = orc.grid(n, n, n, h)
    _, _, Z = _xyz(g)
    Cf = np.ascontiguousarray(0.5 * (1 + np.tanh((0.5 - Z) / (1.5 * h))))
    z = np.zeros(g.shape)
    grav, dt = 9.81, 1e-3
    out = orc.time_step_full(g, Cf, z, z, z, None, levels, 1000.0, 1.0, 1e-3, 1e-5, grav, 0.0, dt, 1e-10, 300, hs_tol=1e-11, hs_cycles=300)
    speed = max(np.abs(a).max() for a in out[1:4])
    assert speed < 0.05 * grav * dt, speed / (grav * dt)
    grad_c = np.abs(np.diff(Cf, axis=0)).max() / h
    assert np.abs(out[0] - Cf).max() < 0.1 * grav * dt * dt * grad_c      # a fraction of the free-fall displacement
    # dp_hs/dz = -rho g in both layers (stage 1 did its job inside the step)
    dpdz = (out[4][2:] - out[4][:-2]) / (2 * h)
    assert np.allclose(dpdz[0:2, 4, 4], -1000.0 * grav, rtol=1e-2)


def test_static_drop_spurious_currents_are_bounded(orc):
    """A drop at rest without gravity: the surface-tension force sigma kappa grad C is balanced by p_hs (Young-Laplace),
    so the step leaves only spurious currents -- a small fraction of the velocity the unbalanced force would create."""
    n, levels = 24, 3
    h = 1.0 / n
    g = orc.grid(n, n, n, h)
    X, Y, Z = _xyz(g)
    r = np.sqrt((X - 0.5) ** 2 + (Y - 0.5) ** 2 + (Z - 0.5) ** 2)
    Cf = np.ascontiguousarray(0.5 * (1 - np.tanh((r - 0.25) / (2 * h))))
    z = np.zeros(g.shape)
    rho_l, rho_g, sig, dt = 10.0, 1.0, 1.0, 1e-3
    out = orc.time_step_full(g, Cf, z, z, z, None, levels, rho_l, rho_g, 1e-3, 1e-4, 0.0, sig, dt, 1e-10, 300, hs_tol=1e-11, hs_cycles=400)
    _, _, st = orc.hydrostatic_rhs(g, Cf, rho_l, rho_g, 0.0, sig)
    unbalanced = orc.mom_forcing(g, Cf, None, None, BCP, 0.0, st, rho_l, rho_g, dt, (z, z, z))
    ref = max(np.abs(a).max() for a in unbalanced)
    speed = max(np.abs(a).max() for a in out[1:4])
    assert ref > 0 and speed < 0.25 * ref, speed / ref
