"""Pins of the oracle's explicit residuals: vof_residual, momentum predictor, pressure RHS and
projection (readings C9, C10).  The paper gives no worked example for these, so the pins
are special cases that reduce to hand-derivable forms, invariants and the printed constants.
Beyond them parity against the paper is UNPINNED (stated in oracle.c and DESIGN.md).
"""
import os

import numpy as np
import pytest

from workloads import configs

N, D = 0, 1
HERE = os.path.dirname(os.path.abspath(__file__))


def _rand(shape, seed):
    return np.random.default_rng(seed).standard_normal(shape)


def _constants():
    out = {}
    for line in open(os.path.join(HERE, "golden", "vof_constants.txt")):
        line = line.split("#")[0].split()
        if len(line) == 2:
            out[line[0]] = float(line[1])
    return out


def _vof_1d(C, u, v, w, h, dt, cst, detector=3):
    """The scheme of Eqs. 16, 27, 29, 33, 35-42 reduced BY HAND to fields that vary along x only:
    every 3x3x3 filter collapses to its 1-D factor because the mass factors sum to one, the y/z
    diffusion terms vanish, and S^y = S^z = 0 (or -1 under the override).  Constants are read from
    the paper's printed values (tests/golden/vof_constants.txt)."""
    Cp = np.pad(C, 1, mode="edge")
    Cx = (Cp[2:] - Cp[:-2]) / (2 * h)
    adv = u * Cx
    ap = np.pad(adv, 1, mode="edge")
    a = cst["alpha_a"] * (ap[:-2] - 2 * adv + ap[2:]) / 6.0
    kabs = cst["alpha_kabs"] * h * np.abs(a) / (cst["eps_k"] + np.abs(Cx) / 3.0)
    S = (C - Cp[:-2]) * (Cp[2:] - C)
    if detector == 5:                         # Eq. 34: min of the three products over i-2 .. i+2; halo = reflection
        C2 = np.pad(C, 2, mode="symmetric")
        d = np.diff(C2)                       # d[m] = C2[m+1] - C2[m]; cell i sits at C2[i+2]
        n = len(C)
        S = np.minimum(np.minimum(d[0:n] * d[1:n + 1], d[1:n + 1] * d[2:n + 2]), d[2:n + 2] * d[3:n + 3])
    S = np.where((C > cst["C_hi"]) | (C < cst["C_lo"]), -1.0, S)
    wp = -np.maximum(-1.0, np.minimum(0.0, cst["K_plus"] * S))
    wm = np.minimum(1.0, np.maximum(0.0, cst["K_minus"] * S))
    g2 = Cx ** 2
    us = Cx * (u * Cx) / (cst["eps_x"] + g2)
    kneg = -cst["beta"] * (u * u + v * v + w * w) / (cst["eps_x"] + g2 * np.abs(us) / 3.0)
    kmin, kmax = cst["alpha_min"] * h * h / dt, cst["alpha_max"] * h * h / dt
    kraw = wp * cst["K_cal"] * kabs + wm * kneg / h
    kx = np.maximum(-kmin, np.minimum(kmax, kraw))
    kp = np.pad(kx, 1, mode="edge")
    diff = (0.5 * (kx + kp[:-2]) * (C - Cp[:-2]) + 0.5 * (kx + kp[2:]) * (C - Cp[2:])) / (h * h)
    return adv + diff, kraw, kmin, kmax


@pytest.mark.parametrize("axis", [2, 1, 0])
def test_vof_one_dimensional_profile(orc, axis):
    """A smeared step advected along one axis, against the hand-reduced 1-D scheme; the case is
    built so that both clip bounds of Eq. 41 and both branches of Eq. 35 are exercised."""
    cst = _constants()
    n, h, dt = 24, 0.05, 0.004
    i = np.arange(n)
    C = 0.5 * (1 + np.tanh((i - 11.3) / 1.7)) + 0.04 * np.sin(1.9 * i)       # step + wiggles (extrema)
    u = 1.0 + 0.3 * np.cos(0.4 * i)
    v, w = 0.35, -0.2
    ref, kraw, kmin, kmax = _vof_1d(C, u, v, w, h, dt, cst)
    assert (kraw > kmax).any() and (kraw < -kmin).any() and ((kraw < kmax) & (kraw > 0)).any()
    shape = [5, 5, 5]; shape[axis] = n
    bshape = [1, 1, 1]; bshape[axis] = n
    g = orc.grid(shape[2], shape[1], shape[0], h)
    C3 = np.broadcast_to(C.reshape(bshape), shape).copy()
    vel = [np.full(shape, v), np.full(shape, w)]
    comps = [None, None, None]                                               # (u, v, w) = x, y, z components
    comps[2 - axis] = np.broadcast_to(u.reshape(bshape), shape).copy()
    rest = [c for c in range(3) if c != 2 - axis]
    comps[rest[0]], comps[rest[1]] = vel
    sC, Cn = orc.vof_residual(g, C3, comps[0], comps[1], comps[2], dt)
    assert np.abs(sC - ref.reshape(bshape)).max() < 1e-11 * np.abs(ref).max()
    assert np.abs(Cn - (C3 - dt * sC)).max() < 1e-15                         # Eq. 55


@pytest.mark.parametrize("axis", [2, 1, 0])
def test_vof_five_point_detectors_eq34(orc, axis):
    """Eq. 34: the same smeared step with wiggles against the hand-reduced 1-D scheme with the 5-point detector; the
    profile has extrema one cell away from cells where Eq. 33 sees none, so the two detectors differ there (asserted) --
    and nowhere in the monotone part of the step."""
    cst = _constants()
    n, h, dt = 24, 0.05, 0.004
    i = np.arange(n)
    C = 0.5 * (1 + np.tanh((i - 11.3) / 1.7)) + 0.04 * np.sin(1.9 * i)
    u = 1.0 + 0.3 * np.cos(0.4 * i)
    v, w = 0.35, -0.2
    ref5, _, _, _ = _vof_1d(C, u, v, w, h, dt, cst, detector=5)
    ref3, _, _, _ = _vof_1d(C, u, v, w, h, dt, cst, detector=3)
    assert np.abs(ref5 - ref3).max() > 1e-3 * np.abs(ref3).max()
    shape = [5, 5, 5]; shape[axis] = n
    bshape = [1, 1, 1]; bshape[axis] = n
    g = orc.grid(shape[2], shape[1], shape[0], h)
    C3 = np.broadcast_to(C.reshape(bshape), shape).copy()
    comps = [None, None, None]
    comps[2 - axis] = np.broadcast_to(u.reshape(bshape), shape).copy()
    rest = [c for c in range(3) if c != 2 - axis]
    comps[rest[0]], comps[rest[1]] = np.full(shape, v), np.full(shape, w)
    s5, _ = orc.vof_residual(g, C3, comps[0], comps[1], comps[2], dt, detector=5)
    s3, _ = orc.vof_residual(g, C3, comps[0], comps[1], comps[2], dt, detector=3)
    assert np.abs(s5 - ref5.reshape(bshape)).max() < 1e-11 * np.abs(ref5).max()
    assert np.abs(s3 - ref3.reshape(bshape)).max() < 1e-11 * np.abs(ref3).max()


def test_vof_five_point_detector_special_cases(orc):
    """A monotone profile has no sign change anywhere: min{...} >= 0, no positive (anti-)diffusion weight w+ beyond what
    Eq. 33 gives, and where the three products are equal (a linear ramp) both detectors agree exactly.  A single-cell
    spike is seen by the 5-point detector in the two cells on either side of it, by the 3-point one only in the spike."""
    n, h, dt = 16, 0.1, 0.01
    g = orc.grid(n, 4, 4, h)
    i = np.arange(n)
    ramp = np.broadcast_to((0.2 + 0.04 * i).reshape(1, 1, n), g.shape).copy()       # inside (0.05, 0.95): no override
    q = [np.full(g.shape, c) for c in (0.7, 0.0, 0.0)]
    s5, _ = orc.vof_residual(g, ramp, *q, dt, detector=5)
    s3, _ = orc.vof_residual(g, ramp, *q, dt, detector=3)
    assert np.abs(s5 - s3)[:, :, 3:-3].max() < 1e-13        # away from the walls (the reflected halo is an extremum)
    spike = ramp.copy(); spike[:, :, 8] += 0.1                                      # one-cell extremum at i = 8
    s5, _ = orc.vof_residual(g, spike, *q, dt, detector=5)
    s3, _ = orc.vof_residual(g, spike, *q, dt, detector=3)
    differs = np.abs(s5 - s3)[2, 2] > 1e-9
    # the detectors disagree at i = 6 and i = 10 (their own 3-point product is positive, a neighbouring one is negative); the
    # directional coefficients there feed the diffusion stencil of the cells next to them
    assert differs[6:9].all() and differs[9:12].any() and not differs[3:6].any() and not differs[12:13].any()   # walls apart


def test_vof_trivial_cases(orc):
    g = orc.grid(6, 7, 5, 0.1)
    u, v, w = (_rand(g.shape, s) for s in (1, 2, 3))
    z = np.zeros(g.shape)
    sC, _ = orc.vof_residual(g, np.full(g.shape, 0.4), u, v, w, 0.01)
    assert np.abs(sC).max() < 1e-13                                          # uniform C (filter rounding only)
    C = 0.5 + 0.3 * np.tanh(_rand(g.shape, 4))
    sC, Cn = orc.vof_residual(g, C, z, z, z, 0.01)
    assert np.abs(sC).max() == 0.0 and np.array_equal(Cn, C)                 # q = 0


def test_vof_linear_field_interior_is_pure_advection(orc):
    """Linear C, constant q: grad C exact, a = 0, k_abs = 0 and k^x uniform, so away from the
    walls s_C = q . grad C exactly (C9 pins)."""
    n, h = 12, 0.05
    g = orc.grid(n, n, n, h)
    c = (np.arange(n) + 0.5) * h
    C = 0.3 + 0.5 * c[None, None, :] + 0.2 * c[None, :, None] - 0.1 * c[:, None, None]
    q = (0.7, -0.4, 0.9)
    sC, _ = orc.vof_residual(g, C, *(np.full(g.shape, qq) for qq in q), 0.002)
    exact = q[0] * 0.5 + q[1] * 0.2 + q[2] * (-0.1)
    assert np.abs(sC[3:-3, 3:-3, 3:-3] - exact).max() < 1e-11


def test_vof_diffusion_is_conservative_and_axes_permute(orc):
    """sum(s_C - q.grad C) = 0 under copy halos (collapsed Eq. 12 is a flux form), and relabelling
    the axes of the inputs relabels the output."""
    g = orc.grid(9, 9, 9, 0.1)
    C = 0.5 + 0.45 * np.tanh(2 * _rand(g.shape, 5))
    u, v, w = (_rand(g.shape, s) for s in (6, 7, 8))
    dt = 0.003
    sC, _ = orc.vof_residual(g, C, u, v, w, dt)
    adv = sum(q * orc.apply_filter(g, (N,) * 6, orc.filter_weights(g, a), C) for q, a in ((u, "x"), (v, "y"), (w, "z")))
    assert abs((sC - adv).sum()) < 1e-9 * np.abs(sC - adv).sum()
    assert np.abs(sC - adv).max() > 1e-3                                     # the diffusion is active
    # swap x <-> z: arrays transpose (2,1,0), u <-> w
    t = lambda a: np.ascontiguousarray(a.transpose(2, 1, 0))
    sT, _ = orc.vof_residual(g, t(C), t(w), t(v), t(u), dt)
    assert np.abs(t(sT) - sC).max() < 1e-10 * np.abs(sC).max()
    # swap x <-> y
    t2 = lambda a: np.ascontiguousarray(a.transpose(0, 2, 1))
    sT, _ = orc.vof_residual(g, t2(C), t2(v), t2(u), t2(w), dt)
    assert np.abs(t2(sT) - sC).max() < 1e-10 * np.abs(sC).max()


def test_vof_nonuniform_spacing_uses_eq26(orc):
    """dx != dy != dz: Eq. 26 and Eqs. 38/42 with per-direction spacing; 1-D profile along y."""
    cst = _constants()
    n, dt = 20, 0.002
    hx, hy, hz = 0.05, 0.08, 0.11
    j = np.arange(n)
    C = 0.5 * (1 + np.tanh((j - 9.4) / 1.5))
    vv = 0.8 + 0.1 * np.sin(0.7 * j)
    g = orc.grid(4, n, 4, hx, hy, hz)
    shape = g.shape
    C3 = np.broadcast_to(C[None, :, None], shape).copy()
    v3 = np.broadcast_to(vv[None, :, None], shape).copy()
    sC, _ = orc.vof_residual(g, C3, np.full(shape, 0.1), v3, np.full(shape, -0.3), dt)
    # hand reduction along y
    Cp = np.pad(C, 1, mode="edge"); Cy = (Cp[2:] - Cp[:-2]) / (2 * hy)
    adv = vv * Cy; ap = np.pad(adv, 1, mode="edge")
    a = 2 * (ap[:-2] - 2 * adv + ap[2:]) / 6
    kabs = cst["alpha_kabs"] * np.abs(a) * hy * np.abs(Cy) / (cst["eps_k"] + Cy ** 2 / 3)          # Eq. 26
    S = (C - Cp[:-2]) * (Cp[2:] - C); S = np.where((C > 0.95) | (C < 0.05), -1.0, S)
    wp = -np.maximum(-1, np.minimum(0, 300 * S)); wm = np.minimum(1, np.maximum(0, 300 * S))
    us = Cy * vv * Cy / (1e-4 + Cy ** 2)
    kneg = -0.1 * (0.01 + vv ** 2 + 0.09) / (1e-4 + Cy ** 2 * np.abs(us) / 3)
    kmin, kmax = 1e-4 * hz ** 2 / dt, 0.05 * hx ** 2 / dt
    ky = np.maximum(-kmin, np.minimum(kmax, wp * 3 * kabs + wm * kneg / hy))
    kp = np.pad(ky, 1, mode="edge")
    diff = (0.5 * (ky + kp[:-2]) * (C - Cp[:-2]) + 0.5 * (ky + kp[2:]) * (C - Cp[2:])) / hy ** 2
    assert np.abs(sC - (adv + diff)[None, :, None]).max() < 1e-11 * np.abs(adv + diff).max()


# ---------------------------------------------------------------- momentum (Eqs. 18, 30-32, 45-46)
def test_momentum_uniform_velocity_is_steady(orc):
    g = orc.grid(6, 6, 6, 0.1)
    C = 0.5 + 0.4 * np.tanh(_rand(g.shape, 1))
    q = tuple(np.full(g.shape, c) for c in (0.3, -0.7, 1.1))
    qt, qh = orc.mom_predictor(g, C, q, q, 1000.0, 1.0, 1e-3, 1e-5, 0.01)
    for a, b, c in zip(qt, qh, q):
        assert np.abs(a - c).max() < 1e-13 and np.abs(b - c).max() < 1e-13


def test_momentum_linear_velocity_interior(orc):
    """Linear velocity field: gradients exact, mixed-mass residual 0 so k = mu (linear in x through C),
    diffusion of a linear field with linear k ... choose constant C so k is constant: s = rho q.grad c."""
    n, h, dt = 12, 0.1, 0.01
    g = orc.grid(n, n, n, h)
    c = (np.arange(n) + 0.5) * h
    X, Y, Z = c[None, None, :] + 0 * c[:, None, None] + 0 * c[None, :, None], None, None
    X = np.broadcast_to(c[None, None, :], g.shape); Y = np.broadcast_to(c[None, :, None], g.shape)
    Z = np.broadcast_to(c[:, None, None], g.shape)
    u = 0.2 + 0.5 * X - 0.3 * Y + 0.1 * Z
    v = -0.1 + 0.2 * X + 0.4 * Y - 0.6 * Z
    w = 0.3 - 0.7 * X + 0.1 * Y + 0.2 * Z
    C = np.full(g.shape, 0.25)
    rho = 1000 * 0.25 + 0.75
    un = _rand(g.shape, 3)
    qt, qh = orc.mom_predictor(g, C, (u, v, w), (un, v, w), 1000.0, 1.0, 1e-3, 1e-5, dt)
    s_u = u * 0.5 + v * (-0.3) + w * 0.1                                     # q . grad u  (per unit rho)
    sl = (slice(3, -3),) * 3
    assert np.abs(qt[0][sl] - (un - dt * s_u)[sl]).max() < 1e-12
    assert np.abs(qh[0][sl] - 0.5 * (un + qt[0])[sl]).max() < 1e-15          # Eq. 46
    s_w = u * (-0.7) + v * 0.1 + w * 0.2
    assert np.abs(qt[2][sl] - (w - dt * s_w)[sl]).max() < 1e-12
    assert rho > 0


def test_momentum_viscous_limit_is_eigenmode_decay(orc):
    """Tiny velocity amplitude: advection and PG diffusion are O(eps^2)/O(eps), so
    c~ = c - dt (mu/rho) A c with A the 27-point operator under copy halos; for a cosine mode
    A c = lambda c in closed form (C1-ii)."""
    n, h, dt, eps = 8, 0.125, 0.01, 1e-9
    g = orc.grid(n, n, n, h)
    i = np.arange(n)
    cx, cy, cz = (np.cos(np.pi * m * (i + 0.5) / n) for m in (1, 2, 1))
    mode = cz[:, None, None] * cy[None, :, None] * cx[None, None, :]
    s = [np.sin(np.pi * m / (2 * n)) ** 2 for m in (1, 2, 1)]
    lam = sum(4 / h ** 2 * s[d] * np.prod([1 - 2 / 3 * s[e] for e in range(3) if e != d]) for d in range(3))
    C = np.full(g.shape, 0.5)
    rho, mu = 500.5, 0.5 * 1e-1 + 0.5 * 1e-3
    u = eps * mode
    z = np.zeros(g.shape)
    qt, _ = orc.mom_predictor(g, C, (u, z, z), (u, z, z), 1000.0, 1.0, 1e-1, 1e-3, dt)
    assert np.abs(qt[0] - (1 - dt * mu / rho * lam) * u).max() < 1e-5 * eps * dt * mu / rho * lam


def _mom_1d(c, adv_vel, speed_sum, C, cn, h, dt, rho_l, rho_g, mu_l, mu_g):
    """Eqs. 18 (advection + diffusion part), 27, 29, 30-32, 45-46 reduced BY HAND to fields that vary along ONE axis
    (P:198-220, 284-305, 309-319, 433-441): every 3x3x3 filter collapses to its 1-D factor (the mass factors sum to one);
    `adv_vel` is the velocity component along that axis, `speed_sum` = |u| + |v| + |w| (uniform spacing, Eq. 30).
    Returns (c~, c_half', k_max, k_abs, k_c)."""
    cp = np.pad(c, 1, mode="edge")
    cx = (cp[2:] - cp[:-2]) / (2 * h)
    adv = adv_vel * cx
    ap = np.pad(adv, 1, mode="edge")
    a = 2.0 * (ap[:-2] - 2 * adv + ap[2:]) / 6.0                       # Eq. 29, alpha_a = 2
    kabs = (1.0 / 16.0) * h * np.abs(a) / (1e-7 + np.abs(cx) / 3.0)    # Eq. 27, alpha_kabs = 1/16, eps_k
    kmax = h * speed_sum                                               # Eq. 30
    rho = rho_l * C + rho_g * (1 - C)                                  # Eq. 2
    mu = mu_l * C + mu_g * (1 - C)
    kc = rho * np.minimum(kmax, kabs) + mu                             # Eqs. 31-32, k_square (lost Eq. 28) omitted
    kp = np.pad(kc, 1, mode="edge")
    diff = (0.5 * (kc + kp[:-2]) * (c - cp[:-2]) + 0.5 * (kc + kp[2:]) * (c - cp[2:])) / (h * h)   # Eq. 13 collapsed, 1-D
    s = rho * adv + diff
    ct = cn - dt * s / rho                                             # Eq. 45, sigma = 0
    return ct, 0.5 * (cn + ct), kmax, kabs, kc


@pytest.mark.parametrize("axis", [2, 1, 0])
def test_momentum_one_dimensional_profile_pins_the_petrov_galerkin_coefficient(orc, axis):
    """Velocity components and C varying along one axis, against the hand-reduced 1-D scheme.  The profiles are built so
    that min{k_max, k_abs} takes BOTH branches at many cells with rho and mu varying by orders of magnitude across them:
    dropping rho, dropping the min, a wrong k_max or dropping mu each change c~ far beyond the tolerance (asserted
    below on the hand side, so the case stays discriminating if the profiles are edited)."""
    n, h, dt = 32, 0.05, 0.004
    rho_l, rho_g, mu_l, mu_g = 1000.0, 1.0, 0.5, 0.02
    i = np.arange(n)
    along_of = {2: 0, 1: 1, 0: 2}                                            # component index of the velocity along `axis`
    C = 0.5 * (1 + np.tanh((i - 15.2) / 2.5))                                # rho from 1 to 1000 across the profile
    # cos(2 pi (i - i0) / P) with integer i0 and even P is symmetric about the cells i0 + m P / 2: the central gradient
    # vanishes there while the mixed-mass residual a of Eq. 29 does not (the advecting velocity is not symmetric about
    # them), so k_abs >> k_max at those cells (Eq. 27's eps_k in the denominator) and k_abs << k_max elsewhere
    prof = [0.25 * np.cos(2 * np.pi * i / 8) + 0.05, 0.2 * np.cos(2 * np.pi * (i - 1) / 6) - 0.03,
            0.15 * np.cos(2 * np.pi * (i - 2) / 10) + 0.1]
    prof[along_of[axis]] = 0.22 * np.sin(0.47 * i + 0.3) + 0.06              # the advecting component: no symmetric cells
    prof_n = [p + 0.01 * np.cos(1.3 * i + m) for m, p in enumerate(prof)]    # q_n differs from q_half
    along = along_of[axis]
    speed = sum(np.abs(p) for p in prof)
    shape = [4, 4, 4]; shape[axis] = n
    bshape = [1, 1, 1]; bshape[axis] = n
    g = orc.grid(shape[2], shape[1], shape[0], h)
    b3 = lambda a: np.broadcast_to(a.reshape(bshape), shape).copy()
    qh = tuple(b3(p) for p in prof); qn = tuple(b3(p) for p in prof_n)
    qt, qhn = orc.mom_predictor(g, b3(C), qh, qn, rho_l, rho_g, mu_l, mu_g, dt)
    for comp in range(3):
        ct, chalf, kmax, kabs, kc = _mom_1d(prof[comp], prof[along], speed, C, prof_n[comp], h, dt, rho_l, rho_g, mu_l, mu_g)
        lo, hi = (kabs < kmax) & (kabs > 1e-3 * kmax), kabs > kmax
        # both branches of the min{} are taken (the self-advected component has no cell with k_abs > k_max)
        assert lo.sum() >= 4 and (hi.sum() >= 3 or comp == along), (comp, lo.sum(), hi.sum())
        scale = np.abs(ct - prof_n[comp]).max()
        assert np.abs(qt[comp] - ct.reshape(bshape)).max() < 1e-11 * scale
        assert np.abs(qhn[comp] - chalf.reshape(bshape)).max() < 1e-11 * np.abs(chalf).max()
        # the case discriminates: each plausible slip in Eqs. 30-32 moves c~ by much more than the tolerance
        rho = rho_l * C + rho_g * (1 - C); mu = mu_l * C + mu_g * (1 - C)
        for bad in (np.minimum(kmax, kabs) + mu, rho * kabs + mu, rho * np.minimum(2 * kmax, kabs) + mu,
                    rho * np.minimum(kmax, kabs), rho * np.minimum(kmax, kabs) + mu_l):
            kp = np.pad(bad, 1, mode="edge"); cp = np.pad(prof[comp], 1, mode="edge")
            diff = (0.5 * (bad + kp[:-2]) * (prof[comp] - cp[:-2]) + 0.5 * (bad + kp[2:]) * (prof[comp] - cp[2:])) / (h * h)
            adv = prof[along] * (cp[2:] - cp[:-2]) / (2 * h)
            wrong = prof_n[comp] - dt * (rho * adv + diff) / rho
            assert comp == along or np.abs(wrong - ct).max() > 1e-4 * scale


# ---------------------------------------------------------------- pressure RHS and projection (C10)
def test_pressure_rhs_linear_velocity(orc):
    n, h, dt = 10, 0.1, 0.02
    g = orc.grid(n, n, n, h)
    c = (np.arange(n) + 0.5) * h
    X = np.broadcast_to(c[None, None, :], g.shape); Y = np.broadcast_to(c[None, :, None], g.shape)
    Z = np.broadcast_to(c[:, None, None], g.shape)
    b = orc.pressure_rhs(g, 0.3 * X + Y, 0.5 * Y - Z, -0.2 * Z + X, dt)
    sl = (slice(1, -1),) * 3
    assert np.abs(b[sl] + (0.3 + 0.5 - 0.2) / dt).max() < 1e-11


def test_projection_pins(orc):
    n, h, dt = 10, 0.1, 0.02
    g = orc.grid(n, n, n, h)
    k = np.exp(_rand(g.shape, 1))
    u, v, w = (_rand(g.shape, s) for s in (2, 3, 4))
    # constant p under all-Neumann halos: no change
    uu, vv, ww = orc.project_velocity(g, (N,) * 6, np.full(g.shape, 3.0), k, dt, u, v, w)
    assert np.abs(uu - u).max() < 1e-13 and np.abs(ww - w).max() < 1e-13
    # linear p: exact gradient in the interior
    c = (np.arange(n) + 0.5) * h
    p = 2.0 * c[None, None, :] - 1.5 * c[None, :, None] + 0.5 * c[:, None, None] + np.zeros(g.shape)
    uu, vv, ww = orc.project_velocity(g, (N,) * 6, p, k, dt, u, v, w)
    sl = (slice(1, -1),) * 3
    assert np.abs(uu - (u - dt * k * 2.0))[sl].max() < 1e-12
    assert np.abs(vv - (v + dt * k * 1.5))[sl].max() < 1e-12
    assert np.abs(ww - (w - dt * k * 0.5))[sl].max() < 1e-12
    # Dirichlet top (ghost = -mirror): the z-gradient at the top cells sees p_ghost = -p
    uu, vv, ww = orc.project_velocity(g, (N,) * 5 + (D,), np.ones(g.shape), np.ones(g.shape), 1.0, u, v, w)
    assert np.abs(ww[-1] - (w[-1] + 1.0 / h)).max() < 1e-12 and np.abs(ww[:-1] - w[:-1]).max() < 1e-13


def test_projection_reduces_divergence(orc):
    """RHS -> solve -> project on a smooth field: the FE divergence norm drops (approximate projection, C10 note)."""
    n, h, dt = 16, 1.0 / 16, 0.01
    g = orc.grid(n, n, n, h)
    bc = (N,) * 5 + (D,)
    c = (np.arange(n) + 0.5) * h
    X = np.broadcast_to(c[None, None, :], g.shape); Y = np.broadcast_to(c[None, :, None], g.shape)
    Z = np.broadcast_to(c[:, None, None], g.shape)
    u = np.sin(np.pi * X) * np.cos(np.pi * Y); v = np.cos(2 * np.pi * Y) * Z; w = np.sin(np.pi * Z) * X
    alpha = (X < 0.4).astype(float)
    k = orc.k_from_vof(alpha, 10.0, 1.0)
    b = orc.pressure_rhs(g, u, v, w, dt)
    p, _, rel, _ = orc.solve(g, bc, k, np.zeros(g.shape), b, levels=3, tol=1e-10, max_cycles=100)
    assert rel < 1e-10
    uu, vv, ww = orc.project_velocity(g, bc, p, k, dt, u, v, w)
    b2 = orc.pressure_rhs(g, uu, vv, ww, dt)
    sl = (slice(2, -2),) * 3
    assert np.linalg.norm(b2[sl]) < 0.5 * np.linalg.norm(b[sl])


# ---------------------------------------------------------------- 8(f) next 2: the paper's own stage-3 right-hand side (Eq. 53)
def test_rhs_paper_constant_density_is_rho_times_divergence(orc):
    """rho constant: the rho-gradient terms vanish and Eq. 53's RHS is rho times the FE divergence RHS (already pinned)."""
    g = orc.grid(10, 12, 8, 0.1, 0.08, 0.125)
    r = np.random.default_rng(0)
    u, v, w = (r.standard_normal(g.shape) for _ in range(3))
    for Cval, rho in ((1.0, 1000.0), (0.0, 1.0), (0.25, 250.75)):
        b = orc.pressure_rhs_paper(g, np.full(g.shape, Cval), u, v, w, 1000.0, 1.0, 0.02)
        assert np.allclose(b, rho * orc.pressure_rhs(g, u, v, w, 0.02), rtol=1e-12, atol=1e-9)


def test_rhs_paper_linear_fields_closed_form(orc):
    """u = x, rho = 1 + x (C = x with rho_l = 2, rho_g = 1), v = w = 0: the central difference of the quadratic rho u is
    exact, so away from the x faces  b = -(1/dt) ((1 + 2x) - x) = -(1 + x)/dt = -rho div(q)/dt."""
    n, h, dt = 12, 0.05, 0.01
    g = orc.grid(n, 6, 6, h)
    x = ((np.arange(n) + 0.5) * h).reshape(1, 1, n) + np.zeros(g.shape)
    z = np.zeros(g.shape)
    b = orc.pressure_rhs_paper(g, x, x, z, z, 2.0, 1.0, dt)
    assert np.allclose(b[:, :, 1:-1], -(1.0 + x[:, :, 1:-1]) / dt, rtol=1e-12)
    # a sign or a dropped term would show: the two groups of Eq. 53 separately are -(1 + 2x)/dt and +x/dt
    b_u = orc.pressure_rhs_paper(g, x, x, z, z, 2.0, 1.0, dt) - orc.pressure_rhs_paper(g, z, x, z, z, 2.0, 1.0, dt)
    assert np.allclose(b_u[:, :, 1:-1], -(x[:, :, 1:-1]) / dt, rtol=1e-11)      # rho_g = 1 part removed: -(x * 1)' - ... = -x/dt


def test_time_step_paper_reduces_mass_residual(orc):
    """Two passes of the paper's stage 3 reduce the right-hand side of Eq. 52 (the mass-conservation defect)."""
    from workloads import configs
    w = configs.config5(16, 3)
    g = orc.grid(16, 16, 16, w.h)
    Cf, u, v, ww = (w.fields[q] for q in ("alpha", "u", "v", "w"))
    qn = (u, v, ww)
    qt, qh = orc.mom_predictor(g, Cf, qn, qn, w.rho_l, w.rho_g, w.mu_l, w.mu_g, w.dt)
    qt, _ = orc.mom_predictor(g, Cf, qh, qn, w.rho_l, w.rho_g, w.mu_l, w.mu_g, w.dt)
    b0 = orc.pressure_rhs_paper(g, Cf, qt[0], qt[1], qt[2], w.rho_l, w.rho_g, w.dt)
    Cn, un, vn, wn, p, rel = orc.time_step_paper(g, w.bc, Cf, u, v, ww, 3, w.rho_l, w.rho_g, w.mu_l, w.mu_g, w.dt)
    b2 = orc.pressure_rhs_paper(g, Cf, un, vn, wn, w.rho_l, w.rho_g, w.dt)
    assert np.linalg.norm(b2) < 0.7 * np.linalg.norm(b0)
    assert np.isfinite(p).all() and 0.0 <= Cn.min() + 1e-3 and Cn.max() <= 1.0 + 1e-3


def test_time_step_with_pcg_reaches_the_same_step_and_a_solenoidal_velocity(orc):
    """time_step(solver="pcg") differs from the plain-cycle step only in how A(k) p = b is solved: driven to 1e-11 both give
    the same fields; and the projected velocity then has no FE divergence left (b of the new velocity is ~0 relative to
    b of the predictor), which pins the composition rhs -> solve -> projection with either solver."""
    from workloads import configs
    n, levels = 16, 3
    w = configs.config5(n, levels)
    g = orc.grid(n, n, n, w.h)
    Cf, u, v, ww = (w.fields[q] for q in ("alpha", "u", "v", "w"))
    args = (g, w.bc, Cf, u, v, ww, levels, w.rho_l, w.rho_g, w.mu_l, w.mu_g, w.dt, 1e-11, 400)
    ref = orc.time_step(*args)
    got = orc.time_step(*args, solver="pcg")
    assert got[6] < 1e-11 and ref[6] < 1e-11
    assert got[5] < ref[5]                                   # CG needs fewer V-cycles than the plain iteration
    for a, b in zip(got[:5], ref[:5]):
        assert np.linalg.norm(a - b) <= 1e-8 * max(np.linalg.norm(b), 1e-30)
    qn = (u, v, ww)
    qt, qh = orc.mom_predictor(g, Cf, qn, qn, w.rho_l, w.rho_g, w.mu_l, w.mu_g, w.dt)
    qt, _ = orc.mom_predictor(g, Cf, qh, qn, w.rho_l, w.rho_g, w.mu_l, w.mu_g, w.dt)
    b0 = orc.pressure_rhs(g, qt[0], qt[1], qt[2], w.dt)
    b1 = orc.pressure_rhs(g, got[1], got[2], got[3], w.dt)
    # the projection uses the gradient filters, the operator the Laplacian filters (D M D != K M M exactly): the divergence
    # drops by the discretisation mismatch, not to rounding (0.66 on this 16^3 swirl; a wrong sign in the projection gives > 1)
    assert np.linalg.norm(b1) < 0.8 * np.linalg.norm(b0)


# ---------------------------------------------------------------- 8(f) next 3: hydrostatic + surface-tension pressure (stage 1)
BC_PHS = (0, 0, 0, 0, 0, 1)       # p_hs: zero derivative on the sides and (after folding -rho g into b) the bottom, zero value on top


def test_hydrostatic_column_is_reproduced_exactly(orc):
    """One fluid, no surface tension: p = rho g (H - z) is linear, the FE filters are exact for it, and it satisfies
    dp/dz = -rho g at the bottom and p = 0 on the top face.  So A p = b_hs must hold to rounding, and the multigrid solve of
    A p = b_hs must return it.  Pins the gravity term, its sign, and the bottom boundary fold."""
    nx, ny, nz, h = 8, 6, 16, 0.05
    g = orc.grid(nx, ny, nz, h)
    rho, grav = 1000.0, 9.81
    b, kap, st = orc.hydrostatic_rhs(g, np.ones(g.shape), rho, 1.0, grav, 0.0728)
    assert np.abs(kap).max() < 1e-12 and all(np.abs(a).max() < 1e-12 for a in st)      # no interface: no curvature (rounding only)
    z = ((np.arange(nz) + 0.5) * h).reshape(nz, 1, 1) + np.zeros(g.shape)
    p = rho * grav * (nz * h - z)
    assert np.allclose(orc.apply_operator(g, BC_PHS, None, p), b, rtol=0, atol=1e-8 * rho * grav / h)
    x, cyc, rel, _ = orc.solve(g, BC_PHS, None, np.zeros(g.shape), b, 2, 1e-12, 200)
    assert np.allclose(x, p, rtol=1e-9, atol=1e-9 * rho * grav)


def test_two_layer_hydrostatic_balance(orc):
    """Flat interface (water below air), sigma_t = 0: dp/dz = -rho(z) g in both layers away from the smoothed interface."""
    n, h = 32, 1.0 / 32
    g = orc.grid(8, 8, n, h)
    z = ((np.arange(n) + 0.5) * h).reshape(n, 1, 1) + np.zeros(g.shape)
    Cf = 0.5 * (1 + np.tanh((0.5 - z) / (1.5 * h)))
    b, kap, _ = orc.hydrostatic_rhs(g, Cf, 1000.0, 1.0, 9.81, 0.0)
    # flat interface: no curvature where there is an interface (far away, where |grad C| drops below eps_t, the normal of
    # Eq. 23 decays from 1 to 0 and kappa is not small, but it multiplies grad C ~ 1e-8 there)
    assert np.abs(kap[np.abs(z - 0.5) < 3 * h]).max() < 1e-3          # vs -8 for the sphere below; the rest is eps_t / |grad C|
    _, _, st1 = orc.hydrostatic_rhs(g, Cf, 1000.0, 1.0, 9.81, 1.0)
    assert max(np.abs(a).max() for a in st1) < 1e-3          # vs sigma kappa |grad C| ~ 8 * 20 for the sphere below
    x, _, rel, _ = orc.solve(g, BC_PHS, None, np.zeros(g.shape), b, 3, 1e-11, 400)
    dpdz = (x[2:] - x[:-2]) / (2 * h)
    assert np.allclose(dpdz[2:8, 4, 4], -1000.0 * 9.81, rtol=2e-3)      # in the water
    assert np.allclose(dpdz[-5:-2, 4, 4], -1.0 * 9.81, rtol=5e-3)       # in the air, clear of the smoothed interface


def test_curvature_of_a_sphere(orc):
    """kappa = -div(grad C / |grad C|) (reading N3): for a drop (C = 1 inside a sphere of radius R) the curvature is +2 / r on
    the interface (second-order filters: a few per cent at 12 cells per radius), the force sigma kappa grad C points to the
    centre, and p_hs is higher inside by 2 sigma / R (Young-Laplace)."""
    n = 48
    h = 1.0 / n
    g = orc.grid(n, n, n, h)
    c = (np.arange(n) + 0.5) * h
    Z, Y, X = np.meshgrid(c, c, c, indexing="ij")
    r = np.sqrt((X - 0.5) ** 2 + (Y - 0.5) ** 2 + (Z - 0.5) ** 2)
    R = 0.25
    Cf = 0.5 * (1 - np.tanh((r - R) / (2 * h)))         # 1 inside
    _, kap, st = orc.hydrostatic_rhs(g, Cf, 1000.0, 1.0, 0.0, 1.0)
    shell = np.abs(r - R) < 0.5 * h
    assert shell.sum() > 100
    assert np.allclose(kap[shell] * r[shell], 2.0, rtol=0.05)
    # sigma kappa grad C points along -r_hat: kappa > 0, grad C along -r_hat
    sr = (st[0] * (X - 0.5) + st[1] * (Y - 0.5) + st[2] * (Z - 0.5)) / np.maximum(r, 1e-12)
    assert (sr[shell] < 0).all()
    # Young-Laplace: p_hs is higher inside the drop by 2 sigma / R
    b, _, _ = orc.hydrostatic_rhs(g, Cf, 1000.0, 1.0, 0.0, 1.0)
    x, _, rel, _ = orc.solve(g, (1,) * 6, None, np.zeros(g.shape), b, 4, 1e-10, 300)
    p_in = x[n // 2, n // 2, n // 2]
    p_out = x[n // 2, n // 2, 3]
    assert abs((p_in - p_out) - 2.0 / R) <= 0.1 * 2.0 / R


# ---- reading C7 (revised): rho and mu from the volume fraction limited to [0, 1]; everything else sees C as it is ----------
def _out_of_range_vof(shape, seed):
    """a smooth interface with undershoots to -0.2 and overshoots to 1.25 on both sides of it"""
    nz, ny, nx = shape
    x, y, z = configs.centres(nx, ny, nz, 1.0)
    d = (0.7 * x / nx + 0.4 * y / ny + 0.6 * z / nz) - 0.8
    Cin = 0.5 * (1 + np.tanh(d * 5.0)) + 0.0 * (x + y + z)
    return 1.45 * Cin - 0.2 + 0.02 * _rand(shape, seed)


def test_material_mixtures_limit_the_volume_fraction(orc):
    """Eqs. 2 / 19 with C limited to [0, 1]: closed-form values of k = 1 / rho; and every routine that sees C only through rho
    and mu gives, for an out-of-range C, exactly what it gives for the limited field (dropping the limit anywhere breaks one
    of the equalities; the inputs make rho NEGATIVE without it: 1000 * (-0.2) + 1.2)."""
    rho_l, rho_g, mu_l, mu_g = 1000.0, 1.0, 1e-3, 1e-5
    a = np.array([-0.2, -1e-3, 0.0, 0.3, 1.0, 1.4])
    assert np.allclose(orc.k_from_vof(a, rho_l, rho_g), [1.0, 1.0, 1.0, 1.0 / (300.0 + 0.7), 1e-3, 1e-3], rtol=1e-15)
    shape, h, dt = (10, 12, 14), 0.1, 0.01
    g = orc.grid(shape[2], shape[1], shape[0], h)
    C = _out_of_range_vof(shape, 7)
    Cl = np.clip(C, 0.0, 1.0)
    assert C.min() < -0.1 and C.max() > 1.1 and (rho_l * C + rho_g * (1 - C)).min() < 0
    q = tuple(0.3 * _rand(shape, 20 + c) + 0.2 for c in range(3))
    for vbc in (None, orc.velocity_bc()):
        for r, rl in zip(orc.mom_predictor(g, C, q, q, rho_l, rho_g, mu_l, mu_g, dt, vbc), orc.mom_predictor(g, Cl, q, q, rho_l, rho_g, mu_l, mu_g, dt, vbc)):
            for c in range(3):
                assert np.array_equal(r[c], rl[c]) and np.isfinite(r[c]).all()
    assert np.array_equal(orc.pressure_rhs_paper(g, C, q[0], q[1], q[2], rho_l, rho_g, dt), orc.pressure_rhs_paper(g, Cl, q[0], q[1], q[2], rho_l, rho_g, dt))
    p_hs, p_nh = 1e3 * _rand(shape, 31), 1e3 * _rand(shape, 32)
    st = tuple(1e3 * _rand(shape, 33 + c) for c in range(3))
    pbc = (0, 1, 0, 0, 0, 1)
    f, fl = (orc.mom_forcing(g, c_, p_hs, p_nh, pbc, 9.81, st, rho_l, rho_g, dt, q) for c_ in (C, Cl))
    for c in range(3):
        assert np.array_equal(f[c], fl[c])


def test_only_the_mixtures_are_limited_not_the_interface_terms(orc):
    """hydrostatic_rhs = gravity part (through rho: limited) + surface-tension part (through grad C and the curvature: NOT
    limited).  sigma = 0: equal to the limited field's, bit for bit.  g = 0: C' = 1.45 C - 0.2 has the same normals and
    curvature as C and 1.45 times its gradient, so b(C') = 1.45 b(C) (up to the epsilon of the normalisation) -- a limit on C in
    the curvature or in grad C would flatten C' and break this by O(1)."""
    n, h = 16, 1.0 / 16
    g = orc.grid(n, n, n, h)
    c = (np.arange(n) + 0.5) * h
    Z, Y, X = np.meshgrid(c, c, c, indexing="ij")
    r = np.sqrt((X - 0.5) ** 2 + (Y - 0.45) ** 2 + (Z - 0.55) ** 2)
    C0 = 0.5 * (1 - np.tanh((r - 0.25) / (1.5 * h)))
    C1 = 1.45 * C0 - 0.2
    assert C1.min() < -0.19 and C1.max() > 1.2
    b_g, _, _ = orc.hydrostatic_rhs(g, C1, 1000.0, 1.0, 9.81, 0.0)
    b_gl, _, _ = orc.hydrostatic_rhs(g, np.clip(C1, 0, 1), 1000.0, 1.0, 9.81, 0.0)
    assert np.array_equal(b_g, b_gl) and np.abs(b_g).max() > 0
    b_s0, kap0, st0 = orc.hydrostatic_rhs(g, C0, 1000.0, 1.0, 0.0, 0.0728)
    b_s1, kap1, st1 = orc.hydrostatic_rhs(g, C1, 1000.0, 1.0, 0.0, 0.0728)
    band = np.abs(C0 - 0.5) < 0.4                                   # where the gradient is well above the normalisation's epsilon
    assert np.abs(b_s0[band]).max() > 0
    assert np.abs(b_s1 - 1.45 * b_s0)[band].max() < 2e-3 * np.abs(b_s0[band]).max()
    b_cl, _, _ = orc.hydrostatic_rhs(g, np.clip(C1, 0, 1), 1000.0, 1.0, 0.0, 0.0728)
    assert np.abs(b_cl - 1.45 * b_s0)[band].max() > 0.05 * np.abs(b_s0[band]).max()      # the limited field is a different problem
