"""Pins of the oracle's smoother, transfers, V-cycle and solve (readings C4-C7).

Checked against closed forms, dense linear algebra on grids <= 8^3 and invariants -- never
against a retyped copy of the oracle's own loops.
"""
import numpy as np
import pytest

N, D, DH = 0, 1, 2
BC_MIXES = [(D,) * 6, (N,) * 5 + (D,), (N, D, DH, N, D, DH), (DH,) * 6]


def _rand(shape, seed):
    return np.random.default_rng(seed).standard_normal(shape)


def _dense(orc, g, bc, k):
    n = g.nx * g.ny * g.nz
    A = np.zeros((n, n))
    e = np.zeros(n)
    for c in range(n):
        e[c] = 1.0
        A[:, c] = orc.apply_operator(g, bc, k, e.reshape(g.shape)).ravel()
        e[c] = 0.0
    return A


# ---------------------------------------------------------------- C4: weighted Jacobi
def test_jacobi_fourier_mode_factor(orc):
    """One sweep with b = 0 multiplies a Dirichlet sine mode by 1 - omega*lambda/w0 (closed form)."""
    n = 8
    g = orc.grid(n, n, n, 1.0 / n)
    i = np.arange(n)
    for (mx, my, mz), omega in [((1, 1, 1), 2 / 3), ((3, 5, 2), 0.8), ((8, 8, 8), 2 / 3)]:
        vx, vy, vz = (np.sin(np.pi * m * (i + 0.5) / n) for m in (mx, my, mz))
        vec = vz[:, None, None] * vy[None, :, None] * vx[None, None, :]
        s = [np.sin(np.pi * m / (2 * n)) ** 2 for m in (mx, my, mz)]
        lam = sum(4 * n * n * s[d] * np.prod([1 - 2 / 3 * s[e] for e in range(3) if e != d]) for d in range(3))
        w0 = 8.0 / 3.0 * n * n
        y = orc.jacobi_sweep(g, (D,) * 6, None, vec, np.zeros(g.shape), omega)
        assert np.abs(y - (1 - omega * lam / w0) * vec).max() < 1e-12
    # the worst high-frequency mode (pi,pi,pi) has lambda/w0 = 1/2: smoothing factor 2/3 at omega = 2/3 (C4 note)
    assert abs((1 - (2 / 3) * lam / w0) - 2 / 3) < 1e-12


def test_jacobi_alternating_mode_halves(orc):
    """omega = 1, b = 0: the (pi,0,0) mode (-1)^i maps to -1/2 of itself (C4 pin)."""
    g = orc.grid(8, 4, 4, 0.25)
    vec = np.broadcast_to(((-1.0) ** np.arange(8))[None, None, :], g.shape).copy()
    y = orc.jacobi_sweep(g, (D, D, N, N, N, N), None, vec, np.zeros(g.shape), 1.0)
    assert np.abs(y + 0.5 * vec).max() < 1e-13


@pytest.mark.parametrize("var", [False, True])
def test_jacobi_is_x_plus_omega_dinv_residual(orc, var):
    """x' = x + omega (b - A x) / D with the DENSE matrix of the operator.  D is the conv-layer
    centre coefficient w0 k - 1/2 f(k; w_lap) (reading C2-2, pinned in test_oracle_operator); it
    equals the matrix diagonal except on domain edges/corners, where an edge- or corner-weight
    ghost mirrors onto the cell itself."""
    g = orc.grid(5, 4, 6, 0.2)
    bc = (N, N, N, N, N, D)
    k = np.exp(_rand(g.shape, 1)) if var else None
    A = _dense(orc, g, bc, k)
    w = orc.filter_weights(g, "lap")
    kk = np.ones(g.shape) if k is None else k
    Dc = w[1, 1, 1] * kk - 0.5 * orc.apply_filter(g, (N,) * 6, w, kk)
    inner = np.zeros(g.shape, bool); inner[1:-1, 1:-1, 1:-1] = True
    assert np.allclose(np.diag(A).reshape(g.shape)[inner], Dc[inner], rtol=1e-13)
    x, b = _rand(g.shape, 2), _rand(g.shape, 3)
    ref = x.ravel() + 0.7 * (b.ravel() - A @ x.ravel()) / Dc.ravel()
    y = orc.jacobi_sweep(g, bc, k, x, b, 0.7)
    assert np.abs(y.ravel() - ref).max() < 1e-12 * np.abs(ref).max()
    # and smooth(n) == n single sweeps
    y3 = x
    for _ in range(3):
        y3 = orc.jacobi_sweep(g, bc, k, y3, b, 0.7)
    assert np.array_equal(orc.smooth(g, bc, k, x, b, 0.7, 3), y3)


def test_jacobi_fixed_point_is_direct_solution(orc):
    g = orc.grid(4, 4, 4, 0.25)
    bc = (N, N, N, N, N, D)
    k = np.exp(_rand(g.shape, 7))
    b = _rand(g.shape, 8)
    xs = np.linalg.solve(_dense(orc, g, bc, k), b.ravel()).reshape(g.shape)
    y = orc.jacobi_sweep(g, bc, k, xs, b, 2 / 3)
    assert np.abs(y - xs).max() < 1e-12 * np.abs(xs).max()


# ---------------------------------------------------------------- C5: transfers
def test_restriction_prolongation_pins(orc):
    g = orc.grid(8, 6, 4, 0.1)
    assert np.array_equal(orc.restrict(g, np.ones(g.shape)), np.ones((2, 3, 4)))          # R 1 = 1
    assert np.array_equal(orc.prolong_add(g, np.ones((2, 3, 4)), np.zeros(g.shape)), np.ones(g.shape))
    r, e = _rand(g.shape, 1), _rand((2, 3, 4), 2)
    lhs = 8.0 * (orc.restrict(g, r) * e).sum()                                              # <R r, e>_c * 8
    rhs = (r * orc.prolong_add(g, e, np.zeros(g.shape))).sum()                              # <r, P e>
    assert abs(lhs - rhs) < 1e-12 * abs(rhs)
    # restriction is the block mean, prolongation is np.repeat (library re-statement)
    assert np.allclose(orc.restrict(g, r), r.reshape(2, 2, 3, 2, 4, 2).mean(axis=(1, 3, 5)), atol=1e-15)
    up = np.repeat(np.repeat(np.repeat(e, 2, 0), 2, 1), 2, 2)
    assert np.array_equal(orc.prolong_add(g, e, r), r + up)


def test_k_from_vof(orc):
    """Eqs. 2 and 19: alpha = 1 -> 1/rho_l, alpha = 0 -> 1/rho_g, midpoint -> 2/(rho_l+rho_g)."""
    k = orc.k_from_vof(np.array([[[1.0, 0.0, 0.5, 0.25]]]), 1000.0, 1.0)
    assert np.allclose(k.ravel(), [1e-3, 1.0, 2 / 1001.0, 1 / 250.75], rtol=1e-15)


# ---------------------------------------------------------------- C6: V-cycle and solve
def _two_grid_matrix(orc, g, bc, k, nu1, nu2, nc, omega):
    """Error-propagation matrix of the 2-level cycle assembled by dense algebra from the oracle's
    PIECES (operator, restrict, prolong), not from orc_vcycle."""
    n = g.nx * g.ny * g.nz
    A = _dense(orc, g, bc, k)
    S = np.eye(n) - omega * A / orc.diagonal(g, k).ravel()[:, None]
    gc = orc.grid(g.nx // 2, g.ny // 2, g.nz // 2, 2 * g.hx, 2 * g.hy, 2 * g.hz)
    m = gc.nx * gc.ny * gc.nz
    kc = None if k is None else orc.restrict(g, k)
    Ac = _dense(orc, gc, bc, kc)
    R = np.zeros((m, n)); P = np.zeros((n, m))
    for c in range(n):
        e = np.zeros(n); e[c] = 1
        R[:, c] = orc.restrict(g, e.reshape(g.shape)).ravel()
    for c in range(m):
        e = np.zeros(m); e[c] = 1
        P[:, c] = orc.prolong_add(g, e.reshape(gc.shape), np.zeros(g.shape)).ravel()
    Sc = np.eye(m) - omega * Ac / orc.diagonal(gc, kc).ravel()[:, None]
    # nc Jacobi sweeps from a zero guess: x_c = (I - Sc^nc) Ac^-1 b_c
    Bc = (np.eye(m) - np.linalg.matrix_power(Sc, nc)) @ np.linalg.inv(Ac)
    E = np.linalg.matrix_power(S, nu2) @ (np.eye(n) - P @ Bc @ R @ A) @ np.linalg.matrix_power(S, nu1)
    return A, E


@pytest.mark.parametrize("bc", BC_MIXES)
@pytest.mark.parametrize("var", [False, True])
def test_vcycle_equals_dense_two_grid_operator(orc, bc, var):
    """orc_vcycle (2 levels, 8^3 -> 4^3) applied to (x, b) gives x* + E (x - x*) with E the dense
    two-grid error propagator: pins the order of the steps, the coarse operator and the transfers."""
    g = orc.grid(8, 8, 8, 0.125)
    k = np.exp(_rand(g.shape, 21)) if var else None
    A, E = _two_grid_matrix(orc, g, bc, k, 2, 2, 50, 2 / 3)
    x, b = _rand(g.shape, 22), _rand(g.shape, 23)
    xs = np.linalg.solve(A, b.ravel())
    ref = xs + E @ (x.ravel() - xs)
    y = orc.vcycle(g, bc, k, x, b, levels=2, nu_pre=2, nu_post=2, coarse_sweeps=50, omega=2 / 3)
    assert np.abs(y.ravel() - ref).max() < 1e-10 * np.abs(ref).max()
    rho = np.abs(np.linalg.eigvals(E)).max()
    assert rho < 1.0


def test_solve_converges_to_direct_solution_and_factor(orc):
    """Config-1-like 8^3 problem: solve() reaches the dense solution; the observed asymptotic
    factor equals the spectral radius of the dense two-grid operator; history is monotone."""
    g = orc.grid(8, 8, 8, 0.125)
    bc = (D,) * 6
    A, E = _two_grid_matrix(orc, g, bc, None, 2, 2, 50, 2 / 3)
    b = _rand(g.shape, 31); b -= b.mean()
    x, cycles, rel, hist = orc.solve(g, bc, None, np.zeros(g.shape), b, levels=2, tol=1e-13, max_cycles=60)
    xs = np.linalg.solve(A, b.ravel())
    assert rel < 1e-13 and cycles < 60
    assert np.abs(x.ravel() - xs).max() < 1e-11 * np.abs(xs).max()
    assert (np.diff(hist) < 0).all()
    rho = np.abs(np.linalg.eigvals(E)).max()
    obs = (hist[-1] / hist[-5]) ** 0.25
    assert abs(obs - rho) < 0.05 and rho < 0.3
    # relres reported == ||b - A x|| / ||b|| recomputed densely
    assert abs(rel - np.linalg.norm(b.ravel() - A @ x.ravel()) / np.linalg.norm(b)) < 1e-15


def test_solve_variable_coefficient_three_levels(orc):
    """1000:1 contrast, p_nh boundary conditions, 3 levels 8^3 -> 2^3 against the dense solve."""
    g = orc.grid(8, 8, 8, 0.125)
    bc = (N, N, N, N, N, D)
    alpha = (np.arange(8)[None, None, :] < 3).astype(float) * np.ones(g.shape)
    k = orc.k_from_vof(alpha, 1000.0, 1.0)
    b = _rand(g.shape, 41)
    x, cycles, rel, hist = orc.solve(g, bc, k, np.zeros(g.shape), b, levels=3, tol=1e-12, max_cycles=200)
    xs = np.linalg.solve(_dense(orc, g, bc, k), b.ravel())
    assert rel < 1e-12
    assert np.linalg.norm(x.ravel() - xs) < 1e-9 * np.linalg.norm(xs)


def test_solve_recovers_manufactured_solution(orc):
    """-lap u = 3 pi^2 sin sin sin, 16^3 and 32^3, 3/4 levels: error = discretisation error, O(h^2)."""
    errs = []
    for n, lv in ((16, 3), (32, 4)):
        g = orc.grid(n, n, n, 1.0 / n)
        c = (np.arange(n) + 0.5) / n
        s = np.sin(np.pi * c)
        u = s[:, None, None] * s[None, :, None] * s[None, None, :]
        x, _, rel, _ = orc.solve(g, (D,) * 6, None, np.zeros(g.shape), 3 * np.pi ** 2 * u, levels=lv, tol=1e-11,
                                 max_cycles=40)
        assert rel < 1e-11
        errs.append(np.abs(x - u).max())
        # u is an exact discrete eigenvector (C1-ii), so the solution is (3 pi^2 / lambda_h) u in closed form
        sh = np.sin(np.pi / (2 * n)) ** 2
        lam = 3 * 4 * n * n * sh * (1 - 2 / 3 * sh) ** 2
        assert abs(errs[-1] - (3 * np.pi ** 2 / lam - 1) * u.max()) < 1e-9
    assert 3.5 < errs[0] / errs[1] < 4.5


def test_vcycle_zero_guess_first_sweep_is_pointwise(orc):
    """Fusion equivalence (C6): from x = 0 one generic sweep equals omega b / D."""
    g = orc.grid(6, 6, 6, 0.1)
    k = np.exp(_rand(g.shape, 5)); b = _rand(g.shape, 6)
    y = orc.jacobi_sweep(g, (N,) * 5 + (D,), k, np.zeros(g.shape), b, 2 / 3)
    assert np.abs(y - (2 / 3) * b / orc.diagonal(g, k)).max() < 1e-15 * np.abs(y).max()


@pytest.mark.parametrize("var", [False, True])
def test_two_sweeps_from_zero_are_one_pass_over_the_jacobi_seed(orc, var):
    """The identity behind the CUDA path's seeded correction cycles: with y = b / D, two weighted-Jacobi sweeps
    from x = 0 give x_2 = omega (2 - omega) y - omega^2 D^-1 (A - D) y.  Checked with the oracle's own sweeps, operator and
    diagonal on a mixed-BC, variable-coefficient problem; a wrong weight or sign in either form shows at O(1)."""
    from workloads import rng
    nx, ny, nz, h = 12, 10, 8, 0.05
    g = orc.grid(nx, ny, nz, h)
    bc = (0, 1, 2, 0, 1, 0)
    n = nx * ny * nz
    b = rng.normal(301, n).reshape(nz, ny, nx)
    k = np.exp(-3.0 * rng.uniform01(302, n)).reshape(nz, ny, nx) if var else None
    omega = 2.0 / 3.0
    x2 = orc.smooth(g, bc, k, np.zeros_like(b), b, omega, 2)
    D = orc.diagonal(g, k)
    y = b / D
    Ay = orc.apply_operator(g, bc, k, y)
    seeded = omega * (2.0 - omega) * y - omega ** 2 * (Ay - D * y) / D
    assert np.linalg.norm(seeded - x2) <= 1e-13 * np.linalg.norm(x2)
    x1 = orc.smooth(g, bc, k, np.zeros_like(b), b, omega, 1)
    assert np.linalg.norm(x1 - omega * y) <= 1e-14 * np.linalg.norm(x1)
