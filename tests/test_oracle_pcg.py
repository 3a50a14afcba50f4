"""Pins of the oracle's V-cycle-preconditioned CG (SURVEY 8(f) "next 1"; not in the paper): what the mathematics fixes
about PCG, none of it by re-running the oracle's own loop.
 - the preconditioner (one V(nu, nu) cycle from zero) is a symmetric linear operator: <M u, v> = <u, M v>
 - the iterates converge to the dense direct solution
 - the energy norm of the error decreases at every iteration (the defining optimality of CG with an SPD preconditioner)
 - successive residuals are M-orthogonal, search directions A-conjugate (rebuilt here from the oracle's building blocks)
 - it needs far fewer V-cycles than the plain cycle under a 1000:1 coefficient jump."""
import numpy as np
import pytest

from test_oracle_multigrid import BC_MIXES, _dense, _rand

N, D = 0, 1


def _M(orc, g, bc, k, r, levels, nu=2):
    return orc.vcycle(g, bc, k, np.zeros(g.shape), r, levels, nu, nu)


@pytest.mark.parametrize("bc", BC_MIXES)
@pytest.mark.parametrize("var", [False, True])
def test_preconditioner_is_symmetric(orc, bc, var):
    g = orc.grid(16, 8, 8, 0.1)
    k = np.exp(_rand(g.shape, 3)) if var else None
    u, v = _rand(g.shape, 1), _rand(g.shape, 2)
    Mu, Mv = _M(orc, g, bc, k, u, 2), _M(orc, g, bc, k, v, 2)
    a, b = np.vdot(Mu, v), np.vdot(u, Mv)
    assert abs(a - b) <= 1e-12 * max(abs(a), abs(b))
    # and positive: <M u, u> > 0
    assert np.vdot(Mu, u) > 0


def test_unequal_smoothing_counts_break_symmetry(orc):
    """The pin above must be able to fail: V(2,1) is not symmetric."""
    g = orc.grid(8, 8, 8, 0.125)
    bc = (N,) * 5 + (D,)
    k = np.exp(_rand(g.shape, 3))
    u, v = _rand(g.shape, 1), _rand(g.shape, 2)
    z = np.zeros(g.shape)
    a = np.vdot(orc.vcycle(g, bc, k, z, u, 2, 2, 1), v)
    b = np.vdot(u, orc.vcycle(g, bc, k, z, v, 2, 2, 1))
    assert abs(a - b) > 1e-6 * max(abs(a), abs(b))


@pytest.mark.parametrize("bc", [(D,) * 6, (N,) * 5 + (D,)])
def test_pcg_converges_to_direct_solution_with_monotone_energy_error(orc, bc):
    g = orc.grid(8, 8, 8, 0.125)
    k = np.exp(1.5 * _rand(g.shape, 5))
    b = _rand(g.shape, 6)
    A = _dense(orc, g, bc, k)
    xs = np.linalg.solve(A, b.ravel())
    prev = None
    for iters in range(1, 9):
        x, n, rel, hist = orc.pcg_solve(g, bc, k, np.zeros(g.shape), b, 2, 0.0, iters)
        assert n == iters
        e = x.ravel() - xs
        en = float(e @ (A @ e))
        if prev is not None:
            assert en < prev                       # energy-norm error strictly decreases
        prev = en
        # the reported residual is the true residual
        assert abs(np.linalg.norm(b.ravel() - A @ x.ravel()) / np.linalg.norm(b) - hist[-1]) <= 1e-9 * max(hist[-1], 1e-300) + 1e-13
    x, n, rel, _ = orc.pcg_solve(g, bc, k, np.zeros(g.shape), b, 2, 1e-12, 60)
    assert rel < 1e-12 and np.linalg.norm(x.ravel() - xs) <= 1e-10 * np.linalg.norm(xs)


def test_pcg_orthogonality_relations(orc):
    """Rebuild two iterations from apply_operator / vcycle and check r1 _|_ z0 (M-orthogonal residuals) and
    p1 A-conjugate to p0; then that the oracle's iterate after 2 iterations is x0 + a0 p0 + a1 p1."""
    g = orc.grid(8, 8, 8, 0.125)
    bc = (N,) * 5 + (D,)
    k = np.exp(_rand(g.shape, 8))
    b = _rand(g.shape, 9)
    Aop = lambda v: orc.apply_operator(g, bc, k, v)
    r0 = b.copy(); z0 = _M(orc, g, bc, k, r0, 2); p0 = z0
    q0 = Aop(p0); a0 = np.vdot(r0, z0) / np.vdot(p0, q0)
    r1 = r0 - a0 * q0; z1 = _M(orc, g, bc, k, r1, 2)
    assert abs(np.vdot(r1, z0)) <= 1e-10 * np.linalg.norm(r1) * np.linalg.norm(z0)
    p1 = z1 + (np.vdot(r1, z1) / np.vdot(r0, z0)) * p0
    assert abs(np.vdot(p1, q0)) <= 1e-10 * np.linalg.norm(p1) * np.linalg.norm(q0)
    a1 = np.vdot(r1, z1) / np.vdot(p1, Aop(p1))
    x2, n, _, _ = orc.pcg_solve(g, bc, k, np.zeros(g.shape), b, 2, 0.0, 2)
    assert np.linalg.norm(x2 - (a0 * p0 + a1 * p1)) <= 1e-12 * np.linalg.norm(x2)


def test_pcg_beats_plain_cycles_under_a_density_jump(orc):
    """Bubble-like 1000:1 coefficient (alpha = 0 inside a sphere): SURVEY hard part 4."""
    n = 32
    g = orc.grid(n, n, n, 1.0 / n)
    bc = (N,) * 5 + (D,)
    c = (np.arange(n) + 0.5) / n
    X, Y, Z = np.meshgrid(c, c, c, indexing="ij")
    d = np.sqrt((X.T - 0.5) ** 2 + (Y.T - 0.5) ** 2 + (Z.T - 0.3) ** 2) - 0.2
    alpha = 0.5 * (1 + np.tanh(d / (1.5 / n)))
    k = orc.k_from_vof(np.ascontiguousarray(alpha), 1000.0, 1.0)
    b = _rand(g.shape, 11)
    _, n_pcg, rel_pcg, _ = orc.pcg_solve(g, bc, k, np.zeros(g.shape), b, 4, 1e-8, 100)
    _, n_cyc, rel_cyc, _ = orc.solve(g, bc, k, np.zeros(g.shape), b, 4, 1e-8, 100)
    assert rel_pcg < 1e-8
    assert n_pcg + 1 <= 0.6 * n_cyc, (n_pcg, n_cyc, rel_cyc)
