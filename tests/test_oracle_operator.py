"""Pins of the oracle's filters, operator and boundary conditions (readings C1-C3).

Each test checks the oracle against something the paper or mathematics fixes, not against
a retyped copy of its own formula.
"""
import itertools
import os

import numpy as np
import pytest

N, D, DH = 0, 1, 2  # bc codes
HERE = os.path.dirname(os.path.abspath(__file__))

BC_MIXES = [(D,) * 6, (N,) * 5 + (D,), (N, D, DH, N, D, DH), (DH,) * 6, (N,) * 6]


def _rand(shape, seed):
    return np.random.default_rng(seed).standard_normal(shape)


def test_eq11_printed_weights(orc):
    """Eq. 11: the printed integer slices of w_x, prefactor m_l/(72 dx)."""
    rows = [l.split() for l in open(os.path.join(HERE, "golden", "eq11_wx.txt")) if l.strip() and l[0] != "#"]
    printed = np.array(rows, dtype=float).reshape(3, 3, 3)        # [kk, jj, ii]
    g = orc.grid(8, 8, 8, 0.3, 0.7, 1.1)
    wx = orc.filter_weights(g, "x")                               # nodal = integrated / m_l
    assert np.allclose(wx * 72.0 * g.hx, printed, rtol=0, atol=1e-13)
    # w_y, w_z are the same filter with the axes exchanged
    assert np.allclose(orc.filter_weights(g, "y") * 72.0 * g.hy, printed.transpose(0, 2, 1), atol=1e-13)
    assert np.allclose(orc.filter_weights(g, "z") * 72.0 * g.hz, printed.transpose(2, 1, 0), atol=1e-13)


def _fe_stencils_by_quadrature(hx, hy, hz):
    """Independent derivation: assemble the trilinear-FE stiffness / mass / d-dx rows of the
    centre node of a 2x2x2 patch of hexahedra by 2-point Gauss quadrature (exact here)."""
    gp = np.array([-1.0, 1.0]) / np.sqrt(3.0)
    h = (hx, hy, hz)

    def shape1d(node, xi):      # node in {0,1}; reference coordinate xi in [-1,1]
        return (0.5 * (1 - xi), -0.5) if node == 0 else (0.5 * (1 + xi), 0.5)

    lap = np.zeros((3, 3, 3)); mass = np.zeros((3, 3, 3)); ddx = np.zeros((3, 3, 3))
    for ez, ey, ex in itertools.product((0, 1), repeat=3):         # the 8 elements around the centre node
        a = (1 - ex, 1 - ey, 1 - ez)                               # local index of the centre node in this element
        for bz, by, bx in itertools.product((0, 1), repeat=3):
            b = (bx, by, bz)
            off = (ex + bx - 1, ey + by - 1, ez + bz - 1)          # stencil offset of node b
            for qz, qy, qx in itertools.product(gp, repeat=3):
                q = (qx, qy, qz)
                Na = [shape1d(a[d], q[d]) for d in range(3)]
                Nb = [shape1d(b[d], q[d]) for d in range(3)]
                jac = hx * hy * hz / 8.0
                va = Na[0][0] * Na[1][0] * Na[2][0]
                vb = Nb[0][0] * Nb[1][0] * Nb[2][0]
                ga = [Na[d][1] * 2 / h[d] * np.prod([Na[e][0] for e in range(3) if e != d]) for d in range(3)]
                gb = [Nb[d][1] * 2 / h[d] * np.prod([Nb[e][0] for e in range(3) if e != d]) for d in range(3)]
                idx = (off[2] + 1, off[1] + 1, off[0] + 1)
                lap[idx] += jac * sum(ga[d] * gb[d] for d in range(3))
                mass[idx] += jac * va * vb
                ddx[idx] += jac * va * gb[0]
    return lap, mass, ddx


@pytest.mark.parametrize("h", [(0.25, 0.25, 0.25), (0.5, 0.2, 0.9)])
def test_filters_equal_fe_integrals(orc, h):
    """the filters are the FE basis-function integrals (here by quadrature)."""
    g = orc.grid(4, 4, 4, *h)
    ml = h[0] * h[1] * h[2]
    lap, mass, ddx = _fe_stencils_by_quadrature(*h)
    assert np.allclose(orc.filter_weights(g, "lap") * ml, lap, atol=1e-12 * abs(lap).max())
    assert np.allclose(orc.filter_weights(g, "mass") * ml, mass, atol=1e-13)
    assert np.allclose(orc.filter_weights(g, "x") * ml, ddx, atol=1e-13)
    tot = orc.filter_weights(g, "xx") + orc.filter_weights(g, "yy") + orc.filter_weights(g, "zz")
    assert np.allclose(tot, orc.filter_weights(g, "lap"), atol=1e-12 * abs(lap).max() / ml)
    assert abs(orc.filter_weights(g, "lap").sum()) < 1e-10 * abs(lap).max() / ml      # row sum 0
    assert abs(orc.filter_weights(g, "mass").sum() - 1.0) < 1e-13                     # w_m/m_l sums to 1


def test_uniform_laplacian_weights(orc):
    """On a uniform grid: centre 8/(3h^2), faces 0, edges -1/(6h^2), corners -1/(12h^2)."""
    h = 0.125
    w = orc.filter_weights(orc.grid(4, 4, 4, h), "lap") * h * h
    for kk, jj, ii in itertools.product(range(3), repeat=3):
        nz = (kk != 1) + (jj != 1) + (ii != 1)
        assert abs(w[kk, jj, ii] - [8 / 3, 0.0, -1 / 6, -1 / 12][nz]) < 1e-13


def _mode(n, m, kind, nodes="centre"):
    i = np.arange(n)
    if kind == "sin":
        return np.sin(np.pi * m * (i + 0.5) / n) if nodes == "centre" else np.sin(np.pi * m * (i + 1) / (n + 1))
    return np.cos(np.pi * m * (i + 0.5) / n)


@pytest.mark.parametrize("bc,kind,nodes", [((D,) * 6, "sin", "centre"), ((N,) * 6, "cos", "centre"),
                                           ((DH,) * 6, "sin", "halo")])
def test_closed_form_eigenpairs(orc, bc, kind, nodes):
    """Tensor-product Fourier modes are exact eigenvectors with
    lambda = sum_d (4/h_d^2) s_d prod_{e!=d} (1 - 2/3 s_e), s = sin^2(theta/2) (reading C1-ii, C3)."""
    nx, ny, nz = 12, 10, 8
    g = orc.grid(nx, ny, nz, 1.0 / nx, 1.3 / ny, 0.7 / nz)
    for (mx, my, mz) in [(1, 1, 1), (3, 2, 5), (1, 4, 2)]:
        vec = (_mode(nz, mz, kind, nodes)[:, None, None] * _mode(ny, my, kind, nodes)[None, :, None] *
               _mode(nx, mx, kind, nodes)[None, None, :])
        th = [np.pi * m / (n if nodes == "centre" else n + 1) for m, n in ((mx, nx), (my, ny), (mz, nz))]
        s = [np.sin(t / 2) ** 2 for t in th]
        hh = [g.hx, g.hy, g.hz]
        lam = sum(4 / hh[d] ** 2 * s[d] * np.prod([1 - 2 / 3 * s[e] for e in range(3) if e != d]) for d in range(3))
        y = orc.apply_operator(g, bc, None, vec)
        assert np.abs(y - lam * vec).max() < 1e-10 * lam


def test_isotropic_lowest_eigenvalue_formula(orc):
    """lambda_h = 3 (4/h^2) s (1 - 2/3 s)^2 -> 3 pi^2 from below at O(h^2)."""
    n = 32
    g = orc.grid(n, n, n, 1.0 / n)
    v = _mode(n, 1, "sin")
    vec = v[:, None, None] * v[None, :, None] * v[None, None, :]
    s = np.sin(np.pi / (2 * n)) ** 2
    lam = 3 * 4 * n * n * s * (1 - 2 / 3 * s) ** 2
    assert abs(lam - 29.490142179) < 1e-8
    assert np.abs(orc.apply_operator(g, (D,) * 6, None, vec) - lam * vec).max() < 1e-9


def test_manufactured_solution_second_order(orc):
    """-lap u = 3 pi^2 u, u = sin sin sin with zero Dirichlet faces: error drops 4x per halving
    (solution by a dense direct solve of the oracle's own matrix, 4^3 and 8^3)."""
    errs = []
    for n in (4, 8):
        g = orc.grid(n, n, n, 1.0 / n)
        A = _dense(orc, g, (D,) * 6, None)
        c = (np.arange(n) + 0.5) / n
        u = (np.sin(np.pi * c)[:, None, None] * np.sin(np.pi * c)[None, :, None] * np.sin(np.pi * c)[None, None, :])
        uh = np.linalg.solve(A, (3 * np.pi ** 2 * u).ravel())
        errs.append(np.abs(uh - u.ravel()).max())
    assert 3.3 < errs[0] / errs[1] < 4.7


def _dense(orc, g, bc, k):
    n = g.nx * g.ny * g.nz
    A = np.zeros((n, n))
    e = np.zeros(n)
    for c in range(n):
        e[c] = 1.0
        A[:, c] = orc.apply_operator(g, bc, k, e.reshape(g.shape)).ravel()
        e[c] = 0.0
    return A


@pytest.mark.parametrize("bc", BC_MIXES)
@pytest.mark.parametrize("var", [False, True])
def test_symmetry_and_semidefiniteness(orc, bc, var):
    """<Au,v> = <u,Av> under every BC mix; A is positive semi-definite (C1-iv, C2)."""
    g = orc.grid(7, 6, 5, 0.2)
    k = np.exp(_rand(g.shape, 5)) if var else None
    u, v = _rand(g.shape, 1), _rand(g.shape, 2)
    Au, Av = orc.apply_operator(g, bc, k, u), orc.apply_operator(g, bc, k, v)
    assert abs((Au * v).sum() - (u * Av).sum()) < 1e-12 * np.abs(Au).max() * u.size
    assert (Au * u).sum() > -1e-12


@pytest.mark.parametrize("var", [False, True])
def test_constant_null_space_all_neumann(orc, var):
    g = orc.grid(6, 5, 4, 0.1, 0.2, 0.15)
    k = np.exp(_rand(g.shape, 3)) if var else None
    y = orc.apply_operator(g, (N,) * 6, k, np.ones(g.shape))
    assert np.abs(y).max() < 1e-10


@pytest.mark.parametrize("bc", BC_MIXES)
def test_eq13_literal_equals_difference_form(orc, bc):
    """Eq. 13 written as three stencils == collapsed arithmetic-mean form (C2)."""
    g = orc.grid(6, 7, 5, 0.1, 0.13, 0.09)
    k = np.exp(_rand(g.shape, 11))
    x = _rand(g.shape, 12)
    a = orc.apply_operator(g, bc, k, x)
    b = orc.apply_operator(g, bc, k, x, eq13=True)
    assert np.abs(a - b).max() < 1e-12 * np.abs(a).max()


def test_constant_k_scales_operator_and_diagonal_identity(orc):
    """k == c gives c*A; D = w0 k - 1/2 f(k; w_lap) with copy halos (C2 pins)."""
    g = orc.grid(6, 6, 6, 0.25)
    x = _rand(g.shape, 4)
    bc = (N, N, N, N, N, D)
    a0 = orc.apply_operator(g, bc, None, x)
    a1 = orc.apply_operator(g, bc, np.full(g.shape, 2.5), x)
    assert np.abs(a1 - 2.5 * a0).max() < 1e-11 * np.abs(a0).max()
    k = np.exp(_rand(g.shape, 6))
    w = orc.filter_weights(g, "lap")
    Wk = orc.apply_filter(g, (N,) * 6, w, k)
    assert np.abs(orc.diagonal(g, k) - (w[1, 1, 1] * k - 0.5 * Wk)).max() < 1e-10 * w[1, 1, 1]
    assert np.abs(orc.diagonal(g, None) - w[1, 1, 1]).max() == 0.0
    assert (orc.diagonal(g, k) > 0).all()


def test_bc_ghost_rules(orc):
    """P:256-258 / Fig. 2: the identity filter shifted by one picks out the halo value."""
    g = orc.grid(4, 3, 2, 1.0)
    x = _rand(g.shape, 9)
    for face, (axis, side) in enumerate([(2, 0), (2, -1), (1, 0), (1, -1), (0, 0), (0, -1)]):
        for code, s in ((N, 1.0), (D, -1.0), (DH, 0.0)):
            bc = [N] * 6
            bc[face] = code
            w = np.zeros((3, 3, 3))
            off = [1, 1, 1]
            off[axis] = 0 if side == 0 else 2          # read the neighbour across that face
            w[tuple(off)] = 1.0
            y = orc.apply_filter(g, bc, w, x)
            sl = [slice(None)] * 3
            sl[axis] = side
            assert np.allclose(y[tuple(sl)], s * x[tuple(sl)], atol=0)   # ghost = s * mirror
    # corner ghost: factors multiply
    w = np.zeros((3, 3, 3)); w[0, 0, 0] = 1.0
    y = orc.apply_filter(g, (D, N, D, N, N, N), w, x)
    assert y[0, 0, 0] == x[0, 0, 0] * (-1.0) * (-1.0) * 1.0
