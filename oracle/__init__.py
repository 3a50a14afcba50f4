"""ctypes wrapper around oracle/oracle.c -- the fp64 CPU oracle (TEST INFRASTRUCTURE).

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference leg
may import this package.  It never imports the CUDA package and shares no code with it.
All arrays are float64, C-contiguous, shape (nz, ny, nx).
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "oracle.c")
_LIB = os.path.join(_HERE, "liboracle.so")
_lib = None


class Grid(C.Structure):
    _fields_ = [("nx", C.c_int), ("ny", C.c_int), ("nz", C.c_int),
                ("hx", C.c_double), ("hy", C.c_double), ("hz", C.c_double)]

    @property
    def shape(self):
        return (self.nz, self.ny, self.nx)


def grid(nx, ny, nz, hx, hy=None, hz=None):
    return Grid(nx, ny, nz, hx, hx if hy is None else hy, hx if hz is None else hz)


# ORACLE_SANITIZE=1: the pins run against a build with AddressSanitizer + UndefinedBehaviorSanitizer (no OpenMP, -O1);
# the interpreter must then be started with LD_PRELOAD=$(gcc -print-file-name=libasan.so) (profiles/r02_oracle_sanitizers.md)
_SANITIZE = os.environ.get("ORACLE_SANITIZE", "") == "1"
if _SANITIZE:
    _LIB = os.path.join(_HERE, "liboracle_san.so")


def build(force=False):
    """Compile oracle.c with gcc (plain C99, -O2, OpenMP on the outer z loops)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        flags = ["-O1", "-g", "-fsanitize=address,undefined", "-fno-omit-frame-pointer"] if _SANITIZE else ["-O2", "-fopenmp"]
        subprocess.check_call(["gcc", *flags, "-fPIC", "-shared", "-std=c99", "-Wall", "-o", _LIB, _SRC, "-lm"])
    return _LIB


def lib():
    global _lib
    if _lib is None:
        _lib = C.CDLL(build())
        _lib.orc_norm2.restype = C.c_double
        _lib.orc_solve.restype = C.c_int
        _lib.orc_pcg_solve.restype = C.c_int
        _lib.orc_num_threads.restype = C.c_int
    return _lib


def _p(a):
    if a is None:
        return None
    assert a.dtype == np.float64 and a.flags.c_contiguous
    return a.ctypes.data_as(C.c_void_p)


def _bc(bc):
    return (C.c_int * 6)(*[int(b) for b in bc])


def _f64(a):
    return None if a is None else np.ascontiguousarray(a, dtype=np.float64)


def num_threads():
    return lib().orc_num_threads()


def set_threads(n):
    lib().orc_set_threads(int(n))


FILTERS = {"lap": 0, "x": 1, "y": 2, "z": 3, "xx": 4, "yy": 5, "zz": 6, "mass": 7}


def filter_weights(g, which):
    """(3,3,3) array indexed [kk+1, jj+1, ii+1] of the nodal filter `which`."""
    w = np.zeros(27)
    lib().orc_filter(C.byref(g), FILTERS[which], _p(w))
    return w.reshape(3, 3, 3)


def apply_filter(g, bc, w, field):
    field = _f64(field); w = _f64(w).reshape(27)
    y = np.empty(g.shape)
    lib().orc_apply_filter(C.byref(g), _bc(bc), _p(w), _p(field), _p(y))
    return y


def apply_operator(g, bc, k, x, eq13=False):
    k = _f64(k); x = _f64(x)
    y = np.empty(g.shape)
    fn = lib().orc_apply_operator_eq13 if eq13 else lib().orc_apply_operator
    fn(C.byref(g), _bc(bc), _p(k), _p(x), _p(y))
    return y


def diagonal(g, k):
    k = _f64(k)
    d = np.empty(g.shape)
    lib().orc_diagonal(C.byref(g), _p(k), _p(d))
    return d


def jacobi_sweep(g, bc, k, x, b, omega):
    k = _f64(k); x = _f64(x); b = _f64(b)
    y = np.empty(g.shape)
    lib().orc_jacobi_sweep(C.byref(g), _bc(bc), _p(k), _p(x), _p(b), C.c_double(omega), _p(y))
    return y


def smooth(g, bc, k, x, b, omega, sweeps):
    k = _f64(k); b = _f64(b)
    x = np.array(x, dtype=np.float64, order="C")
    lib().orc_smooth(C.byref(g), _bc(bc), _p(k), _p(x), _p(b), C.c_double(omega), int(sweeps))
    return x


def residual(g, bc, k, x, b):
    k = _f64(k); x = _f64(x); b = _f64(b)
    r = np.empty(g.shape)
    lib().orc_residual(C.byref(g), _bc(bc), _p(k), _p(x), _p(b), _p(r))
    return r


def restrict(g, rf):
    rf = _f64(rf)
    rc = np.empty((g.nz // 2, g.ny // 2, g.nx // 2))
    lib().orc_restrict(C.byref(g), _p(rf), _p(rc))
    return rc


def prolong_add(g, xc, xf):
    xc = _f64(xc)
    xf = np.array(xf, dtype=np.float64, order="C")
    lib().orc_prolong_add(C.byref(g), _p(xc), _p(xf))
    return xf


def k_from_vof(alpha, rho_l, rho_g):
    alpha = _f64(alpha)
    k = np.empty_like(alpha)
    lib().orc_k_from_vof(C.c_size_t(alpha.size), _p(alpha), C.c_double(rho_l), C.c_double(rho_g), _p(k))
    return k


def vcycle(g, bc, k, x, b, levels, nu_pre=2, nu_post=2, coarse_sweeps=50, omega=2.0 / 3.0):
    k = _f64(k); b = _f64(b)
    x = np.array(x, dtype=np.float64, order="C")
    lib().orc_vcycle(C.byref(g), _bc(bc), _p(k), int(levels), int(nu_pre), int(nu_post), int(coarse_sweeps),
                     C.c_double(omega), _p(x), _p(b))
    return x


def solve(g, bc, k, x, b, levels, tol, max_cycles, nu_pre=2, nu_post=2, coarse_sweeps=50, omega=2.0 / 3.0):
    """Returns (x, cycles, relres, history)."""
    k = _f64(k); b = _f64(b)
    x = np.array(x, dtype=np.float64, order="C")
    hist = np.zeros(max(max_cycles, 1))
    rel = C.c_double(0.0)
    n = lib().orc_solve(C.byref(g), _bc(bc), _p(k), int(levels), int(nu_pre), int(nu_post), int(coarse_sweeps),
                        C.c_double(omega), _p(x), _p(b), C.c_double(tol), int(max_cycles), _p(hist), C.byref(rel))
    return x, n, rel.value, hist[:n]


def pcg_solve(g, bc, k, x, b, levels, tol, max_iter, nu=2, coarse_sweeps=50, omega=2.0 / 3.0):
    """V-cycle-preconditioned CG.  Returns (x, iterations, relres, history)."""
    k = _f64(k); b = _f64(b)
    x = np.array(x, dtype=np.float64, order="C")
    hist = np.zeros(max(max_iter, 1))
    rel = C.c_double(0.0)
    n = lib().orc_pcg_solve(C.byref(g), _bc(bc), _p(k), int(levels), int(nu), int(coarse_sweeps), C.c_double(omega),
                            _p(x), _p(b), C.c_double(tol), int(max_iter), _p(hist), C.byref(rel))
    return x, n, rel.value, hist[:n]


def vof_residual(g, Cf, u, v, w, dt, detector=3):
    """detector: 3 = Eq. 33, 5 = the 5-point oscillation detectors of Eq. 34.  Returns (sC, Cnew)."""
    Cf = _f64(Cf); u = _f64(u); v = _f64(v); w = _f64(w)
    s = np.empty(g.shape); cn = np.empty(g.shape)
    lib().orc_vof_residual_ex(C.byref(g), _p(Cf), _p(u), _p(v), _p(w), C.c_double(dt), int(detector), _p(s), _p(cn))
    return s, cn


def _ptr3(arrs):
    return (C.c_void_p * 3)(*[a.ctypes.data for a in arrs])


def mom_predictor(g, Cf, qh, qn, rho_l, rho_g, mu_l, mu_g, dt, vbc=None):
    """qh, qn: 3-tuples (u, v, w).  vbc as in pressure_rhs().  Returns (q_tilde, q_half_new), each a 3-tuple."""
    Cf = _f64(Cf)
    qh = [_f64(a) for a in qh]; qn = [_f64(a) for a in qn]
    qt = [np.empty(g.shape) for _ in range(3)]; qhn = [np.empty(g.shape) for _ in range(3)]
    lib().orc_mom_predictor_bc(C.byref(g), _p(Cf), _ptr3(qh), _ptr3(qn), _vbc(vbc), C.c_double(rho_l), C.c_double(rho_g),
                               C.c_double(mu_l), C.c_double(mu_g), C.c_double(dt), _ptr3(qt), _ptr3(qhn))
    return tuple(qt), tuple(qhn)


def pressure_rhs(g, u, v, w, dt, vbc=None):
    """vbc: None (velocity halos are copies) or the 18 halo codes of velocity_bc()."""
    u = _f64(u); v = _f64(v); w = _f64(w)
    b = np.empty(g.shape)
    lib().orc_pressure_rhs_bc(C.byref(g), _p(u), _p(v), _p(w), _vbc(vbc), C.c_double(dt), _p(b))
    return b


# halo codes (0 copy, 1 odd about the face, 2 zero) of (u, v, w) on the faces x-, x+, y-, y+, z-, z+
FREE_SLIP_OPEN_TOP = (1, 1, 0, 0, 0, 0,   0, 0, 1, 1, 0, 0,   0, 0, 0, 0, 1, 0)


def velocity_bc(walls=(1, 1, 1, 1, 1, 0)):
    """Free-slip halo codes: on a wall face the component normal to it is odd about the face (zero normal
    velocity on the wall), the tangential ones and everything on an open face are copied."""
    out = []
    for comp in range(3):
        out += [1 if walls[f] and f // 2 == comp else 0 for f in range(6)]
    return tuple(out)


def _vbc(vbc):
    return None if vbc is None else (C.c_int * 18)(*[int(b) for b in vbc])


def mom_forcing(g, Cf, p_hs, p_nh, pbc, grav, st, rho_l, rho_g, dt, qt):
    """q~ <- q~ - (dt / rho) (grad p_hs + grad p~_nh - M (s + s_t))  (Eq. 18's forcing terms).  p_hs, p_nh, st may be None.
    Returns the new 3-tuple."""
    Cf = _f64(Cf)
    qt = [np.array(a, dtype=np.float64, order="C") for a in qt]
    st = None if st is None else [_f64(a) for a in st]
    lib().orc_mom_forcing(C.byref(g), _p(Cf), _p(_f64(p_hs)), _p(_f64(p_nh)), _bc(pbc), C.c_double(grav),
                          None if st is None else _ptr3(st), C.c_double(rho_l), C.c_double(rho_g), C.c_double(dt), _ptr3(qt))
    return tuple(qt)


def pressure_rhs_paper(g, Cf, u, v, w, rho_l, rho_g, dt):
    """Eq. 53's right-hand side (constant-coefficient Laplacian, density on the right)."""
    Cf = _f64(Cf); u = _f64(u); v = _f64(v); w = _f64(w)
    b = np.empty(g.shape)
    lib().orc_pressure_rhs_paper(C.byref(g), _p(Cf), _p(u), _p(v), _p(w), C.c_double(rho_l), C.c_double(rho_g),
                                 C.c_double(dt), _p(b))
    return b


def hydrostatic_rhs(g, Cf, rho_l, rho_g, grav, sigma_t):
    """Stage 1.  Returns (b_hs, kappa, (s_tu, s_tv, s_tw))."""
    Cf = _f64(Cf)
    b = np.empty(g.shape); kap = np.empty(g.shape)
    st = [np.empty(g.shape) for _ in range(3)]
    lib().orc_hydrostatic_rhs(C.byref(g), _p(Cf), C.c_double(rho_l), C.c_double(rho_g), C.c_double(grav), C.c_double(sigma_t),
                              _p(b), _p(kap), _ptr3(st))
    return b, kap, tuple(st)


def project_velocity(g, bc, p, k, dt, u, v, w):
    p = _f64(p); k = _f64(k)
    u, v, w = (np.array(a, dtype=np.float64, order="C") for a in (u, v, w))
    lib().orc_project_velocity(C.byref(g), _bc(bc), _p(p), _p(k), C.c_double(dt), _p(u), _p(v), _p(w))
    return u, v, w


def time_step(g, bc, Cf, u, v, w, levels, rho_l, rho_g, mu_l, mu_g, dt, tol, max_cycles,
              nu_pre=2, nu_post=2, coarse_sweeps=50, omega=2.0 / 3.0, solver="mg"):
    """One time step of BASELINE config 5, stages 2-4 of PAPER.md:403-505 under the readings
    C9/C10 of DESIGN.md, composed from the oracle's own steps:
      stage 2: q_half = q_n; two predictor iterations (Eqs. 45-46)
      stage 3: k = 1/rho(C_n); b = -(1/dt) D.q~; solve A(k) p = b from p = 0; q = q~ - dt k G p
               (Eqs. 48, 52-54)
      stage 4: C_new = C_n - dt s~_C(C_n, q) (Eqs. 16, 55)
    solver = "mg": plain V-cycles (the paper); "pcg": pcg_solve (nu_pre == nu_post).
    Returns (C_new, u, v, w, p, cycles, relres)."""
    qn = (u, v, w)
    qt, qh = mom_predictor(g, Cf, qn, qn, rho_l, rho_g, mu_l, mu_g, dt)
    qt, _ = mom_predictor(g, Cf, qh, qn, rho_l, rho_g, mu_l, mu_g, dt)
    k = k_from_vof(Cf, rho_l, rho_g)
    b = pressure_rhs(g, qt[0], qt[1], qt[2], dt)
    if solver == "pcg":
        p, cycles, rel, _ = pcg_solve(g, bc, k, np.zeros(g.shape), b, levels, tol, max_cycles, nu_pre, coarse_sweeps, omega)
    else:
        p, cycles, rel, _ = solve(g, bc, k, np.zeros(g.shape), b, levels, tol, max_cycles, nu_pre, nu_post,
                                  coarse_sweeps, omega)
    un, vn, wn = project_velocity(g, bc, p, k, dt, qt[0], qt[1], qt[2])
    _, Cn = vof_residual(g, Cf, un, vn, wn, dt)
    return Cn, un, vn, wn, p, cycles, rel


def time_step_paper(g, bc, Cf, u, v, w, levels, rho_l, rho_g, mu_l, mu_g, dt, cycles=20, passes=2,
                    nu_pre=2, nu_post=2, coarse_sweeps=50, omega=2.0 / 3.0):
    """One time step with the PAPER'S stage 3: constant-coefficient Laplacian, density on the
    right (Eqs. 52-53), `cycles` multigrid cycles per solve (fixed 20), velocity correction Eq. 54, the
    whole stage carried out `passes` times (twice); p_nh accumulates the corrections.  Stages 2 and 4 as
    time_step().  Returns (C_new, u, v, w, p_nh, relres of the last solve)."""
    qn = (u, v, w)
    qt, qh = mom_predictor(g, Cf, qn, qn, rho_l, rho_g, mu_l, mu_g, dt)
    qt, _ = mom_predictor(g, Cf, qh, qn, rho_l, rho_g, mu_l, mu_g, dt)
    k = k_from_vof(Cf, rho_l, rho_g)
    un, vn, wn = qt
    p = np.zeros(g.shape)
    rel = 0.0
    for _ in range(passes):
        b = pressure_rhs_paper(g, Cf, un, vn, wn, rho_l, rho_g, dt)
        dp, _, rel, _ = solve(g, bc, None, np.zeros(g.shape), b, levels, 0.0, cycles, nu_pre, nu_post, coarse_sweeps, omega)
        un, vn, wn = project_velocity(g, bc, dp, k, dt, un, vn, wn)
        p = p + dp
    _, Cn = vof_residual(g, Cf, un, vn, wn, dt)
    return Cn, un, vn, wn, p, rel


BC_PRESSURE = (0, 0, 0, 0, 0, 1)      # p_hs and p_nh: zero derivative on the sides / bottom, zero value on the top face


def time_step_full(g, Cf, u, v, w, p_nh, levels, rho_l, rho_g, mu_l, mu_g, grav, sigma_t, dt, tol, max_cycles,
                   hs_tol=0.0, hs_cycles=20, walls=(1, 1, 1, 1, 1, 0), nu_pre=2, nu_post=2, coarse_sweeps=50, omega=2.0 / 3.0):
    """One time step of the paper's four-stage method, composed from the oracle's steps:
      stage 1: b_hs, s_t from C^n (Eqs. 20-23, 43-44); A p_hs = b_hs, constant coefficient, from p_hs = 0,
                           `hs_cycles` cycles (the paper's fixed 20) or to `hs_tol`
      stage 2: q_half = q_n; twice: q~ from Eq. 45 with the FULL source of Eq. 18 -- advection + Petrov-Galerkin
                           diffusion (mom_predictor, free-slip velocity halos P:538), then the pressure gradients of
                           p_hs and of the previous p_nh and the buoyancy / surface-tension sources (mom_forcing);
                           q_half = (q_n + q~) / 2 (Eq. 46)
      stage 3 (reading C10): b = -(1/dt) D.q~ with the wall halos; A(1/rho) dp = b; q = q~ - dt k G dp (Eq. 54);
                           p_nh += dp
      stage 4: C_new = C_n - dt s~_C(C_n, q) (Eqs. 16, 55)
    Returns (C_new, u, v, w, p_hs, p_nh_new, cycles, relres)."""
    vbc = velocity_bc(walls)
    b_hs, _, st = hydrostatic_rhs(g, Cf, rho_l, rho_g, grav, sigma_t)
    p_hs, _, _, _ = solve(g, BC_PRESSURE, None, np.zeros(g.shape), b_hs, levels, hs_tol, hs_cycles, nu_pre, nu_post, coarse_sweeps, omega)
    qn = (u, v, w)
    qh = qn
    for _ in range(2):
        qt, _ = mom_predictor(g, Cf, qh, qn, rho_l, rho_g, mu_l, mu_g, dt, vbc)
        qt = mom_forcing(g, Cf, p_hs, p_nh, BC_PRESSURE, grav, st, rho_l, rho_g, dt, qt)
        qh = tuple(0.5 * (a + b) for a, b in zip(qn, qt))
    k = k_from_vof(Cf, rho_l, rho_g)
    b = pressure_rhs(g, qt[0], qt[1], qt[2], dt, vbc)
    dp, cycles, rel, _ = solve(g, BC_PRESSURE, k, np.zeros(g.shape), b, levels, tol, max_cycles, nu_pre, nu_post, coarse_sweeps, omega)
    un, vn, wn = project_velocity(g, BC_PRESSURE, dp, k, dt, qt[0], qt[1], qt[2])
    _, Cn = vof_residual(g, Cf, un, vn, wn, dt)
    return Cn, un, vn, wn, p_hs, (np.zeros(g.shape) if p_nh is None else _f64(p_nh)) + dp, cycles, rel
