"""Thin ctypes binding of libmg_b200.so (include/mg.h).  Argument marshalling only.

Every function has the name and the arguments of its C-ABI entry point; torch tensors are
used for device memory and streams and are passed down as raw device pointers.  Tensors are
contiguous, shape (nz, ny, nx) (x fastest), float32 or float64 matching the solver's dtype.
There is no CPU fallback: if the library cannot be loaded, importing this module raises.
"""
from __future__ import annotations

import ctypes as C
import os

import torch

from . import _build

MG_F32, MG_F64 = 0, 1
MG_BC_NEUMANN, MG_BC_DIRICHLET, MG_BC_DIRICHLET_HALO = 0, 1, 2
MG_OK, MG_NOT_CONVERGED, MG_STAGNATED = 0, 1, 2
MG_EINVAL, MG_ESHAPE, MG_ECUDA, MG_EALLOC = -1, -2, -3, -4

EXPORTS = [
    "mg_create", "mg_destroy", "mg_set_params", "mg_get_params", "mg_set_coefficient",
    "mg_set_coefficient_from_vof", "mg_apply_operator", "mg_smooth", "mg_residual", "mg_vcycle", "mg_solve", "mg_pcg_solve",
    "mg_solve_host", "mg_solve_host_zero", "mg_get_history", "mg_get_history_cycles", "mg_level_info", "mg_vcycle_timed", "mg_launch_count", "mg_set_fused",
    "vof_residual", "mom_predictor", "pressure_rhs", "pressure_rhs_paper", "hydrostatic_rhs", "project_velocity", "flow_time_step", "flow_time_step_pcg", "flow_time_step_paper", "mg_last_error",
    "mom_predictor_bc", "pressure_rhs_bc", "mom_forcing", "hydrostatic_rhs_force", "flow_time_step_full", "flow_time_step_full_ex", "vof_residual_ex", "vof_residual_noalloc",
    "mg_version",
]


class MgGrid(C.Structure):
    _fields_ = [("nx", C.c_int), ("ny", C.c_int), ("nz", C.c_int),
                ("hx", C.c_double), ("hy", C.c_double), ("hz", C.c_double)]


class MgParams(C.Structure):
    _fields_ = [("nu_pre", C.c_int), ("nu_post", C.c_int), ("coarse_sweeps", C.c_int),
                ("sweeps_per_pass", C.c_int), ("omega", C.c_double), ("mixed_precision", C.c_int),
                ("cycles_per_defect", C.c_int)]


class MgError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__("libmg_b200 error %d: %s" % (code, msg))
        self.code = code


def _load():
    # build() is mtime-checked and returns at once when nothing changed: the library that is loaded is never older than
    # csrc/ (a stale .so travelling with a snapshot would otherwise be exercised silently).  If the toolchain is missing
    # the existing library is used and the fact is said aloud.
    try:
        path = _build.build(force=False)
    except Exception as e:  # noqa: BLE001 -- no nvcc on this machine
        path = _build.LIB
        if not os.path.exists(path):
            raise
        import warnings
        warnings.warn("libmg_b200.so could not be checked against csrc/ (%s); loading the existing build" % (str(e).splitlines()[0],))
    lib = C.CDLL(path)
    if any(not hasattr(lib, name) for name in EXPORTS):     # a stale build from before an entry point was added
        del lib
        path = _build.build(force=True)
        lib = C.CDLL(path)
    vp, i, d = C.c_void_p, C.c_int, C.c_double
    pi, pd = C.POINTER(C.c_int), C.POINTER(C.c_double)
    lib.mg_create.argtypes = [C.POINTER(vp), C.POINTER(MgGrid), i, pi, i, vp]
    lib.mg_destroy.argtypes = [vp]; lib.mg_destroy.restype = None
    lib.mg_set_params.argtypes = [vp, C.POINTER(MgParams)]
    lib.mg_get_params.argtypes = [vp, C.POINTER(MgParams)]
    lib.mg_set_coefficient.argtypes = [vp, vp]
    lib.mg_set_coefficient_from_vof.argtypes = [vp, vp, d, d]
    lib.mg_apply_operator.argtypes = [vp, vp, vp]
    lib.mg_smooth.argtypes = [vp, vp, vp, i]
    lib.mg_residual.argtypes = [vp, vp, vp, vp]
    lib.mg_vcycle.argtypes = [vp, vp, vp]
    lib.mg_solve.argtypes = [vp, vp, vp, d, i, pi, pd]
    lib.mg_solve_host.argtypes = [vp, vp, vp, d, i, pi, pd]
    lib.mg_solve_host_zero.argtypes = [vp, vp, vp, d, i, pi, pd]
    lib.mg_pcg_solve.argtypes = [vp, vp, vp, d, i, pi, pd]
    lib.mg_get_history.argtypes = [vp, pd, i]
    lib.mg_get_history_cycles.argtypes = [vp, pi, i]
    lib.mg_level_info.argtypes = [vp, i, pi, pi, pi]; lib.mg_level_info.restype = C.c_longlong
    lib.mg_vcycle_timed.argtypes = [vp, vp, vp, C.POINTER(C.c_float), C.POINTER(C.c_float)]
    lib.mg_launch_count.argtypes = [vp]; lib.mg_launch_count.restype = C.c_longlong
    lib.mg_set_fused.argtypes = [vp, i]
    lib.vof_residual.argtypes = [C.POINTER(MgGrid), i, vp, vp, vp, vp, d, vp, vp, vp]
    lib.vof_residual_ex.argtypes = [C.POINTER(MgGrid), i, vp, vp, vp, vp, d, i, vp, vp, vp]
    lib.vof_residual_noalloc.argtypes = [C.POINTER(MgGrid), i, vp, vp, vp, vp, d, i, vp, vp, vp]
    lib.mom_predictor.argtypes = [C.POINTER(MgGrid), i, vp, C.POINTER(vp), C.POINTER(vp), d, d, d, d, d,
                                  C.POINTER(vp), C.POINTER(vp), vp]
    lib.pressure_rhs.argtypes = [C.POINTER(MgGrid), i, vp, vp, vp, d, vp, vp]
    lib.pressure_rhs_bc.argtypes = [C.POINTER(MgGrid), i, vp, vp, vp, pi, d, vp, vp]
    lib.mom_predictor_bc.argtypes = [C.POINTER(MgGrid), i, vp, C.POINTER(vp), C.POINTER(vp), pi, d, d, d, d, d,
                                     C.POINTER(vp), C.POINTER(vp), vp]
    lib.mom_forcing.argtypes = [C.POINTER(MgGrid), i, vp, vp, vp, pi, d, C.POINTER(vp), d, d, d, C.POINTER(vp), C.POINTER(vp),
                                C.POINTER(vp), vp]
    lib.hydrostatic_rhs_force.argtypes = [C.POINTER(MgGrid), i, vp, d, d, d, d, vp, vp, C.POINTER(vp), vp]
    lib.flow_time_step_full.argtypes = [vp, vp, vp, vp, vp, vp, vp, vp, d, d, d, d, d, d, d, d, i, d, i, pi, pi, pd]
    lib.flow_time_step_full_ex.argtypes = [vp, vp, vp, vp, vp, vp, vp, vp, d, d, d, d, d, d, d, d, i, d, i, pi, i, pi, pd]
    lib.pressure_rhs_paper.argtypes = [C.POINTER(MgGrid), i, vp, vp, vp, vp, d, d, d, vp, vp]
    lib.flow_time_step_paper.argtypes = [vp, vp, vp, vp, vp, vp, d, d, d, d, d, i, i, pd]
    lib.hydrostatic_rhs.argtypes = [C.POINTER(MgGrid), i, vp, d, d, d, d, vp, vp, vp]
    lib.project_velocity.argtypes = [C.POINTER(MgGrid), pi, i, vp, vp, d, vp, vp, vp, vp]
    lib.flow_time_step.argtypes = [vp, vp, vp, vp, vp, vp, d, d, d, d, d, d, i, pi, pd]
    lib.flow_time_step_pcg.argtypes = [vp, vp, vp, vp, vp, vp, d, d, d, d, d, d, i, pi, pd]
    lib.mg_last_error.restype = C.c_char_p
    lib.mg_version.restype = C.c_char_p
    return lib


_lib = _load()


def library_path():
    return _build.LIB


def mg_last_error():
    return _lib.mg_last_error().decode()


def mg_version():
    return _lib.mg_version().decode()


def _check(rc):
    if rc < 0:
        raise MgError(rc, mg_last_error())
    return rc


_TORCH_DTYPE = {MG_F32: torch.float32, MG_F64: torch.float64}


def _dtype_code(t):
    return MG_F32 if t.dtype == torch.float32 else MG_F64


def _dev(t, shape=None, dtype=None, allow_none=False):
    """Device pointer of a contiguous CUDA tensor (marshalling checks only)."""
    if t is None:
        if allow_none:
            return None
        raise ValueError("tensor argument is None")
    if not t.is_cuda or not t.is_contiguous():
        raise ValueError("expected a contiguous CUDA tensor")
    if dtype is not None and t.dtype != dtype:
        raise ValueError("expected dtype %s, got %s" % (dtype, t.dtype))
    if shape is not None and tuple(t.shape) != tuple(shape):
        raise ValueError("expected shape %s, got %s" % (tuple(shape), tuple(t.shape)))
    return C.c_void_p(t.data_ptr())


def _stream_ptr(stream):
    if stream is None:
        stream = torch.cuda.current_stream()
    return C.c_void_p(stream.cuda_stream)


def _grid(nx, ny, nz, hx, hy=None, hz=None):
    return MgGrid(int(nx), int(ny), int(nz), float(hx), float(hx if hy is None else hy), float(hx if hz is None else hz))


class Solver:
    """Handle returned by mg_create; frees the C object when collected."""

    def __init__(self, handle, grid, levels, bc, dtype, stream):
        self.handle, self.grid, self.levels, self.bc, self.dtype, self.stream = handle, grid, levels, tuple(bc), dtype, stream
        self.shape = (grid.nz, grid.ny, grid.nx)
        self.torch_dtype = _TORCH_DTYPE[dtype]

    def close(self):
        if self.handle:
            _lib.mg_destroy(self.handle)
            self.handle = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


def mg_create(grid, levels, bc, dtype=MG_F32, stream=None):
    """grid: MgGrid or (nx, ny, nz, hx[, hy, hz]); bc: 6 codes x-,x+,y-,y+,z-,z+."""
    if not isinstance(grid, MgGrid):
        grid = _grid(*grid)
    if stream is None:
        stream = torch.cuda.current_stream()
    h = C.c_void_p()
    bcarr = (C.c_int * 6)(*[int(b) for b in bc])
    _check(_lib.mg_create(C.byref(h), C.byref(grid), int(levels), bcarr, int(dtype), _stream_ptr(stream)))
    return Solver(h, grid, levels, bc, dtype, stream)


def mg_destroy(s):
    s.close()


def mg_set_params(s, nu_pre=2, nu_post=2, coarse_sweeps=50, sweeps_per_pass=1, omega=2.0 / 3.0, mixed_precision=1,
                  cycles_per_defect=1):
    p = MgParams(int(nu_pre), int(nu_post), int(coarse_sweeps), int(sweeps_per_pass), float(omega), int(mixed_precision),
                 int(cycles_per_defect))
    return _check(_lib.mg_set_params(s.handle, C.byref(p)))


def mg_get_params(s):
    p = MgParams()
    _check(_lib.mg_get_params(s.handle, C.byref(p)))
    return {k: getattr(p, k) for k, _ in MgParams._fields_}


def mg_set_fused(s, fused):
    return _check(_lib.mg_set_fused(s.handle, int(fused)))


def mg_set_coefficient(s, k):
    return _check(_lib.mg_set_coefficient(s.handle, _dev(k, s.shape, s.torch_dtype, allow_none=True)))


def mg_set_coefficient_from_vof(s, alpha, rho_l, rho_g):
    return _check(_lib.mg_set_coefficient_from_vof(s.handle, _dev(alpha, s.shape, s.torch_dtype), float(rho_l), float(rho_g)))


def mg_apply_operator(s, x, y):
    return _check(_lib.mg_apply_operator(s.handle, _dev(x, s.shape, s.torch_dtype), _dev(y, s.shape, s.torch_dtype)))


def mg_residual(s, x, b, r):
    return _check(_lib.mg_residual(s.handle, _dev(x, s.shape, s.torch_dtype), _dev(b, s.shape, s.torch_dtype),
                                   _dev(r, s.shape, s.torch_dtype)))


def mg_smooth(s, x, b, sweeps):
    return _check(_lib.mg_smooth(s.handle, _dev(x, s.shape, s.torch_dtype), _dev(b, s.shape, s.torch_dtype), int(sweeps)))


def mg_vcycle(s, x, b):
    return _check(_lib.mg_vcycle(s.handle, _dev(x, s.shape, s.torch_dtype), _dev(b, s.shape, s.torch_dtype)))


def mg_solve(s, x, b, tol, max_cycles):
    """Returns (status, cycles, relres)."""
    cyc, rel = C.c_int(0), C.c_double(0.0)
    st = _check(_lib.mg_solve(s.handle, _dev(x, s.shape, s.torch_dtype), _dev(b, s.shape, s.torch_dtype), float(tol),
                              int(max_cycles), C.byref(cyc), C.byref(rel)))
    return st, cyc.value, rel.value


def mg_pcg_solve(s, x, b, tol, max_iter):
    """V-cycle-preconditioned CG.  Returns (status, iterations, relres)."""
    it, rel = C.c_int(0), C.c_double(0.0)
    st = _check(_lib.mg_pcg_solve(s.handle, _dev(x, s.shape, s.torch_dtype), _dev(b, s.shape, s.torch_dtype), float(tol),
                                  int(max_iter), C.byref(it), C.byref(rel)))
    return st, it.value, rel.value


def _solve_host(fn, s, x_host, b_host, tol, max_cycles):
    for t in (x_host, b_host):
        if t.is_cuda or not t.is_contiguous() or t.dtype != s.torch_dtype or tuple(t.shape) != s.shape:
            raise ValueError("expected contiguous CPU tensors of the solver's shape and dtype")
    cyc, rel = C.c_int(0), C.c_double(0.0)
    st = _check(fn(s.handle, C.c_void_p(x_host.data_ptr()), C.c_void_p(b_host.data_ptr()), float(tol), int(max_cycles),
                   C.byref(cyc), C.byref(rel)))
    return st, cyc.value, rel.value


def mg_solve_host(s, x_host, b_host, tol, max_cycles):
    """x_host (guess in, solution out), b_host: contiguous CPU tensors (pinned or not).  Returns (status, cycles, relres)."""
    return _solve_host(_lib.mg_solve_host, s, x_host, b_host, tol, max_cycles)


def mg_solve_host_zero(s, x_host, b_host, tol, max_cycles):
    """As mg_solve_host from a zero guess: x_host is output only (not read, not copied to the device)."""
    return _solve_host(_lib.mg_solve_host_zero, s, x_host, b_host, tol, max_cycles)


def mg_get_history(s):
    n = _lib.mg_get_history(s.handle, None, 0)
    buf = (C.c_double * max(n, 1))()
    _lib.mg_get_history(s.handle, buf, n)
    return list(buf[:n])


def mg_get_history_cycles(s):
    """cycles completed when each entry of mg_get_history was taken"""
    n = _lib.mg_get_history_cycles(s.handle, None, 0)
    buf = (C.c_int * max(n, 1))()
    _lib.mg_get_history_cycles(s.handle, buf, n)
    return list(buf[:n])


def mg_level_info(s, level):
    nx, ny, nz = C.c_int(), C.c_int(), C.c_int()
    n = _lib.mg_level_info(s.handle, int(level), C.byref(nx), C.byref(ny), C.byref(nz))
    _check(int(n) if n < 0 else 0)
    return int(n), (nx.value, ny.value, nz.value)


def mg_vcycle_timed(s, x, b):
    """Returns (ms_down[levels], ms_up[levels])."""
    dn = (C.c_float * s.levels)(); up = (C.c_float * s.levels)()
    _check(_lib.mg_vcycle_timed(s.handle, _dev(x, s.shape, s.torch_dtype), _dev(b, s.shape, s.torch_dtype), dn, up))
    return list(dn), list(up)


def mg_launch_count(s):
    return int(_lib.mg_launch_count(s.handle))


def _grid_of(t, h):
    nz, ny, nx = t.shape
    if isinstance(h, (tuple, list)):
        return _grid(nx, ny, nz, *h)
    return _grid(nx, ny, nz, h)


def vof_residual(C_, u, v, w, h, dt, sC_out=None, Cnew_out=None, stream=None):
    g = _grid_of(C_, h)
    sh, dt_ = tuple(C_.shape), C_.dtype
    return _check(_lib.vof_residual(C.byref(g), _dtype_code(C_), _dev(C_), _dev(u, sh, dt_), _dev(v, sh, dt_),
                                    _dev(w, sh, dt_), float(dt), _dev(sC_out, sh, dt_, True), _dev(Cnew_out, sh, dt_, True),
                                    _stream_ptr(stream)))


def vof_residual_ex(C_, u, v, w, h, dt, detector, sC_out=None, Cnew_out=None, stream=None):
    g = _grid_of(C_, h)
    sh, dt_ = tuple(C_.shape), C_.dtype
    return _check(_lib.vof_residual_ex(C.byref(g), _dtype_code(C_), _dev(C_), _dev(u, sh, dt_), _dev(v, sh, dt_),
                                       _dev(w, sh, dt_), float(dt), int(detector), _dev(sC_out, sh, dt_, True),
                                       _dev(Cnew_out, sh, dt_, True), _stream_ptr(stream)))


def vof_residual_noalloc(C_, u, v, w, h, dt, detector=3, sC_out=None, Cnew_out=None, stream=None):
    """vof_residual_ex without any allocation by the library (static device scratch; size limit VOF_NOALLOC_SCRATCH_BYTES of
    include/mg.h, MgError(MG_EINVAL) beyond it).  Calls that overlap on the GPU race on the shared scratch."""
    g = _grid_of(C_, h)
    sh, dt_ = tuple(C_.shape), C_.dtype
    return _check(_lib.vof_residual_noalloc(C.byref(g), _dtype_code(C_), _dev(C_), _dev(u, sh, dt_), _dev(v, sh, dt_),
                                            _dev(w, sh, dt_), float(dt), int(detector), _dev(sC_out, sh, dt_, True),
                                            _dev(Cnew_out, sh, dt_, True), _stream_ptr(stream)))


def _ptr3(ts, sh, dt_, allow_none=False):
    if ts is None:
        if allow_none:
            return None
        raise ValueError("missing tensor triple")
    return (C.c_void_p * 3)(*[_dev(t, sh, dt_).value for t in ts])


def mom_predictor(C_, qh, qn, h, rho_l, rho_g, mu_l, mu_g, dt, qt, qhn=None, stream=None, vbc=None):
    g = _grid_of(C_, h)
    sh, dt_ = tuple(C_.shape), C_.dtype
    return _check(_lib.mom_predictor_bc(C.byref(g), _dtype_code(C_), _dev(C_), _ptr3(qh, sh, dt_), _ptr3(qn, sh, dt_), _vbc(vbc),
                                        float(rho_l), float(rho_g), float(mu_l), float(mu_g), float(dt),
                                        _ptr3(qt, sh, dt_), _ptr3(qhn, sh, dt_, True), _stream_ptr(stream)))


def _vbc(vbc):
    return None if vbc is None else (C.c_int * 18)(*[int(b) for b in vbc])


def velocity_bc(walls=(1, 1, 1, 1, 1, 0)):
    """The 18 halo codes of (u, v, w) for free-slip walls: the wall-normal component is odd about a wall
    (MG_BC_DIRICHLET), everything else is copied (MG_BC_NEUMANN).  Argument marshalling only."""
    return tuple(MG_BC_DIRICHLET if walls[f] and f // 2 == comp else MG_BC_NEUMANN for comp in range(3) for f in range(6))


def pressure_rhs(u, v, w, h, dt, b, stream=None, vbc=None):
    g = _grid_of(u, h)
    sh, dt_ = tuple(u.shape), u.dtype
    return _check(_lib.pressure_rhs_bc(C.byref(g), _dtype_code(u), _dev(u), _dev(v, sh, dt_), _dev(w, sh, dt_), _vbc(vbc), float(dt),
                                       _dev(b, sh, dt_), _stream_ptr(stream)))


def mom_forcing(C_, p_hs, p_nh, pbc, h, grav, force, rho_l, rho_g, dt, qt, qn=None, qhn=None, stream=None):
    """q~ updated in place; p_hs, p_nh, force may be None; qhn (with qn) receives (q_n + q~)/2."""
    g = _grid_of(C_, h)
    sh, dt_ = tuple(C_.shape), C_.dtype
    bcarr = (C.c_int * 6)(*[int(b) for b in pbc])
    return _check(_lib.mom_forcing(C.byref(g), _dtype_code(C_), _dev(C_), _dev(p_hs, sh, dt_, True), _dev(p_nh, sh, dt_, True), bcarr,
                                   float(grav), _ptr3(force, sh, dt_, True), float(rho_l), float(rho_g), float(dt), _ptr3(qt, sh, dt_),
                                   _ptr3(qn, sh, dt_, True), _ptr3(qhn, sh, dt_, True), _stream_ptr(stream)))


def flow_time_step_full(s_hs, s, C_, u, v, w, p_hs, p_nh, rho_l, rho_g, mu_l, mu_g, grav, sigma_t, dt, tol, max_cycles,
                        hs_tol=0.0, hs_cycles=20, walls=(1, 1, 1, 1, 1, 0)):
    """Returns (status, cycles, relres) of the stage-3 solve."""
    cyc, rel = C.c_int(0), C.c_double(0.0)
    sh, dt_ = s.shape, s.torch_dtype
    wl = (C.c_int * 6)(*[int(b) for b in walls])
    st = _check(_lib.flow_time_step_full(s_hs.handle, s.handle, _dev(C_, sh, dt_), _dev(u, sh, dt_), _dev(v, sh, dt_), _dev(w, sh, dt_),
                                         _dev(p_hs, sh, dt_), _dev(p_nh, sh, dt_), float(rho_l), float(rho_g), float(mu_l), float(mu_g),
                                         float(grav), float(sigma_t), float(dt), float(tol), int(max_cycles), float(hs_tol),
                                         int(hs_cycles), wl, C.byref(cyc), C.byref(rel)))
    return st, cyc.value, rel.value


def flow_time_step_full_ex(s_hs, s, C_, u, v, w, p_hs, p_nh, rho_l, rho_g, mu_l, mu_g, grav, sigma_t, dt, tol, max_cycles,
                           hs_tol=0.0, hs_cycles=20, walls=(1, 1, 1, 1, 1, 0), pressure_solver=0):
    """flow_time_step_full with the stage-3 solver chosen: 0 = plain cycles, 1 = V-cycle-preconditioned CG."""
    cyc, rel = C.c_int(0), C.c_double(0.0)
    sh, dt_ = s.shape, s.torch_dtype
    wl = (C.c_int * 6)(*[int(b) for b in walls])
    st = _check(_lib.flow_time_step_full_ex(s_hs.handle, s.handle, _dev(C_, sh, dt_), _dev(u, sh, dt_), _dev(v, sh, dt_), _dev(w, sh, dt_),
                                            _dev(p_hs, sh, dt_), _dev(p_nh, sh, dt_), float(rho_l), float(rho_g), float(mu_l), float(mu_g),
                                            float(grav), float(sigma_t), float(dt), float(tol), int(max_cycles), float(hs_tol),
                                            int(hs_cycles), wl, int(pressure_solver), C.byref(cyc), C.byref(rel)))
    return st, cyc.value, rel.value


def pressure_rhs_paper(C_, u, v, w, h, rho_l, rho_g, dt, b, stream=None):
    g = _grid_of(C_, h)
    sh, dt_ = tuple(C_.shape), C_.dtype
    return _check(_lib.pressure_rhs_paper(C.byref(g), _dtype_code(C_), _dev(C_), _dev(u, sh, dt_), _dev(v, sh, dt_), _dev(w, sh, dt_),
                                          float(rho_l), float(rho_g), float(dt), _dev(b, sh, dt_), _stream_ptr(stream)))


def flow_time_step_paper(s, C_, u, v, w, p, rho_l, rho_g, mu_l, mu_g, dt, cycles=20, passes=2):
    """Returns the relative residual of the last solve."""
    rel = C.c_double(0.0)
    sh, dt_ = s.shape, s.torch_dtype
    _check(_lib.flow_time_step_paper(s.handle, _dev(C_, sh, dt_), _dev(u, sh, dt_), _dev(v, sh, dt_), _dev(w, sh, dt_), _dev(p, sh, dt_),
                                     float(rho_l), float(rho_g), float(mu_l), float(mu_g), float(dt), int(cycles), int(passes),
                                     C.byref(rel)))
    return rel.value


def hydrostatic_rhs(C_, h, rho_l, rho_g, grav, sigma_t, b, kappa_out=None, stream=None, force_out=None):
    g = _grid_of(C_, h)
    sh, dt_ = tuple(C_.shape), C_.dtype
    return _check(_lib.hydrostatic_rhs_force(C.byref(g), _dtype_code(C_), _dev(C_), float(rho_l), float(rho_g), float(grav), float(sigma_t),
                                             _dev(b, sh, dt_), _dev(kappa_out, sh, dt_, True), _ptr3(force_out, sh, dt_, True),
                                             _stream_ptr(stream)))


def project_velocity(p, k, h, bc, dt, u, v, w, stream=None):
    g = _grid_of(p, h)
    sh, dt_ = tuple(p.shape), p.dtype
    bcarr = (C.c_int * 6)(*[int(b) for b in bc])
    return _check(_lib.project_velocity(C.byref(g), bcarr, _dtype_code(p), _dev(p), _dev(k, sh, dt_), float(dt),
                                        _dev(u, sh, dt_), _dev(v, sh, dt_), _dev(w, sh, dt_), _stream_ptr(stream)))


def flow_time_step_pcg(s, C_, u, v, w, p, rho_l, rho_g, mu_l, mu_g, dt, tol, max_iter):
    """Returns (status, iterations, relres)."""
    its, rel = C.c_int(0), C.c_double(0.0)
    sh, dt_ = s.shape, s.torch_dtype
    st = _check(_lib.flow_time_step_pcg(s.handle, _dev(C_, sh, dt_), _dev(u, sh, dt_), _dev(v, sh, dt_), _dev(w, sh, dt_),
                                        _dev(p, sh, dt_), float(rho_l), float(rho_g), float(mu_l), float(mu_g), float(dt),
                                        float(tol), int(max_iter), C.byref(its), C.byref(rel)))
    return st, its.value, rel.value


def flow_time_step(s, C_, u, v, w, p, rho_l, rho_g, mu_l, mu_g, dt, tol, max_cycles):
    """Returns (status, cycles, relres)."""
    cyc, rel = C.c_int(0), C.c_double(0.0)
    sh, dt_ = s.shape, s.torch_dtype
    st = _check(_lib.flow_time_step(s.handle, _dev(C_, sh, dt_), _dev(u, sh, dt_), _dev(v, sh, dt_), _dev(w, sh, dt_),
                                    _dev(p, sh, dt_), float(rho_l), float(rho_g), float(mu_l), float(mu_g), float(dt),
                                    float(tol), int(max_cycles), C.byref(cyc), C.byref(rel)))
    return st, cyc.value, rel.value


def mom_predictor_bc(C_, qh, qn, vbc, h, rho_l, rho_g, mu_l, mu_g, dt, qt, qhn=None, stream=None):
    return mom_predictor(C_, qh, qn, h, rho_l, rho_g, mu_l, mu_g, dt, qt, qhn, stream, vbc)


def pressure_rhs_bc(u, v, w, vbc, h, dt, b, stream=None):
    return pressure_rhs(u, v, w, h, dt, b, stream, vbc)


def hydrostatic_rhs_force(C_, h, rho_l, rho_g, grav, sigma_t, b, kappa_out=None, force_out=None, stream=None):
    return hydrostatic_rhs(C_, h, rho_l, rho_g, grav, sigma_t, b, kappa_out, stream, force_out)
