"""GPU parity beyond BASELINE.json's sizes: 1024 x 1024 x 512 (5.4e8 points, 2 GiB per fp32 field, so byte offsets pass 2^31 and
element offsets 2^29) -- a size the oracle cannot run in a test -- checked on EVERY point through a reflection identity.

Mirroring a problem across a Neumann face (ghost = mirror value) gives a problem on the doubled domain whose operator,
Jacobi sweep, restriction, prolongation and coarsest sweeps all commute with the reflection: every point of the mirrored grid sees
exactly the neighbour values its mirror image sees.  So with the same number of levels (the big grid's coarsest level is the small
one's mirrored too) the V-cycle of the mirrored problem is the mirrored V-cycle of the small problem, and the oracle's 256^3
result checks the 1024 x 1024 x 512 GPU result block by block (16 x and y blocks, 2 z blocks, each plain or flipped).  Across the
bottom face the mirror turns the z pair (Neumann, Dirichlet) into (Dirichlet, Dirichlet).  In fp32 the two differ only by the
order in which a point adds its left / right neighbours."""
import numpy as np
import pytest

from workloads import configs
from test_gpu_mg import TOL, as_f64, make_solver, mg, quantise, to_dev  # noqa: F401
from _parity import MAXABS_FACTOR

pytestmark = pytest.mark.gpu
N, D = configs.BC_NEUMANN, configs.BC_DIRICHLET
MX, MY = 4, 4          # copies along x and y (plain, flipped, plain, flipped); along z: (flipped, plain)


def _mirror_dev(a):
    """small host field (fp64, already quantised to fp32) -> mirrored device field"""
    import torch
    t = torch.from_numpy(np.ascontiguousarray(a, dtype=np.float32)).cuda()
    t = torch.cat([t.flip(0), t], 0)
    for ax, m in ((1, MY), (2, MX)):
        pair = torch.cat([t, t.flip(ax)], ax)
        t = torch.cat([pair] * (m // 2), ax)
    return t.contiguous()


def _check_blocks(dev, ref, tol, what, factor=MAXABS_FACTOR):
    """every block of the device field against the small reference (fp64), with the bounds of tests/_parity.py"""
    nz, ny, nx = ref.shape
    host = dev.cpu().numpy()
    assert host.shape == (2 * nz, MY * ny, MX * nx)
    num = 0.0
    worst = 0.0
    for bz in range(2):
        for by in range(MY):
            for bx in range(MX):
                blk = host[bz * nz:(bz + 1) * nz, by * ny:(by + 1) * ny, bx * nx:(bx + 1) * nx].astype(np.float64)
                if bz == 0: blk = blk[::-1]
                if by % 2: blk = blk[:, ::-1]
                if bx % 2: blk = blk[:, :, ::-1]
                d = blk - ref
                num += float((d * d).sum())
                worst = max(worst, float(np.abs(d).max()))
    den = 2 * MY * MX * float((ref * ref).sum())
    rel, mx = np.sqrt(num / den), worst / np.abs(ref).max()
    assert rel <= tol and mx <= factor * tol, "%s: rel L2 %.3e (bound %.1e), max-abs %.3e (bound %.1e)" % (what, rel, tol, mx, factor * tol)


def test_mirrored_rising_bubble_1024x1024x512(mg, orc):
    import torch
    w = configs.config3()                                   # 256^3, 7 levels, faces (N, N, N, N, N, D)
    g = orc.grid(w.nx, w.ny, w.nz, w.h)
    alpha = quantise(w.fields["alpha"], "f32")
    b = quantise(orc.pressure_rhs(g, w.fields["u"], w.fields["v"], w.fields["w"], 1.0), "f32")
    k = orc.k_from_vof(alpha, w.rho_l, w.rho_g)
    x0 = quantise(0.01 * b, "f32")
    shape = (2 * w.nz, MY * w.ny, MX * w.nx)
    assert np.prod(shape) * 4 >= 2 ** 31
    s = make_solver(mg, shape, w.h, w.levels, (N, N, N, N, D, D), "f32")
    d_alpha = _mirror_dev(alpha)
    mg.mg_set_coefficient_from_vof(s, d_alpha, w.rho_l, w.rho_g)
    del d_alpha
    db = _mirror_dev(b)
    # a1: residual;  a2: three sweeps;  a3-a6: one V(2,2) cycle from a zero guess and one from a non-zero guess
    dx = _mirror_dev(x0)
    dr = torch.empty_like(dx)
    mg.mg_residual(s, dx, db, dr)
    _check_blocks(dr, orc.residual(g, w.bc, k, x0, b), 5 * TOL["f32"], "residual")
    mg.mg_smooth(s, dx, db, 3)
    _check_blocks(dx, orc.smooth(g, w.bc, k, x0, b, w.omega, 3), 3 * TOL["f32"], "3 sweeps")
    dx.zero_()
    mg.mg_vcycle(s, dx, db)
    x1 = orc.vcycle(g, w.bc, k, np.zeros(w.shape), b, w.levels, 2, 2)
    _check_blocks(dx, x1, 1e-4, "V(2,2) cycle 1")
    # second cycle, restarted from the oracle's iterate.  A plain fp32 cycle from a NON-zero guess forms b - A x in fp32; on this
    # problem (1000:1 coefficient, slowly varying lowest mode) the rounding of that residual, amplified by the coarse levels, leaves
    # a smooth offset of 6e-4 relative L2 (1e-4 of max |x|) against the fp64 oracle -- on 256^3 exactly as here (DESIGN.md
    # section 7; it is what the fp64 defect correction of mg_solve removes).  So the oracle bound is 2e-3 for this step, and the
    # reflection identity is checked tightly against the library's own 256^3 result of the same cycle.
    x1 = quantise(x1, "f32")
    del dx
    dx = _mirror_dev(x1)
    mg.mg_vcycle(s, dx, db)
    _check_blocks(dx, orc.vcycle(g, w.bc, k, x1, b, w.levels, 2, 2), 2e-3, "V(2,2) cycle 2", factor=1.0)
    s_small = make_solver(mg, w.shape, w.h, w.levels, w.bc, "f32")
    mg.mg_set_coefficient_from_vof(s_small, to_dev(alpha, "f32"), w.rho_l, w.rho_g)
    dxs = to_dev(x1, "f32")
    mg.mg_vcycle(s_small, dxs, to_dev(b, "f32"))
    _check_blocks(dx, as_f64(dxs), 2e-5, "reflection identity, cycle 2")
    mg.mg_destroy(s_small)
    mg.mg_destroy(s)
