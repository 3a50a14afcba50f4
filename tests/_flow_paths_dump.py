"""Helper of tests/test_gpu_flow_paths.py: runs the explicit stages on a list of odd shapes and dumps every output to an .npz file.
Run as a script in a process of its own (the choice between the TMA-staged and the plain-load kernels is read once per process from
MG_NO_FLOW_TMA)."""
import sys, os
sys.path.insert(0, os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
import numpy as np, torch
import paper_2401_06755_b200 as mg
rs = np.random.RandomState(12345)
shapes = [(1, 1, 4), (1, 2, 8), (2, 1, 4), (3, 5, 12), (17, 3, 4), (16, 4, 128), (15, 5, 132), (33, 9, 260), (1, 7, 256), (40, 1, 64), (2, 2, 4)]
for _ in range(25):
    shapes.append((int(rs.randint(1, 41)), int(rs.randint(1, 21)), 4 * int(rs.randint(1, 66))))
out = {}
for si, shape in enumerate(shapes):
    nz, ny, nx = shape
    g = torch.Generator(device="cpu"); g.manual_seed(si)
    r = lambda: torch.randn(shape, generator=g).cuda()
    C = torch.rand(shape, generator=g).cuda(); u, v, w, p = r(), r(), r(), r()
    k = (torch.rand(shape, generator=g) + 0.1).cuda()
    h, dt = 0.05, 0.003
    sC, Cn, b = (torch.empty_like(C) for _ in range(3))
    mg.vof_residual(C, u, v, w, h, dt, sC, Cn)
    qt = [torch.empty_like(C) for _ in range(3)]; qh = [torch.empty_like(C) for _ in range(3)]
    mg.mom_predictor(C, (u, v, w), (u * 0.9, v * 1.1, w), h, 1000.0, 1.0, 1e-3, 1e-5, dt, qt, qh)
    vbc = mg.velocity_bc((1, 1, 0, 1, 1, 0))
    qt2 = [torch.empty_like(C) for _ in range(3)]
    mg.mom_predictor_bc(C, (u, v, w), (u, v, w), vbc, h, 1000.0, 1.0, 1e-3, 1e-5, dt, qt2, None)
    mg.pressure_rhs(u, v, w, h, dt, b)
    b2 = torch.empty_like(C); mg.pressure_rhs_bc(u, v, w, vbc, h, dt, b2)
    pu, pv, pw = u.clone(), v.clone(), w.clone()
    mg.project_velocity(p, k, h, (0, 1, 0, 0, 2, 1), dt, pu, pv, pw)
    bh, kap = torch.empty_like(C), torch.empty_like(C)
    F = [torch.empty_like(C) for _ in range(3)]
    mg.hydrostatic_rhs_force(C, h, 1000.0, 1.0, 9.81, 0.0728, bh, kap, F)
    fq = [u.clone(), v.clone(), w.clone()]; fh = [torch.empty_like(C) for _ in range(3)]
    mg.mom_forcing(C, p, bh * 0.01, (0, 1, 0, 0, 0, 1), h, 9.81, F, 1000.0, 1.0, dt, fq, (u, v, w), fh)
    bp = torch.empty_like(C); mg.pressure_rhs_paper(C, u, v, w, h, 1000.0, 1.0, dt, bp)
    torch.cuda.synchronize()
    for name, t in [("sC", sC), ("Cn", Cn), ("b", b), ("b2", b2), ("pu", pu), ("pv", pv), ("pw", pw)] + [("qt%d" % c, qt[c]) for c in range(3)] + [("qh%d" % c, qh[c]) for c in range(3)] + [("qtb%d" % c, qt2[c]) for c in range(3)] + [("bh", bh), ("kap", kap)] + [("F%d" % c, F[c]) for c in range(3)] + [("fq%d" % c, fq[c]) for c in range(3)] + [("fh%d" % c, fh[c]) for c in range(3)] + [("bp", bp)]:
        out["%d_%s" % (si, name)] = t.cpu().numpy()
np.savez(sys.argv[1], **out)
print("wrote", sys.argv[1], len(out), "arrays;", len(shapes), "shapes")
