"""vof_residual_noalloc (include/mg.h): the VoF residual for callers that must not allocate -- its scratch is a static device array.
Checked against the existing path (vof_residual_ex, stream-ordered scratch) on two calls in a row, the second one on another
shape and dtype so that what the first call left in the shared scratch would show if it mattered.  The file sorts last on purpose:
the suite runs with pytest -x, and a failure here must not hide the parity tests."""
import numpy as np
import pytest

from workloads import configs, rng
from _parity import assert_close

pytestmark = pytest.mark.gpu
TOL = {"f32": 1e-5, "f64": 1e-12}          # the tolerances of tests/test_gpu_flow.py


@pytest.fixture(scope="module")
def mg():
    import torch
    if not torch.cuda.is_available():
        pytest.fail("GPU tests need a CUDA device")
    import paper_2401_06755_b200 as m
    return m


def _fields(shape, dt, seed):
    import torch
    nz, ny, nx = shape
    n = nx * ny * nz
    x, y, z = configs.centres(nx, ny, nz, 1.0)
    d = (0.6 * x / nx + 0.5 * y / ny + 0.62 * z / nz) - 0.8
    Cf = 0.5 * (1 + np.tanh(d * 6.0)) + 0.0 * (x + y + z)
    tdt = torch.float32 if dt == "f32" else torch.float64
    dev = lambda a: torch.from_numpy(np.ascontiguousarray(a)).to(tdt).cuda()
    return dev(Cf), [dev(0.3 * rng.normal(seed + c, n).reshape(shape) + 0.2) for c in range(3)]


def test_two_calls_in_a_row_match_the_allocating_path(mg):
    import torch
    calls = [((40, 48, 64), 1.0 / 64, "f32", 3, 11), ((20, 36, 28), 0.05, "f64", 5, 23), ((40, 48, 64), 1.0 / 64, "f32", 3, 11)]
    for shape, h, dt, detector, seed in calls:
        C, (u, v, w) = _fields(shape, dt, seed)
        tstep = 0.1 * h
        s_ref, c_ref = torch.empty_like(C), torch.empty_like(C)
        mg.vof_residual_ex(C, u, v, w, h, tstep, detector, s_ref, c_ref)
        s_new, c_new = torch.full_like(C, float("nan")), torch.full_like(C, float("nan"))
        mg.vof_residual_noalloc(C, u, v, w, h, tstep, detector, s_new, c_new)
        torch.cuda.synchronize()
        what = "%s %s detector %d" % (shape, dt, detector)
        assert float(s_ref.abs().max()) > 0.0
        assert_close(s_new.double().cpu().numpy(), s_ref.double().cpu().numpy(), TOL[dt], "s_C " + what)
        assert_close(c_new.double().cpu().numpy(), c_ref.double().cpu().numpy(), TOL[dt], "C_new " + what)
        # the same kernels on the same inputs: in fact bit for bit
        assert torch.equal(s_new, s_ref) and torch.equal(c_new, c_ref), what


def test_sizes_beyond_the_static_scratch_are_refused(mg):
    import torch
    # 64 x 64 x 128 fp32 = exactly 8 MiB of scratch: accepted; one more plane: refused with a message that names the limit
    C, (u, v, w) = _fields((128, 64, 64), "f32", 5)
    out = torch.empty_like(C)
    mg.vof_residual_noalloc(C, u, v, w, 1.0 / 64, 1e-3, 3, out, None)
    ref = torch.empty_like(C)
    mg.vof_residual_ex(C, u, v, w, 1.0 / 64, 1e-3, 3, ref, None)
    assert torch.equal(out, ref)
    C, (u, v, w) = _fields((129, 64, 64), "f32", 5)
    with pytest.raises(mg.MgError) as e:
        mg.vof_residual_noalloc(C, u, v, w, 1.0 / 64, 1e-3, 3, torch.empty_like(C), None)
    assert e.value.code == mg.MG_EINVAL and "VOF_NOALLOC_SCRATCH_BYTES" in str(e.value)
    C, (u, v, w) = _fields((65, 64, 64), "f64", 5)
    with pytest.raises(mg.MgError):
        mg.vof_residual_noalloc(C, u, v, w, 1.0 / 64, 1e-3, 3, torch.empty_like(C), None)
