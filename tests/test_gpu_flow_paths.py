"""The explicit stages have two kernel families with the same arithmetic: flow_tma.cuh (inputs staged by TMA; the fp32 vector path)
and flow_march.cuh (plain loads; everything else).  Parity with the oracle is tested through whichever one a call selects
(tests/test_gpu_flow.py); here the two are compared with EACH OTHER, bit for bit, on 36 shapes the oracle tests do not reach:
single rows and planes, tiles cut by the domain in x, y and z, nx from 4 to 260.  Each family runs in a process of its own."""
import os
import subprocess
import sys

import numpy as np
import pytest

pytestmark = pytest.mark.gpu
HERE = os.path.dirname(os.path.abspath(__file__))


def test_staged_and_plain_load_kernels_agree_bit_for_bit(tmp_path):
    import torch
    if not torch.cuda.is_available():
        pytest.fail("GPU tests need a CUDA device")
    files = []
    for name, env in (("staged", {}), ("plain", {"MG_NO_FLOW_TMA": "1"})):
        f = str(tmp_path / (name + ".npz"))
        e = dict(os.environ); e.pop("MG_NO_FLOW_TMA", None); e.update(env)
        r = subprocess.run([sys.executable, os.path.join(HERE, "_flow_paths_dump.py"), f], env=e, capture_output=True, text=True, timeout=600)
        assert r.returncode == 0, r.stderr[-2000:]
        files.append(np.load(f))
    a, b = files
    assert len(a.files) == len(b.files) == 36 * 28
    for k in a.files:
        assert np.isfinite(a[k]).all(), k
        assert np.array_equal(a[k], b[k]), k
