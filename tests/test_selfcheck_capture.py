"""The one-time self-checks behind CS_ROUTE_AUTO / CS_A1_AUTO must not break a caller's CUDA-graph capture."""
import pytest

torch = pytest.importorskip("torch")

pytestmark = pytest.mark.gpu


def test_selfchecks_stay_out_of_a_stream_capture():
    """The one-time self-checks behind the AUTO routes synchronise the stream; inside a CUDA-graph capture that would
    invalidate the caller's graph.  In a fresh process (nothing checked yet) an AUTO call made during capture must leave
    the capture intact -- it records the routes that need no trust -- and the replayed graph must give the same
    histogram as the eager call.  Runs in a subprocess because the check's state is per process."""
    import subprocess
    import sys
    code = r"""
import numpy as np, torch
from paper_1805_04463_b200 import api, inputs as inp
torch.cuda.set_device(0)
N = 1500
d = torch.from_numpy(inp.sprinkle(inp.GEOM_MINK_CONE, 4, N, 5)).cuda()
bits, bitsT = api.causal_matrix(d, inp.GEOM_MINK_CONE, route=api.A1_FMA)
want = api.interval_hist(bits, bitsT, N, route=api.ROUTE_POPC)
ws = torch.empty(api.interval_hist_workspace(N), dtype=torch.uint8, device="cuda")
hist = torch.zeros(N - 1, dtype=torch.int64, device="cuda")
lib = api.load()
torch.cuda.synchronize()
g = torch.cuda.CUDAGraph()
with torch.cuda.graph(g):
    st = torch.cuda.current_stream().cuda_stream
    rc = lib.cs_interval_hist(bits.data_ptr(), bitsT.data_ptr(), N, -1, hist.data_ptr(), None, ws.data_ptr(), ws.numel(), st)
    assert rc == 0, (rc, lib.cs_last_cuda_error())
    assert lib.cs_a2_tensor_selfcheck(st) == 0          # asked during capture: not run, not cached
hist.fill_(-1)
g.replay(); torch.cuda.synchronize()
assert torch.equal(hist, want), "replayed graph differs"
assert api.a2_tensor_selfcheck() is True                # outside the capture the check runs and passes
assert torch.equal(api.interval_hist(bits, bitsT, N), want)
print("capture ok")
"""
    import os
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    r = subprocess.run([sys.executable, "-c", code], cwd=root, capture_output=True, text=True, timeout=300)
    assert r.returncode == 0 and "capture ok" in r.stdout, r.stdout + r.stderr
