"""The C-ABI library builds, loads on a CPU-only host and exports every symbol the header declares."""
import ctypes
import re

import pytest

from paper_1805_04463_b200 import api, build


@pytest.fixture(scope="module")
def lib():
    build.build()
    return api.load()


def declared_symbols():
    text = open(api.HEADER_PATH).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(cs_[a-z0-9_]+)\s*\(", text)))


def test_header_symbols_exported(lib):
    names = declared_symbols()
    assert len(names) >= 15
    for n in names:
        assert hasattr(lib, n), "libcausalset.so does not export %s" % n
    # the binding marshals exactly the declared entry points
    assert sorted(api._SIGNATURES) == names


def test_host_only_entry_points(lib):
    assert b"sm_100a" in lib.cs_version()
    assert lib.cs_status_string(0) == b"ok"
    assert lib.cs_status_string(-5).startswith(b"workspace")
    for N, want in [(0, 0), (1, 2), (64, 2), (65, 2), (128, 2), (129, 4), (1000, 16), (65536, 1024), (131072, 2048)]:
        assert lib.cs_row_stride_words(N) == want
    assert lib.cs_launch_count() >= 0


def test_argument_errors_need_no_gpu(lib):
    # argument validation happens before any CUDA call
    assert lib.cs_causal_matrix(None, -1, 2, 0, None, None, None) == -1          # CS_ERR_ARG
    assert lib.cs_causal_matrix(None, 8, 2, 7, None, None, None) == -3           # CS_ERR_GEOM
    assert lib.cs_causal_matrix(None, 8, 3, 0, None, None, None) == -2           # CS_ERR_DIM
    assert lib.cs_causal_matrix(None, 8, 6, 1, None, None, None) == -2           # the flat cone stops at 4+1
    assert lib.cs_causal_matrix(None, 8, 2, 0, None, None, None) == -1           # NULL buffers
    assert lib.cs_causal_matrix(None, 0, 2, 0, None, None, None) == 0            # N = 0 is a no-op
    assert lib.cs_causal_matrix_ex(None, 1, 8, 2, 0, 7, None, None, None, 0, None) == -1     # unknown a1 route
    assert lib.cs_causal_matrix_ex(None, 1, 8, 2, 0, 0, None, None, None, 0, None) == -1     # NULL buffers
    assert lib.cs_causal_matrix_ex(None, 0, 8, 2, 0, 0, None, None, None, 0, None) == 0      # B = 0 is a no-op
    assert lib.cs_causal_matrix_workspace(1, 200, 4, 1, 2) == 0                              # N < 256: no tensor route
    assert lib.cs_causal_matrix_workspace(1, 4096, 4, 1, 1) == 0                             # FMA route: no scratch
    assert lib.cs_causal_matrix_workspace(1, 4096, 4, 1, 2) >= 4096 * (128 + 32)             # operand rows + coordinates
    assert lib.cs_a1_tensor_probe(None, 8, 4, None, None, None, 0, None, None) == -1
    # the probe runs the tensor route, which needs N >= 256 (rows of at least one 32-byte TMA box)
    out5 = (ctypes.c_double * 5)()
    p16 = ctypes.c_void_p(16)
    assert lib.cs_a1_tensor_probe(p16, 255, 4, p16, None, None, 0, ctypes.addressof(out5), None) == -1
    assert lib.cs_a1_tensor_probe(p16, 256, 3, p16, None, None, 0, ctypes.addressof(out5), None) == -2
    assert lib.cs_a1_tensor_probe(p16, 256, 4, p16, None, None, 0, ctypes.addressof(out5), None) == -5   # no workspace
    # the pipeline entry points check geometry, dim and the action's dimension before any chunk is built:
    # the 4+1 cone has a causal matrix but no action (Eq. 4.10-4.12 stop at d = 4)
    assert lib.cs_bd_action_batched(p16, 2, 100, 5, 1, p16, None, None, 0, None) == -2
    assert lib.cs_bd_action_batched(p16, 2, 100, 4, 9, p16, None, None, 0, None) == -3
    assert lib.cs_bd_action_batched(p16, 2, 100, 4, 1, p16, None, None, 0, None) == -5                    # then the workspace
    assert lib.cs_bd_action_batched_host(p16, 2, 100, 5, 1, p16, None, None, 0, None) == -2
    assert lib.cs_bd_action_batched_host(p16, 2, 100, 6, 4, p16, None, None, 0, None) == -2              # dS4 points have 7 numbers
    assert lib.cs_action_host(p16, 100, 5, 1, -1, p16, p16, None, 0, None) == -2
    assert lib.cs_action_host(p16, 100, 2, 7, -1, p16, p16, None, 0, None) == -3
    # CS_A1_AUTO: the tensor route from 128 tiles of 256 x 256 pairs up, never below N = 256 (host logic only)
    assert lib.cs_default_a1_route(1, 65536, 4, 1) == 2 and lib.cs_default_a1_route(1, 131072, 2, 2) == 2
    assert lib.cs_default_a1_route(1, 3840, 4, 1) == 1 and lib.cs_default_a1_route(1, 3841, 4, 1) == 2
    assert lib.cs_default_a1_route(1, 1024, 2, 0) == 1 and lib.cs_default_a1_route(4096, 2048, 4, 1) == 2
    assert lib.cs_default_a1_route(100000, 200, 4, 1) == 1
    w1, w2 = lib.cs_causal_matrix_workspace(1, 4096, 4, 1, 2), lib.cs_causal_matrix_workspace(2, 4096, 4, 1, 2)
    assert 0 < w1 < w2 <= 2 * w1 and w1 % 256 == 0
    assert lib.cs_bd_action_batched_workspace(4096, 2048) <= 512 << 20                       # the ensemble chunk keeps it there
    assert lib.cs_bd_action(None, 3, 10, 4, None, None, None) == -1
    assert lib.cs_interval_hist(None, None, 10, -1, None, None, None, 0, None) == -1
    assert lib.cs_interval_hist_workspace(65536, -1, 1, 1) >= 256
    assert lib.cs_interval_hist_workspace(1024, -1, 0, 1) >= 256 + 1024 * 16 * 8
    # CS_ROUTE_AUTO: the tensor route for 1024 <= N <= 2^21, the bit route outside (host logic)
    assert [lib.cs_default_route(n) for n in (0, 1023, 1024, 65536, 1 << 21, (1 << 21) + 1, 1 << 23)] == [1, 1, 4, 4, 4, 1, 1]
    # the entry point with static scratch refuses what its array cannot hold, before touching the device
    assert lib.cs_interval_hist_static_max_n() == 8192
    assert lib.cs_interval_hist_static(ctypes.c_void_p(16), None, 8193, -1, ctypes.c_void_p(16), None, None) == -7
    assert b"N <= 8192" in lib.cs_last_cuda_error() and b"capacity" in lib.cs_status_string(-7)
    assert lib.cs_interval_hist_static(None, None, 10, -1, None, None, None) == -1


def test_missing_library_fails_loudly(monkeypatch, tmp_path):
    monkeypatch.setattr(api, "_lib", None)
    monkeypatch.setattr(api, "LIB_PATH", str(tmp_path / "nope.so"))
    with pytest.raises(RuntimeError, match="no CPU fallback"):
        api.load()
