"""Thin Python binding of libcausalset.so (include/causalset.h): argument marshalling only.

Every function has the name of the C entry point without the `cs_` prefix and
takes/returns torch CUDA tensors (torch is used for device memory and streams
only).  There is no CPU fallback: if the library is missing, or a call returns
an error status, a RuntimeError is raised.

    bits, bitsT = causal_matrix(coords, geometry)        # a1
    hist        = interval_hist(bits, bitsT, N, kmax)    # a2  (Alg. 19/20)
    S           = bd_action(hist, N, dim)                # a3  (Eq. 4.10-4.12)
"""
from __future__ import annotations

import ctypes
import os

import torch

GEOM_MINK2_LIGHTCONE = 0
GEOM_MINK_CONE = 1
GEOM_DS2_SLAB = 2

GEOM_FLRW_POLAR = 3   # include/causalset.h
GEOM_DS4_SPHERICAL = 4
ROUTE_AUTO = 0
ROUTE_POPC = 1
ROUTE_TENSOR = 2
ROUTE_TENSOR_FP4 = 3
ROUTE_TENSOR_PAIR = 4
A1_AUTO = 0           # cs_a1_route
A1_FMA = 1
A1_TENSOR = 2

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libcausalset.so")       # the in-tree build, nothing else
HEADER_PATH = os.path.join(os.path.dirname(_HERE), "include", "causalset.h")

_i64 = ctypes.c_int64
_p = ctypes.c_void_p
_int = ctypes.c_int
_sz = ctypes.c_size_t

_SIGNATURES = {
    "cs_version": (ctypes.c_char_p, []),
    "cs_status_string": (ctypes.c_char_p, [_int]),
    "cs_last_cuda_error": (ctypes.c_char_p, []),
    "cs_row_stride_words": (_i64, [_i64]),
    "cs_causal_matrix": (_int, [_p, _i64, _int, _int, _p, _p, _p]),
    "cs_causal_matrix_batched": (_int, [_p, _i64, _i64, _int, _int, _p, _p, _p]),
    "cs_causal_matrix_workspace": (_sz, [_i64, _i64, _int, _int, _int]),
    "cs_default_a1_route": (_int, [_i64, _i64, _int, _int]),
    "cs_causal_matrix_ex": (_int, [_p, _i64, _i64, _int, _int, _int, _p, _p, _p, _sz, _p]),
    "cs_a1_tensor_selfcheck": (_int, [_p]),
    "cs_a2_tensor_selfcheck": (_int, [_p]),
    "cs_a1_tensor_probe": (_int, [_p, _i64, _int, _p, _p, _p, _sz, _p, _p]),
    "cs_transpose_bits": (_int, [_p, _i64, _p, _p]),
    "cs_degrees": (_int, [_p, _p, _i64, _p, _p, _p]),
    "cs_relation_stats": (_int, [_p, _i64, _p, _p]),
    "cs_interval_hist_workspace": (_sz, [_i64, _i64, _int, _int]),
    "cs_interval_hist": (_int, [_p, _p, _i64, _i64, _p, _p, _p, _sz, _p]),
    "cs_interval_hist_ex": (_int, [_p, _p, _i64, _i64, _i64, _i64, _int, _p, _p, _p, _sz, _p]),
    "cs_interval_hist_stats": (_int, [_p, _p, _p]),
    "cs_interval_hist_static_max_n": (_i64, []),
    "cs_interval_hist_static": (_int, [_p, _p, _i64, _i64, _p, _p, _p]),
    "cs_interval_hist_batched_workspace": (_sz, [_i64, _i64, _int]),
    "cs_interval_hist_batched": (_int, [_p, _p, _i64, _i64, _i64, _int, _p, _p, _sz, _p]),
    "cs_default_route": (_int, [_i64]),
    "cs_bd_action": (_int, [_p, _i64, _i64, _int, _p, _p, _p]),
    "cs_poset_workspace": (_sz, [_i64]),
    "cs_chain_heights": (_int, [_p, _p, _i64, _i64, _p, _p, _p, _sz, _p]),
    "cs_greedy_antichain": (_int, [_p, _p, _i64, _i64, _p, _p, _p, _sz, _p]),
    "cs_smeared_action": (_int, [_p, _i64, _i64, _int, ctypes.c_double, _p, _p]),
    "cs_bd_action_batched_workspace": (_sz, [_i64, _i64]),
    "cs_bd_action_batched": (_int, [_p, _i64, _i64, _int, _int, _p, _p, _p, _sz, _p]),
    "cs_bd_action_batched_host_workspace": (_sz, [_i64, _i64, _int]),
    "cs_bd_action_batched_host": (_int, [_p, _i64, _i64, _int, _int, _p, _p, _p, _sz, _p]),
    "cs_action_host_workspace": (_sz, [_i64, _i64]),
    "cs_action_host": (_int, [_p, _i64, _int, _int, _i64, _p, _p, _p, _sz, _p]),
    "cs_launch_count": (_i64, []),
    "cs_peak_probe": (_int, [_int, _i64, _p, _sz, _p, _p]),
}

_lib = None


def load() -> ctypes.CDLL:
    """Load libcausalset.so; raises if it has not been built (no fallback)."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise RuntimeError(
                "libcausalset.so is missing (%s): build it with `python -m paper_1805_04463_b200.build`; "
                "there is no CPU fallback" % LIB_PATH)
        lib = ctypes.CDLL(LIB_PATH)
        for name, (res, args) in _SIGNATURES.items():
            fn = getattr(lib, name)
            fn.restype = res
            fn.argtypes = args
        _lib = lib
    return _lib


def _check(rc: int, what: str):
    if rc != 0:
        lib = load()
        msg = lib.cs_status_string(rc).decode()
        cuda = lib.cs_last_cuda_error().decode()
        raise RuntimeError("%s failed: %s (%d)%s" % (what, msg, rc, (" -- " + cuda) if cuda else ""))


def _stream() -> int:
    return torch.cuda.current_stream().cuda_stream


def _dptr(t) -> int:
    return 0 if t is None else t.data_ptr()


def _need_cuda(t: torch.Tensor, dtype, name: str):
    if not (isinstance(t, torch.Tensor) and t.is_cuda and t.dtype == dtype and t.is_contiguous()):
        raise TypeError("%s must be a contiguous CUDA tensor of dtype %s" % (name, dtype))


def version() -> str:
    return load().cs_version().decode()


def row_stride_words(N: int) -> int:
    return int(load().cs_row_stride_words(N))


def launch_count() -> int:
    return int(load().cs_launch_count())


def default_route(N: int) -> int:
    return int(load().cs_default_route(N))


PEAK_KINDS = {"mxf4_pair": 0, "i8": 1, "popc": 2, "dfma": 3, "ffma": 4, "ffma2": 5, "hbm_write": 6, "hbm_copy": 7,
              "tmem_ld4": 8, "tmem_ld8": 9, "mxf4_pair_n128": 10, "mxf4_pair_n128_dep": 11}


def peak_probe(kind: str, iters: int, workspace: torch.Tensor):
    """-> (units, seconds, units per clock per SM) of one peak probe (include/causalset.h, cs_peak_kind)."""
    out = (ctypes.c_double * 3)()
    _check(load().cs_peak_probe(PEAK_KINDS[kind], iters, _dptr(workspace), workspace.numel(), ctypes.addressof(out),
                                _stream()), "cs_peak_probe")
    return float(out[0]), float(out[1]), float(out[2])


def causal_matrix_workspace(B: int, N: int, dim: int, geometry: int, route: int = A1_AUTO) -> int:
    return int(load().cs_causal_matrix_workspace(B, N, dim, geometry, route))


def default_a1_route(B: int, N: int, dim: int, geometry: int) -> int:
    return int(load().cs_default_a1_route(B, N, dim, geometry))


def causal_matrix(coords: torch.Tensor, geometry: int, want_transpose: bool = True, route: int = A1_AUTO,
                  workspace: torch.Tensor | None = None):
    """coords [N][dim] fp64 (CUDA, time-sorted) -> (bits, bitsT) int64 tensors [N][stride]
    holding the uint64 bit rows (bitsT is None if want_transpose is False)."""
    _need_cuda(coords, torch.float64, "coords")
    N, dim = coords.shape
    stride = row_stride_words(N)
    bits = torch.empty((N, stride), dtype=torch.int64, device=coords.device)
    bitsT = torch.empty((N, stride), dtype=torch.int64, device=coords.device) if want_transpose else None
    _check(load().cs_causal_matrix_ex(_dptr(coords), 1, N, dim, geometry, route, _dptr(bits), _dptr(bitsT),
                                      _dptr(workspace), workspace.numel() if workspace is not None else 0, _stream()),
           "cs_causal_matrix_ex")
    return bits, bitsT


def causal_matrix_batched(coords: torch.Tensor, geometry: int, want_transpose: bool = True, route: int = A1_AUTO,
                          workspace: torch.Tensor | None = None):
    _need_cuda(coords, torch.float64, "coords")
    B, N, dim = coords.shape
    stride = row_stride_words(N)
    bits = torch.empty((B, N, stride), dtype=torch.int64, device=coords.device)
    bitsT = torch.empty((B, N, stride), dtype=torch.int64, device=coords.device) if want_transpose else None
    _check(load().cs_causal_matrix_ex(_dptr(coords), B, N, dim, geometry, route, _dptr(bits), _dptr(bitsT),
                                      _dptr(workspace), workspace.numel() if workspace is not None else 0, _stream()),
           "cs_causal_matrix_ex")
    return bits, bitsT


def a1_tensor_selfcheck() -> bool:
    """True if this device's tensor cores accumulate like the model the tensor a1 route's error band assumes."""
    rc = load().cs_a1_tensor_selfcheck(_stream())
    if rc < 0:
        _check(rc, "cs_a1_tensor_selfcheck")
    return rc == 1


def a2_tensor_selfcheck() -> bool:
    """True if this device's tensor cores add subnormal fp32 partial sums exactly, which the tensor a2 route rests on."""
    rc = load().cs_a2_tensor_selfcheck(_stream())
    if rc < 0:
        _check(rc, "cs_a2_tensor_selfcheck")
    return rc == 1


def a1_tensor_probe(coords: torch.Tensor):
    """CS_A1_TENSOR on one flat-cone causet (dim 4 or 5) with its counters on ->
    (bits, bitsT, {"max_err_u", "max_acc_err_u", "max_err_over_margin", "rows_fp64", "rows_total"})."""
    _need_cuda(coords, torch.float64, "coords")
    N, dim = coords.shape
    stride = row_stride_words(N)
    bits = torch.empty((N, stride), dtype=torch.int64, device=coords.device)
    bitsT = torch.empty((N, stride), dtype=torch.int64, device=coords.device)
    ws = _workspace(causal_matrix_workspace(1, N, dim, GEOM_MINK_CONE, A1_TENSOR), coords.device)
    out = (ctypes.c_double * 5)()
    _check(load().cs_a1_tensor_probe(_dptr(coords), N, dim, _dptr(bits), _dptr(bitsT), _dptr(ws), ws.numel(),
                                     ctypes.addressof(out), _stream()), "cs_a1_tensor_probe")
    return bits, bitsT, {"max_err_u": float(out[0]), "rows_fp64": int(out[1]), "rows_total": int(out[2]),
                         "max_err_over_margin": float(out[3]), "max_acc_err_u": float(out[4])}


def transpose_bits(bits: torch.Tensor, N: int) -> torch.Tensor:
    _need_cuda(bits, torch.int64, "bits")
    out = torch.empty_like(bits)
    _check(load().cs_transpose_bits(_dptr(bits), N, _dptr(out), _stream()), "cs_transpose_bits")
    return out


def relation_stats(bits: torch.Tensor, N: int) -> torch.Tensor:
    """-> int64[2] CUDA tensor {R, W_alg}."""
    _need_cuda(bits, torch.int64, "bits")
    out = torch.empty(2, dtype=torch.int64, device=bits.device)
    _check(load().cs_relation_stats(_dptr(bits), N, _dptr(out), _stream()), "cs_relation_stats")
    return out


def clamp_kmax(N: int, kmax: int) -> int:
    top = max(N - 2, 0)
    return top if (kmax < 0 or kmax > top) else kmax


def interval_hist_workspace(N: int, kmax: int = -1, have_bitsT: bool = True, route: int = ROUTE_AUTO) -> int:
    return int(load().cs_interval_hist_workspace(N, kmax, int(have_bitsT), route))


def _workspace(nbytes: int, device) -> torch.Tensor:
    return torch.empty(max(nbytes, 256), dtype=torch.uint8, device=device)


def interval_hist(bits: torch.Tensor, bitsT, N: int, kmax: int = -1, route: int = ROUTE_AUTO,
                  row_begin: int = 0, row_end: int | None = None, workspace: torch.Tensor | None = None,
                  return_relations: bool = False):
    """-> hist int64[kmax+1] (CUDA); with return_relations also int64[1] n_relations."""
    _need_cuda(bits, torch.int64, "bits")
    if bitsT is not None:
        _need_cuda(bitsT, torch.int64, "bitsT")
    k = clamp_kmax(N, kmax)
    hist = torch.empty(k + 1, dtype=torch.int64, device=bits.device)
    nrel = torch.empty(1, dtype=torch.int64, device=bits.device) if return_relations else None
    need = interval_hist_workspace(N, kmax, bitsT is not None, route)
    ws = workspace if workspace is not None else _workspace(need, bits.device)
    row_end = N if row_end is None else row_end
    _check(load().cs_interval_hist_ex(_dptr(bits), _dptr(bitsT), N, kmax, row_begin, row_end, route,
                                      _dptr(hist), _dptr(nrel), _dptr(ws), ws.numel(), _stream()),
           "cs_interval_hist_ex")
    return (hist, nrel) if return_relations else hist


def interval_hist_static_max_n() -> int:
    return int(load().cs_interval_hist_static_max_n())


def interval_hist_static(bits: torch.Tensor, bitsT, N: int, kmax: int = -1, hist: torch.Tensor | None = None,
                         return_relations: bool = False):
    """a2 through cs_interval_hist_static: for callers that cannot allocate device memory (inside an allocator
    hook, under a fixed memory budget, plugins that only get their buffers).  The library's scratch is a static
    device array, so no workspace is passed and nothing is allocated by the library; N <= interval_hist_static_max_n().
    Pass `hist` (int64[kmax+1] after clamping) to keep this wrapper from allocating the output as well.
    Calls share the one array per device: do not let two of them overlap on the GPU.
    -> hist int64[kmax+1] (CUDA); with return_relations also int64[1] n_relations."""
    _need_cuda(bits, torch.int64, "bits")
    if bitsT is not None:
        _need_cuda(bitsT, torch.int64, "bitsT")
    k = clamp_kmax(N, kmax)
    if hist is None:
        hist = torch.empty(k + 1, dtype=torch.int64, device=bits.device)
    else:
        _need_cuda(hist, torch.int64, "hist")
        if hist.numel() < k + 1:
            raise ValueError("hist needs %d entries" % (k + 1))
    nrel = torch.empty(1, dtype=torch.int64, device=bits.device) if return_relations else None
    _check(load().cs_interval_hist_static(_dptr(bits), _dptr(bitsT), N, kmax, _dptr(hist), _dptr(nrel), _stream()),
           "cs_interval_hist_static")
    return (hist, nrel) if return_relations else hist


def interval_hist_stats(workspace: torch.Tensor):
    """-> (stages_executed, stages_total, blocks_empty, blocks_examined) of the last a2 call on `workspace`."""
    out = (ctypes.c_int64 * 4)()
    _check(load().cs_interval_hist_stats(_dptr(workspace), ctypes.addressof(out), _stream()), "cs_interval_hist_stats")
    return tuple(int(x) for x in out)


def interval_hist_batched(bits: torch.Tensor, bitsT: torch.Tensor, N: int, kmax: int = -1,
                          route: int = ROUTE_AUTO, workspace: torch.Tensor | None = None) -> torch.Tensor:
    """bits, bitsT [B][N][stride] -> hist int64[B][kmax+1] (CUDA), one launch for all causets."""
    _need_cuda(bits, torch.int64, "bits")
    _need_cuda(bitsT, torch.int64, "bitsT")
    B = bits.shape[0]
    k = clamp_kmax(N, kmax)
    hist = torch.empty((B, k + 1), dtype=torch.int64, device=bits.device)
    need = int(load().cs_interval_hist_batched_workspace(B, N, route))
    ws = workspace if workspace is not None else _workspace(need, bits.device)
    _check(load().cs_interval_hist_batched(_dptr(bits), _dptr(bitsT), B, N, kmax, route, _dptr(hist),
                                           _dptr(ws), ws.numel(), _stream()), "cs_interval_hist_batched")
    return hist


def bd_action(hist: torch.Tensor, N: int, dim: int, return_bracket: bool = False):
    """-> fp64[1] CUDA tensor (and int64[1] bracket)."""
    _need_cuda(hist, torch.int64, "hist")
    action = torch.empty(1, dtype=torch.float64, device=hist.device)
    bracket = torch.empty(1, dtype=torch.int64, device=hist.device) if return_bracket else None
    _check(load().cs_bd_action(_dptr(hist), hist.numel() - 1, N, dim, _dptr(action), _dptr(bracket), _stream()),
           "cs_bd_action")
    return (action, bracket) if return_bracket else action


def degrees(bits: torch.Tensor, bitsT: torch.Tensor, N: int):
    """-> (outdeg, indeg) int64[N] on the device."""
    _need_cuda(bits, torch.int64, "bits")
    _need_cuda(bitsT, torch.int64, "bitsT")
    outdeg = torch.empty(N, dtype=torch.int64, device=bits.device)
    indeg = torch.empty(N, dtype=torch.int64, device=bits.device)
    _check(load().cs_degrees(_dptr(bits), _dptr(bitsT), N, _dptr(outdeg), _dptr(indeg), _stream()), "cs_degrees")
    return outdeg, indeg


def chain_heights(bits: torch.Tensor, bitsT: torch.Tensor, N: int, source: int = -1):
    """-> (height int32[N], longest int64[1]) on the device: elements of the longest chain ending at each
    element (starting at `source` if >= 0); Algorithm 11 for the pair (source, j) is height[j] - 1."""
    _need_cuda(bits, torch.int64, "bits")
    _need_cuda(bitsT, torch.int64, "bitsT")
    height = torch.empty(N, dtype=torch.int32, device=bits.device)
    longest = torch.empty(1, dtype=torch.int64, device=bits.device)
    ws = _workspace(int(load().cs_poset_workspace(N)), bits.device)
    _check(load().cs_chain_heights(_dptr(bits), _dptr(bitsT), N, source, _dptr(height), _dptr(longest),
                                   _dptr(ws), ws.numel(), _stream()), "cs_chain_heights")
    return height, longest


def greedy_antichain(bits: torch.Tensor, bitsT: torch.Tensor, N: int, seed: int):
    """Algorithm 13 -> (member int64[stride] holding the uint64 bitset, size int64[1]) on the device."""
    _need_cuda(bits, torch.int64, "bits")
    _need_cuda(bitsT, torch.int64, "bitsT")
    member = torch.empty(row_stride_words(N), dtype=torch.int64, device=bits.device)
    size = torch.empty(1, dtype=torch.int64, device=bits.device)
    ws = _workspace(int(load().cs_poset_workspace(N)), bits.device)
    _check(load().cs_greedy_antichain(_dptr(bits), _dptr(bitsT), N, seed, _dptr(member), _dptr(size),
                                      _dptr(ws), ws.numel(), _stream()), "cs_greedy_antichain")
    return member, size


def smeared_action(hist: torch.Tensor, N: int, dim: int, eps: float) -> torch.Tensor:
    """Smeared action S_eps (Eq. 4.13-4.18) from the full histogram -> fp64[1] CUDA tensor."""
    _need_cuda(hist, torch.int64, "hist")
    action = torch.empty(1, dtype=torch.float64, device=hist.device)
    _check(load().cs_smeared_action(_dptr(hist), hist.numel() - 1, N, dim, float(eps), _dptr(action), _stream()),
           "cs_smeared_action")
    return action


def bd_action_batched_workspace(B: int, N: int) -> int:
    return int(load().cs_bd_action_batched_workspace(B, N))


def bd_action_batched(coords: torch.Tensor, geometry: int, workspace: torch.Tensor | None = None,
                      return_hist4: bool = False):
    """coords [B][N][dim] -> actions fp64[B] (and hist4 int64[B][4])."""
    _need_cuda(coords, torch.float64, "coords")
    B, N, dim = coords.shape
    actions = torch.empty(B, dtype=torch.float64, device=coords.device)
    hist4 = torch.empty((B, 4), dtype=torch.int64, device=coords.device) if return_hist4 else None
    ws = workspace if workspace is not None else _workspace(bd_action_batched_workspace(B, N), coords.device)
    _check(load().cs_bd_action_batched(_dptr(coords), B, N, dim, geometry, _dptr(actions), _dptr(hist4),
                                       _dptr(ws), ws.numel(), _stream()), "cs_bd_action_batched")
    return (actions, hist4) if return_hist4 else actions


def bd_action_batched_host(coords_host: torch.Tensor, geometry: int, workspace: torch.Tensor | None = None,
                           actions_host: torch.Tensor | None = None, hist4_host: torch.Tensor | None = None,
                           device="cuda"):
    """Ensemble end to end from HOST buffers (pinned for overlap): coords [B][N][dim] -> (actions_host fp64[B],
    hist4_host int64[B][4]); H2D copies overlap the kernels chunk by chunk."""
    if coords_host.is_cuda or coords_host.dtype != torch.float64 or not coords_host.is_contiguous():
        raise TypeError("coords_host must be a contiguous CPU float64 tensor")
    B, N, dim = coords_host.shape
    if actions_host is None:
        actions_host = torch.empty(B, dtype=torch.float64).pin_memory()
    if hist4_host is None:
        hist4_host = torch.empty((B, 4), dtype=torch.int64).pin_memory()
    need = int(load().cs_bd_action_batched_host_workspace(B, N, dim))
    ws = workspace if workspace is not None else _workspace(need, device)
    _check(load().cs_bd_action_batched_host(coords_host.data_ptr(), B, N, dim, geometry, actions_host.data_ptr(),
                                            hist4_host.data_ptr(), _dptr(ws), ws.numel(), _stream()),
           "cs_bd_action_batched_host")
    return actions_host, hist4_host


def action_host_workspace(N: int, kmax: int = -1) -> int:
    return int(load().cs_action_host_workspace(N, kmax))


def action_host(coords_host: torch.Tensor, geometry: int, kmax: int = -1, workspace: torch.Tensor | None = None,
                hist_host: torch.Tensor | None = None, action_host_out: torch.Tensor | None = None,
                device="cuda"):
    """End to end from HOST buffers (pinned preferred): -> (hist_host int64[kmax+1], action_host fp64[1])."""
    if coords_host.is_cuda or coords_host.dtype != torch.float64 or not coords_host.is_contiguous():
        raise TypeError("coords_host must be a contiguous CPU float64 tensor")
    N, dim = coords_host.shape
    k = clamp_kmax(N, kmax)
    if hist_host is None:
        hist_host = torch.empty(k + 1, dtype=torch.int64).pin_memory()
    if action_host_out is None:
        action_host_out = torch.empty(1, dtype=torch.float64).pin_memory()
    ws = workspace if workspace is not None else _workspace(action_host_workspace(N, kmax), device)
    _check(load().cs_action_host(coords_host.data_ptr(), N, dim, geometry, kmax, hist_host.data_ptr(),
                                 action_host_out.data_ptr(), _dptr(ws), ws.numel(), _stream()), "cs_action_host")
    return hist_host, action_host_out
