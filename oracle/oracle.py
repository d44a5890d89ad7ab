"""ctypes loader for oracle/causet_oracle.c (ORACLE -- test infrastructure only).

`build()` compiles the C file with gcc (-O2 -fopenmp -ffp-contract=off, no
-ffast-math, no -march=native so that the .so built on one host runs on
another) into oracle/libcauset_oracle.so.  Everything here is argument
marshalling; the arithmetic lives in the C file, where each function cites
the passage of PAPER.md it follows.
"""
from __future__ import annotations

import ctypes
import os
import subprocess

import numpy as np

GEOM_MINK2_LIGHTCONE = 0
GEOM_MINK_CONE = 1
GEOM_DS2_SLAB = 2
GEOM_FLRW_POLAR = 3
GEOM_DS4_SPHERICAL = 4

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "causet_oracle.c")
_SO = os.path.join(_HERE, "libcauset_oracle.so")
_lib = None

_i64 = ctypes.c_int64
_p = ctypes.c_void_p


def build(force: bool = False) -> str:
    """Compile the oracle library if it is missing or older than its source."""
    if (not force) and os.path.exists(_SO) and os.path.getmtime(_SO) >= os.path.getmtime(_SRC):
        return _SO
    cmd = ["gcc", "-O2", "-std=c11", "-D_GNU_SOURCE", "-fopenmp", "-ffp-contract=off", "-mpopcnt",
           "-fPIC", "-shared", "-o", _SO, _SRC, "-lm"]
    subprocess.run(cmd, check=True)
    return _SO


def _load():
    global _lib
    if _lib is None:
        build()
        lib = ctypes.CDLL(_SO)
        lib.orc_relation.restype = ctypes.c_int
        lib.orc_relation.argtypes = [_p, _p, ctypes.c_int, ctypes.c_int]
        lib.orc_causal_matrix_bytes.restype = ctypes.c_int
        lib.orc_causal_matrix_bytes.argtypes = [_p, _i64, ctypes.c_int, ctypes.c_int, _p]
        lib.orc_causal_matrix_bits.restype = ctypes.c_int
        lib.orc_causal_matrix_bits.argtypes = [_p, _i64, ctypes.c_int, ctypes.c_int, _p, _i64]
        lib.orc_transpose_bits.restype = None
        lib.orc_transpose_bits.argtypes = [_p, _i64, _i64, _p]
        lib.orc_degrees.restype = None
        lib.orc_degrees.argtypes = [_p, _i64, _i64, _p, _p]
        lib.orc_pack_bytes.restype = None
        lib.orc_pack_bytes.argtypes = [_p, _i64, _p, _i64]
        lib.orc_unpack_bits.restype = None
        lib.orc_unpack_bits.argtypes = [_p, _i64, _i64, _p]
        lib.orc_interval_hist_alg19.restype = None
        lib.orc_interval_hist_alg19.argtypes = [_p, _i64, _p]
        lib.orc_interval_hist_alg20.restype = ctypes.c_int
        lib.orc_interval_hist_alg20.argtypes = [_p, _i64, _i64, _i64, _i64, _i64, _p, _p, _p, ctypes.c_int]
        lib.orc_count_relations.restype = None
        lib.orc_count_relations.argtypes = [_p, _i64, _i64, _p, _p]
        lib.orc_bd_action.restype = ctypes.c_double
        lib.orc_bd_action.argtypes = [_p, _i64, _i64, ctypes.c_int, _p]
        lib.orc_chain_pair.restype = _i64
        lib.orc_chain_pair.argtypes = [_p, _i64, _i64, _i64]
        lib.orc_chain_heights.restype = _i64
        lib.orc_chain_heights.argtypes = [_p, _i64, _i64, _p]
        lib.orc_greedy_antichain.restype = _i64
        lib.orc_greedy_antichain.argtypes = [_p, _i64, _i64, _p]
        lib.orc_smear_f.restype = ctypes.c_double
        lib.orc_smear_f.argtypes = [ctypes.c_int, _i64, ctypes.c_double]
        lib.orc_smeared_action.restype = ctypes.c_double
        lib.orc_smeared_action.argtypes = [_p, _i64, _i64, ctypes.c_int, ctypes.c_double]
        lib.orc_max_threads.restype = ctypes.c_int
        lib.orc_max_threads.argtypes = []
        _lib = lib
    return _lib


def _ptr(a: np.ndarray):
    return a.ctypes.data_as(_p)


def row_stride_words(N: int) -> int:
    """Row stride in uint64 blocks: ceil(N/64) rounded up to an even count
    (128-bit aligned rows; the paper aligns rows to 256 bits)."""
    w = (N + 63) // 64
    return w + (w & 1)


def _coords(coords, dim=None) -> np.ndarray:
    c = np.ascontiguousarray(coords, dtype=np.float64)
    assert c.ndim == 2
    return c


def relation(xi, xj, geom: int) -> bool:
    xi = np.ascontiguousarray(xi, dtype=np.float64)
    xj = np.ascontiguousarray(xj, dtype=np.float64)
    return bool(_load().orc_relation(_ptr(xi), _ptr(xj), int(xi.shape[0]), int(geom)))


def causal_matrix_bytes(coords, geom: int) -> np.ndarray:
    c = _coords(coords)
    N, dim = c.shape
    C = np.zeros((N, N), dtype=np.uint8)
    rc = _load().orc_causal_matrix_bytes(_ptr(c), N, dim, int(geom), _ptr(C))
    if rc != 0:
        raise ValueError("oracle: bad dim/geometry")
    return C


def causal_matrix_bits(coords, geom: int, stride: int | None = None) -> np.ndarray:
    c = _coords(coords)
    N, dim = c.shape
    stride = row_stride_words(N) if stride is None else stride
    bits = np.zeros((N, stride), dtype=np.uint64)
    rc = _load().orc_causal_matrix_bits(_ptr(c), N, dim, int(geom), _ptr(bits), stride)
    if rc != 0:
        raise ValueError("oracle: bad dim/geometry/stride")
    return bits


def transpose_bits(bits: np.ndarray, N: int) -> np.ndarray:
    bits = np.ascontiguousarray(bits, dtype=np.uint64)
    out = np.zeros_like(bits)
    _load().orc_transpose_bits(_ptr(bits), N, bits.shape[1], _ptr(out))
    return out


def degrees(bits: np.ndarray, N: int):
    """(outdeg, indeg) int64 arrays of the relation."""
    bits = np.ascontiguousarray(bits, dtype=np.uint64)
    o = np.zeros(N, dtype=np.int64)
    i = np.zeros(N, dtype=np.int64)
    _load().orc_degrees(_ptr(bits), N, bits.shape[1], _ptr(o), _ptr(i))
    return o, i


def pack_bytes(C: np.ndarray, stride: int | None = None) -> np.ndarray:
    C = np.ascontiguousarray(C, dtype=np.uint8)
    N = C.shape[0]
    stride = row_stride_words(N) if stride is None else stride
    bits = np.zeros((N, stride), dtype=np.uint64)
    _load().orc_pack_bytes(_ptr(C), N, _ptr(bits), stride)
    return bits


def unpack_bits(bits: np.ndarray, N: int) -> np.ndarray:
    bits = np.ascontiguousarray(bits, dtype=np.uint64)
    C = np.zeros((N, N), dtype=np.uint8)
    _load().orc_unpack_bits(_ptr(bits), N, bits.shape[1], _ptr(C))
    return C


def interval_hist_alg19(C: np.ndarray) -> np.ndarray:
    """Tier-0: Algorithm 19 on the byte matrix.  Returns hist[0..N-2] (int64)."""
    C = np.ascontiguousarray(C, dtype=np.uint8)
    N = C.shape[0]
    hist = np.zeros(max(N - 1, 0), dtype=np.int64)
    if N >= 2:
        _load().orc_interval_hist_alg19(_ptr(C), N, _ptr(hist))
    return hist


def interval_hist_alg20(bits: np.ndarray, N: int, row_begin: int = 0, row_end: int | None = None,
                        nthreads: int = 0, row_step: int = 1, timing: dict | None = None):
    """Tier-1: Algorithm 20 on bit rows i = row_begin, row_begin+row_step, ... < row_end.
    Returns (hist[0..N-2], word_ops, threads); timing["loop_seconds"] gets the pair-loop wall time."""
    bits = np.ascontiguousarray(bits, dtype=np.uint64)
    row_end = N if row_end is None else row_end
    hist = np.zeros(max(N - 1, 0), dtype=np.int64)
    wops = np.zeros(1, dtype=np.int64)
    secs = ctypes.c_double(0.0)
    T = _load().orc_interval_hist_alg20(_ptr(bits), N, bits.shape[1], row_begin, row_end, row_step,
                                        _ptr(hist), _ptr(wops), ctypes.byref(secs), nthreads)
    if timing is not None:
        timing["loop_seconds"] = secs.value
    if T < 0:
        raise RuntimeError("oracle: alg20 failed (%d)" % T)
    return hist, int(wops[0]), int(T)


def count_relations(bits: np.ndarray, N: int):
    bits = np.ascontiguousarray(bits, dtype=np.uint64)
    R = np.zeros(1, dtype=np.int64)
    W = np.zeros(1, dtype=np.int64)
    _load().orc_count_relations(_ptr(bits), N, bits.shape[1], _ptr(R), _ptr(W))
    return int(R[0]), int(W[0])


def bd_action(hist: np.ndarray, N: int, dim: int):
    """Returns (S, bracket) with bracket the exact integer I_d (eighths for dim 3)."""
    hist = np.ascontiguousarray(hist, dtype=np.int64)
    br = np.zeros(1, dtype=np.int64)
    S = _load().orc_bd_action(_ptr(hist), hist.shape[0], N, dim, _ptr(br))
    return float(S), int(br[0])


def chain_pair(C: np.ndarray, i: int, j: int) -> int:
    """Algorithm 11: links of the longest chain from i to j (0 if unrelated)."""
    C = np.ascontiguousarray(C, dtype=np.uint8)
    return int(_load().orc_chain_pair(_ptr(C), C.shape[0], i, j))


def chain_heights(C: np.ndarray, source: int = -1):
    """-> (height int32[N], longest): elements of the longest chain ending at each element."""
    C = np.ascontiguousarray(C, dtype=np.uint8)
    N = C.shape[0]
    h = np.zeros(N, dtype=np.int32)
    best = int(_load().orc_chain_heights(_ptr(C), N, source, _ptr(h)))
    return h, best


def greedy_antichain(C: np.ndarray, seed: int) -> np.ndarray:
    """Algorithm 13 -> member uint8[N]."""
    C = np.ascontiguousarray(C, dtype=np.uint8)
    N = C.shape[0]
    m = np.zeros(N, dtype=np.uint8)
    _load().orc_greedy_antichain(_ptr(C), N, seed, _ptr(m))
    return m


def smear_f(dim: int, m: int, eps: float) -> float:
    return float(_load().orc_smear_f(dim, m, eps))


def smeared_action(hist: np.ndarray, N: int, dim: int, eps: float) -> float:
    hist = np.ascontiguousarray(hist, dtype=np.int64)
    return float(_load().orc_smeared_action(_ptr(hist), hist.shape[0], N, dim, eps))


def max_threads() -> int:
    return int(_load().orc_max_threads())


def action_pipeline(coords, geom: int, tier: int = 1):
    """coords -> (bits, hist, S, bracket) through the oracle only."""
    c = _coords(coords)
    N, dim = c.shape
    if tier == 0:
        C = causal_matrix_bytes(c, geom)
        bits = pack_bytes(C)
        hist = interval_hist_alg19(C)
    else:
        bits = causal_matrix_bits(c, geom)
        hist, _, _ = interval_hist_alg20(bits, N)
    # FLRW_POLAR (six numbers per point) and DS4_SPHERICAL (seven) describe 3+1 dimensional events; the paper
    # prints no action for 4+1 dimensions (Eq. 4.10-4.12 stop at d = 4): the bracket and S are then None
    sdim = 4 if geom in (GEOM_FLRW_POLAR, GEOM_DS4_SPHERICAL) else dim
    if sdim > 4:
        return bits, hist, None, None
    S, br = bd_action(hist, N, sdim)
    return bits, hist, S, br
