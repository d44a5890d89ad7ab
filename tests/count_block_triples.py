"""How many (I, K, J) block triples of the a2 contraction are live under different element orders?

    python tests/count_block_triples.py [--N 65536] [--block 256]

count(i, j) = sum_k C_ik C_kj needs no order of the elements (Alg. 19/20), and the
interval histogram and the action are invariant under relabelling.  The tensor a2 route executes one 256 x 256 x 256
stage per (I, K, J) triple of blocks and can skip a stage when block (I, K) or block (K, J) of the bit matrix is
empty (and the whole tile when block (I, J) is: no related pair to tally).  This script counts, on the oracle's
matrix of the headline workload (config 3), the triples that stay live

    live = |{(I, K, J) : block(I,K) != 0 and block(K,J) != 0 and block(I,J) != 0}|        (all K)

for (a) the time order the library uses, (b) a k-d clustering of the points into space-time cells of `block` points,
(c) time slabs of 16 blocks with a spatial k-d clustering inside each slab.  It calls the oracle and numpy only (CPU,
about six minutes on 8 cores at N = 65536); the numbers are quoted in DESIGN.md section 5.  Test infrastructure, not product code.
"""
from __future__ import annotations

import argparse
import os
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def kd_cells(points: np.ndarray, idx: np.ndarray, axes, leaf: int, depth: int = 0):
    """Recursive median split of the points `idx` along the cycling `axes` into leaves of `leaf` points; returns the
    leaves in depth-first order (neighbouring leaves are neighbouring cells)."""
    if idx.shape[0] <= leaf:
        return [idx]
    ax = axes[depth % len(axes)]
    order = idx[np.argsort(points[idx, ax], kind="stable")]
    half = (order.shape[0] // (2 * leaf)) * leaf or leaf
    return kd_cells(points, order[:half], axes, leaf, depth + 1) + kd_cells(points, order[half:], axes, leaf, depth + 1)


def orders(coords: np.ndarray, block: int):
    """name -> cell index of every element (cells of `block` elements; the last one may be ragged)."""
    N, dim = coords.shape
    out = {"a_time_order": np.arange(N) // block}
    leaves = kd_cells(coords, np.arange(N), list(range(dim)), block)
    cell = np.empty(N, dtype=np.int64)
    for c, leaf in enumerate(leaves):
        cell[leaf] = c
    out["b_kd_spacetime_cells"] = cell
    slab = 16 * block
    cell = np.empty(N, dtype=np.int64)
    c = 0
    for s0 in range(0, N, slab):
        for leaf in kd_cells(coords, np.arange(s0, min(N, s0 + slab)), list(range(1, dim)), block):
            cell[leaf] = c
            c += 1
    out["c_time_slabs_spatial_kd"] = cell
    return out


def block_occupancy(bits: np.ndarray, N: int, cell: np.ndarray, ncell: int, chunk: int = 1024) -> np.ndarray:
    """E[a][b] = some related pair i -< j has cell(i) = a and cell(j) = b."""
    E = np.zeros((ncell, ncell), dtype=bool)
    col_order = np.argsort(cell, kind="stable")
    starts = np.searchsorted(cell[col_order], np.arange(ncell))
    for r0 in range(0, N, chunk):
        rows = bits[r0:r0 + chunk]
        C = np.unpackbits(rows.view(np.uint8), axis=1, bitorder="little")[:, :N]
        C = C[:, col_order]
        occ = np.add.reduceat(C, starts, axis=1, dtype=np.int32) > 0           # [rows][cell of j]
        rc = cell[r0:r0 + rows.shape[0]]
        for a in np.unique(rc):
            E[a] |= occ[rc == a].any(axis=0)
    return E


def live_triples(E: np.ndarray) -> int:
    Ei = E.astype(np.int64)
    return int(((Ei @ Ei) * Ei).sum())


def live_triples_bruteforce(E: np.ndarray) -> int:
    n = E.shape[0]
    return sum(1 for i in range(n) for k in range(n) for j in range(n) if E[i, k] and E[k, j] and E[i, j])


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--N", type=int, default=0)
    ap.add_argument("--block", type=int, default=256)
    args = ap.parse_args()
    import oracle
    from paper_1805_04463_b200 import inputs as inp
    oracle.build()
    cfg = inp.CONFIGS[3]
    N = args.N or cfg.N
    coords = inp.make_config_coords(cfg, N=N)
    bits = oracle.causal_matrix_bits(coords, cfg.geometry)
    R, _ = oracle.count_relations(bits, N)
    ncell = (N + args.block - 1) // args.block
    print("config 3 (%s), N = %d, %d relations (%.1f %% of the pairs), %d cells of %d" %
          (cfg.name, N, R, 200.0 * R / (N * (N - 1.0)), ncell, args.block))
    base = None
    for name, cell in orders(coords, args.block).items():
        E = block_occupancy(bits, N, cell, ncell)
        live = live_triples(E)
        base = base or live
        print("%-26s non-empty blocks %6d of %d   live (I,K,J) triples %9d   = %.3f x the time order" %
              (name, int(E.sum()), ncell * ncell, live, live / base))


if __name__ == "__main__":
    main()
