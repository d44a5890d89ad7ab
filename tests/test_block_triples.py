"""The block-triple counter behind DESIGN.md section 5's element-order comparison (tests/count_block_triples.py)."""
import os
import sys

import numpy as np

sys.path.insert(0, os.path.dirname(os.path.abspath(__file__)))
import count_block_triples as cbt  # noqa: E402

from paper_1805_04463_b200 import inputs as inp  # noqa: E402


def test_orders_partition_and_counter_matches_brute_force(oracle):
    N, block = 700, 64
    coords = inp.sprinkle(inp.GEOM_MINK_CONE, 4, N, 3)
    bits = oracle.causal_matrix_bits(coords, inp.GEOM_MINK_CONE)
    C = oracle.unpack_bits(bits, N).astype(bool)
    ncell = (N + block - 1) // block
    lives = {}
    for name, cell in cbt.orders(coords, block).items():
        counts = np.bincount(cell, minlength=ncell)
        assert counts.sum() == N and counts.max() <= block and len(counts) == ncell, name
        E = cbt.block_occupancy(bits, N, cell, ncell, chunk=100)
        want = np.zeros((ncell, ncell), dtype=bool)
        ii, jj = np.nonzero(C)
        want[cell[ii], cell[jj]] = True
        assert np.array_equal(E, want), name
        lives[name] = cbt.live_triples(E)
        assert lives[name] == cbt.live_triples_bruteforce(E), name
    # in time order the block matrix is upper triangular: live triples need I <= K <= J
    E = cbt.block_occupancy(bits, N, np.arange(N) // block, ncell)
    assert not np.tril(E, -1).any()
