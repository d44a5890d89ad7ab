"""Pins of the oracle's chain / antichain functions (NEXT-3; Algorithms 11 and 13)
against things other than the oracle: closed forms, a textbook routine (patience sorting for the longest
increasing subsequence), brute force over all subsets of tiny posets, and the defining properties of a
maximal antichain.  CPU only."""
import bisect
import itertools

import numpy as np
import pytest

from paper_1805_04463_b200 import inputs as inp


def _matrix(oracle, geom, dim, N, seed):
    coords = inp.sprinkle(geom, dim, N, seed)
    return coords, oracle.causal_matrix_bytes(coords, geom)


def _random_poset(rng, N, p):
    """transitive closure of a random upper-triangular relation"""
    C = np.triu(rng.random((N, N)) < p, 1)
    R = C.copy()
    for k in range(N):
        R |= np.outer(R[:, k], R[k, :])
    return R.astype(np.uint8)


def test_chain_closed_forms(oracle):
    N = 50
    chain = np.triu(np.ones((N, N), dtype=np.uint8), 1)              # total order
    h, best = oracle.chain_heights(chain)
    assert best == N and np.array_equal(h, np.arange(1, N + 1))
    assert oracle.chain_pair(chain, 0, N - 1) == N - 1               # links = elements - 1
    assert oracle.chain_pair(chain, 3, 4) == 1 and oracle.chain_pair(chain, 4, 3) == 0
    h, best = oracle.chain_heights(chain, source=10)
    assert best == N - 10 and np.array_equal(h[:10], np.zeros(10)) and h[10] == 1 and h[-1] == N - 10
    anti = np.zeros((N, N), dtype=np.uint8)
    h, best = oracle.chain_heights(anti)
    assert best == 1 and np.all(h == 1)
    assert oracle.chain_heights(np.zeros((0, 0), dtype=np.uint8))[1] == 0


def test_longest_chain_is_longest_increasing_subsequence(oracle):
    """1+1 light-cone diamond: i -< j iff u and v both increase, so the longest chain is the longest
    strictly increasing subsequence of v in u order -- patience sorting, O(N log N), independent."""
    for N, seed in ((300, 1), (1500, 2)):
        coords, C = _matrix(oracle, inp.GEOM_MINK2_LIGHTCONE, 2, N, seed)
        order = np.argsort(coords[:, 0], kind="stable")
        piles = []
        for v in coords[order, 1]:
            k = bisect.bisect_left(piles, v)
            if k == len(piles):
                piles.append(v)
            else:
                piles[k] = v
        h, best = oracle.chain_heights(C)
        assert best == len(piles)
        assert 1.2 * np.sqrt(N) < best < 2.0 * np.sqrt(N)            # -> 2 sqrt(N) from below (Vershik-Kerov)


def test_chain_brute_force_small(oracle):
    rng = np.random.default_rng(3)
    for N, p in ((9, 0.25), (12, 0.15), (12, 0.4)):
        C = _random_poset(rng, N, p)
        best_bf = 0
        ending = np.zeros(N, dtype=int)
        for r in range(1, N + 1):
            for sub in itertools.combinations(range(N), r):
                if all(C[a, b] for a, b in zip(sub, sub[1:])):       # consecutive related => a chain (transitive)
                    best_bf = max(best_bf, r)
                    ending[sub[-1]] = max(ending[sub[-1]], r)
        h, best = oracle.chain_heights(C)
        assert best == best_bf and np.array_equal(h, ending)


@pytest.mark.parametrize("geom,dim", [(inp.GEOM_MINK2_LIGHTCONE, 2), (inp.GEOM_MINK_CONE, 4), (inp.GEOM_DS2_SLAB, 2)])
def test_algorithm_11_agrees_with_heights(oracle, geom, dim):
    """Alg. 11 (recursive, memoised, per pair) against the height definition with a source."""
    N = 260
    _, C = _matrix(oracle, geom, dim, N, 11)
    rng = np.random.default_rng(5)
    rel = np.argwhere(C)
    for i, j in rel[rng.choice(len(rel), 25, replace=False)]:
        h, _ = oracle.chain_heights(C, source=int(i))
        assert oracle.chain_pair(C, int(i), int(j)) == h[j] - 1
    i, j = np.argwhere(C == 0)[5]
    if i < j:
        assert oracle.chain_pair(C, int(i), int(j)) == 0


def _check_maximal_antichain(C, member, seed):
    idx = np.flatnonzero(member)
    assert member[seed]
    sym = C | C.T
    assert not sym[np.ix_(idx, idx)].any()                           # no two members related
    others = np.flatnonzero(member == 0)
    assert sym[np.ix_(others, idx)].any(axis=1).all()                # every other element is related to a member


def test_greedy_antichain_properties(oracle):
    N = 40
    chain = np.triu(np.ones((N, N), dtype=np.uint8), 1)
    m = oracle.greedy_antichain(chain, 7)
    assert m.sum() == 1 and m[7]
    anti = np.zeros((N, N), dtype=np.uint8)
    assert oracle.greedy_antichain(anti, 3).sum() == N
    for geom, dim, N in ((inp.GEOM_MINK2_LIGHTCONE, 2, 300), (inp.GEOM_MINK_CONE, 3, 250), (inp.GEOM_DS2_SLAB, 2, 300)):
        _, C = _matrix(oracle, geom, dim, N, 4)
        for seed in (0, N // 2, N - 1):
            _check_maximal_antichain(C, oracle.greedy_antichain(C, seed), seed)


def test_greedy_antichain_step_by_step(oracle):
    """Algorithm 13 re-walked with Python sets on small random posets, including its tie rule (first j
    with the largest c)."""
    rng = np.random.default_rng(9)
    for N, p in ((14, 0.2), (25, 0.1), (25, 0.3)):
        C = _random_poset(rng, N, p)
        J = [set(np.flatnonzero(C[j] | C[:, j])) for j in range(N)]
        for seed in range(0, N, 5):
            xi = set(range(N)) - J[seed] - {seed}
            A = {seed} | xi
            while xi:
                sigma, k = 0, None
                for j in sorted(xi):
                    c = len(A - J[j])
                    if c > sigma:
                        sigma, k = c, j
                A -= J[k]
                xi -= J[k] | {k}
            m = oracle.greedy_antichain(C, seed)
            assert set(np.flatnonzero(m)) == A


def test_greedy_antichain_width_bound(oracle):
    """A maximal antichain can be no larger than the width; on tiny posets the width by brute force."""
    rng = np.random.default_rng(1)
    C = _random_poset(rng, 13, 0.2)
    sym = C | C.T
    width = max(r for r in range(1, 14) for sub in itertools.combinations(range(13), r)
                if not sym[np.ix_(sub, sub)].any())
    for seed in range(13):
        assert 1 <= oracle.greedy_antichain(C, seed).sum() <= width
