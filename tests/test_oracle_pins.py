"""Pins for the oracle (CPU only).  Each test checks oracle/ against something
other than itself: a closed form, an invariant, brute force on tiny inputs, an
independent algorithm, or a number PAPER.md prints.  Citations: PAPER.md lines.
"""
import itertools
import math
import os
from fractions import Fraction

import numpy as np
import pytest

from paper_1805_04463_b200 import inputs as inp

GOLDEN = os.path.join(os.path.dirname(__file__), "golden")


# ----------------------------------------------------------------------------- helpers
def brute_force_hist(C):
    """Interval sizes by explicit set membership: |J+(i) & J-(j)|."""
    N = C.shape[0]
    future = [set(np.nonzero(C[i])[0].tolist()) for i in range(N)]
    past = [set(np.nonzero(C[:, j])[0].tolist()) for j in range(N)]
    hist = np.zeros(max(N - 1, 0), dtype=np.int64)
    for i in range(N):
        for j in future[i]:
            hist[len(future[i] & past[j])] += 1
    return hist


def transitive_closure(C):
    C = C.astype(bool)
    N = C.shape[0]
    for k in range(N):
        C = C | (C[:, k:k + 1] & C[k:k + 1, :])
    return C.astype(np.uint8)


def hist_both_tiers(orc, C):
    N = C.shape[0]
    h0 = orc.interval_hist_alg19(C)
    bits = orc.pack_bytes(C)
    h1, wops, _ = orc.interval_hist_alg20(bits, N)
    return h0, h1, bits, wops


def all_geoms():
    return [
        (inp.GEOM_MINK2_LIGHTCONE, 2, 11),
        (inp.GEOM_MINK_CONE, 2, 12),
        (inp.GEOM_MINK_CONE, 3, 13),
        (inp.GEOM_MINK_CONE, 4, 14),
        (inp.GEOM_DS2_SLAB, 2, 15),
    ]


# ----------------------------------------------------------------------------- stage 1
def test_relation_hand_cases(oracle):
    L, Cn, D = inp.GEOM_MINK2_LIGHTCONE, inp.GEOM_MINK_CONE, inp.GEOM_DS2_SLAB
    # light cone (ds^2 = -2 du dv): strict in both coordinates
    assert oracle.relation([0.1, 0.2], [0.3, 0.4], L)
    assert not oracle.relation([0.1, 0.5], [0.3, 0.4], L)
    assert not oracle.relation([0.1, 0.2], [0.1, 0.4], L)      # du = 0: null, not related
    assert not oracle.relation([0.3, 0.4], [0.1, 0.2], L)      # wrong time order
    # flat cone: dt^2 >= |dx|^2, null related (reading A1), past not related
    assert oracle.relation([0, 0, 0, 0], [1.0, 0.5, 0.5, 0.5], Cn)          # 1 >= 0.75
    assert not oracle.relation([0, 0, 0, 0], [1.0, 0.6, 0.6, 0.6], Cn)      # 1 < 1.08
    assert oracle.relation([0.0, 0.0], [1.0, 1.0], Cn)                      # null
    assert oracle.relation([0.0, 0.0], [1.0, -1.0], Cn)
    assert not oracle.relation([1.0, 0.0], [0.0, 0.0], Cn)                  # dt < 0
    assert oracle.relation([0, 0, 0], [5.0, 3.0, 4.0], Cn)                  # 25 >= 25
    assert not oracle.relation([0, 0, 0], [5.0, 3.0, 4.5], Cn)
    # de Sitter slab: angular distance wraps around the circle
    assert oracle.relation([-1.0, 0.1], [-0.7, 6.2], D)        # min(6.1, 0.183..) = 0.183 <= 0.3
    assert not oracle.relation([-1.0, 0.1], [-0.9, 6.2], D)    # 0.183 > 0.1
    assert not oracle.relation([-1.0, 1.0], [-0.5, 3.0], D)    # 2.0 > 0.5
    assert oracle.relation([-1.0, 1.0], [-0.5, 1.5], D)        # 0.5 >= 0.5 (null related)


def test_ds_relation_matches_paper_form(oracle):
    """The paper's form pi - |pi - |dtheta|| equals min(a, 2pi-a)
    in exact arithmetic; away from the null cone both give the same relation."""
    rng = np.random.default_rng(5)
    n_checked = 0
    for _ in range(4000):
        e1, e2 = np.sort(rng.uniform(-1.2, -0.2, 2))
        t1, t2 = rng.uniform(0, 2 * np.pi, 2)
        paper = np.pi - abs(np.pi - abs(t1 - t2))
        if abs(paper - (e2 - e1)) < 1e-9:
            continue
        n_checked += 1
        assert oracle.relation([e1, t1], [e2, t2], inp.GEOM_DS2_SLAB) == (paper <= e2 - e1)
    assert n_checked > 3900


@pytest.mark.parametrize("geom,dim,seed", all_geoms())
def test_matrix_structure_transitive_acyclic(oracle, geom, dim, seed):
    """Upper triangular (acyclic under the time order) and
    transitive: (C.C > 0) => C."""
    N = 700
    coords = inp.sprinkle(geom, dim, N, seed)
    C = oracle.causal_matrix_bytes(coords, geom)
    assert np.array_equal(C, np.triu(C, 1))
    two_step = (C.astype(np.float32) @ C.astype(np.float32)) > 0
    assert not np.any(two_step & (C == 0))
    # direct re-evaluation of the predicate in numpy for the flat cone (different code path)
    if geom == inp.GEOM_MINK_CONE:
        d = coords[None, :, :] - coords[:, None, :]
        s = np.zeros((N, N))
        for a in range(1, dim):
            s = s + d[:, :, a] * d[:, :, a]
        ref = (d[:, :, 0] >= 0) & (d[:, :, 0] * d[:, :, 0] >= s)
        ref = np.triu(ref, 1)
        assert np.array_equal(C.astype(bool), ref)


@pytest.mark.parametrize("N", [0, 1, 2, 63, 64, 65, 130, 1000])
def test_bit_layout_and_padding(oracle, N):
    """LSB-first blocks, zero padding, pack/unpack/transposes agree."""
    coords = inp.sprinkle(inp.GEOM_MINK2_LIGHTCONE, 2, N, 3) if N else np.zeros((0, 2))
    C = oracle.causal_matrix_bytes(coords, inp.GEOM_MINK2_LIGHTCONE)
    bits = oracle.causal_matrix_bits(coords, inp.GEOM_MINK2_LIGHTCONE)
    stride = oracle.row_stride_words(N)
    assert bits.shape == (N, stride) and stride % 2 == 0 and stride * 64 >= N
    assert np.array_equal(bits, oracle.pack_bytes(C))
    assert np.array_equal(oracle.unpack_bits(bits, N), C)
    # independent unpack with numpy: little-endian bit order
    if N:
        nb = np.unpackbits(bits.view(np.uint8), axis=1, bitorder="little")
        assert np.array_equal(nb[:, :N], C)
        assert not nb[:, N:].any()
        bT = oracle.transpose_bits(bits, N)
        assert np.array_equal(oracle.unpack_bits(bT, N), C.T)


# ----------------------------------------------------------------------------- stage 2
@pytest.mark.parametrize("N", [2, 3, 5, 64, 65, 300])
def test_chain_closed_form(oracle, N):
    """Total order: pair (i,j) has j-i-1 interior elements => N_k = N-1-k."""
    coords = inp.chain_lightcone(N)
    C = oracle.causal_matrix_bytes(coords, inp.GEOM_MINK2_LIGHTCONE)
    assert C.sum() == N * (N - 1) // 2
    h0, h1, _, _ = hist_both_tiers(oracle, C)
    expect = np.arange(N - 1, 0, -1, dtype=np.int64)
    assert np.array_equal(h0, expect)
    assert np.array_equal(h1, expect)
    # actions of the chain: I2 = N, I4 = N-1 (N >= 5), from N_k = N-1-k
    S2, I2 = oracle.bd_action(h0, N, 2)
    assert I2 == N - 2 * max(N - 1, 0) + 4 * max(N - 2, 0) - 2 * max(N - 3, 0)
    if N >= 4:
        assert I2 == N and S2 == 2.0 * N
    S4, I4 = oracle.bd_action(h0, N, 4)
    if N >= 5:
        assert I4 == N - 1
        assert S4 == pytest.approx(4 / math.sqrt(6) * (N - 1), rel=1e-15)


@pytest.mark.parametrize("N", [1, 2, 64, 257])
def test_antichain(oracle, N):
    coords = inp.antichain_lightcone(N)
    C = oracle.causal_matrix_bytes(coords, inp.GEOM_MINK2_LIGHTCONE)
    assert C.sum() == 0
    h0, h1, _, _ = hist_both_tiers(oracle, C)
    assert not h0.any() and not h1.any()
    for dim in (2, 4):
        _, I = oracle.bd_action(h0, N, dim)
        assert I == N


def test_exhaustive_small_posets(oracle):
    """Every transitive strictly-upper-triangular 0/1 matrix with N <= 5."""
    n_posets = 0
    for N in range(2, 6):
        pairs = [(i, j) for i in range(N) for j in range(i + 1, N)]
        for mask in range(1 << len(pairs)):
            C = np.zeros((N, N), dtype=np.uint8)
            for b, (i, j) in enumerate(pairs):
                if (mask >> b) & 1:
                    C[i, j] = 1
            if not np.array_equal(transitive_closure(C), C):
                continue
            n_posets += 1
            expect = brute_force_hist(C)
            h0, h1, _, _ = hist_both_tiers(oracle, C)
            assert np.array_equal(h0, expect), (N, mask)
            assert np.array_equal(h1, expect), (N, mask)
    # labelled-by-linear-extension partial orders on 2..5 points: 2, 7, 40, 357
    assert n_posets == 2 + 7 + 40 + 357


@pytest.mark.parametrize("N,p,seed", [(8, 0.5, 0), (33, 0.2, 1), (64, 0.1, 2), (64, 0.03, 3), (100, 0.05, 4)])
def test_random_transitive_closures_bruteforce(oracle, N, p, seed):
    rng = np.random.default_rng(seed)
    C = np.triu((rng.random((N, N)) < p).astype(np.uint8), 1)
    C = transitive_closure(C)
    expect = brute_force_hist(C)
    h0, h1, bits, wops = hist_both_tiers(oracle, C)
    assert np.array_equal(h0, expect)
    assert np.array_equal(h1, expect)
    R, W = oracle.count_relations(bits, N)
    assert R == int(C.sum()) == int(expect.sum())
    ii, jj = np.nonzero(C)
    assert W == wops == int(((jj >> 6) - (ii >> 6) + 1).sum())


def test_nontransitive_input_follows_alg19_definition(oracle):
    """Alg. 19 counts k with i<k and k<j as matrix entries; on a non-transitive
    matrix tier-0 and tier-1 still agree with the matrix-product definition."""
    rng = np.random.default_rng(9)
    N = 90
    C = np.triu((rng.random((N, N)) < 0.3).astype(np.uint8), 1)
    prod = C.astype(np.int64) @ C.astype(np.int64)
    expect = np.bincount(prod[C == 1], minlength=N - 1).astype(np.int64)
    h0, h1, _, _ = hist_both_tiers(oracle, C)
    assert np.array_equal(h0, expect)
    assert np.array_equal(h1, expect)


@pytest.mark.parametrize("geom,dim,seed", all_geoms())
@pytest.mark.parametrize("N", [64, 1000])
def test_tier1_equals_tier0_and_moments(oracle, geom, dim, seed, N):
    """Alg. 20 == Alg. 19 on every geometry (N=1000 is not a multiple of 64), and
    sum_k N_k = R,  sum_k k N_k = sum_m indeg(m) outdeg(m) (number of 3-chains)."""
    coords = inp.sprinkle(geom, dim, N, seed + N)
    C = oracle.causal_matrix_bytes(coords, geom)
    h0, h1, bits, _ = hist_both_tiers(oracle, C)
    assert np.array_equal(h0, h1)
    R = int(C.sum())
    assert int(h0.sum()) == R
    indeg = C.sum(axis=0).astype(np.int64)
    outdeg = C.sum(axis=1).astype(np.int64)
    assert int((np.arange(N - 1) * h0).sum()) == int((indeg * outdeg).sum())
    # row-range additivity of tier-1 (used for sampled parity at full size)
    ha, wa, _ = oracle.interval_hist_alg20(bits, N, 0, N // 3)
    hb, wb, _ = oracle.interval_hist_alg20(bits, N, N // 3, N)
    assert np.array_equal(ha + hb, h1)


@pytest.mark.parametrize("geom,dim,N,step", [(inp.GEOM_MINK_CONE, 4, 1000, 7), (inp.GEOM_DS2_SLAB, 2, 777, 5),
                                             (inp.GEOM_MINK2_LIGHTCONE, 2, 130, 64)])
def test_tier1_row_step_partitions_the_rows(oracle, geom, dim, N, step):
    """The stride of Alg. 20's outer loop (`row_step`, the sample bench.py times for the CPU
    baseline and the reference arm): rows row_begin + m * row_step, nothing else.  The residue classes add up to the
    whole histogram and the whole word count; one class equals the sum of its rows taken one at a time, from an
    offset start too; N is not a multiple of the stride."""
    coords = inp.sprinkle(geom, dim, N, 900 + N)
    bits = oracle.causal_matrix_bits(coords, geom)
    full, wfull, _ = oracle.interval_hist_alg20(bits, N)
    parts = [oracle.interval_hist_alg20(bits, N, s0, N, row_step=step) for s0 in range(step)]
    assert np.array_equal(sum(p[0] for p in parts), full)
    assert sum(p[1] for p in parts) == wfull
    assert full.sum() > 0 and sum(1 for p in parts if p[0].sum() > 0) >= min(step, 3)
    for s0, row_end in ((0, N), (step - 1, N), (3, N - 11)):
        got, wgot, _ = oracle.interval_hist_alg20(bits, N, s0, row_end, row_step=step)
        rows = [oracle.interval_hist_alg20(bits, N, i, i + 1) for i in range(s0, row_end, step)]
        assert np.array_equal(got, sum(r[0] for r in rows)) and wgot == sum(r[1] for r in rows)
    # a stride larger than the range touches its first row only
    one, wone, _ = oracle.interval_hist_alg20(bits, N, 2, 10, row_step=100)
    ref, wref, _ = oracle.interval_hist_alg20(bits, N, 2, 3)
    assert np.array_equal(one, ref) and wone == wref


def test_tier1_equals_tier0_N2048(oracle):
    cfg = inp.CONFIGS[5]
    coords = inp.make_config_coords(cfg, batch_index=1)
    C = oracle.causal_matrix_bytes(coords, cfg.geometry)
    h0, h1, _, _ = hist_both_tiers(oracle, C)
    assert np.array_equal(h0, h1)
    # soft sanity: ordering fraction of the 3+1 diamond is about 1/10 (Myrheim-Meyer; not in PAPER.md)
    frac = C.sum() / (cfg.N * (cfg.N - 1) / 2)
    assert 0.07 < frac < 0.13


# ----------------------------------------------------------------------------- 1+1 diamond: independent algorithms
def count_inversions(a):
    """Textbook merge-sort inversion count."""
    a = list(a)
    if len(a) < 2:
        return 0, a
    mid = len(a) // 2
    il, left = count_inversions(a[:mid])
    ir, right = count_inversions(a[mid:])
    merged, i, j, inv = [], 0, 0, il + ir
    while i < len(left) and j < len(right):
        if left[i] <= right[j]:
            merged.append(left[i]); i += 1
        else:
            merged.append(right[j]); j += 1; inv += len(left) - i
    merged += left[i:] + right[j:]
    return inv, merged


def sat_histogram(coords):
    """Interval sizes in the light-cone diamond from a summed-area table over the
    rank grid: |I(i,j)| = points strictly inside the rectangle (u_i,u_j)x(v_i,v_j)."""
    N = coords.shape[0]
    ru = np.argsort(np.argsort(coords[:, 0], kind="stable"), kind="stable")
    rv = np.argsort(np.argsort(coords[:, 1], kind="stable"), kind="stable")
    G = np.zeros((N + 1, N + 1), dtype=np.int32)
    G[ru + 1, rv + 1] = 1
    P = G.cumsum(axis=0, dtype=np.int32).cumsum(axis=1, dtype=np.int32)  # P[a][b] = #{ru<a, rv<b}
    hist = np.zeros(N - 1, dtype=np.int64)
    R = 0
    for i in range(N):
        rel = (ru > ru[i]) & (rv > rv[i])
        a0, b0 = ru[i] + 1, rv[i] + 1
        a1, b1 = ru[rel], rv[rel]
        cnt = P[a1, b1] - P[a0, b1] - P[a1, b0] + P[a0, b0]
        hist += np.bincount(cnt, minlength=N - 1)
        R += int(rel.sum())
    return hist, R


@pytest.mark.parametrize("N,tier", [(1024, 0), (4096, 1)])
def test_lightcone_diamond_sat_and_inversions(oracle, N, tier):
    cfg = inp.CONFIGS[1]
    coords = inp.make_config_coords(cfg, N=N)
    bits = oracle.causal_matrix_bits(coords, cfg.geometry)
    R, _ = oracle.count_relations(bits, N)
    # R = N(N-1)/2 - inversions of the v-ranks taken in u-order
    order = np.argsort(coords[:, 0], kind="stable")
    inv, _ = count_inversions(coords[order, 1].tolist())
    assert R == N * (N - 1) // 2 - inv
    # expected relation fraction of the 2-D diamond: E[R] = N(N-1)/4, Kendall variance
    sd = math.sqrt(N * (N - 1) * (2 * N + 5) / 72)
    assert abs(R - N * (N - 1) / 4) < 4.5 * sd
    expect, R_sat = sat_histogram(coords)
    assert R_sat == R
    if tier == 0:
        hist = oracle.interval_hist_alg19(oracle.unpack_bits(bits, N))
    else:
        hist, _, _ = oracle.interval_hist_alg20(bits, N)
    assert np.array_equal(hist, expect)


# ----------------------------------------------------------------------------- stage 3
def _read_table(name):
    rows = []
    with open(os.path.join(GOLDEN, name)) as f:
        for line in f:
            line = line.split("#")[0].strip()
            if line:
                rows.append(line.split())
    return rows


def _prefactor(dim):
    return {2: 2.0,
            3: (1 / math.gamma(5 / 3)) * (math.pi / (3 * math.sqrt(2))) ** (2 / 3),
            4: 4 / math.sqrt(6)}[dim]


def test_action_coefficients_three_statements(oracle):
    """Eq. 4.10-4.12 (golden), Eq. 4.5-4.7 (golden, sign flipped) and the eps -> 1
    limit of Eq. 4.16-4.18 agree, and the oracle reproduces them term by term."""
    act = {int(r[0]): [Fraction(x) for x in r[2:6]] for r in _read_table("bd_action_coefficients.txt")}
    dal = {int(r[0]): (Fraction(r[1]), [Fraction(x) for x in r[2:6]]) for r in _read_table("dalembertian_coefficients.txt")}
    N = 1000
    for dim in (2, 3, 4):
        a, b = dal[dim]
        assert [-(a * x) for x in b] == act[dim]                      # statement 2 vs statement 1
        for m in range(0, 8):                                           # statement 3
            f = oracle.smear_f(dim, m, 1.0)
            # S_eps at eps=1: bracket N - a*sum n_m f(m-1)  =>  c_{m+1} = -a f(m)
            c = float(act[dim][m]) if m < 4 else 0.0
            assert -float(a) * f == pytest.approx(c, abs=1e-15), (dim, m)
        S0, _ = oracle.bd_action(np.zeros(4, dtype=np.int64), N, dim)
        assert S0 == pytest.approx(_prefactor(dim) * N, rel=1e-15)
        for m in range(4):
            h = np.zeros(6, dtype=np.int64)
            h[m] = 7
            S, _ = oracle.bd_action(h, N, dim)
            assert S == pytest.approx(_prefactor(dim) * (N + 7 * float(act[dim][m])), rel=1e-14)
        h = np.zeros(6, dtype=np.int64); h[4] = 5; h[5] = 9             # n_5, n_6 do not enter
        assert oracle.bd_action(h, N, dim)[0] == S0


def test_action_short_hist_and_int64_range(oracle):
    # missing entries are zero (reading A9)
    assert oracle.bd_action(np.array([3], dtype=np.int64), 10, 4)[1] == 10 - 3
    assert oracle.bd_action(np.zeros(0, dtype=np.int64), 10, 2)[1] == 10
    # counts far above 2^31 stay exact in the integer bracket
    h = np.array([3_000_000_000, 2_500_000_000, 2_000_000_001, 1_999_999_999], dtype=np.int64)
    _, I = oracle.bd_action(h, 131072, 4)
    assert I == 131072 - 3_000_000_000 + 9 * 2_500_000_000 - 16 * 2_000_000_001 + 8 * 1_999_999_999


def test_smeared_action_reduces_to_local_at_eps_1(oracle):
    coords = inp.sprinkle(inp.GEOM_DS2_SLAB, 2, 600, 77)
    bits = oracle.causal_matrix_bits(coords, inp.GEOM_DS2_SLAB)
    hist, _, _ = oracle.interval_hist_alg20(bits, 600)
    for dim in (2, 3, 4):
        S, _ = oracle.bd_action(hist, 600, dim)
        assert oracle.smeared_action(hist, 600, dim, 1.0) == pytest.approx(S, rel=1e-12)


def test_smear_f_against_paper_form(oracle):
    """Eq. 4.16-4.18 as printed (with the 1/(1-eps) factors), rational arithmetic."""
    for eps in (Fraction(1, 64), Fraction(1, 3)):
        q = 1 - eps
        for m in (0, 1, 2, 3, 10, 40):
            f2 = q ** m * (1 - 2 * m * eps / q + Fraction(m * (m - 1), 2) * eps ** 2 / q ** 2)
            f3 = q ** m * (1 - Fraction(27, 8) * m * eps / q + Fraction(9, 8) * m * (m - 1) * eps ** 2 / q ** 2)
            f4 = q ** m * (1 - 9 * m * eps / q + 8 * m * (m - 1) * eps ** 2 / q ** 2
                           - Fraction(4, 3) * m * (m - 1) * (m - 2) * eps ** 3 / q ** 3)
            for dim, f in ((2, f2), (3, f3), (4, f4)):
                assert oracle.smear_f(dim, m, float(eps)) == pytest.approx(float(f), rel=1e-12, abs=1e-15)


def test_smeared_action_against_exact_rational(oracle):
    """Eq. 4.13-4.15 with Eq. 4.16-4.18 exactly as printed, in rational arithmetic, on a real histogram
    (the bracket cancels to ~1e-3 of its terms here): pins the oracle's long-double sum, index shift
    n_m f(m-1) and prefactors.  Irrational prefactors are applied in floating point at the end."""
    N = 400
    coords = inp.sprinkle(inp.GEOM_DS2_SLAB, 2, N, 5)
    hist, _, _ = oracle.interval_hist_alg20(oracle.causal_matrix_bits(coords, inp.GEOM_DS2_SLAB), N)
    for eps in (Fraction(1, 64), Fraction(1, 5), Fraction(3, 4)):
        q = 1 - eps
        sums = {2: Fraction(0), 3: Fraction(0), 4: Fraction(0)}
        for mm in range(1, N):                                   # the paper's m = 1 .. N-1, n_m = hist[m-1]
            n_m = int(hist[mm - 1]) if mm - 1 < hist.shape[0] else 0
            if n_m == 0:
                continue
            m = mm - 1
            sums[2] += n_m * q ** m * (1 - 2 * m * eps / q + Fraction(m * (m - 1), 2) * eps ** 2 / q ** 2)
            sums[3] += n_m * q ** m * (1 - Fraction(27, 8) * m * eps / q + Fraction(9, 8) * m * (m - 1) * eps ** 2 / q ** 2)
            sums[4] += n_m * q ** m * (1 - 9 * m * eps / q + 8 * m * (m - 1) * eps ** 2 / q ** 2
                                       - Fraction(4, 3) * m * (m - 1) * (m - 2) * eps ** 3 / q ** 3)
        e = float(eps)
        want = {2: float(2 * eps * (N - 2 * eps * sums[2])),
                3: (1 / math.gamma(5 / 3)) * (math.pi * e / (3 * math.sqrt(2))) ** (2 / 3) * float(N - eps * sums[3]),
                4: 4 * math.sqrt(e / 6) * float(N - eps * sums[4])}
        for dim in (2, 3, 4):
            got = oracle.smeared_action(hist, N, dim, e)
            assert got == pytest.approx(want[dim], rel=1e-11, abs=1e-9), (dim, eps)


def test_seh_golden():
    eta0, printed, _ = _read_table("ds_slab_seh.txt")[0]
    assert round(4 * math.pi * math.tan(float(eta0)), 3) == float(printed)


def test_degrees_helper(oracle):
    coords = inp.sprinkle(inp.GEOM_MINK_CONE, 3, 333, 21)
    C = oracle.causal_matrix_bytes(coords, inp.GEOM_MINK_CONE)
    o, i = oracle.degrees(oracle.pack_bytes(C), 333)
    assert np.array_equal(o, C.sum(axis=1)) and np.array_equal(i, C.sum(axis=0))


def test_flrw_polar_relation(oracle):
    """Eq. 7.7: hand cases (law of cosines along one ray, opposite rays, the null
    pair is NOT related -- the paper's strict '<'), and agreement with the flat cone in Cartesian
    coordinates for every pair away from the cone (FLRW is conformally flat)."""
    def pt(eta, r, th, ph):
        return np.array([eta, r, math.cos(th), math.sin(th), math.cos(ph), math.sin(ph)])
    g = oracle.GEOM_FLRW_POLAR
    assert oracle.relation(pt(0.0, 0.5, 0.3, 1.0), pt(0.25, 0.7, 0.3, 1.0), g)          # same ray: |dr| = 0.2 < 0.25
    assert not oracle.relation(pt(0.0, 0.5, 0.3, 1.0), pt(0.15, 0.7, 0.3, 1.0), g)      # 0.2 > 0.15
    assert not oracle.relation(pt(0.25, 0.7, 0.3, 1.0), pt(0.0, 0.5, 0.3, 1.0), g)      # time order
    assert oracle.relation(pt(0.0, 0.25, 0.0, 0.0), pt(0.625, 0.25, math.pi, 0.0), g)   # opposite poles: 0.5 < 0.625
    assert not oracle.relation(pt(0.0, 0.25, 0.0, 0.0), pt(0.5, 0.25, math.pi, 0.0), g) # null: strict
    assert not oracle.relation(pt(0.0, 0.0, 0.0, 0.0), pt(0.0, 0.0, 0.0, 0.0), g)       # same event
    N = 400
    c = inp.sprinkle_flrw_polar(N, 12)
    assert np.all(np.diff(c[:, 0]) >= 0) and np.allclose(c[:, 2] ** 2 + c[:, 3] ** 2, 1) and np.allclose(c[:, 4] ** 2 + c[:, 5] ** 2, 1)
    C = oracle.causal_matrix_bytes(c, g)
    x = c[:, 1] * c[:, 3] * c[:, 4]; y = c[:, 1] * c[:, 3] * c[:, 5]; z = c[:, 1] * c[:, 2]
    dt = c[None, :, 0] - c[:, None, 0]
    q = dt ** 2 - ((x[None] - x[:, None]) ** 2 + (y[None] - y[:, None]) ** 2 + (z[None] - z[:, None]) ** 2)
    want = np.triu((dt > 0) & (q > 0), 1)
    clear = np.triu(np.abs(q) > 1e-12, 1)
    assert np.array_equal(C.astype(bool)[clear], want[clear]) and 0.02 < want.mean() < 0.4
    # transitive and acyclic like every other geometry
    Cb = C.astype(bool)
    assert not (Cb.astype(np.int32) @ Cb.astype(np.int32) > 0)[~Cb & np.triu(np.ones_like(Cb), 1)].any()
    # the action pipeline treats it as 3+1 dimensional
    _, hist, S, I = oracle.action_pipeline(c, g)
    assert I == N - hist[0] + 9 * hist[1] - 16 * hist[2] + 8 * hist[3]


# ----------------------------------------------------------------------------- NEXT-4: the other App. A regions
def test_cone_in_five_dimensions(oracle):
    """4+1 flat cone: hand cases incl. the null pair (related, reading A1) and the fourth spatial
    coordinate really entering; numpy re-evaluation of the squared form on a 4+1 diamond; the ordering fraction of
    the d-dimensional diamond falls with d (soft check that a coordinate was not dropped)."""
    g = inp.GEOM_MINK_CONE
    assert oracle.relation([0, 0, 0, 0, 0], [1.0, 0.5, 0.5, 0.5, 0.5], g)           # 1 >= 1: null
    assert not oracle.relation([0, 0, 0, 0, 0], [1.0, 0.5, 0.5, 0.5, 0.51], g)
    assert oracle.relation([0, 0, 0, 0, 0], [1.0, 0, 0, 0, 0.99], g)
    assert not oracle.relation([0, 0, 0, 0, 0], [1.0, 0, 0, 0, 1.01], g)            # only w decides
    assert not oracle.relation([1.0, 0, 0, 0, 0], [0, 0, 0, 0, 0], g)
    N = 500
    c = inp.sprinkle(g, 5, N, 31)
    assert c.shape == (N, 5) and np.all(np.diff(c[:, 0]) >= 0)
    assert np.all(np.abs(c[:, 0]) + np.sqrt((c[:, 1:] ** 2).sum(axis=1)) <= 1.0)
    C = oracle.causal_matrix_bytes(c, g).astype(bool)
    d = c[None, :, :] - c[:, None, :]
    s = np.zeros((N, N))
    for a in range(1, 5):
        s = s + d[:, :, a] * d[:, :, a]
    assert np.array_equal(C, np.triu((d[:, :, 0] >= 0) & (d[:, :, 0] ** 2 >= s), 1))
    frac = {dim: oracle.causal_matrix_bytes(inp.sprinkle(g, dim, 600, 7), g).sum() / (600 * 599 / 2) for dim in (2, 3, 4, 5)}
    assert frac[2] > frac[3] > frac[4] > frac[5] > 0.01
    bits, hist, S, I = oracle.action_pipeline(c, g)                                  # no action printed for d = 5
    assert S is None and hist.sum() == C.sum()


def _ds4_point(eta, psi, th, ph):
    sp = math.sin(psi)
    return np.array([eta, math.cos(eta), math.sin(eta), math.cos(psi), sp * math.cos(th),
                     sp * math.sin(th) * math.cos(ph), sp * math.sin(th) * math.sin(ph)])


def test_ds4_spherical_relation(oracle):
    """3+1 de Sitter, spherical foliation (d eta^2 > d Sigma^2).  Hand cases; the
    arccos form of the great-circle distance away from the cone; on a great circle of the 3-sphere the relation is
    the 1+1 slab's periodic one (GEOM_DS2_SLAB, strictness aside); transitivity; the sprinkler's marginals."""
    g = inp.GEOM_DS4_SPHERICAL
    assert oracle.relation(_ds4_point(0.1, 1.0, 1.0, 1.0), _ds4_point(0.2, 1.0, 1.0, 1.0), g)        # same place, later
    assert not oracle.relation(_ds4_point(0.2, 1.0, 1.0, 1.0), _ds4_point(0.1, 1.0, 1.0, 1.0), g)    # time order
    assert not oracle.relation(_ds4_point(0.2, 1.0, 1.0, 1.0), _ds4_point(0.2, 1.0, 1.0, 1.0), g)    # same event
    assert oracle.relation(_ds4_point(0.0, 0.5, 1.0, 1.0), _ds4_point(0.31, 0.8, 1.0, 1.0), g)       # d psi = 0.3 < 0.31
    assert not oracle.relation(_ds4_point(0.0, 0.5, 1.0, 1.0), _ds4_point(0.29, 0.8, 1.0, 1.0), g)
    assert not oracle.relation(_ds4_point(0.0, 0.1, 0.0, 0.0), _ds4_point(1.4, math.pi - 0.1, 0.0, 0.0), g)  # nearly antipodal
    rng = np.random.default_rng(3)
    n = 0
    for _ in range(3000):
        e1, e2 = np.sort(rng.uniform(0.0, 1.3, 2))
        a = (rng.uniform(0, np.pi), rng.uniform(0, np.pi), rng.uniform(0, 2 * np.pi))
        b = (rng.uniform(0, np.pi), rng.uniform(0, np.pi), rng.uniform(0, 2 * np.pi))
        p, q = _ds4_point(e1, *a), _ds4_point(e2, *b)
        omega = math.acos(max(-1.0, min(1.0, float(p[3:] @ q[3:]))))
        if abs(omega - (e2 - e1)) < 1e-9:
            continue
        n += 1
        assert oracle.relation(p, q, g) == (e2 - e1 > omega)
    assert n > 2900
    # a great circle: psi = th = pi/2, phi free -> the relation of the 1+1 slab on (eta, phi)
    for _ in range(2000):
        e1, e2 = np.sort(rng.uniform(0.0, 1.3, 2))
        f1, f2 = rng.uniform(0, 2 * np.pi, 2)
        d = min(abs(f1 - f2), 2 * np.pi - abs(f1 - f2))
        if abs(d - (e2 - e1)) < 1e-9:
            continue
        assert oracle.relation(_ds4_point(e1, np.pi / 2, np.pi / 2, f1), _ds4_point(e2, np.pi / 2, np.pi / 2, f2), g) == \
            oracle.relation([e1, f1], [e2, f2], inp.GEOM_DS2_SLAB)
    N = 600
    c = inp.sprinkle(g, 7, N, 17)
    assert np.all(np.diff(c[:, 0]) >= 0) and np.allclose((c[:, 3:] ** 2).sum(axis=1), 1) and np.allclose(c[:, 1] ** 2 + c[:, 2] ** 2, 1)
    C = oracle.causal_matrix_bytes(c, g).astype(bool)
    assert np.array_equal(C, np.triu(C, 1)) and 0.005 < C.sum() / (N * (N - 1) / 2) < 0.6
    assert not (C.astype(np.int32) @ C.astype(np.int32) > 0)[~C & np.triu(np.ones_like(C), 1)].any()
    _, hist, S, I = oracle.action_pipeline(c, g)                                     # a 3+1 dimensional spacetime
    assert I == N - hist[0] + 9 * hist[1] - 16 * hist[2] + 8 * hist[3]
    # marginals of the sprinkler: E[sin^2 psi] = 3/4 under (2/pi) sin^2 psi, E[cos th] = 0
    big = inp.sprinkle_ds4_spherical(20000, 5)
    assert abs((1 - big[:, 3] ** 2).mean() - 0.75) < 0.01 and abs(big[:, 4].mean()) < 0.02
    assert big[:, 0].min() >= 0 and big[:, 0].max() <= 1.0 and np.median(big[:, 0]) > 0.7     # sec^4: late times dominate


def test_appendix_a_sprinklers(oracle):
    """The remaining flat / FLRW regions are sprinklers over predicates already pinned: the 1+1 square and the paper's
    own inverse-CDF 2+1 diamond feed the flat cone, the 1+1 cylinder the periodic relation, the dust slab Eq. 7.7 in
    conformal time.  Checks: region bounds, time order, the 2+1 diamond's radial law, and that the dust slab's
    relation agrees with the flat cone in Cartesian conformal coordinates."""
    sq = inp.sprinkle_mink2_square(500, 3, t0=0.5, x0=2.0)
    assert np.all(np.abs(sq[:, 0]) <= 0.5) and np.all(np.abs(sq[:, 1]) <= 2.0) and np.all(np.diff(sq[:, 0]) >= 0)
    cy = inp.sprinkle_mink2_cylinder(500, 4)
    assert np.all((cy[:, 1] >= 0) & (cy[:, 1] < 2 * np.pi)) and np.all(np.diff(cy[:, 0]) >= 0)
    C = oracle.causal_matrix_bytes(cy, inp.GEOM_DS2_SLAB)
    d = np.abs(cy[None, :, 1] - cy[:, None, 1]); d = np.minimum(d, 2 * np.pi - d)
    assert np.array_equal(C.astype(bool), np.triu((cy[None, :, 0] - cy[:, None, 0]) >= d, 1))
    di = inp.sprinkle_mink3_diamond_uv(20000, 5)
    t, r = di[:, 0], np.hypot(di[:, 1], di[:, 2])
    u, v = (t + r) / np.sqrt(2), (t - r) / np.sqrt(2)
    assert np.all(u <= 1 + 1e-12) and np.all(v >= -1e-12) and np.all(v <= u + 1e-12)
    assert abs((u ** 3).mean() - 0.5) < 0.01                  # u* = u^(1/3): u*^3 is uniform
    du = inp.sprinkle_dust_slab(400, 6)
    assert np.all(np.diff(du[:, 0]) >= 0) and np.all(du[:, 1] <= 0.5)
    C = oracle.causal_matrix_bytes(du, inp.GEOM_FLRW_POLAR).astype(bool)
    x = du[:, 1] * du[:, 3] * du[:, 4]; y = du[:, 1] * du[:, 3] * du[:, 5]; z = du[:, 1] * du[:, 2]
    dt = du[None, :, 0] - du[:, None, 0]
    q = dt ** 2 - ((x[None] - x[:, None]) ** 2 + (y[None] - y[:, None]) ** 2 + (z[None] - z[:, None]) ** 2)
    clear = np.triu(np.abs(q) > 1e-12, 1)
    assert np.array_equal(C[clear], np.triu((dt > 0) & (q > 0), 1)[clear]) and C.sum() > 1000


def _cdf_close(sample, cdf, lo, hi, tol):
    qs = np.linspace(lo, hi, 12)[1:-1]
    emp = np.array([(sample < q).mean() for q in qs])
    assert np.max(np.abs(emp - cdf(qs))) < tol, (emp, cdf(qs))


def test_appendix_a_de_sitter_and_dust_lambda_sprinklers(oracle):
    """The de Sitter diamonds / flat slab and the dust + dark energy slab: every
    recipe is checked against the density the paper states for it (marginal and conditional CDFs in closed form),
    and the conformal time of Eq. 7.5 against a direct quadrature of d tau / a."""
    n = 60000
    # 1+1 dS diamond, flat foliation: rho(u, v) ~ 1 / (u + v)^2 on [u0, u0 + w]^2
    w = 0.5; u0 = v0 = -1 / np.sqrt(2)
    c = inp.sprinkle_ds2_diamond_flat(n, 3, w)
    assert c[:, 0].min() >= u0 - 1e-12 and c[:, 0].max() <= u0 + w + 1e-12 and c[:, 1].min() >= v0 - 1e-12 and c[:, 1].max() <= v0 + w + 1e-12
    g = lambda x: np.log(np.abs(x + v0)) - np.log(np.abs(x + v0 + w))
    _cdf_close(c[:, 0], lambda q: (g(q) - g(u0)) / (g(u0 + w) - g(u0)), u0, u0 + w, 0.01)
    band = (c[:, 0] > u0 + 0.2) & (c[:, 0] < u0 + 0.25); um = c[band, 0].mean()
    _cdf_close(c[band, 1], lambda q: (1 / (um + v0) - 1 / (um + q)) / (1 / (um + v0) - 1 / (um + v0 + w)), v0, v0 + w, 0.03)
    # 1+1 dS diamond, spherical foliation: rho ~ sec^2((u + v) / sqrt 2) on [0, w0]^2 (reading A20)
    w0 = 0.8; s2 = np.sqrt(2)
    c = inp.sprinkle_ds2_diamond_spherical(n, 4, w0)
    assert c.min() >= -1e-12 and c.max() <= w0 + 1e-12
    G = lambda x: -np.log(np.cos((x + w0) / s2)) + np.log(np.cos(x / s2))
    _cdf_close(c[:, 0], lambda q: (G(q) - G(0)) / (G(w0) - G(0)), 0, w0, 0.01)
    band = (c[:, 0] > 0.3) & (c[:, 0] < 0.33); um = c[band, 0].mean()
    _cdf_close(c[band, 1], lambda q: (np.tan((um + q) / s2) - np.tan(um / s2)) / (np.tan((um + w0) / s2) - np.tan(um / s2)), 0, w0, 0.03)
    # both feed the light-cone relation: sorted by time, transitive
    C = oracle.causal_matrix_bytes(c[:400], inp.GEOM_MINK2_LIGHTCONE).astype(bool)
    assert not (C.astype(np.int32) @ C.astype(np.int32) > 0)[~C & np.triu(np.ones_like(C), 1)].any()
    # 3+1 dS slab, flat foliation: rho(eta) ~ eta^-4 on [-1, eta0]
    e0 = -0.25
    c = inp.sprinkle_ds4_flat_slab(n, 5, e0, 0.6)
    assert c[:, 0].min() >= -1 - 1e-12 and c[:, 0].max() <= e0 + 1e-12 and np.all(np.diff(c[:, 0]) >= 0)
    _cdf_close(c[:, 0], lambda q: (-q ** -3 - 1) / (-e0 ** -3 - 1), -1, e0, 0.01)
    _cdf_close(c[:, 1] ** 3, lambda q: q / 0.6 ** 3, 0, 0.6 ** 3, 0.01)
    # dust + dark energy: tau from (sinh 3 tau - 3 tau), eta by Eq. 7.5 = integral of d tau / sinh^(2/3)(3 tau / 2)
    from scipy.integrate import quad
    c = inp.sprinkle_dust_lambda_slab(4000, 6, 1.0, 0.5)
    assert np.all(np.diff(c[:, 0]) >= 0) and c[:, 1].max() <= 0.5
    for tau in (0.2, 0.7, 1.0):
        sh = np.sinh(1.5 * tau)
        from scipy.special import hyp2f1
        eta = 2 * np.cbrt(sh) * hyp2f1(1 / 6, 0.5, 7 / 6, -sh * sh)
        assert eta == pytest.approx(quad(lambda t: np.sinh(1.5 * t) ** (-2 / 3), 0, tau)[0], rel=1e-6)
    eta_max = 2 * np.cbrt(np.sinh(1.5)) * hyp2f1(1 / 6, 0.5, 7 / 6, -np.sinh(1.5) ** 2)
    assert 0 < c[:, 0].min() and c[:, 0].max() <= eta_max + 1e-12
    C = oracle.causal_matrix_bytes(c[:500], inp.GEOM_FLRW_POLAR)
    assert C.sum() > 0


def test_appendix_a_diamonds_3p1(oracle):
    """The last three regions of App. A.1: 3+1 dS diamonds (flat and spherical foliation) and the
    3+1 dust diamond.  The printed inverse CDFs are garbled in the extracted text (DESIGN.md
    reading A23); the sprinklers invert the CDFs of the STATED densities, so the pins are those densities integrated
    numerically (scipy quadrature, nothing shared with the sprinklers' closed forms), the paper's printed volumes /
    normalisations (mu of PAPER.md:3889 and 3933, 1981/5940 of PAPER.md:3961), the regions, and the relation they feed."""
    from scipy.integrate import dblquad, quad
    n = 60000
    s2 = np.sqrt(2.0)

    def check(uv, dens, ulo, uhi, vlo, total, tol=0.012):
        u, v = uv
        assert np.all(u >= ulo - 1e-12) and np.all(u <= uhi + 1e-12) and np.all(v >= vlo - 1e-12) and np.all(v <= u + 1e-12)
        for q in np.linspace(ulo, uhi, 7)[1:-1]:                   # marginal CDF of u
            want = dblquad(lambda vv, uu: dens(uu, vv), ulo, q, lambda uu: vlo, lambda uu: uu)[0] / total
            assert abs((u < q).mean() - want) < tol, (q, (u < q).mean(), want)
        lo_q, hi_q = np.quantile(u, [0.50, 0.54])                   # conditional CDF of v in a thin band of u (2400 points)
        band = (u > lo_q) & (u < hi_q)
        um = u[band].mean()
        den = quad(lambda vv: dens(um, vv), vlo, um)[0]
        for q in np.linspace(vlo, um, 6)[1:-1]:
            want = quad(lambda vv: dens(um, vv), vlo, q)[0] / den
            assert abs((v[band] < q).mean() - want) < 0.04, (q, (v[band] < q).mean(), want)

    # flat foliation: rho ~ (u - v)^2 / (u + v)^4, total = mu / 6
    w, u0 = 0.5, -1 / s2
    dens = lambda u, v: (u - v) ** 2 / (u + v) ** 4
    total = dblquad(lambda vv, uu: dens(uu, vv), u0, u0 + w, lambda uu: u0, lambda uu: uu)[0]
    assert inp.ds4_diamond_flat_mu(w, u0) / 6 == pytest.approx(total, rel=1e-9)
    c = inp.sprinkle_ds4_diamond_flat(n, 3, w)
    assert np.all(np.diff(c[:, 0]) >= 0) and c[:, 0].max() < 0 and c[:, 1].min() >= 0
    check(((c[:, 0] + c[:, 1]) / s2, (c[:, 0] - c[:, 1]) / s2), dens, u0, u0 + w, u0, total)
    assert abs(c[:, 2].mean()) < 0.01 and np.allclose(c[:, 2] ** 2 + c[:, 3] ** 2, 1) and np.allclose(c[:, 4] ** 2 + c[:, 5] ** 2, 1)

    # spherical foliation: rho ~ sec^4((u + v)/sqrt 2) sin^2((u - v)/sqrt 2), total = mu / 3
    w0 = 0.8
    dens = lambda u, v: np.sin((u - v) / s2) ** 2 / np.cos((u + v) / s2) ** 4
    total = dblquad(lambda vv, uu: dens(uu, vv), 0, w0, lambda uu: 0, lambda uu: uu)[0]
    mu = np.log(0.5 * (1 + 1 / np.cos(s2 * w0))) - 1 / np.cos(w0 / s2) ** 2 + 1
    assert mu / 3 == pytest.approx(total, rel=1e-9)
    c = inp.sprinkle_ds4_diamond_spherical(n, 4, w0)
    eta = c[:, 0]
    psi = np.arccos(np.clip(c[:, 3], -1, 1))
    assert np.all(np.diff(eta) >= 0) and np.allclose(c[:, 1], np.cos(eta)) and np.allclose(c[:, 2], np.sin(eta))
    assert np.allclose((c[:, 3:] ** 2).sum(axis=1), 1)
    check(((eta + psi) / s2, (eta - psi) / s2), dens, 0, w0, 0, total)

    # dust: rho = 5940 / (1981 u0^12) (u + v)^8 (u - v)^2
    dens = lambda u, v: (u + v) ** 8 * (u - v) ** 2
    total = dblquad(lambda vv, uu: dens(uu, vv), 0, 1, lambda uu: 0, lambda uu: uu)[0]
    assert total == pytest.approx(1981 / 5940, rel=1e-9)
    c = inp.sprinkle_dust_diamond(n, 5, 1.0)
    assert np.all(np.diff(c[:, 0]) >= 0)
    check(((c[:, 0] + c[:, 1]) / s2, (c[:, 0] - c[:, 1]) / s2), dens, 0, 1.0, 0, total)

    # each feeds a predicate that is already pinned: upper triangular, transitive, a non-trivial relation density
    for cc, g in ((inp.sprinkle_ds4_diamond_flat(400, 7), inp.GEOM_FLRW_POLAR),
                  (inp.sprinkle_ds4_diamond_spherical(400, 8), inp.GEOM_DS4_SPHERICAL),
                  (inp.sprinkle_dust_diamond(400, 9), inp.GEOM_FLRW_POLAR)):
        C = oracle.causal_matrix_bytes(cc, g).astype(bool)
        assert np.array_equal(C, np.triu(C, 1)) and 0.02 < C.sum() / (400 * 399 / 2) < 0.9
        assert not (C.astype(np.int32) @ C.astype(np.int32) > 0)[~C & np.triu(np.ones_like(C), 1)].any()
