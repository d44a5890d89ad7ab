"""Parity of the CUDA path (through the C ABI) with the oracle -- bit-exact.

Run on the B200 box:  python -m pytest tests -m gpu -x -q
Every input is seeded and synthetic (paper_1805_04463_b200.inputs); nothing
reads /root/reference at run time.
"""
import numpy as np
import pytest

torch = pytest.importorskip("torch")

from paper_1805_04463_b200 import inputs as inp  # noqa: E402

pytestmark = pytest.mark.gpu

GEOMS = [
    (inp.GEOM_MINK2_LIGHTCONE, 2),
    (inp.GEOM_MINK_CONE, 2),
    (inp.GEOM_MINK_CONE, 3),
    (inp.GEOM_MINK_CONE, 4),
    (inp.GEOM_DS2_SLAB, 2),
    (inp.GEOM_FLRW_POLAR, 6),          # NEXT-4: Eq. 7.7
    (inp.GEOM_MINK_CONE, 5),           # NEXT-4: 4+1 diamond
    (inp.GEOM_DS4_SPHERICAL, 7),       # NEXT-4: 3+1 de Sitter, spherical foliation
]


@pytest.fixture(scope="module")
def api():
    if not torch.cuda.is_available():
        pytest.fail("gpu tests need a CUDA device")
    from paper_1805_04463_b200 import api as _api
    _api.load()
    torch.cuda.set_device(0)
    return _api


ALL_ROUTES = ("ROUTE_POPC", "ROUTE_TENSOR", "ROUTE_TENSOR_FP4", "ROUTE_TENSOR_PAIR")


def routes(api):
    """Every concrete a2 route.  On a compute-capability 10.x device all four must launch: a tensor route that
    stops working fails the test that asked for it instead of quietly leaving the list."""
    major, _ = torch.cuda.get_device_capability()
    if major != 10:
        pytest.fail("the tensor routes need an sm_100 device (found compute capability %d.x)" % major)
    r = []
    for name in ALL_ROUTES:
        cand = getattr(api, name)
        x = torch.zeros((128, 2), dtype=torch.int64, device="cuda")
        try:
            api.interval_hist(x, x, 128, route=cand)
        except RuntimeError as e:
            pytest.fail("a2 route %s does not launch on this device: %s" % (name, e))
        r.append(cand)
    return r


def to_u64(t):
    return t.cpu().numpy().view(np.uint64)


# every predicate is the sign of a bilinear form, some in derived coordinates (cs_build_tc.cu)
TENSOR_A1_GEOMS = (inp.GEOM_MINK2_LIGHTCONE, inp.GEOM_MINK_CONE, inp.GEOM_DS2_SLAB, inp.GEOM_FLRW_POLAR, inp.GEOM_DS4_SPHERICAL)


def a1_routes(api, geom, N):
    """Every concrete a1 route that serves this geometry and size (the tensor route wants rows of >= 32 bytes)."""
    r = [api.A1_FMA]
    if geom in TENSOR_A1_GEOMS and N >= 256:
        r.append(api.A1_TENSOR)
    return r


def gpu_bits(api, coords, geom):
    """The library's default a1 route -- and, asserted bit-identical to it, every other route that serves the geometry,
    so that each a1 test compares all of them with the oracle."""
    d = torch.from_numpy(np.ascontiguousarray(coords)).cuda()
    bits, bitsT = api.causal_matrix(d, geom)
    for route in a1_routes(api, geom, coords.shape[0]):
        b, t = api.causal_matrix(d, geom, route=route)
        assert torch.equal(b, bits) and torch.equal(t, bitsT), "a1 route %d differs from the default route" % route
    torch.cuda.synchronize()
    return bits, bitsT


# ----------------------------------------------------------------------------- a1
@pytest.mark.parametrize("geom,dim", GEOMS)
@pytest.mark.parametrize("N", [1, 2, 63, 64, 65, 255, 256, 257, 1000, 1024, 3001])
def test_causal_matrix_bit_exact(api, oracle, geom, dim, N):
    coords = inp.sprinkle(geom, dim, N, 100 + N + dim)
    o_bits = oracle.causal_matrix_bits(coords, geom)
    bits, bitsT = gpu_bits(api, coords, geom)
    assert np.array_equal(to_u64(bits), o_bits)
    assert np.array_equal(to_u64(bitsT), oracle.transpose_bits(o_bits, N))
    # bits-only call, then the stand-alone transpose
    d = torch.from_numpy(coords).cuda()
    b2, none = api.causal_matrix(d, geom, want_transpose=False)
    assert none is None and torch.equal(b2, bits)
    assert torch.equal(api.transpose_bits(b2, N), bitsT)


def test_causal_matrix_near_null_pairs(api, oracle):
    """Pairs exactly on and one ulp either side of the light cone decide identically."""
    rng = np.random.default_rng(1)
    base = rng.uniform(-0.5, 0.5, (200, 4))
    base[:, 0] = np.sort(rng.uniform(-1, 0, 200))
    fut = base.copy()
    r = np.sqrt((rng.uniform(0.1, 0.4, (200, 3)) ** 2).sum(axis=1))
    dx = rng.normal(size=(200, 3))
    dx = dx / np.linalg.norm(dx, axis=1)[:, None] * r[:, None]
    fut[:, 1:] = base[:, 1:] + dx
    fut[:, 0] = base[:, 0] + r                      # (nearly) null separated partners
    fut2 = fut.copy(); fut2[:, 0] = np.nextafter(fut[:, 0], 10.0)
    fut3 = fut.copy(); fut3[:, 0] = np.nextafter(fut[:, 0], -10.0)
    coords = np.concatenate([base, fut, fut2, fut3])
    coords = coords[np.lexsort((coords[:, 1], coords[:, 0]))]
    o_bits = oracle.causal_matrix_bits(coords, inp.GEOM_MINK_CONE)
    bits, _ = gpu_bits(api, coords, inp.GEOM_MINK_CONE)
    assert np.array_equal(to_u64(bits), o_bits)


def _near_null_set(rng, n, dim):
    """n base points and, for each, partners on the cone and one ulp either side of it (time-sorted)."""
    base = rng.uniform(-0.5, 0.5, (n, dim))
    base[:, 0] = rng.uniform(-1, 0, n)
    r = rng.uniform(0.05, 0.6, n)
    dx = rng.normal(size=(n, dim - 1))
    dx = dx / np.linalg.norm(dx, axis=1)[:, None] * r[:, None]
    fut = base.copy()
    fut[:, 1:] = base[:, 1:] + dx
    fut[:, 0] = base[:, 0] + np.sqrt((dx ** 2).sum(axis=1))
    fut2 = fut.copy(); fut2[:, 0] = np.nextafter(fut[:, 0], 10.0)
    fut3 = fut.copy(); fut3[:, 0] = np.nextafter(fut[:, 0], -10.0)
    coords = np.concatenate([base, fut, fut2, fut3])
    return np.ascontiguousarray(coords[np.lexsort((coords[:, 1], coords[:, 0]))])


@pytest.mark.parametrize("dim", [2, 3, 4, 5])
@pytest.mark.parametrize("scale", [1.0, 2.0 ** 30, 2.0 ** -30, 2.0 ** 45, 2.0 ** -45, 2.0 ** 600, 2.0 ** -600])
def test_causal_matrix_prefilter_bands(api, oracle, dim, scale):
    """The single-precision prefilter of the flat cone never decides a pair the fp64 expression would
    decide differently: thousands of pairs within an ulp of the cone spread over many tiles, at
    coordinate scales inside and outside the prefilter's range (|x| in 2^-40 .. 2^40)."""
    rng = np.random.default_rng(7 + dim)
    coords = _near_null_set(rng, 700, dim) * scale          # N = 2800: 11 tiles per side
    o_bits = oracle.causal_matrix_bits(coords, inp.GEOM_MINK_CONE)
    bits, bitsT = gpu_bits(api, coords, inp.GEOM_MINK_CONE)
    assert np.array_equal(to_u64(bits), o_bits)
    assert np.array_equal(to_u64(bitsT), oracle.transpose_bits(o_bits, coords.shape[0]))


def test_causal_matrix_prefilter_unsorted_inf_nan(api, oracle):
    """Inputs that break the prefilter's preconditions fall back to the fp64 expression: elements not
    sorted by time (dt < 0 must read unrelated), infinite and NaN coordinates, a tile of identical points."""
    rng = np.random.default_rng(11)
    N = 1500
    coords = inp.sprinkle(inp.GEOM_MINK_CONE, 4, N, 5)
    shuffled = np.ascontiguousarray(coords[rng.permutation(N)])
    weird = coords.copy()
    weird[300, 0] = np.inf; weird[301, 2] = -np.inf; weird[700, 0] = np.nan; weird[701, 3] = np.nan
    weird[900:1200] = weird[900]                            # more than one tile of identical points
    late = coords.copy(); late[5, 0] = 2.0                  # one element far out of time order
    for c in (shuffled, weird, late):
        o_bits = oracle.causal_matrix_bits(c, inp.GEOM_MINK_CONE)
        bits, bitsT = gpu_bits(api, c, inp.GEOM_MINK_CONE)
        assert np.array_equal(to_u64(bits), o_bits)
        assert np.array_equal(to_u64(bitsT), oracle.transpose_bits(o_bits, N))


def test_causal_matrix_prefilter_ds_slab(api, oracle):
    """The de Sitter slab's single-precision prefilter: partners exactly on the cone and one ulp either side,
    directly and through the 2 pi wrap-around, plus angles outside [0, 2 pi) and NaN / infinite coordinates."""
    rng = np.random.default_rng(21)
    n = 600
    eta = rng.uniform(-1.2, -0.4, n); th = rng.uniform(0, 2 * np.pi, n)
    d = rng.uniform(0.01, 0.35, n)
    base = np.stack([eta, th], axis=1)
    fwd = np.stack([eta + d, th + d], axis=1)                       # null, same side
    wrap = np.stack([eta + d, np.mod(th - d, 2 * np.pi)], axis=1)   # null, may cross theta = 0
    sets = [base]
    for p in (fwd, wrap):
        for k in (0.0, 10.0, -10.0):
            q = p.copy()
            if k:
                q[:, 0] = np.nextafter(p[:, 0], k)
            sets.append(q)
    coords = np.concatenate(sets)
    coords = np.ascontiguousarray(coords[np.lexsort((coords[:, 1], coords[:, 0]))])
    N = coords.shape[0]
    for variant in range(3):
        c = coords.copy()
        if variant == 1:
            c[:, 1] += 100.0                                        # angles far outside [0, 2 pi)
        if variant == 2:
            c[7, 1] = np.nan; c[300, 0] = np.inf; c[900, 1] = -np.inf; c[1500:1900] = c[1500]
        o_bits = oracle.causal_matrix_bits(c, inp.GEOM_DS2_SLAB)
        bits, bitsT = gpu_bits(api, c, inp.GEOM_DS2_SLAB)
        assert np.array_equal(to_u64(bits), o_bits), variant
        assert np.array_equal(to_u64(bitsT), oracle.transpose_bits(o_bits, N)), variant
    shuffled = np.ascontiguousarray(coords[rng.permutation(N)])     # not time-sorted: d_eta < 0 pairs
    assert np.array_equal(to_u64(gpu_bits(api, shuffled, inp.GEOM_DS2_SLAB)[0]),
                          oracle.causal_matrix_bits(shuffled, inp.GEOM_DS2_SLAB))


def test_causal_matrix_prefilter_ds4_spherical(api, oracle):
    """The bilinear prefilter of the 3+1 de Sitter predicate (cos omega - cos d eta): partners displaced along a great
    circle by exactly d eta and one ulp either side of it, equal times, NaN / infinite / non-unit inputs, unsorted input."""
    rng = np.random.default_rng(31)
    n = 500

    def pts(eta, psi, th, ph):
        sp = np.sin(psi)
        return np.stack([eta, np.cos(eta), np.sin(eta), np.cos(psi), sp * np.cos(th), sp * np.sin(th) * np.cos(ph),
                         sp * np.sin(th) * np.sin(ph)], axis=1)
    eta = rng.uniform(0.0, 0.9, n); psi = rng.uniform(0.2, 2.0, n); th = rng.uniform(0.2, 2.9, n); ph = rng.uniform(0, 6.28, n)
    d = rng.uniform(0.01, 0.4, n)
    sets = [pts(eta, psi, th, ph)]
    for k in (0.0, 10.0, -10.0):
        e2 = eta + d
        if k:
            e2 = np.nextafter(e2, k)
        sets.append(pts(e2, psi + d, th, ph))               # same meridian: omega = d
    sets.append(pts(eta, psi + 0.3, th, ph))                # equal times: never related
    coords = np.concatenate(sets)
    coords = np.ascontiguousarray(coords[np.lexsort((coords[:, 3], coords[:, 0]))])
    N = coords.shape[0]
    for variant in range(7):
        c = coords.copy()
        if variant == 1:
            c[5, 3] = np.nan; c[300, 0] = np.inf; c[900, 4] = -np.inf; c[1200:1500] = c[1200]
        if variant == 2:
            c[:, 3:] *= 3.0                                 # not unit vectors: still the header's expression
        if variant == 3:
            c = np.ascontiguousarray(c[rng.permutation(N)])
        # eta enters the bilinear form through its cosine and sine columns only: whatever the time column itself
        # decides (d eta > 0, NaN differences) has to survive the prefilter of both a1 routes
        if variant == 4:                                    # NaN times, every other column still a valid unit vector
            c[[7, 129, 700, 1300, 2047, 2048, N - 1], 0] = np.nan
        if variant == 5:                                    # infinite times: inf - inf = NaN (unrelated), inf - finite > 0
            c[N - 40:, 0] = np.inf; c[:3, 0] = -np.inf
        if variant == 6:                                    # equal times whose (cos eta, sin eta) columns still differ
            c[1000:1400, 0] = c[1000, 0]; c[2040:2060, 0] = c[2040, 0]
        o_bits = oracle.causal_matrix_bits(c, inp.GEOM_DS4_SPHERICAL)
        if variant in (4, 5, 6):                            # the cases bite: the sign of T alone would relate such pairs
            C = oracle.unpack_bits(o_bits, N)
            rows = {4: [7, 129, 700, 1300, 2047, 2048, N - 1], 5: list(range(N - 40, N)), 6: list(range(1000, 1400))}[variant]
            ref = oracle.unpack_bits(oracle.causal_matrix_bits(coords, inp.GEOM_DS4_SPHERICAL), N)
            if variant == 4:                                # a NaN time is unrelated to everything, in both directions
                assert ref[rows].any() and ref[:, rows].any() and not C[rows].any() and not C[:, rows].any()
            else:
                assert ref[np.ix_(rows, rows)].any() and not C[np.ix_(rows, rows)].any()
        bits, bitsT = gpu_bits(api, c, inp.GEOM_DS4_SPHERICAL)
        assert np.array_equal(to_u64(bits), o_bits), variant
        assert np.array_equal(to_u64(bitsT), oracle.transpose_bits(o_bits, N)), variant


def test_causal_matrix_prefilter_flrw(api, oracle):
    """Eq. 7.7's prefilter runs on Cartesian conformal coordinates formed per point; it may only be used when the
    trigonometric inputs are unit vectors.  Near-null pairs along rays and across them, inputs whose (cos, sin) pairs
    are NOT normalised (the law-of-cosines value then differs from the Cartesian distance), NaN, unsorted."""
    rng = np.random.default_rng(41)
    base = inp.sprinkle_flrw_polar(900, 9)
    extra = base[:300].copy()
    extra[:, 0] = base[:300, 0] + 0.0625
    extra[:, 1] = base[:300, 1] + 0.0625                    # same ray, null separated
    e2 = extra.copy(); e2[:, 0] = np.nextafter(extra[:, 0], 10.0)
    e3 = extra.copy(); e3[:, 0] = np.nextafter(extra[:, 0], -10.0)
    coords = np.concatenate([base, extra, e2, e3])
    coords = np.ascontiguousarray(coords[np.lexsort((coords[:, 1], coords[:, 0]))])
    N = coords.shape[0]
    for variant in range(4):
        c = coords.copy()
        if variant == 1:
            c[::7, 2:4] *= 1.0 + 1e-6                       # cos^2 + sin^2 != 1 on every 7th point
        if variant == 2:
            c[:, 4:6] *= 0.5; c[11, 1] = np.nan; c[700, 0] = np.inf
        if variant == 3:
            c = np.ascontiguousarray(c[rng.permutation(N)])
        o_bits = oracle.causal_matrix_bits(c, inp.GEOM_FLRW_POLAR)
        bits, bitsT = gpu_bits(api, c, inp.GEOM_FLRW_POLAR)
        assert np.array_equal(to_u64(bits), o_bits), variant
        assert np.array_equal(to_u64(bitsT), oracle.transpose_bits(o_bits, N)), variant
    dust = inp.sprinkle_dust_slab(2500, 3)                  # App. A.1.4 through the same predicate
    assert np.array_equal(to_u64(gpu_bits(api, dust, inp.GEOM_FLRW_POLAR)[0]),
                          oracle.causal_matrix_bits(dust, inp.GEOM_FLRW_POLAR))


@pytest.mark.parametrize("geom,dim", [(g, d) for g, d in GEOMS if g in TENSOR_A1_GEOMS])
@pytest.mark.parametrize("N", [256, 257, 511, 1025, 2304, 3001])
def test_causal_matrix_tensor_route(api, oracle, geom, dim, N):
    """a1 on the tensor cores (CS_A1_TENSOR) against the oracle at sizes from one tile up: with the library's pool and with
    a caller's workspace, with and without the transposed output, and as a batch of ragged causets."""
    coords = inp.sprinkle(geom, dim, N, 300 + N + dim)
    o_bits = oracle.causal_matrix_bits(coords, geom)
    d = torch.from_numpy(coords).cuda()
    bits, bitsT = api.causal_matrix(d, geom, route=api.A1_TENSOR)
    assert np.array_equal(to_u64(bits), o_bits)
    assert np.array_equal(to_u64(bitsT), oracle.transpose_bits(o_bits, N))
    nbytes = api.causal_matrix_workspace(1, N, dim, geom, api.A1_TENSOR)
    assert nbytes > 0 and api.causal_matrix_workspace(1, N, dim, geom, api.A1_FMA) == 0
    ws = torch.empty(nbytes, dtype=torch.uint8, device="cuda")
    b2, t2 = api.causal_matrix(d, geom, route=api.A1_TENSOR, workspace=ws)
    assert torch.equal(b2, bits) and torch.equal(t2, bitsT)
    b3, none = api.causal_matrix(d, geom, want_transpose=False, route=api.A1_TENSOR)
    assert none is None and torch.equal(b3, bits)
    with pytest.raises(RuntimeError):      # a workspace that is too small is refused, not overrun
        api.causal_matrix(d, geom, route=api.A1_TENSOR, workspace=ws[:256])
    if N <= 1025:
        ens = np.stack([inp.sprinkle(geom, dim, N, 900 + b) for b in range(3)])
        eb, et = api.causal_matrix_batched(torch.from_numpy(ens).cuda(), geom, route=api.A1_TENSOR)
        for b in range(3):
            ob = oracle.causal_matrix_bits(ens[b], geom)
            assert np.array_equal(to_u64(eb[b]), ob) and np.array_equal(to_u64(et[b]), oracle.transpose_bits(ob, N))


def test_causal_matrix_tensor_route_arguments_and_probe(api, oracle):
    """The tensor route refuses what it does not serve; its probe reports an error of the tensor-core value far inside
    the margin, and rows re-evaluated in fp64 exactly where the input forces them (unsorted input: every row)."""
    assert api.a1_tensor_selfcheck() is True        # the device accumulates like the model: AUTO may take the tensor route
    small = torch.from_numpy(inp.sprinkle(inp.GEOM_MINK_CONE, 4, 100, 1)).cuda()
    with pytest.raises(RuntimeError):      # rows shorter than a TMA box
        api.causal_matrix(small, inp.GEOM_MINK_CONE, route=api.A1_TENSOR)
    with pytest.raises(RuntimeError):      # no such route
        api.causal_matrix(small, inp.GEOM_MINK_CONE, route=3)
    assert api.causal_matrix_workspace(1, 100, 4, inp.GEOM_MINK_CONE, api.A1_TENSOR) == 0
    assert api.default_a1_route(1, 1024, 2, inp.GEOM_MINK2_LIGHTCONE) == api.A1_FMA          # 10 tiles
    assert api.default_a1_route(1, 16384, 2, inp.GEOM_MINK2_LIGHTCONE) == api.A1_TENSOR
    assert api.default_a1_route(4096, 2048, 4, inp.GEOM_MINK_CONE) == api.A1_TENSOR
    for dim in (4, 5):
        coords = inp.sprinkle(inp.GEOM_MINK_CONE, dim, 3000, 17)
        o_bits = oracle.causal_matrix_bits(coords, inp.GEOM_MINK_CONE)
        bits, bitsT, st = api.a1_tensor_probe(torch.from_numpy(coords).cuda())
        assert np.array_equal(to_u64(bits), o_bits)
        assert np.array_equal(to_u64(bitsT), oracle.transpose_bits(o_bits, 3000))
        assert 0.0 < st["max_err_over_margin"] < 0.25 and 0.0 < st["max_acc_err_u"] < 64.0, st
        assert 0 < st["rows_fp64"] < st["rows_total"] / 10, st
        rng = np.random.default_rng(3)
        shuffled = np.ascontiguousarray(coords[rng.permutation(3000)])
        b2, _, st2 = api.a1_tensor_probe(torch.from_numpy(shuffled).cuda())
        assert np.array_equal(to_u64(b2), oracle.causal_matrix_bits(shuffled, inp.GEOM_MINK_CONE))
        assert st2["rows_fp64"] > 0.9 * st2["rows_total"], st2       # (only the tiles whose points happen to be ordered escape)


def test_causal_matrix_tensor_route_ds_slab_ranges(api, oracle):
    """The bilinear form of the 1+1 dS slab (cos dtheta - cos d eta) is the header's expression only while the angles of a
    tile span at most 2 pi and its times at most pi: slabs far wider than that, angles spread over many turns, and a
    sprinkling inside the valid range, all through every a1 route (gpu_bits)."""
    rng = np.random.default_rng(8)
    n = 1500
    for tspan, aspan in ((1.0, 2 * np.pi), (8.0, 2 * np.pi), (1.0, 40.0), (8.0, 40.0), (3.2, 6.4)):
        c = np.stack([rng.uniform(-1.2, -1.2 + tspan, n), rng.uniform(0.0, aspan, n)], axis=1)
        c = np.ascontiguousarray(c[np.lexsort((c[:, 1], c[:, 0]))])
        bits, bitsT = gpu_bits(api, c, inp.GEOM_DS2_SLAB)
        o_bits = oracle.causal_matrix_bits(c, inp.GEOM_DS2_SLAB)
        assert np.array_equal(to_u64(bits), o_bits), (tspan, aspan)
        assert np.array_equal(to_u64(bitsT), oracle.transpose_bits(o_bits, n)), (tspan, aspan)


def test_causal_matrix_tensor_route_degenerate(api, oracle):
    """Identical points (T = 0 for every pair: every row inside the band), NaN rows, huge and tiny scales mixed in one
    causet (the tile range test), all through CS_A1_TENSOR (gpu_bits checks every route)."""
    coords = np.zeros((600, 4)); coords[10:20, 1] = np.nan; coords[300:, 0] = 1.0
    assert np.array_equal(to_u64(gpu_bits(api, coords, inp.GEOM_MINK_CONE)[0]),
                          oracle.causal_matrix_bits(coords, inp.GEOM_MINK_CONE))
    mixed = inp.sprinkle(inp.GEOM_MINK_CONE, 4, 1200, 4)
    mixed[400:800] *= 2.0 ** 50; mixed[800:] *= 2.0 ** -50
    mixed = np.ascontiguousarray(mixed[np.lexsort((mixed[:, 1], mixed[:, 0]))])
    assert np.array_equal(to_u64(gpu_bits(api, mixed, inp.GEOM_MINK_CONE)[0]),
                          oracle.causal_matrix_bits(mixed, inp.GEOM_MINK_CONE))


@pytest.mark.parametrize("dim", [4, 5])
def test_causal_matrix_tensor_route_mixed_exponents(api, oracle, dim):
    """The tensor route's error band (reading A21) inside its accepted range 2^-40 .. 2^40 but with the exponents
    mixed within every tile: points scaled by 2^-15, 1 and 2^15 at random (the margin follows the largest addend of the
    tile while most pairs have a tiny T), and near-null pairs far from the origin, where |h_i|, |h_j| and the products
    are ~2^24 times the value they cancel to.  Every a1 route against the oracle (gpu_bits), and the probe's measured
    error stays inside the margin on such input."""
    rng = np.random.default_rng(50 + dim)
    n = 2600
    mixed = inp.sprinkle(inp.GEOM_MINK_CONE, dim, n, 70 + dim)
    mixed *= np.array([2.0 ** -15, 1.0, 2.0 ** 15])[rng.integers(0, 3, n)][:, None]
    mixed = np.ascontiguousarray(mixed[np.lexsort((mixed[:, 1], mixed[:, 0]))])
    far = _near_null_set(rng, 650, dim)                      # 2600 points: partners on the cone and one ulp off it
    far[:, 0] += 4096.0                                     # h = (t^2 - |x|^2) / 2 ~ 2^20 for every point
    far[:, 1] += 3900.0
    far = np.ascontiguousarray(far[np.lexsort((far[:, 1], far[:, 0]))])
    both = np.concatenate([mixed[: n // 2], far[: n // 2] * 2.0 ** 3])
    both = np.ascontiguousarray(both[np.lexsort((both[:, 1], both[:, 0]))])
    for c in (mixed, far, both):
        o_bits = oracle.causal_matrix_bits(c, inp.GEOM_MINK_CONE)
        bits, bitsT = gpu_bits(api, c, inp.GEOM_MINK_CONE)
        assert np.array_equal(to_u64(bits), o_bits)
        assert np.array_equal(to_u64(bitsT), oracle.transpose_bits(o_bits, c.shape[0]))
        b2, _, st = api.a1_tensor_probe(torch.from_numpy(c).cuda())
        assert np.array_equal(to_u64(b2), o_bits)
        assert st["max_err_over_margin"] < 0.5, st
        assert 0 < st["rows_fp64"] <= st["rows_total"], st


def test_causal_matrix_lightcone_ties(api, oracle):
    """1+1 light cone (two strict fp64 comparisons): coordinates that differ by one fp64 ulp, exact ties, values
    beyond the fp32 range, denormals and NaN.  (An fp32 prefilter was measured for this predicate too and
    dropped: two DSETP per pair are already cheaper than its set-up.)"""
    rng = np.random.default_rng(5)
    n = 500
    u = rng.uniform(0, 1, n); v = rng.uniform(0, 1, n)
    pts = [np.stack([u, v], 1)]
    for du, dv in ((1, 1), (1, 0), (0, 1), (-1, 1), (1, -1)):
        uu = u.copy(); vv = v.copy()
        for _ in range(abs(du)):
            uu = np.nextafter(uu, 2.0 * du)
        for _ in range(abs(dv)):
            vv = np.nextafter(vv, 2.0 * dv)
        pts.append(np.stack([uu, vv], 1))
    coords = np.concatenate(pts)
    for scale in (1.0, 1e300, 1e-300, 1e-42):
        c = coords * scale
        c = np.ascontiguousarray(c[np.lexsort((c[:, 0], (c[:, 0] + c[:, 1]) / 2))])
        if scale == 1.0:
            c[17, 0] = np.nan; c[400, 1] = np.inf; c[1000:1300] = c[1000]
        o_bits = oracle.causal_matrix_bits(c, inp.GEOM_MINK2_LIGHTCONE)
        bits, bitsT = gpu_bits(api, c, inp.GEOM_MINK2_LIGHTCONE)
        assert np.array_equal(to_u64(bits), o_bits), scale
        assert np.array_equal(to_u64(bitsT), oracle.transpose_bits(o_bits, c.shape[0])), scale


def test_degenerate_inputs(api, oracle):
    # identical points, NaN coordinates, N = 0
    coords = np.zeros((70, 4)); coords[10:20, 1] = np.nan
    o_bits = oracle.causal_matrix_bits(coords, inp.GEOM_MINK_CONE)
    bits, bitsT = gpu_bits(api, coords, inp.GEOM_MINK_CONE)
    assert np.array_equal(to_u64(bits), o_bits)
    for r in routes(api):
        h = api.interval_hist(bits, bitsT, 70, route=r)
        assert np.array_equal(h.cpu().numpy(), oracle.interval_hist_alg20(o_bits, 70)[0])
    empty = torch.zeros((0, 2), dtype=torch.float64, device="cuda")
    b, bT = api.causal_matrix(empty, inp.GEOM_DS2_SLAB)
    assert b.numel() == 0
    for N in (0, 1):
        z = torch.zeros((N, api.row_stride_words(N)), dtype=torch.int64, device="cuda")
        h = api.interval_hist(z, z, N)
        assert h.shape == (1,) and int(h[0]) == 0
        assert float(api.bd_action(h, N, 2)[0]) == 2.0 * N


# ----------------------------------------------------------------------------- a2
@pytest.mark.parametrize("geom,dim", GEOMS)
@pytest.mark.parametrize("N", [2, 64, 129, 1000, 2048])
def test_interval_hist_bit_exact(api, oracle, geom, dim, N):
    coords = inp.sprinkle(geom, dim, N, 7 * N + dim)
    o_bits = oracle.causal_matrix_bits(coords, geom)
    if N <= 1000:
        o_hist = oracle.interval_hist_alg19(oracle.unpack_bits(o_bits, N))      # tier-0
    else:
        o_hist, _, _ = oracle.interval_hist_alg20(o_bits, N)                    # tier-1
    R, W = oracle.count_relations(o_bits, N)
    bits, bitsT = gpu_bits(api, coords, geom)
    stats = api.relation_stats(bits, N).cpu().numpy()
    assert (int(stats[0]), int(stats[1])) == (R, W)
    for r in routes(api):
        hist, nrel = api.interval_hist(bits, bitsT, N, route=r, return_relations=True)
        assert np.array_equal(hist.cpu().numpy(), o_hist), "route %d" % r
        assert int(nrel[0]) == R
        # without bitsT (rebuilt in the workspace)
        assert np.array_equal(api.interval_hist(bits, None, N, route=r).cpu().numpy(), o_hist)
        # truncated histogram: larger intervals dropped, still counted as relations
        h3, n3 = api.interval_hist(bits, bitsT, N, kmax=3, route=r, return_relations=True)
        k = min(3, max(N - 2, 0))
        assert np.array_equal(h3.cpu().numpy(), o_hist[:k + 1]) and int(n3[0]) == R
        # row ranges add up
        cut = N // 3 + 1
        ha = api.interval_hist(bits, bitsT, N, route=r, row_begin=0, row_end=cut)
        hb = api.interval_hist(bits, bitsT, N, route=r, row_begin=cut, row_end=N)
        assert np.array_equal((ha + hb).cpu().numpy(), o_hist)
        assert np.array_equal(ha.cpu().numpy(), oracle.interval_hist_alg20(o_bits, N, 0, cut)[0])


@pytest.mark.parametrize("N", [2, 300, 1025])
def test_chain_and_antichain_on_gpu(api, N):
    for r in routes(api):
        bits, bitsT = gpu_bits(api, inp.chain_lightcone(N), inp.GEOM_MINK2_LIGHTCONE)
        h = api.interval_hist(bits, bitsT, N, route=r).cpu().numpy()
        assert np.array_equal(h, np.arange(N - 1, 0, -1))          # N_k = N-1-k
        bits, bitsT = gpu_bits(api, inp.antichain_lightcone(N), inp.GEOM_MINK2_LIGHTCONE)
        assert int(api.interval_hist(bits, bitsT, N, route=r).sum()) == 0


# ----------------------------------------------------------------------------- a3
@pytest.mark.parametrize("dim", [2, 3, 4])
def test_bd_action_matches_oracle(api, oracle, dim):
    rng = np.random.default_rng(dim)
    for n_entries in (1, 2, 3, 4, 9):
        hist = rng.integers(0, 3_000_000_000, n_entries).astype(np.int64)
        N = 131072
        S, I = api.bd_action(torch.from_numpy(hist).cuda(), N, dim, return_bracket=True)
        oS, oI = oracle.bd_action(hist, N, dim)
        assert int(I[0]) == oI
        if dim == 3:   # the prefactor needs Gamma and pow: libm vs correctly rounded constant
            assert float(S[0]) == pytest.approx(oS, rel=1e-15)
        else:
            assert float(S[0]) == oS


# ----------------------------------------------------------------------------- whole path
@pytest.mark.parametrize("cfg_index,N", [(1, 1024), (3, 1500), (4, 2000)])
def test_pipeline_device_and_host_entry(api, oracle, cfg_index, N):
    cfg = inp.CONFIGS[cfg_index]
    coords = inp.make_config_coords(cfg, N=N)
    o_bits, o_hist, o_S, o_I = oracle.action_pipeline(coords, cfg.geometry, tier=0 if N <= 1024 else 1)
    bits, bitsT = gpu_bits(api, coords, cfg.geometry)
    hist = api.interval_hist(bits, bitsT, N)
    S, I = api.bd_action(hist, N, cfg.dim, return_bracket=True)
    assert np.array_equal(to_u64(bits), o_bits)
    assert np.array_equal(hist.cpu().numpy(), o_hist)
    assert int(I[0]) == o_I and float(S[0]) == o_S
    # the host-buffer entry point (H2D + a1 + a2 + a3 + D2H)
    h_host, s_host = api.action_host(torch.from_numpy(coords).pin_memory(), cfg.geometry)
    assert np.array_equal(h_host.numpy(), o_hist) and float(s_host[0]) == o_S
    h_host3, s3 = api.action_host(torch.from_numpy(coords), cfg.geometry, kmax=3)
    assert np.array_equal(h_host3.numpy(), o_hist[:4]) and float(s3[0]) == o_S


def test_batched_ensemble(api, oracle):
    cfg = inp.CONFIGS[5]
    B, N = 6, 2048
    coords = inp.make_ensemble_coords(cfg, B=B)
    actions, hist4 = api.bd_action_batched(torch.from_numpy(coords).cuda(), cfg.geometry, return_hist4=True)
    actions = actions.cpu().numpy(); hist4 = hist4.cpu().numpy()
    for b in range(B):
        _, o_hist, o_S, _ = oracle.action_pipeline(coords[b], cfg.geometry, tier=1)
        assert np.array_equal(hist4[b], o_hist[:4])
        assert actions[b] == o_S
    # the chunked host-buffer entry point: more than one chunk of 512, pinned and pageable memory
    coords = inp.make_ensemble_coords(cfg, B=20, N=300)
    big = np.ascontiguousarray(np.tile(coords, (53, 1, 1))[:1050])
    want = [oracle.action_pipeline(coords[b], cfg.geometry, tier=1) for b in range(20)]
    for host in (torch.from_numpy(big).pin_memory(), torch.from_numpy(big)):
        a_host, h4_host = api.bd_action_batched_host(host, cfg.geometry)
        for b in range(1050):
            assert a_host[b] == want[b % 20][2] and np.array_equal(h4_host[b].numpy(), want[b % 20][1][:4])
    # ragged batched size
    coords = inp.make_ensemble_coords(cfg, B=3, N=333)
    actions = api.bd_action_batched(torch.from_numpy(coords).cuda(), cfg.geometry).cpu().numpy()
    for b in range(3):
        assert actions[b] == oracle.action_pipeline(coords[b], cfg.geometry)[2]


def test_interval_hist_batched_routes(api, oracle):
    """cs_interval_hist_batched: every route, full and truncated histograms, causets of a ragged size."""
    cfg = inp.CONFIGS[5]
    for B, N in ((5, 1300), (3, 2048)):
        coords = inp.make_ensemble_coords(cfg, B=B, N=N)
        bits, bitsT = api.causal_matrix_batched(torch.from_numpy(coords).cuda(), cfg.geometry)
        want = [oracle.action_pipeline(coords[b], cfg.geometry, tier=1)[1] for b in range(B)]
        for r in routes(api) + [api.ROUTE_AUTO]:
            full = api.interval_hist_batched(bits, bitsT, N, route=r).cpu().numpy()
            k3 = api.interval_hist_batched(bits, bitsT, N, kmax=3, route=r).cpu().numpy()
            k100 = api.interval_hist_batched(bits, bitsT, N, kmax=100, route=r).cpu().numpy()
            for b in range(B):
                assert np.array_equal(full[b], want[b]), (r, b)
                assert np.array_equal(k3[b], want[b][:4]), (r, b)
                assert np.array_equal(k100[b], want[b][:101]), (r, b)


def test_interval_hist_empty_block_skipping(api, oracle):
    """N large enough for the pair route to skip K blocks whose 256 x 256 bit block is empty (96+ row tiles):
    a 3+1 diamond, the same points with space stretched (most blocks near the diagonal empty, many tiles with
    no live stage at all), a ragged N, row ranges and kmax = 3; all routes that take this size agree with tier-1."""
    cfg = inp.CONFIGS[3]
    base = inp.sprinkle(cfg.geometry, cfg.dim, 25000, 41)
    stretched = base.copy(); stretched[:, 1:] *= 12.0
    thin = base[:24700].copy(); thin[:, 1:] *= 3.0
    for coords in (base, stretched, thin):
        N = coords.shape[0]
        o_bits = oracle.causal_matrix_bits(coords, cfg.geometry)
        o_hist, _, _ = oracle.interval_hist_alg20(o_bits, N)
        bits, bitsT = gpu_bits(api, coords, cfg.geometry)
        assert np.array_equal(to_u64(bits), o_bits)
        for r in (api.ROUTE_TENSOR_PAIR, api.ROUTE_AUTO):
            hist, nrel = api.interval_hist(bits, bitsT, N, route=r, return_relations=True)
            assert np.array_equal(hist.cpu().numpy(), o_hist)
            assert int(nrel[0]) == int(o_hist.sum())
            assert np.array_equal(api.interval_hist(bits, bitsT, N, kmax=3, route=r).cpu().numpy(), o_hist[:4])
        cut = 14321
        ha = api.interval_hist(bits, bitsT, N, row_begin=0, row_end=cut)
        hb = api.interval_hist(bits, bitsT, N, row_begin=cut, row_end=N)
        assert np.array_equal((ha + hb).cpu().numpy(), o_hist)
        assert np.array_equal(ha.cpu().numpy(), oracle.interval_hist_alg20(o_bits, N, 0, cut)[0])


def test_interval_hist_random_block_patterns(api, oracle):
    """The empty-block logic on arbitrary patterns (a sprinkling only produces monotone ones): a random upper
    triangular relation whose 256 x 256 blocks near the diagonal are emptied at random, a2 on the given bits
    (count = sum_k U[i][k] U[k][j] over related pairs, whatever U is) against tier-1, incl. a row range."""
    rng = np.random.default_rng(77)
    for N, p_empty in ((25000, 0.5), (24900, 0.9), (26000, 0.15)):
        stride = api.row_stride_words(N)
        nT = (N + 255) // 256
        bits = np.zeros((N, stride), dtype=np.uint64)
        for I in range(nT):
            r0, r1 = I * 256, min(N, I * 256 + 256)
            for J in range(I, nT):
                if J - I < 20 and rng.random() < p_empty:
                    continue                                   # an empty block
                if J - I >= 20 and rng.random() < 0.7:
                    continue                                   # keep the matrix sparse: most far blocks empty too
                blk = rng.integers(0, 2 ** 63, size=(r1 - r0, 4), dtype=np.int64).astype(np.uint64)
                blk &= rng.integers(0, 2 ** 63, size=(r1 - r0, 4), dtype=np.int64).astype(np.uint64)
                blk &= rng.integers(0, 2 ** 63, size=(r1 - r0, 4), dtype=np.int64).astype(np.uint64)   # density 1/8
                w0 = J * 4
                w1 = min(stride, w0 + 4)
                bits[r0:r1, w0:w1] = blk[:, : w1 - w0]
        # upper triangular (only the diagonal blocks hold bits at or below the diagonal), nothing at or beyond N
        sh = np.arange(64, dtype=np.uint64)[None, :]
        for I in range(nT):
            r0, r1 = I * 256, min(N, I * 256 + 256)
            rows = np.arange(r0, r1)
            for w in range(I * 4, min(stride, I * 4 + 4)):
                cols = np.arange(w * 64, w * 64 + 64)
                keep = cols[None, :] > rows[:, None]
                bits[r0:r1, w] &= (keep.astype(np.uint64) << sh).sum(axis=1, dtype=np.uint64)
        for w in range(N // 64, stride):
            cols = np.arange(w * 64, w * 64 + 64)
            bits[:, w] &= np.uint64(((cols < N).astype(np.uint64) << sh[0]).sum(dtype=np.uint64))
        o_hist, _, _ = oracle.interval_hist_alg20(bits, N)
        d_bits = torch.from_numpy(bits.view(np.int64)).cuda()
        d_bitsT = api.transpose_bits(d_bits, N)
        hist = api.interval_hist(d_bits, d_bitsT, N, route=api.ROUTE_TENSOR_PAIR)
        assert np.array_equal(hist.cpu().numpy(), o_hist), (N, p_empty)
        part = api.interval_hist(d_bits, d_bitsT, N, route=api.ROUTE_TENSOR_PAIR, row_begin=5000, row_end=5300)
        assert np.array_equal(part.cpu().numpy(), oracle.interval_hist_alg20(bits, N, 5000, 5300)[0])


# ----------------------------------------------------------------------------- full sizes
def _full_size_check(api, oracle, cfg):
    """BASELINE.json's full size, in the launch configuration bench.py times (default route, whole row range):
    bits, the WHOLE histogram and the action element by element against the oracle (tier-1 = Alg. 20,
    PAPER.md:1851-1893; bracket and S of Eq. 4.10-4.12, from the ORACLE's histogram),
    plus the two moment identities and three sampled row ranges."""
    N = cfg.N
    coords = inp.make_config_coords(cfg)
    o_bits = oracle.causal_matrix_bits(coords, cfg.geometry)
    bits, bitsT = gpu_bits(api, coords, cfg.geometry)
    assert np.array_equal(to_u64(bits), o_bits)
    R, W = oracle.count_relations(o_bits, N)
    stats = api.relation_stats(bits, N).cpu().numpy()
    assert (int(stats[0]), int(stats[1])) == (R, W)
    hist, nrel = api.interval_hist(bits, bitsT, N, return_relations=True)
    h = hist.cpu().numpy()
    assert int(nrel[0]) == R and int(h.sum()) == R
    outdeg, indeg = oracle.degrees(o_bits, N)
    assert int((np.arange(N - 1, dtype=np.int64) * h).sum()) == int((outdeg * indeg).sum())
    o_hist, _, _ = oracle.interval_hist_alg20(o_bits, N)
    assert np.array_equal(h, o_hist)
    # the two single-CTA tensor routes (kept as measured alternatives) at the size they were measured at: their
    # global-atomic tail, the 16/32-bit schedule limits and the int8 route's N <= 131072 bound are live here
    for r in (api.ROUTE_TENSOR, api.ROUTE_TENSOR_FP4, api.ROUTE_POPC if N <= 16384 else api.ROUTE_TENSOR_PAIR):
        assert np.array_equal(api.interval_hist(bits, bitsT, N, route=r).cpu().numpy(), o_hist), "route %d" % r
    rng = np.random.default_rng(cfg.index)
    for r0 in sorted(rng.integers(0, N - 64, 3).tolist()):
        part = api.interval_hist(bits, bitsT, N, row_begin=r0, row_end=r0 + 40).cpu().numpy()
        assert np.array_equal(part, oracle.interval_hist_alg20(o_bits, N, r0, r0 + 40)[0])
    S, I = api.bd_action(hist, N, cfg.dim, return_bracket=True)
    oS, oI = oracle.bd_action(o_hist, N, cfg.dim)          # from the oracle's own histogram
    assert int(I[0]) == oI and float(S[0]) == oS
    # the host-buffer entry point bench.py's e2e leg times
    h_host, s_host = api.action_host(torch.from_numpy(coords).pin_memory(), cfg.geometry)
    assert np.array_equal(h_host.numpy(), o_hist) and float(s_host[0]) == oS
    return o_hist, oS


def test_config2_full(api, oracle):
    _full_size_check(api, oracle, inp.CONFIGS[2])


@pytest.mark.slow
def test_config3_full_size(api, oracle):
    """The headline workload (N = 65536, 3+1): every bin of N_k and the action printed by bench.py."""
    _full_size_check(api, oracle, inp.CONFIGS[3])


@pytest.mark.slow
def test_config4_full_size(api, oracle):
    _full_size_check(api, oracle, inp.CONFIGS[4])


def test_headline_size_routes_agree_on_device(api):
    """N = 65536 (empty-block skipping, 16896 shared bins + global-atomic tail all active) without the oracle, so it
    runs in the default GPU suite: the complete pair-route histogram against the POPC route, kmax = 3, a row range."""
    cfg = inp.CONFIGS[3]
    bits, bitsT = gpu_bits(api, inp.make_config_coords(cfg), cfg.geometry)
    N = cfg.N
    ws = torch.empty(api.interval_hist_workspace(N, -1, True, api.ROUTE_TENSOR_PAIR), dtype=torch.uint8, device="cuda")
    pair = api.interval_hist(bits, bitsT, N, route=api.ROUTE_TENSOR_PAIR, workspace=ws)
    executed, total, empty, examined = api.interval_hist_stats(ws)
    popc = api.interval_hist(bits, bitsT, N, route=api.ROUTE_POPC)
    assert torch.equal(pair, popc)
    for r in (api.ROUTE_TENSOR, api.ROUTE_TENSOR_FP4):
        assert torch.equal(api.interval_hist(bits, bitsT, N, route=r), popc), "route %d" % r
    assert torch.equal(api.interval_hist(bits, bitsT, N, kmax=3), popc[:4])
    a = api.interval_hist(bits, bitsT, N, route=api.ROUTE_TENSOR_PAIR, row_begin=30000, row_end=31000)
    b = api.interval_hist(bits, bitsT, N, route=api.ROUTE_POPC, row_begin=30000, row_end=31000)
    assert torch.equal(a, b)
    # the executed-stage counter: dense-triangular total in closed form, fewer executed (empty blocks), none lost
    nT = N // 256
    assert total == nT * (nT + 1) * (nT + 2) // 6
    assert 0 < executed < total and 0 < empty <= examined


@pytest.mark.slow
def test_config5_full_size(api, oracle):
    """The whole ensemble (4096 x N=2048) in the one launch bench-style callers use; every causet's
    N_0..N_3 and action against the oracle (tier-1, itself pinned to tier-0 at this N)."""
    cfg = inp.CONFIGS[5]
    coords = inp.make_ensemble_coords(cfg)
    B = coords.shape[0]
    assert B == 4096 and coords.shape[1] == 2048
    actions, hist4 = api.bd_action_batched(torch.from_numpy(coords).cuda(), cfg.geometry, return_hist4=True)
    actions = actions.cpu().numpy(); hist4 = hist4.cpu().numpy()
    for b in range(B):
        _, o_hist, o_S, _ = oracle.action_pipeline(coords[b], cfg.geometry, tier=1)
        assert np.array_equal(hist4[b], o_hist[:4]), "causet %d" % b
        assert actions[b] == o_S, "causet %d" % b


# ----------------------------------------------------------------------------- NEXT-1: smeared action
_SMEAR_C = {2: (2.0, 0.5, 0.0, 2.0), 3: (27.0 / 8, 9.0 / 8, 0.0, 1.0), 4: (9.0, 8.0, 4.0 / 3, 1.0)}


def _smear_prefactor(dim, eps):
    import math
    if dim == 2:
        return 2.0 * eps
    if dim == 3:
        return (1.0 / math.gamma(5.0 / 3.0)) * (math.pi * eps / (3.0 * math.sqrt(2.0))) ** (2.0 / 3.0)
    return 4.0 * math.sqrt(eps / 6.0)


def _smear_tolerance(hist, dim, eps, S):
    """Bound on |CUDA - oracle| derived from the arithmetic: the CUDA sum is carried
    in double-double (~2^-100) and rounded once (2^-53 |S|, plus the fp64 prefactor: 2^-51 |S| in all); the
    oracle works in x87 long double, u = 2^-64: q = 1 - eps is rounded once, so q^(k-j) is off by <= (k+1) u, and
    each of the <= 4 sub-terms of f_d and their sums round with u -- in all <= (k+8) u A(k), with A(k) the sum of
    the absolute values of the sub-terms of f_d(k, eps)."""
    c1, c2, c3, a = _SMEAR_C[dim]
    k = np.arange(hist.shape[0], dtype=np.float64)
    q = 1.0 - eps

    def qp(j):                      # q^(k-j), 0 where the falling factorial vanishes
        return np.where(k >= j, np.power(q, np.maximum(k - j, 0.0)), 0.0)
    A = qp(0) + c1 * k * eps * qp(1) + c2 * k * (k - 1) * eps ** 2 * qp(2) + c3 * k * (k - 1) * (k - 2) * eps ** 3 * qp(3)
    bound = float((hist.astype(np.float64) * A * (k + 8.0)).sum()) * 2.0 ** -63
    return _smear_prefactor(dim, eps) * a * eps * bound + 2.0 ** -51 * abs(S)


@pytest.mark.parametrize("cfg_id,N,dim", [(2, 1500, 2), (3, 2048, 4), (4, 2000, 2), (3, 1200, 3)])
def test_smeared_action_vs_oracle(api, oracle, cfg_id, N, dim):
    cfg = inp.CONFIGS[cfg_id]
    coords = inp.sprinkle(cfg.geometry, dim, N, 77 + N)
    _, o_hist, _, _ = oracle.action_pipeline(coords, cfg.geometry, tier=1)
    d_hist = torch.from_numpy(o_hist).cuda()
    for eps in (1.0, 0.5, 0.25, 0.1, 2.0 ** -6, 0.013):
        o_S = oracle.smeared_action(o_hist, N, dim, eps)
        S = float(api.smeared_action(d_hist, N, dim, eps)[0])
        assert abs(S - o_S) <= _smear_tolerance(o_hist, dim, eps, o_S), (eps, S, o_S)
    # eps = 1 is the local action (Eq. 4.16-4.18 reduce to the coefficients of Eq. 4.10-4.12)
    S1 = float(api.smeared_action(d_hist, N, dim, 1.0)[0])
    S_local = float(api.bd_action(d_hist, N, dim)[0])
    assert S1 == pytest.approx(S_local, rel=4e-16, abs=0.0)
    # on the device pipeline's own histogram too
    bits, bitsT = gpu_bits(api, coords, cfg.geometry)
    h = api.interval_hist(bits, bitsT, N)
    assert float(api.smeared_action(h, N, dim, 2.0 ** -6)[0]) == float(api.smeared_action(d_hist, N, dim, 2.0 ** -6)[0])


def test_smeared_action_device_vs_exact_rational(api, oracle):
    """The DEVICE value against Eq. 4.13-4.15 with Eq. 4.16-4.18 as printed, evaluated in exact
    rational arithmetic on the same histogram and the same eps (Fraction(float) is exact).  The tolerance is the CUDA
    side's own: the double-double bracket is rounded to fp64 once and multiplied by an fp64 prefactor, 2^-51 |S| for
    the rational prefactor of d = 2, 2^-50 |S| where the prefactor is irrational (its few roundings on either side) --
    four to five orders tighter than the comparison with the oracle's long-double sum, whose error dominates there."""
    import math
    from fractions import Fraction
    N = 1200
    coords = inp.sprinkle(inp.GEOM_MINK_CONE, 4, N, 4242)
    _, hist, _, _ = oracle.action_pipeline(coords, inp.GEOM_MINK_CONE, tier=1)
    d_hist = torch.from_numpy(hist).cuda()
    for e in (2.0 ** -6, 0.2, 0.75, 0.013):
        eps = Fraction(e)
        q = 1 - eps
        sums = {2: Fraction(0), 3: Fraction(0), 4: Fraction(0)}
        qm = Fraction(1)                                         # q^m
        for m in range(hist.shape[0]):                           # the paper's n_{m+1} f(m)
            n = int(hist[m])
            if n:
                r = eps / q
                sums[2] += n * qm * (1 - 2 * m * r + Fraction(m * (m - 1), 2) * r ** 2)
                sums[3] += n * qm * (1 - Fraction(27, 8) * m * r + Fraction(9, 8) * m * (m - 1) * r ** 2)
                sums[4] += n * qm * (1 - 9 * m * r + 8 * m * (m - 1) * r ** 2 - Fraction(4, 3) * m * (m - 1) * (m - 2) * r ** 3)
            qm *= q
        want = {2: (float(2 * eps * (N - 2 * eps * sums[2])), 2.0 ** -51),
                3: ((1 / math.gamma(5 / 3)) * (math.pi * e / (3 * math.sqrt(2))) ** (2 / 3) * float(N - eps * sums[3]), 2.0 ** -50),
                4: (4 * math.sqrt(e / 6) * float(N - eps * sums[4]), 2.0 ** -50)}
        for dim in (2, 3, 4):
            S = float(api.smeared_action(d_hist, N, dim, e)[0])
            w, tol = want[dim]
            assert abs(S - w) <= tol * abs(w), (dim, e, S, w)
            # the bracket really cancels: the test would not see a sloppy sum otherwise
            assert abs(float(N - (2 if dim == 2 else 1) * eps * sums[dim])) < 0.2 * float(sum(abs(int(x)) for x in hist)) or e > 0.5


def test_tensor_selfchecks_pass_on_this_device(api):
    """CS_ROUTE_AUTO / CS_A1_AUTO take the tensor routes only on a device that passed these; on a B200 both must."""
    assert api.a2_tensor_selfcheck() is True
    assert api.a1_tensor_selfcheck() is True
    assert api.a2_tensor_selfcheck() is True                     # the cached answer


@pytest.mark.parametrize("dim", [2, 3, 4])
def test_smeared_action_long_histogram(api, oracle, dim):
    """Every bin up to k = N - 2 at the largest N the entry point takes, large counts, small eps: the terms
    reach ~1e21 while they cancel; still inside the derived bound."""
    N = 131072
    rng = np.random.default_rng(dim)
    k = np.arange(N - 1)
    hist = (rng.integers(1, 1 << 40, N - 1) * np.exp(-k / 30000.0)).astype(np.int64)
    d_hist = torch.from_numpy(hist).cuda()
    for eps in (2.0 ** -10, 2.0 ** -6, 0.37):
        o_S = oracle.smeared_action(hist, N, dim, eps)
        S = float(api.smeared_action(d_hist, N, dim, eps)[0])
        assert abs(S - o_S) <= _smear_tolerance(hist, dim, eps, o_S), (eps, S, o_S)


def test_smeared_action_arguments(api):
    h = torch.zeros(10, dtype=torch.int64, device="cuda")
    for bad in (0.0, -0.5, 1.5, float("nan")):
        with pytest.raises(RuntimeError):
            api.smeared_action(h, 11, 2, bad)
    with pytest.raises(RuntimeError):
        api.smeared_action(h, 11, 5, 0.5)
    assert float(api.smeared_action(h, 11, 4, 0.5)[0]) == 4.0 * (0.5 / 6.0) ** 0.5 * 11


@pytest.mark.slow
def test_smeared_action_tends_to_einstein_hilbert(api):
    """The paper's convergence experiment (Eq. 4.20, Fig. 4.5 right): 1+1 de Sitter slab,
    symmetric cutoff eta0 = 0.5, eps = 2^-6, ten sprinklings; the mean smeared action 'begins to converge' to
    S_EH = 4 pi tan(eta0) = 6.865 around N >= 2^14 while single terms of the series are orders of magnitude
    larger, and sigma_S grows like sqrt(N).  Statistical, but deterministic: the seeds are fixed.  The whole
    pipeline (a1, a2, smeared a3) runs on the device."""
    import math
    target = 4.0 * math.pi * math.tan(0.5)
    sds = {}
    for N in (1 << 14, 1 << 15):
        vals = []
        for seed in range(10):
            c = inp.sprinkle_ds2_slab(N, 9000 + seed, -0.5, 0.5)
            bits, bitsT = api.causal_matrix(torch.from_numpy(c).cuda(), inp.GEOM_DS2_SLAB)
            h = api.interval_hist(bits, bitsT, N)
            vals.append(float(api.smeared_action(h, N, 2, 2.0 ** -6)[0]))
            assert int(h[:3].sum()) > 1000 * abs(vals[-1])           # the series' terms dwarf the result
        mean, sd = float(np.mean(vals)), float(np.std(vals, ddof=1))
        sds[N] = sd
        assert abs(mean - target) < 3.5 * sd / math.sqrt(10), (N, mean, sd)
        assert mean > 0.5 * target                                    # N = 2^12 gives 0.4 +- 0.3: not yet converged
    assert 0.8 < sds[1 << 15] / sds[1 << 14] < 2.5                    # ~ sqrt(2), ten samples each


@pytest.mark.parametrize("geom,dim", GEOMS)
def test_degree_vectors(api, oracle, geom, dim):
    N = 1111
    coords = inp.sprinkle(geom, dim, N, 5 + dim)
    o_bits = oracle.causal_matrix_bits(coords, geom)
    bits, bitsT = gpu_bits(api, coords, geom)
    outdeg, indeg = api.degrees(bits, bitsT, N)
    o_out, o_in = oracle.degrees(o_bits, N)
    assert np.array_equal(outdeg.cpu().numpy(), o_out) and np.array_equal(indeg.cpu().numpy(), o_in)
    # the 3-chain identity on the device's own histogram
    h = api.interval_hist(bits, bitsT, N)
    k = torch.arange(h.numel(), device="cuda", dtype=torch.int64)
    assert int((k * h).sum()) == int((outdeg * indeg).sum())


def test_flrw_polar_pipeline(api, oracle):
    """NEXT-4 (Eq. 7.7): bits incl. pairs on and one ulp off the cone, histogram, 3+1 action, host entry point."""
    N = 1800
    coords = inp.sprinkle_flrw_polar(N, 3)
    # partners along the same ray at exactly / just beyond / just short of null separation
    extra = coords[:200].copy()
    extra[:, 0] = coords[:200, 0] + 0.125
    extra[:, 1] = coords[:200, 1] + 0.125
    e2 = extra.copy(); e2[:, 0] = np.nextafter(extra[:, 0], 10.0)
    e3 = extra.copy(); e3[:, 0] = np.nextafter(extra[:, 0], -10.0)
    coords = np.concatenate([coords, extra, e2, e3])
    coords = np.ascontiguousarray(coords[np.lexsort((coords[:, 1], coords[:, 0]))])
    N = coords.shape[0]
    o_bits, o_hist, o_S, o_I = oracle.action_pipeline(coords, inp.GEOM_FLRW_POLAR, tier=1)
    bits, bitsT = gpu_bits(api, coords, inp.GEOM_FLRW_POLAR)
    assert np.array_equal(to_u64(bits), o_bits)
    hist = api.interval_hist(bits, bitsT, N)
    assert np.array_equal(hist.cpu().numpy(), o_hist)
    S, I = api.bd_action(hist, N, 4, return_bracket=True)
    assert int(I[0]) == o_I and float(S[0]) == o_S
    h_host, s_host = api.action_host(torch.from_numpy(coords).pin_memory(), inp.GEOM_FLRW_POLAR)
    assert np.array_equal(h_host.numpy(), o_hist) and float(s_host[0]) == o_S
    with pytest.raises(RuntimeError):
        api.causal_matrix(torch.zeros((10, 4), dtype=torch.float64, device="cuda"), inp.GEOM_FLRW_POLAR)


# ----------------------------------------------------------------------------- NEXT-3: chains, antichains
def _unpack_member(member, N):
    return np.unpackbits(member.cpu().numpy().view(np.uint8), bitorder="little")[:N]


@pytest.mark.parametrize("geom,dim", GEOMS)
@pytest.mark.parametrize("N", [1, 2, 65, 700, 1500])
def test_chain_heights_bit_exact(api, oracle, geom, dim, N):
    coords = inp.sprinkle(geom, dim, N, 31 * N + dim)
    C = oracle.causal_matrix_bytes(coords, geom)
    bits, bitsT = gpu_bits(api, coords, geom)
    h, longest = api.chain_heights(bits, bitsT, N)
    o_h, o_best = oracle.chain_heights(C)
    assert np.array_equal(h.cpu().numpy(), o_h) and int(longest[0]) == o_best
    rng = np.random.default_rng(N)
    for source in {0, N // 2, int(rng.integers(0, N))}:
        h, longest = api.chain_heights(bits, bitsT, N, source=source)
        o_h, o_best = oracle.chain_heights(C, source=source)
        assert np.array_equal(h.cpu().numpy(), o_h) and int(longest[0]) == o_best
        # Algorithm 11 for a related pair = height - 1
        js = np.flatnonzero(C[source])
        if len(js):
            j = int(js[len(js) // 2])
            assert oracle.chain_pair(C, source, j) == int(h[j]) - 1


def test_chain_heights_closed_forms(api, oracle):
    for N in (300, 1025):
        c = inp.chain_lightcone(N)
        bits, bitsT = gpu_bits(api, c, inp.GEOM_MINK2_LIGHTCONE)
        h, longest = api.chain_heights(bits, bitsT, N)
        assert int(longest[0]) == N and np.array_equal(h.cpu().numpy(), np.arange(1, N + 1))
        a = inp.antichain_lightcone(N)
        bits, bitsT = gpu_bits(api, a, inp.GEOM_MINK2_LIGHTCONE)
        h, longest = api.chain_heights(bits, bitsT, N)
        assert int(longest[0]) == 1 and bool((h == 1).all())
        m, size = api.greedy_antichain(bits, bitsT, N, 5)
        assert int(size[0]) == N and _unpack_member(m, N).all()
    z = torch.zeros((0, 0), dtype=torch.int64, device="cuda")
    assert int(api.chain_heights(z, z, 0)[1][0]) == 0
    with pytest.raises(RuntimeError):
        api.chain_heights(bits, bitsT, N, source=N)
    with pytest.raises(RuntimeError):
        api.greedy_antichain(bits, bitsT, N, -1)


@pytest.mark.parametrize("geom,dim,N", [(inp.GEOM_MINK2_LIGHTCONE, 2, 900), (inp.GEOM_MINK_CONE, 4, 1100),
                                        (inp.GEOM_MINK_CONE, 3, 333), (inp.GEOM_DS2_SLAB, 2, 1000)])
def test_greedy_antichain_bit_exact(api, oracle, geom, dim, N):
    coords = inp.sprinkle(geom, dim, N, 17 + N)
    C = oracle.causal_matrix_bytes(coords, geom)
    bits, bitsT = gpu_bits(api, coords, geom)
    for seed in (0, N // 3, N - 1):
        m, size = api.greedy_antichain(bits, bitsT, N, seed)
        want = oracle.greedy_antichain(C, seed)
        assert np.array_equal(_unpack_member(m, N), want) and int(size[0]) == int(want.sum())
        assert int(m.cpu().numpy().view(np.uint64)[(N + 63) // 64:].sum()) == 0     # padding words stay zero


def test_longest_chain_config2_is_lis(api):
    """Full config 2 (N = 16384): the longest chain of the 1+1 diamond is the longest increasing subsequence
    (patience sorting on the host: a property that holds at any size)."""
    import bisect
    cfg = inp.CONFIGS[2]
    coords = inp.make_config_coords(cfg)
    bits, bitsT = gpu_bits(api, coords, cfg.geometry)
    h, longest = api.chain_heights(bits, bitsT, cfg.N)
    piles = []
    for v in coords[np.argsort(coords[:, 0], kind="stable"), 1]:
        k = bisect.bisect_left(piles, v)
        if k == len(piles):
            piles.append(v)
        else:
            piles[k] = v
    assert int(longest[0]) == len(piles)
    hh = h.cpu().numpy()
    assert hh.min() == 1 and np.array_equal(np.unique(hh), np.arange(1, len(piles) + 1))


# ----------------------------------------------------------------------------- NEXT-4: row sharding on one GPU
def test_row_sharding_matches_single_launch(api):
    """bench.py --shard on one device: the row ranges dist.shard_rows hands to 2, 3 and 8 ranks, run one after the
    other through cs_interval_hist_ex and summed, give the single-launch histogram of config 2 bit for bit."""
    from paper_1805_04463_b200 import dist as csd
    cfg = inp.CONFIGS[2]
    bits, bitsT = gpu_bits(api, inp.make_config_coords(cfg), cfg.geometry)
    full = api.interval_hist(bits, bitsT, cfg.N)
    for world in (2, 3, 8):
        total = torch.zeros_like(full)
        for r0, r1 in csd.shard_rows(cfg.N, world):
            total += api.interval_hist(bits, bitsT, cfg.N, row_begin=r0, row_end=r1)
        assert torch.equal(total, full), world


# ----------------------------------------------------------------------------- sanitizer target
def test_small_everything(api, oracle):
    """Every kernel of the library once on a small input (all four a2 routes, the batched ensemble, the cooperative
    poset kernels, the smeared action, the host entry points), checked against the oracle.  This is the command
    compute-sanitizer runs (profiles/r2_sanitizer.md):
        compute-sanitizer --tool memcheck python -m pytest tests/test_gpu_parity.py -q -k small_everything"""
    cfg = inp.CONFIGS[3]
    N = 700
    coords = inp.make_config_coords(cfg, N=N)
    o_bits, o_hist, o_S, o_I = oracle.action_pipeline(coords, cfg.geometry, tier=1)
    bits, bitsT = gpu_bits(api, coords, cfg.geometry)
    assert np.array_equal(to_u64(bits), o_bits)
    for r in routes(api):
        assert np.array_equal(api.interval_hist(bits, bitsT, N, route=r).cpu().numpy(), o_hist), r
        assert np.array_equal(api.interval_hist(bits, None, N, kmax=3, route=r).cpu().numpy(), o_hist[:4]), r
    S, I = api.bd_action(api.interval_hist(bits, bitsT, N), N, cfg.dim, return_bracket=True)
    assert int(I[0]) == o_I and float(S[0]) == o_S
    ens = inp.make_ensemble_coords(inp.CONFIGS[5], B=3, N=600)
    actions, hist4 = api.bd_action_batched(torch.from_numpy(ens).cuda(), cfg.geometry, return_hist4=True)
    a_host, _ = api.bd_action_batched_host(torch.from_numpy(ens).pin_memory(), cfg.geometry)
    for b in range(3):
        _, oh, oS, _ = oracle.action_pipeline(ens[b], cfg.geometry, tier=1)
        assert np.array_equal(hist4[b].cpu().numpy(), oh[:4]) and float(actions[b]) == oS == float(a_host[b])
    C = oracle.causal_matrix_bytes(coords, cfg.geometry)
    h, longest = api.chain_heights(bits, bitsT, N)
    assert np.array_equal(h.cpu().numpy(), oracle.chain_heights(C)[0])
    m, size = api.greedy_antichain(bits, bitsT, N, 3)
    assert np.array_equal(_unpack_member(m, N), oracle.greedy_antichain(C, 3))
    d_hist = torch.from_numpy(o_hist).cuda()
    assert abs(float(api.smeared_action(d_hist, N, 4, 0.25)[0]) - oracle.smeared_action(o_hist, N, 4, 0.25)) \
        <= _smear_tolerance(o_hist, 4, 0.25, oracle.smeared_action(o_hist, N, 4, 0.25))
    h_host, s_host = api.action_host(torch.from_numpy(coords).pin_memory(), cfg.geometry)
    assert np.array_equal(h_host.numpy(), o_hist) and float(s_host[0]) == o_S


def test_ds4_spherical_and_cone5_pipelines(api, oracle):
    """NEXT-4: the 3+1 de Sitter slab (spherical foliation) through the whole path incl. the host entry point (a 3+1
    dimensional action), and the 4+1 flat diamond up to its histogram (the paper prints no action for d = 5)."""
    N = 2100
    c = inp.sprinkle(inp.GEOM_DS4_SPHERICAL, 7, N, 8)
    o_bits, o_hist, o_S, o_I = oracle.action_pipeline(c, inp.GEOM_DS4_SPHERICAL, tier=1)
    bits, bitsT = gpu_bits(api, c, inp.GEOM_DS4_SPHERICAL)
    assert np.array_equal(to_u64(bits), o_bits)
    hist = api.interval_hist(bits, bitsT, N)
    assert np.array_equal(hist.cpu().numpy(), o_hist)
    S, I = api.bd_action(hist, N, 4, return_bracket=True)
    assert int(I[0]) == o_I and float(S[0]) == o_S
    h_host, s_host = api.action_host(torch.from_numpy(c).pin_memory(), inp.GEOM_DS4_SPHERICAL)
    assert np.array_equal(h_host.numpy(), o_hist) and float(s_host[0]) == o_S
    c5 = inp.sprinkle(inp.GEOM_MINK_CONE, 5, N, 9)
    o_bits, o_hist, _, _ = oracle.action_pipeline(c5, inp.GEOM_MINK_CONE, tier=1)
    bits, bitsT = gpu_bits(api, c5, inp.GEOM_MINK_CONE)
    assert np.array_equal(to_u64(bits), o_bits)
    assert np.array_equal(api.interval_hist(bits, bitsT, N).cpu().numpy(), o_hist)
    with pytest.raises(RuntimeError):
        api.bd_action(hist, N, 5)
    with pytest.raises(RuntimeError):
        api.causal_matrix(torch.zeros((10, 6), dtype=torch.float64, device="cuda"), inp.GEOM_DS4_SPHERICAL)


def test_appendix_a_3p1_diamonds_pipeline(api, oracle):
    """NEXT-4, the last three regions of App. A.1 (3+1 dS diamonds, flat and spherical foliation; 3+1
    dust diamond): each sprinkling through a1 (every route), a2 and a3 against the oracle."""
    N = 1800
    for sprinkler, geom in ((inp.sprinkle_ds4_diamond_flat, inp.GEOM_FLRW_POLAR),
                            (inp.sprinkle_ds4_diamond_spherical, inp.GEOM_DS4_SPHERICAL),
                            (inp.sprinkle_dust_diamond, inp.GEOM_FLRW_POLAR)):
        c = sprinkler(N, 21)
        o_bits, o_hist, o_S, o_I = oracle.action_pipeline(c, geom, tier=1)
        bits, bitsT = gpu_bits(api, c, geom)
        assert np.array_equal(to_u64(bits), o_bits), sprinkler.__name__
        hist = api.interval_hist(bits, bitsT, N)
        assert np.array_equal(hist.cpu().numpy(), o_hist) and o_hist.sum() > N
        S, I = api.bd_action(hist, N, 4, return_bracket=True)
        assert int(I[0]) == o_I and float(S[0]) == o_S
        h_host, s_host = api.action_host(torch.from_numpy(c).pin_memory(), geom)
        assert np.array_equal(h_host.numpy(), o_hist) and float(s_host[0]) == o_S


@pytest.mark.slow
def test_larger_N_properties(api, oracle):
    """NEXT-4 'larger N': N = 262144 (8 GiB per bit matrix, 1024 x 1024 tiles) in the 1+1 de Sitter slab.  The oracle's
    tier-1 would need ~10 minutes here, so the checks are the ones that hold at any size: sum_k N_k = R,
    sum_k k N_k = sum_m indeg(m) outdeg(m), additivity of row ranges (the --shard split of 4 ranks), and six sampled
    rows whose per-pair interval sizes are recounted on the host from the definition, popcount(bits[i] & bitsT[j])."""
    from paper_1805_04463_b200 import dist as csd
    N = 1 << 18
    coords = inp.sprinkle_ds2_slab(N, 2718)
    bits, bitsT = gpu_bits(api, coords, inp.GEOM_DS2_SLAB)
    stats = api.relation_stats(bits, N).cpu().numpy()
    hist, nrel = api.interval_hist(bits, bitsT, N, return_relations=True)
    assert int(nrel[0]) == int(stats[0]) == int(hist.sum())
    outdeg, indeg = api.degrees(bits, bitsT, N)
    k = torch.arange(hist.numel(), device="cuda", dtype=torch.int64)
    assert int((k * hist).sum()) == int((outdeg * indeg).sum())
    total = torch.zeros_like(hist)
    for r0, r1 in csd.shard_rows(N, 4):
        total += api.interval_hist(bits, bitsT, N, row_begin=r0, row_end=r1)
    assert torch.equal(total, hist)
    # sampled rows i: count(i, j) = popcount(bits[i] & bitsT[j]) over the related j, histogrammed with numpy
    hb = bits.cpu().numpy().view(np.uint64); hbT = bitsT.cpu().numpy().view(np.uint64)
    rng = np.random.default_rng(5)
    for i in rng.integers(0, N - 1000, 6).tolist():
        part = api.interval_hist(bits, bitsT, N, row_begin=i, row_end=i + 1).cpu().numpy()
        js = np.flatnonzero(np.unpackbits(hb[i].view(np.uint8), bitorder="little")[:N])
        cnt = np.array([int(np.unpackbits((hb[i] & hbT[j]).view(np.uint8)).sum()) for j in js], dtype=np.int64)
        want = np.bincount(cnt, minlength=part.shape[0])[:part.shape[0]]
        assert np.array_equal(part, want), i
