"""Seeded synthetic sprinklings (inputs only -- none of the method's arithmetic).

This module is the one piece shared by the oracle-side tests and the CUDA
path: it draws point coordinates with a counter-based SplitMix64 generator,
sorts them by time, and hands the same fp64 buffer to both sides.  It never
evaluates a causal relation, an interval or an action.

The paper's workloads are themselves synthetic Poisson sprinklings
(App. A.1); `N` is fixed instead of
Poisson-distributed (reading A10).  Recipes:

  config 1/2  1+1 flat diamond in light-cone coordinates, u,v ~ U[0,1)
              (PAPER.md:3715-3729), sorted by ((u+v)/2, u, index)
  config 3/5  3+1 flat diamond |t|+|x|<=1 by rejection from the cube
              [-1,1)^4 (same distribution as PAPER.md:3745-3759 up to shift and
              scale; reading A11), sorted by (t, x, index)
  config 4    1+1 de Sitter slab, eta in [-1.2,-0.2] with density ~ sec^2(eta):
              eta = atan(tan a + u (tan b - tan a)), theta = 2 pi u
              (PAPER.md:3781-3795 generalised to an asymmetric slab; A12),
              sorted by (eta, theta, index)
"""
from __future__ import annotations

import dataclasses

import numpy as np

GEOM_MINK2_LIGHTCONE = 0
GEOM_MINK_CONE = 1
GEOM_DS2_SLAB = 2
GEOM_FLRW_POLAR = 3
GEOM_DS4_SPHERICAL = 4

_GAMMA = np.uint64(0x9E3779B97F4A7C15)
_M1 = np.uint64(0xBF58476D1CE4E5B9)
_M2 = np.uint64(0x94D049BB133111EB)
_MASK = (1 << 64) - 1

SEED_BASE = 180504463 * 10


def splitmix64(seed: int, start: int, count: int) -> np.ndarray:
    """Outputs number start .. start+count-1 of SplitMix64 seeded with `seed`
    (output n is mix(seed + (n+1)*gamma)); returned as uint64."""
    n = np.arange(start + 1, start + count + 1, dtype=np.uint64)
    with np.errstate(over="ignore"):
        z = np.uint64(seed & _MASK) + n * _GAMMA
        z = (z ^ (z >> np.uint64(30))) * _M1
        z = (z ^ (z >> np.uint64(27))) * _M2
        z = z ^ (z >> np.uint64(31))
    return z


def uniform01(seed: int, start: int, count: int) -> np.ndarray:
    """fp64 uniforms in [0,1): (z >> 11) * 2^-53."""
    z = splitmix64(seed, start, count)
    return (z >> np.uint64(11)).astype(np.float64) * (1.0 / 9007199254740992.0)


def _sort_rows(coords: np.ndarray, k0: np.ndarray, k1: np.ndarray) -> np.ndarray:
    idx = np.arange(coords.shape[0])
    order = np.lexsort((idx, k1, k0))  # primary k0, then k1, then original index
    return np.ascontiguousarray(coords[order])


def sprinkle_mink2_lightcone(N: int, seed: int) -> np.ndarray:
    """[N][2] = (u, v), draws per point in the order u, v."""
    r = uniform01(seed, 0, 2 * N).reshape(N, 2)
    t = (r[:, 0] + r[:, 1]) / 2.0
    return _sort_rows(r, t, r[:, 0])


def sprinkle_mink4_diamond(N: int, seed: int) -> np.ndarray:
    """[N][4] = (t, x, y, z); trial n uses draws 4n..4n+3 as t,x,y,z = 2u-1 and
    is accepted iff |t| + sqrt(x^2+y^2+z^2) <= 1; the first N accepted trials."""
    out = np.empty((N, 4), dtype=np.float64)
    have = 0
    trial = 0
    while have < N:
        batch = max(4096, int((N - have) * 8.5))
        r = 2.0 * uniform01(seed, 4 * trial, 4 * batch).reshape(batch, 4) - 1.0
        ok = np.abs(r[:, 0]) + np.sqrt(r[:, 1] ** 2 + r[:, 2] ** 2 + r[:, 3] ** 2) <= 1.0
        acc = r[ok]
        take = min(N - have, acc.shape[0])
        out[have:have + take] = acc[:take]
        have += take
        trial += batch
    return _sort_rows(out, out[:, 0], out[:, 1])


def sprinkle_ds2_slab(N: int, seed: int, eta_a: float = -1.2, eta_b: float = -0.2) -> np.ndarray:
    """[N][2] = (eta, theta), draws per point in the order eta, theta."""
    r = uniform01(seed, 0, 2 * N).reshape(N, 2)
    ta, tb = np.tan(eta_a), np.tan(eta_b)
    eta = np.arctan(ta + r[:, 0] * (tb - ta))
    theta = (2.0 * np.pi) * r[:, 1]
    c = np.stack([eta, theta], axis=1)
    return _sort_rows(c, eta, theta)


def sprinkle_flrw_polar(N: int, seed: int, eta0: float = 1.0, r0: float = 0.7) -> np.ndarray:
    """[N][6] = (eta, r, cos th, sin th, cos ph, sin ph) for the Eq. 7.7 predicate: conformal time
    eta ~ U[0, eta0), points uniform in the ball r < r0 (r = r0 u^(1/3), cos th = 2u - 1, ph = 2 pi u); draws per
    point in the order eta, r, th, ph.  The trigonometric values are part of the input."""
    r = uniform01(seed, 0, 4 * N).reshape(N, 4)
    eta = eta0 * r[:, 0]
    rad = r0 * np.cbrt(r[:, 1])
    ct = 2.0 * r[:, 2] - 1.0
    st = np.sqrt(np.maximum(0.0, 1.0 - ct * ct))
    ph = (2.0 * np.pi) * r[:, 3]
    c = np.stack([eta, rad, ct, st, np.cos(ph), np.sin(ph)], axis=1)
    return _sort_rows(c, eta, rad)


# ---- the other regions of the paper's Appendix A.1, each with the paper's own recipe ---------
def _invert_monotone(f, u: np.ndarray, lo: float, hi: float, iters: int = 70) -> np.ndarray:
    """x in [lo, hi] with f(x) = u for an increasing f, by bisection (the paper: "must be inverted numerically");
    a fixed iteration count keeps the result a deterministic function of u."""
    a = np.full(u.shape, lo, dtype=np.float64)
    b = np.full(u.shape, hi, dtype=np.float64)
    for _ in range(iters):
        mid = 0.5 * (a + b)
        below = f(mid) < u
        a = np.where(below, mid, a)
        b = np.where(below, b, mid)
    return 0.5 * (a + b)


def sprinkle_mink2_square(N: int, seed: int, t0: float = 1.0, x0: float = 1.0) -> np.ndarray:
    """1+1 square: t* = (2u-1) t0, x* = (2u-1) x0; [N][2] = (t, x) for GEOM_MINK_CONE."""
    r = uniform01(seed, 0, 2 * N).reshape(N, 2)
    c = np.stack([(2.0 * r[:, 0] - 1.0) * t0, (2.0 * r[:, 1] - 1.0) * x0], axis=1)
    return _sort_rows(c, c[:, 0], c[:, 1])


def sprinkle_mink2_cylinder(N: int, seed: int, t0: float = 1.0) -> np.ndarray:
    """1+1 cylinder, ds^2 = -dt^2 + d theta^2: t* = (2u-1) t0, theta* = 2 pi u; [N][2] = (t, theta).
    Its relation is the periodic one of GEOM_DS2_SLAB (the de Sitter slab is conformal to this cylinder)."""
    r = uniform01(seed, 0, 2 * N).reshape(N, 2)
    c = np.stack([(2.0 * r[:, 0] - 1.0) * t0, (2.0 * np.pi) * r[:, 1]], axis=1)
    return _sort_rows(c, c[:, 0], c[:, 1])


def sprinkle_mink3_diamond_uv(N: int, seed: int, u0: float = 1.0) -> np.ndarray:
    """2+1 diamond by the paper's inverse CDFs: u* = u^(1/3) u0, v* = u* (1 - sqrt(1 - u)),
    theta* = 2 pi u, with t = (u+v)/sqrt 2, r = (u-v)/sqrt 2; [N][3] = (t, x, y) for GEOM_MINK_CONE."""
    r = uniform01(seed, 0, 3 * N).reshape(N, 3)
    u = np.cbrt(r[:, 0]) * u0
    v = u * (1.0 - np.sqrt(1.0 - r[:, 1]))
    th = (2.0 * np.pi) * r[:, 2]
    t = (u + v) / np.sqrt(2.0)
    rad = (u - v) / np.sqrt(2.0)
    c = np.stack([t, rad * np.cos(th), rad * np.sin(th)], axis=1)
    return _sort_rows(c, c[:, 0], c[:, 1])


def sprinkle_mink5_diamond(N: int, seed: int) -> np.ndarray:
    """4+1 flat diamond |t| + |x| <= 1 (the region of PAPER.md:3761-3777 up to shift and scale) by rejection from the
    cube [-1,1)^5, as config 3 does in 3+1 (reading A11); [N][5] = (t, x, y, z, w) for GEOM_MINK_CONE."""
    return _sprinkle_mink_low(N, 5, seed)


def sprinkle_ds4_spherical(N: int, seed: int, eta0: float = 1.0) -> np.ndarray:
    """3+1 de Sitter slab, spherical foliation: eta in [0, eta0] with density ~ sec^4 eta, psi with
    density ~ sin^2 psi (u = (2 psi - sin 2 psi) / 2 pi "must be inverted numerically"), theta* = arccos(1 - 2u),
    phi* = 2 pi u; draws per point in the order eta, psi, theta, phi.  The eta CDF is (tan eta + tan^3 eta / 3) /
    (tan eta0 + tan^3 eta0 / 3) (the integral of sec^4), inverted numerically as well.
    [N][7] = (eta, cos eta, sin eta, X0, X1, X2, X3), X the unit 4-vector of (psi, theta, phi): the trigonometric
    values are part of the input (reading A18)."""
    r = uniform01(seed, 0, 4 * N).reshape(N, 4)
    t0 = np.tan(eta0)
    norm = t0 + t0 ** 3 / 3.0
    tan_eta = _invert_monotone(lambda t: (t + t ** 3 / 3.0) / norm, r[:, 0], 0.0, t0)
    eta = np.arctan(tan_eta)
    psi = _invert_monotone(lambda p: (2.0 * p - np.sin(2.0 * p)) / (2.0 * np.pi), r[:, 1], 0.0, np.pi)
    ct = 1.0 - 2.0 * r[:, 2]
    st = np.sqrt(np.maximum(0.0, 1.0 - ct * ct))
    ph = (2.0 * np.pi) * r[:, 3]
    sp = np.sin(psi)
    c = np.stack([eta, np.cos(eta), np.sin(eta), np.cos(psi), sp * ct, sp * st * np.cos(ph), sp * st * np.sin(ph)], axis=1)
    return _sort_rows(c, eta, c[:, 3])


def sprinkle_dust_slab(N: int, seed: int, tau0: float = 1.0, r0: float = 0.5) -> np.ndarray:
    """3+1 dust (Einstein-de Sitter) slab: tau* = tau0 u^(1/3), r* = r0 u^(1/3),
    theta* = arccos(1 - 2u), phi* = 2 pi u.  The relation of a conformally flat FLRW spacetime is Eq. 7.7 in conformal
    time: with a = (3 tau / 2)^(2/3) (alpha~ = 1), eta = int d tau / a = 2 (3 tau / 2)^(1/3).
    [N][6] = (eta, r, cos th, sin th, cos ph, sin ph) for GEOM_FLRW_POLAR."""
    r = uniform01(seed, 0, 4 * N).reshape(N, 4)
    tau = tau0 * np.cbrt(r[:, 0])
    eta = 2.0 * np.cbrt(1.5 * tau)
    rad = r0 * np.cbrt(r[:, 1])
    ct = 1.0 - 2.0 * r[:, 2]
    st = np.sqrt(np.maximum(0.0, 1.0 - ct * ct))
    ph = (2.0 * np.pi) * r[:, 3]
    c = np.stack([eta, rad, ct, st, np.cos(ph), np.sin(ph)], axis=1)
    return _sort_rows(c, eta, rad)


def sprinkle_ds4_flat_slab(N: int, seed: int, eta0: float = -0.25, r0: float = 0.6) -> np.ndarray:
    """3+1 de Sitter slab, flat foliation ("3+1 Dimensional Slab (Flat Foliation)"), conformal time
    eta in [-1, eta0]: eta* = [u (1 + eta0^-3) - 1]^(-1/3), r* = u^(1/3) r0, theta* = arccos(1 - 2u), phi* = 2 pi u.
    Conformally flat, so the relation is Eq. 7.7: [N][6] = (eta, r, cos th, sin th, cos ph, sin ph) for GEOM_FLRW_POLAR."""
    r = uniform01(seed, 0, 4 * N).reshape(N, 4)
    eta = 1.0 / np.cbrt(r[:, 0] * (1.0 + eta0 ** -3) - 1.0)
    rad = r0 * np.cbrt(r[:, 1])
    ct = 1.0 - 2.0 * r[:, 2]
    st = np.sqrt(np.maximum(0.0, 1.0 - ct * ct))
    ph = (2.0 * np.pi) * r[:, 3]
    c = np.stack([eta, rad, ct, st, np.cos(ph), np.sin(ph)], axis=1)
    return _sort_rows(c, eta, rad)


def sprinkle_dust_lambda_slab(N: int, seed: int, tau0: float = 1.0, r0: float = 0.5) -> np.ndarray:
    """3+1 dust + dark energy slab: tau from u = (sinh 3 tau - 3 tau) / (sinh 3 tau0 - 3 tau0)
    ("must be inverted numerically"), r* = r0 u^(1/3), theta*, phi* as above; conformal time by Eq. 7.5
    (PAPER.md:3167), eta_M = 2 sinh^(1/3)(3 tau / 2) 2F1(1/6, 1/2; 7/6; -sinh^2(3 tau / 2)) with alpha~ = 1.
    [N][6] for GEOM_FLRW_POLAR."""
    from scipy.special import hyp2f1
    r = uniform01(seed, 0, 4 * N).reshape(N, 4)
    norm = np.sinh(3.0 * tau0) - 3.0 * tau0
    tau = _invert_monotone(lambda t: (np.sinh(3.0 * t) - 3.0 * t) / norm, r[:, 0], 0.0, tau0)
    sh = np.sinh(1.5 * tau)
    eta = 2.0 * np.cbrt(sh) * hyp2f1(1.0 / 6.0, 0.5, 7.0 / 6.0, -sh * sh)
    rad = r0 * np.cbrt(r[:, 1])
    ct = 1.0 - 2.0 * r[:, 2]
    st = np.sqrt(np.maximum(0.0, 1.0 - ct * ct))
    ph = (2.0 * np.pi) * r[:, 3]
    c = np.stack([eta, rad, ct, st, np.cos(ph), np.sin(ph)], axis=1)
    return _sort_rows(c, eta, rad)


def sprinkle_ds2_diamond_flat(N: int, seed: int, w: float = 0.5) -> np.ndarray:
    """1+1 de Sitter diamond, flat foliation, ds^2 = -4 lambda^2 du dv / (u + v)^2 on [u0, u0 + w]^2 with
    u0 = v0 = -1/sqrt 2: mu = (u0+v0+w)^2 / ((u0+v0)(u0+v0+2w)), beta = (u0+v0)/(u0+v0+w) mu^u,
    u* = (beta (v0+w) - v0) / (1 - beta), gamma = w u / (u* + v0 + w), v* = (gamma u* + v0) / (1 - gamma).
    Conformal to the flat light-cone diamond: [N][2] = (u, v) for GEOM_MINK2_LIGHTCONE."""
    r = uniform01(seed, 0, 2 * N).reshape(N, 2)
    u0 = v0 = -1.0 / np.sqrt(2.0)
    mu = (u0 + v0 + w) ** 2 / ((u0 + v0) * (u0 + v0 + 2.0 * w))
    beta = (u0 + v0) / (u0 + v0 + w) * mu ** r[:, 0]
    u = (beta * (v0 + w) - v0) / (1.0 - beta)
    gamma = w * r[:, 1] / (u + v0 + w)
    v = (gamma * u + v0) / (1.0 - gamma)
    c = np.stack([u, v], axis=1)
    return _sort_rows(c, (u + v) / 2.0, u)


def sprinkle_ds2_diamond_spherical(N: int, seed: int, w0: float = 0.8) -> np.ndarray:
    """1+1 de Sitter diamond, spherical foliation, density ~ sec^2((u + v)/sqrt 2) on [0, w0]^2:
    mu = (1 + sec(sqrt 2 w0)) / 2, u* = sqrt 2 arctan[(1 - mu^-u) cot(w0 / sqrt 2)],
    v* = sqrt 2 arctan[u tan((u* + w0)/sqrt 2) + (1 - u) tan(u* / sqrt 2)] - u*.
    (The extracted text prints the first tangent without its factor u; with it the expression is the inverse of the
    conditional CDF of the stated density, reading A20.)  [N][2] = (u, v) for GEOM_MINK2_LIGHTCONE."""
    r = uniform01(seed, 0, 2 * N).reshape(N, 2)
    s2 = np.sqrt(2.0)
    mu = (1.0 + 1.0 / np.cos(s2 * w0)) / 2.0
    u = s2 * np.arctan((1.0 - mu ** (-r[:, 0])) / np.tan(w0 / s2))
    v = s2 * np.arctan(r[:, 1] * np.tan((u + w0) / s2) + (1.0 - r[:, 1]) * np.tan(u / s2)) - u
    c = np.stack([u, v], axis=1)
    return _sort_rows(c, (u + v) / 2.0, u)


def _polar6(t, rad, r_theta, r_phi):
    """(eta, r, cos th, sin th, cos ph, sin ph) rows with theta* = arccos(1 - 2u), phi* = 2 pi u."""
    ct = 1.0 - 2.0 * r_theta
    st = np.sqrt(np.maximum(0.0, 1.0 - ct * ct))
    ph = (2.0 * np.pi) * r_phi
    return np.stack([t, rad, ct, st, np.cos(ph), np.sin(ph)], axis=1)


def ds4_diamond_flat_mu(w: float, u0: float) -> float:
    """mu of the 3+1 dS diamond, flat foliation: ln[(w + 2u0)^2 / (4 u0 (w + u0))] - (w / (w + 2u0))^2."""
    return float(np.log((w + 2.0 * u0) ** 2 / (4.0 * u0 * (w + u0))) - (w / (w + 2.0 * u0)) ** 2)


def sprinkle_ds4_diamond_flat(N: int, seed: int, w: float = 0.5) -> np.ndarray:
    """3+1 de Sitter diamond, flat foliation: rho(u, v) = (6 / mu) (u - v)^2 / (u + v)^4 on
    u in [u0, u0 + w], v in [u0, u], u0 = -1/sqrt 2 (as in the 1+1 diamond; w < 1/sqrt 2).  The
    printed u*, v* (Lambert W, a cubic) are garbled in the extracted text; both are inverse CDFs of the stated
    density, which has them in closed form (reading A23), inverted here by bisection:
      F(u)     = (6 / mu) [G(u) - G(u0)],  G(x) = ln|x + u0| / 3 + 2 u0 / (3 (x + u0)) - 2 u0^2 / (3 (x + u0)^2) - ln|x| / 6
      F(v | u) = [K(u + v) - K(u + u0)] / [K(2u) - K(u + u0)],  K(s) = -4 u^2 / (3 s^3) + 2 u / s^2 - 1 / s.
    Conformally flat with eta = (u + v) / sqrt 2 < 0, r = (u - v) / sqrt 2: [N][6] for GEOM_FLRW_POLAR."""
    r = uniform01(seed, 0, 4 * N).reshape(N, 4)
    u0 = -1.0 / np.sqrt(2.0)
    mu = ds4_diamond_flat_mu(w, u0)

    def G(x):
        a = x + u0
        return np.log(np.abs(a)) / 3.0 + 2.0 * u0 / (3.0 * a) - 2.0 * u0 * u0 / (3.0 * a * a) - np.log(np.abs(x)) / 6.0
    u = _invert_monotone(lambda x: 6.0 * (G(x) - G(u0)) / mu, r[:, 0], u0, u0 + w)

    def K(sv):
        return -4.0 * u * u / (3.0 * sv ** 3) + 2.0 * u / sv ** 2 - 1.0 / sv
    span = K(2.0 * u) - K(u + u0)
    t = _invert_monotone(lambda q: np.where(span > 0, (K(u + u0 + q * (u - u0)) - K(u + u0)) / np.where(span > 0, span, 1.0), q),
                         r[:, 1], 0.0, 1.0)
    v = u0 + t * (u - u0)
    c = _polar6((u + v) / np.sqrt(2.0), (u - v) / np.sqrt(2.0), r[:, 2], r[:, 3])
    return _sort_rows(c, c[:, 0], c[:, 1])


def sprinkle_ds4_diamond_spherical(N: int, seed: int, w0: float = 0.8) -> np.ndarray:
    """3+1 de Sitter diamond, spherical foliation: rho(u, v) ~ sec^4((u + v)/sqrt 2)
    sin^2((u - v)/sqrt 2) on u in [0, w0], v in [0, u].  The printed u(u*), u(v*) are cut off in the extracted text and
    "must be inverted numerically" anyway; the stated density is sampled in eta = (u + v)/sqrt 2, psi = (u - v)/sqrt 2
    (constant Jacobian; reading A23): 0 <= psi <= psi_m(eta) = min(eta, sqrt 2 w0 - eta),
      p(eta) ~ sec^4(eta) (psi_m - sin(2 psi_m)/2),  F(psi | eta) = (psi - sin(2 psi)/2) / (psi_m - sin(2 psi_m)/2),
    the first through a cumulative Simpson table (8192 panels), both inverted by bisection.
    [N][7] = (eta, cos eta, sin eta, X0..X3) for GEOM_DS4_SPHERICAL (w0 < pi / (2 sqrt 2))."""
    r = uniform01(seed, 0, 4 * N).reshape(N, 4)
    top = np.sqrt(2.0) * w0

    def area(pm):
        return pm - 0.5 * np.sin(2.0 * pm)
    n = 8192
    grid = np.linspace(0.0, top, 2 * n + 1)
    f = area(np.minimum(grid, top - grid)) / np.cos(grid) ** 4
    h = grid[1] - grid[0]
    cum = np.concatenate([[0.0], np.cumsum((f[0:-2:2] + 4.0 * f[1:-1:2] + f[2::2]) * (h / 3.0))])
    eta = _invert_monotone(lambda x: np.interp(x, grid[::2], cum) / cum[-1], r[:, 0], 0.0, top)
    pm = np.minimum(eta, top - eta)
    am = area(pm)
    t = _invert_monotone(lambda q: np.where(am > 0, area(q * pm) / np.where(am > 0, am, 1.0), q), r[:, 1], 0.0, 1.0)
    psi = t * pm
    ct = 1.0 - 2.0 * r[:, 2]
    st = np.sqrt(np.maximum(0.0, 1.0 - ct * ct))
    ph = (2.0 * np.pi) * r[:, 3]
    sp = np.sin(psi)
    c = np.stack([eta, np.cos(eta), np.sin(eta), np.cos(psi), sp * ct, sp * st * np.cos(ph), sp * st * np.sin(ph)], axis=1)
    return _sort_rows(c, eta, psi)


def sprinkle_dust_diamond(N: int, seed: int, u0: float = 1.0) -> np.ndarray:
    """3+1 dust diamond: rho(u, v) = 5940 / (1981 u0^12) (u + v)^8 (u - v)^2 on u in [0, u0],
    v in [0, u]; u* = u0 u^(1/12); v* from the printed eleventh-degree polynomial (partly garbled in the extracted text),
    "must be inverted numerically": it is the conditional CDF of the stated density,
      F(v | u) = [Q(u + v) - Q(u)] / [Q(2u) - Q(u)],  Q(s) = 4 u^2 s^9 / 9 - 2 u s^10 / 5 + s^11 / 11
    (reading A23), inverted by bisection.  Conformally flat in eta = (u + v)/sqrt 2, r = (u - v)/sqrt 2
    (the conformal factor ~ (u + v)^4 does not enter the relation): [N][6] for GEOM_FLRW_POLAR."""
    r = uniform01(seed, 0, 4 * N).reshape(N, 4)
    u = u0 * r[:, 0] ** (1.0 / 12.0)

    def Q(sv):
        return 4.0 * u * u * sv ** 9 / 9.0 - 2.0 * u * sv ** 10 / 5.0 + sv ** 11 / 11.0
    span = Q(2.0 * u) - Q(u)
    t = _invert_monotone(lambda q: np.where(span > 0, (Q(u + q * u) - Q(u)) / np.where(span > 0, span, 1.0), q), r[:, 1], 0.0, 1.0)
    v = t * u
    c = _polar6((u + v) / np.sqrt(2.0), (u - v) / np.sqrt(2.0), r[:, 2], r[:, 3])
    return _sort_rows(c, c[:, 0], c[:, 1])


def chain_lightcone(N: int) -> np.ndarray:
    """Total order: u_i = v_i = i/N (sorted already)."""
    u = np.arange(N, dtype=np.float64) / max(N, 1)
    return np.ascontiguousarray(np.stack([u, u], axis=1))


def antichain_lightcone(N: int) -> np.ndarray:
    """Mutually unrelated points: u_i = i/N, v_i = 1 - i/N, sorted by time."""
    u = np.arange(N, dtype=np.float64) / max(N, 1)
    c = np.stack([u, 1.0 - u], axis=1)
    return _sort_rows(c, (c[:, 0] + c[:, 1]) / 2.0, c[:, 0])


@dataclasses.dataclass(frozen=True)
class Config:
    """One BASELINE.json workload."""
    index: int          # 1..5
    name: str
    N: int
    dim: int
    geometry: int
    batch: int = 1      # >1: independent causets (config 5)
    kmax: int = -1      # -1: full histogram (k = 0..N-2)

    @property
    def seed(self) -> int:
        return SEED_BASE + self.index


CONFIGS = {
    1: Config(1, "mink2_diamond_N1024", 1024, 2, GEOM_MINK2_LIGHTCONE),
    2: Config(2, "mink2_diamond_N16384", 16384, 2, GEOM_MINK2_LIGHTCONE),
    3: Config(3, "mink4_diamond_N65536", 65536, 4, GEOM_MINK_CONE),
    4: Config(4, "ds2_slab_N131072", 131072, 2, GEOM_DS2_SLAB),
    5: Config(5, "mink4_ensemble_4096xN2048", 2048, 4, GEOM_MINK_CONE, batch=4096, kmax=3),
}


def sprinkle(geometry: int, dim: int, N: int, seed: int) -> np.ndarray:
    if geometry == GEOM_MINK2_LIGHTCONE and dim == 2:
        return sprinkle_mink2_lightcone(N, seed)
    if geometry == GEOM_MINK_CONE and dim == 4:
        return sprinkle_mink4_diamond(N, seed)
    if geometry == GEOM_MINK_CONE and dim == 5:
        return sprinkle_mink5_diamond(N, seed)
    if geometry == GEOM_DS4_SPHERICAL and dim == 7:
        return sprinkle_ds4_spherical(N, seed)
    if geometry == GEOM_MINK_CONE and dim in (2, 3):
        # lower-dimensional flat diamonds: take the first `dim` coordinates of a
        # cube rejection restricted to those coordinates
        return _sprinkle_mink_low(N, dim, seed)
    if geometry == GEOM_DS2_SLAB and dim == 2:
        return sprinkle_ds2_slab(N, seed)
    if geometry == GEOM_FLRW_POLAR and dim == 6:
        return sprinkle_flrw_polar(N, seed)
    raise ValueError("no sprinkler for geometry=%d dim=%d" % (geometry, dim))


def _sprinkle_mink_low(N: int, dim: int, seed: int) -> np.ndarray:
    out = np.empty((N, dim), dtype=np.float64)
    have = 0
    trial = 0
    while have < N:
        batch = max(4096, int((N - have) * (4 if dim < 5 else 18)))
        r = 2.0 * uniform01(seed, dim * trial, dim * batch).reshape(batch, dim) - 1.0
        ok = np.abs(r[:, 0]) + np.sqrt((r[:, 1:] ** 2).sum(axis=1)) <= 1.0
        acc = r[ok]
        take = min(N - have, acc.shape[0])
        out[have:have + take] = acc[:take]
        have += take
        trial += batch
    return _sort_rows(out, out[:, 0], out[:, 1])


def make_config_coords(cfg: Config, N: int | None = None, batch_index: int = 0) -> np.ndarray:
    """Coordinates of config `cfg` (optionally at a reduced N, for tests).
    Config 5: causet `batch_index` uses seed cfg.seed*4096 + batch_index."""
    n = cfg.N if N is None else N
    seed = cfg.seed if cfg.batch == 1 else cfg.seed * 4096 + batch_index
    return sprinkle(cfg.geometry, cfg.dim, n, seed)


def make_ensemble_coords(cfg: Config, B: int | None = None, N: int | None = None) -> np.ndarray:
    """[B][N][dim] for the batched config."""
    b = cfg.batch if B is None else B
    return np.ascontiguousarray(np.stack([make_config_coords(cfg, N, i) for i in range(b)], axis=0))
