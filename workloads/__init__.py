"""Seeded synthetic inputs shaped like the paper's workloads.

This module serves BOTH the CUDA path and the oracle and therefore holds none of
the method's arithmetic: only a counter-based RNG (SplitMix64), the draws of
orbital elements, and the textbook elements -> Cartesian conversion.  The
paper's own initial-condition files are
not available; these stand in for them.

Units: G = 1, AU, M_sun, time unit = 1 day / k with the Gaussian constant k, so
dt(6 d) = 6 k.  All state is heliocentric (x, v), SoA arrays of shape (3, N).
"""
from __future__ import annotations

import numpy as np

K_GAUSS = 0.01720209895
M_EARTH = 3.0034893e-6          # M_sun
RHO_2GCC = 3.3673417e6          # 2 g/cm^3 in M_sun / AU^3
DAY = K_GAUSS                   # one day in code time units

_M64 = np.uint64(0xFFFFFFFFFFFFFFFF)


def splitmix64_uniform(seed: int, count: int, offset: int = 0) -> np.ndarray:
    """u_k in [0,1), k = offset .. offset+count-1, of the SplitMix64 stream of `seed`."""
    with np.errstate(over="ignore"):
        k = np.arange(offset + 1, offset + count + 1, dtype=np.uint64)
        z = np.uint64(seed & 0xFFFFFFFFFFFFFFFF) + k * np.uint64(0x9E3779B97F4A7C15)
        z = (z ^ (z >> np.uint64(30))) * np.uint64(0xBF58476D1CE4E5B9)
        z = (z ^ (z >> np.uint64(27))) * np.uint64(0x94D049BB133111EB)
        z = z ^ (z >> np.uint64(31))
    return (z >> np.uint64(11)).astype(np.float64) * (1.0 / 9007199254740992.0)


def _rayleigh(u, sigma):
    return sigma * np.sqrt(-2.0 * np.log1p(-u))


def _log_uniform(u, lo, hi):
    return lo * (hi / lo) ** u


def elements_to_cartesian(mu, a, e, inc, Om, om, M):
    """Textbook two-body elements -> heliocentric position/velocity (vectorised)."""
    E = M + e * np.sin(M)
    for _ in range(60):
        E = E - (E - e * np.sin(E) - M) / (1.0 - e * np.cos(E))
    cE, sE = np.cos(E), np.sin(E)
    b = np.sqrt(1.0 - e * e)
    n = np.sqrt(mu / a**3)
    xp, yp = a * (cE - e), a * b * sE
    rr = a * (1.0 - e * cE)
    vxp, vyp = -a * a * n * sE / rr, a * a * n * b * cE / rr
    cO, sO, co, so, ci, si = np.cos(Om), np.sin(Om), np.cos(om), np.sin(om), np.cos(inc), np.sin(inc)
    r11, r12 = cO * co - sO * so * ci, -cO * so - sO * co * ci
    r21, r22 = sO * co + cO * so * ci, -sO * so + cO * co * ci
    r31, r32 = so * si, co * si
    x = np.stack([r11 * xp + r12 * yp, r21 * xp + r22 * yp, r31 * xp + r32 * yp])
    v = np.stack([r11 * vxp + r12 * vyp, r21 * vxp + r22 * vyp, r31 * vxp + r32 * vyp])
    return x, v


def _draw(seed, n, offset, mass, a, e, inc, m0=1.0):
    """Per body, in fixed order: mass, a, e, i, Omega, omega, M (7 uniforms)."""
    u = splitmix64_uniform(seed, 7 * n, 7 * offset).reshape(n, 7).T
    m = mass(u[0])
    aa = a(u[1])
    ee = np.minimum(e(u[2]), 0.9)
    ii = inc(u[3])
    Om, om, M = 2 * np.pi * u[4], 2 * np.pi * u[5], 2 * np.pi * u[6]
    x, v = elements_to_cartesian(m0 + m, aa, ee, ii, Om, om, M)
    return m, x, v


def _radius(m):
    return np.cbrt(3.0 * m / (4.0 * np.pi * RHO_2GCC))


def _pack(mode, m0, m, x, v, *, n_massive, n_test=0, n_systems=1, dt_days, order, n_steps, name):
    return dict(name=name, mode=mode, m0=np.atleast_1d(np.asarray(m0, dtype=np.float64)),
                m=np.ascontiguousarray(m), radius=_radius(m),
                x=np.ascontiguousarray(x), v=np.ascontiguousarray(v),
                n_massive=n_massive, n_test=n_test, n_systems=n_systems,
                dt=dt_days * DAY, order=order, n_steps=n_steps,
                G=1.0, n1=3.0, n2=0.4, bs_eps=1e-12)


def config0(seed=0, n=15):
    """BASELINE.json configs[0]: tiny massive mode, 15 bodies, order 2, dt 6 d, 1000 steps."""
    m, x, v = _draw(seed, n, 0, lambda u: _log_uniform(u, 1e-7, 1e-5), lambda u: 0.5 + 3.5 * u,
                    lambda u: _rayleigh(u, 0.01), lambda u: _rayleigh(u, 0.005))
    return _pack(0, 1.0, m, x, v, n_massive=n, dt_days=6.0, order=2, n_steps=1000, name="cfg0")


def config1(seed=1, n=2048):
    """configs[1]: planetesimal disc, 2048 equal masses totalling 2 M_earth, Sigma ~ a^-1.5."""
    mb = 2.0 * M_EARTH / n
    m, x, v = _draw(seed, n, 0, lambda u: np.full_like(u, mb),
                    lambda u: (np.sqrt(0.5) + u * (np.sqrt(4.0) - np.sqrt(0.5))) ** 2,
                    lambda u: _rayleigh(u, 0.01), lambda u: _rayleigh(u, 0.005))
    return _pack(0, 1.0, m, x, v, n_massive=n, dt_days=6.0, order=2, n_steps=10000, name="cfg1")


def config2(seed=2, n_massive=8, n_test=1_000_000):
    """configs[2]: 8 massive bodies + 1e6 massless test particles."""
    mm, xm, vm = _draw(seed, n_massive, 0, lambda u: _log_uniform(u, 1e-6, 1e-3),
                       lambda u: 0.4 + 29.6 * u, lambda u: 0.05 * u, lambda u: _rayleigh(u, 0.005))
    mt, xt, vt = _draw(seed, n_test, n_massive, lambda u: np.zeros_like(u), lambda u: 0.5 + 4.5 * u,
                       lambda u: _rayleigh(u, 0.05), lambda u: _rayleigh(u, 0.03))
    m = np.concatenate([mm, mt])
    x = np.concatenate([xm, xt], axis=1)
    v = np.concatenate([vm, vt], axis=1)
    return _pack(1, 1.0, m, x, v, n_massive=n_massive, n_test=n_test, dt_days=6.0, order=2,
                 n_steps=1000, name="cfg2")


def config3(seed=3, n_systems=4096, n_per=16):
    """configs[3]: independent systems of 16 bodies drawn as config 0, per-system seed."""
    ms, xs, vs = [], [], []
    for s in range(n_systems):
        m, x, v = _draw(seed * (1 << 20) + s, n_per, 0, lambda u: _log_uniform(u, 1e-7, 1e-5),
                        lambda u: 0.5 + 3.5 * u, lambda u: _rayleigh(u, 0.01),
                        lambda u: _rayleigh(u, 0.005))
        ms.append(m); xs.append(x); vs.append(v)
    m = np.concatenate(ms)
    x = np.concatenate(xs, axis=1)
    v = np.concatenate(vs, axis=1)
    return _pack(2, np.ones(n_systems), m, x, v, n_massive=n_per, n_systems=n_systems, dt_days=6.0,
                 order=2, n_steps=10000, name="cfg3")


def config4(seed=4, n=2048, order=4):
    """configs[4]: encounter-heavy annulus a = 0.9-1.1 AU, orders 4 and 6, dt 2 d."""
    m, x, v = _draw(seed, n, 0, lambda u: _log_uniform(u, 1e-8, 1e-6), lambda u: 0.9 + 0.2 * u,
                    lambda u: _rayleigh(u, 0.05), lambda u: _rayleigh(u, 0.02))
    return _pack(0, 1.0, m, x, v, n_massive=n, dt_days=2.0, order=order, n_steps=5000, name="cfg4")


CONFIGS = {0: config0, 1: config1, 2: config2, 3: config3, 4: config4}


def shard_bounds(n, rank, world):
    """Balanced contiguous split of n units over world ranks: [lo, hi) of this rank."""
    return (n * rank) // world, (n * (rank + 1)) // world


def shard(w, rank, world):
    """The part of workload w that rank `rank` of `world` integrates (no data-path collective).

    Test-particle mode: the massive bodies are replicated on every rank and integrated redundantly, the
    particles are partitioned.  Multi-system mode: the systems are partitioned.  Massive mode does not
    shard (every force evaluation needs all positions): ValueError -- replicas only.
    """
    if not 0 <= rank < world:
        raise ValueError("rank %d outside world %d" % (rank, world))
    if w["mode"] == 0:
        raise ValueError("massive mode does not shard: replicas only")
    out = dict(w)
    if w["mode"] == 1:
        nm = w["n_massive"]
        lo, hi = shard_bounds(w["n_test"], rank, world)
        idx = np.concatenate([np.arange(nm), nm + np.arange(lo, hi)])
        out["n_test"] = hi - lo
    else:
        nm = w["n_massive"]
        lo, hi = shard_bounds(w["n_systems"], rank, world)
        idx = np.arange(lo * nm, hi * nm)
        out["n_systems"] = hi - lo
        out["m0"] = np.ascontiguousarray(w["m0"][lo:hi])
    out["m"] = np.ascontiguousarray(w["m"][idx])
    out["radius"] = np.ascontiguousarray(w["radius"][idx])
    out["x"] = np.ascontiguousarray(w["x"][:, idx])
    out["v"] = np.ascontiguousarray(w["v"][:, idx])
    out["shard"] = (rank, world, int(lo), int(hi))
    return out
