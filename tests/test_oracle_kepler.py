"""Pins for the oracle's Kepler drift and Stumpff functions (Eq. 9; L230).

The reference is the analytic two-body orbit evaluated from orbital elements with
mpmath at 40 digits (Kepler's equation in E or H), i.e. not the oracle's formula.
"""
import mpmath as mp
import numpy as np
import pytest

import oracle

mp.mp.dps = 40


def analytic_orbit(mu, a, e, M):
    """Position/velocity in the orbital plane at mean anomaly M (elliptic a>0, hyperbolic a<0)."""
    mu, a, e, M = map(mp.mpf, (mu, a, e, M))
    if e < 1:
        E = mp.findroot(lambda E: E - e * mp.sin(E) - M, M + e * mp.sin(M), tol=mp.mpf(10) ** -38, maxsteps=200)
        r = a * (1 - e * mp.cos(E))
        n = mp.sqrt(mu / a**3)
        x, y = a * (mp.cos(E) - e), a * mp.sqrt(1 - e * e) * mp.sin(E)
        vx, vy = -a * a * n * mp.sin(E) / r, a * a * n * mp.sqrt(1 - e * e) * mp.cos(E) / r
    else:
        aa = -a
        H = mp.findroot(lambda H: e * mp.sinh(H) - H - M, mp.asinh(M / e), tol=mp.mpf(10) ** -38, maxsteps=200)
        r = aa * (e * mp.cosh(H) - 1)
        n = mp.sqrt(mu / aa**3)
        x, y = aa * (e - mp.cosh(H)), aa * mp.sqrt(e * e - 1) * mp.sinh(H)
        vx, vy = -aa * aa * n * mp.sinh(H) / r, aa * aa * n * mp.sqrt(e * e - 1) * mp.cosh(H) / r
    return (x, y), (vx, vy), n


ROT = np.array([[0.36, 0.48, -0.8], [-0.8, 0.6, 0.0], [0.48, 0.64, 0.6]])  # orthonormal


def to3(p):
    return ROT.T @ np.array([float(p[0]), float(p[1]), 0.0])


@pytest.mark.parametrize("e", [0.0, 0.01, 0.3, 0.7, 0.9, 0.99, 1.5, 3.0])
@pytest.mark.parametrize("frac", [0.013, 0.2, -0.11, 0.9])
def test_single_drift_matches_analytic_orbit(e, frac):
    """One drift of |h| <= one period (or time unit, hyperbolic) vs the analytic orbit, 1e-13 relative."""
    mu = 1.3
    a = 1.7 if e < 1 else -1.7
    M0 = 0.4 if e < 1 else -0.8
    (p0, v0, n) = analytic_orbit(mu, a, e, M0)
    h = frac * (2 * mp.pi / n if e < 1 else 3 / n)
    (p1, v1, _) = analytic_orbit(mu, a, e, M0 + n * h)
    # rotate with mpmath-evaluated coordinates rounded to double at the end
    q, V, it = oracle.kepler_drift(mu, float(h), to3(p0), to3(v0))
    q1, V1 = to3(p1), to3(v1)
    # 1e-13 relative (north_star).  Near e = 1 the map amplifies the 1e-16 rounding of the
    # double-precision INPUT state by ~1/|1-e|, which no solver can undo: widen there only.
    tol = 1e-13 * max(1.0, 0.1 / abs(1 - e))
    assert np.linalg.norm(q - q1) <= tol * np.linalg.norm(q1)
    assert np.linalg.norm(V - V1) <= tol * np.linalg.norm(V1)
    assert 0 < it <= 60


def test_invariants_and_phase_over_1e4_orbits():
    """north_star: "two-body drift must match the analytic orbit to 1e-13 relative over 1e4 orbits" (reading R-18).
    650 146 repeated 6-day drifts = 1e4 orbits at a = 1.04 AU, e = 0.043.
    (i) The invariants -- energy, angular momentum vector, eccentricity vector -- hold to a few 1e-13: they random-walk
        with the ~6.5e5 roundings.  Measured on this oracle: |dE/E| = 1.9e-13, |dL|/|L| = 9.1e-14, |dA| = 1.5e-13
        (absolute, |A| = e = 0.043); the bounds below are ~2.5x those, not the 1e-13 of a single drift.
    (ii) The along-track PHASE cannot hold 1e-13 in FP64: the mean anomaly alone carries eps * 2 pi * 1e4 = 1.4e-11, and
        an energy error dE shifts the mean motion by 1.5 dE/E, so the phase error is bounded by 1.5 * (2 pi 1e4) *
        max|dE/E| over the run.  The position against the analytic orbit (mpmath, 40 digits, Kepler's equation solved
        at the final time) is asserted against that bound.  Measured: 1.2e-9 relative (bound 1.9e-8)."""
    mu, h = 1.0, 6 * 0.01720209895
    q = np.array([1.0, 0.0, 0.0]); V = np.array([0.0, 1.02, 0.05])
    q0, V0 = q.copy(), V.copy()
    def inv(q, V):
        E = 0.5 * V @ V - mu / np.linalg.norm(q)
        L = np.cross(q, V)
        A = np.cross(V, L) / mu - q / np.linalg.norm(q)
        return E, L, A
    E0, L0, A0 = inv(q, V)
    a = -mu / (2 * E0)
    norbits = 1e4
    nsteps = int(norbits * 2 * np.pi * a**1.5 / h)
    lib = oracle.lib()
    worst_dE = 0.0
    for k in range(nsteps):
        assert lib.ora_kepler_drift(mu, h, q, V) > 0
        if k % 1000 == 999:
            worst_dE = max(worst_dE, abs(inv(q, V)[0] - E0) / abs(E0))
    E1, L1, A1 = inv(q, V)
    worst_dE = max(worst_dE, abs(E1 - E0) / abs(E0))
    assert worst_dE <= 5e-13
    assert np.linalg.norm(L1 - L0) <= 2.5e-13 * np.linalg.norm(L0)
    assert np.linalg.norm(A1 - A0) <= 4e-13
    # analytic position at t = nsteps * h from the initial state, in mpmath: elements, Kepler's equation, f and g
    mq, mv = [mp.mpf(x) for x in q0], [mp.mpf(x) for x in V0]
    dot = lambda u, w: sum(x * y for x, y in zip(u, w))
    r0 = mp.sqrt(dot(mq, mq))
    am = 1 / (2 / r0 - dot(mv, mv) / mu)
    n = mp.sqrt(mu / am**3)
    ecosE, esinE = 1 - r0 / am, dot(mq, mv) / mp.sqrt(mu * am)
    ecc = mp.sqrt(ecosE**2 + esinE**2)
    Ea = mp.atan2(esinE, ecosE)
    T = mp.mpf(h) * nsteps
    M1 = Ea - esinE + n * T
    Eb = mp.findroot(lambda E: E - ecc * mp.sin(E) - M1, M1, tol=mp.mpf(10) ** -35)
    dE = Eb - Ea
    f, g = 1 - am / r0 * (1 - mp.cos(dE)), T - (dE - mp.sin(dE)) / n
    q1 = [f * x + g * v for x, v in zip(mq, mv)]
    err = float(mp.sqrt(sum((mp.mpf(float(u)) - w) ** 2 for u, w in zip(q, q1))) / mp.sqrt(dot(q1, q1)))
    bound = 1.5 * 2 * np.pi * norbits * worst_dE + 2.2e-16 * 2 * np.pi * norbits
    print("phase error after 1e4 orbits: %.3e relative (bound %.3e, max |dE/E| %.3e)" % (err, bound, worst_dE))
    assert err <= bound
    assert err <= 2e-8


def test_drift_group_property_and_reversal():
    mu = 1.0
    q0 = np.array([0.8, 0.1, -0.05]); V0 = np.array([-0.1, 1.2, 0.02])
    qa, Va, _ = oracle.kepler_drift(mu, 0.3, q0, V0)
    qb, Vb, _ = oracle.kepler_drift(mu, 0.45, qa, Va)
    qc, Vc, _ = oracle.kepler_drift(mu, 0.75, q0, V0)
    assert np.allclose(qb, qc, rtol=0, atol=5e-15) and np.allclose(Vb, Vc, rtol=0, atol=5e-15)
    qd, Vd, _ = oracle.kepler_drift(mu, -0.75, qc, Vc)
    assert np.allclose(qd, q0, rtol=0, atol=5e-15) and np.allclose(Vd, V0, rtol=0, atol=5e-15)


@pytest.mark.parametrize("x", [0.0, 1e-9, -1e-7, 0.3, -0.7, 1.0, -1.0, 1.0000001, 9.0, 40.0, -25.0, 300.0])
def test_stumpff_against_mpmath(x):
    c = oracle.stumpff(x)
    X = mp.mpf(x)
    if x == 0:
        ref = [1, 1, mp.mpf(1) / 2, mp.mpf(1) / 6]
    else:
        s = mp.sqrt(X)  # complex for X<0: cos(i y) = cosh y etc.
        ref = [mp.cos(s), mp.sin(s) / s, (1 - mp.cos(s)) / X, (s - mp.sin(s)) / s**3]
    for k in range(4):
        r = float(mp.re(ref[k]))
        # closed forms lose a little to cancellation in (1-c0)/x at large |x|
        assert abs(c[k] - r) <= 4e-16 * max(abs(r), 1.0) * (1 + abs(x)), (k, c[k], r)
