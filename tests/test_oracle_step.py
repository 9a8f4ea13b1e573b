"""Pins for the composed maps: Eq. 7 (L98-108), the per-step algorithm (L144-166) and the
higher-order compositions (L168-170)."""
import numpy as np
import pytest

import oracle
import workloads
from workloads import DAY


def test_yoshida_order_conditions():
    """[R-6] sum w = 1, sum w^3 = 0 (order 4), and sum w^5 = 0 too (order 6, solution A)."""
    w4, w6 = oracle.yoshida(4), oracle.yoshida(6)
    assert len(w4) == 3 and len(w6) == 7
    assert abs(w4.sum() - 1) < 1e-15 and abs((w4**3).sum()) < 1e-14
    assert np.array_equal(w6, w6[::-1])
    assert abs(w6.sum() - 1) < 1e-14 and abs((w6**3).sum()) < 1e-13 and abs((w6**5).sum()) < 1e-12
    assert np.array_equal(oracle.yoshida(2), [1.0])


def _max_energy_error(w, order, dt_days, T_days, **kw):
    s = oracle.System(1.0, w["m"], w["x"], w["v"], **kw)
    E0, _ = s.energy()
    worst = 0.0
    for _ in range(int(T_days / dt_days)):
        s.step(1, dt_days * DAY, order)
        worst = max(worst, abs((s.energy()[0] - E0) / E0))
    return worst, s


@pytest.mark.parametrize("order,lo,hi", [(2, 3.5, 4.6), (4, 13, 20), (6, 45, 130)])
def test_energy_error_scales_as_dt_to_the_order_without_encounters(order, lo, hi):
    """K == 1 (n1 = n2 = 0): the democratic-heliocentric Wisdom-Holman limit (L92)."""
    w = workloads.config0()
    e1, _ = _max_energy_error(w, order, 24, 960, n1=0.0, n2=0.0)
    e2, _ = _max_energy_error(w, order, 12, 960, n1=0.0, n2=0.0)
    assert lo < e1 / e2 < hi, (e1, e2)


def _close_pair_system():
    """two 1e-4 planets on neighbouring orbits that meet inside r_crit within a few steps"""
    m = np.array([1e-4, 1e-4, 3e-5])
    a = np.array([1.0, 1.03, 2.2]); e = np.array([0.0, 0.0, 0.05])
    M = np.array([0.0, -0.03, 1.0])
    x, v = workloads.elements_to_cartesian(1.0 + m, a, e, np.array([0.0, 0.01, 0.02]),
                                           np.zeros(3), np.zeros(3), M)
    return dict(m=m, x=np.ascontiguousarray(x), v=np.ascontiguousarray(v))


@pytest.mark.parametrize("order,dt_days,lo,hi", [(2, 2.0, 3.5, 4.6), (4, 4.0, 13, 20), (6, 8.0, 45, 90)])
def test_energy_error_scaling_with_pairs_inside_rcrit(order, dt_days, lo, hi):
    """|dE/E| ~ dt^p for p = 2, 4, 6 on a run WITH pairs inside r_crit (n2 = 0, so r_crit does not
    depend on dt; the pair spends the whole run inside 3 R_H and Bulirsch-Stoer runs in every map).  Halving dt must
    divide the error by 2^p: this is what constrains reading R-4 (r_crit frozen over the substeps of a step -- a
    substep that moved the changeover boundary would not be the same one-parameter map and the h^3 / h^5 terms of the
    composition would not cancel).  Measured: 4.00, 16.04, 64.7 (dt chosen per order above the 1e-14 floor)."""
    w = _close_pair_system()
    kw = dict(n1=6.0, n2=0.0)
    ea, s = _max_energy_error(w, order, dt_days, 120, **kw)
    assert s.stats()["groups"] >= 15          # BS really ran, in every map
    eb, _ = _max_energy_error(w, order, dt_days / 2, 120, **kw)
    assert lo < ea / eb < hi, (order, ea, eb, ea / eb)


def test_time_reversal_of_the_map_with_frozen_rcrit():
    """[R-13] S2(-h) S2(h) = identity when r_crit is frozen, encounters included."""
    w = _close_pair_system()
    s = oracle.System(1.0, w["m"], w["x"], w["v"], n1=6.0, n2=0.0)
    s.accel_now(2 * DAY)                      # fixes rc
    q0, V0, _ = s.demo()
    for _ in range(5):
        s.map_s2(2 * DAY)
    assert len(s.encounters()[1]) >= 1
    for _ in range(5):
        s.map_s2(-2 * DAY)
    q1, V1, _ = s.demo()
    assert np.abs(q1 - q0).max() < 5e-11 and np.abs(V1 - V0).max() < 5e-11


def test_angular_momentum_conserved_by_full_steps():
    w = workloads.config4(n=256)
    s = oracle.System(1.0, w["m"], w["x"], w["v"])
    _, L0 = s.energy()
    s.step(20, w["dt"], 4)
    _, L1 = s.energy()
    assert s.stats()["groups"] > 0
    assert np.linalg.norm(L1 - L0) <= 1e-12 * np.linalg.norm(L0)


def _brute_force_pairs(s, h):
    """S2's encounter set rebuilt from the oracle's component functions, every pair tested by
    dense sampling of Eq. 10 (numpy), no prechecker."""
    lib = oracle.lib()
    n = s.n
    q, V, rc = s.demo()
    a, _ = oracle.accel(s.G, s.m, q, rc)
    V = V + 0.5 * h * a
    lib.ora_sun_kick(n, n, s.m0, s.m, V, q, 0.5 * h)
    q0, V0 = q.copy(), V.copy()
    for i in range(n):
        qi, Vi, _ = oracle.kepler_drift(s.G * s.m0, h, q0[:, i], V0[:, i])
        q[:, i], V[:, i] = qi, Vi
    t = np.linspace(0, 1, 20001)
    out, margin = set(), {}
    for i in range(n):
        for j in range(i + 1, n):
            d0, d1 = q0[:, j] - q0[:, i], q[:, j] - q[:, i]
            w0, w1 = V0[:, j] - V0[:, i], V[:, j] - V[:, i]
            P0, P1, Pd0, Pd1 = d0 @ d0, d1 @ d1, 2 * d0 @ w0, 2 * d1 @ w1
            P = (P0 * (1 + 2 * t) * (1 - t) ** 2 + P1 * t**2 * (3 - 2 * t)
                 + Pd0 * t * (1 - t) ** 2 * h + Pd1 * t**2 * (t - 1) * h)
            rcij = max(rc[i], rc[j])
            margin[(i, j)] = P.min() / rcij**2 - 1
            if P.min() < rcij**2:
                out.add((i, j))
    return out, margin


@pytest.mark.parametrize("seed", [0, 11, 12])
def test_encounter_sets_match_brute_force_small_n(seed):
    """N <= 16: candidate -> confirm pipeline == all-pairs brute force, and == the no-cull mode [R-9]."""
    w = workloads.config4(seed=seed, n=16)
    w["m"] = w["m"] * 3000                     # Hill radii large enough for several encounters
    sA = oracle.System(1.0, w["m"], w["x"], w["v"])
    sB = oracle.System(1.0, w["m"], w["x"], w["v"]); sB.set_cull(0)
    total = 0
    for step in range(12):
        sA.accel_now(w["dt"]); sB.accel_now(w["dt"])
        want, margin = _brute_force_pairs(sA, w["dt"])
        sA.map_s2(w["dt"]); sB.map_s2(w["dt"])
        got = set(map(tuple, sA.encounters()[1])); got_nocull = set(map(tuple, sB.encounters()[1]))
        assert got == got_nocull
        diff = {p for p in want ^ got if abs(margin[p]) > 1e-6}   # dense sampling resolution
        assert not diff, (step, diff)
        total += len(got)
        qa, Va, _ = sA.demo(); qb, Vb, _ = sB.demo()
        assert np.array_equal(qa, qb) and np.array_equal(Va, Vb)
    assert total >= 5


def test_massless_particles_are_independent_and_match_tiny_masses():
    """Test-particle mode (L334-342): a particle's path does not depend on other particles, and
    equals that of a body of negligible mass in massive mode."""
    w = workloads.config2(n_massive=3, n_test=40)
    # put a few particles next to planet 1 so that particle groups form
    x, v = w["x"].copy(), w["v"].copy()
    V = oracle.helio_to_demo(1.0, w["m"], v, 3)
    rc1 = oracle.rcrit(1.0, 1.0, 3.0, 0.4, w["dt"], w["m"], x, V)[1]
    for k in range(5):                         # radial offsets of 0.25..1.25 r_crit, Keplerian shear
        f = 0.25 * (k + 1) * rc1 / np.linalg.norm(x[:, 1])
        x[:, 3 + k] = x[:, 1] * (1 + f); v[:, 3 + k] = v[:, 1] * (1 - 0.5 * f)
    full = oracle.System(1.0, w["m"], x, v, n_massive=3)
    full.step(6, w["dt"], 2)
    assert full.stats()["groups"] > 0
    xf, vf = full.state()
    keep = [0, 1, 2, 3, 5, 20]
    sub = oracle.System(1.0, w["m"][keep], np.ascontiguousarray(x[:, keep]), np.ascontiguousarray(v[:, keep]), n_massive=3)
    sub.step(6, w["dt"], 2)
    xs, vs = sub.state()
    assert np.array_equal(xs, xf[:, keep]) and np.array_equal(vs, vf[:, keep])
    # the same six bodies all "massive", the particles with mass 1e-30
    m2 = w["m"][keep].copy(); m2[3:] = 1e-30
    allm = oracle.System(1.0, m2, np.ascontiguousarray(x[:, keep]), np.ascontiguousarray(v[:, keep]))
    # particles then carry a Hill radius of ~0; r_crit = n2 tau v as for test particles
    allm.step(6, w["dt"], 2)
    xm, vm = allm.state()
    assert np.abs(xm - xs).max() < 1e-9 and np.abs(vm - vs).max() < 1e-9


def test_multi_system_is_a_loop_over_independent_systems():
    w = workloads.config3(n_systems=3)
    sim = oracle.Sim(w)
    sim.step(5)
    x, v = sim.state()
    one = oracle.System(1.0, w["m"][16:32], w["x"][:, 16:32], w["v"][:, 16:32])
    one.step(5, w["dt"], 2)
    x1, v1 = one.state()
    assert np.array_equal(x[:, 16:32], x1) and np.array_equal(v[:, 16:32], v1)
