"""Pins for the oracle's collisions, ejections and removal (section 3.2.7-3.2.8).

What the paper fixes: the pair merges when r_ij < R_i + R_j; linear momentum is conserved; the internal energy
U = 1/2 mu v_ij^2 - G m_i m_j / r_ij; the index rule; the ghost; the detection "between the Bulirsch-Stoer steps with the
code of the encounter detection".  The references here are closed forms of the two-body problem (free-fall time,
periapsis of a hyperbolic fly-by), conservation laws, and runs without the colliding body."""
import numpy as np
import pytest

import oracle
import workloads

G = 1.0


def _pair(r0, b, vinf, m=(3e-6, 1e-6), centre=(50.0, 0.0, 0.0)):
    """two bodies far from a negligible star, approaching along x with impact parameter b and relative speed vinf"""
    m = np.array(m)
    q = np.array([[centre[0] - r0 * m[1] / m.sum(), centre[0] + r0 * m[0] / m.sum()], [centre[1] - b * m[1] / m.sum(), centre[1] + b * m[0] / m.sum()], [0.0, 0.0]])
    V = np.array([[vinf * m[1] / m.sum(), -vinf * m[0] / m.sum()], [0.0, 0.0], [0.0, 0.0]])
    return m, q, V


def test_free_fall_collision_time():
    """Two bodies released at rest at separation r0 touch (separation R_i + R_j) after the closed-form free-fall time
    t_c = sqrt(r0^3 / (2 mu)) (sqrt(x (1 - x)) + arccos(sqrt(x))), x = (R_i + R_j) / r0, mu = G (m_i + m_j): the oracle
    reports no collision over 0.9 t_c and one over 1.1 t_c (the star is 1e-20: a pure two-body problem; rc is large, so
    the whole pair force is integrated by Bulirsch-Stoer)."""
    m, q, V = _pair(1e-3, 0.0, 0.0)
    R = np.array([3e-5, 2e-5])
    x = R.sum() / 1e-3
    tc = np.sqrt(1e-9 / (2 * G * m.sum())) * (np.sqrt(x * (1 - x)) + np.arccos(np.sqrt(x)))
    rc = np.array([1.0, 1.0])
    out = oracle.bs_group_collide(G, 1e-20, m, rc, R, q, V, 0.9 * tc)
    assert len(out[7]) == 0 and np.array_equal(out[4], [0, 0])
    out = oracle.bs_group_collide(G, 1e-20, m, rc, R, q, V, 1.1 * tc)
    assert len(out[7]) == 1 and np.array_equal(out[4], [0, 2])


@pytest.mark.parametrize("factor,hit", [(1.1, True), (0.9, False)])
def test_collision_iff_periapsis_inside_the_radii(factor, hit):
    """Hyperbolic fly-by with impact parameter b and speed v at infinity: periapsis d_p = -a + sqrt(a^2 + b^2),
    a = mu / v^2.  Radii summing to 1.1 d_p collide, to 0.9 d_p do not (the Hermite minimum over a Bulirsch-Stoer step
    is an interpolation: 10 % is far more than its error)."""
    b, vinf = 2e-4, 0.05
    m, q, V = _pair(5e-3, b, vinf)
    a = G * m.sum() / vinf**2
    # the pair starts at finite distance: energy and angular momentum give the exact periapsis
    r0 = np.hypot(5e-3, b)
    E = 0.5 * vinf**2 - G * m.sum() / r0
    Lz = b * vinf
    dp = (-G * m.sum() + np.sqrt((G * m.sum()) ** 2 + 2 * E * Lz**2)) / (2 * E)
    assert 0 < dp < b and a > 0
    R = np.array([0.6, 0.4]) * factor * dp
    out = oracle.bs_group_collide(G, 1e-20, m, np.array([1.0, 1.0]), R, q, V, 2 * 5e-3 / vinf)
    assert (len(out[7]) == 1) == hit


def test_merge_conserves_mass_momentum_and_accounts_the_energy():
    """Across a merge: sum m and sum m V unchanged to rounding (L316 "linear momentum is conserved"); the merged position
    is the centre of mass; U = 1/2 mu v^2 - G m_i m_j / r at the merge state (L318-322); E + U of the isolated pair is
    conserved; the spin is the pair's orbital angular momentum about its centre of mass (L324); the heavier body keeps
    its index."""
    m, q, V = _pair(1e-3, 2.8e-4, 0.05)          # periapsis ~ 2.5e-5: half the sum of the radii
    R = np.array([3e-5, 2e-5])
    P0 = (m * V).sum(1); M0 = m.sum()
    mu = m.prod() / m.sum()
    d0, w0 = q[:, 0] - q[:, 1], V[:, 0] - V[:, 1]
    E0 = 0.5 * mu * w0 @ w0 - G * m.prod() / np.linalg.norm(d0)     # energy of the relative motion (the centre of mass moves freely)
    L0 = mu * np.cross(d0, w0)
    q1, V1, m1, R1, kind, spin, U, ev = oracle.bs_group_collide(G, 1e-20, m, np.array([1.0, 1.0]), R, q, V, 0.5)
    assert len(ev) == 1 and np.array_equal(kind, [0, 2])
    assert m1[0] == M0 and m1[1] == 0.0 and R1[1] == 0.0
    assert abs(R1[0] ** 3 - (R[0] ** 3 + R[1] ** 3)) < 1e-15 * R1[0] ** 3 * 4
    assert np.abs((m1 * V1).sum(1) - P0).max() <= 1e-12 * np.abs(m * np.abs(V).max()).sum()   # the Bulirsch-Stoer steps before the merge round too
    assert abs(U - E0) <= 1e-8 * abs(E0)                      # all the relative energy went into U (kinetic and potential parts are ~30 |E0| each, integrated to 1e-12)
    assert np.abs(spin[:, 0] - L0).max() <= 1e-9 * np.linalg.norm(L0)
    assert ev[0][2] == 0 and ev[0][3] == 1 and ev[0][1] == 0 and abs(ev[0][20] - U) < 1e-20
    # the report holds the two states of the last Bulirsch-Stoer step before the collision: still apart
    assert np.linalg.norm(ev[0][8:11] - ev[0][14:17]) > R.sum()
    # the ghost sits on its parking orbit
    assert q1[0, 1] == 2000.0 and V1[1, 1] == np.sqrt(G * 1e-20 / 2000.0)


def test_index_rule():
    """L324: the index of the more massive body; the smaller index if the masses are equal."""
    for masses, survivor in [((1e-6, 3e-6), 1), ((3e-6, 1e-6), 0), ((2e-6, 2e-6), 0)]:
        m, q, V = _pair(1e-3, 0.0, 0.01, m=masses)
        out = oracle.bs_group_collide(G, 1e-20, m, np.array([1.0, 1.0]), np.array([3e-5, 3e-5]), q, V, 0.5)
        assert out[4][survivor] == 0 and out[4][1 - survivor] == 2 and out[7][0][2] == survivor


def _colliding_system():
    """three planets about a solar-mass star; body 1 sits 0.003 AU ahead of body 0 on the same orbit and moves 1 %
    slower: they touch (radii 4e-4 + 3e-4) after ~13 days"""
    m = np.array([3e-6, 1e-6, 2e-6])
    x = np.array([[1.0, 1.0003, -2.5], [0.0, 0.003, 0.0], [0.0, 0.0, 0.01]])   # 3e-4 off the line: no singular head-on passage
    v = np.array([[0.0, 0.0, 0.0], [1.0, 0.99, -np.sqrt(1 / 2.5)], [0.0, 0.0, 0.0]])
    R = np.array([4e-4, 3e-4, 1e-4])
    return dict(m=m, x=np.ascontiguousarray(x), v=np.ascontiguousarray(v), R=R)


def test_full_step_collision_energy_bookkeeping_and_ghost():
    """Whole time steps (L153-166 with "do collisions"): E + U is conserved across the step with the collision as well
    as the integrator conserves E in the steps without one; the ghost is massless, parked, and never met again."""
    w = _colliding_system()
    s = oracle.System(1.0, w["m"], w["x"], w["v"])
    s.set_collisions(w["R"])
    E0 = s.energy()[0]
    seen = None
    for k in range(40):
        s.step(1, 2 * workloads.DAY, 2)
        if seen is None and len(s.events()):
            seen = k
    assert seen is not None
    ev = s.events()
    assert len(ev) == 1 and ev[0][1] == 0 and {int(ev[0][2]), int(ev[0][3])} == {0, 1} and ev[0][0] == seen
    m, R, kind, spin = s.bodies()
    assert kind[1] == 2 and m[1] == 0.0 and m[0] == 4e-6 and kind[0] == 0 and kind[2] == 0
    E1 = s.energy()[0]
    U = s.internal_energy()
    assert abs(U) > 1e-3 * abs(E0) * 1e-3                      # not trivial
    assert abs((E1 + U - E0) / E0) < 1e-7, ((E1 - E0) / E0, U / E0)
    assert abs((E1 - E0) / E0) > 100 * abs((E1 + U - E0) / E0)  # without U the books do not balance
    x, v = s.state()
    assert abs(np.linalg.norm(x[:, 1]) - 2000.0) < 1e-3         # on its parking orbit (it still drifts, and feels the kicks)


def test_test_particle_collision_removes_the_particle_only():
    """L336: a test particle that hits a planetesimal is reported and removed; it has no effect on the planetesimal."""
    w = workloads.config2(n_massive=3, n_test=6)
    x, v = w["x"].copy(), w["v"].copy()
    x[:, 4] = x[:, 1] * (1 + 2e-4); v[:, 4] = v[:, 1] * (1 - 3e-4)         # particle 4 next to planet 1
    R = np.full(9, 1e-5); R[1] = 3e-4
    a = oracle.System(1.0, w["m"], x, v, n_massive=3); a.set_collisions(R)
    keep = [0, 1, 2, 3, 5, 6, 7, 8]
    b = oracle.System(1.0, w["m"][keep], np.ascontiguousarray(x[:, keep]), np.ascontiguousarray(v[:, keep]), n_massive=3); b.set_collisions(R[keep])
    a.step(10, w["dt"], 2); b.step(10, w["dt"], 2)
    ev = a.events()
    assert len(ev) == 1 and ev[0][1] == 1 and ev[0][2] == 1 and ev[0][3] == 4
    xa, va = a.state(); xb, vb = b.state()
    assert np.array_equal(xa[:, keep], xb) and np.array_equal(va[:, keep], vb)
    assert a.bodies()[2][4] == 2 and a.internal_energy() == 0.0


def test_ejections_and_stop_of_the_system():
    """L330-332: beyond Rcut or inside RcutSun -> reported, removed.  L378-384: fewer than Nmin bodies left -> the system
    stops (all its bodies removed)."""
    w = workloads.config0(n=6)
    s = oracle.System(1.0, w["m"], w["x"], w["v"])
    r = np.linalg.norm(w["x"], axis=0)
    far, near = int(r.argmax()), int(r.argmin())
    s.set_collisions(w["radius"], True, rcut=0.5 * (np.sort(r)[-1] + np.sort(r)[-2]), rcut_sun=0.5 * (np.sort(r)[0] + np.sort(r)[1]))
    s.step(1, w["dt"], 2)
    ev = s.events()
    kinds = {int(e[2]): int(e[1]) for e in ev}
    assert kinds == {far: 2, near: 3}
    m, R, kind, _ = s.bodies()
    assert kind[far] == 2 and kind[near] == 2 and m[far] == 0 and (kind == 2).sum() == 2
    s2 = oracle.System(1.0, w["m"], w["x"], w["v"])
    s2.set_collisions(w["radius"], True, rcut=0.5 * (np.sort(r)[-1] + np.sort(r)[-2]), nmin=6)
    s2.step(1, w["dt"], 2)
    ev = s2.events()
    assert len(ev) == 6 and ev[0][1] == 2 and all(e[1] == 4 for e in ev[1:])
    assert (s2.bodies()[2] == 2).all()


def test_collisions_off_is_the_point_mass_path():
    """the default (no call of set_collisions) and collisions switched off are the same, bit for bit"""
    w = _colliding_system()
    a = oracle.System(1.0, w["m"], w["x"], w["v"])
    b = oracle.System(1.0, w["m"], w["x"], w["v"]); b.set_collisions(w["R"], False)
    a.step(12, 2 * workloads.DAY, 2); b.step(12, 2 * workloads.DAY, 2)      # point masses: they pass each other
    assert np.array_equal(a.state()[0], b.state()[0]) and len(b.events()) == 0
