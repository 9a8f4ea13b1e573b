"""Parity of collisions, ejections and removal between the CUDA path and the
oracle: event records (kind, step and bodies exact; states, masses, U to tolerance), the bodies afterwards, the
state, and the energy books E + U."""
import numpy as np
import pytest

import oracle
import workloads

pytestmark = pytest.mark.gpu
STATE_TOL = 1e-9


@pytest.fixture(scope="module")
def G():
    import paper_1404_2324_b200 as G
    from paper_1404_2324_b200 import build
    build.build()
    return G


def relerr(a, b):
    return np.linalg.norm(a - b, axis=0) / np.linalg.norm(b, axis=0)


def sort_events(e):
    return e[np.lexsort((e[:, 3], e[:, 2], e[:, 1], e[:, 0]))] if len(e) else e


def compare(g, o, min_events, kinds=None):
    x, v = g.get_state_host()
    assert g.status() == 0
    xo, vo = o.state()
    eg, eo = sort_events(g.events()), sort_events(o.events())
    assert len(eg) == len(eo) and len(eo) >= min_events, (len(eg), len(eo))
    assert np.array_equal(eg[:, :4], eo[:, :4])                     # step, kind, surviving body, removed body
    if len(eo):
        assert np.allclose(eg[:, 4:], eo[:, 4:], rtol=1e-8, atol=1e-18)
        if kinds is not None:
            assert set(eo[:, 1].astype(int)) == set(kinds), set(eo[:, 1].astype(int))
    m, R, kind, spin, U = g.bodies()
    mo, Ro, ko, so = o.bodies()
    assert np.array_equal(kind, ko)
    assert np.allclose(m, mo, rtol=1e-15, atol=0) and np.allclose(R, Ro, rtol=1e-14, atol=0)
    assert np.allclose(spin, so, rtol=1e-7, atol=1e-20)
    assert np.allclose(U, o.internal_energy(), rtol=1e-8, atol=1e-22)
    alive = ko != 2
    assert relerr(x[:, alive], xo[:, alive]).max(initial=0.0) < STATE_TOL and relerr(v[:, alive], vo[:, alive]).max(initial=0.0) < STATE_TOL
    assert relerr(x[:, ~alive], xo[:, ~alive]).max(initial=0.0) < 1e-9       # the parked bodies too
    return eo


def _colliding_triple():
    m = np.array([3e-6, 1e-6, 2e-6])
    x = np.array([[1.0, 1.0003, -2.5], [0.0, 0.003, 0.0], [0.0, 0.0, 0.01]])
    v = np.array([[0.0, 0.0, 0.0], [1.0, 0.99, -np.sqrt(1 / 2.5)], [0.0, 0.0, 0.0]])
    R = np.array([4e-4, 3e-4, 1e-4])
    return dict(name="triple", mode=0, m0=np.array([1.0]), m=m, radius=R, x=x, v=v, n_massive=3, n_test=0, n_systems=1,
                dt=2 * workloads.DAY, order=2, G=1.0, n1=3.0, n2=0.4, bs_eps=1e-12)


def test_two_planets_merge(G):
    """the three-planet system of the oracle's pin: one collision, the books E + U balance on both sides"""
    w = _colliding_triple()
    g = G.from_workload(w); g.set_collisions(True)
    o = oracle.Sim(w); o.set_collisions(True)
    E0 = g.energy()[0]
    g.step(20, w["dt"], 2); o.step(20, w["dt"], 2)
    ev = compare(g, o, 1, kinds=[0])
    assert len(ev) == 1
    E1 = g.energy()[0]
    U = g.bodies()[4]
    assert abs((E1 + U - E0) / E0)[0] < 1e-7 and abs((E1 - E0) / E0)[0] > 1e-5
    g.close()


@pytest.mark.parametrize("make,inflate,order,nsteps", [
    (lambda: workloads.config4(n=400), 400.0, 2, 12),           # pairs and triples: the block layout notices, the generic one merges
    (lambda: workloads.config4(n=1200), 300.0, 4, 4),           # fourth order: three maps per step
    (lambda: workloads.config1(n=1500), 1000.0, 2, 6),          # groups of up to ~20 bodies: the cluster layout notices
])
def test_many_collisions(G, make, inflate, order, nsteps):
    """discs with radii inflated so that tens of pairs collide within a few steps; events, merged bodies and
    trajectories against the oracle, pair lists and labels after every step"""
    w = dict(make(), order=order)
    w["radius"] = w["radius"] * inflate
    g = G.from_workload(w, max_pairs=400000); g.set_collisions(True)
    o = oracle.Sim(w, cap=400000); o.set_collisions(True)
    for _ in range(nsteps):
        g.step(1, w["dt"], order); o.step(1, w["dt"], order)
        pairs, ncand, labels = g.encounters()
        co, eo, lo = o.encounters()
        assert ncand == len(co) and np.array_equal(pairs, eo) and np.array_equal(labels, lo)
    compare(g, o, 3, kinds=[0])
    g.close()


def test_test_particle_hits_a_planet(G):
    """L336: the particle is reported and removed, the planet does not notice"""
    w = workloads.config2(n_massive=3, n_test=300)
    x, v = w["x"].copy(), w["v"].copy()
    for k in range(20):                                      # particles next to planet 1, on their way into it
        f = 2e-4 * (1 + 0.2 * k)
        x[:, 3 + k] = x[:, 1] * (1 + f); v[:, 3 + k] = v[:, 1] * (1 - 1.5 * f)
    R = np.full(303, 1e-5); R[1] = 3e-4
    w = dict(w, x=x, v=v, radius=R)
    g = G.from_workload(w); g.set_collisions(True)
    o = oracle.Sim(w); o.set_collisions(True)
    g.step(10, w["dt"], 2); o.step(10, w["dt"], 2)
    ev = compare(g, o, 3, kinds=[1])
    assert all(e[2] == 1 for e in ev)
    g.close()


def test_multi_system_collisions_ejections_and_stop(G):
    """mode 2: per-system collisions, Rcut / RcutSun, and the stop of a system that falls below Nmin (L378-384)"""
    w = workloads.config3(n_systems=24, n_per=12)
    w["m"] = w["m"] * 300
    w["radius"] = w["radius"] * 300
    g = G.from_workload(w); g.set_collisions(True, rcut=3.9, rcut_sun=0.52, n_min=11)
    o = oracle.Sim(w); o.set_collisions(True, rcut=3.9, rcut_sun=0.52, nmin=11)
    g.step(40, w["dt"], 2); o.step(40, w["dt"], 2)
    ev = compare(g, o, 5)
    assert {2, 4} <= set(ev[:, 1].astype(int))
    g.close()


def test_ejection_and_stop_single_system(G):
    w = workloads.config0(n=6)
    r = np.sort(np.linalg.norm(w["x"], axis=0))
    for nmin in (0, 6):
        g = G.from_workload(w); g.set_collisions(True, rcut=0.5 * (r[-1] + r[-2]), rcut_sun=0.5 * (r[0] + r[1]), n_min=nmin)
        o = oracle.Sim(w); o.set_collisions(True, rcut=0.5 * (r[-1] + r[-2]), rcut_sun=0.5 * (r[0] + r[1]), nmin=nmin)
        g.step(3, w["dt"], 2); o.step(3, w["dt"], 2)
        ev = compare(g, o, 2)
        assert (len(ev) == 6) if nmin else (2 <= len(ev) < 6)
        g.close()


def test_collisions_off_is_bitwise_the_point_mass_path(G):
    w = workloads.config4(n=300)
    a = G.from_workload(w)
    b = G.from_workload(w); b.set_collisions(False)
    c = G.from_workload(w); c.set_collisions(True)               # real radii: nothing collides in 5 steps
    for g in (a, b, c):
        g.step(5, w["dt"], 4)
    xa, va = a.get_state_host(); xb, vb = b.get_state_host(); xc, vc = c.get_state_host()
    assert np.array_equal(xa, xb) and np.array_equal(va, vb)
    assert np.array_equal(xa, xc) and np.array_equal(va, vc) and len(c.events()) == 0
    for g in (a, b, c):
        assert g.status() == 0
        g.close()
