"""Pins for the encounter search (Eq. 10-12), grouping (Appendix,
L537-551) and the Bulirsch-Stoer integration of groups (L116, L314, L505)."""
import mpmath as mp
import numpy as np
import pytest
from scipy.sparse import coo_matrix
from scipy.sparse.csgraph import connected_components

import oracle
import workloads


def eq10(t, P0, P1, Pd0, Pd1, h):
    """Eq. 10 (L120) typed from the paper, independent of the oracle's Eq. 12 code."""
    return (P0 * (1 + 2 * t) * (1 - t) ** 2 + P1 * t**2 * (3 - 2 * t)
            + Pd0 * t * (1 - t) ** 2 * h + Pd1 * t**2 * (t - 1) * h)


@pytest.mark.parametrize("seed", range(12))
def test_hermite_min_equals_dense_minimum_of_eq10(seed):
    """[R-2] with the printed sign of `a` the critical points are wrong and this fails."""
    rng = np.random.default_rng(seed)
    P0, P1 = rng.uniform(0.1, 2.0, 2)
    Pd0, Pd1 = rng.uniform(-8, 8, 2)
    h = rng.choice([-1, 1]) * rng.uniform(0.05, 0.5)
    t = np.linspace(0, 1, 200001)
    dense = eq10(t, P0, P1, Pd0, Pd1, h).min()
    got = oracle.hermite_min(P0, P1, Pd0, Pd1, h)
    assert got <= dense + 1e-15
    assert abs(got - dense) <= 1e-9 * max(1.0, abs(dense))


def test_hermite_exact_for_uniform_relative_motion():
    """Straight-line relative motion: P(t) is a quadratic, the cubic Hermite fit is exact and
    Delta is the analytic closest approach |d0 x dv|^2/|dv|^2."""
    d0 = np.array([0.3, -0.2, 0.1]); dv = np.array([-1.0, 0.9, 0.05]); h = 0.5
    d1 = d0 + h * dv
    D = oracle.hermite_min(d0 @ d0, d1 @ d1, 2 * d0 @ dv, 2 * d1 @ dv, h)
    assert abs(D - np.linalg.norm(np.cross(d0, dv)) ** 2 / (dv @ dv)) < 1e-15
    # receding pair: minimum at the start; backwards in time the same pair approaches
    d0 = np.array([0.3, 0.0, 0.0]); dv = np.array([1.0, 0.0, 0.0])
    d1 = d0 + h * dv
    assert oracle.hermite_min(d0 @ d0, d1 @ d1, 2 * d0 @ dv, 2 * d1 @ dv, h) == d0 @ d0
    d1 = d0 - 0.2 * dv
    assert abs(oracle.hermite_min(d0 @ d0, d1 @ d1, 2 * d0 @ dv, 2 * d1 @ dv, -0.2) - d1 @ d1) < 1e-16


@pytest.mark.parametrize("seed", range(6))
def test_group_labels_are_min_index_of_connected_component(seed):
    rng = np.random.default_rng(seed)
    n = 300
    pairs = rng.integers(0, n, size=(rng.integers(1, 260), 2)).astype(np.int32)
    pairs = pairs[pairs[:, 0] != pairs[:, 1]]
    link = oracle.group(n, pairs)
    g = coo_matrix((np.ones(len(pairs)), (pairs[:, 0], pairs[:, 1])), shape=(n, n))
    _, comp = connected_components(g, directed=False)
    want = np.array([np.flatnonzero(comp == comp[i]).min() for i in range(n)])
    assert np.array_equal(link, want)
    # a long chain given in the worst order
    chain = np.array([[i, i + 1] for i in range(n - 1)][::-1], dtype=np.int32)
    assert np.all(oracle.group(n, chain) == 0)


# ---------------------------------------------------------------- Bulirsch-Stoer
mp.mp.dps = 40


def test_bs_single_body_group_is_the_kepler_flow():
    """A group of one body feels only the fixed star (L314): BS must equal the analytic orbit
    (here through the separately pinned Kepler drift) to ~eps."""
    mu = 1.0
    q0 = np.array([[1.0], [0.1], [-0.02]]); V0 = np.array([[-0.05], [0.93], [0.03]])
    for h in (0.1032, -0.1032, 0.9):
        q, V, st = oracle.bs_group(1.0, mu, [1e-6], [0.05], q0, V0, h)
        qk, Vk, _ = oracle.kepler_drift(mu, h, q0[:, 0], V0[:, 0])
        assert np.linalg.norm(q[:, 0] - qk) <= 3e-12 * np.linalg.norm(qk)
        assert np.linalg.norm(V[:, 0] - Vk) <= 3e-12 * np.linalg.norm(Vk)
        assert st[0] >= 1


def test_bs_circular_binary_closed_form():
    """m0 = 0 and separation below 0.1 rc (K = 0, the whole pair force is in H_A, Eq. 1):
    two equal masses on a circular orbit rotate rigidly by omega h, omega^2 = G(2m)/d^3."""
    G, m, d = 1.0, 2e-3, 0.01
    om = np.sqrt(G * 2 * m / d**3)
    q0 = np.array([[d / 2, -d / 2], [0, 0], [0, 0.0]])
    V0 = np.array([[0, 0], [om * d / 2, -om * d / 2], [0, 0.0]])
    h = 0.37
    q, V, st = oracle.bs_group(G, 0.0, [m, m], [1.0, 1.0], q0, V0, h)
    c, s = np.cos(om * h), np.sin(om * h)
    # 3.7 revolutions in st[0] accepted BS steps, each good to eps = 1e-12 relative
    tol = 1e-12 * st[0]
    assert np.allclose(q[:, 0], [d / 2 * c, d / 2 * s, 0], rtol=0, atol=tol * d)
    assert np.allclose(V[:, 1], [om * d / 2 * s, -om * d / 2 * c, 0], rtol=0, atol=tol * om * d)
    assert 1 <= st[0] < 200


def _HA(G, m0, m, rc, q, V):
    return oracle.energy(G, m0, m, q, V, rc)[2][0]


def test_bs_conserves_HA_and_reverses():
    """Three bodies inside each other's changeover zone: H_A of Eq. 1 (with 1-K) is the
    conserved quantity of the BS flow, only with the weight 1-(K - r K') [R-1]."""
    G, m0 = 1.0, 1.0
    m = np.array([3e-5, 1e-5, 2e-5]); rc = np.array([0.03, 0.02, 0.025])
    q0 = np.array([[1.0, 1.012, 0.995], [0.0, 0.008, -0.01], [0.0, 0.001, 0.002]])
    V0 = np.array([[0.0, -0.02, 0.03], [1.0, 0.99, 1.01], [0.0, 0.005, -0.004]])
    h = 0.1032
    q, V, _ = oracle.bs_group(G, m0, m, rc, q0, V0, h)
    H0, H1 = _HA(G, m0, m, rc, q0, V0), _HA(G, m0, m, rc, q, V)
    assert abs(H1 - H0) <= 1e-11 * abs(H0)
    qb, Vb, _ = oracle.bs_group(G, m0, m, rc, q, V, -h)
    assert np.allclose(qb, q0, rtol=0, atol=1e-11) and np.allclose(Vb, V0, rtol=0, atol=1e-11)
    # the interaction matters at this level (else the test proves nothing)
    qk = np.array([oracle.kepler_drift(1.0, h, q0[:, i], V0[:, i])[0] for i in range(3)]).T
    assert np.abs(qk - q).max() > 1e-8
    # angular momentum of the group about the fixed star
    L0 = (m * np.cross(q0.T, V0.T).T).sum(1); L1 = (m * np.cross(q.T, V.T).T).sum(1)
    assert np.linalg.norm(L1 - L0) <= 1e-11 * np.linalg.norm(L0)


def test_bs_tolerance_is_honoured_against_tight_run():
    G, m0 = 1.0, 1.0
    m = np.array([3e-5, 1e-5]); rc = np.array([0.03, 0.02])
    q0 = np.array([[1.0, 1.012], [0.0, 0.008], [0.0, 0.001]])      # a fly-by through the zone
    V0 = np.array([[0.0, -0.02], [1.0, 0.99], [0.0, 0.005]])
    qa, Va, sa = oracle.bs_group(G, m0, m, rc, q0, V0, 0.1032, 1e-12)
    qb, Vb, sb = oracle.bs_group(G, m0, m, rc, q0, V0, 0.1032, 1e-15)
    assert np.abs(qa - qb).max() <= 1e-12 and np.abs(Va - Vb).max() <= 1e-12
    assert sb[1] >= sa[1]
