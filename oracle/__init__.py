"""ctypes front end of the CPU oracle (oracle/genga_oracle.c).

TEST INFRASTRUCTURE, NOT THE PRODUCT: only tests/, __graft_entry__.smoke() and
bench.py's cpu_baseline / --impl reference legs may import this package.  It
shares nothing with paper_1404_2324_b200/ and never imports it.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "genga_oracle.c")
_LIB = os.path.join(_HERE, "libgenga_oracle.so")


def build(force: bool = False) -> str:
    """Compile the oracle with gcc (plain -O2, no fast-math, no FMA contraction)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        subprocess.check_call(["gcc", "-O2", "-std=c11", "-ffp-contract=off", "-fPIC", "-shared",
                               "-o", _LIB, _SRC, "-lm"])
    return _LIB


_lib = None
_dp = np.ctypeslib.ndpointer(dtype=np.float64, flags="C_CONTIGUOUS")
_ip = np.ctypeslib.ndpointer(dtype=np.int32, flags="C_CONTIGUOUS")
_lp = np.ctypeslib.ndpointer(dtype=np.int64, flags="C_CONTIGUOUS")


def lib():
    global _lib
    if _lib is not None:
        return _lib
    L = C.CDLL(build())
    d, i, l, vp = C.c_double, C.c_int, C.c_int64, C.c_void_p
    sig = {
        "ora_changeover": (None, [d, d, C.POINTER(d), C.POINTER(d)]),
        "ora_kick_weight": (d, [d, d]),
        "ora_rcrit": (None, [i, d, d, d, d, d, _dp, _dp, _dp, _dp]),
        "ora_accel": (i, [i, i, d, _dp, _dp, _dp, _dp, i, _ip, l, _lp]),
        "ora_sun_kick": (None, [i, i, d, _dp, _dp, _dp, d]),
        "ora_stumpff": (None, [d, _dp]),
        "ora_kepler_drift": (i, [d, d, _dp, _dp]),
        "ora_drift_all": (i, [i, d, d, _dp, _dp, vp]),
        "ora_hermite_min": (d, [d, d, d, d, d]),
        "ora_confirm": (i, [i, _dp, _dp, _dp, _dp, _dp, d, _ip, l, _ip, l, _lp]),
        "ora_group": (None, [i, _ip, l, _ip]),
        "ora_bs_group": (i, [i, d, d, _dp, _dp, _dp, _dp, d, d, vp]),
        "ora_energy": (None, [i, i, d, d, _dp, _dp, _dp, vp, _dp, _dp, vp]),
        "ora_helio_to_demo": (None, [i, i, d, _dp, _dp, _dp]),
        "ora_demo_to_helio": (None, [i, i, d, _dp, _dp, _dp]),
        "ora_create": (vp, [i, i, d, d, d, d, d, l]),
        "ora_destroy": (None, [vp]),
        "ora_set_cull": (None, [vp, i]),
        "ora_set_state": (None, [vp, _dp, _dp, _dp]),
        "ora_get_state": (None, [vp, _dp, _dp]),
        "ora_get_demo": (None, [vp, _dp, _dp, _dp]),
        "ora_set_demo": (None, [vp, _dp, _dp]),
        "ora_map_s2": (i, [vp, d]),
        "ora_step": (i, [vp, l, d, i]),
        "ora_yoshida": (i, [i, _dp]),
        "ora_get_encounters": (None, [vp, _ip, _lp, _ip, _lp, _ip]),
        "ora_get_stats": (None, [vp, _lp]),
        "ora_system_energy": (d, [vp, _dp]),
        "ora_accel_now": (i, [vp, d, _dp, _dp]),
        "ora_set_collisions": (None, [vp, vp, i, d, d, i]),
        "ora_get_events": (l, [vp, vp, l]),
        "ora_get_bodies": (None, [vp, vp, vp, vp, vp]),
        "ora_internal_energy": (d, [vp]),
        "ora_bs_group_collide": (i, [i, d, d, _dp, _dp, _dp, _ip, _dp, _dp, _dp, d, d, _dp, _dp, l, _lp]),
    }
    for name, (res, args) in sig.items():
        f = getattr(L, name)
        f.restype, f.argtypes = res, args
    _lib = L
    return L


ERR = {0: "ok", -1: "invalid argument", -2: "pair list capacity exceeded",
       -3: "Kepler solver did not converge", -4: "Bulirsch-Stoer step underflow"}


class OracleError(RuntimeError):
    pass


EV = 24          # doubles per event record: step, kind, i, j, m_i, m_j, R_i, R_j, q_i[3], V_i[3], q_j[3], V_j[3], U, spin[3]


def _chk(rc):
    if rc != 0:
        raise OracleError(ERR.get(rc, str(rc)))


# ---------------------------------------------------------------- thin per-function helpers
def changeover(r, rc):
    K, dK = C.c_double(), C.c_double()
    lib().ora_changeover(r, rc, C.byref(K), C.byref(dK))
    return K.value, dK.value


def kick_weight(r, rc):
    return lib().ora_kick_weight(r, rc)


def stumpff(x):
    c = np.zeros(4)
    lib().ora_stumpff(x, c)
    return c


def kepler_drift(mu, h, q, V):
    q = np.array(q, dtype=np.float64)
    V = np.array(V, dtype=np.float64)
    it = lib().ora_kepler_drift(mu, h, q, V)
    if it < 0:
        _chk(it)
    return q, V, it


def yoshida(order):
    w = np.zeros(7)
    return w[: lib().ora_yoshida(order, w)].copy()


def hermite_min(P0, P1, Pd0, Pd1, h):
    return lib().ora_hermite_min(P0, P1, Pd0, Pd1, h)


def rcrit(G, m0, n1, n2, tau, m, q, V):
    n = len(m)
    rc = np.zeros(n)
    lib().ora_rcrit(n, G, m0, n1, n2, tau, np.ascontiguousarray(m), np.ascontiguousarray(q),
                    np.ascontiguousarray(V), rc)
    return rc


def accel(G, m, q, rc, n_massive=None, record=True, cap=None):
    n = len(m)
    nm = n if n_massive is None else n_massive
    cap = cap or max(16, n * 64)
    a = np.zeros((3, n))
    cand = np.zeros((cap, 2), dtype=np.int32)
    nc = np.zeros(1, dtype=np.int64)
    _chk(lib().ora_accel(n, nm, G, np.ascontiguousarray(m), np.ascontiguousarray(q),
                         np.ascontiguousarray(rc), a, int(record), cand, cap, nc))
    return a, cand[: nc[0]].copy()


def group(n, pairs):
    pairs = np.ascontiguousarray(pairs, dtype=np.int32).reshape(-1, 2)
    link = np.zeros(n, dtype=np.int32)
    lib().ora_group(n, pairs, len(pairs), link)
    return link


def bs_group(G, m0, m, rc, q, V, h, eps=1e-12):
    q = np.array(q, dtype=np.float64, order="C")
    V = np.array(V, dtype=np.float64, order="C")
    stats = np.zeros(2, dtype=np.int64)
    _chk(lib().ora_bs_group(len(m), G, m0, np.ascontiguousarray(m, dtype=np.float64),
                            np.ascontiguousarray(rc, dtype=np.float64), q, V, h, eps,
                            stats.ctypes.data))
    return q, V, stats


def bs_group_collide(G, m0, m, rc, R, q, V, h, kind=None, eps=1e-12):
    """one group integrated over h with collisions; returns q, V, m, R, kind, spin, U, events"""
    ng = len(m)
    m = np.array(m, dtype=np.float64); R = np.array(R, dtype=np.float64)
    q = np.array(q, dtype=np.float64, order="C"); V = np.array(V, dtype=np.float64, order="C")
    kind = np.zeros(ng, dtype=np.int32) if kind is None else np.array(kind, dtype=np.int32)
    spin = np.zeros((3, ng)); U = np.zeros(1); ev = np.zeros((64, EV)); nev = np.zeros(1, dtype=np.int64)
    _chk(lib().ora_bs_group_collide(ng, G, m0, m, np.ascontiguousarray(rc, dtype=np.float64), R, kind, spin, q, V, h, eps,
                                    U, ev, 64, nev))
    return q, V, m, R, kind, spin, U[0], ev[: nev[0]]


def energy(G, m0, m, q, V, rc=None, n_massive=None):
    n = len(m)
    nm = n if n_massive is None else n_massive
    E, L, parts = np.zeros(1), np.zeros(3), np.zeros(3)
    rcp = None if rc is None else np.ascontiguousarray(rc).ctypes.data
    rc_keep = None if rc is None else np.ascontiguousarray(rc)
    rcp = None if rc_keep is None else rc_keep.ctypes.data
    lib().ora_energy(nm, n, G, m0, np.ascontiguousarray(m), np.ascontiguousarray(q),
                     np.ascontiguousarray(V), rcp, E, L, parts.ctypes.data)
    return E[0], L, parts


def helio_to_demo(m0, m, v, n_massive=None):
    n = len(m)
    V = np.zeros((3, n))
    lib().ora_helio_to_demo(n, n if n_massive is None else n_massive, m0, np.ascontiguousarray(m),
                            np.ascontiguousarray(v), V)
    return V


def demo_to_helio(m0, m, V, n_massive=None):
    n = len(m)
    v = np.zeros((3, n))
    lib().ora_demo_to_helio(n, n if n_massive is None else n_massive, m0, np.ascontiguousarray(m),
                            np.ascontiguousarray(V), v)
    return v


# ---------------------------------------------------------------- one system
class System:
    """One star + n bodies (first n_massive massive, the rest test particles)."""

    def __init__(self, m0, m, x, v, n_massive=None, G=1.0, n1=3.0, n2=0.4, bs_eps=1e-12, cap=None):
        self.n = len(m)
        self.nm = self.n if n_massive is None else n_massive
        self.cap = int(cap or max(64, 32 * self.n))
        self.h = lib().ora_create(self.n, self.nm, G, float(m0), n1, n2, bs_eps, self.cap)
        if not self.h:
            raise OracleError("ora_create failed")
        self.m0, self.G = float(m0), G
        self.m = np.ascontiguousarray(m, dtype=np.float64)
        lib().ora_set_state(self.h, self.m, np.ascontiguousarray(x, dtype=np.float64),
                            np.ascontiguousarray(v, dtype=np.float64))

    def __del__(self):
        if getattr(self, "h", None):
            lib().ora_destroy(self.h)
            self.h = None

    def set_cull(self, cull):
        lib().ora_set_cull(self.h, int(cull))

    def step(self, n_steps, dt, order=2):
        _chk(lib().ora_step(self.h, int(n_steps), float(dt), int(order)))

    def map_s2(self, h):
        _chk(lib().ora_map_s2(self.h, float(h)))

    def state(self):
        x, v = np.zeros((3, self.n)), np.zeros((3, self.n))
        lib().ora_get_state(self.h, x, v)
        return x, v

    def demo(self):
        q, V, rc = np.zeros((3, self.n)), np.zeros((3, self.n)), np.zeros(self.n)
        lib().ora_get_demo(self.h, q, V, rc)
        return q, V, rc

    def set_demo(self, q, V):
        lib().ora_set_demo(self.h, np.ascontiguousarray(q), np.ascontiguousarray(V))

    def energy(self):
        L = np.zeros(3)
        E = lib().ora_system_energy(self.h, L)
        return E, L

    def accel_now(self, dt):
        a, rc = np.zeros((3, self.n)), np.zeros(self.n)
        _chk(lib().ora_accel_now(self.h, float(dt), a, rc))
        return a, rc

    def encounters(self):
        """(candidates, confirmed pairs, labels) of the last drift substep, pairs sorted."""
        cand = np.zeros((self.cap, 2), dtype=np.int32)
        enc = np.zeros((self.cap, 2), dtype=np.int32)
        nc, ne = np.zeros(1, dtype=np.int64), np.zeros(1, dtype=np.int64)
        label = np.zeros(self.n, dtype=np.int32)
        lib().ora_get_encounters(self.h, cand, nc, enc, ne, label)
        cand, enc = cand[: nc[0]], enc[: ne[0]]
        cand = cand[np.lexsort((cand[:, 1], cand[:, 0]))] if len(cand) else cand
        enc = enc[np.lexsort((enc[:, 1], enc[:, 0]))] if len(enc) else enc
        return cand.copy(), enc.copy(), label

    # ---- collisions, ejections, removal
    def set_collisions(self, radius, collisions=True, rcut=0.0, rcut_sun=0.0, nmin=0):
        R = np.ascontiguousarray(radius, dtype=np.float64)
        lib().ora_set_collisions(self.h, R.ctypes.data, int(collisions), float(rcut), float(rcut_sun), int(nmin))

    def events(self):
        """event records (EV doubles each, see genga_oracle.c): all events since creation"""
        n = lib().ora_get_events(self.h, None, 0)
        buf = np.zeros((max(n, 1), EV))
        lib().ora_get_events(self.h, buf.ctypes.data, n)
        return buf[:n]

    def bodies(self):
        m, R, kind, spin = np.zeros(self.n), np.zeros(self.n), np.zeros(self.n, dtype=np.int32), np.zeros((3, self.n))
        lib().ora_get_bodies(self.h, m.ctypes.data, R.ctypes.data, kind.ctypes.data, spin.ctypes.data)
        return m, R, kind, spin

    def internal_energy(self):
        return lib().ora_internal_energy(self.h)

    def stats(self):
        out = np.zeros(6, dtype=np.int64)
        lib().ora_get_stats(self.h, out)
        return dict(kepler_iters=int(out[0]), bs_steps=int(out[1]), bs_rhs=int(out[2]),
                    force_evals=int(out[3]), groups=int(out[4]), max_group=int(out[5]))


class Sim:
    """A workload dict from `workloads` run by the oracle in any of the three modes.
    Multi-simulation mode is a loop over independent systems."""

    def __init__(self, w, cap=None):
        self.w = w
        self.ns = int(w.get("n_systems", 1))
        n = w["x"].shape[1]
        self.per = n // self.ns
        kw = dict(G=w["G"], n1=w["n1"], n2=w["n2"], bs_eps=w["bs_eps"], cap=cap)
        self.sys = []
        for s in range(self.ns):
            sl = slice(s * self.per, (s + 1) * self.per)
            nm = w["n_massive"] if w["mode"] != 2 else self.per
            self.sys.append(System(w["m0"][s], w["m"][sl], w["x"][:, sl], w["v"][:, sl],
                                   n_massive=nm, **kw))

    def set_collisions(self, collisions=True, rcut=0.0, rcut_sun=0.0, nmin=0):
        for k, s in enumerate(self.sys):
            sl = slice(k * self.per, (k + 1) * self.per)
            s.set_collisions(self.w["radius"][sl], collisions, rcut, rcut_sun, nmin)

    def events(self):
        """all events, body indices global, in the order (system, occurrence)"""
        out = []
        for k, s in enumerate(self.sys):
            e = s.events().copy()
            if len(e):
                e[:, 2] += k * self.per
                e[:, 3] = np.where(e[:, 3] >= 0, e[:, 3] + k * self.per, e[:, 3])
                out.append(e)
        return np.concatenate(out) if out else np.zeros((0, EV))

    def bodies(self):
        m, R, kind, spin = zip(*[s.bodies() for s in self.sys])
        return np.concatenate(m), np.concatenate(R), np.concatenate(kind), np.concatenate(spin, axis=1)

    def internal_energy(self):
        return np.array([s.internal_energy() for s in self.sys])

    def step(self, n_steps, dt=None, order=None):
        dt = self.w["dt"] if dt is None else dt
        order = self.w["order"] if order is None else order
        for s in self.sys:
            s.step(n_steps, dt, order)

    def state(self):
        xs, vs = zip(*[s.state() for s in self.sys])
        return np.concatenate(xs, axis=1), np.concatenate(vs, axis=1)

    def energy(self):
        E, L = zip(*[s.energy() for s in self.sys])
        return np.array(E), np.array(L)

    def encounters(self):
        """Pairs in global body indices, sorted; labels global."""
        cands, encs, labels = [], [], []
        for k, s in enumerate(self.sys):
            c, e, l = s.encounters()
            cands.append(c + k * self.per); encs.append(e + k * self.per); labels.append(l + k * self.per)
        return np.concatenate(cands), np.concatenate(encs), np.concatenate(labels)
