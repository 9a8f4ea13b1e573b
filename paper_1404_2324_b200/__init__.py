"""Python binding of libgenga_b200.so (the C-ABI of include/genga.h).

Argument marshalling only: every step of the method runs in the library's CUDA kernels.
PyTorch supplies device memory (the workspace and state tensors) and the stream.  There is
no CPU fallback: importing works without a GPU (so the symbols can be inspected), but
creating a context without the library or without a CUDA device raises.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libgenga_b200.so")

MODE_MASSIVE, MODE_TEST_PARTICLE, MODE_MULTI_SYSTEM = 0, 1, 2
OK, EINVAL, ECAPACITY, EKEPLER, EBS, ECUDA = 0, -1, -2, -3, -4, -5

# every symbol include/genga.h declares
SYMBOLS = [
    "genga_workspace_bytes", "genga_create", "genga_destroy", "genga_set_state", "genga_set_state_host",
    "genga_step", "genga_get_state", "genga_get_state_host", "genga_set_state_ragged_host", "genga_get_state_ragged_host", "genga_set_system_params_host",
    "genga_energy", "genga_encounters", "genga_bs_trace", "genga_set_collisions", "genga_events", "genga_bodies",
    "genga_status", "genga_accelerations", "genga_kepler_drift", "genga_counters", "genga_time_kernel", "genga_profile_step",
    "genga_eval_fast", "genga_fp64_probe", "genga_strerror",
    "genga_last_cuda_error", "genga_kick_accel_noalloc", "genga_noalloc_last_error",
]

NOALLOC_MAX_BODIES = 2048           # GENGA_NOALLOC_MAX_BODIES of include/genga.h


class genga_config(C.Structure):
    _fields_ = [("mode", C.c_int32), ("n_massive", C.c_int32), ("n_test", C.c_int64),
                ("n_systems", C.c_int32), ("flags", C.c_int32),
                ("G", C.c_double), ("n1", C.c_double), ("n2", C.c_double), ("bs_eps", C.c_double),
                ("max_pairs", C.c_int64), ("workspace", C.c_void_p), ("workspace_bytes", C.c_size_t),
                ("stream", C.c_void_p)]


class GengaError(RuntimeError):
    def __init__(self, code, where=""):
        self.code = code
        msg = load().genga_strerror(code).decode()
        if code == ECUDA:
            msg += ": " + load().genga_last_cuda_error().decode()
        super().__init__("%s: %s (%d)" % (where, msg, code))


_lib = None


def load():
    """dlopen the library (built by `python -m paper_1404_2324_b200.build`) and type its entry points."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise RuntimeError("CUDA library %s is missing: run `python -m paper_1404_2324_b200.build` "
                           "(there is no CPU fallback)" % LIB_PATH)
    L = C.CDLL(LIB_PATH)
    vp, d, i, l, dp = C.c_void_p, C.c_double, C.c_int, C.c_int64, C.c_void_p
    cfgp = C.POINTER(genga_config)
    sig = {
        "genga_workspace_bytes": (C.c_size_t, [cfgp]),
        "genga_create": (i, [cfgp, C.POINTER(vp)]),
        "genga_destroy": (i, [vp]),
        "genga_set_state": (i, [vp, dp, dp, dp, dp, dp]),
        "genga_set_state_host": (i, [vp, dp, dp, dp, dp, dp]),
        "genga_step": (i, [vp, l, d, i]),
        "genga_get_state": (i, [vp, dp, dp]),
        "genga_get_state_host": (i, [vp, dp, dp]),
        "genga_set_state_ragged_host": (i, [vp, vp, dp, dp, dp, dp, dp]),
        "genga_get_state_ragged_host": (i, [vp, dp, dp]),
        "genga_set_system_params_host": (i, [vp, dp, dp]),
        "genga_energy": (i, [vp, dp, dp]),
        "genga_encounters": (i, [vp, vp, l, C.POINTER(l), C.POINTER(l), vp]),
        "genga_bs_trace": (i, [vp, vp, l, C.POINTER(l)]),
        "genga_set_collisions": (i, [vp, i, d, d, i]),
        "genga_events": (i, [vp, vp, l, C.POINTER(l)]),
        "genga_bodies": (i, [vp, vp, vp, vp, vp, vp]),
        "genga_status": (i, [vp]),
        "genga_accelerations": (i, [vp, d, dp, dp]),
        "genga_kepler_drift": (i, [vp, l, d, d, dp, dp]),
        "genga_counters": (i, [vp, vp]),
        "genga_time_kernel": (i, [vp, i, i, d, C.POINTER(d)]),
        "genga_profile_step": (i, [vp, l, d, i, vp]),
        "genga_eval_fast": (i, [vp, i, l, dp, dp]),
        "genga_fp64_probe": (i, [vp, C.POINTER(d)]),
        "genga_strerror": (C.c_char_p, [i]),
        "genga_last_cuda_error": (C.c_char_p, []),
        "genga_kick_accel_noalloc": (i, [vp, l, d, dp, dp, dp, dp]),
        "genga_noalloc_last_error": (C.c_char_p, []),
    }
    for name, (res, args) in sig.items():
        f = getattr(L, name)
        f.restype, f.argtypes = res, args
    _lib = L
    return L


def _chk(code, where):
    if code != 0:
        raise GengaError(code, where)


def _hp(a):
    return a.ctypes.data          # the address as an int: the argtypes make it a void*; the caller keeps `a` alive


class Genga:
    """One simulation context.  State arrays are (3, Ntot) float64, heliocentric."""

    def __init__(self, mode, n_massive, n_test=0, n_systems=1, G=1.0, n1=3.0, n2=0.4, bs_eps=1e-12,
                 max_pairs=None, device="cuda:0", stream=None, flags=0):
        import torch
        if not torch.cuda.is_available():
            raise RuntimeError("paper_1404_2324_b200 needs a CUDA device (sm_100a); there is no CPU fallback")
        self.torch = torch
        self.lib = load()
        self.device = torch.device(device)
        self.mode, self.nm, self.nt, self.ns = int(mode), int(n_massive), int(n_test), int(n_systems)
        self.ntot = self.ns * self.nm if mode == MODE_MULTI_SYSTEM else self.nm + self.nt
        if max_pairs is None:
            max_pairs = max(4096, 64 * self.nm * (self.ns if mode == MODE_MULTI_SYSTEM else 1), 2 * self.nt)
        self.max_pairs = int(max_pairs)
        with torch.cuda.device(self.device):
            self.stream = stream if stream is not None else torch.cuda.Stream(device=self.device)
            cfg = genga_config(mode, n_massive, n_test, n_systems, int(flags), G, n1, n2, bs_eps, self.max_pairs, None, 0,
                               self.stream.cuda_stream)
            nbytes = self.lib.genga_workspace_bytes(C.byref(cfg))
            if nbytes == 0:
                raise GengaError(EINVAL, "genga_workspace_bytes")
            self.workspace = torch.empty(nbytes + 256, dtype=torch.uint8, device=self.device)
            base = (self.workspace.data_ptr() + 255) // 256 * 256
            cfg.workspace, cfg.workspace_bytes = base, nbytes
            self.cfg = cfg
            h = C.c_void_p()
            _chk(self.lib.genga_create(C.byref(cfg), C.byref(h)), "genga_create")
            self.h = h

    def close(self):
        if getattr(self, "h", None):
            self.stream.synchronize()
            self.lib.genga_destroy(self.h)
            self.h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    # ---- state ------------------------------------------------------------------------
    def _dev(self, a):
        t = self.torch
        if isinstance(a, t.Tensor):
            a = a.to(device=self.device, dtype=t.float64).contiguous()
        else:
            a = t.as_tensor(np.ascontiguousarray(a, dtype=np.float64), device=self.device)
        return a

    def _order_before(self):
        """the context's stream waits for the work the caller queued on torch's current stream (the tensors passed in)"""
        self.stream.wait_stream(self.torch.cuda.current_stream(self.device))

    def _order_after(self):
        """torch's current stream waits for the work this call queued on the context's stream"""
        self.torch.cuda.current_stream(self.device).wait_stream(self.stream)

    def set_state(self, m0, m, radius, x, v):
        """Device path: arguments are moved to the device first (if they are not there),
        then handed to genga_set_state as device pointers."""
        args = [self._dev(np.atleast_1d(m0) if not hasattr(m0, "shape") else m0), self._dev(m),
                self._dev(radius), self._dev(x), self._dev(v)]
        self.torch.cuda.current_stream(self.device).synchronize()
        with self.torch.cuda.stream(self.stream):
            _chk(self.lib.genga_set_state(self.h, *[a.data_ptr() for a in args]), "genga_set_state")
        self.stream.synchronize()

    def set_state_host(self, m0, m, radius, x, v):
        """Host path: numpy (or pinned torch CPU) arrays go through genga_set_state_host."""
        arrs = [np.ascontiguousarray(a, dtype=np.float64) for a in (np.atleast_1d(m0), m, radius, x, v)]
        _chk(self.lib.genga_set_state_host(self.h, *[_hp(a) for a in arrs]), "genga_set_state_host")

    def step(self, n_steps, dt, order=2):
        _chk(self.lib.genga_step(self.h, int(n_steps), float(dt), int(order)), "genga_step")

    def get_state(self):
        """Device tensors (x, v), each (3, Ntot)."""
        t = self.torch
        x = t.empty((3, self.ntot), dtype=t.float64, device=self.device)
        v = t.empty((3, self.ntot), dtype=t.float64, device=self.device)
        self._order_before()
        _chk(self.lib.genga_get_state(self.h, x.data_ptr(), v.data_ptr()), "genga_get_state")
        self.stream.synchronize()
        return x, v

    def get_state_host(self, x=None, v=None):
        x = np.empty((3, self.ntot)) if x is None else x
        v = np.empty((3, self.ntot)) if v is None else v
        _chk(self.lib.genga_get_state_host(self.h, _hp(x), _hp(v)), "genga_get_state_host")
        return x, v

    def set_state_ragged_host(self, n_bodies, m0, m, radius, x, v):
        """Multi-system mode, variable bodies per system: packed arrays, see include/genga.h."""
        nb = np.ascontiguousarray(n_bodies, dtype=np.int32)
        if nb.shape != (self.ns,):
            raise ValueError("n_bodies must have one entry per system")
        self._nreal = int(nb.sum())
        arrs = [np.ascontiguousarray(a, dtype=np.float64) for a in (np.atleast_1d(m0), m, radius, x, v)]
        if arrs[1].size != self._nreal or arrs[2].size != self._nreal or arrs[3].size != 3 * self._nreal or arrs[4].size != 3 * self._nreal:
            raise ValueError("packed arrays do not match sum(n_bodies)")
        _chk(self.lib.genga_set_state_ragged_host(self.h, _hp(nb), *[_hp(a) for a in arrs]), "genga_set_state_ragged_host")

    def set_system_params_host(self, n1, n2):
        """Multi-system mode: n1, n2 of Eq. 6 per system."""
        a, b = (np.ascontiguousarray(np.broadcast_to(np.asarray(q, dtype=np.float64), (self.ns,))) for q in (n1, n2))
        _chk(self.lib.genga_set_system_params_host(self.h, _hp(a), _hp(b)), "genga_set_system_params_host")

    def get_state_ragged_host(self):
        x, v = np.empty((3, self._nreal)), np.empty((3, self._nreal))
        _chk(self.lib.genga_get_state_ragged_host(self.h, _hp(x), _hp(v)), "genga_get_state_ragged_host")
        return x, v

    def energy(self):
        E, L = np.zeros(self.ns if self.mode == MODE_MULTI_SYSTEM else 1), np.zeros((self.ns if self.mode == MODE_MULTI_SYSTEM else 1, 3))
        _chk(self.lib.genga_energy(self.h, _hp(E), _hp(L)), "genga_energy")
        return E, L

    def encounters(self, with_labels=True):
        pairs = np.zeros((self.max_pairs, 2), dtype=np.int32)
        npairs, ncand = C.c_int64(), C.c_int64()
        labels = np.zeros(self.ntot, dtype=np.int32) if with_labels else None
        _chk(self.lib.genga_encounters(self.h, _hp(pairs), self.max_pairs, C.byref(npairs), C.byref(ncand),
                                       _hp(labels) if with_labels else None), "genga_encounters")
        return pairs[: npairs.value].copy(), int(ncand.value), labels

    def set_collisions(self, collisions=True, rcut=0.0, rcut_sun=0.0, n_min=0):
        _chk(self.lib.genga_set_collisions(self.h, int(collisions), float(rcut), float(rcut_sun), int(n_min)), "genga_set_collisions")

    def events(self):
        """event records (n, 24), see include/genga.h"""
        buf = np.zeros((4096, 24))
        n = C.c_int64()
        _chk(self.lib.genga_events(self.h, _hp(buf), 4096, C.byref(n)), "genga_events")
        return buf[: min(n.value, 4096)].copy()

    def bodies(self):
        """(m, radius, kind, spin, U) as they are now"""
        ns = self.ns if self.mode == MODE_MULTI_SYSTEM else 1
        m, R, kind = np.zeros(self.ntot), np.zeros(self.ntot), np.zeros(self.ntot, dtype=np.int32)
        spin, U = np.zeros((3, self.ntot)), np.zeros(ns)
        _chk(self.lib.genga_bodies(self.h, _hp(m), _hp(R), _hp(kind), _hp(spin), _hp(U)), "genga_bodies")
        return m, R, kind, spin, U

    def bs_trace(self):
        """records (n, layout, accepted, rejected, cycles, member) of the groups integrated in the last substep"""
        out = np.zeros((4096, 4), dtype=np.int32)
        n = C.c_int64()
        _chk(self.lib.genga_bs_trace(self.h, _hp(out), 4096, C.byref(n)), "genga_bs_trace")
        r = out[: min(n.value, 4096)]
        return np.stack([r[:, 0] & 0xffff, r[:, 0] >> 16, r[:, 1] & 0xffff, r[:, 1] >> 16, r[:, 2], r[:, 3]], axis=1)

    def status(self):
        return self.lib.genga_status(self.h)

    def accelerations(self, dt):
        t = self.torch
        a = t.empty((3, self.ntot), dtype=t.float64, device=self.device)
        rc = t.empty(self.ntot, dtype=t.float64, device=self.device)
        self._order_before()
        _chk(self.lib.genga_accelerations(self.h, float(dt), a.data_ptr(), rc.data_ptr()), "genga_accelerations")
        self.stream.synchronize()
        return a, rc

    def kepler_drift(self, mu, h, x, v):
        """In-place drift of device tensors x, v of shape (3, n)."""
        n = x.shape[1]
        self._order_before()
        _chk(self.lib.genga_kepler_drift(self.h, n, float(mu), float(h), x.data_ptr(), v.data_ptr()), "genga_kepler_drift")
        self._order_after()

    def counters(self):
        out = np.zeros(16, dtype=np.int64)
        _chk(self.lib.genga_counters(self.h, _hp(out)), "genga_counters")
        keys = ["steps", "force_evals", "interactions", "launches", "groups", "max_group", "bs_steps", "candidates", "bs_rejects"]
        return dict(zip(keys, map(int, out)))

    PHASES = ["rcrit", "kick", "front", "confirm", "group", "bs", "back", "total"]

    def profile_step(self, n_steps, dt, order=2):
        """ms per step of each phase (genga_profile_step)."""
        ms = np.zeros(8)
        _chk(self.lib.genga_profile_step(self.h, int(n_steps), float(dt), int(order), _hp(ms)), "genga_profile_step")
        return dict(zip(self.PHASES, map(float, ms)))

    def eval_fast(self, which, x):
        """x: device float64 tensor; returns f(x) for f = x^-1/2, x^-3/2, 1/x (which = 0, 1, 2)."""
        out = self.torch.empty_like(x)
        self._order_before()
        _chk(self.lib.genga_eval_fast(self.h, int(which), x.numel(), x.data_ptr(), out.data_ptr()), "genga_eval_fast")
        self.stream.synchronize()
        return out

    def time_kernel(self, which, reps, dt):
        ms = C.c_double()
        _chk(self.lib.genga_time_kernel(self.h, int(which), int(reps), float(dt), C.byref(ms)), "genga_time_kernel")
        return ms.value

    def fp64_probe(self):
        tf = C.c_double()
        _chk(self.lib.genga_fp64_probe(self.h, C.byref(tf)), "genga_fp64_probe")
        return tf.value

    def synchronize(self):
        self.stream.synchronize()


def from_workload(w, **kw):
    """Context for a dict produced by the `workloads` module, state loaded (device path)."""
    g = Genga(w["mode"], w["n_massive"], w.get("n_test", 0), w.get("n_systems", 1), G=w["G"], n1=w["n1"],
              n2=w["n2"], bs_eps=w["bs_eps"], **kw)
    g.set_state(w["m0"], w["m"], w["radius"], w["x"], w["v"])
    return g


def kick_accel_noalloc(G, m, x, rcrit, a, stream=None):
    """genga_kick_accel_noalloc (include/genga.h): kick accelerations of one system of n <= NOALLOC_MAX_BODIES massive
    bodies into `a`, no context, no workspace, no allocation (the scratch is a static device array of the library; calls
    that overlap on the GPU race on it).  m, rcrit: device float64 tensors of n; x, a: device float64 (3, n), contiguous.
    Enqueues on `stream` (a torch stream; default: the current one) and does not synchronise."""
    import torch
    n = int(m.numel())
    for t, size in ((m, n), (rcrit, n), (x, 3 * n), (a, 3 * n)):
        if t.dtype != torch.float64 or not t.is_cuda or not t.is_contiguous() or t.numel() != size:
            raise ValueError("kick_accel_noalloc wants contiguous float64 CUDA tensors of n, n, 3 n and 3 n elements")
    st = (stream or torch.cuda.current_stream(m.device)).cuda_stream
    L = load()
    with torch.cuda.device(m.device):
        code = L.genga_kick_accel_noalloc(st, n, float(G), m.data_ptr(), x.data_ptr(), rcrit.data_ptr(), a.data_ptr())
    if code != 0:
        raise GengaError(code, "genga_kick_accel_noalloc: " + L.genga_noalloc_last_error().decode())
    return a
