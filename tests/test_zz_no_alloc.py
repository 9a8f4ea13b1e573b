"""genga_kick_accel_noalloc (include/genga.h, csrc/noalloc.cu): the entry point that allocates nothing -- its scratch
memory is a static device array of the library -- against the existing path (genga_accelerations, which works in the
caller's workspace), on the same positions, masses and critical radii.  Tolerance: the 1e-12 relative per body that
tests/test_gpu_parity.py uses for accelerations (the two paths add the pairs up in different orders).

Collected last on purpose (pytest -x: a failure here hides nothing behind it).  Passes alone in a fresh
process and after the other tests: the scratch array keeps the last call's contents and a call must not depend on them.
"""
import numpy as np
import pytest

import workloads

pytestmark = pytest.mark.gpu

ACC_TOL = 1e-12


@pytest.fixture(scope="module")
def G():
    import paper_1404_2324_b200 as G
    from paper_1404_2324_b200 import build
    build.build()
    return G


def existing_path(G, w):
    """(m, x, rcrit, a) as device tensors: state and kick accelerations from a context (workspace allocated by torch)."""
    import torch
    g = G.from_workload(w)
    a, rc = g.accelerations(w["dt"])
    x, _ = g.get_state()
    m = torch.as_tensor(np.ascontiguousarray(w["m"], dtype=np.float64), device=x.device)
    g.synchronize()
    return g, m, x.contiguous(), rc.contiguous(), a


def relerr(a, b):
    a, b = a.cpu().numpy(), b.cpu().numpy()
    return np.linalg.norm(a - b, axis=0) / np.linalg.norm(b, axis=0)


def test_two_calls_in_a_row_match_the_existing_path(G):
    import torch
    cases = [workloads.config1(), workloads.config1(n=777), workloads.config4(n=33, order=4), workloads.config1()]
    refs = [existing_path(G, w) for w in cases]          # every allocation happens here, before the calls under test
    outs = [torch.full_like(r[4], float("nan")) for r in refs]
    torch.cuda.synchronize()
    before = torch.cuda.memory_allocated()
    # back to back on one stream (calls that overlap on the GPU would race on the shared scratch array): a large system, a
    # smaller one that leaves the first one's records and partial sums behind in the array, a tiny one, the first again
    for w, (g, m, x, rc, _), out in zip(cases, refs, outs):
        G.kick_accel_noalloc(w["G"], m, x, rc, out)
    torch.cuda.synchronize()
    assert torch.cuda.memory_allocated() == before
    for w, (g, m, x, rc, a), out in zip(cases, refs, outs):
        err = relerr(out, a)
        assert np.isfinite(err).all() and err.max() <= ACC_TOL, (w["name"], err.max())
    # the same input twice gives the same bits (fixed summation order), whatever ran in between
    assert torch.equal(outs[0], outs[3])
    for g, *_ in refs:
        g.close()


def test_sizes_beyond_the_static_array_are_rejected(G):
    import torch
    n = G.NOALLOC_MAX_BODIES + 1
    m = torch.ones(n, dtype=torch.float64, device="cuda")
    x = torch.rand((3, n), dtype=torch.float64, device="cuda")
    a = torch.zeros((3, n), dtype=torch.float64, device="cuda")
    with pytest.raises(G.GengaError) as e:
        G.kick_accel_noalloc(1.0, m, x, m, a)
    assert e.value.code == G.EINVAL and "GENGA_NOALLOC_MAX_BODIES" in str(e.value)
    torch.cuda.synchronize()
    assert float(a.abs().max()) == 0.0                    # nothing was launched
    # the largest size that fits still works, and an empty system is a no-op
    n = G.NOALLOC_MAX_BODIES
    G.kick_accel_noalloc(1.0, m[:n].contiguous(), x[:, :n].contiguous(), 1e-3 * m[:n].contiguous(), a[:, :n].contiguous())
    e0 = torch.empty(0, dtype=torch.float64, device="cuda")
    G.kick_accel_noalloc(1.0, e0, e0.reshape(3, 0), e0, e0.reshape(3, 0))
    torch.cuda.synchronize()
