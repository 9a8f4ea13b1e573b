"""CPU-side checks of the boundary: the library loads, exports every symbol include/genga.h
declares, and its host-only logic (config validation, workspace sizing, error strings) works.
No compute call is made here."""
import ctypes as C
import os
import re
import subprocess
import sys

import pytest

import paper_1404_2324_b200 as G
from paper_1404_2324_b200 import build as B

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    B.build()
    return G.load()


def declared_symbols():
    src = open(os.path.join(ROOT, "include", "genga.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(genga_[a-z0-9_]+)\s*\(", src)))


def test_library_exports_every_declared_symbol(lib):
    names = declared_symbols()
    assert "genga_step" in names and "genga_encounters" in names and len(names) >= 16
    for n in names:
        assert hasattr(lib, n), n
    assert sorted(G.SYMBOLS) == names
    out = subprocess.run(["nm", "-D", "--defined-only", G.LIB_PATH], capture_output=True, text=True).stdout
    exported = set(re.findall(r"\bT (genga_\w+)", out))
    assert exported == set(names)


def test_library_is_sm100a_and_names_no_batch_memcpy():
    out = subprocess.run(["cuobjdump", "-lelf", G.LIB_PATH], capture_output=True, text=True).stdout
    assert "sm_100a" in out


def _cfg(mode, nm, nt=0, ns=1, **kw):
    d = dict(G=1.0, n1=3.0, n2=0.4, bs_eps=1e-12, max_pairs=1000)
    d.update(kw)
    return G.genga_config(mode, nm, nt, ns, 0, d["G"], d["n1"], d["n2"], d["bs_eps"], d["max_pairs"], None, 0, None)


def test_workspace_size_and_limits(lib):
    ok = [_cfg(0, 1), _cfg(0, 2048), _cfg(1, 32, 1_000_000), _cfg(1, 8, 0), _cfg(2, 16, 0, 100_000)]
    sizes = [lib.genga_workspace_bytes(C.byref(c)) for c in ok]
    assert all(s > 0 and s % 256 == 0 for s in sizes)
    assert sizes[1] > sizes[0] and sizes[2] > 16 * 8 * 1_000_000
    bad = [_cfg(0, 0), _cfg(0, 2049), _cfg(0, 10, 5), _cfg(1, 33, 10), _cfg(1, 8, 1_000_001), _cfg(2, 17, 0, 10),
           _cfg(2, 16, 0, 100_001), _cfg(3, 5), _cfg(0, 5, G=0.0), _cfg(0, 5, bs_eps=0.0), _cfg(0, 5, max_pairs=0), _cfg(0, 5, max_pairs=2**31)]
    for c in bad:
        assert lib.genga_workspace_bytes(C.byref(c)) == 0
    assert lib.genga_workspace_bytes(None) == 0


def test_null_and_invalid_arguments_are_rejected_without_a_device(lib):
    h = C.c_void_p()
    assert lib.genga_create(None, C.byref(h)) == G.EINVAL
    assert lib.genga_create(C.byref(_cfg(0, 5)), C.byref(h)) == G.EINVAL       # NULL workspace
    assert lib.genga_destroy(None) == G.EINVAL
    assert lib.genga_step(None, 1, 0.1, 2) == G.EINVAL
    assert lib.genga_status(None) == G.EINVAL
    for code in (0, -1, -2, -3, -4, -5, -99):
        assert len(lib.genga_strerror(code)) > 0
    assert b"capacity" in lib.genga_strerror(G.ECAPACITY)


def test_product_does_not_touch_the_oracle():
    """The product path may not import, link or read anything under oracle/."""
    pkg = os.path.join(ROOT, "paper_1404_2324_b200")
    for root, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                txt = open(os.path.join(root, f)).read()
                assert "import oracle" not in txt and "genga_oracle" not in txt and "ora_" not in txt, f
    otxt = open(os.path.join(ROOT, "oracle", "__init__.py")).read() + open(os.path.join(ROOT, "oracle", "genga_oracle.c")).read()
    assert "import paper_1404_2324_b200" not in otxt and "libgenga_b200" not in otxt and "csrc" not in otxt


def test_context_creation_fails_loudly_without_cuda():
    import torch
    if torch.cuda.is_available():
        pytest.skip("CUDA present")
    with pytest.raises(RuntimeError, match="no CPU fallback"):
        G.Genga(0, 4)
