"""CPU-side checks of the C-ABI boundary: the library builds for sm_100a, exports every symbol
include/tpcca.h declares, its host-only entry points work, and without a GPU it fails LOUDLY
(there is no CPU fallback).  No compute calls here."""
import ctypes as C
import os
import re
import subprocess

import numpy as np
import pytest

import tpcsynth

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def pkg():
    import paper_2208_07412_b200 as p
    p.load_library()
    return p


def declared_symbols():
    txt = open(os.path.join(ROOT, "include", "tpcca.h")).read()
    txt = re.sub(r"/\*.*?\*/", "", txt, flags=re.S)
    return sorted(set(re.findall(r"\b(tpcca_[a-z_]+)\s*\(", txt)))


def test_library_exports_every_declared_symbol(pkg):
    syms = declared_symbols()
    assert len(syms) >= 12 and "tpcca_create" in syms and "tpcca_get_tracks" in syms
    lib = C.CDLL(pkg.library_path())
    for s in syms:
        assert hasattr(lib, s), s
    assert sorted(pkg.abi_symbols()) == syms
    out = subprocess.run(["nm", "-D", "--defined-only", pkg.library_path()], capture_output=True, text=True).stdout
    for s in syms:
        assert re.search(rf"\bT {s}\b", out), s


def test_library_holds_sm100a_code_only(pkg):
    out = subprocess.run(["cuobjdump", "-lelf", pkg.library_path()], capture_output=True, text=True).stdout
    archs = set(re.findall(r"sm_\d+a?", out))
    assert archs == {"sm_100a"}, archs


def test_python_binding_does_not_import_the_oracle():
    """The product path never routes through oracle/ (and the oracle never imports the product)."""
    for root, _, files in os.walk(os.path.join(ROOT, "paper_2208_07412_b200")):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                txt = open(os.path.join(root, f)).read()
                assert not re.search(r"^\s*(from|import)\s+oracle\b", txt, flags=re.M), f
                assert "liboracle" not in txt and "tpcca_oracle" not in txt, f
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith((".py", ".cpp")):
            txt = open(os.path.join(ROOT, "oracle", f)).read()
            assert "paper_2208_07412_b200 import" not in txt and "libtpcca" not in txt, f


def test_workspace_bytes_host_only(pkg):
    from paper_2208_07412_b200.binding import workspace_bytes
    P = tpcsynth.default_params(n_sectors=36)
    a = workspace_bytes(P, 1_000_000)
    b = workspace_bytes(P, 2_000_000)
    c = workspace_bytes(P, 2_000_000, max_start_hits=1_000_000)
    assert 0 < a < b < c
    # config-3 footprint fits one B200 (180 GB) with room to spare
    Ptf = tpcsynth.default_params(n_sectors=36, z_hi=250.0 + tpcsynth.V_DRIFT * 128 * tpcsynth.ORBIT_US)
    big = workspace_bytes(Ptf, 160_000_000)
    assert big < 100e9
    # bad tables are rejected with a message
    bad = P.copy()
    bad.grid_ny = bad.grid_ny.copy(); bad.grid_ny[3] = 0
    with pytest.raises(pkg.TpccaError) as e:
        workspace_bytes(bad, 1000)
    assert e.value.code == -1 and "grid_ny" in str(e.value)


def test_no_gpu_means_loud_failure(pkg):
    import torch
    if torch.cuda.is_available():
        pytest.skip("a GPU is present")
    P = tpcsynth.default_params(n_sectors=1)
    with pytest.raises(pkg.TpccaError) as e:
        pkg.Tracker(P, max_clusters=100)
    assert e.value.code == -3
    # straight through the C-ABI as well
    from paper_2208_07412_b200.binding import _make_params
    lib = pkg.load_library()
    p, keep = _make_params(P)
    h = C.c_void_p()
    rc = lib.tpcca_create(C.byref(p), 0, None, C.c_void_p(256), 1 << 30, 100, 0, C.byref(h))
    assert rc == -3 and not h.value
    assert b"no CPU path" in lib.tpcca_last_error(None)
