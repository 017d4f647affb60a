"""C-ABI boundary checks that need no GPU: the library builds for sm_100a, loads, exports every symbol that
include/mdpd.h declares, sizes its workspace sensibly (host logic), and FAILS LOUDLY without a CUDA device."""
import ctypes as C
import os
import re

import numpy as np
import pytest

import mdpd_workloads as wl

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def pk():
    from paper_1903_10134_b200 import build
    build()
    import paper_1903_10134_b200 as pk
    return pk


def declared_symbols():
    src = open(os.path.join(ROOT, "include", "mdpd.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(mdpd_[a-z_]+)\s*\(", src)))


def test_every_declared_symbol_is_exported(pk):
    names = declared_symbols()
    assert len(names) >= 15 and "mdpd_step" in names
    L = pk.lib()
    for s in names:
        assert hasattr(L, s), s
    assert sorted(pk.SYMBOLS) == names


def test_params_struct_matches_header(pk):
    """18 float + 4 uint32 fields in the header's order = 88 bytes, no padding."""
    assert C.sizeof(pk.mdpd_params) == 22 * 4
    src = open(os.path.join(ROOT, "include", "mdpd.h")).read()
    body = re.search(r"typedef struct \{(.*?)\} mdpd_params;", src, flags=re.S).group(1)
    body = re.sub(r"/\*.*?\*/", "", body, flags=re.S)
    fields = []
    for decl in body.split(";"):
        decl = decl.strip()
        if not decl:
            continue
        for nm in decl.split(None, 1)[1].split(","):
            fields.append(re.sub(r"\[.*\]", "", nm.strip()))
    assert fields == [f[0] for f in pk.mdpd_params._fields_]


def test_workspace_bytes_host_logic(pk):
    p = pk.make_params(wl.default_params((55.0, 55.0, 55.0)))
    n = 998_250
    b = pk.lib().mdpd_workspace_bytes(C.byref(p), n, 0, None)
    # state (pos, vel x2, force, xbuild) = 96 B/particle; the list dominates: a few hundred bytes per particle
    assert 96 * n < b < 1200 * n
    md = (C.c_uint32 * 3)(128, 128, 128)
    assert pk.lib().mdpd_workspace_bytes(C.byref(p), n, 1, md) >= b + 128 ** 3 - 4096
    # 32 M particles fit a 180 GB B200 with room to spare
    p = pk.make_params(wl.default_params((175.0, 175.0, 175.0)))
    assert pk.lib().mdpd_workspace_bytes(C.byref(p), 32_156_250, 0, None) < 60e9
    # invalid parameters -> 0
    for bad in (dict(rd=1.5), dict(s=-0.5), dict(s=5.0), dict(skin=-1.0), dict(dt=0.0), dict(reorder_every=3)):
        q = pk.make_params(wl.default_params((10.0, 10.0, 10.0), **bad))
        assert pk.lib().mdpd_workspace_bytes(C.byref(q), 100, 0, None) == 0, bad
    q = pk.make_params(wl.default_params((3.0, 10.0, 10.0)))     # fewer than 3 cells of rc + skin along x (R4)
    assert pk.lib().mdpd_workspace_bytes(C.byref(q), 100, 0, None) == 0


def test_no_cpu_fallback(pk):
    """Without a CUDA device mdpd_create returns MDPD_ECUDA and the binding raises; nothing computes on the CPU."""
    import torch
    if torch.cuda.is_available():
        pytest.skip("a GPU is present")
    h = C.c_void_p()
    assert pk.lib().mdpd_create(C.byref(h), 0, None) == -3
    assert not h.value
    with pytest.raises(RuntimeError):
        pk.Simulation(wl.default_params((10.0, 10.0, 10.0)))


def test_product_never_imports_the_oracle():
    for dirpath, _, files in os.walk(os.path.join(ROOT, "paper_1903_10134_b200")):
        for f in files:
            if f.endswith((".py", ".cu", ".h", ".cuh")):
                txt = open(os.path.join(dirpath, f)).read()
                assert "oracle" not in txt.replace("(the fp64 CPU oracle)", "").replace("shares nothing with oracle/", ""), f
    txt = open(os.path.join(ROOT, "oracle", "mdpd_ref.py")).read()
    assert "import paper_1903_10134_b200" not in txt and "from paper_1903_10134_b200" not in txt
