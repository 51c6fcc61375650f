"""CPU-side checks of the C-ABI boundary: the library loads, exports every symbol the header
declares, and rejects bad arguments before touching the GPU (no compute calls here)."""
import ctypes as C
import os
import re

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def B():
    from paper_1210_1017_b200 import build
    build.build_library()
    from paper_1210_1017_b200 import binding
    return binding


def _declared_symbols():
    text = open(os.path.join(ROOT, "include", "sph_b200.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(sph_[a-z_0-9]+)\s*\(", text)))


def test_library_exports_every_declared_symbol(B):
    names = _declared_symbols()
    assert len(names) >= 15
    lib = C.CDLL(B.LIB_PATH)
    for name in names:
        assert hasattr(lib, name), f"{name} declared in sph_b200.h but not exported"
    assert sorted(B.EXPORTS) == names


def test_struct_layouts_match_header(B):
    # sizes implied by the header on LP64: params 19 words; particles 7 words of 8; view 40 B + 16 pointers
    assert C.sizeof(B.sph_params) == 4 * 19
    assert C.sizeof(B.sph_particles) == 8 * 7
    assert C.sizeof(B.sph_view) == 8 + 12 + 4 + 4 + 4 + 8 + 16 * 8


def test_workspace_bytes_and_argument_errors(B):
    from paper_1210_1017_b200 import workloads as W
    w = W.dam_break(16)
    p = B.make_params(w.params)
    b1 = B.sph_workspace_bytes(p, w.n, 1)
    b16 = B.sph_workspace_bytes(p, w.n, 16)
    assert 0 < b1 < b16 < 400 * w.n + (1 << 22)
    assert B.sph_workspace_bytes(p, (1 << 28) + 1, 1) == 0    # n too large
    assert B.sph_workspace_bytes(p, w.n, 17) == 0             # too many slabs
    big = dict(w.params)
    big["dom_max"] = (1e4, 1e4, 1e4)                          # > 2^28 cells
    assert B.sph_workspace_bytes(B.make_params(big), 10, 1) == 0

    # sph_init refuses a missing workspace before any CUDA call
    ctx = C.c_void_p()
    part = B.sph_particles()
    part.n = w.n
    part.pos = w.pos.ctypes.data
    part.vel = w.vel.ctypes.data
    part.rho = w.rho.ctypes.data
    rc = B._lib.sph_init(C.byref(ctx), C.byref(p), C.byref(part), 1, None, 0, None)
    assert rc == -2 and not ctx.value
    bad = B.make_params(w.params)
    bad.gamma = 0
    assert B._lib.sph_init(C.byref(ctx), C.byref(bad), C.byref(part), 1, None, 0, None) == -1
    assert B._lib.sph_init(C.byref(ctx), C.byref(B.make_params(big)), C.byref(part), 1, None, 0, None) == -3
    assert B.sph_strerror(0) == "ok" and "slab" in B.sph_strerror(-4)
    for code in range(-8, 1):
        assert B.sph_strerror(code) != "unknown error"


def test_no_cpu_fallback_without_device(B):
    import torch
    if torch.cuda.is_available():
        pytest.skip("GPU present")
    from paper_1210_1017_b200 import workloads as W
    w = W.dam_break(6)
    with pytest.raises(RuntimeError):
        B.Sph(w.params, w.pos, w.vel, w.rho, w.type)


def test_product_does_not_import_oracle():
    pkg = os.path.join(ROOT, "paper_1210_1017_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                text = open(os.path.join(dirpath, f)).read()
                assert not re.search(r"^\s*(from|import)\s+oracle", text, flags=re.M), f
                assert "liborc" not in text and "sph_physics" not in text and "orc_" not in text, f
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith((".py", ".c")):
            text = open(os.path.join(ROOT, "oracle", f)).read()
            assert "paper_1210_1017_b200" not in text and "sph_b200" not in text, f
