"""CPU-side checks of the boundary: libsph.so loads and exports every symbol include/sph.h
declares; argument checks that need no GPU behave as documented."""
import ctypes as C
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    from paper_2603_19764_b200 import build, binding
    build.build()
    return binding.load()


def declared_symbols():
    src = open(os.path.join(ROOT, "include", "sph.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(sph_[a-z_0-9]+)\s*\(", src)))


def test_header_and_binding_agree():
    from paper_2603_19764_b200 import binding
    assert declared_symbols() == sorted(binding.SYMBOLS)


def test_library_exports_every_declared_symbol(lib):
    for s in declared_symbols():
        assert hasattr(lib, s), s


def test_struct_layout_matches_header():
    from paper_2603_19764_b200 import binding as B
    assert C.sizeof(B.sph_material) == 11 * 4
    assert C.sizeof(B.sph_params) == 6 * 4 + 4 + 4 + 8 * 11 * 4 + 4 + 4 * 4
    assert C.sizeof(B.sph_state) == 19 * C.sizeof(C.c_void_p)


def test_argument_errors_without_gpu(lib):
    from paper_2603_19764_b200 import binding as B
    assert lib.sph_workspace_bytes(None, 100) == 0
    p = B.sph_params()
    assert lib.sph_workspace_bytes(C.byref(p), 100) == 0           # n_materials = 0
    ctx = C.c_void_p()
    assert lib.sph_init(C.byref(ctx), None, 10, None, 0, None) == B.EINVAL
    assert lib.sph_density(None) == B.EINVAL
    assert lib.sph_step(None, None, 0, 0.0, None) == B.EINVAL
    assert lib.sph_strerror(B.EORDER).decode().startswith("pass called")
    assert lib.sph_strerror(0).decode() == "ok"
    lib.sph_destroy(None)


def test_retired_and_unknown_flag_bits_are_refused(lib):
    """Bit 8 once meant the opposite Jaumann choice, 128 and 256 selected kernels that no longer exist: a caller that
    still passes one of them must hear about it (sph.h), not get something else silently."""
    from paper_2603_19764_b200 import binding as B, workloads as W
    p = B.make_params(W.Params())
    assert lib.sph_workspace_bytes(C.byref(p), 100) > 0
    for bit in (8, 128, 256, 1024, 1 << 31):
        q = B.make_params(W.Params())
        q.flags |= bit
        assert lib.sph_workspace_bytes(C.byref(q), 100) == 0, bit
        ctx = C.c_void_p()
        assert lib.sph_init(C.byref(ctx), C.byref(q), 100, C.c_void_p(256), 1 << 30, None) == B.EINVAL, bit
    for bit in (1, 2, 4, 16, 32, 64, 512):
        q = B.make_params(W.Params())
        q.flags |= bit
        assert lib.sph_workspace_bytes(C.byref(q), 100) > 0, bit
    assert B.JAUMANN_AS_PRINTED == W.FLAG_JAUMANN_AS_PRINTED == 512


def test_no_cpu_fallback_when_library_missing(monkeypatch, tmp_path):
    from paper_2603_19764_b200 import binding as B
    monkeypatch.setattr(B, "_lib", None)
    monkeypatch.setattr(B, "LIB_PATH", str(tmp_path / "nope.so"))
    with pytest.raises(RuntimeError, match="no CPU fallback"):
        B.load()


def test_product_does_not_import_the_oracle():
    pkg = os.path.join(ROOT, "paper_2603_19764_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                txt = open(os.path.join(dirpath, f)).read()
                assert "oracle" not in txt.replace("oracle/", "").replace("the oracle", "").replace("CPU oracle", "") \
                    or f in ("workloads.py",), f
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith((".py", ".c")):
            txt = open(os.path.join(ROOT, "oracle", f)).read()
            assert "import paper_2603" not in txt and "from paper_2603" not in txt and "libsph" not in txt
