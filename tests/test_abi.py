"""No-GPU checks of the boundary: the C-ABI library builds for sm_100a, loads, and exports every symbol
that include/echo.h declares; host-only calls validate their arguments.  No compute call is made."""
import ctypes as C
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def libpath():
    from paper_2401_03008_b200 import build
    return build.build()


def declared_symbols():
    text = open(os.path.join(ROOT, "include", "echo.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(echo_[a-z0-9_]+)\s*\(", text)))


def test_header_declares_the_north_star_calls():
    syms = declared_symbols()
    for name in ("echo_create", "echo_set_primitives", "echo_step", "echo_get_primitives", "echo_con2prim",
                 "echo_div_b", "echo_diagnostics"):
        assert name in syms


def test_library_exports_every_declared_symbol(libpath):
    L = C.CDLL(libpath)
    for name in declared_symbols():
        assert hasattr(L, name), name


def test_binding_signature_table_matches_header(libpath):
    from paper_2401_03008_b200 import binding
    assert sorted(binding.SIGNATURES) == declared_symbols()
    binding.lib()


def test_host_only_calls(libpath):
    from paper_2401_03008_b200 import binding
    L = binding.lib()
    assert not L.echo_create(0, 1, 1, 4.0 / 3.0, 0.3)
    assert not L.echo_create(8, 8, 8, 0.9, 0.3)
    assert not L.echo_create(8, 8, 8, 4.0 / 3.0, -1.0)
    assert not L.echo_create(2, 70000, 2, 4.0 / 3.0, 0.3)                # the z-sweep puts y on gridDim.z
    h2 = L.echo_create(2, 70000, 1, 4.0 / 3.0, 0.3)                      # a flat grid does not
    assert h2
    L.echo_destroy(h2)
    h = L.echo_create(8, 6, 4, 4.0 / 3.0, 0.3)
    assert h
    n = 8 * 6 * 4
    assert L.echo_workspace_bytes(h) >= 44 * 8 * n
    assert L.echo_step(h, 1, float("inf")) == binding.ECHO_ESTATE       # not bound: refused on the host
    assert L.echo_bind(h, None, 0, None) == binding.ECHO_ENOMEM
    assert L.echo_last_error(h)
    L.echo_destroy(h)


def test_product_does_not_import_the_oracle():
    """The product path shares nothing with oracle/ and has no CPU fallback."""
    pkg = os.path.join(ROOT, "paper_2401_03008_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                text = open(os.path.join(dirpath, f)).read()
                assert "import oracle" not in text and "from oracle" not in text, f
                assert "echo_oracle" not in text, f
