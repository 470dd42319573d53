"""The C-ABI library loads and exports every symbol include/tfa.h declares (no GPU needed)."""
import ctypes
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def header_symbols():
    txt = open(os.path.join(ROOT, "include", "tfa.h")).read()
    txt = re.sub(r"/\*.*?\*/", "", txt, flags=re.S)
    return sorted(set(re.findall(r"\b(tfa_[a-z_0-9]+)\s*\(", txt)))


@pytest.fixture(scope="module")
def lib():
    from paper_1809_02532_b200 import build
    path = build.build()
    return ctypes.CDLL(path)


def test_header_and_binding_agree():
    from paper_1809_02532_b200 import _lib
    assert header_symbols() == sorted(_lib.SYMBOLS)


def test_every_declared_symbol_is_exported(lib):
    for name in header_symbols():
        assert hasattr(lib, name), name


def test_struct_layouts_match_the_header(lib):
    """ctypes mirrors vs the sizes implied by the header: 6 doubles; 27 doubles + 2 int32."""
    from paper_1809_02532_b200 import _lib
    assert ctypes.sizeof(_lib.Physics) == 6 * 8
    assert ctypes.sizeof(_lib.Numerics) == (1 + 18 + 2 + 4 + 2) * 8 + 8
    L = _lib.load()
    p = _lib.Physics()
    L.tfa_default_physics(ctypes.byref(p))
    assert (p.gamma_gas, p.mass_ratio, p.c, p.gamma_psi, p.chi_phi, p.rusanov_alpha) == (5.0 / 3.0, 25.0, 20.0, 1, 1, 1)
    n = _lib.Numerics()
    L.tfa_default_numerics(ctypes.byref(n), ctypes.byref(p))
    assert n.fd_delta == 1e-6 and n.fd_ref[9] == 1.0 / 25.0 and n.fd_ref[8] == 1.0
    assert n.term_mask == 7 and n.ausm_Minf[1] == 0.1 and n.ausm_beta == 0.125
    assert L.tfa_version().decode().startswith("tfa")


def test_defaults_agree_with_the_oracle(orc, lib):
    """Both sides state the same default constants (they are declared twice, independently)."""
    from paper_1809_02532_b200 import _lib
    L = _lib.load()
    p = _lib.Physics()
    L.tfa_default_physics(ctypes.byref(p))
    n = _lib.Numerics()
    L.tfa_default_numerics(ctypes.byref(n), ctypes.byref(p))
    po = orc.physics_c()
    no = orc.default_numerics(po)
    assert bytes(p) == bytes(po)
    assert bytes(n) == bytes(no)


def test_product_does_not_import_the_oracle():
    pkg = os.path.join(ROOT, "paper_1809_02532_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                src = open(os.path.join(dirpath, f)).read()
                for pat in (r"^\s*(import|from)\s+oracle", r"#include\s+[\"<].*(oracle|tfo)", r"liboracle",
                            r"\btfo_"):
                    assert not re.search(pat, src, flags=re.M), (f, pat)
