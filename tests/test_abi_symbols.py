"""CPU-only: the C-ABI library builds/loads and exports every symbol include/kg.h declares;
host-only entry points (Bessel coefficients, argument validation) behave."""
import ctypes as C
import os
import re

import numpy as np
import scipy.special

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _declared():
    src = open(os.path.join(ROOT, "include", "kg.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(kg_[a-z0-9_]+)\s*\(", src)))


def test_library_exports_every_declared_symbol():
    from paper_1307_0288_b200 import build
    lib = C.CDLL(build.build())
    names = _declared()
    for must in ("kg_create_hamiltonian", "kg_dos_moments", "kg_evolve", "kg_apply_velocity",
                 "kg_vac", "kg_msd", "kg_moments", "kg_evolve_x", "kg_destroy_hamiltonian",
                 "kg_last_error", "kg_create_hamiltonian_csr", "kg_workspace_bytes"):
        assert must in names
    for name in names:
        assert hasattr(lib, name), name


def test_bessel_terms_host():
    from paper_1307_0288_b200 import binding as B
    assert B.bessel_terms(np.pi)[0] == 21                        # P:474 "about 20"
    for x, want in ((3.15, 21), (6.3, 28), (14.7, 42), (25.2, 57)):   # configs 1-5
        n_p, j = B.bessel_terms(x)
        assert n_p == want
        assert np.max(np.abs(j - scipy.special.jv(np.arange(n_p), x))) < 1e-15
        assert abs(j[0] ** 2 + 2 * np.sum(j[1:] ** 2) - 1) < 2e-15


def test_argument_validation_without_gpu():
    from paper_1307_0288_b200 import binding as B
    lib = B._lib
    out = C.c_void_p()
    a = np.zeros(4, np.int32); d = np.zeros(4)
    rc = lib.kg_create_hamiltonian(C.byref(out), 0, 1, a.ctypes.data, a.ctypes.data, d.ctypes.data,
                                   None, d.ctypes.data, 0.0, 0.0, 1.0, None)
    assert rc == B.KG_EINVAL and b"n must be" in lib.kg_last_error()
    rc = lib.kg_create_hamiltonian(C.byref(out), 4, 1, a.ctypes.data, a.ctypes.data, d.ctypes.data,
                                   None, d.ctypes.data, 0.0, 0.0, -1.0, None)
    assert rc == B.KG_EINVAL
    rc = lib.kg_create_hamiltonian(C.byref(out), 4, 40, a.ctypes.data, a.ctypes.data, d.ctypes.data,
                                   None, d.ctypes.data, 0.0, 0.0, 1.0, None)
    assert rc == B.KG_EUNSUPPORTED
    rc = lib.kg_create_hamiltonian(C.byref(out), 4, 1, None, a.ctypes.data, d.ctypes.data,
                                   None, d.ctypes.data, 0.0, 0.0, 1.0, None)
    assert rc == B.KG_EINVAL
    assert lib.kg_dos_moments(None, None, 1, 4, None, None) == B.KG_EINVAL
    assert lib.kg_destroy_hamiltonian(None) == B.KG_OK


def test_product_does_not_import_oracle():
    """The product path must not route through the oracle (and vice versa)."""
    pkg = os.path.join(ROOT, "paper_1307_0288_b200")
    pat = re.compile(r"^\s*(from|import)\s+\.*oracle|kgo\.|libkgo|#include\s+\"kgo", re.M)
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                assert not pat.search(open(os.path.join(dirpath, f)).read()), f
    pat = re.compile(r"^\s*(from|import)\s+paper_1307_0288_b200|libkg\.so|#include\s+\"kg", re.M)
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith((".py", ".c", ".h")):
            assert not pat.search(open(os.path.join(ROOT, "oracle", f)).read()), f
