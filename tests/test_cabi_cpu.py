"""CPU-side checks of the boundary: the library builds/loads and exports every symbol include/rpa_b200.h declares;
without a GPU the product path fails loudly (no fallback)."""
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def declared_symbols():
    text = open(os.path.join(ROOT, "include", "rpa_b200.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(rpa_[a-z0-9_]+)\s*\(", text)))


def test_library_exports_every_declared_symbol():
    import paper_2405_20258_b200 as rpa
    lib = rpa.load_library()
    syms = declared_symbols()
    assert "rpa_create" in syms and "rpa_correlation_energy" in syms and len(syms) >= 12
    for s in syms:
        assert hasattr(lib, s), f"{s} declared in rpa_b200.h but not exported"
    assert sorted(rpa.EXPORTED_SYMBOLS) == syms


def test_no_cpu_fallback():
    import torch
    import paper_2405_20258_b200 as rpa
    if torch.cuda.is_available():
        pytest.skip("GPU present")
    with pytest.raises(rpa.RpaError) as ei:
        rpa.rpa_create([1, 0, 0, 0, 1, 0, 0, 0, 1], [8, 8, 8], [[0, 0, 0]], [1.0], [[0, 0, 0]])
    assert ei.value.code == -3


def test_product_never_imports_oracle():
    pkg = os.path.join(ROOT, "paper_2405_20258_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                src = open(os.path.join(dirpath, f)).read()
                assert "oracle" not in src.replace("no CPU fallback", ""), f"{f} mentions the oracle"
    osrc = open(os.path.join(ROOT, "oracle", "rpa_oracle.py")).read()
    assert "import paper_2405_20258_b200" not in osrc and "from paper_2405_20258_b200" not in osrc


def test_no_process_wide_state_in_the_library():
    """Kernel attributes and tuning switches are per context (a process may hold contexts on several devices): no
    function-local `static` variable and no getenv outside rpa_create."""
    csrc = os.path.join(ROOT, "paper_2405_20258_b200", "csrc")
    for f in sorted(os.listdir(csrc)):
        src = open(os.path.join(csrc, f)).read()
        src = re.sub(r"//[^\n]*", "", src)
        for m in re.finditer(r"^[ \t]+static\s+(?!constexpr|inline|__device__|__forceinline__)[^;(]*[=;]", src, flags=re.M):
            raise AssertionError(f"{f}: function-local static state: {m.group(0).strip()}")
        if f != "api.cu":
            assert "getenv" not in src, f"{f} reads the environment outside rpa_create"
    api = open(os.path.join(csrc, "api.cu")).read()
    body = api[api.index("int rpa_create("):api.index("int rpa_destroy(")]
    assert api.count("getenv(") == body.count("getenv(")


def test_binding_rejects_misshaped_arrays_before_the_call():
    """The C ABI takes raw pointers: the binding must refuse any array whose shape disagrees with the sizes it passes
    (checked before any pointer is taken, so this runs without a GPU and without a library context)."""
    import numpy as np
    import torch
    import paper_2405_20258_b200 as rpa
    ctx = rpa.RpaContext(None, 0, n_g=5, n_pw=7)
    c128, f64 = torch.complex128, torch.float64
    z = lambda *s: torch.zeros(s, dtype=c128)
    r = lambda *s: torch.zeros(s, dtype=f64)
    bad_calls = [
        lambda: rpa.rpa_mtxel(ctx, z(2, 6), z(3, 7), z(2, 3, 5)),                      # psi_v has the wrong n_pw
        lambda: rpa.rpa_mtxel(ctx, z(2, 7), z(3, 7), z(2, 3, 4)),                      # M has the wrong n_g
        lambda: rpa.rpa_mtxel(ctx, z(2, 7), z(3, 7), z(3, 2, 5)),                      # M transposed
        lambda: rpa.rpa_chi0_static(ctx, z(2, 3, 5), r(2), r(4), False, z(5, 5)),      # e_c disagrees with M
        lambda: rpa.rpa_chi0_static(ctx, z(2, 3, 5), r(2), r(3), False, z(5, 4)),      # chi0 not n_g x n_g
        lambda: rpa.rpa_subspace_basis(ctx, z(5, 5), 2, 0.0, z(2, 4), r(2)),           # C rows not n_g long
        lambda: rpa.rpa_subspace_basis(ctx, z(5, 5), 2, 0.0, z(2, 5), r(3)),           # lambda not n_eig long
        lambda: rpa.rpa_chi_subspace_freq(ctx, z(2, 3, 5), r(2), r(3), z(2, 5), 2, r(4), False, z(4, 2, 3)),   # chi_s not square
        lambda: rpa.rpa_chi_subspace_freq(ctx, z(2, 3, 5), r(2), r(3), None, 4, r(4), False, z(4, 4, 4)),      # full basis needs n_eig = n_g
        lambda: rpa.rpa_chi_subspace_freq_occ(ctx, z(2, 3, 5), r(2), r(3), r(2), r(2), z(2, 5), 2, r(4), False, z(4, 2, 2)),   # f_c
        lambda: rpa.rpa_correlation_energy(ctx, z(4, 2, 2), 2, r(3)),                  # weights disagree with chi_s
        lambda: rpa.rpa_epsilon_inverse(ctx, z(4, 2, 2), z(4, 2, 3)),
        lambda: rpa.rpa_energy_host(ctx, np.zeros((2, 7), complex), np.zeros((3, 6), complex), np.zeros(2), np.zeros(3), 2, 2, 0.0,
                                    np.zeros(4), np.zeros(4)),                          # psi_c has the wrong n_pw
        lambda: rpa.rpa_energy_host(ctx, np.zeros((2, 7), complex), np.zeros((3, 7), complex), np.zeros(2), np.zeros(3), 2, 6, 0.0,
                                    np.zeros(4), np.zeros(4)),                          # n_eig > n_g
    ]
    for i, call in enumerate(bad_calls):
        with pytest.raises(TypeError):
            call()
            raise AssertionError(f"bad call {i} was accepted")
    ctx.handle = None
