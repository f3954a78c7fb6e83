"""Library host logic on the CPU: the C-ABI library loads and exports every declared symbol, argument
validation, and the host-built matrices (the paper's recursion (42)-(44) in binary128 + Jacobi SVD)
against the oracle's (Wigner-d l-recurrence + Householder QR) -- two independent routes."""
import ctypes as C
import re
import os

import numpy as np
import pytest

import oracle
from paper_1104_3408_b200 import Shell, SpError, binding

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_library_exports_every_declared_symbol():
    hdr = open(os.path.join(ROOT, "include", "spshell.h")).read()
    declared = set(re.findall(r"\b(sp_[a-z0-9_]+)\s*\(", hdr))
    assert declared == set(binding.EXPORTED_SYMBOLS)
    L = binding.lib()
    for s in declared:
        assert hasattr(L, s), s


def test_argument_validation():
    L = binding.lib()
    h = C.c_void_p()
    bad = [(9, 8, 15, 1.0, 3.0, 6), (1, 8, 16, 1.0, 3.0, 6), (9, 1, 2, 1.0, 3.0, 0), (9, 8, 16, 3.0, 1.0, 6),
           (9, 8, 16, 0.0, 1.0, 6), (9, 8, 16, 1.0, 3.0, 8), (9, 8, 16, 1.0, 3.0, -1)]
    for a in bad:
        assert L.sp_shell_create(*a[:3], a[3], a[4], a[5], C.byref(h)) == 1, a
    assert L.sp_shell_create(9, 8, 16, 1.0, 3.0, 6, C.byref(h)) == 0
    # hot calls before sp_build_matrices
    assert L.sp_cartesian_gradient(h, 8, 1, 8, 8, 0, None) == 2
    assert L.sp_get_matrix(h, 0, 0, 0, None, None, None) == 2
    assert binding.status_string(2) == "SP_ERR_NOT_BUILT"
    assert L.sp_shell_destroy(h) == 0


@pytest.mark.parametrize("cfg", [(9, 8, 16, 1.0, 3.0, 6), (17, 24, 48, 1.8, 10.0, 19), (33, 48, 96, 1.8, 20.0, 43), (5, 7, 14, 1.0, 2.0, 4)])
def test_host_matrices_match_oracle(cfg):
    Nr, Nt, Np, rmin, rmax, L = cfg
    sh = Shell(Nr, Nt, Np, rmin, rmax, L, host_only=True)
    cd = sh.get_matrix(0)
    ref = oracle.cheb_diff(Nr, rmin, rmax)
    assert np.max(np.abs(cd - ref)) <= 4e-16 * np.max(np.abs(ref)) * 4
    assert np.max(np.abs(sh.get_matrix(1) - oracle.fourier_diff(2 * Nt)[:Nt])) < 1e-14 * Nt
    assert np.max(np.abs(sh.get_matrix(2) - oracle.fourier_diff(Np))) < 1e-14 * Nt
    # Fourier rows (eq. 23-24 with B = sin, reading Q1): round trip synthesis(analysis) = identity on modes <= L
    A, S = sh.get_matrix(3), sh.get_matrix(4)
    assert A.shape == (2 * L + 1, Np) and S.shape == (Np, 2 * L + 1)
    assert np.max(np.abs(A @ S - np.eye(2 * L + 1))) < 1e-14
    ph = 2 * np.pi * np.arange(Np) / Np
    for m in range(1, L + 1):
        assert np.max(np.abs(S[:, 2 * m - 1] - np.cos(m * ph))) < 1e-13 and np.max(np.abs(S[:, 2 * m] - np.sin(m * ph))) < 1e-13
    worst = 0.0
    for n in range(-3, 4):
        for m in range(0, L + 1):
            worst = max(worst, np.max(np.abs(sh.get_matrix(5, n, m) - oracle.filter_matrix(Nt, L, n, m))))
    assert worst < 1e-13, worst


@pytest.mark.parametrize("Nt,L", [(8, 6), (24, 19), (7, 4)])
def test_filter_matrices_equatorial_reflection(Nt, L):
    """sY_lm(pi - theta) = (-1)^(l+m) (-s)Y_lm(theta) and the Gauss grid (eq. 3) is symmetric about the equator, so with R the
    reversal of the latitudes F^{-n}_m = R F^n_m R (F is quadratic in P, the signs cancel); F^0_m is centrosymmetric.  Holds for
    the oracle's matrices and for the library's host build: the basis of an even/odd fold of the theta step."""
    sh = Shell(9, Nt, 2 * Nt, 1.0, 3.0, L, host_only=True)
    for get in (lambda n, m: oracle.filter_matrix(Nt, L, n, m), lambda n, m: sh.get_matrix(5, n, m)):
        for n in range(0, 4):
            for m in range(0, L + 1):
                Fp, Fm = get(n, m), get(-n, m)
                assert np.max(np.abs(Fm - Fp[::-1, ::-1])) < 1e-13


def test_ghg_spatial_degree_and_layout():
    """Host logic of the GHG path: the graded kept degree L + d(u^mu) of eq. 59 (g_tt 0, g_tx 1, g_xx 2; d_iab one
    more spatial index), evaluated behind the ABI (sp_ghg_graded_degree), capped at Ntheta - 1; and the tensor layout."""
    from paper_1104_3408_b200 import Shell
    from paper_1104_3408_b200.binding import SpError
    from paper_1104_3408_b200.ghg import ghg_tensors
    sh = Shell(7, 12, 24, 1.0, 2.0, 5, build=False)
    d = [sh.ghg_graded_degree(q) - 5 for q in range(50)]
    assert d[0] == 0 and d[1] == 1 and d[4] == 2 and d[20] == 1 and d[21] == 2 and d[24] == 3
    assert [d.count(q) for q in range(4)] == [2, 9, 21, 18]
    assert [Shell(7, 12, 24, 1.0, 2.0, 10, build=False).ghg_graded_degree(q) for q in (0, 1, 4, 24)] == [10, 11, 11, 11]   # cap
    import pytest
    with pytest.raises(SpError):
        sh.ghg_graded_degree(50)
    t = ghg_tensors()
    assert sorted(sum((x["fields"] for x in t), [])) == list(range(50))


def test_header_compiles_as_plain_c_and_cxx(tmp_path):
    """The boundary is a C ABI: include/spshell.h must compile as C99 and as C++ on its own, warnings as errors, and a C program
    using every declared entry point must link against the library (no CUDA or C++ type may leak into the signatures)."""
    import subprocess
    hdr = os.path.join(ROOT, "include", "spshell.h")
    src = tmp_path / "use.c"
    src.write_text(
        '#include "spshell.h"\n#include <stdio.h>\n'
        "int main(void) {\n"
        "    sp_shell *s = 0; double dt = 0; int L = 0; size_t g, f, w;\n"
        "    if (sp_shell_create(9, 8, 16, 1.0, 3.0, 6, &s) != SP_OK) return 1;\n"
        "    if (sp_wave_dt(s, 4.0, &dt) != SP_OK || !(dt > 0)) return 2;\n"
        "    if (sp_ghg_graded_degree(s, 24, &L) != SP_OK || L != 7) return 3;\n"
        "    if (sp_workspace_bytes(s, 1, &g, &f, &w) != SP_OK || f == 0) return 4;\n"
        "    if (sp_tensor_filter_noalloc(s, 0, 0, 0, 0, 0, 0) != SP_ERR_INVALID_ARG) return 5;\n"
        '    printf("%s %u\\n", sp_status_string(SP_ERR_SCRATCH_LIMIT), (unsigned)SP_NOALLOC_SCRATCH_BYTES);\n'
        "    return sp_shell_destroy(s) == SP_OK ? 0 : 6;\n}\n")
    inc = os.path.join(ROOT, "include")
    subprocess.run(["gcc", "-std=c99", "-Wall", "-Wextra", "-Werror", "-pedantic", "-fsyntax-only", "-x", "c", hdr], check=True)
    subprocess.run(["g++", "-std=c++17", "-Wall", "-Wextra", "-Werror", "-fsyntax-only", "-x", "c++", hdr], check=True)
    exe = tmp_path / "use"
    libdir = os.path.dirname(binding.library_path())
    subprocess.run(["gcc", "-std=c99", "-Wall", "-Werror", "-I", inc, str(src), "-o", str(exe), "-L", libdir, "-lspshell",
                    "-Wl,-rpath," + libdir], check=True)
    r = subprocess.run([str(exe)], capture_output=True, text=True)
    assert r.returncode == 0, (r.returncode, r.stderr)
    assert "SCRATCH_LIMIT" in r.stdout and str(32 * 1024 * 1024) in r.stdout
