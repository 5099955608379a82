"""CPU-side checks of the C-ABI boundary: the library loads, exports every symbol declared in
include/cans_poisson.h, and rejects bad arguments before touching the GPU."""
import ctypes
import os
import re
import subprocess
import tempfile

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
HEADER = os.path.join(ROOT, "include", "cans_poisson.h")


@pytest.fixture(scope="module")
def binding():
    from paper_2001_05234_b200 import build
    build.build()
    from paper_2001_05234_b200 import binding as b
    return b


def declared_functions():
    """Every function declared in include/*.h (the API header and the probe header)."""
    names = set()
    inc = os.path.dirname(HEADER)
    for fn in sorted(os.listdir(inc)):
        if fn.endswith(".h"):
            txt = open(os.path.join(inc, fn)).read()
            txt = re.sub(r"/\*.*?\*/", "", txt, flags=re.S)
            names.update(re.findall(r"\b(cans_[a-z0-9_]+)\s*\(", txt))
    return sorted(names)


def test_header_symbols_are_exported(binding):
    lib = ctypes.CDLL(binding.LIB_PATH)
    names = declared_functions()
    assert "cans_poisson_plan_create" in names and "cans_poisson_solve" in names and "cans_projection" in names
    for name in names:
        assert hasattr(lib, name), f"{name} declared in the header but not exported"
    assert set(binding.EXPORTED_SYMBOLS) == set(names)


def test_version_and_error_strings(binding):
    assert re.match(r"^\d+\.\d+$", binding.version())
    assert isinstance(binding.last_error(), str)


PP_NN = (("P", "P"), ("P", "P"), ("N", "N"))


@pytest.mark.parametrize("kwargs,status", [
    (dict(nx=1, ny=32, nz=32), 1),
    (dict(nx=32, ny=32, nz=32, lx=-1.0), 1),
    (dict(nx=32, ny=32, nz=32, bc=(("P", "N"), ("P", "P"), ("N", "N"))), 1),      # one-sided periodic
    (dict(nx=32, ny=32, nz=32, bc=(("X", "X"), ("P", "P"), ("N", "N"))), 1),      # unknown letter
    (dict(nx=32, ny=32, nz=1025, bc=(("P", "P"), ("P", "P"), ("P", "P"))), 3),    # nz <= 1024 (periodic z as well)
    (dict(nx=40, ny=32, nz=32), 3),                                                # 40 = 2^3*5
    (dict(nx=32, ny=32, nz=2000), 3),
    (dict(nx=32, ny=32, nz=4, dzf=[0.5, 0.5, -0.5, 0.5], dzc=[0.5] * 5), 1),
    # periodic z: the wrap spacing dzc[0] = dzc[nz] must be single-valued
    (dict(nx=32, ny=32, nz=4, bc=(("P", "P"), ("P", "P"), ("P", "P")), dzf=[0.2, 0.3, 0.3, 0.2], dzc=[0.2, 0.25, 0.3, 0.25, 0.21]), 1),
])
def test_plan_create_rejects_bad_arguments_without_a_gpu(binding, kwargs, status):
    args = dict(nx=32, ny=32, nz=32, lx=1.0, ly=1.0, lz=1.0, bc=PP_NN, dzc=None, dzf=None)
    args.update(kwargs)
    with pytest.raises(binding.CansError) as ei:
        binding.PoissonPlan(**args)
    assert ei.value.status == status
    assert binding.last_error() != ""


@pytest.mark.parametrize("bc,stagger,status", [
    ((("N", "N"), ("P", "P"), ("D", "D")), 0, 2),      # faces along a non-periodic x: DST-I / DCT-I family, not implemented
    ((("P", "P"), ("D", "N"), ("D", "D")), 1, 2),
    ((("P", "P"), ("P", "P"), ("N", "N")), 2, 2),      # faces along z: no lower 'N' (the lower boundary face has no slot)
    ((("P", "P"), ("P", "P"), ("N", "D")), 2, 2),
    ((("P", "P"), ("P", "P"), ("D", "D")), 3, 1),
])
def test_helmholtz_plan_rejects_unsupported_staggering_without_a_gpu(binding, bc, stagger, status):
    with pytest.raises(binding.CansError) as ei:
        binding.PoissonPlan(32, 32, 32, 1.0, 1.0, 1.0, bc, stagger=stagger)
    assert ei.value.status == status


def test_host_tables_match_their_definitions():
    """plan_tables.hpp is host logic: compile it with g++ and check twiddles / eigenvalue tables against
    closed forms (cos/sin of exact rational angles; sum of eigenvalues = trace of the stencil matrix)."""
    src = r'''
#include <cstdio>
#include "plan_tables.hpp"
using namespace cans;
int main() {
    for (int n : {16, 48, 768, 1024}) {
        FftRadices f; if (!fft_lookup(n, &f)) return 1;
        if (f.r1 * f.r2 * f.r3 != n) return 2;
        auto t = make_pass_twiddles(f);
        printf("tw %d %zu %.17g %.17g\n", n, t.size() / 2, t[2 * 5], t[2 * 5 + 1]);
        for (int kind = 0; kind < 5; ++kind) {
            auto lam = make_lambda_positions(n, kind, 1.0);
            double s = 0; for (double v : lam) s += v;
            printf("lam %d %d %.17g %.17g %.17g\n", n, kind, s, lam[0], lam[1]);
        }
    }
    double re, im; unit_root(1, 8, &re, &im); printf("root %.17g %.17g\n", re, im);
    unit_root(5, 12, &re, &im); printf("root %.17g %.17g\n", re, im);
    return 0;
}'''
    with tempfile.TemporaryDirectory() as td:
        cpp = os.path.join(td, "t.cpp")
        with open(cpp, "w") as fh:
            fh.write(src)
        exe = os.path.join(td, "t")
        subprocess.check_call(["g++", "-O1", "-std=c++17", "-I",
                               os.path.join(ROOT, "paper_2001_05234_b200", "csrc"), cpp, "-o", exe])
        out = subprocess.check_output([exe], text=True).splitlines()
    roots = [l.split() for l in out if l.startswith("root")]
    assert float(roots[0][1]) == np.sqrt(0.5) and float(roots[0][2]) == -np.sqrt(0.5)
    assert abs(float(roots[1][1]) - np.cos(2 * np.pi * 5 / 12)) < 2e-16
    assert abs(float(roots[1][2]) + np.sin(2 * np.pi * 5 / 12)) < 2e-16
    seen = 0
    for l in out:
        w = l.split()
        if w[0] == "tw":
            n = int(w[1])
            # entry 5 of pass 1, k = 1: W_n^5
            assert abs(float(w[3]) - np.cos(2 * np.pi * 5 / n)) < 2e-16
            assert abs(float(w[4]) + np.sin(2 * np.pi * 5 / n)) < 2e-16
            seen += 1
        if w[0] == "lam":
            n, kind = int(w[1]), int(w[2])
            # trace of the n x n second-difference matrix with the ghost rule: PP -2n, NN -2n+2, DD -2n-2, ND / DN -2n
            trace = {0: -2.0 * n, 1: -2.0 * n + 2, 2: -2.0 * n - 2, 3: -2.0 * n, 4: -2.0 * n}[kind]
            assert abs(float(w[3]) - trace) < 1e-9 * n
            if kind < 3:
                assert float(w[4]) == (0.0 if kind != 2 else -4.0)
            else:
                # positions (0, 1) hold modes (0, n-1) for ND and (n-1, 0) for DN: -4 sin^2(pi (2q+1) / (4n))
                lo, hi = (-4 * np.sin(np.pi * (2 * q + 1) / (4 * n)) ** 2 for q in (0, n - 1))
                want = (lo, hi) if kind == 3 else (hi, lo)
                assert abs(float(w[4]) - want[0]) < 1e-15 and abs(float(w[5]) - want[1]) < 1e-14
            seen += 1
    assert seen == 24
