"""The C oracle rebuilt with -fsanitize=address,undefined and exercised on small lattices in a child process
(SURVEY.md sec. 5): out-of-bounds indexing or undefined behaviour in the checker itself would abort the child."""
import os
import subprocess
import sys
import tempfile

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

CHILD = r"""
import ctypes, os, sys
import numpy as np
sys.path.insert(0, %(root)r)
import oracle, lattice_inputs as li
oracle._LIB = %(lib)r            # load the sanitised build instead of the regular one
oracle.build = lambda force=False: %(lib)r
for dims, bc in [((4, 4, 4, 4), (1, 1, 1, -1)), ((2, 4, 6, 8), tuple(np.exp(1j * np.array([0.3, -1.1, 2.0, 3.14]))))]:
    U = li.random_su3_links(dims, seed=3)
    psi = li.gaussian_spinor(dims, seed=4)
    oracle.dslash_full(U, psi, dims, bc)
    oracle.dslash_full(U.astype(np.complex64), psi.astype(np.complex64), dims, bc)
    for p in (0, 1):
        oracle.dslash_eo(U, psi, dims, bc, p)
    for eo in (0, 1):
        oracle.apply_M(U, psi, dims, bc, 0.13, eo)
        oracle.apply_M_tm(U, psi, dims, bc, 0.13, 0.2, eo)
    X, Y, Z, T = dims
    corners = [[0, 0, 0, 0], [X - 1, Y - 1, Z - 1, T - 1], [0, Y - 1, 0, T - 1], [X - 2, 0, Z - 1, 1]]
    oracle.dslash_sites(U, psi, dims, bc, corners)
    oracle.apply_M_sites(U, psi, dims, bc, 0.13, 1, [c for c in corners if sum(c) %% 2 == 0])
print("sanitised oracle ok")
"""


def test_oracle_under_asan_and_ubsan():
    libasan = subprocess.run(["gcc", "-print-file-name=libasan.so"], capture_output=True, text=True).stdout.strip()
    if not os.path.isabs(libasan) or not os.path.exists(libasan):
        pytest.skip("libasan not available")
    with tempfile.TemporaryDirectory() as tmp:
        lib = os.path.join(tmp, "liboracle_san.so")
        subprocess.check_call(["gcc", "-O1", "-g", "-std=c99", "-fopenmp", "-fPIC", "-shared", "-fsanitize=address,undefined",
                               "-fno-sanitize-recover=all", "-o", lib, os.path.join(ROOT, "oracle", "wilson_oracle.c"), "-lm"])
        env = dict(os.environ, LD_PRELOAD=libasan, ASAN_OPTIONS="detect_leaks=0", OMP_NUM_THREADS="2")
        r = subprocess.run([sys.executable, "-c", CHILD % {"root": ROOT, "lib": lib}], env=env, capture_output=True, text=True,
                           timeout=600)
        assert r.returncode == 0 and "sanitised oracle ok" in r.stdout, (r.stdout[-300:], r.stderr[-2000:])
