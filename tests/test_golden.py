"""Exact-integer fixtures (tests/golden/, written by tests/golden/make_fixtures.py from textbook
identities in pure integer arithmetic): the symmetric Pascal matrix (Cholesky factor = upper Pascal
matrix, inverse = signed Pascal matrix) and the min(i,j) matrix (factor = upper triangle of ones).
The oracle must reproduce them (CPU test), and so must the CUDA path through the C ABI (GPU test).
All entries are small integers, so every product is exactly representable: the tolerances below only
leave room for the square roots and divisions of the factorisation.
"""
import os

import numpy as np
import pytest
import torch

import oracle
from paper_2502_02460_b200 import workloads as wl

GOLDEN = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden")


def load(name):
    out, key, rows_left = {}, None, 0
    with open(os.path.join(GOLDEN, name + ".txt")) as f:
        for line in f:
            line = line.strip()
            if not line or line.startswith("#"):
                continue
            tok = line.split()
            if rows_left == 0:
                if tok[0] == "N":
                    out["N"] = int(tok[1])
                else:
                    key, rows_left = tok[0], int(tok[1])
                    out[key] = []
            else:
                out[key].append([float(x) for x in tok])
                rows_left -= 1
    return {k: (np.array(v, dtype=np.float64) if k != "N" else v) for k, v in out.items()}


def rel(a, b):
    return np.linalg.norm(a - b) / np.linalg.norm(b)


@pytest.mark.parametrize("name", ["pascal8", "minij12"])
def test_fixture_is_self_consistent(name):
    g = load(name)
    assert np.array_equal(g["U"].T @ g["U"], g["S"])
    assert np.array_equal(g["U"] @ g["V"], np.eye(g["N"]))
    assert np.array_equal(g["V"].T @ g["H"] @ g["V"], g["Ht"])
    assert np.array_equal(g["V"] @ g["Ct"], g["C"])


@pytest.mark.parametrize("name", ["pascal8", "minij12"])
def test_oracle_reproduces_the_fixture(name):
    g = load(name)
    U = oracle.cholesky(g["S"])
    assert rel(U, g["U"]) <= 1e-13 and np.count_nonzero(np.tril(U, -1)) == 0
    V = oracle.invert_upper(g["U"])                 # each stage on the exact input of the fixture
    assert rel(V, g["V"]) <= 1e-14
    Ht = oracle.to_standard(g["H"], g["V"])
    assert np.array_equal(Ht, g["Ht"])              # integer inputs: exact, both triangles
    C = oracle.backtransform(g["V"], g["Ct"])
    assert np.array_equal(C, g["C"])
    # chained: the oracle's own factor goes on through the later stages
    Vc = oracle.invert_upper(U)
    assert rel(oracle.to_standard(g["H"], Vc), g["Ht"]) <= 1e-10     # cond(pascal8) ~ 2e7 amplifies the factor's rounding
    # complex128 entry points on the same (real) data
    Uz = oracle.cholesky(g["S"].astype(np.complex128))
    assert rel(Uz, g["U"]) <= 1e-13


@pytest.mark.gpu
@pytest.mark.parametrize("cplx", [False, True])
@pytest.mark.parametrize("name", ["pascal8", "minij12"])
def test_cuda_path_reproduces_the_fixture(name, cplx):
    from paper_2502_02460_b200 import gs
    g = load(name)
    N = g["N"]
    dt = torch.complex128 if cplx else torch.float64

    def dev(a):
        return wl.to_colmajor(torch.from_numpy(a).to(dt).cuda())

    plan = gs.Plan(N, 3, dtype=gs.GS_COMPLEX128 if cplx else gs.GS_REAL64)
    U = dev(g["S"])
    plan.cholesky(U)
    assert plan.last_info() == 0
    assert rel(U.cpu().numpy(), g["U"]) <= 1e-13
    assert torch.count_nonzero(torch.tril(U, -1)) == 0
    # each stage on the exact input of the fixture
    Uex, V = dev(g["U"]), wl.colmajor_empty(N, N, dtype=dt, device="cuda")
    plan.invert_triangular(Uex, V)
    assert rel(V.cpu().numpy(), g["V"]) <= 1e-14
    Ht = wl.colmajor_zeros(N, N, dtype=dt, device="cuda")
    plan.to_standard(dev(g["H"]), dev(g["V"]), Ht)
    plan.last_info()
    assert np.array_equal(np.triu(Ht.cpu().numpy()), np.triu(g["Ht"]).astype(Ht.cpu().numpy().dtype))   # integer data: exact
    C = wl.colmajor_empty(N, 3, dtype=dt, device="cuda")
    plan.backtransform(dev(g["V"]), dev(g["Ct"]), C)
    plan.last_info()
    assert np.array_equal(C.cpu().numpy(), g["C"].astype(C.cpu().numpy().dtype))
    plan.close()
