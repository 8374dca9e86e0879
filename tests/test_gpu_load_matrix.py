"""linac_load_matrix_u32 against the oracle's written-out
definition, and the paper's workflow on top of it (eq. 6): build the matrix of monomials on the device, append
f(X) and solve for the coefficients with linac_solve_u32."""
import numpy as np
import pytest
import torch

import linac_inputs as gen
from gpu_util import require_cuda, from_device

pytestmark = pytest.mark.gpu
P31 = 2147483647
P29 = 2147483629


@pytest.fixture(autouse=True, scope="module")
def _cuda():
    require_cuda()


@pytest.mark.parametrize("n_rows,n_basis,n_cols,d,p", [(1, 1, 1, 1, P31), (300, 7, 1000, 6, P31), (257, 40, 513, 3, P29),
                                                       (64, 5, 300, 0, P31), (50, 3, 260, 12, 7), (33, 2, 70, 4, 2)])
def test_matches_the_definition(oracle, n_rows, n_basis, n_cols, d, p):
    import paper_2605_25863_b200 as L
    rng = np.random.default_rng(n_rows + n_cols)
    bases = rng.integers(0, 2**32, size=(n_rows, n_basis), dtype=np.uint64).astype(np.uint32)     # includes entries >= p
    lind = rng.integers(-1, n_basis + 1, size=(n_cols, d)).astype(np.int32)                        # -1 and n_basis: no factor
    want = oracle.load_matrix_modp(bases, lind, p)
    got = L.load_matrix_u32(torch.from_numpy(bases.view(np.int32)).cuda(), torch.from_numpy(lind).cuda(), p)
    assert np.array_equal(from_device(got), want)
    # into a padded output: the padding must stay untouched
    out = torch.full((n_rows, n_cols + 3), -559038737, dtype=torch.int32, device="cuda")
    L.load_matrix_u32(torch.from_numpy(bases.view(np.int32)).cuda(), torch.from_numpy(lind).cuda(), p, out=out[:, :n_cols])
    o = from_device(out)
    assert np.array_equal(o[:, :n_cols], want) and (o[:, n_cols:] == np.uint32(0xDEADBEEF)).all()


def test_interpolation_workflow_recovers_the_coefficients(oracle):
    """Eq. 6 of the paper: all monomials of degree <= 5 in three variables (56 of them), sampled at 80 points; the
    right-hand side is a known polynomial, so the solve must return its coefficients exactly."""
    import itertools
    import paper_2605_25863_b200 as L
    p = P31
    nvar, deg, npts = 3, 5, 80
    monos = [m for m in itertools.product(range(deg + 1), repeat=nvar) if sum(m) <= deg]
    lind = np.full((len(monos), deg), -1, dtype=np.int32)
    for c, m in enumerate(monos):
        idx = [v for v in range(nvar) for _ in range(m[v])]
        lind[c, :len(idx)] = idx
    x = gen.uniform_matrix(npts, nvar, p, seed=51)
    coeff = gen.uniform_matrix(len(monos), 1, p, seed=52)
    a_dev = L.load_matrix_u32(torch.from_numpy(x.view(np.int32)).cuda(), torch.from_numpy(lind).cuda(), p)
    a_host = from_device(a_dev)
    assert np.array_equal(a_host, oracle.load_matrix_modp(x, lind, p))
    f = oracle.matmul_modp(a_host, coeff, p)                                   # f(X_r) = sum_c coeff_c m_c(X_r)
    aug = torch.cat([a_dev, torch.from_numpy(f.view(np.int32)).cuda()], dim=1).contiguous()
    rank_a, piv, cons, sol = L.solve_u32(aug, len(monos), p)
    assert rank_a == len(monos) and bool(cons[0])
    assert np.array_equal(from_device(sol), coeff)
