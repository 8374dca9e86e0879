"""Pins for the F_p oracle (oracle/linac_oracle.c) against things other than itself.

Every check here is a definition, a brute force over a tiny field, a closed form, Python big-int
arithmetic or an independent library (sympy GF(p)); see SURVEY.md section 8(c) "What pins each part".
"""
import os

import numpy as np
import pytest

import helpers as H
import linac_inputs as gen

P31 = 2147483647      # 2^31 - 1   (configs c1, c3, c5)
P29 = 2147483629      # config c2
SMALL_PRIMES = [2, 3, 5, 7, 11, 13, 251, 65521]


# ---------------------------------------------------------------- modular arithmetic
@pytest.mark.parametrize("p", SMALL_PRIMES)
def test_inverse_exhaustive_small_primes(oracle, p):
    for a in range(1, p) if p < 70000 else []:
        inv = oracle.inv_modp(a, p)
        assert 0 < inv < p and a * inv % p == 1


@pytest.mark.parametrize("p", [P31, P29])
def test_inverse_random_big_primes_vs_python_and_fermat(oracle, p):
    rng = np.random.default_rng(11)
    for a in [1, 2, p - 1, p - 2, (p + 1) // 2] + [int(x) for x in rng.integers(1, p, size=20000)]:
        inv = oracle.inv_modp(a, p)
        assert inv == pow(a, -1, p)                  # Python big-int inverse
        assert inv == oracle.pow_modp(a, p - 2, p)   # Fermat route agrees with Euclid route


def test_pow_vs_python(oracle):
    rng = np.random.default_rng(12)
    for p in [7, 65521, P29, P31]:
        for _ in range(2000):
            a, e = int(rng.integers(0, p)), int(rng.integers(0, 2**62))
            assert oracle.pow_modp(a, e, p) == pow(a, e, p)


def test_matmul_vs_bigint(oracle):
    rng = np.random.default_rng(13)
    for p in [2, 7, P29, P31]:
        a = rng.integers(0, p, size=(9, 13), dtype=np.uint64).astype(np.uint32)
        b = rng.integers(0, p, size=(13, 5), dtype=np.uint64).astype(np.uint32)
        assert np.array_equal(oracle.matmul_modp(a, b, p), H.matmul_big(a, b, p))
    # worst case operands p-1 (catches 64-bit overflow in an accumulate-then-reduce mistake)
    a = np.full((3, 300), P31 - 1, dtype=np.uint32)
    b = np.full((300, 2), P31 - 1, dtype=np.uint32)
    assert np.array_equal(oracle.matmul_modp(a, b, P31), H.matmul_big(a, b, P31))
    assert np.array_equal(oracle.matmul_modp(a, b, P31, nthreads=4), H.matmul_big(a, b, P31))


# ---------------------------------------------------------------- hand-worked fixture
def _read_fixture(path):
    out, lines = {}, [l.strip() for l in open(path) if l.strip() and not l.startswith("#")]
    i = 0
    while i < len(lines):
        tok = lines[i].split()
        if tok[0] in ("p", "rank"):
            out[tok[0]] = int(tok[1]); i += 1
        elif tok[0] == "pivots":
            out["pivots"] = [int(x) for x in tok[1:]]; i += 1
        else:
            r, c = int(tok[1]), int(tok[2])
            out[tok[0]] = np.array([[int(x) for x in lines[i + 1 + k].split()] for k in range(r)],
                                   dtype=np.uint32).reshape(r, c)
            i += 1 + r
    return out


def test_handworked_f7_example(oracle):
    fx = _read_fixture(os.path.join(os.path.dirname(__file__), "golden", "rref_f7_handworked.txt"))
    r, rank, piv = oracle.rref_modp(fx["A"], fx["p"])
    assert rank == fx["rank"] and list(piv) == fx["pivots"]
    assert np.array_equal(r, fx["R"])
    k = oracle.nullspace_modp(r, fx["p"], rank, piv)
    assert np.array_equal(k, fx["K"])


# ---------------------------------------------------------------- brute force on tiny fields
@pytest.mark.parametrize("p,shape", [(2, (5, 6)), (2, (6, 4)), (3, (4, 5)), (3, (5, 3)), (5, (3, 4)), (5, (4, 3)),
                                      (2, (6, 6)), (3, (4, 4))])
def test_rref_structure_rowspace_and_rank_bruteforce(oracle, p, shape):
    rng = np.random.default_rng(100 + p * 31 + shape[0] * 7 + shape[1])
    for trial in range(12):
        a = rng.integers(0, p, size=shape).astype(np.uint32)
        if trial % 3 == 0 and shape[0] > 2:          # force rank deficiency
            a[-1] = (a[0].astype(np.int64) + 2 * a[1].astype(np.int64)) % p
        if trial % 4 == 1:
            a[:, shape[1] // 2] = 0                  # a zero column (free column in the middle)
        r, rank, piv = oracle.rref_modp(a, p)
        pivots = H.is_rref(r, p)
        assert pivots is not None, (a, r)
        assert pivots == list(piv) and rank == len(pivots)
        assert H.row_space_set(a, p) == H.row_space_set(r, p)         # row-equivalent
        assert H.kernel_count(a, p) == p ** (shape[1] - rank)          # brute-force rank
        k = oracle.nullspace_modp(r, p, rank, piv)
        assert k.shape == (shape[1], shape[1] - rank)
        assert not H.matmul_big(a, k, p).any() if k.size else True     # A.K = 0 (eq. 9)


@pytest.mark.parametrize("p", [2, 3, 5, 7, 13])
@pytest.mark.parametrize("n", [1, 2, 3, 4, 5, 6])
def test_det_vs_leibniz(oracle, p, n):
    rng = np.random.default_rng(200 + p + 17 * n)
    for trial in range(6 if n < 6 else 3):
        a = rng.integers(0, p, size=(n, n)).astype(np.uint32)
        if trial == 1 and n > 1:
            a[n - 1] = a[0]
        d = oracle.det_modp(a, p)
        assert d == H.det_leibniz(a, p)
        _, rank, _ = oracle.rref_modp(a, p)
        assert (d != 0) == (rank == n)


# ---------------------------------------------------------------- uniqueness / invariants
@pytest.mark.parametrize("p", [5, 251, P29, P31])
def test_pivot_rule_independence_idempotence_invariance(oracle, p):
    rng = np.random.default_rng(300 + p % 1000)
    for shape in [(7, 11), (11, 7), (9, 9), (1, 6), (6, 1)]:
        a = rng.integers(0, p, size=shape, dtype=np.uint64).astype(np.uint32)
        if shape[0] > 3:
            a[3] = H.matmul_big(rng.integers(0, p, size=(1, 3), dtype=np.uint64).astype(np.uint32), a[:3], p)[0]
        r0, rank0, piv0 = oracle.rref_modp(a, p, oracle.PIVOT_FIRST)
        for rule in (oracle.PIVOT_LAST, oracle.PIVOT_MAX):              # reading Q1: RREF is unique
            r1, rank1, piv1 = oracle.rref_modp(a, p, rule)
            assert rank1 == rank0 and np.array_equal(piv1, piv0) and np.array_equal(r1, r0)
        r2, rank2, piv2 = oracle.rref_modp(r0, p)                       # idempotent
        assert rank2 == rank0 and np.array_equal(r2, r0) and np.array_equal(piv2, piv0)
        ga = H.random_row_ops(a, p, rng)                                # RREF(G.A) = RREF(A)
        r3, rank3, _ = oracle.rref_modp(ga, p)
        assert rank3 == rank0 and np.array_equal(r3, r0)
        assert H.is_rref(r0, p) == list(piv0)
        r4, _, _ = oracle.rref_modp(a, p, nthreads=4)                   # threaded build is bit-identical
        assert np.array_equal(r4, r0)


def test_permutation_matrix_reduces_to_identity(oracle):
    rng = np.random.default_rng(5)
    n = 23
    perm = rng.permutation(n)
    pm = np.zeros((n, n), dtype=np.uint32)
    pm[np.arange(n), perm] = 1
    r, rank, piv = oracle.rref_modp(pm, P31)
    assert rank == n and np.array_equal(r, np.eye(n, dtype=np.uint32)) and list(piv) == list(range(n))


def test_entries_ge_p_are_reduced_first(oracle):
    """Reading Q5: inputs >= p are taken mod p."""
    p = 7
    a = np.array([[9, 14, 8], [7, 15, 3]], dtype=np.uint32)
    r, rank, piv = oracle.rref_modp(a, p)
    r2, rank2, piv2 = oracle.rref_modp(a % p, p)
    assert np.array_equal(r, r2) and rank == rank2 == 2


def test_padding_columns_untouched(oracle):
    """Reading Q8: columns cols..ld-1 are never read as data and never written."""
    import ctypes as C
    p, rows, cols, ld = P29, 6, 5, 8
    rng = np.random.default_rng(9)
    buf = np.full((rows, ld), 0xDEADBEEF, dtype=np.uint32)
    a = rng.integers(0, p, size=(rows, cols), dtype=np.uint64).astype(np.uint32)
    buf[:, :cols] = a
    rank = C.c_int64()
    piv = np.zeros(5, dtype=np.int32)
    rc = oracle.lib().oracle_rref_modp(buf.ctypes.data_as(C.POINTER(C.c_uint32)), rows, cols, ld, p, 0, 1,
                                       C.byref(rank), piv.ctypes.data_as(C.POINTER(C.c_int32)))
    assert rc == 0
    assert (buf[:, cols:] == 0xDEADBEEF).all()
    r, rk, _ = oracle.rref_modp(a, p)
    assert np.array_equal(buf[:, :cols], r) and rank.value == rk


@pytest.mark.parametrize("shape", [(0, 5), (5, 0), (1, 1), (1, 9), (9, 1), (40, 3), (3, 40)])
def test_degenerate_shapes(oracle, shape):
    """Reading Q17."""
    rng = np.random.default_rng(17)
    a = rng.integers(0, P31, size=shape, dtype=np.uint64).astype(np.uint32)
    r, rank, piv = oracle.rref_modp(a, P31)
    assert r.shape == shape and rank <= min(shape)
    if min(shape) > 0:
        assert H.is_rref(r, P31) == list(piv)
    z, rank0, _ = oracle.rref_modp(np.zeros(shape, dtype=np.uint32), P31)
    assert rank0 == 0 and not z.any()


# ---------------------------------------------------------------- product rank, RREF(B.C) = RREF(C)
@pytest.mark.parametrize("p", [P29, P31, 13])
def test_product_of_factors_has_rank_r_and_rref_of_right_factor(oracle, p):
    m, r, n = 40, 17, 45
    a, b, c = gen.lowrank_factors(m, r, n, p, seed_b=2, seed_c=3)
    assert np.array_equal(a, H.matmul_big(b, c, p))                    # the generator's own product is exact
    ra, rank_a, piv_a = oracle.rref_modp(a, p)
    rb, rank_b, _ = oracle.rref_modp(b, p)
    rc, rank_c, piv_c = oracle.rref_modp(c, p)
    if rank_b == r:                                                    # B has full column rank (w.h.p.)
        assert rank_a == rank_c
        assert np.array_equal(ra[:rank_c], rc[:rank_c]) and not ra[rank_c:].any()
        assert np.array_equal(piv_a, piv_c)
    if p > 1000:
        assert rank_a == r                                             # exact rank r w.h.p. for big p


# ---------------------------------------------------------------- Vandermonde closed forms
@pytest.mark.parametrize("p", [P31, P29, 251])
def test_vandermonde_full_rank_det_and_interpolation(oracle, p):
    rng = np.random.default_rng(77)
    n = 12
    x = [int(v) for v in rng.choice(min(p, 10**6), size=n, replace=False)]
    v = np.array([[pow(xi, k, p) for k in range(n)] for xi in x], dtype=np.uint32)
    r, rank, piv = oracle.rref_modp(v, p)
    assert rank == n and np.array_equal(r, np.eye(n, dtype=np.uint32))
    det = 1
    for i in range(n):
        for j in range(i + 1, n):
            det = det * (x[j] - x[i]) % p
    assert oracle.det_modp(v, p) == det                                # prod_{i<j} (x_j - x_i)
    q = [int(c) for c in rng.integers(0, p, size=n)]                   # polynomial coefficients
    y = np.array([[sum(q[k] * pow(xi, k, p) for k in range(n)) % p] for xi in x], dtype=np.uint32)
    aug, rank2, piv2 = oracle.rref_modp(np.hstack([v, y]), p)          # (V | y) -> (I | q)  (eq. 12)
    assert rank2 == n and list(piv2) == list(range(n))
    assert [int(t) for t in aug[:, n]] == q


@pytest.mark.parametrize("p", [P31, 65521])
def test_inverse_via_augmented_identity(oracle, p):
    n = 15
    a = gen.uniform_matrix(n, n, p, seed=21)
    aug = np.hstack([a, np.eye(n, dtype=np.uint32)])
    r, rank, _ = oracle.rref_modp(aug, p)
    assert rank == n and np.array_equal(r[:, :n], np.eye(n, dtype=np.uint32))
    assert np.array_equal(H.matmul_big(a, r[:, n:], p), np.eye(n, dtype=np.uint32))


# ---------------------------------------------------------------- independent library (sympy GF(p))
@pytest.mark.parametrize("p,shape", [(P31, (24, 30)), (P29, (30, 24)), (7, (20, 26)), (P31, (40, 40))])
def test_rref_vs_sympy_gf(oracle, p, shape):
    from sympy import GF
    from sympy.polys.matrices import DomainMatrix
    rng = np.random.default_rng(400 + shape[0])
    a = rng.integers(0, p, size=shape, dtype=np.uint64).astype(np.uint32)
    a[5] = H.matmul_big(rng.integers(0, p, size=(1, 4), dtype=np.uint64).astype(np.uint32), a[:4], p)[0]
    a[:, 3] = 0
    dom = GF(p, symmetric=False)
    dm = DomainMatrix([[dom(int(v)) for v in row] for row in a], shape, dom)
    rr, pivots = dm.rref()
    ref = np.array([[int(v) % p for v in row] for row in rr.to_list()], dtype=np.uint32)
    r, rank, piv = oracle.rref_modp(a, p)
    assert list(piv) == list(pivots) and rank == len(pivots)
    assert np.array_equal(r, ref)


# ---------------------------------------------------------------- null space
@pytest.mark.parametrize("p", [P29, 5])
def test_nullspace_identity_and_structure(oracle, p):
    a, _, _ = gen.lowrank_factors(30, 11, 37, p, seed_b=5, seed_c=6)
    r, rank, piv = oracle.rref_modp(a, p)
    k = oracle.nullspace_modp(r, p, rank, piv)
    assert k.shape == (37, 37 - rank)
    assert not H.matmul_big(a, k, p).any()                             # A.K = 0 with the ORIGINAL A (eq. 9)
    assert not oracle.matmul_modp(a, k, p).any()
    free = [c for c in range(37) if c not in set(int(x) for x in piv)]
    minus_identity = (np.eye(len(free), dtype=np.int64) * (p - 1)).astype(np.uint32)
    assert np.array_equal(k[free, :], minus_identity)                  # "minus the identity"
    for kk, ck in enumerate(piv):
        assert np.array_equal(k[ck, :], r[kk, free])
    # columns of K are independent and there are cols - rank of them
    _, rank_k, _ = oracle.rref_modp(np.ascontiguousarray(k.T), p)
    assert rank_k == 37 - rank


def test_sparse_dependent_generator_rank(oracle):
    """Config c5's recipe at a size the oracle does in no time: rank = rows - rows//period."""
    rows = cols = 300
    a = gen.sparse_dependent_rows(0, rows, rows, cols, P31, seed=7, seed_dep=8)
    _, rank, piv = oracle.rref_modp(a, P31)
    assert rank == rows - rows // 50
    assert 0.85 < (a[np.arange(rows) % 50 != 49] == 0).mean() < 0.95


# ------------------------------------------------------------------ solve_modp
def test_solve_modp_against_brute_force_and_plain_products(oracle):
    import itertools
    rng = np.random.default_rng(11)
    # (1) tiny fields: consistency must equal "some x in F_p^cols solves it" by enumeration; a returned x must solve it
    for p, rows, cols in [(2, 4, 4), (3, 3, 4), (3, 5, 3), (5, 3, 3), (2, 6, 5)]:
        for trial in range(12):
            a = rng.integers(0, p, size=(rows, cols)).astype(np.uint32)
            if trial % 3 == 0:
                a[:, -1] = a[:, 0]                                   # force rank deficiency
            b = rng.integers(0, p, size=(rows, 3)).astype(np.uint32)
            cons, x = oracle.solve_modp(a, b, p)
            allx = np.array(list(itertools.product(range(p), repeat=cols)), dtype=np.int64).T      # cols x p^cols
            prod = (a.astype(np.int64) @ allx) % p
            for j in range(3):
                solvable = bool((prod == b[:, j:j + 1].astype(np.int64)).all(axis=0).any())
                assert bool(cons[j]) == solvable
                if solvable:
                    assert np.array_equal((a.astype(np.int64) @ x[:, j].astype(np.int64)) % p, b[:, j].astype(np.int64))
                else:
                    assert not x[:, j].any()
    # (2) a big prime: manufactured solutions b = A.y are consistent and A.x = b (x need not equal y when A is singular);
    #     full-rank square A gives x = y exactly (eq. 12)
    p = 2147483629
    a = gen.uniform_matrix(40, 40, p, seed=5)
    y = gen.uniform_matrix(40, 4, p, seed=6)
    b = oracle.matmul_modp(a, y, p)
    cons, x = oracle.solve_modp(a, b, p)
    assert cons.all() and np.array_equal(x, y)
    a2, _, _ = gen.lowrank_factors(30, 12, 45, p, seed_b=7, seed_c=8)
    y2 = gen.uniform_matrix(45, 2, p, seed=9)
    b2 = np.hstack([oracle.matmul_modp(a2, y2, p), gen.uniform_matrix(30, 1, p, seed=10)])       # last one: random -> inconsistent w.h.p.
    cons2, x2 = oracle.solve_modp(a2, b2, p)
    assert list(cons2) == [True, True, False]
    assert np.array_equal(oracle.matmul_modp(a2, x2[:, :2], p), b2[:, :2])
    # free variables are zero: x is supported on the pivot columns of A
    _, rank, piv = oracle.rref_modp(a2, p)
    free = np.setdiff1d(np.arange(45), piv[:rank])
    assert not x2[free].any()


# ------------------------------------------------------------------ rank_factor_modp (eq. 7)
def test_rank_factor_modp_pins(oracle):
    import itertools
    # (1) worked by hand over F_7: row 2 = 2 x row 1; (1,0,1) - (1,2,3) = (0,5,5) -> x 3 = (0,1,1); (1,2,3) - 2(0,1,1) = (1,0,1)
    a = np.array([[1, 2, 3], [2, 4, 6], [1, 0, 1]], dtype=np.uint32)
    c, r, j = oracle.rank_factor_modp(a, 7)
    assert list(j) == [0, 1]
    assert np.array_equal(r, np.array([[1, 0, 1], [0, 1, 1]], dtype=np.uint32))
    assert np.array_equal(c, np.array([[1, 2], [2, 4], [1, 0]], dtype=np.uint32))
    # (2) tiny fields: C.R = A with plain integers, and C has full column rank by enumeration of all non-zero x
    rng = np.random.default_rng(13)
    for p, rows, cols in [(2, 5, 6), (3, 4, 5), (5, 4, 3), (2, 6, 4), (3, 5, 5)]:
        for trial in range(10):
            a = rng.integers(0, p, size=(rows, cols)).astype(np.uint32)
            if trial % 2 == 0:
                a[:, 1] = a[:, 0]
                a[-1] = (a[0] + a[1]) % p
            c, r, j = oracle.rank_factor_modp(a, p)
            k = len(j)
            assert c.shape == (rows, k) and r.shape == (k, cols)
            assert np.array_equal((c.astype(np.int64) @ r.astype(np.int64)) % p, a.astype(np.int64))
            if k:
                allx = np.array(list(itertools.product(range(p), repeat=k)), dtype=np.int64).T[:, 1:]   # non-zero x
                assert ((c.astype(np.int64) @ allx) % p != 0).any(axis=0).all()
    # (3) a big prime, entries >= p on input, rank-deficient by construction: C.R = A mod p by the (big-int pinned) product
    p = 2147483629
    a, _, _ = gen.lowrank_factors(37, 9, 52, p, seed_b=21, seed_c=22)
    a = a.copy()
    a[3, 5] += p                                                    # still < 2^32; the same residue
    c, r, j = oracle.rank_factor_modp(a, p)
    assert len(j) == 9 and c.max() < p
    assert np.array_equal(oracle.matmul_modp(c, r, p), a % np.uint32(p))
    # zero matrix and empty shapes: rank 0, empty factors
    c, r, j = oracle.rank_factor_modp(np.zeros((3, 4), dtype=np.uint32), 7)
    assert c.shape == (3, 0) and r.shape == (0, 4) and len(j) == 0


# ------------------------------------------------------------------ load_matrix_modp
def test_load_matrix_modp_pins(oracle):
    rng = np.random.default_rng(12)
    p = 2147483629
    bases = gen.uniform_matrix(9, 6, p, seed=13)
    lind = rng.integers(-1, 6, size=(11, 5)).astype(np.int32)              # -1 = no factor
    a = oracle.load_matrix_modp(bases, lind, p)
    for r in range(9):                                                      # Python big integers, no modular shortcuts
        for c in range(11):
            prod = 1
            for t in range(5):
                if lind[c, t] >= 0:
                    prod *= int(bases[r, lind[c, t]])
            assert int(a[r, c]) == prod % p
    # closed form: columns x^0 .. x^7 of a Vandermonde matrix (index 0 repeated c times, padded with -1)
    x = gen.uniform_matrix(20, 1, p, seed=14)
    lv = np.full((8, 7), -1, dtype=np.int32)
    for c in range(8):
        lv[c, :c] = 0
    v = oracle.load_matrix_modp(x, lv, p)
    assert np.array_equal(v, np.array([[pow(int(xi), c, p) for c in range(8)] for xi in x[:, 0]], dtype=np.uint32))
    # d = 1 is a gather of columns; d = 0 the all-ones matrix; entries >= p are reduced
    g = oracle.load_matrix_modp(bases, np.array([[3], [0], [5]], dtype=np.int32), p)
    assert np.array_equal(g, bases[:, [3, 0, 5]])
    assert (oracle.load_matrix_modp(bases, np.zeros((4, 0), dtype=np.int32), p) == 1).all()
    big = np.array([[p + 5, 7]], dtype=np.uint32)
    assert oracle.load_matrix_modp(big, np.array([[0, 1]], dtype=np.int32), p)[0, 0] == 35
