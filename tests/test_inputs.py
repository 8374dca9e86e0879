"""The seeded generators: determinism, ranges, the counter definition re-typed with Python ints."""
import numpy as np

import linac_inputs as gen

M64 = (1 << 64) - 1


def splitmix_py(seed, idx):
    z = (seed + 0x9E3779B97F4A7C15 * (idx + 1)) & M64
    z = ((z ^ (z >> 30)) * 0xBF58476D1CE4E5B9) & M64
    z = ((z ^ (z >> 27)) * 0x94D049BB133111EB) & M64
    return z ^ (z >> 31)


def test_uniform_matches_counter_definition_and_is_chunk_invariant():
    p, rows, cols, seed = 2147483647, 37, 53, 4
    a = gen.uniform_matrix(rows, cols, p, seed, chunk_rows=8)
    for r, c in [(0, 0), (1, 2), (36, 52), (17, 31)]:
        assert int(a[r, c]) == (splitmix_py(seed, r * cols + c) * p) >> 64
    assert np.array_equal(a, gen.uniform_matrix(rows, cols, p, seed, chunk_rows=1000))
    assert np.array_equal(a[10:20], gen.uniform_rows(10, 10, cols, p, seed))
    assert a.max() < p
    big = gen.uniform_matrix(256, 256, p, 1)
    assert abs(big.mean() / p - 0.5) < 0.01


def test_large_counter_no_overflow():
    # idx beyond 2^32 (the N = 10^5 config has 10^10 elements)
    rows, cols, p, seed = 100000, 100000, 2147483647, 7
    row = gen.uniform_rows(99999, 1, cols, p, seed)[0]
    for c in (0, 5, 99999):
        assert int(row[c]) == (splitmix_py(seed, 99999 * cols + c) * p) >> 64


def test_sparse_dependent_rows_recipe():
    p, rows, cols = 2147483647, 200, 96
    full = gen.sparse_dependent_rows(0, rows, rows, cols, p, 7, 8)
    assert np.array_equal(full[60:130], gen.sparse_dependent_rows(60, 70, rows, cols, p, 7, 8))
    dep, src, alpha = gen.sparse_dependent_plan(rows, p, 8)
    assert list(dep) == [49, 99, 149, 199] and (src % 50 != 49).all() and (alpha >= 1).all()
    for d, i in enumerate(dep):
        comb = sum(full[src[d, t]].astype(object) * int(alpha[d, t]) for t in range(3)) % p
        assert (comb == full[i]).all()
    indep = full[np.arange(rows) % 50 != 49]
    assert 0.86 < (indep == 0).mean() < 0.94


def test_normal_system():
    a, b = gen.shifted_normal_system(300, 8, 5, 6)
    g = a - np.diag(np.diag(a)) 
    assert abs(g.mean()) < 0.02 and abs(g.std() - 1.0) < 0.02 and abs(b.std() - 1.0) < 0.05
    assert np.allclose(np.diag(a).mean(), 4 * np.sqrt(300), atol=0.3)
    a2, _ = gen.shifted_normal_system(300, 8, 5, 6)
    assert np.array_equal(a, a2)


def test_torch_generators_match_numpy_bit_for_bit():
    """gen_torch (used to build config c5 on the device) against gen, on the CPU."""
    import torch
    from linac_inputs import gen_torch
    p = 2147483647
    u = gen_torch.uniform_rows(5, 7, 33, p, seed=4, device="cpu").numpy().view(np.uint32)
    assert np.array_equal(u, gen.uniform_rows(5, 7, 33, p, seed=4))
    rows = cols = 230
    want = gen.sparse_dependent_rows(0, rows, rows, cols, p, seed=7, seed_dep=8)
    got = gen_torch.sparse_dependent_rows(0, rows, rows, cols, p, seed=7, seed_dep=8).numpy().view(np.uint32)
    assert np.array_equal(got, want)
    part = gen_torch.sparse_dependent_rows(90, 70, rows, cols, p, seed=7, seed_dep=8).numpy().view(np.uint32)
    assert np.array_equal(part, want[90:160])
    dst = torch.zeros((rows, cols), dtype=torch.int32)
    gen_torch.fill_c5(dst, dict(p=p, seed=7, seed_dep=8, period=50, terms=3), block_rows=64)
    assert np.array_equal(dst.numpy().view(np.uint32), want)
    assert 0.05 < (want != 0).mean() < 0.2 and (want[49] != 0).mean() > 0.2      # sparse rows, denser combinations
