"""Config c5 at FULL size (10^5 x 10^5 over F_{2^31-1}, 90% zeros, every 50th row a combination of three others):
the oracle cannot finish this, so correctness is certified by properties that hold at any size
("beyond-oracle certificates"; BASELINE.json north_star: the null-space identity and
re-reduction of random row subsets).  The matrix is generated on the device (linac_inputs.gen_torch, bit-identical
to the numpy generator) and regenerated block by block for the checks, because the call works in place.

  (i)   structure: R[:r, pivots] = I, rows >= r are zero, entries canonical            (device scan)
  (ii)  row space: for random v, A.v = A[:, pivots].(R.v) for EVERY row of A           (Freivalds, 3 vectors)
  (iii) exact:     sampled rows a of A satisfy a = a[pivots].R on sampled columns      (CPU oracle matmul)
  (iv)  A.K = 0:   sampled rows exactly on the CPU; every row through A.(K.w) = 0      (eq. 9)
  (v)   rank = rows - rows/50 = 98 000, the rank the generator fixes (w.h.p. the pivots are 0..r-1)
The same generator at an oracle-sized shape is compared byte for byte in test_gpu_fp.py.
"""
import numpy as np
import pytest
import torch

import linac_inputs as gen
from linac_inputs import gen_torch

pytestmark = pytest.mark.gpu


def matvec_mod_p(blk: torch.Tensor, x: torch.Tensor, p: int) -> torch.Tensor:
    """(blk @ x) mod p, blk int64 [n, c] with entries < 2^31, x int64 [c] or [c, k]; plain torch integer ops."""
    if x.dim() == 1:
        return (blk * x[None, :] % p).sum(dim=1) % p
    return torch.stack([(blk * x[None, :, j] % p).sum(dim=1) % p for j in range(x.shape[1])], dim=1)


@pytest.mark.timeout(1500)
def test_config_c5_certificates(oracle):
    import paper_2605_25863_b200 as L
    if not torch.cuda.is_available():
        raise RuntimeError("GPU test selected but no CUDA device is visible (there is no CPU fallback)")
    free_b, _ = torch.cuda.mem_get_info()
    cfg = gen.CONFIGS["c5"]
    n, p = cfg["rows"], cfg["p"]
    if free_b < 60e9:
        pytest.skip("config c5 needs about 60 GB of device memory")
    dev = torch.device("cuda")
    blk_rows = 256
    plan = gen.sparse_dependent_plan(n, p, cfg["seed_dep"], cfg["period"], cfg["terms"])

    def a_block(r0, nr):
        t = gen_torch.sparse_dependent_rows(r0, nr, n, n, p, cfg["seed"], cfg["seed_dep"], cfg["period"], cfg["terms"],
                                            device=dev, plan=plan)
        return t.to(torch.int64)

    d = torch.empty((n, n), dtype=torch.int32, device=dev)
    gen_torch.fill_c5(d, cfg, block_rows=blk_rows)
    rank, piv, k = L.nullspace_u32(d, p)
    st = L.last_stats()
    print("c5: rank", rank, "launches", st["kernel_launches"], "swaps", st["row_swaps"], "device ms", st["ms_total"])

    # (v) rank and pivots
    r = n - n // cfg["period"]
    assert rank == r
    pivn = piv.numpy()
    assert np.array_equal(pivn, np.arange(r)), "pivot columns are 0..r-1 w.h.p. for this generator"
    assert k.shape == (n, n - r)

    # (i) structure (pivots are the first r columns)
    for r0 in range(0, n, 2048):
        blk = d[r0:r0 + 2048]
        assert int(blk.min()) >= 0                                  # int32 view of canonical residues < 2^31
        if r0 < r:
            top = blk[:min(2048, r - r0), :r]
            eye = torch.zeros_like(top)
            idx = torch.arange(top.shape[0], device=dev)
            eye[idx, r0 + idx] = 1
            assert torch.equal(top, eye)
        if r0 + 2048 > r:
            assert not blk[max(0, r - r0):].any(), "rows beyond the rank must be zero"

    # (ii) Freivalds: A.v = A[:, :r].(R.v)  <=>  A.(v - [R.v; 0]) = 0 for every row, three random vectors
    nv = 3
    v = torch.from_numpy(np.stack([gen.uniform_rows(0, 1, n, p, seed=900 + j)[0] for j in range(nv)], axis=1)
                         .astype(np.int64)).to(dev)
    w = torch.zeros((n, nv), dtype=torch.int64, device=dev)
    for r0 in range(0, r, blk_rows):
        nr = min(blk_rows, r - r0)
        w[r0:r0 + nr] = matvec_mod_p(d[r0:r0 + nr].to(torch.int64), v, p)
    u = (v - w) % p                                                 # rows >= r of w are zero
    # (iv) Freivalds for the kernel: A.(K.z) = 0
    z = torch.from_numpy(gen.uniform_rows(0, 1, n - r, p, seed=950)[0].astype(np.int64)).to(dev)
    kz = torch.zeros(n, dtype=torch.int64, device=dev)
    for r0 in range(0, n, 4096):
        kz[r0:r0 + 4096] = matvec_mod_p(k[r0:r0 + 4096].to(torch.int64), z, p)
    rhs = torch.cat([u, kz[:, None]], dim=1)
    bad = 0
    for r0 in range(0, n, blk_rows):
        nr = min(blk_rows, n - r0)
        bad += int(matvec_mod_p(a_block(r0, nr), rhs, p).count_nonzero())
    assert bad == 0, f"{bad} (row, vector) pairs violate A.v = A[:,piv].(R.v) or A.K.z = 0"

    # (iii) + (iv) exact checks on sampled rows with the CPU oracle's plain matmul
    rng = np.random.default_rng(5)
    rows_s = np.sort(rng.choice(n, size=8, replace=False))
    rows_s[0] = cfg["period"] - 1                                   # include a dependent row
    cols_s = np.sort(np.concatenate([rng.choice(r, size=192, replace=False), r + rng.choice(n - r, size=320, replace=False)]))
    a_s = np.concatenate([gen.sparse_dependent_rows(int(i), 1, n, n, p, cfg["seed"], cfg["seed_dep"]) for i in rows_s])
    r_cols = d[:r][:, torch.from_numpy(cols_s).to(dev)].cpu().numpy().view(np.uint32)       # r x 512
    assert np.array_equal(oracle.matmul_modp(np.ascontiguousarray(a_s[:, :r]), np.ascontiguousarray(r_cols), p,
                                             nthreads=oracle.max_threads()), a_s[:, cols_s])
    k_cols = np.sort(rng.choice(n - r, size=256, replace=False))
    k_s = k[:, torch.from_numpy(k_cols).to(dev)].cpu().numpy().view(np.uint32)              # n x 256
    assert not oracle.matmul_modp(a_s, np.ascontiguousarray(k_s), p, nthreads=oracle.max_threads()).any()
    # K's free rows are -I
    kf = k[r:, :]
    assert int((kf == p - 1).sum()) == n - r and int(kf.count_nonzero()) == n - r
    assert torch.equal(kf.diagonal(), torch.full((n - r,), p - 1, dtype=torch.int32, device=dev))
