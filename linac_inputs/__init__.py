"""Seeded synthetic inputs for the Linac hot path (shared by tests, oracle timing and bench).

This module holds NONE of the method's arithmetic (no elimination, no inverse, no
reduction trick): it only draws numbers.  Both the CPU oracle (`oracle/`) and the CUDA
path (`paper_2605_25863_b200/`) are fed from here; neither imports the other.

Recipe (the paper measures on "100% dense, fully random square
matrices in F_{2^31-1}", PAPER.md:308 -- not a public data set, so these stand in for it):

    h(seed, idx) = splitmix64_finaliser(seed + 0x9E3779B97F4A7C15 * (idx + 1))   (mod 2^64)
    uniform in [0, p):  mulhi64(h, p)          (bias < 2^-33, deterministic)
    idx = r * cols + c  as a 64-bit counter

so any element / row of any config can be re-created without the rest (needed to certify
the N = 10^5 config without holding a second 40 GB copy).  `linac_inputs/gen_torch.py`
implements the same counter-based generator with torch integer ops (so it can run on the device),
bit-identically.
"""
from .gen import (  # noqa: F401
    splitmix64,
    uniform_mod_p,
    uniform_matrix,
    uniform_rows,
    uniform_mod_p64,
    uniform_matrix_u64,
    lowrank_factors,
    sparse_dependent_rows,
    sparse_dependent_plan,
    normal_matrix,
    shifted_normal_system,
    CONFIGS,
)
