"""Seeded synthetic inputs for the QR-CTMRG hot path (BASELINE.json `configs`).

This module is the ONLY code shared by the CPU oracle (`oracle/`) and the CUDA
path (`paper_2505_00494_b200/`).  It holds no arithmetic of the method itself
(no contraction, no QR, no normalisation of an iterate): it only draws the
random tensors the configs prescribe and puts them in the symmetric, scaled
form BASELINE.json states.  DESIGN.md §"Input recipe" restates it.

Recipe (BASELINE.json configs[0]):
  * one PRNG stream `numpy.random.default_rng(seed)`, draw order A, C, T;
  * A (d,D,D,D,D) i.i.d. N(0,1), averaged over the 8 permutations of its four
    auxiliary legs that form the dihedral group of the square (legs stored in
    cyclic order u,l,d,r), then scaled to max|A| = 1;
  * C0 (chi,chi) N(0,1) symmetrised, Frobenius-normalised;
  * T0 (chi,D*D,chi) N(0,1) symmetrised in its two chi legs, Frobenius-normalised.

The paper's own workloads are optimised Heisenberg / J1-J2 iPEPS tensors
 that do not exist here; these random C4v tensors of the
same shapes stand in for them.
"""
from __future__ import annotations

import numpy as np

# Dihedral group of the square acting on leg positions (u,l,d,r) = (0,1,2,3):
# new leg i <- old leg PERMS[g][i].  Four rotations, four reflections.
C4V_PERMS = (
    (0, 1, 2, 3), (1, 2, 3, 0), (2, 3, 0, 1), (3, 0, 1, 2),
    (0, 3, 2, 1), (2, 1, 0, 3), (1, 0, 3, 2), (3, 2, 1, 0),
)

# (d, D, chi, seed, iterations, tol) for the BASELINE.json configs; cfg3 has two chi.
CONFIGS = {
    "cfg0": dict(d=2, D=2, chi=8, seed=0, iters=50, tol=1e-12),
    "cfg1": dict(d=2, D=3, chi=36, seed=1, iters=500, tol=1e-10),
    "cfg2": dict(d=2, D=4, chi=64, seed=2, iters=300, tol=1e-10),
    "cfg3a": dict(d=2, D=5, chi=100, seed=3, iters=200, tol=1e-10),
    "cfg3b": dict(d=2, D=5, chi=150, seed=3, iters=200, tol=1e-10),
    "cfg4": dict(d=2, D=7, chi=196, seed=4, iters=100, tol=1e-10),
}


def c4v_symmetrize(A: np.ndarray) -> np.ndarray:
    """Average a (d,D,D,D,D) tensor over the 8 aux-leg permutations of C4V_PERMS."""
    out = np.zeros_like(A)
    for p in C4V_PERMS:
        out += A.transpose(0, 1 + p[0], 1 + p[1], 1 + p[2], 1 + p[3])
    return out / len(C4V_PERMS)


def gen_config(d: int, D: int, chi: int, seed: int):
    """Return (A, C0, T0) as C-contiguous float64 arrays for one config."""
    g = np.random.default_rng(seed)
    b = D * D
    A = g.standard_normal((d, D, D, D, D))
    A = c4v_symmetrize(A)
    A = A / np.max(np.abs(A))
    C0 = g.standard_normal((chi, chi))
    C0 = 0.5 * (C0 + C0.T)
    C0 = C0 / np.sqrt(np.sum(C0 * C0))
    T0 = g.standard_normal((chi, b, chi))
    T0 = 0.5 * (T0 + T0.transpose(2, 1, 0))
    T0 = T0 / np.sqrt(np.sum(T0 * T0))
    return (np.ascontiguousarray(A), np.ascontiguousarray(C0),
            np.ascontiguousarray(T0))


def gen_named(name: str):
    """(A, C0, T0, cfg_dict) for a BASELINE.json config name ('cfg0' ... 'cfg4')."""
    c = CONFIGS[name]
    A, C0, T0 = gen_config(c["d"], c["D"], c["chi"], c["seed"])
    return A, C0, T0, dict(c)


def random_isometry(rows: int, cols: int, seed: int) -> np.ndarray:
    """A seeded rows x cols matrix with orthonormal columns (for sub-step parity
    tests that need 'some isometry' in place of Q)."""
    g = np.random.default_rng(seed)
    q, _ = np.linalg.qr(g.standard_normal((rows, cols)))
    return np.ascontiguousarray(q)
