"""Seeded synthetic inputs shared by the oracle tests and the CUDA path.

This module holds NONE of the method's arithmetic (no Pauli algebra, no ranking, no
phases): it only draws the random arrays both sides receive and names the five
BASELINE.json configurations.  The oracle (oracle/) and the product
(paper_2606_28952_b200/) each turn these arrays into operators on their own.

Recipes (BASELINE.json `configs`):
  * h_pq ~ N(0,1), symmetrised as (B + B^T)/2.
  * g_pqrs = sum_{L<rank} A^L_pq A^L_rs with A^L = (B + B^T)/2, B_ij ~ N(0, 0.3)
    (0.3 = standard deviation) -> real, 8-fold symmetric, chemist notation (pq|rs).
  * psi: re, im ~ N(0,1), normalised to unit 2-norm, complex128.
  * thetas ~ N(0, 0.05).
The paper's own workloads are PySCF molecular integrals (Table 2) which are
not available offline; these dense seeded integrals stand in for them (same M/G regime,
same sector sizes).
"""
from __future__ import annotations

import dataclasses
import math

import numpy as np


@dataclasses.dataclass(frozen=True)
class Config:
    name: str
    kind: str          # "molecular" | "hubbard"
    n_orb: int
    n_alpha: int
    n_beta: int
    seed_ints: int
    seed_psi: int
    seed_theta: int = 0
    hubbard_t: float = 1.0
    hubbard_u: float = 4.0

    @property
    def n_qubits(self) -> int:
        return 2 * self.n_orb

    @property
    def dim_alpha(self) -> int:
        return math.comb(self.n_orb, self.n_alpha)

    @property
    def dim_beta(self) -> int:
        return math.comb(self.n_orb, self.n_beta)

    @property
    def dim(self) -> int:
        return self.dim_alpha * self.dim_beta


# BASELINE.json configs[0..4]; seeds from SURVEY.md §8(d).
CONFIGS = {
    "q12": Config("q12", "molecular", 6, 3, 3, 1001, 2001),
    "q24": Config("q24", "molecular", 12, 6, 6, 1002, 2002, 3002),
    "q28_hubbard": Config("q28_hubbard", "hubbard", 14, 7, 7, 0, 2003),
    "q32": Config("q32", "molecular", 16, 8, 8, 1004, 2004),
    "q56": Config("q56", "molecular", 28, 4, 4, 1005, 2005),
}
CONFIG_ORDER = ["q12", "q24", "q28_hubbard", "q32", "q56"]


def integrals(n_orb: int, seed: int, rank: int | None = None):
    """(h[n,n], g[n,n,n,n]) float64; g in chemist notation (pq|rs), 8-fold symmetric."""
    rank = n_orb if rank is None else rank
    rng = np.random.default_rng(seed)
    b = rng.standard_normal((n_orb, n_orb))
    h = 0.5 * (b + b.T)
    a = rng.standard_normal((rank, n_orb, n_orb)) * 0.3
    a = 0.5 * (a + a.transpose(0, 2, 1))
    g = np.einsum("lpq,lrs->pqrs", a, a, optimize=True)
    return np.ascontiguousarray(h), np.ascontiguousarray(g)


def random_state(dim: int, seed: int) -> np.ndarray:
    """Random normalised complex128 vector, re, im ~ N(0,1)."""
    rng = np.random.default_rng(seed)
    psi = np.empty(dim, dtype=np.complex128)
    v = psi.view(np.float64)
    chunk = 1 << 24
    parts = []
    for i in range(0, 2 * dim, chunk):
        j = min(2 * dim, i + chunk)
        v[i:j] = rng.standard_normal(j - i)
        parts.append(float(np.sum(np.square(v[i:j]))))
    # the squared norm by numpy's own (single-threaded, pairwise) sums per chunk: np.dot is a threaded BLAS reduction
    # whose rounding, and with it the last bit of EVERY amplitude, changed with the host's thread count
    nrm = math.sqrt(math.fsum(parts))
    v /= nrm
    return psi


def thetas(n: int, seed: int, sd: float = 0.05) -> np.ndarray:
    rng = np.random.default_rng(seed)
    return rng.standard_normal(n) * sd


def uccsd_excitations(n_orb: int, n_alpha: int, n_beta: int):
    """Excitation index list in the order of SURVEY.md §8(c) U10.

    Each entry is (creators, annihilators) in SPIN-ORBITAL indices (alpha p -> p, beta p ->
    n_orb + p), T = prod a^dag_{creators} prod a_{annihilators} written left to right, i.e.
    singles T = a^dag_a a_i, doubles T = a^dag_a a^dag_b a_j a_i with a<b, i<j.
    Pure index bookkeeping, no operator arithmetic.
    """
    occ_a = list(range(n_alpha))
    vir_a = list(range(n_alpha, n_orb))
    occ_b = [n_orb + p for p in range(n_beta)]
    vir_b = [n_orb + p for p in range(n_beta, n_orb)]
    out = []
    for occ, vir in ((occ_a, vir_a), (occ_b, vir_b)):
        for i in occ:
            for a in vir:
                out.append(((a,), (i,)))
    for occ, vir in ((occ_a, vir_a), (occ_b, vir_b)):
        for ii, i in enumerate(occ):
            for j in occ[ii + 1:]:
                for ai, a in enumerate(vir):
                    for b in vir[ai + 1:]:
                        out.append(((a, b), (j, i)))
    for i in occ_a:
        for a in vir_a:
            for j in occ_b:
                for b in vir_b:
                    out.append(((a, b), (j, i)))
    return out


def tfim_terms(n_qubits: int, J: float = 0.25, h: float = 1.0):
    """Open transverse-field Ising chain H = J sum Z_i Z_{i+1} + h sum X_i (Eq. 40: J = 1/4, h = 1) as
    (x masks, z masks, coefficients) of its 2 N - 1 Pauli strings.  Index bookkeeping only."""
    x, z, c = [], [], []
    for i in range(n_qubits - 1):
        x.append(0), z.append((1 << i) | (1 << (i + 1))), c.append(J)
    for i in range(n_qubits):
        x.append(1 << i), z.append(0), c.append(h)
    return np.array(x, np.uint64), np.array(z, np.uint64), np.array(c, np.complex128)
