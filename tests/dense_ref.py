"""Independent dense/sparse reference matrices used ONLY to pin the oracle (tests/, `not gpu`).

Nothing here is shared with oracle/ or the CUDA path: Pauli sums become explicit Kronecker
products of 2x2 matrices, fermionic operators become explicit occupation-number matrices.
Qubit k = bit k of the basis index = k-th factor from the RIGHT of the Kronecker product.
"""
import numpy as np
import scipy.sparse as sp

I2 = np.eye(2, dtype=complex)
SX = np.array([[0, 1], [1, 0]], dtype=complex)
SY = np.array([[0, -1j], [1j, 0]], dtype=complex)
SZ = np.array([[1, 0], [0, -1]], dtype=complex)
PAULI = {(0, 0): I2, (1, 0): SX, (1, 1): SY, (0, 1): SZ}  # PAPER.md:93 Eq. 8


def pauli_string_matrix(x: int, z: int, nq: int):
    """Sparse 2^nq matrix of the true Pauli string (x){I,X,Y,Z} with masks (x, z)."""
    m = sp.identity(1, dtype=complex, format="csr")
    for k in range(nq - 1, -1, -1):  # leftmost factor = highest qubit
        a, b = (x >> k) & 1, (z >> k) & 1
        m = sp.kron(m, sp.csr_matrix(PAULI[(a, b)]), format="csr")
    return m


def pauli_sum_matrix(xs, zs, cs, nq: int):
    dim = 1 << nq
    acc = sp.csr_matrix((dim, dim), dtype=complex)
    for x, z, c in zip(xs, zs, cs):
        acc = acc + complex(c) * pauli_string_matrix(int(x), int(z), nq)
    return acc


def creation_matrix(P: int, nq: int):
    """a^dag_P in the occupation-number basis |s>, bit P of s = occupation of spin-orbital P.
    a^dag_P |s> = (-1)^{# occupied below P} |s + P> if P is empty, else 0."""
    dim = 1 << nq
    rows, cols, vals = [], [], []
    for s in range(dim):
        if (s >> P) & 1:
            continue
        sign = -1.0 if bin(s & ((1 << P) - 1)).count("1") & 1 else 1.0
        rows.append(s | (1 << P))
        cols.append(s)
        vals.append(sign)
    return sp.csr_matrix((vals, (rows, cols)), shape=(dim, dim), dtype=complex)


def molecular_h_matrix(h, g):
    """H of SURVEY §8(c) item 2 (Eq. 2, reading U3) from fermionic matrices."""
    n = h.shape[0]
    nq = 2 * n
    cre = [creation_matrix(P, nq) for P in range(nq)]
    ann = [c.conj().T.tocsr() for c in cre]
    dim = 1 << nq
    H = sp.csr_matrix((dim, dim), dtype=complex)
    for p in range(n):
        for q in range(n):
            for s in range(2):
                H = H + h[p, q] * (cre[p + s * n] @ ann[q + s * n])
            for r in range(n):
                for u in range(n):
                    for s in range(2):
                        for t in range(2):
                            P, Q, R, U = p + s * n, q + s * n, r + t * n, u + t * n
                            H = H + 0.5 * g[p, q, r, u] * (cre[P] @ cre[R] @ ann[U] @ ann[Q])
    return H


def slater_condon_energy(h, g, occ_a, occ_b):
    """Energy of a single determinant from the integrals:
    E = sum_{i,s} h_ii + 1/2 sum_{is,jt} [(ii|jj) - delta_st (ij|ji)]."""
    e = 0.0
    occ = [(i, 0) for i in occ_a] + [(i, 1) for i in occ_b]
    for i, _ in occ:
        e += h[i, i]
    for i, s in occ:
        for j, t in occ:
            e += 0.5 * g[i, i, j, j]
            if s == t:
                e -= 0.5 * g[i, j, j, i]
    return e


def bits(w: int):
    return [k for k in range(64) if (w >> k) & 1]
