"""Raw (unmerged) Jordan-Wigner term lists: the INPUT of bs_group_xmask (step a1).

PAPER.md:163-194 (Alg. 1) expands every one-body ladder product into 4 and every two-body ladder
product into 16 binary-symplectic strings and leaves sorting/merging to the canonical reduction
(PAPER.md:157).  This module does exactly that expansion with vectorised numpy on the host and
nothing more: no merge, no sort, no drop -- those run on the device in bs_group_xmask.  It shares no
code with oracle/ (which builds the operator by operator products into an ordered map).

Conventions (include/bs.h): qubit k = bit k; blocked spin ordering (alpha p -> qubit p, beta p ->
qubit n_orb + p); the returned coefficients are those of the TRUE Pauli strings.

Ladder operators in XZ-ordered form R(x,z) = (x)_k sx^{x_k} sz^{z_k} (Eq. 23; Eq. 13):
    a_P^dag = 1/2 R(b, lt) + 1/2 R(b, lt|b),   a_P = 1/2 R(b, lt) - 1/2 R(b, lt|b),
    b = 1<<P, lt = b - 1.
Product rule (Eq. 19-21): R(x1,z1) R(x2,z2) = (-1)^{popc(z1 & x2)} R(x1^x2, z1^z2).
True-Pauli coefficient: c = C (-i)^{popc(x & z)}.
"""
from __future__ import annotations

import itertools

import numpy as np

_U1 = np.uint64(1)


def _popc_parity(v: np.ndarray) -> np.ndarray:
    """parity of popcount of each uint64."""
    v = v.copy()
    for s in (32, 16, 8, 4, 2, 1):
        v ^= v >> np.uint64(s)
    return (v & _U1).astype(np.int64)


def _popc(v: np.ndarray) -> np.ndarray:
    return np.bitwise_count(v).astype(np.int64)


def ladder_product_terms(idx: np.ndarray, dagger, coef: np.ndarray):
    """All 2^k raw strings of coef[i] * prod_j op_j(idx[i, j]), op_j = a^dag if dagger[j] else a.

    idx: int64[N, k] spin-orbital (= qubit) indices; coef: float64 or complex128 [N].
    Returns x, z (uint64[N * 2^k]) and c (complex128), block j of N entries = choice pattern j.
    """
    idx = np.asarray(idx, np.int64)
    N, k = idx.shape
    coef = np.asarray(coef, np.complex128)
    bit = _U1 << idx.astype(np.uint64)            # [N, k]
    lt = bit - _U1
    xs, zs, cs = [], [], []
    for pattern in itertools.product((0, 1), repeat=k):
        x = np.zeros(N, np.uint64)
        z = np.zeros(N, np.uint64)
        sign = np.zeros(N, np.int64)              # exponent of (-1)
        for j in range(k):
            zj = lt[:, j] | bit[:, j] if pattern[j] else lt[:, j]
            sign += _popc_parity(z & bit[:, j])   # popc(z_acc & x_j)
            if pattern[j] and not dagger[j]:
                sign += 1                          # the -1/2 of the annihilator's second string
            x ^= bit[:, j]
            z ^= zj
        ny = _popc(x & z) & 3
        # c = C (-i)^ny with C = coef * 2^-k * (-1)^sign
        phase = np.array([1, -1j, -1, 1j], np.complex128)[ny]
        c = coef * (0.5 ** k) * np.where(sign & 1, -1.0, 1.0) * phase
        xs.append(x)
        zs.append(z)
        cs.append(c)
    return np.concatenate(xs), np.concatenate(zs), np.concatenate(cs)


def molecular_raw_terms(h: np.ndarray, g: np.ndarray):
    """Raw strings of H = sum_{pq,s} h_pq a^dag_{ps} a_{qs}
                       + 1/2 sum_{pqrs} sum_{s,t} (pq|rs) a^dag_{ps} a^dag_{rt} a_{st} a_{qs}
    (Eq. 2, spin-orbital form; reading U3).  g is chemist notation (pq|rs)."""
    n = h.shape[0]
    xs, zs, cs = [], [], []
    p, q = np.meshgrid(np.arange(n), np.arange(n), indexing="ij")
    p, q = p.ravel(), q.ravel()
    for s in (0, 1):
        x, z, c = ladder_product_terms(np.stack([p + s * n, q + s * n], 1), (True, False), h[p, q])
        xs.append(x), zs.append(z), cs.append(c)
    P, Q, R, S = (a.ravel() for a in np.meshgrid(*([np.arange(n)] * 4), indexing="ij"))
    gv = 0.5 * g[P, Q, R, S]
    for s in (0, 1):
        for t in (0, 1):
            i1, i2, i3, i4 = P + s * n, R + t * n, S + t * n, Q + s * n
            keep = (i1 != i2) & (i3 != i4)        # a^dag a^dag = a a = 0 on equal indices
            idx = np.stack([i1[keep], i2[keep], i3[keep], i4[keep]], 1)
            x, z, c = ladder_product_terms(idx, (True, True, False, False), gv[keep])
            xs.append(x), zs.append(z), cs.append(c)
    return np.concatenate(xs), np.concatenate(zs), np.concatenate(cs)


def hubbard_raw_terms(n_sites: int, t: float, U: float):
    """Open 1D Fermi-Hubbard chain: H = -t sum_{i,s} (a^dag_{is} a_{i+1,s} + h.c.) + U sum_i n_ia n_ib."""
    L = n_sites
    xs, zs, cs = [], [], []
    i = np.arange(L - 1)
    for s in (0, 1):
        for a, b in ((i, i + 1), (i + 1, i)):
            x, z, c = ladder_product_terms(np.stack([a + s * L, b + s * L], 1), (True, False),
                                           np.full(L - 1, -t))
            xs.append(x), zs.append(z), cs.append(c)
    j = np.arange(L)
    x, z, c = ladder_product_terms(np.stack([j, j, j + L, j + L], 1), (True, False, True, False),
                                   np.full(L, U))
    xs.append(x), zs.append(z), cs.append(c)
    return np.concatenate(xs), np.concatenate(zs), np.concatenate(cs)


def excitation_generator_terms(excitations):
    """Raw strings of the anti-Hermitian generators T - T^dag (Eq. 39), one run per
    excitation, T = prod a^dag_{creators} prod a_{annihilators}.

    `excitations`: list of (creators, annihilators) tuples of spin-orbital indices.  Each generator's
    2^k + 2^k raw strings are merged on the host per generator (equal (x,z) keys summed, exact zeros
    removed) because BS_MODE_SEQUENCE keeps runs verbatim.  Returns x, z, c and seq_offsets.
    """
    X, Z, Cc, offs = [], [], [], [0]
    for cre, ann in excitations:
        k = len(cre) + len(ann)
        fwd = np.array([list(cre) + list(ann)], np.int64)
        bwd = np.array([list(ann)[::-1] + list(cre)[::-1]], np.int64)   # T^dag
        dag_f = tuple([True] * len(cre) + [False] * len(ann))
        dag_b = tuple([True] * len(ann) + [False] * len(cre))
        x1, z1, c1 = ladder_product_terms(fwd, dag_f, np.array([1.0]))
        x2, z2, c2 = ladder_product_terms(bwd, dag_b, np.array([-1.0]))
        x, z, c = np.concatenate([x1, x2]), np.concatenate([z1, z2]), np.concatenate([c1, c2])
        order = np.lexsort((z, x))
        x, z, c = x[order], z[order], c[order]
        head = np.ones(len(x), bool)
        head[1:] = (x[1:] != x[:-1]) | (z[1:] != z[:-1])
        seg = np.cumsum(head) - 1
        cm = np.zeros(seg[-1] + 1, np.complex128)
        np.add.at(cm, seg, c)
        xm, zm = x[head], z[head]
        nz = np.abs(cm) > 2.0 ** -(k + 4)          # genuine |c| = 2^-(k-1); cancellations are exact 0
        X.append(xm[nz]), Z.append(zm[nz]), Cc.append(cm[nz])
        offs.append(offs[-1] + int(nz.sum()))
    return np.concatenate(X), np.concatenate(Z), np.concatenate(Cc), np.array(offs, np.int64)
