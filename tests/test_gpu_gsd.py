"""Generalised singles and doubles (tUCCGSD; universality) through bs_apply_pauli_rotations.

A GSD pool drops the occupied -> virtual restriction of UCCSD: singles a^dag_p a_q and doubles a^dag_p a^dag_q a_r a_s over
ANY orbitals of matching spin.  That brings in what the UCCSD lists never contain: several generators with the SAME X
mask (the three pairings of four orbitals; every shared-index double n_p a^dag_q a_s has the X mask of the single
a^dag_q a_s), generators of 4 Pauli strings that carry a number projector (|f| in {0, 1} with f = 0 INSIDE the sector),
and pairs that touch occupied and virtual orbitals alike.  Oracle: the fermionic Givens rotation of oracle/ (pinned on
shared-index doubles by P9), generator by generator, on a random state; full-vector comparison.
"""
import itertools

import numpy as np
import pytest

import synth_inputs as si
from common import rel_l2

pytestmark = pytest.mark.gpu


def gsd_pool(n, rng, n_doubles):
    """All generalised singles of both spins, then `n_doubles` seeded generalised doubles (same-spin and opposite-spin,
    shared indices allowed), then for a few index quadruples all three pairings, which share one X mask.  Index
    bookkeeping only: (creators, annihilators) in spin-orbital indices."""
    pool = []
    for s in range(2):
        for p, q in itertools.permutations(range(n), 2):
            if p > q:
                pool.append(((s * n + p,), (s * n + q,)))
    spin_orb = list(range(2 * n))

    def spin(P):
        return P // n
    doubles = []
    while len(doubles) < n_doubles:
        p, q, r, s = (int(v) for v in rng.choice(spin_orb, 4))
        if p == q or r == s or {p, q} == {r, s}:
            continue
        if sorted((spin(p), spin(q))) != sorted((spin(r), spin(s))):      # S_z conserved: stays in the sector
            continue
        doubles.append(((p, q), (r, s)))
    pool += doubles
    for a, b, c, d in ((0, 2, 3, 5), (n + 1, n + 2, n + 4, n + 5), (1, 4, n + 0, n + 3)):
        for cre, ann in (((a, b), (c, d)), ((a, c), (b, d)), ((a, d), (b, c))):
            if sorted((spin(cre[0]), spin(cre[1]))) == sorted((spin(ann[0]), spin(ann[1]))):
                pool.append((cre, ann))
    return pool


@pytest.mark.parametrize("n,na,nb,n_doubles", [(6, 3, 3, 300), (8, 4, 3, 400)])
def test_gsd_pool_rotations_against_fermionic_oracle(n, na, nb, n_doubles):
    import torch
    from oracle import oracle as orc
    from paper_2606_28952_b200 import bs
    from paper_2606_28952_b200 import jw_terms as jw
    rng = np.random.default_rng(100 + n)
    pool = gsd_pool(n, rng, n_doubles)
    order = rng.permutation(len(pool))                    # generators of equal X mask end up apart AND adjacent
    pool = [pool[i] for i in order]
    th = rng.standard_normal(len(pool)) * 0.3
    X, Z, Cc, offs = jw.excitation_generator_terms(pool)
    gens = bs.bs_group_xmask(X, Z, Cc, 2 * n, 0.0, bs.BS_MODE_SEQUENCE, offs)
    xg = X[offs[:-1]]
    assert len(np.unique(xg)) < 0.75 * len(pool)          # the pool really shares X masks (166 of 338, 312 of 464)
    n_str = np.diff(offs)
    assert set(np.unique(n_str)) == {2, 4, 8}             # singles, shared-index doubles, doubles (T - T^dag merged)
    shared = [k for k, (cre, ann) in enumerate(pool) if set(cre) & set(ann)]
    assert len(shared) >= 20                              # shared-index doubles: number projector x single
    sec, osec = bs.bs_sector_build(n, na, nb), orc.Sector(n, na, nb)
    psi = si.random_state(osec.dim, 5)
    d = torch.from_numpy(psi.copy()).cuda()
    bs.bs_apply_pauli_rotations(gens, sec, th, d)
    want = psi.copy()
    for (cre, ann), t in zip(pool, th):
        osec.rot_fermionic(want, list(cre), list(ann), float(t))
    got = d.cpu().numpy()
    assert rel_l2(got, want) <= 1e-12
    assert abs(np.linalg.norm(got) - 1.0) <= 1e-12
    # the whole list once more on the rotated state (both sides)
    bs.bs_apply_pauli_rotations(gens, sec, th, d)
    for (cre, ann), t in zip(pool, th):
        osec.rot_fermionic(want, list(cre), list(ann), float(t))
    assert rel_l2(d.cpu().numpy(), want) <= 1e-12
