"""Point-group symmetry blocking (Eq. 29-31; "sDet" of Table 2) against the oracle.

Synthetic D2h labels: every orbital gets an irrep 0..7, the symmetry-forbidden integrals of the seeded recipe are
zeroed (h_pq unless irrep p = irrep q; (pq|rs) unless the four labels XOR to 0), so H conserves the irrep of a
configuration = XOR of the labels of its occupied spin-orbitals.  The oracle gets the restriction by brute force: the
allowed configurations are listed with numpy from the oracle's own string lists (in the documented block order), the
blocked vector is embedded into the sector vector, the oracle applies H there, and the block is read back.
"""
import numpy as np
import pytest

import synth_inputs as si
from common import rel_l2

pytestmark = pytest.mark.gpu


def _sym_integrals(n, seed, labels):
    h, g = si.integrals(n, seed)
    lab = np.asarray(labels)
    h = h * (lab[:, None] == lab[None, :])
    x = lab[:, None, None, None] ^ lab[None, :, None, None] ^ lab[None, None, :, None] ^ lab[None, None, None, :]
    return np.ascontiguousarray(h), np.ascontiguousarray(g * (x == 0))


def _blocked_index(osec, labels, target):
    """Sector index of every amplitude of the blocked vector, in the layout include/bs.h documents."""
    a, b = osec.strings()

    def irrep(strs):
        out = np.zeros(len(strs), np.int64)
        for p, lab in enumerate(labels):
            out ^= np.where((strs >> np.uint64(p)) & np.uint64(1), lab, 0).astype(np.int64)
        return out
    ia, ib = irrep(a), irrep(b)
    idx = []
    for r in range(8):
        rows = np.nonzero(ia == r)[0]
        cols = np.nonzero(ib == (r ^ target))[0]
        idx.append((rows[:, None] * osec.dim_beta + cols[None, :]).ravel())
    return np.concatenate(idx), ia, ib


@pytest.mark.parametrize("n,na,nb,labels,target", [
    (12, 6, 6, [0, 1, 2, 3, 4, 5, 6, 7, 0, 1, 2, 3], 0),       # q24-sized, D2h-like: 8 irreps
    (12, 6, 6, [0, 1, 2, 3, 4, 5, 6, 7, 0, 1, 2, 3], 5),
    (9, 3, 5, [0, 1, 2, 3, 0, 1, 2, 3, 0], 3),                 # C2v-like: 4 irreps, some blocks empty
])
def test_symmetry_blocked_apply_and_energy(n, na, nb, labels, target):
    import torch
    from oracle import oracle as orc
    from paper_2606_28952_b200 import bs
    h, g = _sym_integrals(n, 1002, labels)
    ref = orc.molecular_h(h, g)
    op = bs.bs_jw_molecular(h, g)
    sec, osec = bs.bs_sector_build(n, na, nb), orc.Sector(n, na, nb)
    sym = bs.bs_symsector_build(sec, labels, target)
    idx, ia, ib = _blocked_index(osec, labels, target)
    assert sym.dim == len(idx) and len(np.unique(idx)) == len(idx)
    assert np.array_equal(sym.dim_alpha, np.bincount(ia, minlength=8))
    assert np.array_equal(sym.dim_beta, np.bincount(ib, minlength=8))
    if len(set(labels)) == 8:
        assert sym.dim < osec.dim / 7                                  # the working space shrinks by ~ |G| = 8
    psi_b = si.random_state(sym.dim, 31)
    full = np.zeros(osec.dim, np.complex128)
    full[idx] = psi_b
    want_full = osec.apply_grouped(ref, full)
    mask = np.ones(osec.dim, bool)
    mask[idx] = False
    assert np.abs(want_full[mask]).max() <= 1e-13                       # H conserves the irrep (the integrals were zeroed)
    d_b = torch.from_numpy(psi_b).cuda()
    d_full = torch.full((osec.dim,), float("nan"), dtype=torch.complex128, device="cuda")
    bs.bs_sym_scatter(sym, d_b, d_full)
    assert np.array_equal(d_full.cpu().numpy(), full)                   # embedding, bit for bit
    d_back = torch.empty_like(d_b)
    bs.bs_sym_gather(sym, d_full, d_back)
    assert np.array_equal(d_back.cpu().numpy(), psi_b)
    d_out = torch.empty_like(d_b)
    bs.bs_sym_apply(op, sym, d_b, d_out)
    assert rel_l2(d_out.cpu().numpy(), want_full[idx]) <= 1e-12
    e = bs.bs_sym_expect(op, sym, d_b)
    assert abs(e - orc.vdot(full, want_full)) <= 1e-10 and abs(e.imag) <= 1e-10


def test_symsector_errors():
    from paper_2606_28952_b200 import bs
    sec = bs.bs_sector_build(6, 3, 3)
    with pytest.raises(bs.BsError):
        bs.bs_symsector_build(sec, [0, 1, 2, 3, 4, 9], 0)
    with pytest.raises(bs.BsError):
        bs.bs_symsector_build(sec, [0] * 6, 8)
    with pytest.raises(bs.BsError):
        bs.bs_symsector_build(bs.bs_sector_build(12), [0] * 12, 0)
