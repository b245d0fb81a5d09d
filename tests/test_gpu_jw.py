"""GPU parity of the device-side Jordan-Wigner construction (bs_jw_molecular, bs_jw_hubbard; PAPER.md:163-194,
Alg. 1) against the oracle's operator route: keys and offsets bit-exact, coefficients to 1e-13 * max|c|
(the device sums the 4/16-term expansions in its own emission order)."""
import numpy as np
import pytest

import synth_inputs as si
from common import oracle_operator, rel_l2

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def bs():
    from paper_2606_28952_b200 import bs as _bs
    return _bs


def _check_tables(op, ref):
    xg, offs, zz, cc, ww = op.export()
    exg, first = np.unique(ref.x, return_index=True)
    assert op.n_terms == len(ref) and np.array_equal(xg, exg)
    assert np.array_equal(offs, np.concatenate([first, [len(ref)]]))
    assert np.array_equal(zz, ref.z)
    assert np.abs(cc - ref.c).max() <= 1e-13 * np.abs(ref.c).max()
    assert np.abs(cc.imag).max() == 0.0            # every true coefficient of a real Hamiltonian is real (pin P3)


@pytest.mark.parametrize("name", ["q12", "q24", "q32", "q56"])   # q56: 3.9e7 raw strings, the route bench.py times
def test_jw_molecular_tables(bs, name):
    cfg = si.CONFIGS[name]
    h, g = si.integrals(cfg.n_orb, cfg.seed_ints)
    op = bs.bs_jw_molecular(h, g)
    _check_tables(op, oracle_operator(name))


def test_jw_hubbard_tables_and_apply(bs):
    import torch
    from oracle import oracle as orc
    op = bs.bs_jw_hubbard(14, 1.0, 4.0)
    _check_tables(op, oracle_operator("q28_hubbard"))
    assert op.n_terms == 95 and op.n_groups == 27
    ref = orc.hubbard_h(6, 1.0, 4.0)
    op6 = bs.bs_jw_hubbard(6, 1.0, 4.0)
    sec, osec = bs.bs_sector_build(6, 3, 2), orc.Sector(6, 3, 2)
    psi = si.random_state(osec.dim, 1)
    d_in = torch.from_numpy(psi).cuda()
    d_out = torch.empty_like(d_in)
    bs.bs_apply(op6, sec, d_in, d_out)
    assert rel_l2(d_out.cpu().numpy(), osec.apply(ref, psi)) <= 1e-12


def test_jw_molecular_apply_and_errors(bs):
    import torch
    from oracle import oracle as orc
    h, g = si.integrals(5, 42)
    op = bs.bs_jw_molecular(h, g)
    ref = orc.molecular_h(h, g)
    for na, nb in [(2, 3), (5, 0), (1, 1)]:
        sec, osec = bs.bs_sector_build(5, na, nb), orc.Sector(5, na, nb)
        psi = si.random_state(osec.dim, 3)
        d_in = torch.from_numpy(psi).cuda()
        d_out = torch.empty_like(d_in)
        bs.bs_apply(op, sec, d_in, d_out)
        want = osec.apply(ref, psi)
        assert rel_l2(d_out.cpu().numpy(), want) <= 1e-12
        assert abs(bs.bs_expect(op, sec, d_in) - orc.vdot(psi, want)) <= 1e-10
    with pytest.raises(ValueError):
        bs.bs_jw_molecular(h, g[:4])
    with pytest.raises(bs.BsError):
        bs.bs_jw_hubbard(1, 1.0, 4.0)
