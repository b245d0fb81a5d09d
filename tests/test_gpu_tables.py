"""GPU parity, integer work (bit-exact bar): a1/a2 grouping tables and a3 sector tables vs the oracle.

SURVEY.md 8(c): x, z, offsets, strings, ranks and dimensions must agree bit for bit.  Coefficients are
bit-exact when both sides sum duplicates in the same order (test_group_coefficients_bit_exact);
the harness route sums the 4/16-term expansions in a different order than the oracle's ordered map,
so there the bar is 1e-13 * max|c| (rounding of <= ~1e3 additions of O(1) numbers).
"""
import numpy as np
import pytest

import synth_inputs as si
from common import oracle_operator, raw_terms

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def bs():
    from paper_2606_28952_b200 import bs as _bs
    return _bs


def _fold(c, x, z):
    """w = c (-i)^{ny} by exact swaps/negations (no rounding)."""
    ny = np.bitwise_count(x & z).astype(np.int64) & 3
    w = c.copy()
    w[ny == 1] = c[ny == 1].imag - 1j * c[ny == 1].real
    w[ny == 2] = -c[ny == 2]
    w[ny == 3] = -c[ny == 3].imag + 1j * c[ny == 3].real
    return w


def _expected_groups(x):
    xg, first = np.unique(x, return_index=True)
    offs = np.concatenate([first, [len(x)]]).astype(np.int64)
    return xg, offs


@pytest.mark.parametrize("name", ["q12", "q24", "q28_hubbard"])
def test_group_tables_bit_exact_from_raw_terms(bs, name):
    cfg = si.CONFIGS[name]
    ref = oracle_operator(name)
    x, z, c = raw_terms(name)
    op = bs.bs_group_xmask(x, z, c, cfg.n_qubits, 1e-12)
    xg, offs, zz, cc, ww = op.export()
    exg, eoffs = _expected_groups(ref.x)
    assert op.n_terms == len(ref) and op.n_groups == len(exg)
    assert np.array_equal(xg, exg)
    assert np.array_equal(offs, eoffs)
    assert np.array_equal(zz, ref.z)
    scale = np.abs(ref.c).max()
    assert np.abs(cc - ref.c).max() <= 1e-13 * scale
    xs = np.repeat(xg, np.diff(offs))
    assert np.array_equal(ww.view(np.float64), _fold(cc, xs, zz).view(np.float64))


def test_group_coefficients_bit_exact(bs):
    """Shuffled input with every term split into 0.75 c + 0.25 c (exact in binary): stable sort +
    in-input-order summation must reproduce c bit for bit."""
    ref = oracle_operator("q12")
    rng = np.random.default_rng(7)
    M = len(ref)
    perm = rng.permutation(M)
    x = np.concatenate([ref.x[perm], ref.x[perm][::-1]])
    z = np.concatenate([ref.z[perm], ref.z[perm][::-1]])
    c = np.concatenate([0.75 * ref.c[perm], 0.25 * ref.c[perm][::-1]])
    op = bs.bs_group_xmask(x, z, c, 12, 1e-12)
    xg, offs, zz, cc, _ = op.export()
    assert np.array_equal(zz, ref.z)
    assert np.array_equal(cc.view(np.float64), ref.c.view(np.float64))
    assert np.array_equal(xg, _expected_groups(ref.x)[0])


def test_group_input_order_summation(bs):
    """(1e16 + 1) - 1e16 in input order is 0 (1e16 + 1 rounds to 1e16); in another order it is 1."""
    x = np.array([3, 3, 3, 5], np.uint64)
    z = np.array([1, 1, 1, 0], np.uint64)
    c = np.array([1e16, 1.0, -1e16, 2.0], np.complex128)
    op = bs.bs_group_xmask(x, z, c, 4, 0.5)
    xg, offs, zz, cc, _ = op.export()
    assert op.n_terms == 1 and xg.tolist() == [5] and cc[0] == 2.0
    c2 = np.array([1e16, -1e16, 1.0, 2.0], np.complex128)
    op2 = bs.bs_group_xmask(x, z, c2, 4, 0.5)
    assert op2.n_terms == 2 and op2.export()[3][0] == 1.0


def test_group_edge_cases(bs):
    e = np.zeros(0, np.uint64)
    op = bs.bs_group_xmask(e, e, np.zeros(0, np.complex128), 8)
    assert op.n_terms == 0 and op.n_groups == 0 and op.export()[1].tolist() == [0]
    # everything cancels
    x = np.array([1, 1], np.uint64)
    op = bs.bs_group_xmask(x, x, np.array([0.5, -0.5], np.complex128), 8)
    assert op.n_terms == 0 and op.n_groups == 0
    # 64-bit masks, unsigned order (top bit set sorts last)
    x = np.array([1 << 63, 1, (1 << 63) | 1], np.uint64)
    z = np.array([0, 1 << 63, 5], np.uint64)
    op = bs.bs_group_xmask(x, z, np.ones(3, np.complex128), 64)
    assert op.export()[0].tolist() == [1, 1 << 63, (1 << 63) | 1]
    # bits above n_qubits are rejected, outputs untouched
    with pytest.raises(bs.BsError) as ei:
        bs.bs_group_xmask(np.array([256], np.uint64), np.array([0], np.uint64), np.ones(1, np.complex128), 8)
    assert ei.value.status == bs.BS_ERR_ARG


def test_group_sequence_mode(bs):
    from paper_2606_28952_b200 import jw_terms as jw
    ex = si.uccsd_excitations(6, 3, 3)
    X, Z, Cc, offs = jw.excitation_generator_terms(ex)
    op = bs.bs_group_xmask(X, Z, Cc, 12, 0.0, bs.BS_MODE_SEQUENCE, offs)
    xg, o, zz, cc, ww = op.export()
    assert op.n_groups == len(ex) and np.array_equal(o, offs)
    assert np.array_equal(zz, Z) and np.array_equal(cc, Cc) and np.array_equal(xg, X[offs[:-1]])
    assert np.array_equal(ww.view(np.float64), _fold(Cc, X, Z).view(np.float64))
    bad = X.copy()
    bad[1] ^= np.uint64(1)
    with pytest.raises(bs.BsError) as ei:
        bs.bs_group_xmask(bad, Z, Cc, 12, 0.0, bs.BS_MODE_SEQUENCE, offs)
    assert ei.value.status == bs.BS_ERR_ARG


@pytest.mark.parametrize("n,na,nb", [(6, 3, 3), (12, 6, 6), (14, 7, 7), (16, 8, 8), (28, 4, 4), (10, 0, 10),
                                     (9, 2, 5), (20, 2, 3)])
def test_sector_tables_bit_exact(bs, n, na, nb):
    from oracle import oracle as orc
    ref = orc.Sector(n, na, nb)
    sec = bs.bs_sector_build(n, na, nb)
    assert (sec.dim, sec.dim_alpha, sec.dim_beta) == (ref.dim, ref.dim_alpha, ref.dim_beta)
    a, b = sec.export()
    ra, rb = ref.strings()
    assert np.array_equal(a, ra) and np.array_equal(b, rb)
    rng = np.random.default_rng(n * 100 + na)
    # in-sector configurations (random pairs of strings), their neighbours, and random words
    ia = rng.integers(0, ref.dim_alpha, 20000)
    ib = rng.integers(0, ref.dim_beta, 20000)
    inside = ra[ia] | (rb[ib] << np.uint64(n))
    flips = inside ^ (np.uint64(1) << rng.integers(0, 2 * n, 20000).astype(np.uint64))
    rnd = rng.integers(0, 1 << 62, 20000, dtype=np.uint64) & np.uint64((1 << (2 * n)) - 1)
    ends = np.array([ra[0] | (rb[0] << np.uint64(n)), ra[-1] | (rb[-1] << np.uint64(n))], np.uint64)
    cfgs = np.concatenate([inside, flips, rnd, ends])
    got = sec.rank(cfgs)
    assert np.array_equal(got, ref.index(cfgs))
    assert np.array_equal(got[:20000], ia * ref.dim_beta + ib)
    assert got[-2] == 0 and got[-1] == ref.dim - 1


def test_sector_full_space_and_errors(bs):
    sec = bs.bs_sector_build(12)
    assert sec.dim == 4096 and sec.full
    cfgs = np.array([0, 5, 4095, 4096], np.uint64)
    assert sec.rank(cfgs).tolist() == [0, 5, 4095, -1]
    for args in [(0, 0, 0), (33, 1, 1), (6, 7, 1), (6, -1, 2)]:
        with pytest.raises(bs.BsError) as ei:
            bs.bs_sector_build(*args)
        assert ei.value.status == bs.BS_ERR_ARG
