"""GPU parity of every apply-kernel path against the oracle on the same operators.

The library picks its path per (operator, sector): v2 row kernel (default), windowed source rows when a
row exceeds shared memory, beta-only groups on the transposed problem or in-row, and the v1 kernel as
fallback.  The environment switches below (read when a plan is built) force each path on sizes the
definition-mode oracle finishes in seconds; each runs in a fresh interpreter because plans are cached.
"""
import os
import subprocess
import sys

import pytest

pytestmark = pytest.mark.gpu
ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

SCRIPT = r"""
import sys, os
sys.path.insert(0, sys.argv[1]); sys.path.insert(0, os.path.join(sys.argv[1], 'tests'))
import numpy as np, torch
import synth_inputs as si
from common import oracle_operator, raw_terms, rel_l2
from oracle import oracle as orc
from paper_2606_28952_b200 import bs, jw_terms as jw
want_kernel = sys.argv[2]
rng = np.random.default_rng(3)
cases = []
for name in ('q12', 'q24'):
    cfg = si.CONFIGS[name]
    cases.append((name, oracle_operator(name), raw_terms(name), cfg.n_orb, cfg.n_alpha, cfg.n_beta))
ref8 = orc.hubbard_h(8, 1.0, 4.0)
cases.append(('hub8', ref8, jw.hubbard_raw_terms(8, 1.0, 4.0), 8, 4, 3))
ref10 = orc.hubbard_h(10, 1.0, 4.0)
cases.append(('hub10', ref10, jw.hubbard_raw_terms(10, 1.0, 4.0), 10, 5, 4))     # light path (D_beta = 210 >= 64)
cases.append(('hub10h', ref10, jw.hubbard_raw_terms(10, 1.0, 4.0), 10, 5, 5))    # light path, list slots by table (l_max = 9 bonds)
h, g = si.integrals(7, 77)
cases.append(('mol7', orc.molecular_h(h, g), jw.molecular_raw_terms(h, g), 7, 2, 5))
h, g = si.integrals(9, 79)                                                          # n = 9 pads the K-resolved kernel's 12 columns
cases.append(('mol9', orc.molecular_h(h, g), jw.molecular_raw_terms(h, g), 9, 3, 5))
cases.append(('mol9b', orc.molecular_h(h, g), jw.molecular_raw_terms(h, g), 9, 4, 2))
# two list-mode alpha masks sharing one column list, the second uniform but owning only a SUBSET of the listed tables
# (n = 10: NN and NNN beta hops with one weight under x_a = 0; V * (alpha hop 0-1) * (NN beta hop j) under x_a = {0,1})
def _hop(P, Q, scale):
    a = orc.ladder_product([P, Q], [1, 0], scale); b = orc.ladder_product([Q, P], [1, 0], scale)
    return [a, b]
parts = []
for j in range(9): parts += _hop(10 + j, 11 + j, -1.0)
for j in range(8): parts += _hop(10 + j, 12 + j, -1.0)
for j in range(9):
    for (P, Q) in ((0, 1), (1, 0)):
        for (R, S) in ((10 + j, 11 + j), (11 + j, 10 + j)):
            parts.append(orc.ladder_product([P, Q, R, S], [1, 0, 1, 0], 0.7))
tl = (np.concatenate([p.x for p in parts]), np.concatenate([p.z for p in parts]), np.concatenate([p.c for p in parts]))
# chain with nearest- and next-nearest-neighbour hops of equal weight on both spins + U n n: light-shaped, and the NNN
# hops carry a JW sign (Z on the site in between), so the light kernel's signed list entries are exercised
parts = []
for sp in (0, 10):
    for j in range(9): parts += _hop(sp + j, sp + j + 1, -1.0)
    for j in range(8): parts += _hop(sp + j, sp + j + 2, -1.0)
for j in range(10): parts.append(orc.ladder_product([j, j, 10 + j, 10 + j], [1, 0, 1, 0], 4.0))
nnn = (np.concatenate([p.x for p in parts]), np.concatenate([p.z for p in parts]), np.concatenate([p.c for p in parts]))
# generic complex operator (multi-key, POPC signs, complex weights)
M = 400
x = rng.integers(0, 1 << 12, M, dtype=np.uint64); x[:60] = 0; x[60:150] = 0b000011; x[150:260] = 0b000101000011
x[260:300] = 0b011000000000
z = rng.integers(0, 1 << 12, M, dtype=np.uint64)
c = rng.standard_normal(M) + 1j * rng.standard_normal(M)
for name, ref, raw, n, na, nb in cases + [('generic', None, (x, z, c), 6, 3, 2), ('twolist', None, tl, 10, 5, 5),
                                        ('hubnnn', None, nnn, 10, 5, 4)]:
    op = bs.bs_group_xmask(*raw, 2 * n, 1e-12 if ref is not None else 0.0)
    if ref is None:
        xg, offs, zz, cc, _ = op.export()
        ref = orc.PauliOp(np.repeat(xg, np.diff(offs)), zz, cc)
    sec, osec = bs.bs_sector_build(n, na, nb), orc.Sector(n, na, nb)
    desc = bs.bs_plan_describe(op, sec)
    assert want_kernel in desc or want_kernel == 'kres{', (want_kernel, desc)
    if name in ('q24', 'mol9') and want_kernel in ('rows_v2', 'kres{'):
        assert ('kres{' in desc) == (os.environ.get('BS_NO_KRES') is None), desc
        assert ('k2{' in desc and 'k2_t{' in desc) == (os.environ.get('BS_NO_K2') is None), desc
    if name in ('hub10', 'hub10h', 'hubnnn') and want_kernel == 'rows_v2':
        assert ('+light' in desc) == (os.environ.get('BS_NO_LIGHT') is None), desc
    psi = si.random_state(osec.dim, 5)
    want = osec.apply_grouped(ref, psi) if osec.dim > 100000 else osec.apply(ref, psi)
    d_in = torch.from_numpy(psi).cuda(); d_out = torch.full_like(d_in, float('nan'))
    bs.bs_apply(op, sec, d_in, d_out)
    err = rel_l2(d_out.cpu().numpy(), want)
    e = bs.bs_expect(op, sec, d_in)
    de = abs(e - orc.vdot(psi, want))
    # row slab + fused epilogue on the same path
    lo, hi = osec.dim_alpha // 3, (2 * osec.dim_alpha) // 3 + 1
    d_slab = torch.zeros_like(d_in); bs.bs_apply_rows(op, sec, d_in, d_slab, lo, hi)
    slab = d_slab.cpu().numpy(); Db = osec.dim_beta
    err_s = rel_l2(slab[lo * Db:hi * Db], want[lo * Db:hi * Db])
    assert np.all(slab[:lo * Db] == 0) and np.all(slab[hi * Db:] == 0)
    acc0 = si.random_state(osec.dim, 6); d_acc = torch.from_numpy(acc0).cuda(); d_o2 = torch.zeros_like(d_in)
    bs.bs_apply_axpby(op, sec, d_in, d_o2, 0.5 - 2j, 1.5j, d_acc)
    w2 = (0.5 - 2j) * want + 1.5j * psi
    err_a = max(rel_l2(d_o2.cpu().numpy(), w2), rel_l2(d_acc.cpu().numpy(), acc0 + w2))
    print(name, desc.split(' ')[0], f"{err:.2e} {de:.2e} {err_s:.2e} {err_a:.2e}")
    assert err <= 1e-12 and de <= 1e-10 and err_s <= 1e-12 and err_a <= 1e-12, (name, err, de, err_s, err_a)
print('PATH OK')
"""


@pytest.mark.parametrize("env,kernel", [
    ({}, "rows_v2"),
    ({"BS_NO_LIGHT": "1", "BS_NO_KRES": "1", "BS_NO_K2": "1", "BS_NO_CDIAG": "1"}, "rows_v2"),   # column-list pass and row axpys only
    ({"BS_K2_SLAB_MB": "1", "BS_K2_MIN": "1", "BS_NO_HOPSPLIT": "1"}, "kres{"),              # several column slabs of the K2 scratch
    ({"BS_KRES_KC": "64", "BS_KRES_SLAB_MB": "2", "BS_K2_MMA": "0"}, "kres{"),   # more K chunks, several scratch slabs, DFMA k_aa
    ({"BS_KRES_KC": "32", "BS_KRES_MIN": "1", "BS_KRES_MMA": "0"}, "kres{"),   # DFMA form of the K-resolved contraction
    ({"BS_KRES_STAGES": "3", "BS_KRES_MIN": "1"}, "kres{"),                    # three pipeline buffers in k_ab (default: two)
    ({"BS_KRES_STAGES": "3", "BS_KRES_KC": "64", "BS_KRES_MMA": "0"}, "kres{"),
    ({"BS_KRES_BIG": "1", "BS_KRES_MIN": "1"}, "kres{"),                       # the 16-compute-warp (96-register) build of k_ab
    ({"BS_KRES_BIG": "1", "BS_KRES_KC": "96", "BS_KRES_STAGES": "3"}, "kres{"),
    ({"BS_K2_NT": "2", "BS_K2_MIN": "1"}, "kres{"),   # k_aa_mma target tiles of 16 / 24 / 32: <2, 4, 1>, <3, 2, 3>, <4, 2, 3>
    ({"BS_K2_NT": "3", "BS_K2_MIN": "1", "BS_K2_SLAB_MB": "1"}, "kres{"),
    ({"BS_K2_NT": "4", "BS_K2_MIN": "1"}, "kres{"),
    ({"BS_K2_NO_CTILE": "1", "BS_K2_MIN": "1"}, "kres{"),   # coupling tiles evaluated inside k_aa_mma instead of at plan time
    ({"BS_LIGHT_COMPACT": "1", "BS_LIGHT_ORDER": "0", "BS_LIGHT_SIGN": "1"}, "rows_v2"),   # light kernel: compacted list, one phase order, signed entries
    ({"BS_LIGHT_ORDER": "1", "BS_LIGHT_THREADS": "1024"}, "rows_v2"),
    ({"BS_KERNEL": "v1"}, "sector_v1"),
    ({"BS_KERNEL": "v2inrow"}, "kernel="),      # q24's beta-only groups do not fit in-row: falls back to v1 there
    ({"BS_ROW_WIN": "24"}, "n_win="),                                  # windowed rows, one column list per window
    ({"BS_ROW_WIN": "24", "BS_ROW_NO_SPLIT": "1"}, "n_win="),          # windowed rows, one list with a window test
    ({"BS_ROW_WIN": "24", "BS_KERNEL": "v2inrow"}, "kernel="),
])
def test_kernel_path(env, kernel):
    e = dict(os.environ)
    e.update(env)
    r = subprocess.run([sys.executable, "-c", SCRIPT, ROOT, kernel], env=e, capture_output=True, text=True, timeout=900)
    assert r.returncode == 0 and "PATH OK" in r.stdout, r.stdout[-3000:] + r.stderr[-3000:]


def test_wide_beta_space_uses_v1_fallback():
    """D_beta > 32767 does not fit the u16 column tables: the v1 kernel must take over and stay exact."""
    import numpy as np
    import torch

    import synth_inputs as si
    from common import rel_l2
    from oracle import oracle as orc
    from paper_2606_28952_b200 import bs
    L = 18
    op = bs.bs_jw_hubbard(L, 1.0, 4.0)
    ref = orc.hubbard_h(L, 1.0, 4.0)
    sec, osec = bs.bs_sector_build(L, 1, 9), orc.Sector(L, 1, 9)
    assert osec.dim_beta == 48620 and "sector_v1" in bs.bs_plan_describe(op, sec)
    psi = si.random_state(osec.dim, 12)
    want = osec.apply_grouped(ref, psi)
    d_in = torch.from_numpy(psi).cuda()
    d_out = torch.empty_like(d_in)
    bs.bs_apply(op, sec, d_in, d_out)
    assert rel_l2(d_out.cpu().numpy(), want) <= 1e-12
    assert abs(bs.bs_expect(op, sec, d_in) - orc.vdot(psi, want)) <= 1e-10
    # the mirrored sector (wide alpha space) also falls back
    sec2, osec2 = bs.bs_sector_build(L, 9, 1), orc.Sector(L, 9, 1)
    assert "sector_v1" in bs.bs_plan_describe(op, sec2)
    psi2 = si.random_state(osec2.dim, 13)
    d2 = torch.from_numpy(psi2).cuda()
    o2 = torch.empty_like(d2)
    bs.bs_apply(op, sec2, d2, o2)
    assert rel_l2(o2.cpu().numpy(), osec2.apply_grouped(ref, psi2)) <= 1e-12
