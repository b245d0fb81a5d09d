"""GPU parity at BASELINE.json's full sizes, in the launch configuration bench.py times.

configs[2] (28 qubits): 100 Taylor-12 steps, norm and energy conservation to 1e-10 (reading U9: fixed
spectral shift, Rayleigh quotient), plus the first step against the oracle's own Taylor step.
configs[3], configs[4] (32 / 56 qubits): the oracle cannot form the full vector in seconds, so the
definition is evaluated per sampled target (orc_apply_sampled visits every string for every sampled
target) and on complete alpha rows (fast mode, itself pinned to the definition by P12); Hermiticity
<phi|H psi> = conj(<H phi|psi>) and <psi|H|psi> = vdot(psi, H psi) hold at any size.
"""
import numpy as np
import pytest

import synth_inputs as si
from common import oracle_operator, raw_terms, rel_l2

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def bs():
    from paper_2606_28952_b200 import bs as _bs
    return _bs


def test_q28_hubbard_taylor_100_steps(bs):
    import torch
    from oracle import oracle as orc
    cfg = si.CONFIGS["q28_hubbard"]
    op = bs.bs_group_xmask(*raw_terms("q28_hubbard"), 28, 1e-12)
    sec = bs.bs_sector_build(14, 7, 7)
    psi0 = si.random_state(cfg.dim, cfg.seed_psi)
    d = torch.from_numpy(psi0).cuda()
    work = torch.empty(2 * sec.dim, dtype=torch.complex128, device="cuda")
    e0 = bs.bs_expect(op, sec, d).real
    bs.bs_taylor_step(op, sec, d, work, 0.05, 12, e0)
    # first step vs the oracle's Taylor step (12 oracle applies)
    ref = oracle_operator("q28_hubbard")
    osec = orc.Sector(14, 7, 7)
    want = psi0.copy()
    osec.taylor_step(ref, want, 0.05, 12, e0)
    assert rel_l2(d.cpu().numpy(), want) <= 1e-12
    for _ in range(99):
        bs.bs_taylor_step(op, sec, d, work, 0.05, 12, e0)
    nrm2 = bs.bs_vdot(sec, d, d).real
    e = bs.bs_expect(op, sec, d)
    assert abs(np.sqrt(nrm2) - 1.0) <= 1e-10
    assert abs(e.real / nrm2 - e0) <= 1e-10                 # Rayleigh quotient (reading U9)
    assert abs(e.imag) <= 1e-10


@pytest.mark.parametrize("name,n_samples,n_rows", [("q32", 4096, 2), ("q56", 256, 1)])
def test_full_size_sampled(bs, name, n_samples, n_rows):
    import torch
    from oracle import oracle as orc
    cfg = si.CONFIGS[name]
    ref = oracle_operator(name)
    op = bs.bs_group_xmask(*raw_terms(name), cfg.n_qubits, 1e-12)
    xg, offs, zz, cc, _ = op.export()
    assert np.array_equal(zz, ref.z) and np.array_equal(np.repeat(xg, np.diff(offs)), ref.x)   # bit-exact tables
    assert np.abs(cc - ref.c).max() <= 1e-13 * np.abs(ref.c).max()
    sec, osec = bs.bs_sector_build(cfg.n_orb, cfg.n_alpha, cfg.n_beta), orc.Sector(cfg.n_orb, cfg.n_alpha, cfg.n_beta)
    psi = si.random_state(cfg.dim, cfg.seed_psi)
    d_in = torch.from_numpy(psi).cuda()
    d_out = torch.empty_like(d_in)
    bs.bs_apply(op, sec, d_in, d_out)
    rng = np.random.default_rng(9)
    targets = np.sort(rng.integers(0, cfg.dim, n_samples))
    got = d_out[torch.from_numpy(targets).cuda()].cpu().numpy()
    want = osec.apply_sampled(ref, psi, targets)
    assert rel_l2(got, want) <= 1e-12
    Db = osec.dim_beta
    rows = [0, osec.dim_alpha - 1, osec.dim_alpha // 2][:n_rows]
    for r in rows:
        want_row = osec.apply_sampled(ref, psi, np.arange(r * Db, (r + 1) * Db, max(1, Db // 128), dtype=np.int64))
        got_row = d_out[r * Db:(r + 1) * Db:max(1, Db // 128)].cpu().numpy()
        assert rel_l2(got_row, want_row) <= 1e-12
    e = bs.bs_expect(op, sec, d_in)
    assert abs(e - bs.bs_vdot(sec, d_in, d_out)) <= 1e-10 and abs(e.imag) <= 1e-10
    # Hermiticity with an independent phi
    phi = torch.from_numpy(si.random_state(cfg.dim, cfg.seed_psi + 7)).cuda()
    lhs = bs.bs_vdot(sec, phi, d_out)                        # <phi|H psi>
    bs.bs_apply(op, sec, phi, d_out)
    rhs = bs.bs_vdot(sec, d_out, d_in)                       # <H phi|psi>
    assert abs(lhs - rhs) <= 1e-10
