"""GPU parity at BASELINE.json's full sizes, in the launch configuration bench.py times.

configs[2] (28 qubits): 100 Taylor-12 steps, norm and energy conservation to 1e-10 (reading U9: fixed
spectral shift, Rayleigh quotient), plus the first step against the oracle's own Taylor step.
configs[3], configs[4] (32 / 56 qubits): the oracle needs minutes to hours for the full vector, so its full-vector
energy, per-row functionals of H psi and 65,536 sampled amplitudes (by the term-by-term definition) are stored under
tests/golden/ by a script that calls only oracle/ (make_fullsize_golden.py); complete alpha rows are evaluated live.
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


def _golden_module():
    """tests/golden/make_fullsize_golden.py as a module (for its seeded sample_targets)."""
    import importlib.util
    import os
    path = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden", "make_fullsize_golden.py")
    spec = importlib.util.spec_from_file_location("make_fullsize_golden", path)
    mod = importlib.util.module_from_spec(spec)
    spec.loader.exec_module(mod)
    return mod


def _golden(name):
    """Full-size goldens written from oracle/ only by tests/golden/make_fullsize_golden.py (H psi) and
    tests/golden/make_rotation_golden.py (the *_rot files); see their docstrings."""
    import os
    path = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden", f"fullsize_{name}.npz")
    if not os.path.exists(path):
        script = "make_rotation_golden.py" if name.endswith("_rot") else f"make_fullsize_golden.py {name}"
        pytest.skip(f"{path} not generated yet (minutes to hours of oracle time): run tests/golden/{script}")
    return np.load(path)


@pytest.mark.parametrize("name", ["q24", "q32", "q56"])
def test_full_size_against_oracle_goldens(bs, name):
    """configs[1], [3], [4] in the launch configuration bench.py times (operator from the device-side JW route):
    energy to 1e-10 against the oracle's full-vector energy, EVERY alpha row through two functionals of H psi
    (sum_j conj(psi) H psi and sum_j |H psi|^2 per row) against the oracle's, 65,536 sampled amplitudes against
    the term-by-term definition, 4 complete alpha rows (first, last, middle, one random) against the oracle's slab
    mode evaluated live, Hermiticity with an independent vector."""
    import torch
    from oracle import oracle as orc
    gold_mod = _golden_module()
    gold = _golden(name)
    cfg = si.CONFIGS[name]
    ref = oracle_operator(name)
    h, g = si.integrals(cfg.n_orb, cfg.seed_ints)
    op = bs.bs_jw_molecular(h, g)                              # the route bench.py times
    xg, offs, zz, cc, _ = op.export()
    assert np.array_equal(zz, ref.z) and np.array_equal(np.repeat(xg, np.diff(offs)), ref.x)   # bit-exact tables
    assert np.abs(cc - ref.c).max() <= 1e-13 * np.abs(ref.c).max()
    sec, osec = bs.bs_sector_build(cfg.n_orb, cfg.n_alpha, cfg.n_beta), orc.Sector(cfg.n_orb, cfg.n_alpha, cfg.n_beta)
    psi = si.random_state(cfg.dim, cfg.seed_psi)
    d_in = torch.from_numpy(psi).cuda()
    d_out = torch.empty_like(d_in)
    bs.bs_apply(op, sec, d_in, d_out)
    Da, Db = osec.dim_alpha, osec.dim_beta
    # energy (north star: 1e-10 Hartree absolute) and its imaginary part
    e = bs.bs_expect(op, sec, d_in)
    e_gold = complex(gold["energy"][0], gold["energy"][1])
    assert abs(e - e_gold) <= 1e-10 and abs(e.imag) <= 1e-10
    assert abs(e - bs.bs_vdot(sec, d_in, d_out)) <= 1e-10
    # every alpha row: two functionals of H psi against the oracle's (relative to the row's own scale)
    row_e = (d_in.view(Da, Db).conj() * d_out.view(Da, Db)).sum(1).cpu().numpy()
    row_n2 = (d_out.view(Da, Db).abs() ** 2).sum(1).cpu().numpy()
    scale = np.sqrt(gold["row_n2"] * (np.abs(psi.reshape(Da, Db)) ** 2).sum(1))     # Cauchy-Schwarz bound of |row_e|
    assert np.abs(row_e - gold["row_e"]).max() <= 1e-12 * scale.max()
    assert np.abs(row_n2 - gold["row_n2"]).max() <= 1e-12 * gold["row_n2"].max()
    assert abs(float(row_n2.sum()) - float(gold["hnorm2"])) <= 1e-11 * float(gold["hnorm2"])
    # 65,536 sampled amplitudes against the definition (stored), 512 of them re-evaluated live by the oracle
    targets = gold_mod.sample_targets(cfg.dim)
    got = d_out[torch.from_numpy(targets).cuda()].cpu().numpy()
    assert rel_l2(got, gold["sample_val"]) <= 1e-12
    live = targets[:: len(targets) // 512]
    assert rel_l2(osec.apply_sampled(ref, psi, live), gold["sample_val"][:: len(targets) // 512]) <= 1e-13
    # 4 complete alpha rows, element by element
    rng = np.random.default_rng(11)
    for r in (0, Da - 1, Da // 2, int(rng.integers(1, Da - 1))):
        want_row = osec.apply_grouped_slab(ref, psi, r, r + 1).reshape(-1)
        assert rel_l2(d_out[r * Db:(r + 1) * Db].cpu().numpy(), want_row) <= 1e-12
    # Hermiticity with an independent phi
    phi = torch.from_numpy(si.random_state(cfg.dim, cfg.seed_psi + 7)).cuda()
    lhs = bs.bs_vdot(sec, phi, d_out)                        # <phi|H psi>
    bs.bs_apply(op, sec, phi, d_out)
    rhs = bs.bs_vdot(sec, d_out, d_in)                       # <H phi|psi>
    assert abs(lhs - rhs) <= 1e-10


def test_q32_uccsd_rotations(bs):
    """a6 beyond 24 qubits (Table 2 "Trotter" column): at D_beta = 12,870 a row pair no longer
    fits shared memory, so runs of generators go through the pair-list kernel, one launch per generator.
    (i) 16 orbitals, (2, 8) electrons (D_beta = 12,870 as in configs[3], D = 1.5e6 so that the single-threaded oracle
    finishes): 600 of its 2,759 UCCSD generators, in list order, on a random state, full-vector comparison with the
    oracle's fermionic Givens rotations.  (ii) configs[3] itself, all 5,792 generators (43,264 Pauli strings): norm, and
    (iii) the rotated vector against the oracle's result for the whole list (stored golden)."""
    import torch
    from oracle import oracle as orc
    from paper_2606_28952_b200 import jw_terms as jw
    n, na, nb = 16, 2, 8
    ex = si.uccsd_excitations(n, na, nb)
    assert len(ex) == 2759
    th_all = si.thetas(len(ex), 3004)
    rng = np.random.default_rng(21)
    pick = sorted(set(range(300)) | set(rng.choice(len(ex), 300, replace=False).tolist()))
    sub = [ex[i] for i in pick]
    th = th_all[pick]
    X, Z, Cc, offs = jw.excitation_generator_terms(sub)
    gens = bs.bs_group_xmask(X, Z, Cc, 2 * n, 0.0, bs.BS_MODE_SEQUENCE, offs)
    sec, osec = bs.bs_sector_build(n, na, nb), orc.Sector(n, na, nb)
    psi = si.random_state(osec.dim, 77)
    d = torch.from_numpy(psi).cuda()
    bs.bs_apply_pauli_rotations(gens, sec, th, d)
    for (cre, ann), t in zip(sub, th):
        osec.rot_fermionic(psi, cre, ann, t)
    assert rel_l2(d.cpu().numpy(), psi) <= 1e-12
    del gens, d
    cfg = si.CONFIGS["q32"]
    ex = si.uccsd_excitations(cfg.n_orb, cfg.n_alpha, cfg.n_beta)
    assert len(ex) == 5792
    X, Z, Cc, offs = jw.excitation_generator_terms(ex)
    gens = bs.bs_group_xmask(X, Z, Cc, cfg.n_qubits, 0.0, bs.BS_MODE_SEQUENCE, offs)
    sec = bs.bs_sector_build(cfg.n_orb, cfg.n_alpha, cfg.n_beta)
    d = torch.from_numpy(si.random_state(cfg.dim, cfg.seed_psi)).cuda()
    bs.bs_apply_pauli_rotations(gens, sec, si.thetas(len(ex), 3004), d)
    assert abs(np.sqrt(bs.bs_vdot(sec, d, d).real) - 1.0) <= 1e-10
    # (iii) the rotated vector against the oracle's fermionic Givens rotations over the WHOLE list
    # (tests/golden/make_rotation_golden.py, oracle/ only): every row and column through its complex sum, every row
    # through its norm, 65,536 sampled amplitudes and four complete rows element by element
    z = _golden("q32_rot")
    assert int(z["n_generators"]) == len(ex) and int(z["theta_seed"]) == 3004
    d2 = d.view(cfg.dim_alpha, cfg.dim_beta)
    assert rel_l2(d2.sum(dim=1).cpu().numpy(), z["row_sum"]) <= 1e-11
    assert rel_l2(d2.sum(dim=0).cpu().numpy(), z["col_sum"]) <= 1e-11
    assert rel_l2((d2.real ** 2 + d2.imag ** 2).sum(dim=1).cpu().numpy(), z["row_n2"]) <= 1e-12
    idx = torch.from_numpy(z["sample_idx"]).cuda()
    assert rel_l2(d[idx].cpu().numpy(), z["sample_val"]) <= 1e-12
    rows = torch.from_numpy(z["rows"]).cuda()
    assert rel_l2(d2[rows].cpu().numpy(), z["row_val"]) <= 1e-12
