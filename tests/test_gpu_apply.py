"""GPU parity, floating-point work: a4 apply, a5 expectation, a6 rotations, a7 Taylor vs the oracle.

Bars (BASELINE.json north_star): H|psi> <= 1e-12 relative L2; energies <= 1e-10 absolute.
Sizes here are ones the definition-mode oracle finishes in seconds (configs 1-3 and small cases);
the full-size configs 4-5 are in test_gpu_fullsize.py.
"""
import numpy as np
import pytest

import synth_inputs as si
from common import oracle_operator, raw_terms, rel_l2, to_device, to_host

pytestmark = pytest.mark.gpu

TOL_L2 = 1e-12
TOL_E = 1e-10


@pytest.fixture(scope="module")
def bs():
    from paper_2606_28952_b200 import bs as _bs
    return _bs


@pytest.fixture(scope="module")
def orc():
    from oracle import oracle as _o
    return _o


def _gpu_op(bs, name):
    cfg = si.CONFIGS[name]
    x, z, c = raw_terms(name)
    return bs.bs_group_xmask(x, z, c, cfg.n_qubits, 1e-12)


def _apply(bs, op, sec, psi_np):
    import torch
    d_in = to_device(psi_np)
    d_out = torch.full_like(d_in, complex(np.nan, np.nan))
    bs.bs_apply(op, sec, d_in, d_out)
    torch.cuda.synchronize()
    return to_host(d_out), d_in


def test_q12_sector_and_full_space(bs, orc):
    cfg = si.CONFIGS["q12"]
    ref = oracle_operator("q12")
    op = _gpu_op(bs, "q12")
    # sector (dim 400)
    osec = orc.Sector(6, 3, 3)
    sec = bs.bs_sector_build(6, 3, 3)
    psi = si.random_state(cfg.dim, cfg.seed_psi)
    want = osec.apply(ref, psi)
    got, d_psi = _apply(bs, op, sec, psi)
    assert rel_l2(got, want) <= TOL_L2
    e = bs.bs_expect(op, sec, d_psi)
    assert abs(e - orc.vdot(psi, want)) <= TOL_E and abs(e.imag) <= TOL_E
    # full 4096-dim space, state embedded from the sector plus a generic full-space state
    ofull = orc.Sector(12)
    full = bs.bs_sector_build(12)
    psi_f = si.random_state(4096, cfg.seed_psi + 1)
    want_f = ofull.apply(ref, psi_f)
    got_f, d_f = _apply(bs, op, full, psi_f)
    assert rel_l2(got_f, want_f) <= TOL_L2
    assert abs(bs.bs_expect(op, full, d_f) - orc.vdot(psi_f, want_f)) <= TOL_E
    a, b = osec.strings()
    cfgs = (a[:, None] | (b[None, :] << np.uint64(6))).ravel()
    emb = np.zeros(4096, np.complex128)
    emb[cfgs.astype(np.int64)] = psi
    got_e, _ = _apply(bs, op, full, emb)
    assert rel_l2(got_e[cfgs.astype(np.int64)], want) <= TOL_L2     # sector = restriction of full space
    mask = np.ones(4096, bool)
    mask[cfgs.astype(np.int64)] = False
    assert np.abs(got_e[mask]).max() <= 1e-13                       # H conserves (N_alpha, N_beta)


@pytest.mark.parametrize("mode", ["sector", "full"])
def test_odd_ny_operator_phase_convention(bs, orc, mode):
    """Reading U2: a UCC generator (every ny odd) through bs_apply; i^{ny} on the target would flip the sign."""
    from paper_2606_28952_b200 import jw_terms as jw
    ex = si.uccsd_excitations(6, 3, 3)
    picks = [ex[1], ex[20], ex[-1], ex[len(ex) // 2]]
    X, Z, Cc, _ = jw.excitation_generator_terms(picks)
    op = bs.bs_group_xmask(X, Z, Cc, 12, 1e-14)
    x_all, z_all, c_all = [], [], []
    for cre, ann in picks:
        o = orc.excitation_generator(cre, ann)
        x_all.append(o.x), z_all.append(o.z), c_all.append(o.c)
    order = np.lexsort((np.concatenate(z_all), np.concatenate(x_all)))
    ref = orc.PauliOp(np.concatenate(x_all)[order], np.concatenate(z_all)[order], np.concatenate(c_all)[order])
    if mode == "sector":
        osec, sec, dim = orc.Sector(6, 3, 3), bs.bs_sector_build(6, 3, 3), 400
    else:
        osec, sec, dim = orc.Sector(12), bs.bs_sector_build(12), 4096
    psi = si.random_state(dim, 99)
    want = osec.apply(ref, psi)
    got, _ = _apply(bs, op, sec, psi)
    assert np.linalg.norm(want) > 0.1
    assert rel_l2(got, want) <= TOL_L2


def test_complex_coefficients_and_sector_projection(bs, orc):
    """Generic complex, non-number-conserving Pauli sum: bs_apply must give P_sector H P_sector psi."""
    rng = np.random.default_rng(5)
    M = 300
    x = rng.integers(0, 1 << 10, M, dtype=np.uint64)
    x[:40] = 0
    x[40:80] = np.uint64(0b0000000011)           # alpha single excitation 0 <-> 1
    x[80:120] = np.uint64(0b0011000011)          # alpha 0 <-> 1 and beta 1 <-> 2
    x[120:140] = np.uint64(0b1111000000)         # beta double excitation
    z = rng.integers(0, 1 << 10, M, dtype=np.uint64)
    c = rng.standard_normal(M) + 1j * rng.standard_normal(M)
    op = bs.bs_group_xmask(x, z, c, 10, 0.0)
    xg, offs, zz, cc, _ = op.export()
    ref = orc.PauliOp(np.repeat(xg, np.diff(offs)), zz, cc)
    for (na, nb) in [(2, 3), (0, 5), (5, 5), (1, 1)]:
        osec, sec = orc.Sector(5, na, nb), bs.bs_sector_build(5, na, nb)
        psi = si.random_state(osec.dim, 11 + na)
        got, d_psi = _apply(bs, op, sec, psi)
        want = osec.apply(ref, psi)
        assert rel_l2(got, want) <= TOL_L2
        assert abs(bs.bs_expect(op, sec, d_psi) - orc.vdot(psi, want)) <= TOL_E
    ofull, full = orc.Sector(10), bs.bs_sector_build(10)
    psi = si.random_state(1024, 3)
    got, _ = _apply(bs, op, full, psi)
    assert rel_l2(got, ofull.apply(ref, psi)) <= TOL_L2


def test_apply_argument_errors(bs):
    import torch
    op = _gpu_op(bs, "q12")
    sec = bs.bs_sector_build(6, 3, 3)
    psi = torch.zeros(400, dtype=torch.complex128, device="cuda")
    with pytest.raises(bs.BsError) as ei:
        bs._check(bs._lib.bs_apply(op._h, sec._h, psi.data_ptr(), psi.data_ptr(), None))
    assert ei.value.status == bs.BS_ERR_ARG
    sec7 = bs.bs_sector_build(7, 3, 3)
    big = torch.zeros(sec7.dim, dtype=torch.complex128, device="cuda")
    with pytest.raises(bs.BsError) as ei:
        bs.bs_apply(op, sec7, big, torch.zeros_like(big))
    assert ei.value.status == bs.BS_ERR_MISMATCH
    with pytest.raises(bs.BsError):
        bs._check(bs._lib.bs_apply(op._h, sec._h, psi.data_ptr() + 8, psi.data_ptr(), None))


def test_apply_rows_writes_only_its_slab(bs, orc):
    import torch
    ref = oracle_operator("q12")
    op = _gpu_op(bs, "q12")
    osec, sec = orc.Sector(6, 3, 3), bs.bs_sector_build(6, 3, 3)
    psi = si.random_state(400, 1)
    want = osec.apply(ref, psi)
    d_in = to_device(psi)
    d_out = torch.full_like(d_in, 7.0)
    bs.bs_apply_rows(op, sec, d_in, d_out, 3, 11)
    got = to_host(d_out)
    assert np.all(got[:60] == 7.0) and np.all(got[220:] == 7.0)
    assert rel_l2(got[60:220], want[60:220]) <= TOL_L2
    bs.bs_apply_rows(op, sec, d_in, d_out, 5, 5)           # empty slab is a no-op
    with pytest.raises(bs.BsError):
        bs.bs_apply_rows(op, sec, d_in, d_out, 5, 21)


def test_apply_axpby_and_vdot(bs, orc):
    import torch
    ref = oracle_operator("q12")
    op = _gpu_op(bs, "q12")
    osec, sec = orc.Sector(6, 3, 3), bs.bs_sector_build(6, 3, 3)
    psi, acc0 = si.random_state(400, 1), si.random_state(400, 2)
    hp = osec.apply(ref, psi)
    alpha, beta = 0.3 - 0.7j, -1.1 + 0.2j
    d_in, d_out, d_acc = to_device(psi), torch.zeros(400, dtype=torch.complex128, device="cuda"), to_device(acc0)
    bs.bs_apply_axpby(op, sec, d_in, d_out, alpha, beta, d_acc)
    want = alpha * hp + beta * psi
    assert rel_l2(to_host(d_out), want) <= TOL_L2
    assert rel_l2(to_host(d_acc), acc0 + want) <= TOL_L2
    v = bs.bs_vdot(sec, d_in, d_out)
    assert abs(v - orc.vdot(psi, want)) <= TOL_E
    v2 = bs.bs_vdot(sec, d_in, d_out)
    assert v == v2                                         # deterministic reduction


def test_q24_uccsd_state_apply_energy(bs, orc):
    """Config 2: HF -> 1,818 grouped Pauli rotations (GPU) vs fermionic Givens rotations (oracle), then
    H|psi> and the energy."""
    import torch
    from paper_2606_28952_b200 import jw_terms as jw
    cfg = si.CONFIGS["q24"]
    ex = si.uccsd_excitations(cfg.n_orb, cfg.n_alpha, cfg.n_beta)
    assert len(ex) == 1818
    th = si.thetas(len(ex), cfg.seed_theta)
    X, Z, Cc, offs = jw.excitation_generator_terms(ex)
    assert len(X) == 14112
    gens = bs.bs_group_xmask(X, Z, Cc, 24, 0.0, bs.BS_MODE_SEQUENCE, offs)
    sec, osec = bs.bs_sector_build(12, 6, 6), orc.Sector(12, 6, 6)
    psi = np.zeros(cfg.dim, np.complex128)
    psi[0] = 1.0                                           # HF determinant = sector index 0
    d_psi = to_device(psi)
    bs.bs_apply_pauli_rotations(gens, sec, th, d_psi)
    for (cre, ann), t in zip(ex, th):
        osec.rot_fermionic(psi, cre, ann, t)
    got = to_host(d_psi)
    assert abs(np.linalg.norm(got) - 1.0) <= 1e-12
    assert rel_l2(got, psi) <= TOL_L2
    ref = oracle_operator("q24")
    op = _gpu_op(bs, "q24")
    want = osec.apply_grouped(ref, psi)
    d_in = to_device(psi)
    d_out = torch.empty_like(d_in)
    bs.bs_apply(op, sec, d_in, d_out)
    assert rel_l2(to_host(d_out), want) <= TOL_L2
    samp = np.random.default_rng(0).integers(0, cfg.dim, 512)
    assert rel_l2(to_host(d_out)[samp], osec.apply_sampled(ref, psi, samp)) <= TOL_L2   # definition, per target
    e = bs.bs_expect(op, sec, d_in)
    assert abs(e - orc.vdot(psi, want)) <= TOL_E
    assert bs.bs_expect(op, sec, d_in) == e                # bit-reproducible


def test_rotations_small_and_errors(bs, orc):
    from paper_2606_28952_b200 import jw_terms as jw
    ex = si.uccsd_excitations(6, 3, 3)
    th = si.thetas(len(ex), 5, sd=0.4)
    X, Z, Cc, offs = jw.excitation_generator_terms(ex)
    gens = bs.bs_group_xmask(X, Z, Cc, 12, 0.0, bs.BS_MODE_SEQUENCE, offs)
    for osec, sec in [(orc.Sector(6, 3, 3), bs.bs_sector_build(6, 3, 3)), (orc.Sector(12), bs.bs_sector_build(12))]:
        psi = si.random_state(osec.dim, 8)
        d = to_device(psi)
        bs.bs_apply_pauli_rotations(gens, sec, th, d)
        for (cre, ann), t in zip(ex, th):
            osec.rot_fermionic(psi, cre, ann, t)
        assert rel_l2(to_host(d), psi) <= TOL_L2
        bs.bs_apply_pauli_rotations(gens, sec, np.zeros(len(ex)), d)      # theta = 0: identity
        assert rel_l2(to_host(d), psi) <= 1e-15
    # a generator that leaves the (3,3) sector: a^dag_0 - a_0 = -i Y_0
    leak = bs.bs_group_xmask(np.array([1], np.uint64), np.array([1], np.uint64), np.array([-1j]), 12, 0.0,
                             bs.BS_MODE_SEQUENCE, np.array([0, 1], np.int64))
    sec = bs.bs_sector_build(6, 3, 3)
    d = to_device(si.random_state(400, 1))
    with pytest.raises(bs.BsError) as ei:
        bs.bs_apply_pauli_rotations(leak, sec, np.array([0.1]), d)
    assert ei.value.status == bs.BS_ERR_LEAVES_SECTOR
    # non-commuting strings in one run: i X_0 X_1 (ny = 0) and i Y_0 X_1 (ny = 1)
    nc = bs.bs_group_xmask(np.array([3, 3], np.uint64), np.array([0, 1], np.uint64),
                           np.array([1j, 1j]), 12, 0.0, bs.BS_MODE_SEQUENCE, np.array([0, 2], np.int64))
    with pytest.raises(bs.BsError) as ei:
        bs.bs_apply_pauli_rotations(nc, sec, np.array([0.1]), d)
    assert ei.value.status == bs.BS_ERR_NOT_COMMUTING


def test_taylor_step_small_hubbard(bs, orc):
    import torch
    from paper_2606_28952_b200 import jw_terms as jw
    L = 8
    ref = orc.hubbard_h(L, 1.0, 4.0)
    op = bs.bs_group_xmask(*jw.hubbard_raw_terms(L, 1.0, 4.0), 2 * L, 1e-12)
    osec, sec = orc.Sector(L, 4, 4), bs.bs_sector_build(L, 4, 4)
    psi = si.random_state(osec.dim, 4)
    d = to_device(psi)
    work = torch.empty(2 * sec.dim, dtype=torch.complex128, device="cuda")
    e0 = bs.bs_expect(op, sec, d).real
    assert abs(e0 - orc.energy(osec, ref, psi).real) <= TOL_E
    for _ in range(5):
        bs.bs_taylor_step(op, sec, d, work, 0.05, 12, e0)
        osec.taylor_step(ref, psi, 0.05, 12, e0)
    assert rel_l2(to_host(d), psi) <= TOL_L2
    assert abs(bs.bs_vdot(sec, d, d).real - 1.0) <= 1e-12


@pytest.mark.parametrize("order", [2, 3, 4, 7, 12, 13])
def test_taylor_step_orders(bs, orc, order):
    """bs_taylor_step accumulates the terms in pairs (even launches add input + output): even and odd orders, the
    shortest ones included, on the light-kernel path (10 sites, 5 + 5) against the oracle's Eq. 6-7 loop."""
    import torch
    from paper_2606_28952_b200 import jw_terms as jw
    L = 10
    ref = orc.hubbard_h(L, 1.0, 4.0)
    op = bs.bs_group_xmask(*jw.hubbard_raw_terms(L, 1.0, 4.0), 2 * L, 1e-12)
    osec, sec = orc.Sector(L, 5, 5), bs.bs_sector_build(L, 5, 5)
    psi = si.random_state(osec.dim, 14)
    d = to_device(psi)
    work = torch.empty(2 * sec.dim, dtype=torch.complex128, device="cuda")
    e0 = bs.bs_expect(op, sec, d).real
    for _ in range(2):
        bs.bs_taylor_step(op, sec, d, work, 0.03, order, e0)
        osec.taylor_step(ref, psi, 0.03, order, e0)
    assert rel_l2(to_host(d), psi) <= TOL_L2


def test_q28_hubbard_single_apply(bs, orc):
    """Config 3 operator at full size: one apply vs the definition-mode oracle (95 terms x 1.2e7)."""
    cfg = si.CONFIGS["q28_hubbard"]
    ref = oracle_operator("q28_hubbard")
    op = _gpu_op(bs, "q28_hubbard")
    osec, sec = orc.Sector(14, 7, 7), bs.bs_sector_build(14, 7, 7)
    psi = si.random_state(cfg.dim, cfg.seed_psi)
    want = osec.apply(ref, psi)
    got, d_psi = _apply(bs, op, sec, psi)
    assert rel_l2(got, want) <= TOL_L2
    e = bs.bs_expect(op, sec, d_psi)
    assert abs(e - orc.vdot(psi, want)) <= TOL_E
    assert abs(e.real - 14.0) < 0.1                         # Tr H / D = U N_a N_b / L = 14 (pin P10)


def test_rotations_shuffled_order_and_per_launch_path(bs, orc):
    """Shuffled generator order breaks the runs that the closed-cell batching relies on: isolated generators take
    the per-generator kernel, short runs the cell kernels; BS_ROT_PER_LAUNCH=1 forces the per-generator path for
    the ordered list.  All must agree with the fermionic Givens oracle."""
    import os
    import subprocess
    import sys
    from paper_2606_28952_b200 import jw_terms as jw
    ex = si.uccsd_excitations(7, 3, 4)
    rng = np.random.default_rng(21)
    order = rng.permutation(len(ex))
    ex_s = [ex[i] for i in order]
    th = si.thetas(len(ex_s), 9, sd=0.3)
    X, Z, Cc, offs = jw.excitation_generator_terms(ex_s)
    gens = bs.bs_group_xmask(X, Z, Cc, 14, 0.0, bs.BS_MODE_SEQUENCE, offs)
    osec, sec = orc.Sector(7, 3, 4), bs.bs_sector_build(7, 3, 4)
    psi = si.random_state(osec.dim, 2)
    d = to_device(psi)
    bs.bs_apply_pauli_rotations(gens, sec, th, d)
    for (cre, ann), t in zip(ex_s, th):
        osec.rot_fermionic(psi, cre, ann, t)
    assert rel_l2(to_host(d), psi) <= TOL_L2
    code = (
        "import sys, os; sys.path.insert(0, sys.argv[1]); sys.path.insert(0, os.path.join(sys.argv[1], 'tests'))\n"
        "import numpy as np, torch, synth_inputs as si\n"
        "from oracle import oracle as orc\n"
        "from paper_2606_28952_b200 import bs, jw_terms as jw\n"
        "ex = si.uccsd_excitations(6, 3, 3); th = si.thetas(len(ex), 5, sd=0.4)\n"
        "X, Z, C, offs = jw.excitation_generator_terms(ex)\n"
        "g = bs.bs_group_xmask(X, Z, C, 12, 0.0, bs.BS_MODE_SEQUENCE, offs)\n"
        "sec, osec = bs.bs_sector_build(6, 3, 3), orc.Sector(6, 3, 3)\n"
        "psi = si.random_state(400, 8); d = torch.from_numpy(psi.copy()).cuda()\n"
        "n0 = bs.bs_launch_count(); bs.bs_apply_pauli_rotations(g, sec, th, d); n1 = bs.bs_launch_count()\n"
        "for (cre, ann), t in zip(ex, th): osec.rot_fermionic(psi, cre, ann, t)\n"
        "err = np.linalg.norm(d.cpu().numpy() - psi) / np.linalg.norm(psi)\n"
        "print('LAUNCHES', n1 - n0, 'ERR', err); assert err <= 1e-12\n")
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    counts = {}
    # BS_ROT_IN_PLACE: the cell kernels work on the state vector itself (the path of sectors whose cells exceed
    # shared memory, configs 4-5) -- same launch count as the shared-memory cells
    # BS_ROT_ORBIT=1: cells of {row pair} x {orbit of columns} (opt-in for sectors whose rows exceed shared memory)
    # BS_ROT_CLUSTER=2: every row-pair run on a cluster of two blocks, one row each, partners through distributed shared
    # memory (opt-in with =1 for sectors whose row pair exceeds one block's shared memory)
    for key, env in (("cells", {}), ("per_launch", {"BS_ROT_PER_LAUNCH": "1"}), ("in_place", {"BS_ROT_IN_PLACE": "1"}),
                     ("orbit", {"BS_ROT_ORBIT": "1"}), ("cluster", {"BS_ROT_CLUSTER": "2"}),
                     ("cstr", {"BS_ROT_CSTR": "1"}), ("in_place_table", {"BS_ROT_IN_PLACE": "1", "BS_ROT_CSTR": "0"})):
        r = subprocess.run([sys.executable, "-c", code, root], env=dict(os.environ, **env), capture_output=True,
                           text=True, timeout=600)
        assert r.returncode == 0, r.stdout[-2000:] + r.stderr[-2000:]
        counts[key] = int(r.stdout.split("LAUNCHES")[1].split()[0])
    assert counts["per_launch"] > 3 * counts["cells"]      # batching really reduces the launch count
    assert counts["in_place"] == counts["cells"]
    assert counts["cells"] <= counts["orbit"] < counts["per_launch"]
    assert counts["cluster"] == counts["cells"] == counts["cstr"] == counts["in_place_table"]


def test_apply_and_rotations_are_bit_reproducible(bs):
    """No floating-point atomics and a fixed summation order: repeated runs give identical bits (a shared-memory or
    global-memory race in the row kernel or the rotation cell kernels would show up here as run-to-run noise)."""
    import torch
    from paper_2606_28952_b200 import jw_terms as jw
    cfg = si.CONFIGS["q24"]
    op = _gpu_op(bs, "q24")
    sec = bs.bs_sector_build(12, 6, 6)
    d_in = to_device(si.random_state(cfg.dim, 17))
    ref_out = torch.empty_like(d_in)
    bs.bs_apply(op, sec, d_in, ref_out)
    out = torch.empty_like(d_in)
    for _ in range(10):
        out.fill_(float("nan"))
        bs.bs_apply(op, sec, d_in, out)
        assert torch.equal(torch.view_as_real(out), torch.view_as_real(ref_out))
    ex = si.uccsd_excitations(cfg.n_orb, cfg.n_alpha, cfg.n_beta)
    th = si.thetas(len(ex), cfg.seed_theta)
    X, Z, Cc, offs = jw.excitation_generator_terms(ex)
    gens = bs.bs_group_xmask(X, Z, Cc, 24, 0.0, bs.BS_MODE_SEQUENCE, offs)
    states = []
    for _ in range(4):
        psi = torch.zeros(cfg.dim, dtype=torch.complex128, device="cuda")
        psi[0] = 1.0
        bs.bs_apply_pauli_rotations(gens, sec, th, psi)
        states.append(psi)
    for s in states[1:]:
        assert torch.equal(torch.view_as_real(s), torch.view_as_real(states[0]))
    hub = bs.bs_jw_hubbard(10, 1.0, 4.0)
    hsec = bs.bs_sector_build(10, 5, 5)
    hin = to_device(si.random_state(hsec.dim, 3))
    h0 = torch.empty_like(hin)
    bs.bs_apply(hub, hsec, hin, h0)
    for _ in range(10):
        h1 = torch.empty_like(hin)
        bs.bs_apply(hub, hsec, hin, h1)
        assert torch.equal(torch.view_as_real(h1), torch.view_as_real(h0))


def test_degenerate_operators_and_sectors(bs, orc):
    """Empty operator, identity-only operator, one-dimensional sectors, fully occupied spin."""
    import torch
    e = np.zeros(0, np.uint64)
    op_empty = bs.bs_group_xmask(e, e, np.zeros(0, np.complex128), 12)
    op_id = bs.bs_group_xmask(np.zeros(1, np.uint64), np.zeros(1, np.uint64), np.array([2.5 - 1j]), 12)
    ref = oracle_operator("q12")
    op = _gpu_op(bs, "q12")
    for (na, nb) in [(3, 3), (0, 0), (6, 6), (6, 0), (0, 1), (5, 6)]:
        sec, osec = bs.bs_sector_build(6, na, nb), orc.Sector(6, na, nb)
        psi = si.random_state(osec.dim, 50 + na + nb)
        d_in = to_device(psi)
        d_out = torch.full_like(d_in, complex(np.nan, np.nan))
        bs.bs_apply(op_empty, sec, d_in, d_out)
        assert np.all(to_host(d_out) == 0)
        assert bs.bs_expect(op_empty, sec, d_in) == 0
        bs.bs_apply(op_id, sec, d_in, d_out)
        assert rel_l2(to_host(d_out), (2.5 - 1j) * psi) <= 1e-15
        bs.bs_apply(op, sec, d_in, d_out)
        want = osec.apply(ref, psi)
        # (0,0) is the vacuum: H|vac> = 0 exactly and both sides return rounding residue of cancelling
        # coefficients (~1e-15), so the error is measured against max(||want||, 1) there
        assert np.linalg.norm(to_host(d_out) - want) <= TOL_L2 * max(np.linalg.norm(want), 1.0), (na, nb)
        assert abs(bs.bs_expect(op, sec, d_in) - orc.vdot(psi, want)) <= TOL_E
    full = bs.bs_sector_build(12)
    d_in = to_device(si.random_state(4096, 1))
    d_out = torch.full_like(d_in, 1.0)
    bs.bs_apply(op_empty, full, d_in, d_out)
    assert np.all(to_host(d_out) == 0)


def test_rotations_on_degenerate_sectors(bs, orc):
    """Number-conserving generators on sectors where no pair exists (full / empty spin) act as the identity; on a
    half-empty sector only the generators of the populated spin act."""
    from paper_2606_28952_b200 import jw_terms as jw
    ex = si.uccsd_excitations(5, 2, 2)
    th = si.thetas(len(ex), 77, sd=0.5)
    X, Z, Cc, offs = jw.excitation_generator_terms(ex)
    gens = bs.bs_group_xmask(X, Z, Cc, 10, 0.0, bs.BS_MODE_SEQUENCE, offs)
    for (na, nb) in [(5, 5), (0, 0), (5, 0), (0, 3), (2, 5), (1, 4)]:
        sec, osec = bs.bs_sector_build(5, na, nb), orc.Sector(5, na, nb)
        psi = si.random_state(osec.dim, 9 + na + 7 * nb)
        d = to_device(psi)
        bs.bs_apply_pauli_rotations(gens, sec, th, d)
        for (cre, ann), t in zip(ex, th):
            osec.rot_fermionic(psi, cre, ann, t)
        assert rel_l2(to_host(d), psi) <= TOL_L2, (na, nb)
