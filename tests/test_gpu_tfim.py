"""GPU parity in the full 2^N space on the paper's dynamics model (Eq. 40-43): the open
transverse-field Ising chain H = J sum Z_i Z_{i+1} + h sum X_i (J = 1/4, h = 1) and the layered ansatz of
single-string rotations exp(-i w Z_j Z_{j+1}) (diagonal generators, x = 0) and exp(-i w X_i) / exp(-i w Y_i).

Oracle: the definition-mode apply of oracle/ in the full space; a single-string rotation is evaluated as
exp(-i w P) psi = cos(w) psi - i sin(w) (P psi) (P^2 = 1) with P psi from the oracle's term-by-term apply, so the
rotation kernels are checked against something that shares no code with them."""
import numpy as np
import pytest

import synth_inputs as si
from common import rel_l2

pytestmark = pytest.mark.gpu


def tfim_terms(N, J=0.25, h=1.0):
    x, z, c = [], [], []
    for i in range(N - 1):
        x.append(0), z.append((1 << i) | (1 << (i + 1))), c.append(J)
    for i in range(N):
        x.append(1 << i), z.append(0), c.append(h)
    return np.array(x, np.uint64), np.array(z, np.uint64), np.array(c, np.complex128)


def layered_generators(N, L, rng):
    """Eq. 41-43: per layer 19 ZZ rotations then 20 single-qubit rotations (X in even layers, Y in odd)."""
    x, z, w = [], [], []
    for layer in range(L):
        for j in range(N - 1):
            x.append(0), z.append((1 << j) | (1 << (j + 1)))
        for i in range(N):
            x.append(1 << i), z.append((1 << i) if layer % 2 else 0)
        w.extend(rng.standard_normal(2 * N - 1) * 0.4)
    return np.array(x, np.uint64), np.array(z, np.uint64), np.array(w)


@pytest.mark.parametrize("N,L", [(10, 3), (20, 2)])
def test_tfim_apply_and_layered_circuit(N, L):
    import torch
    from oracle import oracle as orc
    from paper_2606_28952_b200 import bs
    x, z, c = tfim_terms(N)
    op = bs.bs_group_xmask(x, z, c, N, 0.0)
    assert op.n_groups == N + 1 and op.n_terms == 2 * N - 1
    xg, offs, zz, cc, _ = op.export()
    ref = orc.PauliOp(np.repeat(xg, np.diff(offs)), zz, cc)
    sec, osec = bs.bs_sector_build(N), orc.Sector(N)
    psi = si.random_state(1 << N, 40 + N)
    want = osec.apply(ref, psi)
    d_in = torch.from_numpy(psi).cuda()
    d_out = torch.empty_like(d_in)
    bs.bs_apply(op, sec, d_in, d_out)
    assert rel_l2(d_out.cpu().numpy(), want) <= 1e-12
    assert abs(bs.bs_expect(op, sec, d_in) - orc.vdot(psi, want)) <= 1e-10
    # layered circuit on |0...0>, one generator per Pauli string: A = -i P, psi <- exp(w A) psi
    gx, gz, w = layered_generators(N, L, np.random.default_rng(N))
    gens = bs.bs_group_xmask(gx, gz, np.full(len(gx), -1j), N, 0.0, bs.BS_MODE_SEQUENCE,
                             np.arange(len(gx) + 1, dtype=np.int64))
    state = np.zeros(1 << N, np.complex128)
    state[0] = 1.0
    d = torch.from_numpy(state).cuda()
    bs.bs_apply_pauli_rotations(gens, sec, w, d)
    for k in range(len(gx)):
        p = orc.PauliOp(gx[k:k + 1], gz[k:k + 1], np.ones(1, np.complex128))
        state = np.cos(w[k]) * state - 1j * np.sin(w[k]) * osec.apply(p, state)
    got = d.cpu().numpy()
    assert abs(np.linalg.norm(got) - 1.0) <= 1e-12
    assert rel_l2(got, state) <= 1e-12
    # energy of the circuit state through the fused expectation
    assert abs(bs.bs_expect(op, sec, d) - orc.vdot(state, osec.apply(ref, state))) <= 1e-10


def test_diagonal_generator_in_a_sector():
    """x = 0 generators also work on (N_alpha, N_beta) sectors: exp(-i w n_p n_q)-type phases (Z strings)."""
    import torch
    from oracle import oracle as orc
    from paper_2606_28952_b200 import bs
    # generators: two diagonal Z strings, the sector-conserving alpha hop i/2 (Y0 X1 - X0 Y1), one more diagonal
    gx = np.array([0, 0, 3, 3, 0], np.uint64)
    gz = np.array([0b000101, 0b110000000000, 0b01, 0b10, 0b1], np.uint64)   # Y0 X1 (z=01) and X0 Y1 (z=10)
    gc = np.array([-1j, -1j, 0.5j, -0.5j, -1j])
    offs = np.array([0, 1, 2, 4, 5], np.int64)
    w = np.array([0.3, -0.7, 0.45, 1.1])
    gens = bs.bs_group_xmask(gx, gz, gc, 12, 0.0, bs.BS_MODE_SEQUENCE, offs)
    sec, osec = bs.bs_sector_build(6, 3, 3), orc.Sector(6, 3, 3)
    psi = si.random_state(400, 3)
    d = torch.from_numpy(psi.copy()).cuda()
    bs.bs_apply_pauli_rotations(gens, sec, w, d)
    state = psi.copy()
    for j in range(4):
        s = slice(offs[j], offs[j + 1])
        a = orc.PauliOp(gx[s], gz[s], gc[s])
        # exp(w A) by its Taylor series with the oracle apply (A is anti-Hermitian, |w| ||A|| <= 1.1)
        term, acc = state.copy(), state.copy()
        for k in range(1, 40):
            term = osec.apply(a, term) * (w[j] / k)
            acc += term
        state = acc
    assert rel_l2(d.cpu().numpy(), state) <= 1e-12
    assert abs(np.linalg.norm(d.cpu().numpy()) - 1.0) <= 1e-12


@pytest.mark.parametrize("N", [10, 14])
def test_tfim_taylor_propagation_in_the_full_space(N):
    """a7 on a number-non-conserving operator: shifted order-12 Taylor steps (Eq. 6-7; dt = 0.05 as in
    PAPER.md:473) of the TFIM chain in the full 2^N space against the oracle's own propagator, started from the
    paper's initial state |0...0>; norm and energy conserved."""
    import torch
    from oracle import oracle as orc
    from paper_2606_28952_b200 import bs
    x, z, c = si.tfim_terms(N)
    op = bs.bs_group_xmask(x, z, c, N, 0.0)
    ref = orc.PauliOp(x, z, c)
    sec, osec = bs.bs_sector_build(N), orc.Sector(N)
    psi = np.zeros(1 << N, np.complex128)
    psi[0] = 1.0
    d = torch.from_numpy(psi.copy()).cuda()
    work = torch.empty(2 << N, dtype=torch.complex128, device="cuda")
    e0 = bs.bs_expect(op, sec, d).real
    assert abs(e0 - 0.25 * (N - 1)) <= 1e-12                            # <0|H|0> = J (N - 1): every Z_i Z_{i+1} = +1
    for _ in range(6):
        bs.bs_taylor_step(op, sec, d, work, 0.05, 12, e0)
        osec.taylor_step(ref, psi, 0.05, 12, e0)
    got = d.cpu().numpy()
    assert rel_l2(got, psi) <= 1e-12
    assert abs(np.linalg.norm(got) - 1.0) <= 1e-12
    assert abs(bs.bs_expect(op, sec, d).real - e0) <= 1e-10
    # total transverse magnetisation sum_i <X_i> (Figure 5's observable) through the same fused expectation
    mx = bs.bs_group_xmask(x[N - 1:], z[N - 1:], np.ones(N, np.complex128), N, 0.0)
    want = orc.vdot(psi, osec.apply(orc.PauliOp(x[N - 1:], z[N - 1:], np.ones(N, np.complex128)), psi))
    assert abs(bs.bs_expect(mx, sec, d) - want) <= 1e-10
