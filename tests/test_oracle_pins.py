"""Pins of the CPU oracle against what the paper and the mathematics fix.

All `not gpu`.  The references here (tests/dense_ref.py, closed forms, golden files) share
nothing with oracle/bs_oracle.cpp.
"""
import math
import os

import numpy as np
import pytest
import scipy.linalg
import scipy.sparse.linalg

import synth_inputs as S
from oracle import oracle as O
import dense_ref as R

GOLD = os.path.join(os.path.dirname(__file__), "golden")


def _rand_state(dim, seed):
    return S.random_state(dim, seed)


# ---------------------------------------------------------------- P1 encoding + product rule
def test_p1_single_qubit_product_table_vs_matrices():
    # R(a,b) = sx^a sz^b (Eq. 13); product rule Eq. 19-21
    def rmat(a, b):
        return np.linalg.matrix_power(R.SX, a) @ np.linalg.matrix_power(R.SZ, b)
    for a1 in (0, 1):
        for b1 in (0, 1):
            for a2 in (0, 1):
                for b2 in (0, 1):
                    xo, zo, co = O.pauli_mul(a1, b1, 1.0, a2, b2, 1.0)
                    assert np.allclose(rmat(a1, b1) @ rmat(a2, b2), co * rmat(xo, zo))


def test_p1_golden_pauli_table_true_paulis():
    # golden/pauli_table.txt: XY = iZ etc.  True Pauli = (+i)^{ab} sx^a sz^b  (sigma_y = i sx sz).
    enc = {"I": (0, 0), "X": (1, 0), "Y": (1, 1), "Z": (0, 1)}
    for line in open(os.path.join(GOLD, "pauli_table.txt")):
        if line.startswith("#") or not line.strip():
            continue
        l, r, ph, res = line.split()
        (a1, b1), (a2, b2) = enc[l], enc[r]
        c1, c2 = 1j ** (a1 * b1), 1j ** (a2 * b2)  # XZ-form coefficient of the true Pauli
        xo, zo, co = O.pauli_mul(a1, b1, c1, a2, b2, c2)
        assert (xo, zo) == enc[res]
        c_true = co * (-1j) ** (xo & zo)            # back to true-Pauli coefficient (U1)
        assert abs(c_true - 1j ** int(ph)) < 1e-15


def test_p1_type_recovery_identities():
    # Eq. 9-11 on every (a,b)
    for (a, b), name in (((0, 0), "I"), ((1, 0), "X"), ((1, 1), "Y"), ((0, 1), "Z")):
        ty = a & b
        tx, tz = a ^ ty, b ^ ty
        assert {"I": (0, 0, 0), "X": (1, 0, 0), "Y": (0, 1, 0), "Z": (0, 0, 1)}[name] == (tx, ty, tz)


def test_p1_multi_qubit_product_vs_kronecker():
    rng = np.random.default_rng(5)
    nq = 5
    for _ in range(20):
        x1, z1, x2, z2 = (int(v) for v in rng.integers(0, 1 << nq, 4))
        # true-Pauli coefficient 1 -> XZ-form coefficient i^{ny}
        c1, c2 = 1j ** bin(x1 & z1).count("1"), 1j ** bin(x2 & z2).count("1")
        xo, zo, co = O.pauli_mul(x1, z1, c1, x2, z2, c2)
        c_true = co * (-1j) ** bin(xo & zo).count("1")
        lhs = R.pauli_string_matrix(x1, z1, nq) @ R.pauli_string_matrix(x2, z2, nq)
        rhs = c_true * R.pauli_string_matrix(xo, zo, nq)
        assert abs(lhs - rhs).max() < 1e-14


# ---------------------------------------------------------------- P2 ladder operators
def test_p2_ladder_is_one_zero_projector_and_jw_matrix():
    op = O.ladder_product([0], [1])
    m = R.pauli_sum_matrix(op.x, op.z, op.c, 1).toarray()
    assert np.allclose(m, [[0, 0], [1, 0]])  # a^dag = |1><0|
    nq = 4
    for P in range(nq):
        op = O.ladder_product([P], [1])
        assert abs(R.pauli_sum_matrix(op.x, op.z, op.c, nq) - R.creation_matrix(P, nq)).max() < 1e-15
        op = O.ladder_product([P], [0])
        assert abs(R.pauli_sum_matrix(op.x, op.z, op.c, nq) - R.creation_matrix(P, nq).conj().T).max() < 1e-15


def test_p2_anticommutators_as_pauli_sums():
    nq = 6
    eye = np.eye(1 << nq)
    for P in range(nq):
        for Q in range(nq):
            ad_a = O.ladder_product([P, Q], [1, 0])
            a_ad = O.ladder_product([Q, P], [0, 1])
            m = R.pauli_sum_matrix(ad_a.x, ad_a.z, ad_a.c, nq) + R.pauli_sum_matrix(a_ad.x, a_ad.z, a_ad.c, nq)
            assert np.allclose(m.toarray(), eye if P == Q else 0 * eye)
            aa = O.ladder_product([P, Q], [0, 0])
            aa2 = O.ladder_product([Q, P], [0, 0])
            m = R.pauli_sum_matrix(aa.x, aa.z, aa.c, nq) + R.pauli_sum_matrix(aa2.x, aa2.z, aa2.c, nq)
            assert abs(m).max() < 1e-15


def test_p2_term_counts_4_and_16():
    # a one-/two-body term expands into 4 / 16 Pauli strings
    assert len(O.ladder_product([3, 1], [1, 0])) == 4
    assert len(O.ladder_product([5, 3, 2, 0], [1, 1, 0, 0])) == 16


# ---------------------------------------------------------------- P3 counts (closed forms)
def _closed_form_counts(n):
    c2, c4 = math.comb(n, 2), math.comb(n, 4)
    G = 1 + 2 * c2 + 2 * c4 + c2 * c2
    M = 12 * c4 + 4 * c2 * c2 + 4 * (2 * n - 1) * c2 + 1 + 2 * n + math.comb(2 * n, 2)
    return G, M


@pytest.mark.parametrize("n", [2, 3, 4, 6])
def test_p3_molecular_counts_and_classes(n):
    h, g = S.integrals(n, 1000 + n)
    op = O.molecular_h(h, g)
    G, M = _closed_form_counts(n)
    assert len(op) == M and op.n_groups == G
    assert np.abs(op.c.imag).max() == 0.0
    # canonical order: sorted by (x, z), unique
    keys = list(zip(op.x.tolist(), op.z.tolist()))
    assert keys == sorted(set(keys))
    # N_g per class (popc x_alpha, popc x_beta)
    ma = (1 << n) - 1
    expect = {(0, 0): 1 + 2 * n + math.comb(2 * n, 2), (2, 0): 2 * (2 * n - 1), (0, 2): 2 * (2 * n - 1),
              (4, 0): 6, (0, 4): 6, (2, 2): 4}
    xs, counts = np.unique(op.x, return_counts=True)
    for x, cnt in zip(xs.tolist(), counts.tolist()):
        cls = (bin(x & ma).count("1"), bin(x >> n).count("1"))
        assert expect[cls] == cnt
    # every string has an even number of Y
    ny = np.array([bin(int(a) & int(b)).count("1") for a, b in zip(op.x, op.z)])
    assert (ny % 2 == 0).all()


def test_p3_config_counts_match_survey_table():
    # config 1 G=286 M=1819; Hubbard L=14: G=27 M=95
    assert _closed_form_counts(6) == (286, 1819)
    assert _closed_form_counts(12) == (5479, 29737)
    assert _closed_form_counts(16) == (18281, 94849)
    assert _closed_form_counts(28) == (184591, 901993)
    op = O.hubbard_h(14, 1.0, 4.0)
    assert (len(op), op.n_groups) == (95, 27)


# ---------------------------------------------------------------- P4 dense Kronecker vs fermionic
@pytest.mark.parametrize("n", [2, 3, 6])
def test_p4_molecular_dense_equals_fermionic_matrix(n):
    # n = 6 is config 1 itself (12 qubits, the survey's "<= 12 qubits"): 4096 x 4096, sparse on both sides
    h, g = S.integrals(n, 1001 if n == 6 else 77 + n)
    op = O.molecular_h(h, g)
    nq = 2 * n
    Hp = R.pauli_sum_matrix(op.x, op.z, op.c, nq).toarray()
    Hf = R.molecular_h_matrix(h, g).toarray()
    assert np.abs(Hp - Hf).max() < 1e-13
    assert np.abs(Hp - Hp.conj().T).max() < 1e-13
    # number conserving per spin
    ma = (1 << n) - 1
    rows, cols = np.nonzero(np.abs(Hp) > 1e-13)
    for t, s in zip(rows.tolist(), cols.tolist()):
        assert bin(t & ma).count("1") == bin(s & ma).count("1")
        assert bin(t >> n).count("1") == bin(s >> n).count("1")


def test_p4_hubbard_dense_equals_fermionic_matrix():
    L, t, U = 3, 1.0, 4.0
    op = O.hubbard_h(L, t, U)
    nq = 2 * L
    cre = [R.creation_matrix(P, nq) for P in range(nq)]
    ann = [c.conj().T for c in cre]
    H = 0
    for s in range(2):
        for i in range(L - 1):
            P, Q = i + s * L, i + 1 + s * L
            H = H - t * (cre[P] @ ann[Q] + cre[Q] @ ann[P])
    for i in range(L):
        H = H + U * (cre[i] @ ann[i] @ cre[i + L] @ ann[i + L])
    assert abs(R.pauli_sum_matrix(op.x, op.z, op.c, nq) - H).max() < 1e-14


# ---------------------------------------------------------------- P5 Slater-Condon
def test_p5_slater_condon_all_determinants_n3():
    n = 3
    h, g = S.integrals(n, 31)
    op = O.molecular_h(h, g)
    for na in range(n + 1):
        for nb in range(n + 1):
            sec = O.Sector(n, na, nb)
            sa, sb = sec.strings()
            for i, a in enumerate(sa.tolist()):
                for j, b in enumerate(sb.tolist()):
                    e = np.zeros(sec.dim, complex)
                    e[i * sec.dim_beta + j] = 1
                    got = O.energy(sec, op, e)
                    ref = R.slater_condon_energy(h, g, R.bits(a), R.bits(b))
                    assert abs(got - ref) < 1e-12


def test_p5_slater_condon_hf_and_random_dets_config1():
    cfg = S.CONFIGS["q12"]
    h, g = S.integrals(cfg.n_orb, cfg.seed_ints)
    op = O.molecular_h(h, g)
    sec = O.Sector(6, 3, 3)
    sa, sb = sec.strings()
    rng = np.random.default_rng(3)
    idxs = [0] + rng.integers(0, sec.dim, 12).tolist()
    for idx in idxs:
        e = np.zeros(sec.dim, complex)
        e[idx] = 1
        a, b = int(sa[idx // sec.dim_beta]), int(sb[idx % sec.dim_beta])
        assert abs(O.energy(sec, op, e) - R.slater_condon_energy(h, g, R.bits(a), R.bits(b))) < 1e-11


# ---------------------------------------------------------------- P6 apply vs dense (config 1)
@pytest.fixture(scope="module")
def config1():
    cfg = S.CONFIGS["q12"]
    h, g = S.integrals(cfg.n_orb, cfg.seed_ints)
    op = O.molecular_h(h, g)
    Hd = R.pauli_sum_matrix(op.x, op.z, op.c, 12).tocsr()
    return cfg, op, Hd


def test_p6_full_space_apply_vs_dense_4096(config1):
    cfg, op, Hd = config1
    full = O.Sector(12)
    psi = _rand_state(4096, cfg.seed_psi)
    out = full.apply(op, psi)
    ref = Hd @ psi
    assert np.linalg.norm(out - ref) / np.linalg.norm(ref) < 1e-13


def test_p6_sector_apply_is_restriction_of_full_space(config1):
    cfg, op, Hd = config1
    sec = O.Sector(6, 3, 3)
    assert sec.dim == 400
    sa, sb = sec.strings()
    cfgs = (sa[:, None] | (sb[None, :] << np.uint64(6))).reshape(-1)   # index = ia*Db + ib (U4)
    psi = _rand_state(400, cfg.seed_psi)
    emb = np.zeros(4096, complex)
    emb[cfgs.astype(np.int64)] = psi
    ref_full = Hd @ emb
    out = sec.apply(op, psi)
    assert np.linalg.norm(out - ref_full[cfgs.astype(np.int64)]) / np.linalg.norm(out) < 1e-13
    # H conserves the sector: nothing leaks outside
    leak = ref_full.copy()
    leak[cfgs.astype(np.int64)] = 0
    assert np.abs(leak).max() < 1e-12
    # energy against the dense quadratic form
    e = O.energy(sec, op, psi)
    assert abs(e - np.vdot(emb, ref_full)) < 1e-12
    assert abs(e.imag) < 1e-13


def test_p6_hermiticity_of_apply(config1):
    cfg, op, _ = config1
    sec = O.Sector(6, 3, 3)
    phi, psi = _rand_state(400, 11), _rand_state(400, 12)
    lhs = O.vdot(phi, sec.apply(op, psi))
    rhs = np.conj(O.vdot(psi, sec.apply(op, phi)))
    assert abs(lhs - rhs) < 1e-13


# ---------------------------------------------------------------- P7 phase convention (odd ny)
def test_p7_odd_ny_operator_vs_dense():
    # a UCC generator has only odd-ny strings: pins i^{ny} on the source
    n = 3
    gen = O.excitation_generator([4], [0])          # a^dag_4 a_0 - h.c. on 6 qubits
    ny = np.array([bin(int(a) & int(b)).count("1") for a, b in zip(gen.x, gen.z)])
    assert (ny % 2 == 1).all() and len(gen) == 2
    Gd = R.pauli_sum_matrix(gen.x, gen.z, gen.c, 2 * n)
    full = O.Sector(2 * n)
    psi = _rand_state(64, 5)
    assert np.linalg.norm(full.apply(gen, psi) - Gd @ psi) < 1e-14
    gen2 = O.excitation_generator([2, 5], [3, 0])   # alpha-beta double
    assert len(gen2) == 8
    Gd2 = R.pauli_sum_matrix(gen2.x, gen2.z, gen2.c, 2 * n)
    assert np.linalg.norm(full.apply(gen2, psi) - Gd2 @ psi) < 1e-14
    assert abs(Gd2 + Gd2.conj().T).max() < 1e-15     # anti-Hermitian
    # single Y string: <1|Y|0> = i
    y = O.PauliOp([1], [1], [1.0])
    out = O.Sector(1).apply(y, np.array([1.0, 0.0], complex))
    assert np.allclose(out, [0, 1j])


# ---------------------------------------------------------------- P8 sector tables
@pytest.mark.parametrize("n,N", [(6, 3), (12, 6), (14, 7), (16, 8), (10, 0), (10, 10), (20, 4)])
def test_p8_sector_strings(n, N):
    sec = O.Sector(n, N, N)
    sa, _ = sec.strings()
    assert len(sa) == math.comb(n, N) == sec.dim_alpha
    assert (np.diff(sa.astype(np.int64)) > 0).all() if len(sa) > 1 else True
    assert int(sa[0]) == (1 << N) - 1                       # HF string has rank 0 (U5)
    assert int(sa[-1]) == ((1 << N) - 1) << (n - N)
    assert all(bin(int(w)).count("1") == N for w in sa[:: max(1, len(sa) // 200)])
    # combinatorial-number-system rank equals the position (independent formula)
    for pos in list(range(0, len(sa), max(1, len(sa) // 50))) + [len(sa) - 1]:
        rank = sum(math.comb(p, i + 1) for i, p in enumerate(R.bits(int(sa[pos]))))
        assert rank == pos


def test_p8_sector_index_and_golden_dimensions():
    sec = O.Sector(6, 3, 3)
    sa, sb = sec.strings()
    cfgs = (sa[:, None] | (sb[None, :] << np.uint64(6))).reshape(-1)
    assert (sec.index(cfgs) == np.arange(400)).all()
    assert (sec.index(np.array([0, 1, 0b111111], np.uint64)) == -1).all()
    for line in open(os.path.join(GOLD, "table2_det.txt")):
        if line.startswith("#") or not line.strip():
            continue
        _, ne, no, det = line.split()
        ne, no, det = int(ne), int(no), float(det)
        d = math.comb(no, ne // 2) ** 2
        assert abs(d - det) / det < 0.05, (line, d)
    # the five BASELINE.json sector dimensions
    assert [S.CONFIGS[k].dim for k in S.CONFIG_ORDER] == [400, 853776, 11778624, 165636900, 419225625]


# ---------------------------------------------------------------- P9 rotations
def _dense_generator(cre, ann, nq):
    c = [R.creation_matrix(P, nq) for P in range(nq)]
    a = [m.conj().T for m in c]
    T = None
    for P in cre:
        T = c[P] if T is None else T @ c[P]
    for P in ann:
        T = T @ a[P]
    return (T - T.conj().T).toarray()


# the last two are generalised doubles with a shared index (tUCCGSD): a^dag_3 a^dag_5 a_3 a_1 = -n_3 a^dag_5 a_1,
# an X mask of two bits with a number projector attached; creators and annihilators overlap
@pytest.mark.parametrize("cre,ann", [((4,), (0,)), ((2, 5), (3, 0)), ((1, 2), (5, 4)), ((2,), (1,)),
                                     ((3, 5), (3, 1)), ((4, 1), (2, 1))])
def test_p9_fermionic_rotation_vs_dense_expm(cre, ann):
    nq = 6
    Gd = _dense_generator(cre, ann, nq)
    full = O.Sector(nq)
    psi = _rand_state(64, 9)
    th = 0.37
    ref = scipy.linalg.expm(th * Gd) @ psi
    got = psi.copy()
    full.rot_fermionic(got, cre, ann, th)
    assert np.linalg.norm(got - ref) < 1e-14
    assert abs(np.linalg.norm(got) - 1) < 1e-14
    full.rot_fermionic(got, cre, ann, -th)
    assert np.linalg.norm(got - psi) < 1e-14
    zero = psi.copy()
    full.rot_fermionic(zero, cre, ann, 0.0)
    assert np.array_equal(zero, psi)
    assert np.abs(Gd @ Gd @ Gd + Gd).max() < 1e-14             # G^3 = -G
    # Pauli form of the same generator = oracle Pauli sum; product of single-string rotations
    gen = O.excitation_generator(cre, ann)
    assert np.abs(R.pauli_sum_matrix(gen.x, gen.z, gen.c, nq).toarray() - Gd).max() < 1e-15
    v = psi.copy()
    for x, z, c in zip(gen.x, gen.z, gen.c):
        P = R.pauli_string_matrix(int(x), int(z), nq).toarray()
        assert abs(c.real) < 1e-15                              # c = i * real
        a = th * c.imag                                         # exp(i a P) = cos a + i sin a P
        v = math.cos(a) * v + 1j * math.sin(a) * (P @ v)
    assert np.linalg.norm(v - ref) < 1e-14


def test_p9_sector_rotation_matches_full_space():
    n, na, nb = 3, 2, 1
    sec, full = O.Sector(n, na, nb), O.Sector(2 * n)
    sa, sb = sec.strings()
    cfgs = (sa[:, None] | (sb[None, :] << np.uint64(n))).reshape(-1).astype(np.int64)
    psi = _rand_state(sec.dim, 4)
    emb = np.zeros(64, complex)
    emb[cfgs] = psi
    for (cre, ann), th in zip(S.uccsd_excitations(n, na, nb), S.thetas(100, 1)):
        sec.rot_fermionic(psi, cre, ann, th)
        full.rot_fermionic(emb, cre, ann, th)
    assert np.linalg.norm(emb[cfgs] - psi) < 1e-14
    assert abs(np.linalg.norm(psi) - 1) < 1e-14


def test_p9_uccsd_list_counts():
    ex = S.uccsd_excitations(12, 6, 6)
    assert len(ex) == 1818 and sum(len(c) == 1 for c, _ in ex) == 72
    # Pauli-string count of the generators: singles 2, doubles 8
    assert len(O.excitation_generator(*ex[0])) == 2
    assert len(O.excitation_generator(*ex[-1])) == 8
    assert len(O.excitation_generator(*ex[100])) == 8


# ---------------------------------------------------------------- P10 Hubbard
def _ground_energy(sec, op):
    D = sec.dim
    lin = scipy.sparse.linalg.LinearOperator((D, D), matvec=lambda v: sec.apply(op, v.astype(complex)), dtype=complex)
    if D <= 64:
        M = np.column_stack([sec.apply(op, np.eye(D, dtype=complex)[:, k].copy()) for k in range(D)])
        return np.linalg.eigvalsh(M)[0]
    return scipy.sparse.linalg.eigsh(lin, k=1, which="SA", tol=1e-12)[0][0]


def test_p10_hubbard_dimer_golden():
    for line in open(os.path.join(GOLD, "hubbard_dimer.txt")):
        if line.startswith("#") or not line.strip():
            continue
        t, U, e0 = (float(v) for v in line.split())
        op = O.hubbard_h(2, t, U, eps_drop=1e-14)
        assert abs(_ground_energy(O.Sector(2, 1, 1), op) - e0) < 1e-12


def test_p10_hubbard_free_fermion_band_energy():
    L, N = 6, 3
    op = O.hubbard_h(L, 1.0, 0.0)
    e_band = 2 * sum(-2.0 * math.cos(k * math.pi / (L + 1)) for k in range(1, N + 1))
    assert abs(_ground_energy(O.Sector(L, N, N), op) - e_band) < 1e-10


def test_p10_hubbard_trace_and_site_product_state():
    L, N, U = 6, 3, 4.0
    op = O.hubbard_h(L, 1.0, U)
    sec = O.Sector(L, N, N)
    tr = sum(O.energy(sec, op, np.eye(sec.dim, dtype=complex)[k].copy()).real for k in range(sec.dim))
    assert abs(tr / sec.dim - U * N * N / L) < 1e-12
    sa, sb = sec.strings()
    for idx in (0, 17, 123, 399):
        a, b = int(sa[idx // sec.dim_beta]), int(sb[idx % sec.dim_beta])
        e = np.zeros(sec.dim, complex)
        e[idx] = 1
        assert abs(O.energy(sec, op, e) - U * bin(a & b).count("1")) < 1e-13


# ---------------------------------------------------------------- P11 Taylor
def test_p11_taylor_vs_dense_expm_and_reversibility():
    L, N = 4, 2
    op = O.hubbard_h(L, 1.0, 4.0)
    sec = O.Sector(L, N, N)
    D = sec.dim
    Hm = np.column_stack([sec.apply(op, np.eye(D, dtype=complex)[:, k].copy()) for k in range(D)])
    psi0 = _rand_state(D, 21)
    e0 = O.energy(sec, op, psi0).real
    dt = 0.05
    psi = psi0.copy()
    for _ in range(10):
        sec.taylor_step(op, psi, dt, 12, e0)
    ref = scipy.linalg.expm(-1j * Hm * dt * 10) @ psi0
    assert np.linalg.norm(psi - ref) < 1e-12
    assert abs(np.linalg.norm(psi) - 1) < 1e-12
    assert abs(O.energy(sec, op, psi).real - e0) < 1e-11
    for _ in range(10):
        sec.taylor_step(op, psi, -dt, 12, e0)
    assert np.linalg.norm(psi - psi0) < 1e-12


def test_p11_taylor_full_space_tfim_vs_dense_expm():
    """The propagator on a number-non-conserving operator in the full 2^N space: the open TFIM chain of PAPER.md:469-473
    (Eq. 40, J = 1/4, h = 1, dt = 0.05) from |0...0> against scipy's expm of the Kronecker-product matrix."""
    N = 8
    x, z, c = S.tfim_terms(N)
    Hm = R.pauli_sum_matrix([int(v) for v in x], [int(v) for v in z], list(c), N).toarray()
    assert np.abs(Hm - Hm.conj().T).max() == 0
    op, sec = O.PauliOp(x, z, c), O.Sector(N)
    psi = np.zeros(1 << N, np.complex128)
    psi[0] = 1.0
    e0 = O.energy(sec, op, psi).real
    assert abs(e0 - 0.25 * (N - 1)) < 1e-14                  # every Z_i Z_{i+1} = +1 on |0...0>, <X_i> = 0
    for _ in range(8):
        sec.taylor_step(op, psi, 0.05, 12, e0)
    v0 = np.zeros(1 << N, np.complex128)
    v0[0] = 1.0
    assert np.linalg.norm(psi - scipy.linalg.expm(-1j * Hm * 0.4) @ v0) < 1e-12
    assert abs(np.linalg.norm(psi) - 1) < 1e-12


# ---------------------------------------------------------------- P12 fast mode and sampled mode
@pytest.mark.parametrize("kind", ["molecular", "hubbard", "generator", "full"])
def test_p12_grouped_and_sampled_equal_definition(kind):
    if kind == "molecular":
        h, g = S.integrals(5, 8)
        op, sec = O.molecular_h(h, g), O.Sector(5, 2, 3)
    elif kind == "hubbard":
        op, sec = O.hubbard_h(7, 1.0, 4.0), O.Sector(7, 3, 4)
    elif kind == "generator":
        op, sec = O.excitation_generator([3, 8], [6, 1]), O.Sector(5, 2, 2)
    else:
        h, g = S.integrals(4, 8)
        op, sec = O.molecular_h(h, g), O.Sector(8)
    psi = _rand_state(sec.dim, 33)
    ref = sec.apply(op, psi)
    fast = sec.apply_grouped(op, psi)
    assert np.linalg.norm(fast - ref) <= 1e-13 * max(1.0, np.linalg.norm(ref))
    tg = np.random.default_rng(0).integers(0, sec.dim, 50)
    smp = sec.apply_sampled(op, psi, tg)
    assert np.abs(smp - ref[tg]).max() < 1e-13
    # row slab of the fast mode writes only its rows
    if sec.n_alpha >= 0:
        slab = sec.apply_grouped(op, psi, 1, 3)
        db = sec.dim_beta
        assert np.array_equal(slab[db:3 * db], fast[db:3 * db]) and not slab[:db].any() and not slab[3 * db:].any()
        # slab mode with the beta search hoisted (the writer of the full-size goldens): every slab vs the definition
        da = sec.dim_alpha
        for lo, hi in ((0, da), (0, 1), (1, 3), (da - 2, da)):
            got = sec.apply_grouped_slab(op, psi, lo, hi).reshape(-1)
            want = ref[lo * db:hi * db]
            assert np.linalg.norm(got - want) <= 1e-13 * max(1.0, np.linalg.norm(ref))
