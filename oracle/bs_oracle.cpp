// oracle/bs_oracle.cpp -- TEST INFRASTRUCTURE ONLY.
//
// Plain, slow, obviously-correct CPU oracle for the operator-state multiplication path of
// arxiv/paper_2606_28952 (§2.2-2.5).  Only tests/, __graft_entry__.smoke() and
// bench.py's cpu_baseline / --impl reference legs may load this library.  It shares NO code
// with the CUDA library under paper_2606_28952_b200/csrc (no headers, tables or helpers).
//
// Everything is fp64 (complex128 amplitudes); energies accumulate in long double.
// Every function cites the passage it follows.  Readings of silent/ambiguous points are the
// ones listed in DESIGN.md ("Readings").
//
// Pins (tests/test_oracle_*.py, all `-m "not gpu"`):
//   orc_pauli_mul ........ 16-entry single-qubit product table vs 2x2 matrices (P1)
//   orc_ladder ........... anticommutators as Pauli sums; dense a^dag = |1><0| (P2)
//   orc_molecular_h ...... closed-form counts G(n), M(n); dense Kronecker vs fermionic
//                          occupation-number matrices; Hermitian; Slater-Condon (P3-P5)
//   orc_hubbard_h ........ dimer ground energy, U=0 band energy, trace, M=95/G=27 (P10)
//   orc_apply_terms ...... dense 4096x4096 matvec; sector = restriction; Hermiticity (P6, P7)
//   orc_sector_strings ... binomial counts, rank of HF string, monotone (P8)
//   orc_rot_fermionic .... dense expm, norm, theta/-theta, product of Pauli rotations (P9)
//   orc_taylor_step ...... high-order sub-stepped series at 6 sites; reversibility (P11)
//   orc_apply_grouped .... equals orc_apply_terms (P12)
//   orc_apply_sampled .... equals orc_apply_terms on the sampled targets
//   orc_apply_grouped_slab  equals orc_apply_terms on every row slab (P12)
#include <algorithm>
#include <cmath>
#include <complex>
#include <cstdint>
#include <cstring>
#include <map>
#include <utility>
#include <vector>
#ifdef _OPENMP
#include <omp.h>
#endif

using cd = std::complex<double>;
using u64 = uint64_t;
using i64 = int64_t;

namespace {

inline int popc(u64 v) { return __builtin_popcountll(v); }
// popcnt(v) mod 2 of a 32-bit word by xor-folding (each fold halves the width and keeps the parity); written
// without the popcount builtin so that the compiler can vectorise loops over it (orc_apply_grouped_slab)
inline uint32_t parity32(uint32_t v) { v ^= v >> 16; v ^= v >> 8; v ^= v >> 4; v ^= v >> 2; v ^= v >> 1; return v & 1u; }

// ---------------------------------------------------------------------------------------
// Pauli strings in XZ-ordered form R(X,Z) = (x)_k sx^{a_k} sz^{b_k}  (Eq. 13)
// with X = OR a_k<<k, Z = OR b_k<<k (Eq. 14-15; qubit k = bit k).
// A Pauli sum is a map (X,Z) -> C, C the coefficient of R(X,Z)        (Eq. 16-18).
// ---------------------------------------------------------------------------------------
struct Key {
    u64 x, z;
    bool operator<(const Key& o) const { return x < o.x || (x == o.x && z < o.z); }
};
using PauliSum = std::map<Key, cd>;
using TermList = std::vector<std::pair<Key, cd>>;

// Product of two XZ-form strings: Eq. 19-21:
//   X_m = X_k ^ X_l, Z_m = Z_k ^ Z_l, Lambda_m = Lambda_k Lambda_l (-1)^{popcnt(Z_k & X_l)}.
inline std::pair<Key, cd> mul_term(const Key& a, cd ca, const Key& b, cd cb) {
    Key m{a.x ^ b.x, a.z ^ b.z};
    double sgn = (popc(a.z & b.x) & 1) ? -1.0 : 1.0;
    return {m, ca * cb * sgn};
}

// Operator product with key accumulation, Eq. 22.
TermList mul(const TermList& A, const TermList& B) {
    PauliSum acc;
    for (auto& a : A)
        for (auto& b : B) {
            auto m = mul_term(a.first, a.second, b.first, b.second);
            acc[m.first] += m.second;
        }
    return TermList(acc.begin(), acc.end());
}

// JW ladder operators, Eq. 23: a_P^dag = 1/2 (X_P - iY_P) Z_{P-1}...Z_0,
// a_P = 1/2 (X_P + iY_P) Z_{P-1}...Z_0.  With sigma_y = i sx sz:
// -iY = sx sz, +iY = -sx sz, so in XZ form
//   a_P^dag = 1/2 R(1<<P, lt) + 1/2 R(1<<P, lt | 1<<P),   a_P = 1/2 R(..) - 1/2 R(..),
// lt = (1<<P) - 1 the Z chain on qubits below P.
TermList ladder(int P, bool dagger) {
    u64 bit = u64(1) << P, lt = bit - 1;
    TermList t;
    t.push_back({Key{bit, lt}, cd(0.5, 0.0)});
    t.push_back({Key{bit, lt | bit}, cd(dagger ? 0.5 : -0.5, 0.0)});
    return t;
}

void add_into(PauliSum& H, const TermList& T, cd scale) {
    for (auto& t : T) H[t.first] += scale * t.second;
}

// (-i)^m and i^m for integer m.
inline cd pow_i(int m) {
    switch (m & 3) {
        case 0: return cd(1, 0);
        case 1: return cd(0, 1);
        case 2: return cd(-1, 0);
        default: return cd(0, -1);
    }
}
inline cd pow_mi(int m) { return pow_i(-m & 3); }

// XZ-form coefficient C -> coefficient c of the true Pauli string (x){I,X,Y,Z}:
// R(X,Z) has sx sz = -i sigma_y on each Y position, so C R = C (-i)^{ny} P and c = C (-i)^{ny},
// ny = popcnt(X & Z)   (reading U1).
struct Op {
    std::vector<u64> x, z;
    std::vector<cd> c;  // true-Pauli coefficients, sorted by (x, z) ascending
};

Op* finish(const PauliSum& H, double eps_drop) {
    Op* op = new Op;
    for (auto& kv : H) {  // std::map iterates in (x,z) ascending order = canonical order
        cd c = kv.second * pow_mi(popc(kv.first.x & kv.first.z));
        if (std::abs(c) < eps_drop) continue;   // PAPER.md:157 (eps_drop)
        op->x.push_back(kv.first.x);
        op->z.push_back(kv.first.z);
        op->c.push_back(c);
    }
    return op;
}

// ---------------------------------------------------------------------------------------
// Sector: alpha strings = all n-bit words of popcount N in increasing numeric order
// (Eq. 25/28/38; readings U4, U5).  Brute force over all 2^n words.
// index(a, b) = pos(a) * D_b + pos(b); position by binary search in the sorted list.
// Full space (n_alpha < 0): n "orbitals" means n qubits and index = the word itself.
// ---------------------------------------------------------------------------------------
std::vector<u64> enum_strings(int n, int N) {
    std::vector<u64> s;
    for (u64 w = 0; w < (u64(1) << n); ++w)
        if (popc(w) == N) s.push_back(w);
    return s;
}

struct Sector {
    bool full;
    int n;  // orbitals per spin (sector) or qubits (full)
    std::vector<u64> sa, sb;
    i64 Da, Db, D;
    u64 mask_a;
    Sector(int n_, int na, int nb) : n(n_) {
        full = (na < 0);
        if (full) {
            Da = 1; Db = 1; D = i64(1) << n; mask_a = 0;
        } else {
            sa = enum_strings(n, na);
            sb = enum_strings(n, nb);
            Da = (i64)sa.size(); Db = (i64)sb.size(); D = Da * Db;
            mask_a = (u64(1) << n) - 1;
        }
    }
    static i64 pos(const std::vector<u64>& v, u64 w) {
        auto it = std::lower_bound(v.begin(), v.end(), w);
        return (it != v.end() && *it == w) ? (i64)(it - v.begin()) : -1;
    }
    i64 index(u64 cfg) const {
        if (full) return (cfg >> n) ? -1 : (i64)cfg;
        if (n < 32 && (cfg >> (2 * n))) return -1;
        i64 ia = pos(sa, cfg & mask_a), ib = pos(sb, cfg >> n);
        return (ia < 0 || ib < 0) ? -1 : ia * Db + ib;
    }
    u64 config(i64 idx) const {
        if (full) return (u64)idx;
        return sa[idx / Db] | (sb[idx % Db] << n);
    }
};

// One term applied to the whole sector: Eq. 26 for a single Pauli string
//   out[s ^ x] += c * i^{ny} * (-1)^{popcnt(z & s)} * psi[s]     (reading U2, source form).
// For a fixed term s -> s^x is injective, so the loop over sources has no write conflicts.
void apply_one_term(const Sector& S, u64 x, u64 z, cd c, const cd* psi, cd* out) {
    cd ciy = c * pow_i(popc(x & z));
    if (S.full) {
#pragma omp parallel for schedule(static)
        for (i64 s = 0; s < S.D; ++s) {
            u64 t = (u64)s ^ x;
            if (t >> S.n) continue;
            double sg = (popc(z & (u64)s) & 1) ? -1.0 : 1.0;
            out[t] += ciy * sg * psi[s];
        }
        return;
    }
    // valid alpha sources (s_a ^ x_a again a sector string) and valid beta sources, then
    // their product; nothing else can contribute.
    u64 xa = x & S.mask_a, xb = x >> S.n;
    if (S.n < 32 && (x >> (2 * S.n))) return;
    std::vector<std::pair<i64, i64>> va, vb;  // (source pos, target pos)
    for (i64 i = 0; i < S.Da; ++i) {
        i64 t = Sector::pos(S.sa, S.sa[i] ^ xa);
        if (t >= 0) va.push_back({i, t});
    }
    for (i64 j = 0; j < S.Db; ++j) {
        i64 t = Sector::pos(S.sb, S.sb[j] ^ xb);
        if (t >= 0) vb.push_back({j, t});
    }
#pragma omp parallel for schedule(static)
    for (i64 ii = 0; ii < (i64)va.size(); ++ii) {
        i64 i = va[ii].first, ti = va[ii].second;
        for (auto& pb : vb) {
            i64 j = pb.first, tj = pb.second;
            u64 s = S.sa[i] | (S.sb[j] << S.n);
            double sg = (popc(z & s) & 1) ? -1.0 : 1.0;
            out[ti * S.Db + tj] += ciy * sg * psi[i * S.Db + j];
        }
    }
}

}  // namespace

extern "C" {

int orc_num_threads() {
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

// ---- operators -------------------------------------------------------------------------
void orc_op_free(void* h) { delete (Op*)h; }
i64 orc_op_size(void* h) { return (i64)((Op*)h)->x.size(); }
void orc_op_export(void* h, u64* x, u64* z, double* c_reim) {
    Op* op = (Op*)h;
    size_t M = op->x.size();
    std::memcpy(x, op->x.data(), M * 8);
    std::memcpy(z, op->z.data(), M * 8);
    std::memcpy(c_reim, op->c.data(), M * 16);
}

// Single products exposed for the pins P1/P2.
// (x1,z1,C1)*(x2,z2,C2) in XZ form, Eq. 19-21.
void orc_pauli_mul(u64 x1, u64 z1, const double* c1, u64 x2, u64 z2, const double* c2,
                   u64* xo, u64* zo, double* co) {
    auto m = mul_term(Key{x1, z1}, cd(c1[0], c1[1]), Key{x2, z2}, cd(c2[0], c2[1]));
    *xo = m.first.x; *zo = m.first.z; co[0] = m.second.real(); co[1] = m.second.imag();
}

// Pauli sum (true-Pauli coefficients, canonical order) of a product of ladder operators
// a^(dag)_{idx[0]} a^(dag)_{idx[1]} ... (dag[k] != 0 -> creation), times `scale`.
void* orc_ladder_product(const int* idx, const int* dag, int n_ops, const double* scale, double eps_drop) {
    TermList T;
    T.push_back({Key{0, 0}, cd(1, 0)});
    for (int k = 0; k < n_ops; ++k) T = mul(T, ladder(idx[k], dag[k] != 0));
    PauliSum H;
    add_into(H, T, cd(scale[0], scale[1]));
    return finish(H, eps_drop);
}

// Anti-Hermitian excitation generator T - T^dag as a Pauli sum, T = prod a^dag_{cre} prod a_{ann}
// written left to right (Eq. 39: tau_k); used to cross-check the grouped-rotation
// closed form against the fermionic definition.
void* orc_excitation_generator(const int* cre, int n_cre, const int* ann, int n_ann, double eps_drop) {
    TermList T, Td;
    T.push_back({Key{0, 0}, cd(1, 0)});
    Td = T;
    for (int k = 0; k < n_cre; ++k) T = mul(T, ladder(cre[k], true));
    for (int k = 0; k < n_ann; ++k) T = mul(T, ladder(ann[k], false));
    for (int k = n_ann - 1; k >= 0; --k) Td = mul(Td, ladder(ann[k], true));   // (AB)^dag = B^dag A^dag
    for (int k = n_cre - 1; k >= 0; --k) Td = mul(Td, ladder(cre[k], false));
    PauliSum H;
    add_into(H, T, cd(1, 0));
    add_into(H, Td, cd(-1, 0));
    return finish(H, eps_drop);
}

// Molecular Hamiltonian (Eq. 2; reading U3), spin-orbital P = p (alpha),
// n + p (beta) ("blocked spin ordering"):
//   H = sum_{pq,s} h_pq a^dag_{ps} a_{qs}
//     + 1/2 sum_{pqrs} sum_{s,t} (pq|rs) a^dag_{ps} a^dag_{rt} a_{st} a_{qs},
// JW-mapped by ladder-operator products (Eq. 23 + Eq. 19-22), accumulated by (X,Z) key,
// converted to true-Pauli coefficients, |c| < eps_drop dropped, sorted by (x, z).
void* orc_molecular_h(int n, const double* h, const double* g, double eps_drop) {
    std::vector<TermList> cre(2 * n), ann(2 * n);
    for (int P = 0; P < 2 * n; ++P) { cre[P] = ladder(P, true); ann[P] = ladder(P, false); }
    std::vector<PauliSum> part(n);  // one accumulator per p, merged in p order (deterministic)
#pragma omp parallel for schedule(dynamic, 1)
    for (int p = 0; p < n; ++p) {
        PauliSum& H = part[p];
        for (int q = 0; q < n; ++q) {
            for (int s = 0; s < 2; ++s) {
                int P = p + s * n, Q = q + s * n;
                add_into(H, mul(cre[P], ann[Q]), cd(h[p * n + q], 0));
            }
            for (int r = 0; r < n; ++r)
                for (int sidx = 0; sidx < n; ++sidx) {
                    double v = g[((size_t(p) * n + q) * n + r) * n + sidx];  // (pq|rs)
                    for (int s = 0; s < 2; ++s)
                        for (int t = 0; t < 2; ++t) {
                            int P = p + s * n, Q = q + s * n, R = r + t * n, Sx = sidx + t * n;
                            // a^dag_{ps} a^dag_{rt} a_{st} a_{qs}
                            TermList T = mul(mul(cre[P], cre[R]), mul(ann[Sx], ann[Q]));
                            add_into(H, T, cd(0.5 * v, 0));
                        }
                }
        }
    }
    PauliSum H;
    for (int p = 0; p < n; ++p)
        for (auto& kv : part[p]) H[kv.first] += kv.second;
    return finish(H, eps_drop);
}

// 1-D Fermi-Hubbard chain, open boundaries (BASELINE.json configs[2]):
//   H = -t sum_{i=0}^{L-2} sum_s (a^dag_{is} a_{i+1,s} + h.c.) + U sum_i n_{i,alpha} n_{i,beta}.
void* orc_hubbard_h(int L, double t, double U, double eps_drop) {
    PauliSum H;
    for (int s = 0; s < 2; ++s)
        for (int i = 0; i + 1 < L; ++i) {
            int P = i + s * L, Q = i + 1 + s * L;
            add_into(H, mul(ladder(P, true), ladder(Q, false)), cd(-t, 0));
            add_into(H, mul(ladder(Q, true), ladder(P, false)), cd(-t, 0));
        }
    for (int i = 0; i < L; ++i) {
        TermList na = mul(ladder(i, true), ladder(i, false));
        TermList nb = mul(ladder(i + L, true), ladder(i + L, false));
        add_into(H, mul(na, nb), cd(U, 0));
    }
    return finish(H, eps_drop);
}

// ---- sector ----------------------------------------------------------------------------
void* orc_sector_new(int n, int n_alpha, int n_beta) { return new Sector(n, n_alpha, n_beta); }
void orc_sector_free(void* s) { delete (Sector*)s; }
void orc_sector_dims(void* s, i64* D, i64* Da, i64* Db) {
    Sector* S = (Sector*)s; *D = S->D; *Da = S->Da; *Db = S->Db;
}
void orc_sector_strings(void* s, u64* a, u64* b) {
    Sector* S = (Sector*)s;
    std::memcpy(a, S->sa.data(), S->sa.size() * 8);
    std::memcpy(b, S->sb.data(), S->sb.size() * 8);
}
void orc_sector_index(void* s, const u64* cfg, i64 n, i64* idx) {
    Sector* S = (Sector*)s;
    for (i64 k = 0; k < n; ++k) idx[k] = S->index(cfg[k]);
}

// ---- apply -----------------------------------------------------------------------------
// Definition mode: out = sum_k (term k applied to psi), terms in the order given (Eq. 26).
void orc_apply_terms(void* s, const u64* x, const u64* z, const double* c_reim, i64 M,
                     const double* psi_reim, double* out_reim) {
    Sector* S = (Sector*)s;
    const cd* psi = (const cd*)psi_reim;
    cd* out = (cd*)out_reim;
    for (i64 i = 0; i < S->D; ++i) out[i] = cd(0, 0);
    for (i64 k = 0; k < M; ++k)
        apply_one_term(*S, x[k], z[k], cd(c_reim[2 * k], c_reim[2 * k + 1]), psi, out);
}

// The same definition evaluated for a list of target indices only (configs 4-5 where the
// full term-by-term sweep is too slow): out[j] = sum_k <t_j| c_k P_k |psi>, every term k
// visited for every target, source s = t ^ x_k, Eq. 26 read for one output element.
void orc_apply_sampled(void* s, const u64* x, const u64* z, const double* c_reim, i64 M,
                       const double* psi_reim, const i64* targets, i64 n_targets, double* out_reim) {
    Sector* S = (Sector*)s;
    const cd* psi = (const cd*)psi_reim;
    cd* out = (cd*)out_reim;
#pragma omp parallel for schedule(dynamic, 16)
    for (i64 j = 0; j < n_targets; ++j) {
        u64 t = S->config(targets[j]);
        cd acc(0, 0);
        for (i64 k = 0; k < M; ++k) {
            u64 src = t ^ x[k];
            i64 is = S->index(src);
            if (is < 0) continue;
            cd ciy = cd(c_reim[2 * k], c_reim[2 * k + 1]) * pow_i(popc(x[k] & z[k]));
            double sg = (popc(z[k] & src) & 1) ? -1.0 : 1.0;
            acc += ciy * sg * psi[is];
        }
        out[j] = acc;
    }
}

// Fast mode: X-mask grouping + target-configuration gather, Eq. 24 + Eq. 27
// over the alpha-row range [row_lo, row_hi) (full space: index range).  Terms must be in
// canonical order (sorted by x) so that equal x are adjacent.  Thread-parallel over targets
// (PAPER.md:225).  Writes out only for the requested rows.  This is the timed CPU baseline.
void orc_apply_grouped(void* s, const u64* x, const u64* z, const double* c_reim, i64 M,
                       const double* psi_reim, double* out_reim, i64 row_lo, i64 row_hi) {
    Sector* S = (Sector*)s;
    const cd* psi = (const cd*)psi_reim;
    cd* out = (cd*)out_reim;
    std::vector<i64> offs;  // group boundaries
    for (i64 k = 0; k < M; ++k)
        if (k == 0 || x[k] != x[k - 1]) offs.push_back(k);
    offs.push_back(M);
    i64 G = (i64)offs.size() - 1;
    std::vector<cd> C(M);  // C_k = c_k i^{ny_k} (XZ-form coefficient of Eq. 18)
    for (i64 k = 0; k < M; ++k) C[k] = cd(c_reim[2 * k], c_reim[2 * k + 1]) * pow_i(popc(x[k] & z[k]));
    if (S->full) {
#pragma omp parallel for schedule(static)
        for (i64 t = row_lo; t < row_hi; ++t) {
            cd acc(0, 0);
            for (i64 g = 0; g < G; ++g) {
                u64 src = (u64)t ^ x[offs[g]];
                if (src >> S->n) continue;
                cd ph(0, 0);
                for (i64 k = offs[g]; k < offs[g + 1]; ++k) ph += (popc(z[k] & src) & 1) ? -C[k] : C[k];
                acc += ph * psi[src];
            }
            out[t] = acc;
        }
        return;
    }
#pragma omp parallel for schedule(dynamic, 1)
    for (i64 i = row_lo; i < row_hi; ++i) {
        cd* orow = out + i * S->Db;
        for (i64 j = 0; j < S->Db; ++j) orow[j] = cd(0, 0);
        for (i64 g = 0; g < G; ++g) {
            u64 xg = x[offs[g]];
            if (S->n < 32 && (xg >> (2 * S->n))) continue;
            u64 xa = xg & S->mask_a, xb = xg >> S->n;
            u64 srca = S->sa[i] ^ xa;
            i64 ia = Sector::pos(S->sa, srca);
            if (ia < 0) continue;
            for (i64 j = 0; j < S->Db; ++j) {
                u64 srcb = S->sb[j] ^ xb;
                i64 ib = Sector::pos(S->sb, srcb);
                if (ib < 0) continue;
                u64 src = srca | (srcb << S->n);
                cd ph(0, 0);
                for (i64 k = offs[g]; k < offs[g + 1]; ++k) ph += (popc(z[k] & src) & 1) ? -C[k] : C[k];
                orow[j] += ph * psi[ia * S->Db + ib];
            }
        }
    }
}

// The same Eq. 27 gather for an alpha-row slab [row_lo, row_hi), written to a slab-sized buffer
// out_slab[(i - row_lo) * D_b + j], with the beta-string search of Eq. 28 ("two
// smaller spin-string index searches") done ONCE per distinct beta mask instead of once per
// (row, group, column): whether s_b[j] ^ x_b is a sector string, and where it sits, does not depend
// on the row.  Same loops and same arithmetic as orc_apply_grouped otherwise.  Used to write the
// full-size goldens of configs 4-5 (tests/golden/make_fullsize_golden.py), where the per-row search
// makes orc_apply_grouped take days.  Pinned against orc_apply_terms (P12).  Sector mode only.
void orc_apply_grouped_slab(void* s, const u64* x, const u64* z, const double* c_reim, i64 M,
                            const double* psi_reim, double* out_slab_reim, i64 row_lo, i64 row_hi) {
    Sector* S = (Sector*)s;
    if (S->full) return;
    const cd* psi = (const cd*)psi_reim;
    cd* out = (cd*)out_slab_reim;
    std::vector<i64> offs;
    for (i64 k = 0; k < M; ++k)
        if (k == 0 || x[k] != x[k - 1]) offs.push_back(k);
    offs.push_back(M);
    i64 G = (i64)offs.size() - 1;
    std::vector<cd> C(M);  // C_k = c_k i^{ny_k} (Eq. 18)
    for (i64 k = 0; k < M; ++k) C[k] = cd(c_reim[2 * k], c_reim[2 * k + 1]) * pow_i(popc(x[k] & z[k]));
    // per distinct beta mask: the (target column j, source column ib, source string) triples with
    // s_b[j] ^ x_b in the sector
    struct BetaPairs { std::vector<int32_t> tj, ib; std::vector<uint32_t> src; };  // spin strings have n <= 32 bits
    std::map<u64, BetaPairs> beta_pairs;
    for (i64 g = 0; g < G; ++g) {
        u64 xg = x[offs[g]];
        if (S->n < 32 && (xg >> (2 * S->n))) continue;
        u64 xb = xg >> S->n;
        if (beta_pairs.count(xb)) continue;
        BetaPairs& v = beta_pairs[xb];
        for (i64 j = 0; j < S->Db; ++j) {
            i64 ib = Sector::pos(S->sb, S->sb[j] ^ xb);
            if (ib < 0) continue;
            v.tj.push_back((int32_t)j); v.ib.push_back((int32_t)ib); v.src.push_back((uint32_t)S->sb[ib]);
        }
    }
#pragma omp parallel for schedule(dynamic, 1)
    for (i64 i = row_lo; i < row_hi; ++i) {
        cd* orow = out + (i - row_lo) * S->Db;
        for (i64 j = 0; j < S->Db; ++j) orow[j] = cd(0, 0);
        std::vector<double> ph_re(S->Db), ph_im(S->Db);  // phase sum of the group, per valid target column
        for (i64 g = 0; g < G; ++g) {
            u64 xg = x[offs[g]];
            if (S->n < 32 && (xg >> (2 * S->n))) continue;
            u64 xa = xg & S->mask_a, xb = xg >> S->n;
            u64 srca = S->sa[i] ^ xa;
            i64 ia = Sector::pos(S->sa, srca);
            if (ia < 0) continue;
            const BetaPairs& bp = beta_pairs.find(xb)->second;
            const i64 np = (i64)bp.tj.size();
            for (i64 p = 0; p < np; ++p) { ph_re[p] = 0; ph_im[p] = 0; }
            // Eq. 31 (reading U7): the sign (-1)^{popcnt(z & s)} of Eq. 27 splits into an alpha
            // factor, the same for the whole row, and a beta factor: popcnt(z & s) = popcnt(z_a & s_a) + popcnt(z_b & s_b).
            // Strings in the order given; for each string the loop runs over the valid columns.
            for (i64 k = offs[g]; k < offs[g + 1]; ++k) {
                double sa = (popc(z[k] & S->mask_a & srca) & 1) ? -1.0 : 1.0;
                double cre = sa * C[k].real(), cim = sa * C[k].imag();
                uint32_t zb = (uint32_t)(z[k] >> S->n);
                const uint32_t* __restrict src = bp.src.data();
                double* __restrict pre = ph_re.data();
                double* __restrict pim = ph_im.data();
                for (i64 p = 0; p < np; ++p) {
                    double sb = 1.0 - 2.0 * (double)(int32_t)parity32(zb & src[p]);
                    pre[p] += sb * cre;
                    pim[p] += sb * cim;
                }
            }
            const cd* prow = psi + ia * S->Db;
            for (i64 p = 0; p < np; ++p) orow[bp.tj[p]] += cd(ph_re[p], ph_im[p]) * prow[bp.ib[p]];
        }
    }
}

// <a|b> = sum conj(a_i) b_i, long double accumulation (Eq. 5, PAPER.md:71 with b = H psi).
void orc_vdot(const double* a_reim, const double* b_reim, i64 D, double* res) {
    long double re = 0, im = 0;
    for (i64 i = 0; i < D; ++i) {
        long double ar = a_reim[2 * i], ai = a_reim[2 * i + 1], br = b_reim[2 * i], bi = b_reim[2 * i + 1];
        re += ar * br + ai * bi;
        im += ar * bi - ai * br;
    }
    res[0] = (double)re; res[1] = (double)im;
}

// ---- rotations (fermionic definition, no Pauli strings) ----------------------------------
// exp(theta (T - T^dag)) psi with T = a^dag_{cre[0]} a^dag_{cre[1]} .. a_{ann[0]} a_{ann[1]} ..
// (spin-orbital indices, operators applied right to left)  -- Eq. 39, §2.5
// (PAPER.md:347); SURVEY.md §8(c) item 6.  For every sector configuration s with T|s> = sg|t>:
//   psi'[s] = cos(th) psi[s] - sg sin(th) psi[t],   psi'[t] = sg sin(th) psi[s] + cos(th) psi[t].
// Written for excitation operators (disjoint creator and annihilator index sets); generalised doubles that share an
// index (a^dag_p a^dag_q a_p a_s = -n_p a^dag_q a_s) also satisfy T^2 = 0 and are covered by the same update (pin P9).
static bool apply_ops(u64 s, const int* cre, int n_cre, const int* ann, int n_ann, u64* t, int* sg) {
    int sign = 1;
    u64 w = s;
    for (int k = n_ann - 1; k >= 0; --k) {  // rightmost operator acts first
        u64 bit = u64(1) << ann[k];
        if (!(w & bit)) return false;
        if (popc(w & (bit - 1)) & 1) sign = -sign;
        w ^= bit;
    }
    for (int k = n_cre - 1; k >= 0; --k) {
        u64 bit = u64(1) << cre[k];
        if (w & bit) return false;
        if (popc(w & (bit - 1)) & 1) sign = -sign;
        w |= bit;
    }
    *t = w; *sg = sign;
    return true;
}

void orc_rot_fermionic(void* s, const int* cre, int n_cre, const int* ann, int n_ann, double theta,
                       double* psi_reim) {
    Sector* S = (Sector*)s;
    cd* psi = (cd*)psi_reim;
    double c = std::cos(theta), sn = std::sin(theta);
    // The iterations are independent: iteration i touches psi[i] and psi[it] only when T|i> != 0, then T|it> = 0
    // (T^2 = 0 on a configuration it has just excited), so iteration `it` touches nothing, and T is injective on its
    // support, so no other source reaches `it`.  Same arithmetic per pair as the serial loop, in any order.
#pragma omp parallel for schedule(static)
    for (i64 i = 0; i < S->D; ++i) {
        u64 cfg = S->config(i), t;
        int sg;
        if (!apply_ops(cfg, cre, n_cre, ann, n_ann, &t, &sg)) continue;
        i64 it = S->index(t);
        if (it < 0) continue;
        cd a = psi[i], b = psi[it];
        psi[i] = c * a - double(sg) * sn * b;
        psi[it] = double(sg) * sn * a + c * b;
    }
}

// ---- Taylor propagation --------------------------------------------------------------------
// psi(t+dt) = e^{-i E_s dt} sum_{k=0}^{order} (-i dt)^k / k! (H - E_s)^k psi
// (Eq. 6-7; BASELINE.json configs[2]; reading U9: fixed spectral shift E_s).
void orc_taylor_step(void* s, const u64* x, const u64* z, const double* c_reim, i64 M,
                     double dt, int order, double e_shift, double* psi_reim) {
    Sector* S = (Sector*)s;
    i64 D = S->D;
    cd* psi = (cd*)psi_reim;
    std::vector<cd> term(psi, psi + D), hv(D), acc(psi, psi + D);
    for (int k = 1; k <= order; ++k) {
        orc_apply_grouped(s, x, z, c_reim, M, (const double*)term.data(), (double*)hv.data(), 0,
                          S->full ? D : S->Da);
        cd f = cd(0, -dt) / double(k);
        for (i64 i = 0; i < D; ++i) {
            term[i] = f * (hv[i] - e_shift * term[i]);
            acc[i] += term[i];
        }
    }
    cd ph = std::exp(cd(0, -e_shift * dt));
    for (i64 i = 0; i < D; ++i) psi[i] = ph * acc[i];
}

}  // extern "C"
