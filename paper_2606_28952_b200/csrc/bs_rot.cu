// a6 grouped Pauli rotations (section 2.5; Eq. 39).
//
// Generator A = sum_k c_k P_k, all strings sharing one x != 0 and mutually commuting, A^dag = -A.
// With F(t) = sum_k w_k (-1)^{popc(z_k & t)} = <t|A|t^x> (target form, w_k = c_k (-i)^{ny_k}) the
// operator is block diagonal on the pairs {t, u = t^x}: A|u> = F(t)|t>, A|t> = F(u)|u>,
// F(u) = -conj F(t), A^2 = -|F|^2 on the pair, hence
//   exp(theta A) = cos(theta r) + A sin(theta r)/r,  r = |F(t)|,
//   psi'[t] = cos(theta r) psi[t] + sin(theta r)/r F(t) psi[u],
//   psi'[u] = cos(theta r) psi[u] - sin(theta r)/r conj(F(t)) psi[t].
// Routing (pairing) and phase accumulation are computed once per pair and group.
// The pair is owned by the thread of its smaller index, so the update is in place and race free.
#include <algorithm>

#include "bs_internal.cuh"

namespace {

__device__ __forceinline__ double flipd(double v, u32 par) {
    return __hiloint2double(__double2hiint(v) ^ (int)(par << 31), __double2loint(v));
}

__device__ __forceinline__ double2 phase_sum(const u64* __restrict__ z, const double2* __restrict__ w, int k0, int k1,
                                             u64 t) {
    double fr = 0.0, fi = 0.0;
    for (int k = k0; k < k1; ++k) {
        const u32 par = (u32)__popcll(__ldg(z + k) & t) & 1u;
        const double2 wk = __ldg(w + k);
        fr += flipd(wk.x, par);
        fi += flipd(wk.y, par);
    }
    return make_double2(fr, fi);
}

// sc1 = (sin theta, cos theta) precomputed on the host for the common case |F| = 1 (fermionic excitation
// generators: |f| is 0 or 1); other moduli take the sincos path.
__device__ __forceinline__ void rotate_pair(double2* __restrict__ psi, i64 it, i64 iu, double2 F, double theta,
                                            double2 sc1) {
    const double r2 = F.x * F.x + F.y * F.y;
    if (r2 == 0.0) return;
    double sn, cs;
    if (r2 == 1.0) {
        sn = sc1.x;
        cs = sc1.y;
    } else {
        const double r = hypot(F.x, F.y);
        sincos(theta * r, &sn, &cs);
        sn /= r;
    }
    const double2 a = psi[it], b = psi[iu];
    // psi'[t] = cs a + sn F b ; psi'[u] = cs b - sn conj(F) a
    psi[it] = make_double2(cs * a.x + sn * (F.x * b.x - F.y * b.y), cs * a.y + sn * (F.x * b.y + F.y * b.x));
    psi[iu] = make_double2(cs * b.x - sn * (F.x * a.x + F.y * a.y), cs * b.y - sn * (F.x * a.y - F.y * a.x));
}

__global__ void __launch_bounds__(256)
k_rot_sector(SpinTab A, SpinTab B, int n_orb, u64 x, const u64* __restrict__ z, const double2* __restrict__ w, int k0,
             int k1, double theta, double2 sc1, double2* __restrict__ psi) {
    // grid: x = column blocks, y = alpha rows (no 64-bit division); the alpha test is uniform per block
    const u32 row = blockIdx.y, col = blockIdx.x * blockDim.x + threadIdx.x;
    const u32 xa = (u32)(x & ((u64(1) << n_orb) - 1)), xb = (u32)(x >> n_orb);
    const u32 ta = A.str[row];
    if (2 * __popc(ta & xa) != __popc(xa)) return;  // partner outside the sector: F = 0 there (leak check)
    if (col >= B.D) return;
    const u32 tb = B.str[col];
    if (2 * __popc(tb & xb) != __popc(xb)) return;
    const u32 urow = xa ? spin_rank(A, ta ^ xa) : row;
    if (urow < row) return;  // the pair belongs to its smaller index (x != 0, so iu != i)
    const u32 ucol = xb ? spin_rank(B, tb ^ xb) : col;
    if (urow == row && ucol < col) return;
    const i64 i = (i64)row * B.D + col, iu = (i64)urow * B.D + ucol;
    rotate_pair(psi, i, iu, phase_sum(z, w, k0, k1, (u64)ta | ((u64)tb << n_orb)), theta, sc1);
}

// One-off validation of a generator list against a sector: for every generator (blockIdx.y) and
// every sector configuration t whose partner t^x lies outside the sector, F(t) must vanish;
// otherwise exp(theta A) would leak out of the sector and its restriction would not be unitary.
__global__ void __launch_bounds__(256)
k_rot_leak_check(SpinTab A, SpinTab B, int n_orb, const u64* __restrict__ xg, const i64* __restrict__ offs,
                 const u64* __restrict__ z, const double2* __restrict__ w, i64 gen_lo, int* __restrict__ leak_flag) {
    const i64 i = blockIdx.x * (i64)blockDim.x + threadIdx.x;
    if (i >= A.D * B.D) return;
    const i64 j = gen_lo + blockIdx.y;
    const u64 x = xg[j];
    const u32 row = (u32)(i / B.D), col = (u32)(i - (i64)row * B.D);
    const u32 ta = A.str[row], tb = B.str[col];
    const u32 xa = (u32)(x & ((u64(1) << n_orb) - 1)), xb = (u32)(x >> n_orb);
    if ((2 * __popc(ta & xa) == __popc(xa)) && (2 * __popc(tb & xb) == __popc(xb))) return;
    const double2 F = phase_sum(z, w, (int)offs[j], (int)offs[j + 1], (u64)ta | ((u64)tb << n_orb));
    if (hypot(F.x, F.y) > 1e-12) atomicExch(leak_flag, 1);
}

__global__ void __launch_bounds__(256)
k_rot_full(i64 D, u64 x, const u64* __restrict__ z, const double2* __restrict__ w, int k0, int k1, double theta,
           double2 sc1, double2* __restrict__ psi) {
    const i64 i = blockIdx.x * (i64)blockDim.x + threadIdx.x;
    if (i >= D) return;
    const i64 iu = i ^ (i64)x;
    if (iu < i) return;
    rotate_pair(psi, i, iu, phase_sum(z, w, k0, k1, (u64)i), theta, sc1);
}

}  // namespace

extern "C" int bs_apply_pauli_rotations(bs_op_t gen, bs_sector_t s, const double* thetas, int64_t n_rot,
                                        void* psi_inout, void* cuda_stream) {
    BS_REQUIRE(gen && s, BS_ERR_ARG, "bs_apply_pauli_rotations: NULL handle");
    BS_REQUIRE(gen->mode == BS_MODE_SEQUENCE, BS_ERR_ARG,
               "bs_apply_pauli_rotations: generators must be grouped with BS_MODE_SEQUENCE");
    BS_REQUIRE(gen->n_qubits == s->n_qubits, BS_ERR_MISMATCH, "generators have %d qubits, sector has %d", gen->n_qubits,
               s->n_qubits);
    BS_REQUIRE(n_rot == gen->G, BS_ERR_ARG, "bs_apply_pauli_rotations: n_rot (%lld) != generator count (%lld)",
               (long long)n_rot, (long long)gen->G);
    BS_REQUIRE(n_rot == 0 || thetas, BS_ERR_ARG, "bs_apply_pauli_rotations: thetas is NULL");
    BS_REQUIRE(psi_inout && (reinterpret_cast<uintptr_t>(psi_inout) & 15u) == 0, BS_ERR_ARG,
               "psi is NULL or not 16-byte aligned");
    // validation: x != 0, anti-Hermitian (c purely imaginary), mutually commuting (equal ny parity)
    for (i64 j = 0; j < gen->G; ++j) {
        const u64 x = gen->h_xg[j];
        BS_REQUIRE(x != 0, BS_ERR_ARG, "generator %lld has x = 0 (diagonal generators are not rotations of pairs)",
                   (long long)j);
        int par0 = -1;
        for (i64 k = gen->h_offs[j]; k < gen->h_offs[j + 1]; ++k) {
            const double re = gen->h_c[2 * k], im = gen->h_c[2 * k + 1];
            BS_REQUIRE(fabs(re) <= 1e-14 * fabs(im) || (re == 0.0), BS_ERR_ARG,
                       "generator %lld is not anti-Hermitian (coefficient %lld has a real part)", (long long)j,
                       (long long)k);
            const int par = __builtin_popcountll(x & gen->h_z[k]) & 1;
            if (par0 < 0) par0 = par;
            BS_REQUIRE(par == par0, BS_ERR_NOT_COMMUTING, "generator %lld: strings do not mutually commute",
                       (long long)j);
        }
    }
    cudaStream_t st = (cudaStream_t)cuda_stream;
    double2* psi = (double2*)psi_inout;
    const unsigned nb = (unsigned)((s->D + 255) / 256);
    if (!s->full && std::find(gen->validated_sectors.begin(), gen->validated_sectors.end(), s->id) ==
                        gen->validated_sectors.end()) {
        BS_CUDA(cudaMemsetAsync(s->d_flag.p, 0, 4, st));
        for (i64 j = 0; j < n_rot; j += 32768) {
            dim3 grid(nb, (unsigned)std::min<i64>(32768, n_rot - j));
            k_rot_leak_check<<<grid, 256, 0, st>>>(s->ta, s->tb, s->n_orb, gen->d_xg.p, gen->d_offs.p, gen->d_z.p,
                                                   gen->d_w.p, j, s->d_flag.p);
            BS_COUNT_LAUNCH(1);
        }
        int leak = 0;
        BS_CUDA(cudaMemcpyAsync(&leak, s->d_flag.p, 4, cudaMemcpyDeviceToHost, st));
        BS_CUDA(cudaStreamSynchronize(st));
        BS_REQUIRE(!leak, BS_ERR_LEAVES_SECTOR, "a generator maps the sector outside itself");
        gen->validated_sectors.push_back(s->id);
    }
    const dim3 sgrid((unsigned)((s->Db + 255) / 256), (unsigned)std::min<i64>(s->Da, 65535));
    BS_REQUIRE(s->full || s->Da <= 65535, BS_ERR_ARG, "bs_apply_pauli_rotations: more than 65535 alpha strings");
    for (i64 j = 0; j < n_rot; ++j) {
        const int k0 = (int)gen->h_offs[j], k1 = (int)gen->h_offs[j + 1];
        const double2 sc1 = make_double2(sin(thetas[j]), cos(thetas[j]));
        if (s->full)
            k_rot_full<<<nb, 256, 0, st>>>(s->D, gen->h_xg[j], gen->d_z.p, gen->d_w.p, k0, k1, thetas[j], sc1, psi);
        else
            k_rot_sector<<<sgrid, 256, 0, st>>>(s->ta, s->tb, s->n_orb, gen->h_xg[j], gen->d_z.p, gen->d_w.p, k0, k1,
                                                thetas[j], sc1, psi);
    }
    BS_COUNT_LAUNCH(n_rot);
    BS_CUDA(cudaGetLastError());
    return BS_OK;
}
