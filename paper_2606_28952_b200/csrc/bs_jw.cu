// Device-side Jordan-Wigner construction (Alg. 1): every one-body ladder product is
// expanded into 4 and every two-body product into 16 binary-symplectic strings by one thread each, written
// straight into the device arrays that the canonical reduction (a1, bs_group.cu) sorts and merges -- the
// raw term list (0.94 GB at 56 qubits) never exists on the host.
//
// Ladder operators in XZ-ordered form (Eq. 23; Eq. 13): with b = 1 << P, lt = b - 1,
//   a_P^dag = 1/2 R(b, lt) + 1/2 R(b, lt | b),   a_P = 1/2 R(b, lt) - 1/2 R(b, lt | b);
// product rule (Eq. 19-21): R(x1,z1) R(x2,z2) = (-1)^{popc(z1 & x2)} R(x1^x2, z1^z2);
// true-Pauli coefficient: c = C (-i)^{popc(x & z)}.
#include "bs_internal.cuh"

int bs_group_canonical_dev(bs_op* op, const u64* x0, const u64* z0, const double2* c0, i64 M0, double eps,
                           cudaStream_t st);

namespace {

// string number `pattern` (bit j = which of the two strings of operator j) of coef * op_0 op_1 ... op_{k-1}
template <int K>
__device__ __forceinline__ void emit(const int (&idx)[K], u32 dagger_mask, u32 pattern, double coef, u64& xo, u64& zo,
                                     double2& co) {
    u64 x = 0, z = 0;
    u32 sign = 0;
#pragma unroll
    for (int j = 0; j < K; ++j) {
        const u64 bit = u64(1) << idx[j], lt = bit - 1;
        const bool second = (pattern >> j) & 1u;
        sign += (u32)__popcll(z & bit);
        if (second && !((dagger_mask >> j) & 1u)) ++sign;
        x ^= bit;
        z ^= second ? (lt | bit) : lt;
    }
    double v = coef * (1.0 / (1 << K));
    if (sign & 1u) v = -v;
    switch (__popcll(x & z) & 3) {  // (-i)^ny
        case 0: co = make_double2(v, 0.0); break;
        case 1: co = make_double2(0.0, -v); break;
        case 2: co = make_double2(-v, 0.0); break;
        default: co = make_double2(0.0, v); break;
    }
    xo = x;
    zo = z;
}

// H = sum_{pq,s} h_pq a^dag_{ps} a_{qs} + 1/2 sum_{pqrs} sum_{s,t} (pq|rs) a^dag_{ps} a^dag_{rt} a_{st} a_{qs}
// (Eq. 2; reading U3).  Terms 0 .. 8 n^2 - 1: one-body; then 64 n^4 two-body strings.
__global__ void k_jw_molecular(int n, const double* __restrict__ h, const double* __restrict__ g, i64 n1, i64 total,
                               u64* __restrict__ x, u64* __restrict__ z, double2* __restrict__ c) {
    const i64 t = blockIdx.x * (i64)blockDim.x + threadIdx.x;
    if (t >= total) return;
    if (t < n1) {
        const u32 pattern = (u32)(t & 3);
        i64 r = t >> 2;
        const int q = (int)(r % n);
        r /= n;
        const int p = (int)(r % n), s = (int)(r / n);
        const int idx[2] = {p + s * n, q + s * n};
        emit<2>(idx, 0x1u, pattern, h[p * n + q], x[t], z[t], c[t]);
        return;
    }
    i64 r = t - n1;
    const u32 pattern = (u32)(r & 15);
    r >>= 4;
    const int ss = (int)(r % n);
    r /= n;
    const int rr = (int)(r % n);
    r /= n;
    const int q = (int)(r % n);
    r /= n;
    const int p = (int)(r % n);
    const int st = (int)(r / n);  // spin pair: s = st >> 1, t = st & 1
    const int s1 = st >> 1, s2 = st & 1;
    const int idx[4] = {p + s1 * n, rr + s2 * n, ss + s2 * n, q + s1 * n};
    double coef = 0.5 * g[((i64)(p * n + q) * n + rr) * n + ss];
    if (idx[0] == idx[1] || idx[2] == idx[3]) coef = 0.0;  // a^dag a^dag = a a = 0 on equal indices
    emit<4>(idx, 0x3u, pattern, coef, x[t], z[t], c[t]);
}

// H = -t sum_{i,s} (a^dag_{is} a_{i+1,s} + h.c.) + U sum_i n_{i,alpha} n_{i,beta}, open chain
__global__ void k_jw_hubbard(int L, double thop, double U, i64 n1, i64 total, u64* __restrict__ x, u64* __restrict__ z,
                             double2* __restrict__ c) {
    const i64 t = blockIdx.x * (i64)blockDim.x + threadIdx.x;
    if (t >= total) return;
    if (t < n1) {  // (L-1) bonds x 2 spins x 2 directions x 4 strings
        const u32 pattern = (u32)(t & 3);
        i64 r = t >> 2;
        const int dir = (int)(r & 1);
        r >>= 1;
        const int i = (int)(r % (L - 1)), s = (int)(r / (L - 1));
        const int a = i + dir + s * L, b = i + 1 - dir + s * L;
        const int idx[2] = {a, b};
        emit<2>(idx, 0x1u, pattern, -thop, x[t], z[t], c[t]);
        return;
    }
    const i64 r = t - n1;
    const u32 pattern = (u32)(r & 15);
    const int i = (int)(r >> 4);
    const int idx[4] = {i, i, i + L, i + L};
    emit<4>(idx, 0x5u, pattern, U, x[t], z[t], c[t]);  // a^dag a a^dag a
}

int finish_jw(int n_qubits, DevBuf<u64>& x, DevBuf<u64>& z, DevBuf<double2>& c, i64 total, double eps, cudaStream_t st,
              bs_op_t* out) {
    BS_CUDA(cudaGetLastError());
    bs_op* op = new (std::nothrow) bs_op;
    BS_REQUIRE(op, BS_ERR_ALLOC, "bs_jw: host allocation failed");
    op->id = bs_next_id();
    op->n_qubits = n_qubits;
    op->mode = BS_MODE_CANONICAL;
    int rc = bs_group_canonical_dev(op, x.p, z.p, c.p, total, eps, st);
    if (rc != BS_OK) {
        delete op;
        return rc;
    }
    *out = op;
    return BS_OK;
}

}  // namespace

extern "C" int bs_jw_molecular(int n_orb, const double* h, const double* g, double eps_drop, void* cuda_stream,
                               bs_op_t* out) {
    BS_REQUIRE(out && h && g, BS_ERR_ARG, "bs_jw_molecular: NULL argument");
    BS_REQUIRE(n_orb >= 1 && n_orb <= 32, BS_ERR_ARG, "bs_jw_molecular: n_orb must be in [1, 32]");
    int dev_count = 0;
    BS_CUDA(cudaGetDeviceCount(&dev_count));
    BS_REQUIRE(dev_count > 0, BS_ERR_CUDA, "no CUDA device (libbs has no CPU fallback)");
    cudaStream_t st = (cudaStream_t)cuda_stream;
    const i64 n = n_orb, n2 = n * n, n4 = n2 * n2;
    const i64 n1 = 8 * n2, total = n1 + 64 * n4;
    BS_REQUIRE(total < (i64(1) << 31), BS_ERR_ARG, "bs_jw_molecular: too many raw terms");
    DevBuf<double> dh, dg;
    DevBuf<u64> x, z;
    DevBuf<double2> c;
    BS_CUDA(dh.alloc(n2));
    BS_CUDA(dg.alloc(n4));
    BS_CUDA(x.alloc(total));
    BS_CUDA(z.alloc(total));
    BS_CUDA(c.alloc(total));
    BS_CUDA(cudaMemcpyAsync(dh.p, h, n2 * 8, cudaMemcpyHostToDevice, st));
    BS_CUDA(cudaMemcpyAsync(dg.p, g, n4 * 8, cudaMemcpyHostToDevice, st));
    k_jw_molecular<<<(unsigned)((total + 255) / 256), 256, 0, st>>>(n_orb, dh.p, dg.p, n1, total, x.p, z.p, c.p);
    BS_COUNT_LAUNCH(1);
    return finish_jw(2 * n_orb, x, z, c, total, eps_drop, st, out);
}

extern "C" int bs_jw_hubbard(int n_sites, double t, double U, double eps_drop, void* cuda_stream, bs_op_t* out) {
    BS_REQUIRE(out, BS_ERR_ARG, "bs_jw_hubbard: out is NULL");
    BS_REQUIRE(n_sites >= 2 && n_sites <= 32, BS_ERR_ARG, "bs_jw_hubbard: n_sites must be in [2, 32]");
    int dev_count = 0;
    BS_CUDA(cudaGetDeviceCount(&dev_count));
    BS_REQUIRE(dev_count > 0, BS_ERR_CUDA, "no CUDA device (libbs has no CPU fallback)");
    cudaStream_t st = (cudaStream_t)cuda_stream;
    const i64 n1 = (i64)(n_sites - 1) * 2 * 2 * 4, total = n1 + (i64)n_sites * 16;
    DevBuf<u64> x, z;
    DevBuf<double2> c;
    BS_CUDA(x.alloc(total));
    BS_CUDA(z.alloc(total));
    BS_CUDA(c.alloc(total));
    k_jw_hubbard<<<(unsigned)((total + 255) / 256), 256, 0, st>>>(n_sites, t, U, n1, total, x.p, z.p, c.p);
    BS_COUNT_LAUNCH(1);
    return finish_jw(2 * n_sites, x, z, c, total, eps_drop, st, out);
}
