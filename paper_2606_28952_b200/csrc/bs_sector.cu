// a3 sector tables (Eq. 25, 28, 38).
//
// Per spin s: unrank array str_s[D_s] = all n_orb-bit words of popcount N_s in increasing numeric
// order (Gosper's next-combination walk) and a two-chunk rank lookup in the combinatorial number
// system: for w with set bits p_1 < ... < p_k, rank(w) = sum_i C(p_i, i).  Splitting w into a low
// chunk (bits_lo bits) and a high chunk, the low bits contribute lo[low] and the high bits
// contribute hi[popc(low)][high] = sum_j C(bits_lo + q_j, popc(low) + j): two table loads and a
// POPC per rank instead of N_s binomial terms.  This is the "two smaller spin-string index
// searches" of PAPER.md:247 done as lookups.
#include "bs_internal.cuh"

namespace {

struct Binom {
    u64 c[65][34];
    Binom() {
        for (int n = 0; n <= 64; ++n)
            for (int k = 0; k <= 33; ++k) {
                if (k == 0) c[n][k] = 1;
                else if (n == 0) c[n][k] = 0;
                else {
                    u64 v = c[n - 1][k - 1] + c[n - 1][k];
                    c[n][k] = v;
                }
            }
    }
    u64 operator()(int n, int k) const { return (k < 0 || k > 33 || n < 0) ? 0 : (k > n ? 0 : c[n][k]); }
};
const Binom& binom() {
    static Binom b;
    return b;
}

void enum_strings(int n, int N, std::vector<u64>& out) {
    out.clear();
    u64 D = binom()(n, N);
    out.reserve(D);
    if (N == 0) {
        out.push_back(0);
        return;
    }
    u64 w = (u64(1) << N) - 1, lim = u64(1) << n;
    while (w < lim) {
        out.push_back(w);
        u64 c = w & (~w + 1), r = w + c;       // Gosper: next word with the same popcount
        w = (((r ^ w) >> 2) / c) | r;
    }
}

void rank_tables(int n, int N, int& bits_lo, int& bits_hi, std::vector<u32>& lo, std::vector<u32>& hi) {
    bits_lo = (n <= 16) ? n : (n + 1) / 2;
    bits_hi = n - bits_lo;
    const Binom& B = binom();
    lo.assign(size_t(1) << bits_lo, 0);
    for (u32 w = 0; w < (u32(1) << bits_lo); ++w) {
        u64 r = 0;
        int i = 0;
        for (int p = 0; p < bits_lo; ++p)
            if (w >> p & 1) r += B(p, ++i);
        lo[w] = (i <= N) ? (u32)r : 0;
    }
    hi.clear();
    if (bits_hi == 0) return;
    hi.assign(size_t(N + 1) << bits_hi, 0);
    for (int k = 0; k <= N; ++k)
        for (u32 w = 0; w < (u32(1) << bits_hi); ++w) {
            u64 r = 0;
            int j = 0;
            for (int q = 0; q < bits_hi; ++q)
                if (w >> q & 1) r += B(bits_lo + q, k + (++j));
            hi[(size_t(k) << bits_hi) | w] = (k + j <= N) ? (u32)r : 0;
        }
}

__global__ void k_rank_configs(SpinTab A, SpinTab Bt, int n_orb, int full, int n_qubits, const u64* __restrict__ cfg,
                               i64* __restrict__ out, i64 n) {
    i64 i = blockIdx.x * (i64)blockDim.x + threadIdx.x;
    if (i >= n) return;
    u64 c = cfg[i];
    if (full) {
        out[i] = (n_qubits < 64 && (c >> n_qubits)) ? -1 : (i64)c;
        return;
    }
    u64 ma = (n_orb == 64) ? ~u64(0) : ((u64(1) << n_orb) - 1);
    u64 a = c & ma, b = c >> n_orb;
    if ((2 * n_orb < 64 && (c >> (2 * n_orb))) || __popcll(a) != A.N || __popcll(b) != Bt.N) {
        out[i] = -1;
        return;
    }
    out[i] = (i64)spin_rank(A, (u32)a) * Bt.D + (i64)spin_rank(Bt, (u32)b);
}

int build_spin(int n, int N, cudaStream_t st, std::vector<u64>& hs, DevBuf<u32>& dstr, DevBuf<u32>& dlo,
               DevBuf<u32>& dhi, SpinTab& T) {
    enum_strings(n, N, hs);
    std::vector<u32> s32(hs.begin(), hs.end()), lo, hi;
    int bl, bh;
    rank_tables(n, N, bl, bh, lo, hi);
    BS_CUDA(dstr.upload(s32, st));
    BS_CUDA(dlo.upload(lo, st));
    BS_CUDA(dhi.upload(hi, st));
    BS_CUDA(cudaStreamSynchronize(st));  // the host vectors go out of scope
    T.str = dstr.p;
    T.lo = dlo.p;
    T.hi = dhi.p;
    T.bits_lo = bl;
    T.bits_hi = bh;
    T.N = N;
    T.mask_lo = (bl >= 32) ? 0xffffffffu : ((u32(1) << bl) - 1);
    T.D = (i64)hs.size();
    return BS_OK;
}

}  // namespace

extern "C" int bs_sector_build(int n_orb, int n_alpha, int n_beta, void* cuda_stream, bs_sector_t* out) {
    BS_REQUIRE(out, BS_ERR_ARG, "bs_sector_build: out is NULL");
    bool full = (n_alpha < 0 && n_beta < 0);
    if (full) {
        BS_REQUIRE(n_orb >= 1 && n_orb <= 40, BS_ERR_ARG, "bs_sector_build: full space needs 1 <= n_qubits <= 40");
    } else {
        BS_REQUIRE(n_orb >= 1 && n_orb <= 32, BS_ERR_ARG, "bs_sector_build: sector mode needs 1 <= n_orb <= 32");
        BS_REQUIRE(n_alpha >= 0 && n_alpha <= n_orb && n_beta >= 0 && n_beta <= n_orb, BS_ERR_ARG,
                   "bs_sector_build: electron counts out of range");
    }
    int dev_count = 0;
    BS_CUDA(cudaGetDeviceCount(&dev_count));
    BS_REQUIRE(dev_count > 0, BS_ERR_CUDA, "no CUDA device (libbs has no CPU fallback)");
    cudaStream_t st = (cudaStream_t)cuda_stream;
    bs_sector* s = new (std::nothrow) bs_sector;
    BS_REQUIRE(s, BS_ERR_ALLOC, "bs_sector_build: host allocation failed");
    s->id = bs_next_id();
    s->full = full;
    s->n_orb = n_orb;
    s->n_alpha = n_alpha;
    s->n_beta = n_beta;
    std::memset(&s->ta, 0, sizeof(SpinTab));
    std::memset(&s->tb, 0, sizeof(SpinTab));
    int rc = BS_OK;
    if (full) {
        s->n_qubits = n_orb;
        s->Da = 1;
        s->Db = 1;
        s->D = i64(1) << n_orb;
    } else {
        s->n_qubits = 2 * n_orb;
        u64 da = binom()(n_orb, n_alpha), db = binom()(n_orb, n_beta);
        if (da > (u64(1) << 31) || db > (u64(1) << 31)) {
            bs_set_error("bs_sector_build: spin-string space too large");
            delete s;
            return BS_ERR_ARG;
        }
        rc = build_spin(n_orb, n_alpha, st, s->h_sa, s->d_sa, s->d_lo_a, s->d_hi_a, s->ta);
        if (rc == BS_OK) rc = build_spin(n_orb, n_beta, st, s->h_sb, s->d_sb, s->d_lo_b, s->d_hi_b, s->tb);
        s->Da = (i64)da;
        s->Db = (i64)db;
        s->D = s->Da * s->Db;
    }
    if (rc == BS_OK) {
        cudaError_t e = s->d_partials.alloc(1 << 16);
        if (e == cudaSuccess) e = s->d_result.alloc(4);
        if (e == cudaSuccess) e = s->d_flag.alloc(4);
        if (e == cudaSuccess) e = cudaMemsetAsync(s->d_flag.p, 0, 16, st);
        if (e != cudaSuccess) {
            bs_set_error("bs_sector_build: %s", cudaGetErrorString(e));
            rc = BS_ERR_ALLOC;
        }
    }
    if (rc != BS_OK) {
        delete s;
        return rc;
    }
    *out = s;
    return BS_OK;
}

extern "C" int bs_sector_info(bs_sector_t s, int64_t* dim, int64_t* dim_alpha, int64_t* dim_beta) {
    BS_REQUIRE(s, BS_ERR_ARG, "bs_sector_info: NULL handle");
    if (dim) *dim = s->D;
    if (dim_alpha) *dim_alpha = s->Da;
    if (dim_beta) *dim_beta = s->Db;
    return BS_OK;
}

extern "C" int bs_sector_export(bs_sector_t s, uint64_t* alpha_strings, uint64_t* beta_strings) {
    BS_REQUIRE(s, BS_ERR_ARG, "bs_sector_export: NULL handle");
    BS_REQUIRE(!s->full, BS_ERR_ARG, "bs_sector_export: full-space mode has no string tables");
    if (alpha_strings) std::memcpy(alpha_strings, s->h_sa.data(), s->h_sa.size() * 8);
    if (beta_strings) std::memcpy(beta_strings, s->h_sb.data(), s->h_sb.size() * 8);
    return BS_OK;
}

extern "C" int bs_sector_rank(bs_sector_t s, const uint64_t* configs, int64_t n, int64_t* index_out) {
    BS_REQUIRE(s && (n == 0 || (configs && index_out)) && n >= 0, BS_ERR_ARG, "bs_sector_rank: bad argument");
    if (n == 0) return BS_OK;
    DevBuf<u64> dc;
    DevBuf<i64> di;
    BS_CUDA(dc.alloc(n));
    BS_CUDA(di.alloc(n));
    BS_CUDA(cudaMemcpy(dc.p, configs, n * 8, cudaMemcpyHostToDevice));
    k_rank_configs<<<(unsigned)((n + 255) / 256), 256>>>(s->ta, s->tb, s->n_orb, s->full ? 1 : 0, s->n_qubits, dc.p,
                                                         di.p, n);
    BS_COUNT_LAUNCH(1);
    BS_CUDA(cudaGetLastError());
    BS_CUDA(cudaMemcpy(index_out, di.p, n * 8, cudaMemcpyDeviceToHost));
    return BS_OK;
}

extern "C" int bs_sector_destroy(bs_sector_t s) {
    if (!s) return BS_OK;
    bs_plan_purge(0, s->id);
    delete s;
    return BS_OK;
}
