// a4, same-spin double excitations resolved over (N - 2)-electron strings: plan tables and kernels (see bs_k2.cuh).
// PAPER.md:220-231 (Eq. 27-28).
#include <algorithm>

#include "bs_epilogue.cuh"
#include "bs_k2.cuh"

namespace {

constexpr int kAaThreads = 256;

// combinadic (colex) rank of a word with exactly four bits set: C(p1,1) + C(p2,2) + C(p3,3) + C(p4,4)
__host__ __device__ inline u32 rank4(u32 x) {
    u32 r = 0;
#ifdef __CUDA_ARCH__
    u32 p = (u32)__ffs((int)x) - 1u;
#else
    u32 p = (u32)__builtin_ctz(x);
#endif
    r += p;
    x &= x - 1;
#ifdef __CUDA_ARCH__
    p = (u32)__ffs((int)x) - 1u;
#else
    p = (u32)__builtin_ctz(x);
#endif
    r += p * (p - 1) / 2;
    x &= x - 1;
#ifdef __CUDA_ARCH__
    p = (u32)__ffs((int)x) - 1u;
#else
    p = (u32)__builtin_ctz(x);
#endif
    r += p * (p - 1) * (p - 2) / 6;
    x &= x - 1;
#ifdef __CUDA_ARCH__
    p = (u32)__ffs((int)x) - 1u;
#else
    p = (u32)__builtin_ctz(x);
#endif
    r += (u32)((u64)p * (p - 1) * (p - 2) * (p - 3) / 24);
    return r;
}

// block = (family, tile of RT target members); thread = one column per pass over the slab [c0, c0 + W)
template <int RT>
__global__ void __launch_bounds__(kAaThreads)
k_aa(const K2Dev K, const double2* __restrict__ psi, double2* __restrict__ S2, i64 L, i64 c0, i64 W, i64 row_lo,
     i64 row_hi) {
    extern __shared__ __align__(16) unsigned char smem_k2[];
    // the tiles of one family are neighbours in launch order: they stream the same source rows, which L2 then serves
    const int P = K.P, f = blockIdx.y, t0 = blockIdx.x * RT, nt = min(RT, P - t0), tid = threadIdx.x;
    double* sC = reinterpret_cast<double*>(smem_k2);                       // [P + 4][RT] coupling tile, source-major
    u32* srow = reinterpret_cast<u32*>(smem_k2 + (size_t)(P + 4) * RT * 8);  // [P + 4] row of every source member
    const u32* __restrict__ mrow = K.mrow + (size_t)f * P;
    const u32* __restrict__ mpair = K.mpair + (size_t)f * P;
    bool any = false;   // block-uniform: some target of the tile lies in the requested row range
    for (int tt = 0; tt < nt; ++tt) {
        const i64 r = __ldg(mrow + t0 + tt);
        any |= r >= row_lo && r < row_hi;
    }
    if (!any) return;
    const u32 k2 = __ldg(K.fk2 + f);
    for (int idx = tid; idx < (P + 4) * RT; idx += kAaThreads) {
        const int u = idx / RT, tt = idx - u * RT;
        double v = 0.0;
        if (u < P && tt < nt) {
            const u32 pt = __ldg(mpair + t0 + tt), pu = __ldg(mpair + u);
            if (!(pt & pu)) {   // disjoint pairs: a double excitation; its group by the rank of the 4-bit mask
                const u32 g = rank4(pt | pu), t = k2 | pt;
                const u32 s1 = __ldg(K.goff + g + 1);
                for (u32 s = __ldg(K.goff + g); s < s1; ++s)
                    v += flip(__ldg(K.gw + s), (u32)__popc(__ldg(K.gza + s) & t) & 1u);
            }
        }
        sC[idx] = v;
    }
    for (int u = tid; u < P + 4; u += kAaThreads) srow[u] = u < P ? __ldg(mrow + u) : 0u;
    __syncthreads();
    for (i64 c = c0 + tid; c < c0 + W; c += kAaThreads) {
        double2 acc[RT];
#pragma unroll
        for (int tt = 0; tt < RT; ++tt) acc[tt] = make_double2(0.0, 0.0);
        const double2* __restrict__ pc = psi + c;
        double2 a[4], an[4];   // four source rows being consumed, the next four in flight (rows beyond P read row 0
                               // against a zero coupling row)
#pragma unroll
        for (int k = 0; k < 4; ++k) a[k] = __ldg(pc + (i64)srow[k] * L);
        for (int u = 0; u < P; u += 4) {
            if (u + 4 < P) {
#pragma unroll
                for (int k = 0; k < 4; ++k) an[k] = __ldg(pc + (i64)srow[u + 4 + k] * L);
            }
#pragma unroll
            for (int k = 0; k < 4; ++k) {
                const double2* __restrict__ g2 = reinterpret_cast<const double2*>(sC + (u + k) * RT);
#pragma unroll
                for (int t2 = 0; t2 < RT / 2; ++t2) {
                    const double2 g = g2[t2];   // warp-uniform address
                    acc[2 * t2].x += g.x * a[k].x;
                    acc[2 * t2].y += g.x * a[k].y;
                    acc[2 * t2 + 1].x += g.y * a[k].x;
                    acc[2 * t2 + 1].y += g.y * a[k].y;
                }
            }
#pragma unroll
            for (int k = 0; k < 4; ++k) a[k] = an[k];
        }
        double2* __restrict__ so = S2 + ((i64)f * P + t0) * W + (c - c0);
#pragma unroll
        for (int tt = 0; tt < RT; ++tt)
            if (tt < nt) so[(i64)tt * W] = acc[tt];
    }
}

// Tensor-instruction form (mma.sync.m8n8k4.f64, SASS DMMA; same FP64 peak as DFMA, see profiles/r02_fp64_peak.md): a warp
// owns 8 RTW columns (RTW row tiles of 8) x 8 NT targets and keeps the amplitudes of the next DEPTH steps in registers.
// One 16-byte amplitude load per lane and row tile feeds 2 NT DMMAs: with <NT, RTW, DEPTH> = <2, 4, 1> the kernel ran at
// half the tensor pipe because only 32 KB per SM were in flight against ~2,150 cycles of L2 latency
// (profiles/r02b_q32_k_ab_k_aa_full.md); <3, 2, 3> and <4, 2, 3> need 1.5x / 2x fewer bytes per DMMA and hold 1.5x more
// in flight per warp at the same accumulator registers.  A[column][u] = psi[source member u][column] (re and im as separate
// tiles), B[u][target] = the coupling tile, four source members per step.  One B fragment load feeds 8 columns: the
// warp-uniform coupling loads of the DFMA form (65 % of the shared-memory pipe, profiles/r02_q32_k_aa_full.md) shrink 12x.
__host__ __device__ constexpr int k2_gs(int NT) { return 8 * NT + 4; }   // row stride of the coupling tile: conflict-free fragments

// entry (source member u, target tt of the tile at t0) of a family's coupling tile: F_g(t) of the double excitation that
// takes member u to member t0 + tt, 0 if the two pairs overlap or the slot is padding
__device__ __forceinline__ double k2_tile_entry(const K2Dev& K, const u32* __restrict__ mpair, u32 k2, int t0, int nt,
                                                int u, int tt) {
    double v = 0.0;
    if (u < K.P && tt < nt) {
        const u32 pt = __ldg(mpair + t0 + tt), pu = __ldg(mpair + u);
        if (!(pt & pu)) {   // disjoint pairs: a double excitation; its group by the rank of the 4-bit mask
            const u32 g = rank4(pt | pu), t = k2 | pt;
            const u32 s1 = __ldg(K.goff + g + 1);
            for (u32 s = __ldg(K.goff + g); s < s1; ++s)
                v += flip(__ldg(K.gw + s), (u32)__popc(__ldg(K.gza + s) & t) & 1u);
        }
    }
    return v;
}

// fallback of k_aa_mma when the tiles were not evaluated at plan time; not inlined, so that its registers (table
// pointers, string loop) do not count against the contraction loop, which sits at the 128-register cap
__device__ __noinline__ void k2_fill_tile(const K2Dev& K, int f, int t0, int nt, int GS, double* sC) {
    const u32* __restrict__ mpair = K.mpair + (size_t)f * K.P;
    const u32 k2 = __ldg(K.fk2 + f);
    for (int idx = threadIdx.x; idx < (K.P + 4) * GS; idx += kAaThreads) {
        const int u = idx / GS, tt = idx - u * GS;
        sC[idx] = k2_tile_entry(K, mpair, k2, t0, nt, u, tt);
    }
}

// plan time: every (family, target tile) coupling tile of the tensor form, in the layout k_aa_mma keeps in shared memory
template <int NT>
__global__ void __launch_bounds__(kAaThreads) k_aa_tiles(const K2Dev K, double* __restrict__ out) {
    constexpr int RT = 8 * NT, GS = k2_gs(NT);
    const int P = K.P, f = blockIdx.y, t0 = blockIdx.x * RT, nt = min(RT, P - t0);
    const u32* __restrict__ mpair = K.mpair + (size_t)f * P;
    const u32 k2 = __ldg(K.fk2 + f);
    double* o = out + ((size_t)f * K.n_tiles + blockIdx.x) * (size_t)(P + 4) * GS;
    for (int idx = threadIdx.x; idx < (P + 4) * GS; idx += kAaThreads) {
        const int u = idx / GS, tt = idx - u * GS;
        o[idx] = k2_tile_entry(K, mpair, k2, t0, nt, u, tt);
    }
}

template <int NT, int RTW, int DEPTH>
__global__ void __launch_bounds__(kAaThreads, 2)
k_aa_mma(const K2Dev K, const double2* __restrict__ psi, double2* __restrict__ S2, i64 L, i64 c0, i64 W, i64 row_lo,
         i64 row_hi) {
    extern __shared__ __align__(16) unsigned char smem_k2[];
    constexpr int RT = 8 * NT, GS = k2_gs(NT), CW = 8 * RTW;   // CW: columns per warp
    const int P = K.P, f = blockIdx.y, t0 = blockIdx.x * RT, nt = min(RT, P - t0), tid = threadIdx.x;
    double* sC = reinterpret_cast<double*>(smem_k2);                          // [P + 4][GS] coupling tile, source-major
    u32* srow = reinterpret_cast<u32*>(smem_k2 + (size_t)(P + 4) * GS * 8);    // [P + 4] row of every source member
    const u32* __restrict__ mrow = K.mrow + (size_t)f * P;
    bool any = false;   // block-uniform: some target of the tile lies in the requested row range
    for (int tt = 0; tt < nt; ++tt) {
        const i64 r = __ldg(mrow + t0 + tt);
        any |= r >= row_lo && r < row_hi;
    }
    if (!any) return;
    if (K.ctile) {   // the tile was evaluated at plan time: (P + 4) * GS doubles, a multiple of 4: 16-byte copies
        const double2* __restrict__ src =
            reinterpret_cast<const double2*>(K.ctile + ((size_t)f * K.n_tiles + blockIdx.x) * (size_t)(P + 4) * GS);
        double2* dst = reinterpret_cast<double2*>(sC);
        for (int idx = tid; idx < (P + 4) * GS / 2; idx += kAaThreads) dst[idx] = __ldg(src + idx);
    } else {
        k2_fill_tile(K, f, t0, nt, GS, sC);
    }
    for (int u = tid; u < P + 4; u += kAaThreads) srow[u] = u < P ? __ldg(mrow + u) : 0u;
    __syncthreads();
    const int lane = tid & 31, warp = tid >> 5, g = lane >> 2, tq = lane & 3;
    for (i64 cb = c0 + warp * CW; cb < c0 + W; cb += (kAaThreads / 32) * CW) {
        double cr[RTW][NT][2], ci[RTW][NT][2];
#pragma unroll
        for (int i = 0; i < RTW; ++i)
#pragma unroll
            for (int j = 0; j < NT; ++j) cr[i][j][0] = cr[i][j][1] = ci[i][j][0] = ci[i][j][1] = 0.0;
        bool okc[RTW];
        const double2* pc[RTW];
#pragma unroll
        for (int i = 0; i < RTW; ++i) {
            const i64 c = cb + 8 * i + g;
            okc[i] = c < c0 + W;
            pc[i] = psi + (okc[i] ? c : c0);
        }
        double2 q[DEPTH][RTW];   // q[0]: this step's amplitudes; q[1 .. DEPTH-1] and nx: the next DEPTH steps', in flight
#pragma unroll
        for (int d = 0; d < DEPTH; ++d) {
            const bool have = 4 * d < P;
            const i64 ro = have ? (i64)srow[4 * d + tq] * L : 0;
#pragma unroll
            for (int i = 0; i < RTW; ++i) q[d][i] = have ? __ldg(pc[i] + ro) : make_double2(0.0, 0.0);
        }
        for (int u = 0; u < P; u += 4) {
            double2 nx[RTW];
            if (u + 4 * DEPTH < P) {
                const i64 ro = (i64)srow[u + 4 * DEPTH + tq] * L;
#pragma unroll
                for (int i = 0; i < RTW; ++i) nx[i] = __ldg(pc[i] + ro);
            } else {
#pragma unroll
                for (int i = 0; i < RTW; ++i) nx[i] = make_double2(0.0, 0.0);
            }
            double bf[NT];
#pragma unroll
            for (int j = 0; j < NT; ++j) bf[j] = sC[(u + tq) * GS + 8 * j + g];
#pragma unroll
            for (int i = 0; i < RTW; ++i) {
                const double are = okc[i] ? q[0][i].x : 0.0, aim = okc[i] ? q[0][i].y : 0.0;
#pragma unroll
                for (int j = 0; j < NT; ++j) {
                    asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};"
                                 : "+d"(cr[i][j][0]), "+d"(cr[i][j][1]) : "d"(are), "d"(bf[j]));
                    asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};"
                                 : "+d"(ci[i][j][0]), "+d"(ci[i][j][1]) : "d"(aim), "d"(bf[j]));
                }
            }
#pragma unroll
            for (int i = 0; i < RTW; ++i) {
#pragma unroll
                for (int d = 0; d + 1 < DEPTH; ++d) q[d][i] = q[d + 1][i];
                q[DEPTH - 1][i] = nx[i];
            }
        }
        // C fragment: row g of tile i (column cb + 8 i + g), targets 8 j + 2 tq + {0, 1}
#pragma unroll
        for (int i = 0; i < RTW; ++i)
#pragma unroll
            for (int j = 0; j < NT; ++j)
#pragma unroll
                for (int e = 0; e < 2; ++e) {
                    const int tt = 8 * j + 2 * tq + e;
                    if (okc[i] && tt < nt)
                        S2[((i64)f * P + t0 + tt) * W + (cb + 8 * i + g - c0)] = make_double2(cr[i][j][e], ci[i][j][e]);
                }
    }
}

// acc[r][c] += sum_j S2[tf[r][j]][c - c0], j in fixed order
__global__ void __launch_bounds__(256)
k_aa_acc(const u32* __restrict__ tf, int NP2, const double2* __restrict__ S2, double2* __restrict__ acc, i64 L, i64 W,
         i64 c0, i64 row_lo) {
    const i64 cl = blockIdx.x * (i64)blockDim.x + threadIdx.x;
    if (cl >= W) return;
    const i64 r = row_lo + blockIdx.y;
    const u32* __restrict__ t = tf + r * NP2;
    double2 s = make_double2(0.0, 0.0);
    for (int j = 0; j < NP2; ++j) {
        const double2 v = __ldg(S2 + (i64)__ldg(t + j) * W + cl);
        s.x += v.x;
        s.y += v.y;
    }
    double2* o = acc + r * L + c0 + cl;
    double2 a = *o;
    a.x += s.x;
    a.y += s.y;
    *o = a;
}

template <int RT>
cudaError_t kaa_launch(const bs_k2* K, const double2* psi, i64 L, i64 c0, i64 W, i64 row_lo, i64 row_hi, cudaStream_t st,
                       bool set_attr) {
    if (set_attr) return cudaFuncSetAttribute(k_aa<RT>, cudaFuncAttributeMaxDynamicSharedMemorySize, 200 * 1024);   // the ceiling is per kernel,
                                                                  // shared by all plans: never lower it to one plan's size
    dim3 grid((unsigned)K->n_tiles, (unsigned)K->F);
    k_aa<RT><<<grid, kAaThreads, K->smem, st>>>(K->dev, psi, K->d_S2.p, L, c0, W, row_lo, row_hi);
    return cudaGetLastError();
}

template <int NT, int RTW, int DEPTH>
cudaError_t kaa_mma_launch(const bs_k2* K, const double2* psi, i64 L, i64 c0, i64 W, i64 row_lo, i64 row_hi,
                           cudaStream_t st, bool set_attr) {
    if (set_attr)
        return cudaFuncSetAttribute(k_aa_mma<NT, RTW, DEPTH>, cudaFuncAttributeMaxDynamicSharedMemorySize, 200 * 1024);
    dim3 grid((unsigned)K->n_tiles, (unsigned)K->F);
    k_aa_mma<NT, RTW, DEPTH><<<grid, kAaThreads, K->smem, st>>>(K->dev, psi, K->d_S2.p, L, c0, W, row_lo, row_hi);
    return cudaGetLastError();
}

cudaError_t kaa_dispatch(const bs_k2* K, const double2* psi, i64 L, i64 c0, i64 W, i64 row_lo, i64 row_hi,
                         cudaStream_t st, bool set_attr) {
    if (K->mma) switch (K->rt) {   // <target tiles NT, row tiles per warp, prefetch depth>
            case 8: return kaa_mma_launch<1, 4, 1>(K, psi, L, c0, W, row_lo, row_hi, st, set_attr);
            case 16: return kaa_mma_launch<2, 4, 1>(K, psi, L, c0, W, row_lo, row_hi, st, set_attr);
            case 24: return kaa_mma_launch<3, 2, 3>(K, psi, L, c0, W, row_lo, row_hi, st, set_attr);
            default: return kaa_mma_launch<4, 2, 3>(K, psi, L, c0, W, row_lo, row_hi, st, set_attr);
        }
    switch (K->rt) {
        case 4: return kaa_launch<4>(K, psi, L, c0, W, row_lo, row_hi, st, set_attr);
        case 8: return kaa_launch<8>(K, psi, L, c0, W, row_lo, row_hi, st, set_attr);
        case 12: return kaa_launch<12>(K, psi, L, c0, W, row_lo, row_hi, st, set_attr);
        case 16: return kaa_launch<16>(K, psi, L, c0, W, row_lo, row_hi, st, set_attr);
        case 20: return kaa_launch<20>(K, psi, L, c0, W, row_lo, row_hi, st, set_attr);
        case 24: return kaa_launch<24>(K, psi, L, c0, W, row_lo, row_hi, st, set_attr);
        default: return kaa_launch<28>(K, psi, L, c0, W, row_lo, row_hi, st, set_attr);
    }
}

}  // namespace

int bs_k2_build(std::vector<HostGroup>& groups, const std::vector<u64>& row_strings, int n, int N, i64 row_len,
                cudaStream_t st, bs_k2** out) {
    *out = nullptr;
    if (getenv("BS_NO_K2")) return BS_OK;   // test hook (include/bs.h "Environment")
    if (n < 4 || n > 32 || N < 2 || n - N < 2 || row_len < 32) return BS_OK;
    auto qualifies = [](const HostGroup& g) {
        if (g.xb != 0 || __builtin_popcount(g.xa) != 4) return false;
        for (auto& s : g.s)
            if (s.zb != 0 || s.im != 0.0) return false;   // one key (no column-spin sign), real weights
        return true;
    };
    i64 n_q = 0;
    for (auto& g : groups) n_q += qualifies(g);
    const int min_groups = getenv("BS_K2_MIN") ? atoi(getenv("BS_K2_MIN")) : 16;
    if (n_q < min_groups) return BS_OK;
    const i64 rows = (i64)row_strings.size();
    // ---- group strings by the combinadic rank of the 4-bit mask -----------------------------------------------
    const u32 n4 = (u32)((u64)n * (n - 1) * (n - 2) * (n - 3) / 24);
    std::vector<u32> goff(n4 + 1, 0u), gza;
    std::vector<double> gw;
    {
        std::vector<const HostGroup*> by_rank(n4, nullptr);
        for (auto& g : groups)
            if (qualifies(g)) by_rank[rank4(g.xa)] = &g;
        for (u32 r = 0; r < n4; ++r) {
            goff[r] = (u32)gza.size();
            if (by_rank[r])
                for (auto& s : by_rank[r]->s) {
                    gza.push_back(s.za);
                    gw.push_back(s.re);
                }
        }
        goff[n4] = (u32)gza.size();
    }
    // ---- families ---------------------------------------------------------------------------------------------
    std::vector<u32> k2s;   // all (N - 2)-electron strings, increasing
    if (N == 2) k2s.push_back(0u);
    else {
        u64 v = (u64(1) << (N - 2)) - 1, lim = u64(1) << n;
        while (v < lim) {
            k2s.push_back((u32)v);
            const u64 c = v & (~v + 1), r = v + c;
            v = (((r ^ v) >> 2) / c) | r;
        }
    }
    const int F = (int)k2s.size(), P = (n - N + 2) * (n - N + 1) / 2, NP2 = N * (N - 1) / 2;
    auto row_of = [&](u32 w) { return (i64)(std::lower_bound(row_strings.begin(), row_strings.end(), (u64)w) - row_strings.begin()); };
    std::vector<u32> mrow((size_t)F * P), mpair((size_t)F * P), tf((size_t)rows * NP2, 0u);
    for (int f = 0; f < F; ++f) {
        int m = 0;
        for (int q = 1; q < n; ++q) {
            if ((k2s[f] >> q) & 1u) continue;
            for (int p = 0; p < q; ++p) {
                if ((k2s[f] >> p) & 1u) continue;
                const u32 pair = (1u << p) | (1u << q), t = k2s[f] | pair;
                const i64 r = row_of(t);
                mrow[(size_t)f * P + m] = (u32)r;
                mpair[(size_t)f * P + m] = pair;
                // which of the row's own electron pairs this is (pairs of set bits, (i < j) in bit order, j major)
                int j = 0, found = -1;
                for (u32 wj = t; wj && found < 0; wj &= wj - 1) {
                    const int bj = __builtin_ctz(wj);
                    for (u32 wi = t & ((1u << bj) - 1u); wi; wi &= wi - 1, ++j)
                        if (((1u << __builtin_ctz(wi)) | (1u << bj)) == pair) {
                            found = j;
                            break;
                        }
                }
                tf[(size_t)r * NP2 + found] = (u32)((size_t)f * P + m);
                ++m;
            }
        }
    }
    bs_k2* K = new (std::nothrow) bs_k2;
    BS_REQUIRE(K, BS_ERR_ALLOC, "k2 plan allocation failed");
    K->n = n;
    K->N = N;
    K->P = P;
    K->F = F;
    K->NP2 = NP2;
    K->rows = rows;
    K->n_groups = n_q;
    // Tensor-instruction form (default; BS_K2_MMA=0: DFMA form): tiles of 16 targets (8 when the family has <= 8 members).
    // DFMA form: 12 targets per tile -- 2 x 12 DFMA per 16-byte load still hides the load behind arithmetic and two blocks
    // (16 warps) fit an SM; 28-target tiles (1 block, 8 warps) were 3 - 6 % slower on configs 2, 4 and 5.
    K->mma = getenv("BS_K2_MMA") ? atoi(getenv("BS_K2_MMA")) != 0 : true;
    if (K->mma) {
        // target tile of 8 NT members: the fewest padded targets (executed DMMAs), ties to the larger tile (fewer
        // amplitude bytes per DMMA).  Measured on one B200: P = 28 (q24) NT = 4, P = 45 (q32) NT = 3, P = 325 (q56) NT = 3
        // or 4 within 0.3 %: 1 - 2 % of an application over NT = 2 everywhere.
        K->rt = 8;
        if (P > 8) {
            int best = 0;
            for (int nt = 2; nt <= 4; ++nt) {
                const int padded = (P + 8 * nt - 1) / (8 * nt) * (8 * nt);
                if (!best || padded <= (P + 8 * best - 1) / (8 * best) * (8 * best)) best = nt;
            }
            K->rt = 8 * best;
        }
        if (const char* e = getenv("BS_K2_NT")) K->rt = 8 * std::min(4, std::max(1, atoi(e)));   // test hook: target tiles of 8
    }
    else {
        K->rt = std::min(12, (P + 3) / 4 * 4);
        if (const char* e = getenv("BS_K2_RT")) K->rt = std::min(28, std::max(4, atoi(e) / 4 * 4));   // test hook: tile height
    }
    K->n_tiles = (P + K->rt - 1) / K->rt;
    K->smem = (size_t)(P + 4) * (K->mma ? k2_gs(K->rt / 8) : K->rt) * 8 + (size_t)(P + 4) * 4;
    if (K->smem > 200 * 1024 || (i64)F * P >= (i64(1) << 31) || F > 65535) {
        delete K;
        return BS_OK;
    }
    i64 budget = i64(4) << 30;
    if (const char* e = getenv("BS_K2_SLAB_MB")) budget = std::max<i64>(1, atoll(e)) << 20;   // test hook
    K->slab_cols = std::max<i64>(32, std::min<i64>(row_len, budget / ((i64)F * P * 16) / 32 * 32));
    cudaError_t ce = K->d_S2.alloc((size_t)F * P * K->slab_cols);
    if (ce == cudaSuccess) ce = K->d_mrow.upload(mrow, st);
    if (ce == cudaSuccess) ce = K->d_mpair.upload(mpair, st);
    if (ce == cudaSuccess) ce = K->d_fk2.upload(k2s, st);
    if (ce == cudaSuccess) ce = K->d_goff.upload(goff, st);
    if (ce == cudaSuccess) ce = K->d_gza.upload(gza, st);
    if (ce == cudaSuccess) ce = K->d_gw.upload(gw, st);
    if (ce == cudaSuccess) ce = K->d_tf.upload(tf, st);
    if (ce == cudaSuccess) ce = cudaStreamSynchronize(st);
    K2Dev& d = K->dev;
    d.mrow = K->d_mrow.p;
    d.mpair = K->d_mpair.p;
    d.fk2 = K->d_fk2.p;
    d.goff = K->d_goff.p;
    d.gza = K->d_gza.p;
    d.gw = K->d_gw.p;
    d.tf = K->d_tf.p;
    d.P = P;
    d.F = F;
    d.NP2 = NP2;
    d.n_tiles = K->n_tiles;
    d.rt = K->rt;
    d.ctile = nullptr;
    // tensor form: the coupling tiles depend on the operator and the sector only, so they are evaluated here, once, instead
    // of in the prologue of every block of every column-slab launch (15 % of the stall samples of k_aa_mma at configs[3]).
    // 176 MB per spin at configs[3], 390 MB at configs[4]; above 2 GB (or BS_K2_NO_CTILE=1, test hook) the kernel evaluates.
    const size_t tile_doubles = (size_t)(P + 4) * k2_gs(K->rt / 8), n_ctile = (size_t)F * K->n_tiles * tile_doubles;
    const bool no_ctile = getenv("BS_K2_NO_CTILE") && atoi(getenv("BS_K2_NO_CTILE")) != 0;
    if (ce == cudaSuccess && K->mma && !no_ctile && n_ctile * 8 <= (size_t(2) << 30)) {
        ce = K->d_ctile.alloc(n_ctile);
        if (ce == cudaSuccess) {
            dim3 grid((unsigned)K->n_tiles, (unsigned)F);
            switch (K->rt) {
                case 8: k_aa_tiles<1><<<grid, kAaThreads, 0, st>>>(d, K->d_ctile.p); break;
                case 16: k_aa_tiles<2><<<grid, kAaThreads, 0, st>>>(d, K->d_ctile.p); break;
                case 24: k_aa_tiles<3><<<grid, kAaThreads, 0, st>>>(d, K->d_ctile.p); break;
                default: k_aa_tiles<4><<<grid, kAaThreads, 0, st>>>(d, K->d_ctile.p); break;
            }
            BS_COUNT_LAUNCH(1);
            ce = cudaGetLastError();
            if (ce == cudaSuccess) ce = cudaStreamSynchronize(st);
            if (ce == cudaSuccess) d.ctile = K->d_ctile.p;
        }
    }
    if (ce == cudaSuccess) ce = kaa_dispatch(K, nullptr, 0, 0, 0, 0, 0, st, true);
    if (ce != cudaSuccess) {
        bs_set_error("k2 plan: %s", cudaGetErrorString(ce));
        cudaGetLastError();
        delete K;
        return ce == cudaErrorMemoryAllocation ? BS_ERR_ALLOC : BS_ERR_CUDA;
    }
    std::vector<HostGroup> rest;
    for (auto& g : groups) {
        if (!qualifies(g)) rest.push_back(g);
        else K->h_x.push_back(g.xa);
    }
    groups.swap(rest);
    *out = K;
    return BS_OK;
}

int bs_k2_apply(bs_k2* K, const double2* psi, double2* acc, i64 row_len, i64 row_lo, i64 row_hi, i64 col_lo, i64 col_hi,
                cudaStream_t st) {
    for (i64 c0 = col_lo; c0 < col_hi; c0 += K->slab_cols) {
        const i64 W = std::min(K->slab_cols, col_hi - c0);
        BS_CUDA(kaa_dispatch(K, psi, row_len, c0, W, row_lo, row_hi, st, false));
        const dim3 grid((unsigned)((W + 255) / 256), (unsigned)(row_hi - row_lo));
        k_aa_acc<<<grid, 256, 0, st>>>(K->dev.tf, K->NP2, K->d_S2.p, acc, row_len, W, c0, row_lo);
        BS_COUNT_LAUNCH(2);
        BS_CUDA(cudaGetLastError());
    }
    return BS_OK;
}
