// a4, alpha-beta class resolved over (N_beta - 1)-electron strings: plan tables and the k_ab kernel.
// See bs_kres.cuh for the formulation (Eq. 27-28; Eq. 23 for the JW chains).
#include <algorithm>

#include "bs_epilogue.cuh"
#include "bs_kres.cuh"
#include "bs_plan.cuh"

namespace {

// KresG codes: how one entry G[s][r] of a header's coupling matrix is made from the phase factors V_key(t_a)
constexpr u32 kGSingle = 0u << 29;    // +-w (-1)^{popc(za & t_a)}: the group with x_b = {r, s} has one string (the JW case)
constexpr u32 kGPair = 1u << 29;      // V(key) (bit 28: negated): the same with several strings
constexpr u32 kGDiagKey = 2u << 29;   // sum_j V(dense key j) / N_beta - 2 V(dense key0 + low bits): x_b = 0 group, orbital carries a key
constexpr u32 kGDiag = 3u << 29;      // sum_j V(dense key j) / N_beta
constexpr u32 kGNone = 4u << 29;      // 0
constexpr u32 kGType = 7u << 29;
constexpr u32 kGNeg = 1u << 28;
constexpr u32 kGKeyMask = (1u << 28) - 1;
constexpr int kMaxDenseStr = 160;     // strings of an absorbed x_b = 0 group (3 n + 1 for a two-body Hamiltonian)
constexpr int kMaxSegs = 48;          // staged column segments of a K chunk
constexpr int kProducer = 32;         // threads of the producer warp (the last warp of the block)
constexpr int kKresBarBytes = 64;     // full[3] + empty[3] mbarriers at the head of k_ab's shared memory (48 bytes used)

// shared-memory layout of one coupling matrix: row s holds G[s][0..NP), padded to a multiple of 8 columns (zero) and to a
// row stride of 8 k + 4 doubles so that the four rows a half warp reads as an MMA fragment fall on different banks
__host__ __device__ constexpr int kres_gs(int NP) { return (NP + 7) / 8 * 8 + 4; }

// Coupling matrices of rows [row_lo, ...): one block per target row, one warp per alpha mask (entry) of the row.
// G[s][r] = V_{x_a,{r,s}}(t_a) from the header's tables (see the KresG codes), written in the padded shared-memory
// layout of k_ab (row stride kres_gs) so that k_ab fetches a matrix with one bulk copy; every K chunk of the row reuses it.
template <int NP>
__global__ void __launch_bounds__(256)
k_ab_g(const KresDev Kd, double* __restrict__ Gbuf, i64 row_lo) {
    constexpr int GS = kres_gs(NP), GN = NP * GS, GQ = (NP * NP + 31) / 32, DQ = kMaxDenseStr / 32;
    __shared__ double sVd_all[8][64], sStr_all[8][kMaxDenseStr];
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    double* sVd = sVd_all[w];
    double* sStr = sStr_all[w];
    const i64 row = row_lo + blockIdx.x;
    const u32 ta = __ldg(Kd.a_str + row);
    const i64 e0 = __ldg(Kd.row_off + row), e_base = __ldg(Kd.row_off + row_lo);
    const int n_ent = (int)(__ldg(Kd.row_off + row + 1) - e0);
    for (int i = w; i < n_ent; i += 8) {
        const u32 kh = __ldg(reinterpret_cast<const u32*>(Kd.row_ent + e0 + i));
        double* __restrict__ G = Gbuf + (e0 - e_base + i) * GN;
        const KresG* __restrict__ gt = Kd.gtab + (size_t)kh * (NP * NP);
        const KresG* __restrict__ ds = Kd.dstr + (size_t)kh * kMaxDenseStr;
        const unsigned short* __restrict__ kr = Kd.dkr + (size_t)kh * 64;
        const u32 kr0 = __ldg(kr + lane), kr1 = __ldg(kr + lane + 32);
        // the absorbed x_b = 0 group: signed string weights, then one lane per key sums its strings in order;
        // fixed-order butterfly for the total
#pragma unroll
        for (int q = 0; q < DQ; ++q) {
            const KresG d = ds[lane + 32 * q];
            sStr[lane + 32 * q] = flip(d.w, (u32)__popc(d.za & ta) & 1u);
        }
        __syncwarp();
        // key 0 (beta Z mask 0) is the long one for a two-body Hamiltonian (n + 1 strings): the whole warp sums it;
        // the other keys (one or two strings each) take one lane each
        const u32 k0 = __shfl_sync(0xffffffffu, kr0, 0);
        double v0 = 0.0;
        for (u32 t = (k0 & 0xFFu) + lane; t < (k0 >> 8); t += 32) v0 += sStr[t];
        for (int o = 16; o > 0; o >>= 1) v0 += __shfl_xor_sync(0xffffffffu, v0, o);
        double dsum = 0.0;
#pragma unroll
        for (int jj = 0; jj < 2; ++jj) {
            const u32 krj = jj ? kr1 : kr0;
            double v = 0.0;
            if (jj == 0 && lane == 0) v = v0;
            else
                for (u32 t = krj & 0xFFu; t < (krj >> 8); ++t) v += sStr[t];
            sVd[lane + 32 * jj] = v;
            dsum += v;
        }
        for (int o = 16; o > 0; o >>= 1) dsum += __shfl_xor_sync(0xffffffffu, dsum, o);
        __syncwarp();
        auto V = [&](u32 key) {   // groups with several strings per key (not the JW case): from the plan tables
            double f = 0.0;
            const u32 s1 = __ldg(Kd.key_s0 + key + 1);
            for (u32 s = __ldg(Kd.key_s0 + key); s < s1; ++s)
                f += flip(__ldg(&Kd.s_w[s].x), (u32)__popc(__ldg(Kd.s_za + s) & ta) & 1u);
            return f;
        };
#pragma unroll 4
        for (int q = 0; q < GQ; ++q) {
            const int p = lane + 32 * q;
            if (p >= NP * NP) break;
            const KresG g = gt[p];
            const u32 type = g.code & kGType;
            double v = 0.0;
            if (type == kGSingle) v = flip(g.w, (u32)__popc(g.za & ta) & 1u);
            else if (type == kGPair) {
                v = V(g.code & kGKeyMask);
                if (g.code & kGNeg) v = -v;
            } else if (type == kGDiag) v = dsum * Kd.inv_nb;
            else if (type == kGDiagKey) v = dsum * Kd.inv_nb - 2.0 * sVd[g.code & kGKeyMask];
            G[(p / NP) * GS + p % NP] = v;
        }
        for (int q = lane; q < GN; q += 32)
            if (q % GS >= NP) G[q] = 0.0;   // padding columns
        __syncwarp();   // sStr / sVd are rewritten by the warp's next entry
    }
}

// MMA: the contraction runs on the FP64 tensor instruction (mma.sync m8n8k4: same 64 FMA/clk/SM peak as DFMA, but one
// G fragment load feeds 8 K rows and one instruction carries 256 FMA: a quarter of the shared-memory wavefronts and of
// the issue slots of the DFMA form)
// row tiles (8 K each) per warp of the MMA form: 4 up to 16 orbitals; 2 above, where 4 would need > 200 registers and leave
// 7 compute warps per SM (2 tiles: 14 warps at <= 128 registers)
__host__ __device__ constexpr int kres_rtw(int NP) { return NP <= 16 ? 4 : 2; }
// threads per block: DFMA form one thread per K; MMA form one warp per 8 * rtw K; + the producer warp
__host__ __device__ constexpr int kres_threads(int NP, int KC, bool mma) {
    return (mma ? KC / (8 * kres_rtw(NP)) * 32 : KC) + 32;
}

template <int NP, int KCMAX, bool MMA>
__global__ void __launch_bounds__(kres_threads(NP, KCMAX, MMA), 1)
k_ab(const KresDev Kd, const double2* __restrict__ psi, const double* __restrict__ Gbuf, double2* __restrict__ S,
     i64 row_lo) {
    extern __shared__ __align__(128) unsigned char smem_raw[];
    __shared__ uint2 sSeg[kMaxSegs];
    // NS = 2 or 3 pipeline stages: full[NS] (producer + TMA -> compute warps), empty[NS] (compute warps -> producer)
    u64* bar = reinterpret_cast<u64*>(smem_raw);
    constexpr int GS = kres_gs(NP), GN = NP * GS, NT = (NP + 7) / 8;
    const int NS = Kd.n_stages;
    double* sG = reinterpret_cast<double*>(smem_raw + kKresBarBytes);                                        // [NS][NP][GS]
    double2* sbuf = reinterpret_cast<double2*>(smem_raw + kKresBarBytes + (size_t)NS * GN * 8);              // [NS][buf_elems]
    unsigned short* sgo = reinterpret_cast<unsigned short*>(smem_raw + kKresBarBytes + (size_t)NS * GN * 8 +
                                                            (size_t)NS * Kd.buf_elems * 16);               // [NP][KC]
    constexpr int RTW = kres_rtw(NP);
    const int tid = threadIdx.x, KC = Kd.KC, n_cmp = (int)blockDim.x - kProducer;   // K per chunk, compute threads
    const bool producer = tid >= n_cmp;
    const int lane = tid & 31;
    const i64 row = row_lo + blockIdx.x;
    const int chunk = blockIdx.y;
    const u32 ta = __ldg(Kd.a_str + row);
    const int nseg = __ldg(Kd.seg_cnt + chunk);
    u32 sig = 0, in_k = 0;   // in_k: orbitals that every K of this warp holds (no source, no target there: skipped)
    if (!producer) {
        if (!MMA) sig = __ldg(Kd.sigma + (size_t)chunk * KC + tid);
        for (int idx = tid; idx < NP * KC; idx += n_cmp) sgo[idx] = __ldg(Kd.goff + (size_t)chunk * NP * KC + idx);
    } else {
        for (int g = lane; g < nseg; g += 32) sSeg[g] = __ldg(Kd.segs + (size_t)chunk * Kd.max_segs + g);
    }
    if (tid == n_cmp) {
        for (int b = 0; b < NS; ++b) {
            mbar_init(bar + b, 1);                     // full: the producer's arrive.expect_tx; the bulk copies complete the byte count
            mbar_init(bar + NS + b, (u32)n_cmp / 32);  // empty: one arrival per compute warp
        }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
        for (int b = 0; b < NS; ++b) sbuf[(size_t)b * Kd.buf_elems] = make_double2(0.0, 0.0);   // position 0 of every buffer: the zero amplitude (s in K)
    }
    constexpr int ACCN = MMA ? 4 * RTW * NT : NP;   // MMA: RTW row tiles x NT column tiles x (re, im) fragments of two doubles
    double2 acc[ACCN < NP ? NP : ACCN];
#pragma unroll
    for (int r = 0; r < (ACCN < NP ? NP : ACCN); ++r) acc[r] = make_double2(0.0, 0.0);
    const i64 e0 = __ldg(Kd.row_off + row);
    const int n_ent = (int)(__ldg(Kd.row_off + row + 1) - e0);
    const i64 Db = Kd.Db;
    const i64 e_base = __ldg(Kd.row_off + row_lo);
    u32 seg_bytes = 0;   // producer: bytes of one entry's bulk copies

    // ---- producer warp -----------------------------------------------------------------------------------------
    // TMA bulk copies of the chunk's column segments of entry i's source row into buffer b = i mod NS (lane 0)
    auto stage_row = [&](int i, int b) {
        const u32 src_row = __ldg(reinterpret_cast<const u32*>(Kd.row_ent + e0 + i) + 1);
        const double2* __restrict__ src = psi + (i64)src_row * Db;
        unsigned char* dst = reinterpret_cast<unsigned char*>(sbuf + (size_t)b * Kd.buf_elems + 1);
        mbar_expect_tx(bar + b, seg_bytes + (u32)(GN * 8));
        // the entry's coupling matrix, made by k_ab_g for all K chunks of the row
        tma_bulk_g2s(sG + b * GN, Gbuf + (e0 - e_base + i) * GN, (u32)(GN * 8), bar + b);
        for (int g = 0; g < nseg; ++g) {
            const uint2 sg = sSeg[g];
            const unsigned char* sp = reinterpret_cast<const unsigned char*>(src + sg.x);
            const u32 bytes = sg.y * 16u;
            for (u32 o = 0; o < bytes; o += 32768u) tma_bulk_g2s(dst + o, sp + o, min(32768u, bytes - o), bar + b);
            dst += bytes;
        }
    };
    __syncthreads();
    if (producer) {
        // No block barrier in the entry loop: the producer refills buffer b as soon as every compute warp has released
        // it (empty[b]); a compute warp starts entry i as soon as full[i mod NS] completes, whatever the other warps do.
        // Entry i uses buffer b = i mod NS for the (i / NS)-th time: its full barrier completes phase i / NS, and the
        // producer refills it once the empty barrier has completed phase i / NS - 1.  NS = 3 (producer two entries ahead)
        // was built because 12.5 % of the compute warps' stall samples sit on the full-barrier wait; it changes nothing
        // (q32 432.7 vs 433.0 ms): that wait is the slack of warps with fewer active orbitals, which a deeper queue cannot
        // remove.  Two buffers are the default, three a tested hook (BS_KRES_STAGES=3).
        if (lane == 0) {
            for (int g = 0; g < nseg; ++g) seg_bytes += sSeg[g].y * 16u;
            int b = 0;
            u32 use = 0;   // i / NS
            for (int i = 0; i < n_ent; ++i) {
                if (use > 0) mbar_wait(bar + NS + b, (use - 1) & 1u);
                stage_row(i, b);
                if (++b == NS) { b = 0; ++use; }
            }
        }
        return;
    }
    // orbitals that every K of this warp holds have no source and no target there: skipped warp-uniformly
    if (MMA) {
        const int g0 = lane >> 2, tq0 = lane & 3, kw0 = (tid >> 5) * (8 * RTW) + g0;
        in_k = 0xFFFFFFFFu;
        for (int s = tq0; s < NP; s += 4) {
            bool all = true;
            for (int i2 = 0; i2 < RTW; ++i2) all &= sgo[s * KC + kw0 + 8 * i2] == 0;
            if (!all) in_k &= ~(1u << s);
        }
    } else {
        for (int s = 0; s < NP; ++s) in_k |= (sgo[s * KC + tid] == 0 ? 1u : 0u) << s;
    }
    in_k = __reduce_and_sync(0xffffffffu, in_k);
    const u32 act_all = ~in_k & (Kd.n >= 32 ? 0xFFFFFFFFu : ((1u << Kd.n) - 1u));
    if (MMA) {
        // Warp tile: 32 K rows (this warp's K) x NP columns; fragment coordinates g = lane / 4, tq = lane % 4.
        // A[K][s] = sigma_s(K) psi[u_a, K + {s}] (re and im as separate row tiles), B[s][r] = G[s][r], four active
        // orbitals per step.  Row tile i of warp w holds K = 8 RTW w + 8 i + g.
        const int g = lane >> 2, tq = lane & 3, kw = (tid >> 5) * (8 * RTW) + g;
        u32 sigk[RTW];
#pragma unroll
        for (int i2 = 0; i2 < RTW; ++i2) sigk[i2] = __ldg(Kd.sigma + (size_t)chunk * KC + kw + 8 * i2);
        const int n_act = __popc(act_all);
        // this lane's orbital of every step (the (4 step + tq)-th active one), 6 bits each, 63 = none: found once per
        // block instead of at every step of every entry (__fns is a loop)
        u64 my_orb = 0;
        for (int st_ = 0; st_ < 8; ++st_) {
            const u32 s_ = 4 * st_ + tq < (u32)n_act ? __fns(act_all, 0, 4 * st_ + tq + 1) : 63u;
            my_orb |= (u64)(s_ & 63u) << (6 * st_);
        }
        int cb = 0;      // buffer of entry i: i mod NS
        u32 cuse = 0;    // i / NS
        for (int i = 0; i < n_ent; ++i) {
            mbar_wait(bar + cb, cuse & 1u);
            const double* __restrict__ G = sG + cb * GN;
            const double2* __restrict__ buf = sbuf + (size_t)cb * Kd.buf_elems;
            for (int ks = 0; ks < n_act; ks += 4) {
                const u32 s = (u32)(my_orb >> (6 * (ks >> 2))) & 63u;   // this lane's orbital of the step (63: none left)
                const bool valid = s < 32u;
                const u32 sc = valid ? s : 0u;
                double are[RTW], aim[RTW], bf[NT];
#pragma unroll
                for (int i2 = 0; i2 < RTW; ++i2) {
                    const double2 b = buf[valid ? sgo[sc * KC + kw + 8 * i2] : 0];
                    const u32 sg = (sigk[i2] >> sc) & 1u;
                    are[i2] = flip(b.x, sg);
                    aim[i2] = flip(b.y, sg);
                }
#pragma unroll
                for (int j = 0; j < NT; ++j) bf[j] = valid ? G[sc * GS + 8 * j + g] : 0.0;
#pragma unroll
                for (int i2 = 0; i2 < RTW; ++i2)
#pragma unroll
                    for (int j = 0; j < NT; ++j) {
                        double2& cr = acc[(i2 * NT + j) * 2];
                        double2& ci = acc[(i2 * NT + j) * 2 + 1];
                        asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};"
                                     : "+d"(cr.x), "+d"(cr.y) : "d"(are[i2]), "d"(bf[j]));
                        asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};"
                                     : "+d"(ci.x), "+d"(ci.y) : "d"(aim[i2]), "d"(bf[j]));
                    }
            }
            __syncwarp();
            if (lane == 0) mbar_arrive(bar + NS + cb);   // this warp is done with the buffer
            if (++cb == NS) { cb = 0; ++cuse; }
        }
        // C fragment: row g of tile i2 (K = kw + 8 i2), columns 8 j + 2 tq + {0, 1}
#pragma unroll
        for (int i2 = 0; i2 < RTW; ++i2)
#pragma unroll
            for (int j = 0; j < NT; ++j)
#pragma unroll
                for (int e = 0; e < 2; ++e) {
                    const int r = 8 * j + 2 * tq + e;
                    if (r < Kd.n) {
                        const u32 sg = (sigk[i2] >> r) & 1u;
                        const double2 cr = acc[(i2 * NT + j) * 2], ci = acc[(i2 * NT + j) * 2 + 1];
                        S[((i64)blockIdx.x * Kd.n + r) * Kd.DKp + (i64)chunk * KC + kw + 8 * i2] =
                            make_double2(flip(e ? cr.y : cr.x, sg), flip(e ? ci.y : ci.x, sg));
                    }
                }
        return;
    }
    // DFMA form: orbitals walked in ascending order; the gather of the next orbital is issued before the DFMA block of
    // the current one
    const unsigned short* __restrict__ my_go = sgo + tid;
    int cb = 0;      // buffer of entry i: i mod NS
    u32 cuse = 0;    // i / NS
    for (int i = 0; i < n_ent; ++i) {
        mbar_wait(bar + cb, cuse & 1u);
        const double* __restrict__ G = sG + cb * GN;
        const double2* __restrict__ buf = sbuf + (size_t)cb * Kd.buf_elems;
        u32 act = act_all;
        int s = __ffs((int)act) - 1;
        act &= act - 1;
        double2 b = (s >= 0) ? buf[my_go[s * KC]] : make_double2(0.0, 0.0);
        while (s >= 0) {
            const int sn = __ffs((int)act) - 1;   // -1 when none is left
            act &= act - 1;
            double2 bn = make_double2(0.0, 0.0);
            if (sn >= 0) bn = buf[my_go[sn * KC]];
            const u32 sg = (sig >> s) & 1u;
            b.x = flip(b.x, sg);
            b.y = flip(b.y, sg);
            const double2* __restrict__ g2 = reinterpret_cast<const double2*>(G + s * GS);
#pragma unroll
            for (int r2 = 0; r2 < NP / 2; ++r2) {
                const double2 g = g2[r2];   // warp-uniform address: two wavefronts for two columns of G
                acc[2 * r2].x += g.x * b.x;
                acc[2 * r2].y += g.x * b.y;
                acc[2 * r2 + 1].x += g.y * b.x;
                acc[2 * r2 + 1].y += g.y * b.y;
            }
            s = sn;
            b = bn;
        }
        __syncwarp();
        if (lane == 0) mbar_arrive(bar + NS + cb);   // this warp is done with the buffer
        if (++cb == NS) { cb = 0; ++cuse; }
    }
    double2* __restrict__ out = S + ((i64)blockIdx.x * Kd.n) * Kd.DKp + (i64)chunk * KC + tid;
#pragma unroll
    for (int r = 0; r < NP; ++r) {
        if (r < Kd.n) {
            const u32 sg = (sig >> r) & 1u;
            out[(i64)r * Kd.DKp] = make_double2(flip(acc[r].x, sg), flip(acc[r].y, sg));
        }
    }
}

// K per chunk.  DFMA form (one thread per K): compute threads + the producer warp fill whole groups of 4 warps, 512 threads
// at <= 128 registers for up to 16 orbitals, 256 threads at <= 255 registers above.  Tensor form (8 RTW K per warp): 16
// COMPUTE warps, four per SM sub-partition, plus the producer warp (544 threads at <= 120 registers).  With 480 / 224 K the
// tensor form ran 15 / 14 compute warps: the busiest sub-partition carried 12 - 15 % more DMMA work than the mean, which is
// the idle fifth of the tensor pipe that ncu showed (profiles/r02b_q32_k_ab_k_aa_full.md).  The register file is per
// sub-partition (16 K registers): the sub-partition that also hosts the producer warp holds five warps, so the 544-thread
// builds are capped at 96 registers.  Above 16 orbitals (two row tiles per warp) that costs at most 16 bytes of spills
// and the balance wins 8 % (q56 1,107 -> 1,015 ms); up to 16 orbitals (four row tiles, 117 registers) it costs 52 bytes of
// spills: worth it only for sectors with many chunks (q32 438.5 -> 431.8 ms), not for small ones (q24 1.233 -> 1.277 ms),
// which keep the 480 build (`big` = false).
constexpr int kres_kcmax(int NP, bool mma, bool big) {
    return mma ? (NP <= 16 ? (big ? 512 : 480) : 256) : (NP <= 16 ? 480 : 224);
}

template <int NP>
cudaError_t kab_launch(const bs_kres* K, const double2* psi, i64 lo, i64 hi, cudaStream_t st, bool set_attr) {
    auto k = !K->mma ? k_ab<NP, kres_kcmax(NP, false, false), false>
                     : (K->kc_max == kres_kcmax(NP, true, true) ? k_ab<NP, kres_kcmax(NP, true, true), true>
                                                                : k_ab<NP, kres_kcmax(NP, true, false), true>);
    // the ceiling is per kernel and shared by all plans: the opt-in maximum minus the kernel's static shared memory
    if (set_attr) return cudaFuncSetAttribute(k, cudaFuncAttributeMaxDynamicSharedMemorySize, 227 * 1024 - 1024);
    dim3 grid((unsigned)(hi - lo), (unsigned)K->n_chunks);
    k_ab_g<NP><<<(unsigned)(hi - lo), 256, 0, st>>>(K->dev, K->d_G.p, lo);
    k<<<grid, kres_threads(NP, K->KC, K->mma), K->smem, st>>>(K->dev, psi, K->d_G.p, K->d_S.p, lo);
    return cudaGetLastError();
}

cudaError_t kab_dispatch(const bs_kres* K, const double2* psi, i64 lo, i64 hi, cudaStream_t st, bool set_attr) {
    switch (K->NP) {
        case 8: return kab_launch<8>(K, psi, lo, hi, st, set_attr);
        case 12: return kab_launch<12>(K, psi, lo, hi, st, set_attr);
        case 16: return kab_launch<16>(K, psi, lo, hi, st, set_attr);
        case 20: return kab_launch<20>(K, psi, lo, hi, st, set_attr);
        case 24: return kab_launch<24>(K, psi, lo, hi, st, set_attr);
        case 28: return kab_launch<28>(K, psi, lo, hi, st, set_attr);
        default: return kab_launch<32>(K, psi, lo, hi, st, set_attr);
    }
}

// all n-bit words of popcount k in increasing numeric order (k = 0: the empty string)
std::vector<u32> subsets(int n, int k) {
    std::vector<u32> out;
    if (k == 0) {
        out.push_back(0u);
        return out;
    }
    u64 v = (u64(1) << k) - 1, lim = u64(1) << n;
    while (v < lim) {
        out.push_back((u32)v);
        const u64 c = v & (~v + 1), r = v + c;   // next word with the same popcount
        v = (((r ^ v) >> 2) / c) | r;
    }
    return out;
}

}  // namespace

bs_kres::~bs_kres() { delete rp; }

int bs_kres_build(std::vector<HostGroup>& groups, bs_sector* S, cudaStream_t st, bs_kres** out, bool allow_xa0) {
    *out = nullptr;
    if (getenv("BS_NO_KRES")) return BS_OK;   // test hook (include/bs.h "Environment")
    const int n = S->n_orb, Nb = S->n_beta;
    if (n < 5 || n > 32 || Nb < 1 || Nb >= n || S->Db < 64 || S->Db > 32767) return BS_OK;
    // ---- which groups: under an alpha mask, the single-key beta single hops whose Z mask is the JW chain, and the
    // x_b = 0 group when its beta Z masks are single bits (number operators) ------------------------------------
    auto real_w = [](const HostGroup& g) {
        for (auto& s : g.s)
            if (s.im != 0.0) return false;
        return true;
    };
    auto jw_hop = [&](const HostGroup& g) {
        if (__builtin_popcount(g.xb) != 2 || g.s.front().zb != g.s.back().zb || !real_w(g)) return false;
        const int lo = __builtin_ctz(g.xb), hi = 31 - __builtin_clz(g.xb);
        const u32 between = ((1u << hi) - 1u) & ~((2u << lo) - 1u);
        return (g.s.front().zb & ~g.xb) == between;
    };
    auto absorbable = [&](const HostGroup& g) {
        if (g.xb != 0 || g.s.front().zb != 0 || !real_w(g)) return false;
        for (auto& s : g.s)
            if (s.zb != 0 && __builtin_popcount(s.zb) != 1) return false;
        return true;
    };
    const int min_hops = getenv("BS_KRES_MIN") ? atoi(getenv("BS_KRES_MIN")) : 8;
    std::map<u32, int> n_hops;
    for (auto& g : groups)
        if ((g.xa != 0 || allow_xa0) && jw_hop(g)) ++n_hops[g.xa];
    std::vector<HostGroup> mine, rest;
    for (auto& g : groups) {
        auto f = n_hops.find(g.xa);
        const bool take = f != n_hops.end() && f->second >= min_hops &&
                          ((g.xa != 0 && (jw_hop(g) || absorbable(g))) || (g.xa == 0 && allow_xa0 && jw_hop(g)));
        (take ? mine : rest).push_back(g);
    }
    if (mine.empty()) return BS_OK;
    bs_kres* K = new (std::nothrow) bs_kres;
    BS_REQUIRE(K, BS_ERR_ALLOC, "kres plan allocation failed");
    K->rp = new (std::nothrow) bs_rowplan;
    int rc = K->rp ? bs_rowplan_build(K->rp, mine, S->ta, S->tb, st, false) : BS_ERR_ALLOC;
    if (rc != BS_OK) {
        delete K;
        return rc;
    }
    const bs_rowplan* R = K->rp;
    const int NP = (n + 3) & ~3;
    K->n = n;
    K->NP = NP;
    K->Nb = Nb;
    // ---- coupling-matrix tables -------------------------------------------------------------------------------
    const size_t n_hdr = R->h_hdrs.size();
    KresG none{};
    none.code = kGNone;
    std::vector<KresG> gtab(n_hdr * NP * NP, none);
    std::vector<KresG> dstr(n_hdr * kMaxDenseStr, KresG{});   // strings of the absorbed group, zero weight beyond
    std::vector<unsigned short> dkr(n_hdr * 64, 0);           // string range lo | hi << 8 of its keys (empty beyond)
    for (size_t kh = 0; kh < n_hdr; ++kh) {
        const XaHdr& h = R->h_hdrs[kh];
        KresG* gm = gtab.data() + kh * NP * NP;
        for (u32 i = h.item0; i < h.item1; ++i) {
            const RowItem& it = R->h_items[i];
            if (it.tkey == kTkeyIdent) {   // the absorbed x_b = 0 group: F = sum_j V_j (-1)^{n_q(j)} -> diagonal of G
                const u32 d0 = R->h_key_s0[it.key0], d1 = R->h_key_s0[it.key0 + it.nkeys];
                if (it.nkeys > 40 || d1 - d0 > (u32)kMaxDenseStr) {
                    delete K;
                    return BS_OK;
                }
                for (u32 t = d0; t < d1; ++t) {
                    dstr[kh * kMaxDenseStr + (t - d0)].w = R->h_s_w[t].x;
                    dstr[kh * kMaxDenseStr + (t - d0)].za = R->h_s_za[t];
                }
                for (u32 j = 0; j < it.nkeys; ++j)
                    dkr[kh * 64 + j] = (unsigned short)((R->h_key_s0[it.key0 + j] - d0) | ((R->h_key_s0[it.key0 + j + 1] - d0) << 8));
                for (int q = 0; q < n; ++q) gm[q * NP + q].code = kGDiag;
                for (u32 j = 1; j < it.nkeys; ++j) {
                    const int q = __builtin_ctz(R->h_key_dz[it.key0 + j]);
                    gm[q * NP + q].code = kGDiagKey | j;
                }
            } else {
                const uint2 tk = R->h_tkeys[it.tkey];   // {x_b, z_b0}
                const int lo = __builtin_ctz(tk.x), hi = 31 - __builtin_clz(tk.x);
                const u32 s0 = R->h_key_s0[it.key0], s1 = R->h_key_s0[it.key0 + 1];
                // target K + {lo} <- source K + {hi}: the target holds lo, so z_b0's own bit on lo counts (and vice versa)
                const int tgt[2] = {lo, hi}, src[2] = {hi, lo};
                for (int d = 0; d < 2; ++d) {
                    const bool neg = (tk.y >> tgt[d]) & 1u;
                    KresG& e = gm[src[d] * NP + tgt[d]];
                    if (s1 - s0 == 1) {
                        e.w = neg ? -R->h_s_w[s0].x : R->h_s_w[s0].x;
                        e.za = R->h_s_za[s0];
                        e.code = kGSingle;
                    } else e.code = kGPair | it.key0 | (neg ? kGNeg : 0u);
                }
            }
        }
    }
    // ---- K strings, chunks, staged column segments ---------------------------------------------------------------
    const std::vector<u32> Ks = subsets(n, Nb - 1);
    const i64 DK = (i64)Ks.size();
    K->DK = DK;
    auto col_of = [&](u32 w) {
        return (i64)(std::lower_bound(S->h_sb.begin(), S->h_sb.end(), (u64)w) - S->h_sb.begin());
    };
    K->mma = getenv("BS_KRES_MMA") ? atoi(getenv("BS_KRES_MMA")) != 0 : true;   // test hook: 0 = DFMA form
    // the build of k_ab (register budget): the 16-compute-warp build for sectors with at least 8 chunks of it
    bool big = (DK + kres_kcmax(NP, K->mma, true) - 1) / kres_kcmax(NP, K->mma, true) >= 8;
    if (const char* e = getenv("BS_KRES_BIG")) big = atoi(e) != 0;   // test hook: force either build
    const int kc_max = kres_kcmax(NP, K->mma, big);
    K->kc_max = kc_max;
    // chunks of equal size: K strings split evenly over the fewest chunks (q24: 792 K in 2 chunks of 416, not 480 + 312)
    const i64 n_min = (DK + kc_max - 1) / kc_max;
    int KC = (int)std::min<i64>(kc_max, ((DK + n_min - 1) / n_min + 31) / 32 * 32);
    if (const char* e = getenv("BS_KRES_KC")) KC = std::max(32, std::min(kc_max, atoi(e) / 32 * 32));
    const size_t smem_max = 227 * 1024 - 1024;
    std::vector<uint2> segs;
    std::vector<int> segcnt;
    std::vector<unsigned short> goff;
    int n_chunks = 0, max_segs = 0, buf_elems = 0;
    double staged = 0;
    for (;; KC /= 2) {
        if (KC < 32) {
            delete K;
            return BS_OK;   // does not fit: the groups stay on the list path
        }
        n_chunks = (int)((DK + KC - 1) / KC);
        std::vector<std::vector<uint2>> cs(n_chunks);
        goff.assign((size_t)n_chunks * NP * KC, 0);
        max_segs = 0;
        buf_elems = 0;
        staged = 0;
        for (int c = 0; c < n_chunks; ++c) {
            std::vector<u32> need;
            for (i64 k = (i64)c * KC; k < std::min<i64>(DK, (i64)(c + 1) * KC); ++k)
                for (int s = 0; s < n; ++s)
                    if (!((Ks[k] >> s) & 1u)) need.push_back((u32)col_of(Ks[k] | (1u << s)));
            std::sort(need.begin(), need.end());
            need.erase(std::unique(need.begin(), need.end()), need.end());
            std::vector<uint2>& sg = cs[c];
            for (u32 gap = 32;; gap *= 2) {   // merge neighbouring columns into segments (few, long bulk copies)
                sg.clear();
                for (u32 v : need) {
                    if (!sg.empty() && v <= sg.back().x + sg.back().y - 1 + gap) sg.back().y = v - sg.back().x + 1;
                    else sg.push_back(make_uint2(v, 1u));
                }
                if (sg.size() <= (size_t)kMaxSegs) break;
            }
            std::vector<u32> base(sg.size());
            u32 tot = 0;
            for (size_t g = 0; g < sg.size(); ++g) {
                base[g] = 1 + tot;   // position 0 is the zero amplitude
                tot += sg[g].y;
            }
            buf_elems = std::max(buf_elems, (int)tot + 1);
            staged += tot;
            max_segs = std::max(max_segs, (int)sg.size());
            for (i64 k = (i64)c * KC; k < std::min<i64>(DK, (i64)(c + 1) * KC); ++k)
                for (int s = 0; s < n; ++s) {
                    if ((Ks[k] >> s) & 1u) continue;
                    const u32 col = (u32)col_of(Ks[k] | (1u << s));
                    size_t g = std::upper_bound(sg.begin(), sg.end(), col, [](u32 v, const uint2& a) { return v < a.x; }) -
                               sg.begin() - 1;
                    goff[((size_t)c * NP + s) * KC + (k - (i64)c * KC)] = (unsigned short)(base[g] + (col - sg[g].x));
                }
        }
        auto smem_for = [&](int ns) {
            return (size_t)kKresBarBytes + (size_t)ns * NP * kres_gs(NP) * 8 + (size_t)ns * buf_elems * 16 + (size_t)NP * KC * 2;
        };
        const size_t smem = smem_for(2);   // the chunk size is chosen for two buffers, as before
        if (smem <= smem_max && buf_elems <= 65535) {
            // two buffers; BS_KRES_STAGES=3 (test hook) takes a third when it fits at this chunk size: no measured gain
            K->n_stages = 2;
            if (const char* e = getenv("BS_KRES_STAGES")) K->n_stages = (atoi(e) >= 3 && smem_for(3) <= smem_max) ? 3 : 2;
            K->smem = smem_for(K->n_stages);
            segs.assign((size_t)n_chunks * max_segs, make_uint2(0u, 0u));
            segcnt.resize(n_chunks);
            for (int c = 0; c < n_chunks; ++c) {
                segcnt[c] = (int)cs[c].size();
                std::copy(cs[c].begin(), cs[c].end(), segs.begin() + (size_t)c * max_segs);
            }
            break;
        }
    }
    K->KC = KC;
    K->n_chunks = n_chunks;
    K->max_segs = max_segs;
    K->buf_elems = buf_elems;
    K->DKp = (i64)n_chunks * KC;
    K->staged_rows = staged / (double)S->Db;
    std::vector<u32> sigma((size_t)K->DKp, 0u);
    for (i64 k = 0; k < DK; ++k) {
        u32 m = 0;
        for (int p = 0; p < n; ++p) m |= ((u32)__builtin_popcount(Ks[k] & ((1u << p) - 1u)) & 1u) << p;
        sigma[k] = m;
    }
    // ---- gather side: where the N_beta contributions of a target column sit in the scratch ---------------------
    std::vector<u32> comb((size_t)S->Db * Nb);
    for (i64 c = 0; c < S->Db; ++c) {
        u32 tb = (u32)S->h_sb[c];
        int j = 0;
        for (u32 w = tb; w; w &= w - 1, ++j) {
            const int r = __builtin_ctz(w);
            const i64 kidx = std::lower_bound(Ks.begin(), Ks.end(), tb ^ (1u << r)) - Ks.begin();
            comb[(size_t)c * Nb + j] = (u32)((i64)r * K->DKp + kidx);
        }
    }
    if ((i64)n * K->DKp >= (i64(1) << 31)) {
        delete K;
        return BS_OK;
    }
    const i64 per_row = (i64)n * K->DKp * 16;
    i64 budget = i64(4) << 30;
    if (const char* e = getenv("BS_KRES_SLAB_MB")) budget = std::max<i64>(1, atoll(e)) << 20;   // test hook
    K->slab_rows = std::max<i64>(1, std::min<i64>(S->Da, budget / per_row));
    // coupling matrices of one slab (k_ab_g): the most entries any slab of slab_rows rows holds
    std::vector<i64> h_off(S->Da + 1);
    cudaError_t ce = cudaMemcpyAsync(h_off.data(), R->d_row_off.p, (S->Da + 1) * 8, cudaMemcpyDeviceToHost, st);
    if (ce == cudaSuccess) ce = cudaStreamSynchronize(st);
    i64 max_ent = 1;
    for (i64 r0 = 0; r0 < S->Da; r0 += K->slab_rows)
        max_ent = std::max(max_ent, h_off[std::min<i64>(S->Da, r0 + K->slab_rows)] - h_off[r0]);
    K->g_bytes = (size_t)max_ent * NP * kres_gs(NP) * 8;
    if (ce == cudaSuccess) ce = K->d_G.alloc((size_t)max_ent * NP * kres_gs(NP));
    if (ce == cudaSuccess) ce = K->d_S.alloc((size_t)(K->slab_rows * n * K->DKp));
    if (ce == cudaSuccess) ce = K->d_gtab.upload(gtab, st);
    if (ce == cudaSuccess) ce = K->d_dstr.upload(dstr, st);
    if (ce == cudaSuccess) ce = K->d_dkr.upload(dkr, st);
    if (ce == cudaSuccess) ce = K->d_goff.upload(goff, st);
    if (ce == cudaSuccess) ce = K->d_sigma.upload(sigma, st);
    if (ce == cudaSuccess) ce = K->d_segs.upload(segs, st);
    if (ce == cudaSuccess) ce = K->d_segcnt.upload(segcnt, st);
    if (ce == cudaSuccess) ce = K->d_comb.upload(comb, st);
    if (ce == cudaSuccess) ce = cudaStreamSynchronize(st);
    KresDev& d = K->dev;
    d.row_off = R->d_row_off.p;
    d.row_ent = R->d_row_ent.p;
    d.a_str = S->ta.str;
    d.gtab = K->d_gtab.p;
    d.dstr = K->d_dstr.p;
    d.dkr = K->d_dkr.p;
    d.key_s0 = R->d_key_s0.p;
    d.s_za = R->d_s_za.p;
    d.s_w = R->d_s_w.p;
    d.goff = K->d_goff.p;
    d.sigma = K->d_sigma.p;
    d.segs = K->d_segs.p;
    d.seg_cnt = K->d_segcnt.p;
    d.max_segs = max_segs;
    d.KC = KC;
    d.n_chunks = n_chunks;
    d.n = n;
    d.Nb = Nb;
    d.buf_elems = buf_elems;
    d.n_stages = K->n_stages;
    d.Db = S->Db;
    d.DKp = K->DKp;
    d.inv_nb = 1.0 / (double)Nb;
    if (ce == cudaSuccess) ce = kab_dispatch(K, nullptr, 0, 0, st, true);
    if (ce != cudaSuccess) {
        bs_set_error("kres plan: %s", cudaGetErrorString(ce));
        cudaGetLastError();
        delete K;
        return ce == cudaErrorMemoryAllocation ? BS_ERR_ALLOC : BS_ERR_CUDA;
    }
    groups.swap(rest);
    *out = K;
    return BS_OK;
}

// rows [lo, hi) (at most slab_rows) -> scratch S[row - lo][r][K]
int bs_kres_apply(bs_kres* K, const double2* psi, i64 lo, i64 hi, cudaStream_t st) {
    BS_CUDA(kab_dispatch(K, psi, lo, hi, st, false));
    BS_COUNT_LAUNCH(2);
    return BS_OK;
}
