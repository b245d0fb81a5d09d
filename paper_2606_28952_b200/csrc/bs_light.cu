// a4/a5/a7, "light" path of the row kernel for operators with few groups whose apply is bound by HBM rather
// than by the gather count -- lattice models such as the Fermi-Hubbard chain of BASELINE.json configs[2]
// (27 groups, 15 non-zeros per row; Eq. 27 with the spin split of PAPER.md:227-231, Eq. 28).
//
// Shape handled (anything else stays on k_rows): the x_a = 0 entry holds the diagonal (x_b = 0, multi-key) and the
// beta-moving groups, all of them served by a UNIFORM column list (one row-independent weight: hopping terms);
// every other alpha mask is a "simple" entry (one group, x_b = 0, one key: an alpha hop = a row axpy).
//
// One 1024-thread block per SM owns ALL columns (D_beta <= 4096) of every grid-th row:
//   * the column list (u16: source column | sign << 15) is copied to shared memory once per launch: the hop loop
//     reads it with one conflict-free LDS.64 per slot and never touches global memory;
//   * rows are double-buffered by TMA bulk copies (row r + 1 lands while row r is processed);
//   * every phase factor V(t_a) was evaluated at plan time into a per-row table, so there is no V phase, no
//     per-entry barrier and no shared-memory traffic for weights; per-thread column state (beta string, validity)
//     is set up once per launch instead of once per row.
#include <algorithm>

#include "bs_epilogue.cuh"
#include "bs_plan.cuh"
#include "bs_rowplan.cuh"

namespace {

constexpr int kLC = 4;         // columns per thread: column = tid + k * T, T = threads per block
constexpr int kLTmax = 1024;   // T = D_beta / 4 rounded up to a warp: no idle warps (3432 columns -> 864 threads)

__device__ __forceinline__ u32 light_slot(u32 col, u32 T) { return (col % T) * kLC + col / T; }

// list build: entry j of a column = j-th valid listed table as (source column * 16) | sign -- the byte offset of the
// source amplitude in the staged row with the sign in the free low bits -- padded with D_beta * 16 (the zero amplitude
// kept behind each staged row).  D_beta <= 4094 keeps it in 16 bits.
__global__ void k_light_list(SpinTab B, const uint2* __restrict__ tkeys, int n_listed, int l_max, int allow_by_table,
                             int T, unsigned short* __restrict__ L, int* __restrict__ cnt) {
    const u32 col = blockIdx.x * blockDim.x + threadIdx.x;
    const u32 kLW = (u32)T * kLC;
    if (col >= kLW) return;
    const u32 slot = light_slot(col, (u32)T);
    // When some column uses every listed table (l_max == n_listed: the Hubbard chain) compaction saves nothing, and
    // slot t = table t keeps the lanes of a warp on the same hop: neighbouring targets then read neighbouring sources
    // (fewer shared-memory bank conflicts than the compacted order, which mixes hops across lanes).
    const bool by_table = allow_by_table && l_max == n_listed;
    int j = 0;
    if (col < B.D) {
        const u32 tb = B.str[col];
        for (int t = 0; t < n_listed; ++t) {
            const uint2 k = tkeys[t];
            const bool valid = 2 * __popc(tb & k.x) == __popc(k.x);
            if (!valid && !(l_max && by_table)) continue;
            if (l_max)
                L[(i64)j * kLW + slot] =
                    valid ? (unsigned short)((spin_rank(B, tb ^ k.x) << 4) | (u32)(__popc(tb & k.y) & 1)) : (unsigned short)(B.D << 4);
            ++j;
        }
    }
    if (!l_max) cnt[col] = j;
    else for (; j < l_max; ++j) L[(i64)j * kLW + slot] = (unsigned short)(B.D << 4);
}

// V table: for row r the keys of the x_a = 0 header, then one value per simple entry (in entry order)
__global__ void k_light_v(RowPlanDev P, u32 key0, u32 key1, const i64* __restrict__ voff, double* __restrict__ vtab) {
    const i64 row = blockIdx.x;
    const u32 ta = P.A.str[row];
    double* v = vtab + voff[row];
    const u32 nk0 = key1 - key0;
    const i64 e0 = P.row_off[row], e1 = P.row_off[row + 1];
    const u32 total = nk0 + (u32)(e1 - e0 - 1);
    for (u32 i = threadIdx.x; i < total; i += blockDim.x) {
        u32 k;
        if (i < nk0) k = key0 + i;
        else {
            const uint4 en = P.row_ent[e0 + 1 + (i - nk0)];
            k = reinterpret_cast<const u32*>(P.xa_hdr + en.x)[2];  // key0 of the simple entry's header
        }
        double f = 0.0;
        for (u32 s = P.key_s0[k]; s < P.key_s0[k + 1]; ++s) f += flip(P.s_w[s].x, (u32)__popc(P.s_za[s] & ta) & 1u);
        v[i] = f;
    }
}

template <int MODE, int MAXT, bool SIGN>  // MODE 0: final epilogue, 2: expectation partials; MAXT: launch bound (register
                                         // budget); SIGN: some list entry carries a sign (else: plain sums, e.g. NN hops)
__global__ void __launch_bounds__(MAXT, 1)
k_light(const LightDev L, const double2* __restrict__ psi, double2* __restrict__ out, i64 row_lo, i64 row_hi, Epilogue ep,
        double2* __restrict__ partials) {
    extern __shared__ __align__(128) unsigned char smem_raw[];
    __shared__ double2 sh_red[32];
    const RowPlanDev& P = L.P;
    const u32 Db = (u32)P.B.D;
    u64* bar = reinterpret_cast<u64*>(smem_raw);
    double2* rowbuf = reinterpret_cast<double2*>(smem_raw + 16);           // [2][Db + 1]
    unsigned short* slist = reinterpret_cast<unsigned short*>(smem_raw + 16 + 2 * (size_t)(Db + 1) * 16);
    double* slut = reinterpret_cast<double*>(smem_raw + 16 + 2 * (size_t)(Db + 1) * 16 + (size_t)L.l_max * (blockDim.x * kLC) * 2);  // [2][8][16]
    const u32 tid = threadIdx.x, kLT = blockDim.x, kLW = kLT * kLC;
    // rows are dealt round-robin (block b takes rows lo + b, lo + b + grid, ...): at any time the running rows
    // are ~grid consecutive ones, so the alpha-hop source rows (near neighbours in rank) stay L2-resident
    const i64 r0 = row_lo + (i64)blockIdx.x, r1 = row_hi, rs = gridDim.x;
    double2 dot = make_double2(0.0, 0.0);
    if (r0 < r1) {
        u32 col[kLC], scol[kLC], tb[kLC];
        bool ok[kLC];
#pragma unroll
        for (int k = 0; k < kLC; ++k) {
            const u32 c = tid + k * kLT;
            ok[k] = c < Db;
            col[k] = min(c, Db - 1u);   // global loads stay in range
            scol[k] = min(c, Db);       // shared-memory reads of idle columns hit the zero amplitude
            tb[k] = P.B.str[col[k]];
        }
        {   // column list -> shared memory (8 bytes per thread and slot, conflict free)
            const uint2* __restrict__ src = reinterpret_cast<const uint2*>(L.llist);
            uint2* dst = reinterpret_cast<uint2*>(slist);
            for (u32 i = tid; i < (u32)L.l_max * kLT; i += kLT) dst[i] = __ldg(src + i);
        }
        auto stage = [&](i64 r, u32 b) {  // thread 0 only
            const u32 bytes = Db * 16u;
            unsigned char* dstp = reinterpret_cast<unsigned char*>(rowbuf + (size_t)b * (Db + 1));
            const unsigned char* srcp = reinterpret_cast<const unsigned char*>(psi + r * (i64)Db);
            mbar_expect_tx(bar + b, bytes);
            for (u32 o = 0; o < bytes; o += 32768u) tma_bulk_g2s(dstp + o, srcp + o, min(32768u, bytes - o), bar + b);
        };
        // Diagonal by nibble look-up: F(t_a, t_b) = V_0 + sum_j V_j (-1)^{parity(dz_j & t_b)}.  The sign pattern of a
        // column is a constant bit mask (bit j-1 for key j), the row supplies 16-entry tables of partial sums over 4
        // keys each: 4 keys cost one LDS.64 + one DADD per column instead of 4 sign flips and adds.
        u32 smask[kLC];
        const u32 d_key0 = L.lut_nq ? __ldg(reinterpret_cast<const u32*>(P.items + L.item0) + 1) : 0u;
        const u32 d_nk = L.lut_nq ? __ldg(reinterpret_cast<const u32*>(P.items + L.item0) + 2) : 0u;
#pragma unroll
        for (int k = 0; k < kLC; ++k) {
            smask[k] = 0;
            for (u32 j = 1; j < d_nk; ++j)
                smask[k] |= ((u32)__popc(tb[k] & __ldg(P.key_dz + d_key0 + j)) & 1u) << (j - 1);
        }
        auto build_lut = [&](i64 r, u32 b) {  // threads 0 .. 16 * lut_nq - 1
            if (tid < 16u * (u32)L.lut_nq) {
                const u32 q = tid >> 4, pat = tid & 15u;
                const double* __restrict__ v = L.vtab + __ldg(L.voff + r) + (d_key0 - L.key0);
                double f = 0.0;
#pragma unroll
                for (u32 j = 0; j < 4; ++j) {
                    const u32 key = 1 + 4 * q + j;
                    if (key < d_nk) f += flip(__ldg(v + key), (pat >> j) & 1u);
                }
                slut[b * 128 + tid] = f;
            }
        };
        if (L.lut_nq) build_lut(r0, 0u);
        if (tid == 0) {
            mbar_init(bar, 1);
            mbar_init(bar + 1, 1);
            asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
            rowbuf[Db] = make_double2(0.0, 0.0);
            rowbuf[2 * Db + 1] = make_double2(0.0, 0.0);
            stage(r0, 0u);
        }
        __syncthreads();
        const uint4* __restrict__ items4 = reinterpret_cast<const uint4*>(P.items);
        const u32 nk0 = reinterpret_cast<const u32*>(P.xa_hdr)[3] - L.key0;  // keys of the x_a = 0 header (header 0)
        const u32 wid = tid >> 5;
        const bool alpha_first = L.order == 1 ? (wid & 1u) : L.order == 2 ? (wid >= kLT / 64u) : L.order == 3 ? ((wid >> 2) & 1u) : false;
        u32 it_n = 0;
        for (i64 r = r0; r < r1; r += rs, ++it_n) {
            const u32 b = it_n & 1u;
            if (tid == 0 && r + rs < r1) stage(r + rs, b ^ 1u);  // buffer b^1 was released by the barrier ending the previous row
            const double2* __restrict__ srow = rowbuf + (size_t)b * (Db + 1);
            const double* __restrict__ Vr = L.vtab + __ldg(L.voff + r);
            double2 acc[kLC];
#pragma unroll
            for (int k = 0; k < kLC; ++k) acc[k] = make_double2(0.0, 0.0);
            if (MODE == 0 && ep.acc) {  // the fused-axpy epilogue will read the accumulator: pull its lines into L2 now
#pragma unroll
                for (int k = 0; k < kLC; ++k)
                    asm volatile("prefetch.global.L2 [%0];" ::"l"(ep.acc + r * (i64)Db + col[k]));
            }
            if (L.lut_nq && r + rs < r1) build_lut(r + rs, b ^ 1u);  // visible after the barrier that ends this row
            // shared-memory phase: diagonal and beta hops from the staged row
            auto smem_phase = [&]() {
            mbar_wait(bar + b, (it_n >> 1) & 1u);
            if (L.lut_nq) {
                const double* __restrict__ lut = slut + b * 128;
                const double f0 = __ldg(Vr + (d_key0 - L.key0));
#pragma unroll
                for (int k = 0; k < kLC; ++k) {
                    double f = f0;
                    for (int q = 0; q < L.lut_nq; ++q) f += lut[q * 16 + ((smask[k] >> (4 * q)) & 15u)];
                    const double2 a = srow[scol[k]];
                    acc[k].x += f * a.x;
                    acc[k].y += f * a.y;
                }
            }
            // dense x_b = 0 groups of the x_a = 0 entry (the diagonal): V-weighted own amplitude
            for (u32 i = L.lut_nq ? L.item_split : L.item0; i < L.item_split; ++i) {
                const uint4 it = __ldg(items4 + i);  // {tkey = ident, key0, nkeys, single}
                const double* __restrict__ v = Vr + (it.y - L.key0);
                double f[kLC];
                const double f0 = __ldg(v);
#pragma unroll
                for (int k = 0; k < kLC; ++k) f[k] = f0;
                if (it.z > 1) {
                    for (u32 j = 1; j < it.z; ++j) {
                        const u32 m = __ldg(P.key_dz + it.y + j);
                        const double vj = __ldg(v + j);
                        if (it.w) {
                            const int sh = __clz((int)m);
#pragma unroll
                            for (int k = 0; k < kLC; ++k) f[k] += flip(vj, (tb[k] << sh) >> 31);
                        } else {
#pragma unroll
                            for (int k = 0; k < kLC; ++k) f[k] += flip(vj, (u32)__popc(tb[k] & m) & 1u);
                        }
                    }
                }
#pragma unroll
                for (int k = 0; k < kLC; ++k) {
                    const double2 a = srow[scol[k]];
                    acc[k].x += f[k] * a.x;
                    acc[k].y += f[k] * a.y;
                }
            }
            // beta-moving groups: uniform column list from shared memory
            if (L.l_max > 0) {
                const double vu = __ldg(Vr + (L.key_split - L.key0));
                const uint2* __restrict__ sl = reinterpret_cast<const uint2*>(slist) + tid;
                const unsigned char* __restrict__ sbytes = reinterpret_cast<const unsigned char*>(srow);
#pragma unroll 4
                for (int s = 0; s < L.l_max; ++s) {
                    const uint2 e = sl[(u32)s * kLT];
                    const u32 en[kLC] = {e.x & 0xFFFFu, e.x >> 16, e.y & 0xFFFFu, e.y >> 16};
#pragma unroll
                    for (int k = 0; k < kLC; ++k) {
                        const double2 a = *reinterpret_cast<const double2*>(sbytes + (SIGN ? (en[k] & 0xFFF0u) : en[k]));
                        const double f = SIGN ? flip(vu, en[k] & 1u) : vu;
                        acc[k].x += f * a.x;
                        acc[k].y += f * a.y;
                    }
                }
            }
            };
            // global phase: alpha hops are row axpys from global memory / L2 (coalesced 128-bit loads), two entries in flight
            auto alpha_phase = [&]() {
            const i64 e0 = __ldg(P.row_off + r), e1 = __ldg(P.row_off + r + 1);
            i64 e = e0 + 1;
            for (; e + 1 < e1; e += 2) {
                const u32 s0 = __ldg(reinterpret_cast<const u32*>(P.row_ent + e) + 1);
                const u32 s1 = __ldg(reinterpret_cast<const u32*>(P.row_ent + e + 1) + 1);
                const double f0 = __ldg(Vr + nk0 + (u32)(e - e0 - 1)), f1 = __ldg(Vr + nk0 + (u32)(e - e0));
                const double2* __restrict__ p0 = psi + (i64)s0 * Db;
                const double2* __restrict__ p1 = psi + (i64)s1 * Db;
                double2 a[kLC], c[kLC];
#pragma unroll
                for (int k = 0; k < kLC; ++k) {
                    a[k] = __ldg(p0 + col[k]);
                    c[k] = __ldg(p1 + col[k]);
                }
#pragma unroll
                for (int k = 0; k < kLC; ++k) {
                    acc[k].x += f0 * a[k].x + f1 * c[k].x;
                    acc[k].y += f0 * a[k].y + f1 * c[k].y;
                }
            }
            if (e < e1) {
                const u32 s0 = __ldg(reinterpret_cast<const u32*>(P.row_ent + e) + 1);
                const double f0 = __ldg(Vr + nk0 + (u32)(e - e0 - 1));
                const double2* __restrict__ p0 = psi + (i64)s0 * Db;
                double2 a[kLC];
#pragma unroll
                for (int k = 0; k < kLC; ++k) a[k] = __ldg(p0 + col[k]);
#pragma unroll
                for (int k = 0; k < kLC; ++k) {
                    acc[k].x += f0 * a[k].x;
                    acc[k].y += f0 * a[k].y;
                }
            }
            };
            // Half of the warps run the global phase first: all warps leave the row barrier together, so without this
            // the shared-memory pipe idles while every warp waits on L2 and vice versa.
            if (alpha_first) {
                alpha_phase();
                smem_phase();
            } else {
                smem_phase();
                alpha_phase();
            }
#pragma unroll
            for (int k = 0; k < kLC; ++k) {
                if (!ok[k]) continue;
                const i64 idx = r * (i64)Db + col[k];
                const double2 pin = srow[col[k]];
                if (L.stream) finish_target<MODE == 2, true>(acc[k], pin, idx, out, ep, dot);
                else finish_target<MODE == 2, false>(acc[k], pin, idx, out, ep, dot);
            }
            __syncthreads();  // everyone is done with buffer b before row r + 2 is staged into it
        }
    }
    if (MODE == 2) {
        dot = block_sum(dot, sh_red);
        if (threadIdx.x == 0) partials[blockIdx.x] = dot;
    }
}

}  // namespace

// Test hooks (include/bs.h "Environment"), read ONCE when the plan is built and stored in it.
static int env_int(const char* name, int dflt) {
    const char* v = getenv(name);
    return v ? atoi(v) : dflt;
}

template <int MODE, bool SIGN>
static cudaError_t light_set_smem(int maxt, size_t smem) {
    switch (maxt) {
        case 512: return cudaFuncSetAttribute(k_light<MODE, 512, SIGN>, cudaFuncAttributeMaxDynamicSharedMemorySize, 227 * 1024 - 1024);
        case 768: return cudaFuncSetAttribute(k_light<MODE, 768, SIGN>, cudaFuncAttributeMaxDynamicSharedMemorySize, 227 * 1024 - 1024);
        case 896: return cudaFuncSetAttribute(k_light<MODE, 896, SIGN>, cudaFuncAttributeMaxDynamicSharedMemorySize, 227 * 1024 - 1024);
        default: return cudaFuncSetAttribute(k_light<MODE, 1024, SIGN>, cudaFuncAttributeMaxDynamicSharedMemorySize, 227 * 1024 - 1024);
    }
}

// Decides whether the plan has the light shape and builds the shared-memory list image and the V table.
int bs_light_build(bs_rowplan* R, cudaStream_t st) {
    R->light = false;
    if (getenv("BS_NO_LIGHT")) return BS_OK;
    const RowPlanDev& P = R->dev;
    const i64 Da = P.A.D, Db = P.B.D;
    if (R->has_cdiag) return BS_OK;   // k_light does not read the per-column diagonal table
    if (!R->real_w || Db > 4094 || Db < 64 || R->h_hdrs.empty() || R->h_xa[0] != 0) return BS_OK;
    const XaHdr& h0 = R->h_hdrs[0];
    const bool listed = h0.item_split < h0.item1;
    if (listed && !(h0.stage & 2u)) return BS_OK;                 // the list must be uniform
    if (!listed && (h0.stage & 1u)) return BS_OK;                 // beta-moving groups outside the list
    for (u32 i = h0.item0; i < h0.item_split; ++i)
        if (R->h_items[i].tkey != kTkeyIdent) return BS_OK;       // dense part: diagonal-type groups only
    for (size_t x = 1; x < R->h_hdrs.size(); ++x)
        if (!R->h_hdrs[x].simple) return BS_OK;                   // every other alpha mask: a plain row axpy
    // threads per block: a quarter of the columns, rounded up to a warp (BS_LIGHT_THREADS overrides: tests)
    int T = (int)(((Db + kLC - 1) / kLC + 31) / 32 * 32);
    if (int t = env_int("BS_LIGHT_THREADS", 0)) T = std::max(T, std::min(kLTmax, (t + 31) / 32 * 32));
    const int kLW = T * kLC;
    // listed tables must be the first n_listed ones and all used by header 0 (true by construction)
    const int n_listed = listed ? R->n_listed : 0;
    DevBuf<uint2> d_tk;
    DevBuf<int> d_cnt;
    int l_max = 0;
    if (n_listed > 0) {
        std::vector<uint2> tk(R->h_tkeys.begin(), R->h_tkeys.begin() + n_listed);
        BS_CUDA(d_tk.upload(tk, st));
        BS_CUDA(d_cnt.alloc(kLW));
        k_light_list<<<(kLW + 255) / 256, 256, 0, st>>>(P.B, d_tk.p, n_listed, 0, 0, T, nullptr, d_cnt.p);
        std::vector<int> hc(kLW);
        BS_CUDA(cudaMemcpyAsync(hc.data(), d_cnt.p, kLW * 4, cudaMemcpyDeviceToHost, st));
        BS_CUDA(cudaStreamSynchronize(st));
        for (int v : hc) l_max = std::max(l_max, v);
    }
    const size_t smem = 16 + 2 * (size_t)(Db + 1) * 16 + (size_t)l_max * kLW * 2 + 2 * 128 * 8;
    if (smem > 227 * 1024 - 1024) return BS_OK;
    BS_CUDA(R->d_llist.alloc((size_t)std::max(1, l_max) * kLW));
    // slot t = table t for every column when some column uses every table (no compaction: see k_light_list);
    // BS_LIGHT_COMPACT (test hook) compacts anyway
    if (l_max > 0) {
        k_light_list<<<(kLW + 255) / 256, 256, 0, st>>>(P.B, d_tk.p, n_listed, l_max, getenv("BS_LIGHT_COMPACT") ? 0 : 1, T,
                                                        R->d_llist.p, d_cnt.p);
        BS_COUNT_LAUNCH(2);
    }
    bool any_sign = false;   // a sign needs a listed table with z_b0 != 0 (NN hops of a chain have none)
    for (int t = 0; t < n_listed; ++t) any_sign |= R->h_tkeys[t].y != 0;
    R->light_sign = any_sign || env_int("BS_LIGHT_SIGN", 0);
    // V table
    std::vector<i64> roff(Da + 1), voff(Da + 1, 0);
    BS_CUDA(cudaMemcpyAsync(roff.data(), R->d_row_off.p, (Da + 1) * 8, cudaMemcpyDeviceToHost, st));
    BS_CUDA(cudaStreamSynchronize(st));
    const i64 nk0 = (i64)h0.key1 - h0.key0;
    for (i64 r = 0; r < Da; ++r) {
        if (roff[r + 1] - roff[r] < 1) return BS_OK;  // every row must start with the x_a = 0 entry
        voff[r + 1] = voff[r] + nk0 + (roff[r + 1] - roff[r] - 1);
    }
    if (voff[Da] > (i64(1) << 27)) return BS_OK;      // 1 GB of V values: not a light operator
    BS_CUDA(R->d_voff.alloc(Da + 1));
    BS_CUDA(R->d_vtab.alloc((size_t)std::max<i64>(1, voff[Da])));
    BS_CUDA(cudaMemcpyAsync(R->d_voff.p, voff.data(), (Da + 1) * 8, cudaMemcpyHostToDevice, st));
    k_light_v<<<(unsigned)Da, 64, 0, st>>>(P, h0.key0, h0.key1, R->d_voff.p, R->d_vtab.p);
    BS_COUNT_LAUNCH(1);
    BS_CUDA(cudaGetLastError());
    BS_CUDA(cudaStreamSynchronize(st));
    // launch configuration, fixed here: the launch path below does nothing but launch
    int dev = 0;
    BS_CUDA(cudaGetDevice(&dev));
    BS_CUDA(cudaDeviceGetAttribute(&R->light_sms, cudaDevAttrMultiProcessorCount, dev));
    R->light_threads = T;
    R->light_maxt = T <= 512 ? 512 : T <= 768 ? 768 : T <= 896 ? 896 : 1024;
    R->light_stream = env_int("BS_LIGHT_STREAM", 1);
    R->light_order = env_int("BS_LIGHT_ORDER", 3);  // 0: every warp runs the shared-memory phase first
    R->light_lut_nq = 0;
    if (h0.item_split - h0.item0 == 1) {
        const u32 nk = R->h_items[h0.item0].nkeys;
        if (nk >= 2 && nk <= 33) R->light_lut_nq = (int)((nk - 1 + 3) / 4);
    }
    if (R->light_sign) {
        BS_CUDA((light_set_smem<0, true>(R->light_maxt, smem)));
        BS_CUDA((light_set_smem<2, true>(R->light_maxt, smem)));
    } else {
        BS_CUDA((light_set_smem<0, false>(R->light_maxt, smem)));
        BS_CUDA((light_set_smem<2, false>(R->light_maxt, smem)));
    }
    R->light_lmax = l_max;
    R->light_smem = smem;
    R->light = true;
    return BS_OK;
}

// rows [lo, hi) through the light kernel; expect: one dot partial per block
int bs_light_apply(bs_rowplan* R, const double2* psi, double2* out, i64 lo, i64 hi, const Epilogue& ep, bool expect,
                   cudaStream_t st, double2* partials, i64* n_partials) {
    const XaHdr& h0 = R->h_hdrs[0];
    LightDev L;
    L.P = R->dev;
    L.llist = R->d_llist.p;
    L.vtab = R->d_vtab.p;
    L.voff = R->d_voff.p;
    L.l_max = R->light_lmax;
    L.item0 = h0.item0;
    L.item_split = h0.item_split;
    L.key0 = h0.key0;
    L.key_split = h0.key_split;
    L.stream = R->light_stream;
    L.order = R->light_order;
    L.lut_nq = R->light_lut_nq;
    const unsigned grid = (unsigned)std::min<i64>(R->light_sms, hi - lo);
    const unsigned T = (unsigned)R->light_threads;
#define BS_LIGHT(M, MT)                                                                                             \
    if (R->light_sign) k_light<M, MT, true><<<grid, T, R->light_smem, st>>>(L, psi, out, lo, hi, ep, expect ? partials : nullptr); \
    else k_light<M, MT, false><<<grid, T, R->light_smem, st>>>(L, psi, out, lo, hi, ep, expect ? partials : nullptr)
#define BS_LIGHT_MT(M)                                   \
    switch (R->light_maxt) {                             \
        case 512: BS_LIGHT(M, 512); break;               \
        case 768: BS_LIGHT(M, 768); break;               \
        case 896: BS_LIGHT(M, 896); break;               \
        default: BS_LIGHT(M, 1024); break;               \
    }
    if (expect) {
        BS_LIGHT_MT(2)
    } else {
        BS_LIGHT_MT(0)
    }
#undef BS_LIGHT_MT
#undef BS_LIGHT
    BS_COUNT_LAUNCH(1);
    BS_CUDA(cudaGetLastError());
    if (n_partials) *n_partials = grid;
    return BS_OK;
}
