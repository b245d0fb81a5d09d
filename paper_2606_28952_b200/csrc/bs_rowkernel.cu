// a4 apply, v2 row kernel (Eq. 27; Eq. 28).
//
// One thread block owns one target row t_a and a chunk of target columns t_b; every thread owns CPT
// columns (stride = blockDim, so global accesses coalesce) and keeps their accumulators in registers.
// The row's valid alpha masks (precomputed list: mask id, source row, V-slot offset) are processed in
// batches -- one staged entry, or a run of alpha-only entries whose keys fit the V slots:
//   1. phase factors V_gj(t_a) of every key (= distinct beta Z mask of a group) of the batch go to shared
//      memory, one warp per entry, one lane per key: strings are visited once per row, not once per target;
//   2. a staged entry (some group moves the beta string) gets its source row psi[u_a, :] by TMA bulk copies
//      (cp.async.bulk + mbarrier), in windows if the row is larger than shared memory;
//   3. "simple" entries (one group, x_b = 0, one key) are row axpys with coalesced 128-bit loads; general
//      groups read 4 packed u16 table entries per thread (validity, source column, first sign), add the
//      remaining keys (bit-shift sign for single-bit Z masks, POPC otherwise) and gather the amplitude from
//      the staged row (LDS.128) or from global memory;
//   4. the column-list pass serves all single-key x_b != 0 groups of the entry from a per-column compacted
//      list (no invalid lanes, no branches): V from shared memory by table id, amplitude by LDS.128.
// No tensor cores: this is a gather with integer bit math (north star).
#include <algorithm>

#include "bs_epilogue.cuh"
#include "bs_k2.cuh"
#include "bs_kres.cuh"
#include "bs_plan.cuh"
#include "bs_rowplan.cuh"

namespace {

constexpr int MODE_FINAL = 0, MODE_RAW = 1, MODE_EXPECT = 2;

template <bool REALW>
struct VT;
template <>
struct VT<true> {
    using type = double;
    static __device__ __forceinline__ double zero() { return 0.0; }
    static __device__ __forceinline__ void addflip(double& f, double v, u32 par) { f += flip(v, par); }
    static __device__ __forceinline__ void fma(double2& acc, double f, u32 sg, double2 a) {
        f = flip(f, sg);
        acc.x += f * a.x;
        acc.y += f * a.y;
    }
    static __device__ __forceinline__ double from(double2 w) { return w.x; }
    static __device__ __forceinline__ void add_real(double& f, double v) { f += v; }
    static __device__ __forceinline__ double shfl_add(double f, int o) { return f + __shfl_xor_sync(0xffffffffu, f, o); }
};
template <>
struct VT<false> {
    using type = double2;
    static __device__ __forceinline__ double2 zero() { return make_double2(0.0, 0.0); }
    static __device__ __forceinline__ void addflip(double2& f, double2 v, u32 par) {
        f.x += flip(v.x, par);
        f.y += flip(v.y, par);
    }
    static __device__ __forceinline__ void fma(double2& acc, double2 f, u32 sg, double2 a) {
        f.x = flip(f.x, sg);
        f.y = flip(f.y, sg);
        acc.x += f.x * a.x - f.y * a.y;
        acc.y += f.x * a.y + f.y * a.x;
    }
    static __device__ __forceinline__ double2 from(double2 w) { return w; }
    static __device__ __forceinline__ void add_real(double2& f, double v) { f.x += v; }
    static __device__ __forceinline__ double2 shfl_add(double2 f, int o) {
        return make_double2(f.x + __shfl_xor_sync(0xffffffffu, f.x, o), f.y + __shfl_xor_sync(0xffffffffu, f.y, o));
    }
};

// CPT packed u16 table entries of one thread (the table is stored thread-blocked, see bs_rowplan.cu)
template <int CPT>
__device__ __forceinline__ void load_entries(const unsigned short* __restrict__ p, u32 (&e)[CPT]) {
    if (CPT == 4) {
        const uint2 v = __ldg(reinterpret_cast<const uint2*>(p));
        e[0] = v.x & 0xFFFFu;
        e[1] = v.x >> 16;
        e[2 % CPT] = v.y & 0xFFFFu;
        e[3 % CPT] = v.y >> 16;
    } else if (CPT == 2) {
        const u32 v = __ldg(reinterpret_cast<const u32*>(p));
        e[0] = v & 0xFFFFu;
        e[1 % CPT] = v >> 16;
    } else {
        e[0] = __ldg(p);
    }
}

// Remaining keys of a multi-key group for all CPT columns of the thread at once:
// f[c] = v[0] + sum_{j>=1} (+-) v[j], sign = parity(dz_j & tb[c]).  Single-bit dz (the common case: Z on one
// beta orbital) needs no POPC: the tested bit is shifted into the sign position of the high word.
template <bool REALW, int CPT>
__device__ __forceinline__ void multi_key(typename VT<REALW>::type (&f)[CPT],
                                          const typename VT<REALW>::type* __restrict__ v,
                                          const u32* __restrict__ dz, u32 nkeys, u32 single, const u32 (&tb)[CPT]) {
    using V = VT<REALW>;
    if (single) {
        for (u32 j = 1; j < nkeys; ++j) {
            const int sh = __clz((int)__ldg(dz + j));
            const typename V::type vj = v[j];
#pragma unroll
            for (int c = 0; c < CPT; ++c) V::addflip(f[c], vj, (tb[c] << sh) >> 31);
        }
    } else {
        for (u32 j = 1; j < nkeys; ++j) {
            const u32 m = __ldg(dz + j);
            const typename V::type vj = v[j];
#pragma unroll
            for (int c = 0; c < CPT; ++c) V::addflip(f[c], vj, (u32)__popc(tb[c] & m) & 1u);
        }
    }
}

// All items of one row entry (one valid alpha mask) for this thread's CPT columns.
// STAGED: the source row (window [w0, w0 + wn)) is in shared memory; else it is read from global memory
// (only x_b = 0 items then, i.e. source column = target column).
template <bool REALW, int CPT, bool STAGED, bool WINDOWED>
__device__ __forceinline__ void process_entry(const RowPlanDev& P, const uint4* __restrict__ items4, u32 item0, u32 item1,
                                              u32 hkey0, const typename VT<REALW>::type* __restrict__ vbase,
                                              const double2* __restrict__ srow, const double2* __restrict__ srcp,
                                              u32 w0, u32 wn, u32 tpos, const u32 (&col)[CPT], const u32 (&tb)[CPT],
                                              double2 (&acc)[CPT]) {
    using V = VT<REALW>;
    using vt = typename V::type;
    uint4 nxt = __ldg(items4 + item0);
    for (u32 i = item0; i < item1; ++i) {
        const uint4 it = nxt;  // {tkey, key0, nkeys, single}
        if (i + 1 < item1) nxt = __ldg(items4 + i + 1);
        const vt* __restrict__ v = vbase + (it.y - hkey0);
        const vt f0 = v[0];
        if (it.x == kTkeyIdent) {
            // x_b = 0, no beta sign on the first key: same column of the source row
            double2 a[CPT];
#pragma unroll
            for (int c = 0; c < CPT; ++c) {
                if (STAGED) a[c] = (!WINDOWED || (col[c] - w0) < wn) ? srow[col[c] - w0] : make_double2(0.0, 0.0);
                else a[c] = __ldg(srcp + col[c]);
            }
            if (it.z == 1 && !(it.w & 2u)) {
#pragma unroll
                for (int c = 0; c < CPT; ++c) V::fma(acc[c], f0, 0u, a[c]);
            } else {
                vt f[CPT];
#pragma unroll
                for (int c = 0; c < CPT; ++c) f[c] = f0;
                if (it.w & 2u) {   // row-independent (real) part of the diagonal group, tabulated per column
#pragma unroll
                    for (int c = 0; c < CPT; ++c) V::add_real(f[c], __ldg(P.cdiag + col[c]));
                }
                multi_key<REALW, CPT>(f, v, P.key_dz + it.y, it.z, it.w & 1u, tb);
#pragma unroll
                for (int c = 0; c < CPT; ++c) V::fma(acc[c], f[c], 0u, a[c]);
            }
        } else {
            u32 en16[CPT];
            load_entries<CPT>(P.ttab + (i64)it.x * P.tstride + tpos, en16);
            if (it.z == 1) {
#pragma unroll
                for (int c = 0; c < CPT; ++c) {
                    const u32 src = en16[c] & 0x7FFFu;
                    if (en16[c] == 0xFFFFu || (WINDOWED && (src - w0) >= wn)) continue;
                    const double2 a = STAGED ? srow[src - w0] : __ldg(srcp + src);
                    V::fma(acc[c], f0, en16[c] >> 15, a);
                }
            } else {
                vt f[CPT];
#pragma unroll
                for (int c = 0; c < CPT; ++c) f[c] = f0;
                multi_key<REALW, CPT>(f, v, P.key_dz + it.y, it.z, it.w & 1u, tb);
#pragma unroll
                for (int c = 0; c < CPT; ++c) {
                    const u32 src = en16[c] & 0x7FFFu;
                    if (en16[c] == 0xFFFFu || (WINDOWED && (src - w0) >= wn)) continue;
                    const double2 a = STAGED ? srow[src - w0] : __ldg(srcp + src);
                    V::fma(acc[c], f[c], en16[c] >> 15, a);
                }
            }
        }
    }
}

// Column-list pass of a staged entry: every single-key x_b != 0 group under the alpha mask, compacted per
// column (no invalid lanes, no branches): entry = source column | sign << 15 | table id << 16, V from sVx[id].
// Padding entries point at column Db (a zero amplitude kept behind the staged row) with id n_listed (V = 0).
// UNIF: every listed group has the same row-independent weight `vu` (lattice hopping terms): no V lookup.
template <bool REALW, int CPT, bool WINDOWED, bool UNIF>
__device__ __forceinline__ void list_pass(const RowPlanDev& P, const typename VT<REALW>::type* __restrict__ sVx,
                                          typename VT<REALW>::type vu, const double2* __restrict__ srow, u32 w0, u32 wn,
                                          u32 tpos, double2 (&acc)[CPT], int slot0, int l_max) {
    using V = VT<REALW>;
    const u32 stride = (u32)P.tstride;
    const u32* __restrict__ p = P.ltab + (size_t)slot0 * stride + tpos;
    u32 en[CPT], n1[CPT];
    auto load = [&](u32 (&e)[CPT]) {
        if (CPT == 4) {
            const uint4 v = __ldg(reinterpret_cast<const uint4*>(p));
            e[0] = v.x;
            e[1 % CPT] = v.y;
            e[2 % CPT] = v.z;
            e[3 % CPT] = v.w;
        } else {
#pragma unroll
            for (int c = 0; c < CPT; ++c) e[c] = __ldg(p + c);
        }
        p += stride;
    };
    load(n1);
#pragma unroll 1
    for (int j = 0; j < l_max; ++j) {
#pragma unroll
        for (int c = 0; c < CPT; ++c) en[c] = n1[c];
        if (j + 1 < l_max) load(n1);
#pragma unroll
        for (int c = 0; c < CPT; ++c) {
            const u32 src = en[c] & 0x7FFFu;
            if (WINDOWED && (src - w0) >= wn) continue;
            V::fma(acc[c], UNIF ? vu : sVx[en[c] >> 16], (en[c] >> 15) & 1u, srow[src - w0]);
        }
    }
}

template <int MODE, bool REALW, int CPT, int MAXT>
__global__ void __launch_bounds__(MAXT, (MAXT == 1024 ? 1 : (MAXT == 512 ? 2 : 4)))
k_rows(const RowPlanDev P, const double2* __restrict__ psi, double2* __restrict__ out, i64 row_lo, i64 col_lo,
       i64 col_hi, int chunk0, Epilogue ep, double2* __restrict__ partials) {
    using V = VT<REALW>;
    using vt = typename V::type;
    extern __shared__ __align__(128) unsigned char smem_raw[];
    __shared__ double2 sh_red[32];
    u64* bar = reinterpret_cast<u64*>(smem_raw);
    vt* sV = reinterpret_cast<vt*>(smem_raw + 16);
    vt* sVx = reinterpret_cast<vt*>(smem_raw + 16 + (size_t)P.max_keys * 16);
    double2* srow = reinterpret_cast<double2*>(smem_raw + 16 + (size_t)(P.max_keys + P.n_listed + 1) * 16);
    const int tid = threadIdx.x, nt = blockDim.x;
    const i64 row = row_lo + blockIdx.x;
    const u32 Db = (u32)P.B.D;
    const u32 ta = P.A.str[row];
    const u32 chunk = (u32)chunk0 + blockIdx.y;
    const u32 c0 = chunk * (u32)P.chunk_cols;
    const u32 tpos = (chunk * (u32)nt + (u32)tid) * CPT;  // this thread's slot in a thread-blocked table row
    u32 col[CPT], tb[CPT];
    bool ok[CPT];
    double2 acc[CPT];
#pragma unroll
    for (int c = 0; c < CPT; ++c) {
        const u32 cc = c0 + (u32)tid + (u32)c * (u32)nt;
        ok[c] = cc < c0 + (u32)P.chunk_cols && cc < Db && (i64)cc >= col_lo && (i64)cc < col_hi;
        col[c] = min(cc, Db - 1u);  // clamped: loads stay in range, results of !ok columns are never stored
        tb[c] = P.B.str[col[c]];
        acc[c] = make_double2(0.0, 0.0);
    }
    if (tid == 0) {
        mbar_init(bar, 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
        srow[P.win_cols] = make_double2(0.0, 0.0);  // target of the column list's padding entries
    }
    u32 phase = 0;
    const uint4* __restrict__ items4 = reinterpret_cast<const uint4*>(P.items);
    const int warp = tid >> 5, lane = tid & 31, nwarps = nt >> 5;
    const u32 vcap = (u32)P.max_keys;
    const i64 e0 = P.row_off[row], e1 = P.row_off[row + 1];
    i64 e = e0;
    while (e < e1) {
        // ---- batch: one staged entry, or a run of non-staged entries whose keys fit the V slots ---------
        const uint4 first = __ldg(P.row_ent + e);
        const u32 stage = first.w >> 31;
        const u32 kbase = first.z;
        i64 be = e + 1;
        if (!stage) {
            while (be < e1) {
                const uint4 nx = __ldg(P.row_ent + be);
                if ((nx.w >> 31) || nx.z + (nx.w & 0x3FFFFFFFu) - kbase > vcap) break;
                ++be;
            }
        }
        const double2* __restrict__ srow_g = psi + (i64)first.y * Db;  // staged batches have one entry
        const uint4 hs = __ldg(reinterpret_cast<const uint4*>(P.xa_hdr + first.x) + 1);  // stage,simple,item_split,key_split
        const u32 item_end = __ldg(reinterpret_cast<const u32*>(P.xa_hdr + first.x) + 1);
        const bool listed = (stage & 1u) && hs.z < item_end;
        const bool unif = (hs.x & 2u) != 0;  // all listed groups share one row-independent weight
        __syncthreads();  // everyone is done with the previous batch's V slots and staged row
        if (listed) {
            for (int k = tid; k <= P.n_listed; k += nt) sVx[k] = V::zero();
            __syncthreads();
        }
        const int n_win = stage ? P.n_win : 1;
        for (int w = 0; w < n_win; ++w) {
            const u32 w0 = (u32)w * (u32)P.win_cols;
            const u32 wn = stage ? min((u32)P.win_cols, Db - w0) : 0u;
            if (stage) {
                if (w > 0) __syncthreads();  // readers of the previous window are done
                if (tid == 0) {
                    const u32 bytes = wn * 16u;
                    mbar_expect_tx(bar, bytes);
                    for (u32 o = 0; o < bytes; o += 32768u)
                        tma_bulk_g2s(reinterpret_cast<unsigned char*>(srow) + o,
                                     reinterpret_cast<const unsigned char*>(srow_g + w0) + o, min(32768u, bytes - o),
                                     bar);
                }
            }
            if (w == 0) {
                // phase factors of every key of the batch, one warp per entry (overlaps the bulk copy)
                for (i64 j = e + warp; j < be; j += nwarps) {
                    const uint4 en = __ldg(P.row_ent + j);
                    const u32 key0 = __ldg(reinterpret_cast<const u32*>(P.xa_hdr + en.x) + 2);
                    const u32 nk = en.w & 0x3FFFFFFFu;
                    if (nk == 1 && !listed) {
                        // one key with many strings (e.g. a beta hop's beta-spectator sum on the transposed problem): the
                        // lanes share the strings, fixed-order butterfly
                        vt f = V::zero();
                        const u32 s1 = __ldg(P.key_s0 + key0 + 1);
                        for (u32 s = __ldg(P.key_s0 + key0) + lane; s < s1; s += 32)
                            V::addflip(f, V::from(__ldg(P.s_w + s)), (u32)__popc(__ldg(P.s_za + s) & ta) & 1u);
                        for (int o = 16; o > 0; o >>= 1) f = V::shfl_add(f, o);
                        if (lane == 0) sV[en.z - kbase] = f;
                        continue;
                    }
                    for (u32 k = lane; k < nk; k += 32) {
                        vt f = V::zero();
                        const u32 s1 = __ldg(P.key_s0 + key0 + k + 1);
                        for (u32 s = __ldg(P.key_s0 + key0 + k); s < s1; ++s)
                            V::addflip(f, V::from(__ldg(P.s_w + s)), (u32)__popc(__ldg(P.s_za + s) & ta) & 1u);
                        sV[en.z - kbase + k] = f;
                        if (listed && key0 + k >= hs.w) sVx[__ldg(&P.items[hs.z + (key0 + k - hs.w)].tkey)] = f;
                    }
                }
                __syncthreads();
            }
            if (stage) {
                mbar_wait(bar, phase);
                phase ^= 1u;
            }
            for (i64 j = e; j < be; ++j) {
                const uint4 en = __ldg(P.row_ent + j);
                const double2* __restrict__ srcp = psi + (i64)en.y * Db;
                const vt* __restrict__ vbase = sV + (en.z - kbase);
                if (en.w & 0x40000000u) {
                    // "simple" entry: one group, x_b = 0, one key: out[row, :] += V * psi[source row, :]
                    const vt f0 = vbase[0];
                    double2 a[CPT];
#pragma unroll
                    for (int c = 0; c < CPT; ++c) a[c] = __ldg(srcp + col[c]);
#pragma unroll
                    for (int c = 0; c < CPT; ++c) V::fma(acc[c], f0, 0u, a[c]);
                    continue;
                }
                const uint4 h4 = __ldg(reinterpret_cast<const uint4*>(P.xa_hdr + en.x));  // item0,item1,key0,key1
                if (!stage)
                    process_entry<REALW, CPT, false, false>(P, items4, h4.x, h4.y, h4.z, vbase, srow, srcp, 0u, 0u, tpos,
                                                            col, tb, acc);
                else if (n_win == 1) {
                    if (h4.x < hs.z)
                        process_entry<REALW, CPT, true, false>(P, items4, h4.x, hs.z, h4.z, vbase, srow, srcp, 0u, wn,
                                                               tpos, col, tb, acc);
                    if (listed) {
                        if (unif) list_pass<REALW, CPT, false, true>(P, sVx, vbase[hs.w - h4.z], srow, 0u, wn, tpos, acc, 0, P.l_max);
                        else list_pass<REALW, CPT, false, false>(P, sVx, V::zero(), srow, 0u, wn, tpos, acc, 0, P.l_max);
                    }
                } else {
                    if (h4.x < hs.z)
                        process_entry<REALW, CPT, true, true>(P, items4, h4.x, hs.z, h4.z, vbase, srow, srcp, w0, wn,
                                                              tpos, col, tb, acc);
                    if (listed) {
                        if (P.l_woff) {  // this window's own list: no window test, padding hits the zero amplitude
                            const int s0 = __ldg(P.l_woff + w);
                            const int ns = __ldg(P.l_woff + P.n_win + 1 + w * P.l_nchunks + (int)chunk);
                            if (ns > 0) list_pass<REALW, CPT, false, false>(P, sVx, V::zero(), srow, w0, wn, tpos, acc, s0, ns);
                        } else
                            list_pass<REALW, CPT, true, false>(P, sVx, V::zero(), srow, w0, wn, tpos, acc, 0, P.l_max);
                    }
                }
            }
        }
        e = be;
    }
    double2 dot = make_double2(0.0, 0.0);
#pragma unroll
    for (int c = 0; c < CPT; ++c) {
        if (!ok[c]) continue;
        const i64 idx = row * (i64)Db + col[c];
        if (MODE == MODE_RAW) {
            out[idx] = acc[c];
        } else {
            double2 pin = make_double2(0.0, 0.0);
            if (MODE == MODE_EXPECT || ep.use_axpby) pin = psi[idx];
            finish_target<MODE == MODE_EXPECT>(acc[c], pin, idx, out, ep, dot);
        }
    }
    if (MODE == MODE_EXPECT) {
        dot = block_sum(dot, sh_red);
        if (tid == 0) partials[(i64)blockIdx.y * gridDim.x + blockIdx.x] = dot;
    }
}

// out_t[c][r] = in[r][c] for a [R x C] row-major matrix of complex128 (32 x 32 tiles through shared
// memory, both sides coalesced)
__global__ void __launch_bounds__(256) k_transpose(const double2* __restrict__ in, double2* __restrict__ out_t, i64 R,
                                                   i64 C) {
    __shared__ double2 tile[32][33];
    const i64 r0 = (i64)blockIdx.y * 32, c0 = (i64)blockIdx.x * 32;
    const int tx = threadIdx.x & 31, ty = threadIdx.x >> 5;
    for (int j = ty; j < 32; j += 8)
        if (r0 + j < R && c0 + tx < C) tile[j][tx] = in[(r0 + j) * C + c0 + tx];
    __syncthreads();
    for (int j = ty; j < 32; j += 8)
        if (c0 + j < C && r0 + tx < R) out_t[(c0 + j) * R + r0 + tx] = tile[tx][j];
}

// Final pass when the operator ran in parts: for rows [row_lo, row_hi)
//   H psi [r][c] = raw[r][c]  (+ out_t[c][r]: the part applied to the transposed problem, TRANS)
//                             (+ the N_beta K-resolved alpha-beta contributions of the target, from the scratch: KC.comb)
// then the fused epilogue (store / axpby / dot partial).
template <bool EXPECT, bool TRANS>
__global__ void __launch_bounds__(256)
k_transpose_add_finish(const double2* raw, const double2* __restrict__ out_t,
                       const double2* __restrict__ psi, double2* out, i64 Da, i64 Db, i64 row_lo,
                       i64 row_hi, Epilogue ep, KresComb KC, double2* __restrict__ partials) {
    __shared__ double2 tile[32][33];
    __shared__ double2 sh_red[32];
    const i64 r0 = row_lo + (i64)blockIdx.y * 32, c0 = (i64)blockIdx.x * 32;
    const int tx = threadIdx.x & 31, ty = threadIdx.x >> 5;
    if (TRANS) {
        for (int j = ty; j < 32; j += 8)  // tile[j][tx] = out_t[c0 + j][r0 + tx]
            if (c0 + j < Db && r0 + tx < row_hi) tile[j][tx] = out_t[(c0 + j) * Da + r0 + tx];
        __syncthreads();
    }
    double2 dot = make_double2(0.0, 0.0);
    for (int j = ty; j < 32; j += 8) {
        const i64 r = r0 + j, c = c0 + tx;
        if (r < row_hi && c < Db) {
            const i64 idx = r * Db + c;
            double2 a = raw[idx];
            if (TRANS) {
                const double2 b = tile[tx][j];
                a.x += b.x;
                a.y += b.y;
            }
            if (KC.comb) {
                const double2* __restrict__ Sr = KC.S + (r - KC.slab_lo) * (i64)KC.n * KC.DKp;
                for (int e = 0; e < KC.Nb; ++e) {   // fixed order: deterministic
                    const double2 v = __ldg(Sr + __ldg(KC.comb + c * KC.Nb + e));
                    a.x += v.x;
                    a.y += v.y;
                }
            }
            double2 pin = make_double2(0.0, 0.0);
            if (EXPECT || ep.use_axpby) pin = psi[idx];
            finish_target<EXPECT>(a, pin, idx, out, ep, dot);
        }
    }
    if (EXPECT) {
        dot = block_sum(dot, sh_red);
        if (threadIdx.x == 0) partials[(i64)blockIdx.y * gridDim.x + blockIdx.x] = dot;
    }
}

// The opt-in shared-memory ceiling is raised ONCE per kernel instantiation (thread-safe static initialisation; the
// library drives one device per process), not on every launch; occupancy follows the size actually launched.
constexpr int kMaxDynSmem = 227 * 1024 - 1024;   // + the kernels' static shared memory (reduction scratch) stays under the 227 KB opt-in limit

template <int MODE, bool REALW, int CPT>
cudaError_t launch_k_rows_t(const bs_rowplan* R, dim3 grid, cudaStream_t st, const double2* psi, double2* out,
                            i64 row_lo, i64 col_lo, i64 col_hi, int chunk0, const Epilogue& ep, double2* partials) {
    if (R->threads > 512) {
        auto k = k_rows<MODE, REALW, CPT, 1024>;
        static const cudaError_t e = cudaFuncSetAttribute(k, cudaFuncAttributeMaxDynamicSharedMemorySize, kMaxDynSmem);
        if (e != cudaSuccess) return e;
        k<<<grid, R->threads, R->smem, st>>>(R->dev, psi, out, row_lo, col_lo, col_hi, chunk0, ep, partials);
    } else if (R->threads > 256) {
        auto k = k_rows<MODE, REALW, CPT, 512>;
        static const cudaError_t e = cudaFuncSetAttribute(k, cudaFuncAttributeMaxDynamicSharedMemorySize, kMaxDynSmem);
        if (e != cudaSuccess) return e;
        k<<<grid, R->threads, R->smem, st>>>(R->dev, psi, out, row_lo, col_lo, col_hi, chunk0, ep, partials);
    } else {
        auto k = k_rows<MODE, REALW, CPT, 256>;
        static const cudaError_t e = cudaFuncSetAttribute(k, cudaFuncAttributeMaxDynamicSharedMemorySize, kMaxDynSmem);
        if (e != cudaSuccess) return e;
        k<<<grid, R->threads, R->smem, st>>>(R->dev, psi, out, row_lo, col_lo, col_hi, chunk0, ep, partials);
    }
    return cudaGetLastError();
}

template <int MODE>
cudaError_t launch_k_rows(const bs_rowplan* R, cudaStream_t st, const double2* psi, double2* out, i64 row_lo,
                          i64 row_hi, i64 col_lo, i64 col_hi, const Epilogue& ep, double2* partials) {
    const int chunk0 = (int)(col_lo / R->chunk_cols);
    const unsigned n_chunks = (unsigned)((col_hi - 1) / R->chunk_cols - chunk0 + 1);
    dim3 grid((unsigned)(row_hi - row_lo), n_chunks);
    BS_COUNT_LAUNCH(1);
#define BS_ROWS(RW, C) launch_k_rows_t<MODE, RW, C>(R, grid, st, psi, out, row_lo, col_lo, col_hi, chunk0, ep, partials)
    if (R->real_w) return R->cpt == 1 ? BS_ROWS(true, 1) : BS_ROWS(true, 4);
    return R->cpt == 1 ? BS_ROWS(false, 1) : BS_ROWS(false, 4);
#undef BS_ROWS
}

}  // namespace

int bs_light_apply(bs_rowplan* R, const double2* psi, double2* out, i64 lo, i64 hi, const Epilogue& ep, bool expect,
                   cudaStream_t st, double2* partials, i64* n_partials);

// Runs the v2 path for rows [lo, hi).  expect: dot partials instead of stores.
int bs_rows_apply(bs_plan* P, bs_sector* s, const double2* psi, double2* out, i64 lo, i64 hi, const Epilogue& ep,
                  bool expect, cudaStream_t st, i64* n_partials_out, double2** partials_out) {
    bs_rowplan* M = P->rp_main;
    const i64 Da = s->Da, Db = s->Db;
    if (!P->rp_t && !P->kres && !P->k2_main && M->light) {
        if (expect && P->n_partials < 1024) {
            BS_CUDA(P->d_partials.alloc(1024));
            P->n_partials = 1024;
        }
        i64 np = 0;
        int rc = bs_light_apply(M, psi, out, lo, hi, ep, expect, st, P->d_partials.p, &np);
        if (rc != BS_OK) return rc;
        if (n_partials_out) *n_partials_out = expect ? np : 0;
        if (partials_out) *partials_out = P->d_partials.p;
        return BS_OK;
    }
    if (!P->rp_t && !P->kres && !P->k2_main) {
        const i64 nblk = (hi - lo) * ((Db + M->chunk_cols - 1) / M->chunk_cols);
        if (expect && P->n_partials < nblk) {
            BS_CUDA(P->d_partials.alloc(nblk));
            P->n_partials = nblk;
        }
        if (expect) BS_CUDA(launch_k_rows<MODE_EXPECT>(M, st, psi, out, lo, hi, 0, Db, ep, P->d_partials.p));
        else BS_CUDA(launch_k_rows<MODE_FINAL>(M, st, psi, out, lo, hi, 0, Db, ep, nullptr));
        if (n_partials_out) *n_partials_out = nblk;
        if (partials_out) *partials_out = P->d_partials.p;
        return BS_OK;
    }
    // the operator runs in parts: beta-only groups on the transposed problem (rp_t), alpha-beta groups K-resolved (kres)
    bs_rowplan* T = P->rp_t;
    bs_kres* K = P->kres;
    const bool need_t = T || P->k2_t;
    if (need_t && !P->d_psi_t.p) BS_CUDA(P->d_psi_t.alloc(s->D));
    if (need_t && !P->d_out_t.p) BS_CUDA(P->d_out_t.alloc(s->D));
    double2* raw = out;
    if (expect || !ep.store_out) {
        if (!P->d_raw.p) BS_CUDA(P->d_raw.alloc(s->D));
        raw = P->d_raw.p;
    }
    Epilogue none = ep;
    if (need_t) {
        dim3 tg((unsigned)((Db + 31) / 32), (unsigned)((Da + 31) / 32));
        k_transpose<<<tg, 256, 0, st>>>(psi, P->d_psi_t.p, Da, Db);
        BS_COUNT_LAUNCH(1);
        BS_CUDA(cudaGetLastError());
    }
    BS_CUDA(launch_k_rows<MODE_RAW>(M, st, psi, raw, lo, hi, 0, Db, none, nullptr));
    if (P->k2_main) {   // same-spin doubles of the row spin, added to the raw result
        int rc = bs_k2_apply(P->k2_main, psi, raw, Db, lo, hi, 0, Db, st);
        if (rc != BS_OK) return rc;
    }
    if (T) BS_CUDA(launch_k_rows<MODE_RAW>(T, st, P->d_psi_t.p, P->d_out_t.p, 0, Db, lo, hi, none, nullptr));
    else if (need_t) BS_CUDA(cudaMemsetAsync(P->d_out_t.p, 0, (size_t)s->D * 16, st));
    if (P->k2_t) {      // and of the column spin, on the transposed problem (its columns are the alpha rows)
        int rc = bs_k2_apply(P->k2_t, P->d_psi_t.p, P->d_out_t.p, Da, 0, Db, lo, hi, st);
        if (rc != BS_OK) return rc;
    }
    const unsigned fgx = (unsigned)((Db + 31) / 32);
    const i64 nblk = (i64)fgx * ((hi - lo + 31) / 32 + (K ? (hi - lo) / K->slab_rows + 1 : 0));
    if (expect && P->n_partials < nblk) {
        BS_CUDA(P->d_partials.alloc(nblk));
        P->n_partials = nblk;
    }
    // finishing pass, slab by slab when the K-resolved part needs its scratch
    const i64 slab = K ? K->slab_rows : hi - lo;
    i64 pdone = 0;
    for (i64 r0 = lo; r0 < hi; r0 += slab) {
        const i64 r1 = std::min(hi, r0 + slab);
        KresComb kc{};
        if (K) {
            int rc = bs_kres_apply(K, psi, r0, r1, st);
            if (rc != BS_OK) return rc;
            kc.comb = K->d_comb.p;
            kc.S = K->d_S.p;
            kc.Nb = K->Nb;
            kc.n = K->n;
            kc.DKp = K->DKp;
            kc.slab_lo = r0;
        }
        dim3 fg(fgx, (unsigned)((r1 - r0 + 31) / 32));
        double2* part = expect ? P->d_partials.p + pdone : nullptr;
        const double2* ot = need_t ? P->d_out_t.p : nullptr;
#define BS_FINISH(E, TR) k_transpose_add_finish<E, TR><<<fg, 256, 0, st>>>(raw, ot, psi, out, Da, Db, r0, r1, ep, kc, part)
        if (expect) {
            if (need_t) BS_FINISH(true, true);
            else BS_FINISH(true, false);
        } else {
            if (need_t) BS_FINISH(false, true);
            else BS_FINISH(false, false);
        }
#undef BS_FINISH
        BS_COUNT_LAUNCH(1);
        BS_CUDA(cudaGetLastError());
        pdone += (i64)fg.x * fg.y;
    }
    if (n_partials_out) *n_partials_out = expect ? pdone : 0;
    if (partials_out) *partials_out = P->d_partials.p;
    return BS_OK;
}
