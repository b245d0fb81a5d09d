// a4 apply (Eq. 27), a5 expectation (Eq. 5), a7 Taylor driver
// (Eq. 6-7).  Hand-written CUDA for sm_100a; no tensor cores (this is a gather with
// integer bit math, not a contraction).
//
// Sector kernel: one thread block owns a tile of target configurations -- one alpha row t_a and
// kColsPerBlock consecutive beta columns t_b (beta is the contiguous index, reading U4).
// Per valid alpha mask of the row (precomputed list: mask id, source row) it walks the groups
// sharing that alpha mask; per group every thread tests its column (2 popc(t_b & x_b) = popc(x_b)),
// ranks the source column with two table lookups, evaluates the Z-phase sum
//   sum_k w_k (-1)^{popc((za_k & t_a) ^ (zb_k & t_b))}
// (one AND/LOP3 + POPC per string; alpha and beta halves folded with XOR because
// parity(a) ^ parity(b) = parity(a ^ b)), gathers psi[src_row * D_b + src_col] with one 128-bit
// load and accumulates in registers.  Groups with x_b = 0 read their source row contiguously.
#include <algorithm>

#include "bs_epilogue.cuh"
#include "bs_plan.cuh"

extern const int kFullChunkStrings;
int bs_rows_apply(bs_plan* P, bs_sector* s, const double2* psi, double2* out, i64 lo, i64 hi, const Epilogue& ep,
                  bool expect, cudaStream_t st, i64* n_partials_out, double2** partials_out);

namespace {

constexpr int kThreads = 256;
constexpr int kCpt = 2;  // columns per thread
constexpr int kColsPerBlock = kThreads * kCpt;

template <bool EXPECT, bool REALW>
__global__ void __launch_bounds__(kThreads)
k_apply_sector(SpinTab A, SpinTab B, const u32* __restrict__ ga_off, const uint4* __restrict__ ghdr,
               const uint2* __restrict__ szab, const double2* __restrict__ sw, const i64* __restrict__ row_off,
               const uint2* __restrict__ row_ent, const double2* __restrict__ psi, double2* __restrict__ out,
               i64 row_lo, Epilogue ep, double2* __restrict__ partials) {
    __shared__ double2 sh_red[32];
    const i64 row = row_lo + blockIdx.y;
    const i64 Db = B.D;
    const u32 ta = A.str[row];
    u32 col[kCpt], tb[kCpt];
    bool ok[kCpt];
    double2 acc[kCpt];
#pragma unroll
    for (int c = 0; c < kCpt; ++c) {
        col[c] = blockIdx.x * kColsPerBlock + c * kThreads + threadIdx.x;
        ok[c] = col[c] < Db;
        tb[c] = ok[c] ? B.str[col[c]] : 0u;
        acc[c] = make_double2(0.0, 0.0);
    }
    const i64 e0 = row_off[row], e1 = row_off[row + 1];
    for (i64 e = e0; e < e1; ++e) {
        const uint2 ent = __ldg(row_ent + e);
        const u32 g0 = __ldg(ga_off + ent.x), g1 = __ldg(ga_off + ent.x + 1);
        const double2* __restrict__ src_row = psi + (i64)ent.y * Db;
        for (u32 g = g0; g < g1; ++g) {
            const uint4 h = __ldg(ghdr + g);  // {xb, first string, n strings, popc(xb)}
#pragma unroll
            for (int c = 0; c < kCpt; ++c) {
                const bool valid = ok[c] && (2u * (u32)__popc(tb[c] & h.x) == h.w);
                if (!valid) continue;
                const u32 js = h.x ? spin_rank(B, tb[c] ^ h.x) : col[c];
                const double2 v = __ldg(src_row + js);
                double pr = 0.0, pi = 0.0;
                for (u32 k = h.y; k < h.y + h.z; ++k) {
                    const uint2 zz = __ldg(szab + k);
                    const double2 w = __ldg(sw + k);
                    const u32 par = (u32)__popc((zz.x & ta) ^ (zz.y & tb[c])) & 1u;
                    pr += flip(w.x, par);
                    if (!REALW) pi += flip(w.y, par);
                }
                if (REALW) {
                    acc[c].x += pr * v.x;
                    acc[c].y += pr * v.y;
                } else {
                    acc[c].x += pr * v.x - pi * v.y;
                    acc[c].y += pr * v.y + pi * v.x;
                }
            }
        }
    }
    double2 dot = make_double2(0.0, 0.0);
#pragma unroll
    for (int c = 0; c < kCpt; ++c) {
        if (!ok[c]) continue;
        const i64 idx = row * Db + col[c];
        double2 pin = make_double2(0.0, 0.0);
        if (EXPECT || ep.use_axpby) pin = psi[idx];
        finish_target<EXPECT>(acc[c], pin, idx, out, ep, dot);
    }
    if (EXPECT) {
        dot = block_sum(dot, sh_red);
        if (threadIdx.x == 0) partials[(i64)blockIdx.y * gridDim.x + blockIdx.x] = dot;
    }
}

// Full-space kernel (n_alpha = n_beta = -1): index = configuration word, every group is valid for
// every target.  One thread per target; the group/string tables are streamed through shared
// memory in double-buffered chunks by TMA bulk copies signalled on mbarriers.
constexpr int kFullStr = 512;  // strings per chunk (== kFullChunkStrings)
struct __align__(16) FullStage {
    u64 z[kFullStr + 2];
    double2 w[kFullStr + 2];
    u64 xg[kFullStr + 4];
    i64 offs[kFullStr + 4];
};

template <bool EXPECT>
__global__ void __launch_bounds__(kThreads)
k_apply_full(const u64* __restrict__ xg, const i64* __restrict__ offs, const u64* __restrict__ z,
             const double2* __restrict__ w, const FullChunk* __restrict__ chunks, int n_chunks,
             const double2* __restrict__ psi, double2* __restrict__ out, i64 lo, i64 hi, Epilogue ep,
             double2* __restrict__ partials) {
    extern __shared__ __align__(128) unsigned char smem_raw[];
    FullStage* stage = reinterpret_cast<FullStage*>(smem_raw);
    __shared__ u64 bar[2];
    __shared__ double2 sh_red[32];
    const i64 t = lo + blockIdx.x * (i64)kThreads + threadIdx.x;
    const bool ok = t < hi;
    if (threadIdx.x == 0) {
        mbar_init(&bar[0], 1);
        mbar_init(&bar[1], 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();
    auto issue = [&](int c) {
        const FullChunk ch = chunks[c];
        FullStage& S = stage[c & 1];
        const int ns = ch.s1 - ch.s0;                 // s0 is even -> 16-byte aligned sources
        const int gb = ch.g0 & ~1, ng = ch.g1 - gb + 2;  // groups gb .. g1+1 (offs needs one more)
        const u32 bz = round16(ns * 8), bw = ns * 16, bx = round16(ng * 8);
        mbar_expect_tx(&bar[c & 1], bz + bw + 2 * bx);
        tma_bulk_g2s(S.z, z + ch.s0, bz, &bar[c & 1]);
        tma_bulk_g2s(S.w, w + ch.s0, bw, &bar[c & 1]);
        tma_bulk_g2s(S.xg, xg + gb, bx, &bar[c & 1]);
        tma_bulk_g2s(S.offs, offs + gb, bx, &bar[c & 1]);
    };
    if (threadIdx.x == 0 && n_chunks > 0) issue(0);
    double2 acc = make_double2(0.0, 0.0);
    for (int c = 0; c < n_chunks; ++c) {
        if (threadIdx.x == 0 && c + 1 < n_chunks) issue(c + 1);  // stage (c+1)&1 was released by the barrier below
        mbar_wait(&bar[c & 1], (c >> 1) & 1);
        const FullChunk ch = chunks[c];
        const FullStage& S = stage[c & 1];
        const int gb = ch.g0 & ~1;
        if (ok) {
            for (int g = ch.g0; g <= ch.g1; ++g) {
                const u64 x = S.xg[g - gb];
                const int k0 = max((int)S.offs[g - gb], ch.s0) - ch.s0;
                const int k1 = min((int)S.offs[g - gb + 1], ch.s1) - ch.s0;
                const double2 v = __ldg(psi + (t ^ (i64)x));
                double pr = 0.0, pi = 0.0;
                for (int k = k0; k < k1; ++k) {
                    const u32 par = (u32)__popcll(S.z[k] & (u64)t) & 1u;
                    pr += flip(S.w[k].x, par);
                    pi += flip(S.w[k].y, par);
                }
                acc.x += pr * v.x - pi * v.y;
                acc.y += pr * v.y + pi * v.x;
            }
        }
        __syncthreads();  // every thread is done reading stage c&1 before it is refilled
    }
    double2 dot = make_double2(0.0, 0.0);
    if (ok) {
        double2 pin = make_double2(0.0, 0.0);
        if (EXPECT || ep.use_axpby) pin = psi[t];
        finish_target<EXPECT>(acc, pin, t, out, ep, dot);
    }
    if (EXPECT) {
        dot = block_sum(dot, sh_red);
        if (threadIdx.x == 0) partials[blockIdx.x] = dot;
    }
}

// fixed-order final reduction of the per-block partials (deterministic run to run)
__global__ void __launch_bounds__(1024) k_reduce_partials(const double2* __restrict__ partials, i64 n,
                                                         double2* __restrict__ result) {
    __shared__ double2 sh_red[32];
    double2 v = make_double2(0.0, 0.0);
    for (i64 i = threadIdx.x; i < n; i += blockDim.x) {
        v.x += partials[i].x;
        v.y += partials[i].y;
    }
    v = block_sum(v, sh_red);
    if (threadIdx.x == 0) *result = v;
}

// <a|b> partials: grid-stride with a fixed grid, 128-bit loads
__global__ void __launch_bounds__(256) k_vdot(const double2* __restrict__ a, const double2* __restrict__ b, i64 n,
                                              double2* __restrict__ partials) {
    __shared__ double2 sh_red[32];
    double2 v = make_double2(0.0, 0.0);
    for (i64 i = blockIdx.x * (i64)blockDim.x + threadIdx.x; i < n; i += (i64)gridDim.x * blockDim.x) {
        double2 x = a[i], y = b[i];
        v.x += x.x * y.x + x.y * y.y;
        v.y += x.x * y.y - x.y * y.x;
    }
    v = block_sum(v, sh_red);
    if (threadIdx.x == 0) partials[blockIdx.x] = v;
}

Epilogue plain_epilogue() {
    Epilogue ep;
    ep.alpha = make_double2(1.0, 0.0);
    ep.beta = make_double2(0.0, 0.0);
    ep.scale = make_double2(1.0, 0.0);
    ep.acc = nullptr;
    ep.use_axpby = 0;
    ep.add_in = 0;
    ep.store_out = 1;
    ep.scale_acc = 0;
    return ep;
}

int check_state_ptr(const void* p, const char* what) {
    BS_REQUIRE(p, BS_ERR_ARG, "%s is NULL", what);
    BS_REQUIRE((reinterpret_cast<uintptr_t>(p) & 15u) == 0, BS_ERR_ARG, "%s is not 16-byte aligned", what);
    return BS_OK;
}

// launches the apply kernel over rows [lo, hi) (full space: indices); expect != 0 writes partials
int launch_apply(bs_op* op, bs_sector* s, const double2* psi, double2* out, i64 lo, i64 hi, const Epilogue& ep,
                 bool expect, cudaStream_t st, i64* n_partials_out, double2** partials_out) {
    bs_plan* P = nullptr;
    int rc = bs_plan_get(op, s, st, &P);
    if (rc != BS_OK) return rc;
    if (hi <= lo) {
        if (n_partials_out) *n_partials_out = 0;
        return BS_OK;
    }
    if (!s->full && P->rp_main) return bs_rows_apply(P, s, psi, out, lo, hi, ep, expect, st, n_partials_out, partials_out);
    if (s->full) {
        BS_REQUIRE(kFullChunkStrings == kFullStr, BS_ERR_ARG, "internal: chunk size mismatch");
        i64 nblk = (hi - lo + kThreads - 1) / kThreads;
        if (expect && P->n_partials < nblk) {
            BS_CUDA(P->d_partials.alloc(nblk));
            P->n_partials = nblk;
        }
        size_t smem = 2 * sizeof(FullStage);
        if (expect)
            k_apply_full<true><<<(unsigned)nblk, kThreads, smem, st>>>(op->d_xg.p, op->d_offs.p, op->d_z.p, op->d_w.p,
                                                                       P->d_chunks.p, P->n_chunks, psi, out, lo, hi, ep,
                                                                       P->d_partials.p);
        else
            k_apply_full<false><<<(unsigned)nblk, kThreads, smem, st>>>(op->d_xg.p, op->d_offs.p, op->d_z.p, op->d_w.p,
                                                                        P->d_chunks.p, P->n_chunks, psi, out, lo, hi,
                                                                        ep, nullptr);
        if (n_partials_out) *n_partials_out = nblk;
    } else {
        dim3 grid((unsigned)((s->Db + kColsPerBlock - 1) / kColsPerBlock), (unsigned)(hi - lo));
        i64 nblk = (i64)grid.x * grid.y;
        if (expect && P->n_partials < nblk) {
            BS_CUDA(P->d_partials.alloc(nblk));
            P->n_partials = nblk;
        }
        // gridDim.y is limited to 65535: launch in row slabs
        i64 done = 0;
        for (i64 r = lo; r < hi; r += 65535) {
            i64 nr = std::min<i64>(65535, hi - r);
            dim3 g2(grid.x, (unsigned)nr);
            double2* part = expect ? P->d_partials.p + done * grid.x : nullptr;
#define BS_LAUNCH_SECTOR(E, R)                                                                                      \
    k_apply_sector<E, R><<<g2, kThreads, 0, st>>>(s->ta, s->tb, P->d_ga_off.p, P->d_ghdr.p, P->d_szab.p, P->d_sw.p, \
                                                  P->d_row_off.p, P->d_row_ent.p, psi, out, r, ep, part)
            if (expect) {
                if (P->real_w) BS_LAUNCH_SECTOR(true, true);
                else BS_LAUNCH_SECTOR(true, false);
            } else {
                if (P->real_w) BS_LAUNCH_SECTOR(false, true);
                else BS_LAUNCH_SECTOR(false, false);
            }
#undef BS_LAUNCH_SECTOR
            BS_COUNT_LAUNCH(1);
            done += nr;
        }
        if (n_partials_out) *n_partials_out = nblk;
        if (partials_out) *partials_out = P->d_partials.p;
        BS_CUDA(cudaGetLastError());
        return BS_OK;
    }
    BS_COUNT_LAUNCH(1);
    if (partials_out) *partials_out = P->d_partials.p;
    BS_CUDA(cudaGetLastError());
    return BS_OK;
}

int check_pair(bs_op* op, bs_sector* s, const char* fn) {
    BS_REQUIRE(op && s, BS_ERR_ARG, "%s: NULL handle", fn);
    BS_REQUIRE(op->n_qubits == s->n_qubits, BS_ERR_MISMATCH, "%s: operator has %d qubits, sector has %d", fn,
               op->n_qubits, s->n_qubits);
    return BS_OK;
}

}  // namespace

extern "C" int bs_apply_rows(bs_op_t op, bs_sector_t s, const void* psi_in, void* psi_out, int64_t row_lo,
                             int64_t row_hi, void* cuda_stream) {
    int rc = check_pair(op, s, "bs_apply_rows");
    if (rc) return rc;
    if ((rc = check_state_ptr(psi_in, "psi_in")) || (rc = check_state_ptr(psi_out, "psi_out"))) return rc;
    BS_REQUIRE(psi_in != psi_out, BS_ERR_ARG, "bs_apply: psi_in and psi_out must be distinct buffers");
    i64 nrows = s->full ? s->D : s->Da;
    BS_REQUIRE(row_lo >= 0 && row_lo <= row_hi && row_hi <= nrows, BS_ERR_ARG, "bs_apply_rows: bad row range");
    return launch_apply(op, s, (const double2*)psi_in, (double2*)psi_out, row_lo, row_hi, plain_epilogue(), false,
                        (cudaStream_t)cuda_stream, nullptr, nullptr);
}

extern "C" int bs_apply(bs_op_t op, bs_sector_t s, const void* psi_in, void* psi_out, void* cuda_stream) {
    BS_REQUIRE(op && s, BS_ERR_ARG, "bs_apply: NULL handle");
    return bs_apply_rows(op, s, psi_in, psi_out, 0, s->full ? s->D : s->Da, cuda_stream);
}

extern "C" int bs_apply_axpby(bs_op_t op, bs_sector_t s, const void* psi_in, void* psi_out,
                              const double alpha_reim[2], const double beta_reim[2], void* acc, void* cuda_stream) {
    int rc = check_pair(op, s, "bs_apply_axpby");
    if (rc) return rc;
    if ((rc = check_state_ptr(psi_in, "psi_in")) || (rc = check_state_ptr(psi_out, "psi_out"))) return rc;
    BS_REQUIRE(psi_in != psi_out && psi_in != acc && psi_out != acc, BS_ERR_ARG,
               "bs_apply_axpby: psi_in, psi_out and acc must be distinct buffers");
    BS_REQUIRE(alpha_reim && beta_reim, BS_ERR_ARG, "bs_apply_axpby: NULL scalar");
    BS_REQUIRE(!acc || (reinterpret_cast<uintptr_t>(acc) & 15u) == 0, BS_ERR_ARG, "acc is not 16-byte aligned");
    Epilogue ep = plain_epilogue();
    ep.use_axpby = 1;
    ep.alpha = make_double2(alpha_reim[0], alpha_reim[1]);
    ep.beta = make_double2(beta_reim[0], beta_reim[1]);
    ep.acc = (double2*)acc;
    return launch_apply(op, s, (const double2*)psi_in, (double2*)psi_out, 0, s->full ? s->D : s->Da, ep, false,
                        (cudaStream_t)cuda_stream, nullptr, nullptr);
}

static int finish_reduction(bs_sector* s, const double2* partials, i64 n, double result_reim[2], cudaStream_t st) {
    k_reduce_partials<<<1, 1024, 0, st>>>(partials, n, s->d_result.p);
    BS_COUNT_LAUNCH(1);
    BS_CUDA(cudaGetLastError());
    double2 r;
    BS_CUDA(cudaMemcpyAsync(&r, s->d_result.p, 16, cudaMemcpyDeviceToHost, st));
    BS_CUDA(cudaStreamSynchronize(st));
    result_reim[0] = r.x;
    result_reim[1] = r.y;
    return BS_OK;
}

extern "C" int bs_expect(bs_op_t op, bs_sector_t s, const void* psi, double result_reim[2], void* cuda_stream) {
    int rc = check_pair(op, s, "bs_expect");
    if (rc) return rc;
    if ((rc = check_state_ptr(psi, "psi"))) return rc;
    BS_REQUIRE(result_reim, BS_ERR_ARG, "bs_expect: result is NULL");
    cudaStream_t st = (cudaStream_t)cuda_stream;
    i64 np = 0;
    double2* part = nullptr;
    rc = launch_apply(op, s, (const double2*)psi, nullptr, 0, s->full ? s->D : s->Da, plain_epilogue(), true, st, &np,
                      &part);
    if (rc) return rc;
    return finish_reduction(s, part, np, result_reim, st);
}

extern "C" int bs_vdot(bs_sector_t s, const void* a, const void* b, double result_reim[2], void* cuda_stream) {
    BS_REQUIRE(s && result_reim, BS_ERR_ARG, "bs_vdot: NULL argument");
    int rc;
    if ((rc = check_state_ptr(a, "a")) || (rc = check_state_ptr(b, "b"))) return rc;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    const int nblk = 1184;  // 8 blocks per SM on 148 SMs, fixed -> fixed summation order
    k_vdot<<<nblk, 256, 0, st>>>((const double2*)a, (const double2*)b, s->D, s->d_partials.p);
    BS_COUNT_LAUNCH(1);
    BS_CUDA(cudaGetLastError());
    return finish_reduction(s, s->d_partials.p, nblk, result_reim, st);
}

// One shifted Taylor step (reading U9), 'order' fused apply+axpy launches:
//   term_0 = psi, term_k = (-i dt / k) (H - E_s) term_{k-1}, psi <- e^{-i E_s dt} sum_k term_k.
// term_1 cannot be accumulated into psi while psi is still being gathered from, so launch 2 adds
// term_1 + term_2; the last launch applies the global phase to the accumulator and skips the store
// of its own term.
extern "C" int bs_taylor_step(bs_op_t op, bs_sector_t s, void* psi_inout, void* work, double dt, int order,
                              double e_shift, void* cuda_stream) {
    int rc = check_pair(op, s, "bs_taylor_step");
    if (rc) return rc;
    if ((rc = check_state_ptr(psi_inout, "psi")) || (rc = check_state_ptr(work, "work"))) return rc;
    BS_REQUIRE(order >= 2, BS_ERR_ARG, "bs_taylor_step: order must be >= 2");
    cudaStream_t st = (cudaStream_t)cuda_stream;
    double2* psi = (double2*)psi_inout;
    double2* t0 = (double2*)work;
    double2* t1 = t0 + s->D;
    const i64 rows = s->full ? s->D : s->Da;
    const double2 phase = make_double2(cos(e_shift * dt), -sin(e_shift * dt));
    const double2* in = psi;
    double2* outb = t0;
    for (int k = 1; k <= order; ++k) {
        Epilogue ep = plain_epilogue();
        ep.use_axpby = 1;
        // (-i dt / k) (H - E_s): alpha = -i dt/k, beta = +i dt E_s / k
        ep.alpha = make_double2(0.0, -dt / k);
        ep.beta = make_double2(0.0, dt * e_shift / k);
        // psi accumulates the terms in PAIRS: an even launch adds its input u_{k-1} (already staged for the gather) and its
        // output u_k, so odd launches carry no accumulator traffic (32 D bytes instead of 64 D); an odd last term adds alone.
        if (k % 2 == 0) {
            ep.acc = psi;
            ep.add_in = 1;
        } else if (k == order && k >= 3) {
            ep.acc = psi;
            ep.add_in = 0;
        }
        if (k == order) {
            ep.store_out = 0;
            ep.scale_acc = 1;
            ep.scale = phase;
        }
        rc = launch_apply(op, s, in, outb, 0, rows, ep, false, st, nullptr, nullptr);
        if (rc) return rc;
        in = outb;
        outb = (outb == t0) ? t1 : t0;
    }
    return BS_OK;
}
