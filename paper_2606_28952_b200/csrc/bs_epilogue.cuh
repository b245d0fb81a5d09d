// Shared device helpers of the apply kernels: fused epilogue (a4 store / axpby / a5 dot), deterministic
// block reduction, TMA bulk-copy + mbarrier wrappers.
#pragma once
#include "bs_internal.cuh"

struct Epilogue {
    double2 alpha, beta, scale;  // out = scale * (alpha * Hpsi + beta * psi_in [+ acc stuff])
    double2* acc;                // optional accumulator: acc += out (+ psi_in if add_in)
    int use_axpby;               // 0: out = Hpsi
    int add_in;                  // acc += out + psi_in
    int store_out;               // write out
    int scale_acc;               // acc = scale * (acc + out ...) instead of scaling out
};

__device__ __forceinline__ double2 cmul(double2 a, double2 b) {
    return make_double2(a.x * b.x - a.y * b.y, a.x * b.y + a.y * b.x);
}
__device__ __forceinline__ double flip(double v, u32 par) {  // (-1)^par * v by a sign-bit XOR
    return __hiloint2double(__double2hiint(v) ^ (int)(par << 31), __double2loint(v));
}

// block-wide deterministic sum of one double2 per thread -> thread 0
__device__ __forceinline__ double2 block_sum(double2 v, double2* sh) {
    for (int o = 16; o > 0; o >>= 1) {
        v.x += __shfl_down_sync(0xffffffffu, v.x, o);
        v.y += __shfl_down_sync(0xffffffffu, v.y, o);
    }
    int w = threadIdx.x >> 5, l = threadIdx.x & 31;
    if (l == 0) sh[w] = v;
    __syncthreads();
    if (w == 0) {
        int nw = (blockDim.x + 31) >> 5;
        v = (l < nw) ? sh[l] : make_double2(0.0, 0.0);
        for (int o = 16; o > 0; o >>= 1) {
            v.x += __shfl_down_sync(0xffffffffu, v.x, o);
            v.y += __shfl_down_sync(0xffffffffu, v.y, o);
        }
    }
    return v;
}

// STREAM: out / acc are touched once per launch: streaming (evict-first) accesses leave L2 to the state vector
// whose rows are re-read as hop sources
template <bool EXPECT, bool STREAM = false>
__device__ __forceinline__ void finish_target(double2 a, double2 pin, i64 idx, double2* __restrict__ out,
                                              const Epilogue& ep, double2& dot) {
    if (EXPECT) {
        // conj(psi) * Hpsi
        dot.x += pin.x * a.x + pin.y * a.y;
        dot.y += pin.x * a.y - pin.y * a.x;
        return;
    }
    if (ep.use_axpby) {
        double2 r = cmul(ep.alpha, a), b = cmul(ep.beta, pin);
        r.x += b.x;
        r.y += b.y;
        if (ep.acc) {
            double2 c = STREAM ? __ldcs(ep.acc + idx) : ep.acc[idx];
            c.x += r.x;
            c.y += r.y;
            if (ep.add_in) {
                c.x += pin.x;
                c.y += pin.y;
            }
            if (ep.scale_acc) c = cmul(ep.scale, c);
            if (STREAM) __stcs(ep.acc + idx, c);
            else ep.acc[idx] = c;
        }
        if (ep.store_out) {
            if (STREAM) __stcs(out + idx, r);
            else out[idx] = r;
        }
    } else {
        if (STREAM) __stcs(out + idx, a);
        else out[idx] = a;
    }
}

// ---- TMA bulk-copy + mbarrier helpers (cp.async.bulk, SASS: UBLKCP) -----------------------------
__device__ __forceinline__ u32 smem_u32(const void* p) { return (u32)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(u64* bar, u32 count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count));
}
__device__ __forceinline__ void mbar_expect_tx(u64* bar, u32 bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_arrive(u64* bar) {
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void mbar_wait(u64* bar, u32 parity) {
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "WAIT_%=:\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
        "@p bra DONE_%=;\n"
        "bra WAIT_%=;\n"
        "DONE_%=:\n"
        "}\n" ::"r"(smem_u32(bar)), "r"(parity) : "memory");
}
__device__ __forceinline__ void tma_bulk_g2s(void* dst, const void* src, u32 bytes, u64* bar) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(
                     smem_u32(dst)),
                 "l"(src), "r"(bytes), "r"(smem_u32(bar))
                 : "memory");
}
__device__ __forceinline__ u32 round16(u32 b) { return (b + 15u) & ~15u; }

