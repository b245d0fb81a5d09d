// Internal declarations of libbs (not part of the ABI; the ABI is include/bs.h).
#pragma once
#include <cuda_runtime.h>

#include <atomic>
#include <cstdint>
#include <cstdio>
#include <cstring>
#include <map>
#include <mutex>
#include <string>
#include <vector>

#include "bs.h"

using u64 = uint64_t;
using u32 = uint32_t;
using i64 = int64_t;

// ---- errors ---------------------------------------------------------------------------------
void bs_set_error(const char* fmt, ...);
extern std::atomic<int64_t> g_bs_launches;
#define BS_COUNT_LAUNCH(n) (g_bs_launches.fetch_add((n), std::memory_order_relaxed))

#define BS_CUDA(call)                                                                       \
    do {                                                                                    \
        cudaError_t e_ = (call);                                                            \
        if (e_ != cudaSuccess) {                                                            \
            bs_set_error("%s:%d: %s -> %s", __FILE__, __LINE__, #call, cudaGetErrorString(e_)); \
            return (e_ == cudaErrorMemoryAllocation) ? BS_ERR_ALLOC : BS_ERR_CUDA;         \
        }                                                                                   \
    } while (0)

#define BS_REQUIRE(cond, status, ...)   \
    do {                                \
        if (!(cond)) {                  \
            bs_set_error(__VA_ARGS__);  \
            return (status);            \
        }                               \
    } while (0)

// RAII device buffer (library-owned tables only; never state vectors).
template <class T>
struct DevBuf {
    T* p = nullptr;
    size_t n = 0;
    DevBuf() = default;
    DevBuf(const DevBuf&) = delete;
    DevBuf& operator=(const DevBuf&) = delete;
    ~DevBuf() { release(); }
    void release() {
        if (p) cudaFree(p);
        p = nullptr;
        n = 0;
    }
    // allocates n_ elements plus `pad` bytes of slack (bulk copies round sizes up to 16 B)
    cudaError_t alloc(size_t n_, size_t pad = 64) {
        release();
        n = n_;
        return cudaMalloc((void**)&p, n_ * sizeof(T) + pad);
    }
    cudaError_t upload(const std::vector<T>& h, cudaStream_t st) {
        cudaError_t e = alloc(h.size());
        if (e != cudaSuccess || h.empty()) return e;
        return cudaMemcpyAsync(p, h.data(), h.size() * sizeof(T), cudaMemcpyHostToDevice, st);
    }
};

// ---- operator -------------------------------------------------------------------------------
struct bs_op {
    u64 id;        // unique handle id (plan cache key)
    int n_qubits;
    int mode;
    i64 G, M;      // groups, strings
    // host mirrors of the canonical tables (used by bs_op_export and by the plan builder)
    std::vector<u64> h_xg, h_z;
    std::vector<i64> h_offs;
    std::vector<double> h_c, h_w;  // 2*M each
    // device tables (SURVEY 8(a) a2 layout)
    DevBuf<u64> d_xg, d_z;
    DevBuf<i64> d_offs;
    DevBuf<double2> d_w;
    std::vector<u64> validated_sectors;  // sector ids this generator list was leak-checked against
    // per sector id: for every generator the (row, partner row) pairs whose rotation this row owns (a6)
    struct RotRows {
        std::vector<i64> off;   // [G + 1]
        DevBuf<uint2> d_pairs;  // {row, partner row}
        std::vector<i64> coff;  // [G + 1]
        DevBuf<uint2> d_cpairs; // per generator the valid {column, partner column} pairs (x_a = 0: owner side only)
        DevBuf<u32> d_cstr;     // the column spin's string of every d_cpairs entry's first column: read WITH the pair, so the
                                // phase sum does not wait for a second dependent look-up (B.str[column])
        DevBuf<i64> d_off, d_coff;  // device copies of off / coff
        std::vector<i64> roff;  // [G + 1] z-reduced strings of every generator for this sector (exact on valid targets)
        DevBuf<u64> d_rz;
        DevBuf<double2> d_rw;
        DevBuf<i64> d_roff;
        // orbit cells (bs_rot.cu, k_rot_orbit): sub-runs of common-x_a runs whose beta masks touch <= 10 orbitals
        struct OrbitSub {
            i64 j0, j1;        // generators of the sub-run
            int tab;           // index into orbit_tabs (tables shared by sub-runs with the same orbital set U), -1: unusable
            i64 part_off;      // offset of its pair lists in d_opart
            i64 poff_off;      // offset of its [n_gen][12] pair offsets in d_opoff
        };
        struct OrbitU {
            i64 pat_off, out_off;   // offsets into d_opat / d_oout
            int n_pat, n_out, nU;
            int m_off[12];
        };
        std::vector<OrbitSub> orbit_subs;   // sorted by j0; covers every generator of every common-x_a run
        std::vector<OrbitU> orbit_tabs;
        DevBuf<u32> d_opat, d_oout;
        DevBuf<unsigned short> d_opart;
        DevBuf<int> d_opoff;
        DevBuf<double> d_th;    // thetas of the current call
        DevBuf<double2> d_sc;   // (sin, cos) of the thetas
    };
    std::map<u64, RotRows*> rot_rows;
    ~bs_op() {
        for (auto& kv : rot_rows) delete kv.second;
    }
};

// ---- sector ---------------------------------------------------------------------------------
// Device view of one spin's rank/unrank tables.  rank(w) = lo[w & mask_lo] +
// hi[popc(w & mask_lo) << bits_hi | (w >> bits_lo)] for words of the right popcount.
struct SpinTab {
    const u32* str;  // unrank: D words, increasing
    const u32* lo;   // 2^bits_lo entries
    const u32* hi;   // (N+1) * 2^bits_hi entries
    int bits_lo, bits_hi, N;
    u32 mask_lo;
    i64 D;
};

struct bs_sector {
    u64 id;
    bool full;
    int n_orb, n_alpha, n_beta, n_qubits;
    i64 D, Da, Db;
    std::vector<u64> h_sa, h_sb;
    DevBuf<u32> d_sa, d_sb, d_lo_a, d_hi_a, d_lo_b, d_hi_b;
    SpinTab ta, tb;
    // scratch for deterministic reductions (partials of bs_expect / bs_vdot) and flags
    DevBuf<double2> d_partials;
    DevBuf<double2> d_result;
    DevBuf<int> d_flag;
};

__device__ __forceinline__ u32 spin_rank(const SpinTab& t, u32 w) {
    u32 l = w & t.mask_lo;
    u32 r = __ldg(t.lo + l);
    if (t.bits_hi > 0) r += __ldg(t.hi + ((u32)__popc(l) << t.bits_hi | (w >> t.bits_lo)));
    return r;
}

// ---- plan: sector-specific tables of one (operator, sector) pair -------------------------------
struct bs_plan;
int bs_plan_get(bs_op* op, bs_sector* s, cudaStream_t st, bs_plan** out);
void bs_plan_purge(u64 op_id, u64 sector_id);

u64 bs_next_id();
