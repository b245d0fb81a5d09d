// Sector-specific device tables of one (operator, sector) pair ("plan"), built once and cached.
#pragma once
#include "bs_internal.cuh"

// One chunk of the full-space kernel's TMA-staged table stream: strings [s0, s1) (s0 even) and the
// groups [g0, g1] that own them.
struct FullChunk {
    int g0, g1;  // inclusive group range
    int s0, s1;  // string range
};

// host-side group after z-reduction (bs_plan.cu), oriented: xa acts on the row spin, xb on the column spin
struct HostStr {
    u32 za, zb;
    double re, im;
};
struct HostGroup {
    u32 xa, xb;
    std::vector<HostStr> s;  // sorted by (zb, za), merged, non-zero
};

struct bs_rowplan;
struct bs_kres;
struct bs_k2;
int bs_rowplan_build(bs_rowplan* R, const std::vector<HostGroup>& groups, const SpinTab& A, const SpinTab& B,
                     cudaStream_t st, bool with_tables = true);
void bs_rowplan_free(bs_rowplan* R);

struct bs_plan {
    ~bs_plan();
    u64 op_id = 0, sector_id = 0;
    bool full = false;
    bool real_w = false;  // every weight has zero imaginary part (Hermitian real-coefficient H)

    // ---- sector mode -------------------------------------------------------------------------
    // Groups are re-ordered by (xa, xb) with xa = x & (2^n - 1), xb = x >> n.  Groups whose xa or
    // xb has odd popcount can never map the sector into itself and are dropped.  Strings are
    // reduced modulo x (z_s and z_s ^ x_s give the same sign up to the constant (-1)^{popc(x_s)/2}
    // on every valid target) and merged, see DESIGN.md "z-reduction".
    int n_xa = 0;
    i64 n_groups = 0, n_strings = 0, n_row_ent = 0;
    int max_row_ent = 0;
    DevBuf<u32> d_xa;          // [n_xa]     distinct alpha masks, ascending
    DevBuf<u32> d_ga_off;      // [n_xa + 1] group range of each alpha mask
    DevBuf<uint4> d_ghdr;      // [n_groups] {xb, first string, n strings, popc(xb)}
    DevBuf<uint2> d_szab;      // [n_strings] {za, zb}
    DevBuf<double2> d_sw;      // [n_strings] weights
    DevBuf<i64> d_row_off;     // [Da + 1]   per target alpha row: range in d_row_ent
    DevBuf<uint2> d_row_ent;   // {alpha-mask id, source alpha row} for every valid (row, mask)

    // ---- full-space mode ----------------------------------------------------------------------
    std::vector<FullChunk> h_chunks;
    DevBuf<FullChunk> d_chunks;
    int n_chunks = 0;

    // ---- v2 row plans (bs_rowplan.cuh); null -> the v1 kernel is used --------------------------------
    bs_rowplan* rp_main = nullptr;  // D, A, AB groups (and B groups when they are few)
    bs_rowplan* rp_t = nullptr;     // B groups as A groups of the transposed problem (when they are many)
    bs_kres* kres = nullptr;        // alpha-beta groups resolved over (N_beta - 1)-electron strings (bs_kres.cuh)
    bs_k2* k2_main = nullptr;       // same-spin doubles of the row spin resolved over (N - 2)-electron strings (bs_k2.cuh)
    bs_k2* k2_t = nullptr;          // the same for the column spin, on the transposed problem
    int rows_fallback = 0;          // 1: a v2 row plan could not be built (allocation, limits) and the v1 kernel runs
    DevBuf<double2> d_psi_t, d_out_t, d_raw;  // transposed input / output, raw H psi (lazily allocated)

    // partial sums of bs_expect, one per thread block of the apply grid
    DevBuf<double2> d_partials;
    i64 n_partials = 0;
};
