// a4, same-spin double excitations resolved over (N - 2)-electron strings ("K2 resolution").
//
// A group whose X mask has four bits on one spin and none on the other (Eq. 28) moves two electrons
// of that spin: target string t and source string u share exactly N - 2 electrons, K2 = t & u.  All strings K2 + {p, q}
// (p < q outside K2) form a FAMILY of P = C(n - N + 2, 2) rows, every such matrix element lies in exactly one family,
// and inside a family the operator is a dense P x P block (zero where the two pairs share an orbital):
//   out[K2 + pair_t, c] += sum_{pair_u disjoint from pair_t} F_g(K2 + pair_t) psi[K2 + pair_u, c],   x_g = pair_t | pair_u,
// F_g(t) = sum_k w_k (-1)^{popc(z_k & t)} the group's phase sum (Eq. 27).  The row kernel reads one source amplitude
// from L2 per non-zero (28 x 28 = 784 source rows per target row at configs[3], 1,656 at configs[4]: it runs at the
// L2 -> SM bandwidth).  Here a thread block owns (family, tile of 12 target rows): one thread per column keeps the
// tile's accumulators in registers and every source amplitude it loads (coalesced, one row after the other) feeds all
// targets of the tile, with the coupling tile broadcast from shared memory -- 2 x 12 DFMA per 16-byte load.  A target
// row belongs to C(N, 2) families; the blocks write their tiles to a scratch S2[family][member][column] and a second
// kernel adds the C(N, 2) contributions of every target in a fixed order (deterministic, no atomics), column slab by
// column slab so that the scratch stays bounded.
#pragma once
#include "bs_plan.cuh"

struct K2Dev {
    const u32* mrow;    // [F][P] row index of family member m (string K2 | pair)
    const u32* mpair;   // [F][P] the member's pair mask (two bits)
    const u32* fk2;     // [F] the family's K2 string
    const u32* goff;    // [C(n,4) + 1] string range of the group whose 4-bit mask has that combinadic rank (may be empty)
    const u32* gza;     // strings: Z mask on the moving spin
    const double* gw;   //          weight
    const u32* tf;      // [rows][NP2] scratch slot (family * P + member) of the row's j-th electron pair
    const double* ctile;   // [F][n_tiles][(P + 4) * k2_gs] coupling tiles of the tensor form, evaluated once at plan time
                           // (they depend on the operator and the sector only); nullptr: evaluated in the kernel
    int P, F, NP2, n_tiles, rt;
};

struct bs_k2 {
    int n = 0, N = 0, P = 0, F = 0, NP2 = 0, rt = 0, n_tiles = 0;
    i64 rows = 0, slab_cols = 0;
    size_t smem = 0;
    bool mma = true;        // contraction on the FP64 tensor instruction (k_aa_mma), else DFMA (k_aa)
    i64 n_groups = 0;
    std::vector<u32> h_x;   // row-spin X masks of the groups taken (bs_plan_groups)
    DevBuf<u32> d_mrow, d_mpair, d_fk2, d_goff, d_gza, d_tf;
    DevBuf<double> d_gw, d_ctile;
    DevBuf<double2> d_S2;
    K2Dev dev{};
};

// Takes the qualifying groups (x on the ROW spin: four bits; nothing on the column spin) out of `groups`.
// row_strings: the row spin's strings (increasing), n orbitals, N electrons; row_len: amplitudes per row.
int bs_k2_build(std::vector<HostGroup>& groups, const std::vector<u64>& row_strings, int n, int N, i64 row_len,
                cudaStream_t st, bs_k2** out);
// acc[r][c] += (same-spin doubles) psi, rows r in [row_lo, row_hi), columns c in [col_lo, col_hi); psi and acc are
// [rows][row_len] row-major
int bs_k2_apply(bs_k2* K, const double2* psi, double2* acc, i64 row_len, i64 row_lo, i64 row_hi, i64 col_lo, i64 col_hi,
                cudaStream_t st);
