// a4, alpha-beta class resolved over (N_beta - 1)-electron strings ("K resolution").
//
// The dominant share of the non-zeros of a two-body Hamiltonian in an (N_alpha, N_beta) sector (71-72 % at
// BASELINE.json configs[3], configs[4]) couples an alpha move x_a with a beta single hop x_b = {r, s}
// (Eq. 28: X_g = (X_ga, X_gb)).  After the exact phase factorisation of bs_rowplan.cuh every such
// group has ONE key: F_g(t_a, t_b) = V_g(t_a) (-1)^{popc(zb_g & t_b)}, and for Jordan-Wigner strings (Eq. 23,
// PAPER.md:161) zb_g is the chain strictly between r and s.  Write the target beta string as t_b = K + {r} and the
// source as K + {s}, K an (N_beta - 1)-electron string containing neither: the chain sign splits,
//   (-1)^{popc(between(r,s) & K)} = sigma_r(K) sigma_s(K),   sigma_p(K) = (-1)^{popc(K & (2^p - 1))},
// so that for a fixed source row u_a = t_a ^ x_a
//   out[t_a, K + {r}] += sigma_r(K) * sum_s G[s][r] * ( sigma_s(K) psi[u_a, K + {s}] ),
//   G[s][r] = V_{x_a,{r,s}}(t_a) (times the constant sign of zb_g's own bits on r, s), G[r][r] from the x_b = 0 group.
// A small kernel (k_ab_g) evaluates G for every (row, alpha mask) of a slab once -- all K chunks of the row reuse it --
// and a producer warp of k_ab fetches it with the column segments by TMA while the other warps compute.
// One thread owns one K and keeps all n accumulators (one per r) in registers over ALL alpha masks of its row:
// every gathered amplitude psi[u_a, K + {s}] feeds n - N_beta + 1 targets (the column-list pass of k_rows gathers it
// once per target), G comes from shared memory by warp-uniform (broadcast) loads, and the inner loop is plain DFMA:
// the kernel is bound by the FP64 pipe (64 DFMA/clk/SM measured), not by shared-memory gathers.  A block owns a
// chunk of consecutive K and stages, per alpha mask, only the few column segments its K + {s} touch (a fraction of
// the source row) by TMA bulk copies, double buffered.  Accumulators go to a scratch S[row][r][K]; the finishing
// kernel gathers the N_beta contributions of every target (t_b minus each of its electrons) and adds them.
// Groups whose zb is not the JW chain stay on the column-list path of k_rows.
#pragma once
#include "bs_plan.cuh"
#include "bs_rowplan.cuh"

// one entry of a header's coupling matrix: single-string groups carry their weight and alpha Z mask inline
struct __align__(16) KresG {
    double w;
    u32 za;
    u32 code;
};

struct KresDev {
    const i64* row_off;          // kres row plan: valid (kres) alpha masks of every target row
    const uint4* row_ent;        // {header id, source row, -, -}
    const u32* a_str;            // row-spin strings
    const KresG* gtab;           // [n_hdr][NP * NP]: how G[s][r] of a header is made (see bs_kres.cu)
    const KresG* dstr;           // [n_hdr][160] strings (w, za) of the absorbed x_b = 0 group, zero weight beyond the last
    const unsigned short* dkr;   // [n_hdr][64] string range lo | hi << 8 of each of its keys (empty beyond the last)
    const u32* key_s0;           // kres row plan: string range of each key
    const u32* s_za;
    const double2* s_w;
    const unsigned short* goff;  // [n_chunks][NP][KC] staged position of column K + {s} (0: the zero amplitude)
    const u32* sigma;            // [n_chunks * KC] bit p = parity(K & (2^p - 1))
    const uint2* segs;           // [n_chunks][max_segs] {first column, length} of the staged column segments
    const int* seg_cnt;          // [n_chunks]
    int max_segs, KC, n_chunks, n, Nb, buf_elems;
    int n_stages;   // shared-memory buffers of k_ab's producer / consumer pipeline: 3 when they fit, else 2
    i64 Db, DKp;
    double inv_nb;
};

// gather side: the N_beta contributions of one target column, read back from the scratch by the finishing kernel
struct KresComb {
    const u32* comb;             // [Db][Nb]: (r * DKp + rank(K)) | sign << 31, K = t_b minus its j-th electron r
    const double2* S;            // scratch of the current row slab: [row - slab_lo][r][DKp]
    int Nb, n;
    i64 DKp, slab_lo;
};

struct bs_kres {
    bs_rowplan* rp = nullptr;
    int n = 0, NP = 0, Nb = 0, KC = 0, n_chunks = 0, max_segs = 0, buf_elems = 0, n_stages = 2;
    int kc_max = 0;   // the KCMAX instantiation of k_ab this plan launches (its launch bound fixes the register budget)
    i64 DK = 0, DKp = 0, slab_rows = 0;
    size_t smem = 0;
    bool mma = true;             // contraction on the FP64 tensor instruction (else DFMA)
    double staged_rows = 0;      // staged columns per alpha mask, in units of one source row (bs_plan_describe)
    DevBuf<KresG> d_gtab;
    DevBuf<u32> d_sigma, d_comb;
    DevBuf<KresG> d_dstr;
    DevBuf<unsigned short> d_dkr;
    DevBuf<uint2> d_segs;
    DevBuf<int> d_segcnt;
    DevBuf<unsigned short> d_goff;
    DevBuf<double> d_G;          // coupling matrices of one slab, one per (row, alpha mask) (k_ab_g)
    size_t g_bytes = 0;
    DevBuf<double2> d_S;         // scratch for slab_rows rows (allocated at plan build, size in bs_plan_describe)
    KresDev dev{};
    ~bs_kres();
};

struct bs_sector;
// Splits the kres-able groups off `groups` (they are removed from it) and builds the tables; *out stays null when
// nothing qualifies or a limit is hit (the groups then remain in `groups`).
// allow_xa0: also take single-key JW hops under the identity alpha move (the alpha-spectator part of beta single hops,
// split off by the plan builder); never the x = 0 diagonal group.
int bs_kres_build(std::vector<HostGroup>& groups, bs_sector* S, cudaStream_t st, bs_kres** out, bool allow_xa0 = false);
int bs_kres_apply(bs_kres* K, const double2* psi, i64 row_lo, i64 row_hi, cudaStream_t st);
