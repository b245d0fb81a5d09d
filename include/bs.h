/* bs.h -- C ABI of libbs: Pauli-sum operator x sector state-vector multiplication on one B200.
 *
 * Implements the operator-state multiplication path of arxiv/paper_2606_28952 ("BinSim")
 * section 2.4-2.5: a Pauli sum held in binary symplectic form
 * (x mask, z mask, complex coefficient per string; Eq. 12-18) is canonically
 * reduced, grouped by X mask (Eq. 24) and applied to a state
 * vector restricted to an (N_alpha, N_beta) sector (Eq. 25, 28, 38) by
 * target-configuration gathers (Eq. 27).
 *
 * Conventions (DESIGN.md "Readings" U1-U5):
 *   - qubit k = bit k of the 64-bit masks; a string is (x) over k of {I,X,Y,Z} with
 *     (x_k, z_k) = (0,0) I, (1,0) X, (1,1) Y, (0,1) Z                    (Eq. 8).
 *   - coefficients are those of the TRUE Pauli string (not of the XZ-ordered product).
 *   - matrix element: <t| c P |s> = c * (-i)^{ny} * (-1)^{popc(z & t)}, t = s ^ x,
 *     ny = popc(x & z).  The library stores the target-form weight w = c * (-i)^{ny}.
 *   - blocked spin ordering: alpha spin-orbital p = qubit p, beta spin-orbital p = qubit n_orb+p;
 *     bit = 1 means occupied.
 *   - sector vector layout: index(t) = rank_alpha(t_a) * D_beta + rank_beta(t_b), where
 *     t_a = t & (2^n_orb - 1), t_b = t >> n_orb, and rank_s is the combinatorial-number-system
 *     rank (= position among all n_orb-bit words of popcount N_s in increasing numeric order).
 *     Full-space mode (n_alpha = n_beta = -1): index(t) = t.
 *   - all state vectors are complex128, interleaved (re, im), 16-byte aligned DEVICE pointers,
 *     owned by the caller; the library never retains them past the call.
 *
 * Pointers are marked [host] or [device].  Every call returns a bs_status (0 = OK, negative =
 * error, outputs untouched on error) and never throws across the ABI; bs_last_error() gives a
 * thread-local message.  `cuda_stream` is a cudaStream_t passed as void* (NULL = default
 * stream); kernels are enqueued on it and the call returns without synchronising unless stated.
 * There is NO CPU fallback: without a CUDA device every compute entry point returns BS_ERR_CUDA.
 *
 * Threading: the library is not re-entrant per handle.  Calls that use the same operator handle OR the same sector
 * handle share library-owned scratch (cached plan, transposed copies, K-resolution scratch, reduction partials and
 * flags owned by the sector, rotation pair lists owned by the generator handle) and must be issued from one host
 * thread on one stream at a time.  Pairs that share neither handle are independent.  One device per process.
 *
 * Library-owned device memory per (operator, sector) pair, allocated at the first bs_apply / bs_expect of the pair
 * and freed with either handle (bs_plan_info reports the exact byte counts):
 *   - plan tables (row lists: 16 B per valid (alpha row, alpha mask) pair; column tables; 1.2 GB at config 5);
 *   - up to 3 state-vector-sized scratch buffers (transposed psi, transposed result, raw H psi) when beta-only
 *     groups run on the transposed problem (every molecular Hamiltonian): 3 x 16 x dim bytes (20 GB at config 5);
 *   - the scratch of the K-resolved alpha-beta kernel: n_orb x D_K x 16 bytes per alpha row of a slab, at most 4 GiB,
 *     plus its coupling matrices (<= 2.2 GB at config 5); the scratch of the K2-resolved same-spin kernels: 2 x 4 GiB,
 *     plus their coupling tiles evaluated at plan build (2 x 176 MB at config 4, 2 x 390 MB at config 5; none above 2 GB).
 *
 * Environment (TEST HOOKS, not API; every one is read ONCE, when a plan is built, never on a launch path):
 *   BS_KERNEL=v1|v2inrow   force the v1 sector kernel / keep beta-only groups in-row
 *   BS_NO_LIGHT, BS_LIGHT_THREADS, BS_LIGHT_ORDER, BS_LIGHT_STREAM, BS_LIGHT_COMPACT, BS_LIGHT_SIGN   k_light variants
 *   BS_NO_KRES, BS_NO_HOPSPLIT, BS_KRES_KC, BS_KRES_MIN, BS_KRES_SLAB_MB, BS_KRES_MMA, BS_KRES_STAGES, BS_KRES_BIG   K-resolved alpha-beta kernel off / chunk / threshold / slab / DFMA form / pipeline buffers (2 | 3) / 16-compute-warp build on or off
 *   BS_NO_K2, BS_K2_MIN, BS_K2_SLAB_MB, BS_K2_MMA, BS_K2_RT, BS_K2_NT, BS_K2_NO_CTILE   K2-resolved same-spin doubles off / threshold / slab / DFMA form / its tile / tensor form's target tiles of 8 / its coupling tiles evaluated in the kernel, not at plan time
 *   BS_ROT_ORBIT=1   orbit cells (k_rot_orbit) for rotation runs instead of row cells (slower at configs[3]; kept as a
 *                    tested alternative); read once per process
 *   BS_ROT_CSTR=0 | 1   row-cell rotation kernels read a column's string from the sector's table (0) or from a copy kept with
 *                    the pair list (1); default: the copy where amplitudes come through L2 (in place, cluster), the table
 *                    where the cell is in shared memory; read once per process
 *   BS_ROT_CLUSTER=1 | 2   row-pair runs on a thread-block cluster of two, one row per block, partners through distributed
 *                    shared memory (k_rot_cluster_rows): 1 = where the pair exceeds one block's shared memory, 2 = every
 *                    row-pair run (test hook).  Slower than the in-place form at configs[3] (1.62 s vs 1.32 s); kept as a
 *                    tested alternative; read once per process
 *   BS_ROT_IN_PLACE   rotation cells in place (L2) even when they fit shared memory; read once per process
 *   BS_ROW_WIN, BS_ROW_NO_SPLIT, BS_ROW_THREADS, BS_NO_CDIAG   k_rows source-row windows, block size, per-column diagonal table off
 *   BS_ROT_PER_LAUNCH   one launch per rotation generator (no closed-cell batching); read once per process
 */
#ifndef BS_H_
#define BS_H_

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct bs_op*     bs_op_t;     /* grouped Pauli sum, device resident, library owned */
typedef struct bs_sector* bs_sector_t; /* sector tables,     device resident, library owned */
typedef struct bs_symsector* bs_symsector_t; /* point-group block of a sector, library owned */

typedef enum {
    BS_OK = 0,
    BS_ERR_ARG = -1,           /* bad argument (null pointer, size, alignment, n_qubits > 64 ...)  */
    BS_ERR_ALLOC = -2,         /* host or device allocation failed                                */
    BS_ERR_CUDA = -3,          /* CUDA runtime error / no device                                  */
    BS_ERR_MISMATCH = -4,      /* operator and sector disagree on the qubit count                 */
    BS_ERR_NOT_COMMUTING = -5, /* a rotation generator's strings do not mutually commute          */
    BS_ERR_LEAVES_SECTOR = -6  /* a rotation generator maps the sector outside itself             */
} bs_status;

#define BS_MODE_CANONICAL 0
#define BS_MODE_SEQUENCE  1

/* ---- a1 + a2: canonical reduction and X-mask grouping (Eq. 24).
 * x, z [host] u64[M]; coeff_reim [host] double[2M] (true-Pauli coefficients c_k).
 * mode BS_MODE_CANONICAL: sort by key (x major, z minor, unsigned ascending; stable), sum the
 *   coefficients of equal keys in INPUT order, drop |c| < eps_drop (and, also with eps_drop = 0, merged
 *   coefficients that are exactly zero), segment by x.  Runs on the
 *   device (radix sort, segmented sum, compaction).  seq_offsets must be NULL.
 * mode BS_MODE_SEQUENCE: strings [seq_offsets[j], seq_offsets[j+1]) (j < n_seq, seq_offsets[0]=0,
 *   seq_offsets[n_seq]=M) form group j, kept in input order, no merge, no drop; every string of
 *   a run must carry the same x (else BS_ERR_ARG).  Used for rotation generators,
 *   whose order matters.
 * Synchronises the stream before returning (the group count is needed on the host). */
int bs_group_xmask(const uint64_t* x, const uint64_t* z, const double* coeff_reim, int64_t M,
                   int n_qubits, double eps_drop, int mode, const int64_t* seq_offsets,
                   int64_t n_seq, void* cuda_stream, bs_op_t* out);
int bs_op_info(bs_op_t op, int64_t* n_groups, int64_t* n_terms, int* n_qubits);
/* Host copies of the device tables; any pointer may be NULL.  xg u64[G] group masks; offs
 * i64[G+1] string offsets; z u64[M]; c_reim double[2M] true-Pauli coefficients; w_reim
 * double[2M] target-form weights w_k = c_k (-i)^{ny_k}. */
int bs_op_export(bs_op_t op, uint64_t* xg, int64_t* offs, uint64_t* z, double* c_reim, double* w_reim);
int bs_op_destroy(bs_op_t op);

/* ---- device-side Jordan-Wigner construction (Alg. 1) feeding a1/a2 directly: the raw 4/16-term
 * expansions are generated and reduced on the device.  h [host] double[n_orb^2] symmetric one-body integrals,
 * g [host] double[n_orb^4] two-body integrals in chemist notation (pq|rs), row-major g[p][q][r][s];
 * H = sum h_pq a+_{ps} a_{qs} + 1/2 sum (pq|rs) a+_{ps} a+_{rt} a_{st} a_{qs}, blocked spin ordering (2 n_orb qubits).
 * bs_jw_hubbard: open chain, H = -t sum (a+_{is} a_{i+1,s} + h.c.) + U sum n_{i,alpha} n_{i,beta}.
 * The resulting operator is a BS_MODE_CANONICAL operator (same tables as bs_group_xmask on the raw list). */
int bs_jw_molecular(int n_orb, const double* h, const double* g, double eps_drop, void* cuda_stream, bs_op_t* out);
int bs_jw_hubbard(int n_sites, double t, double U, double eps_drop, void* cuda_stream, bs_op_t* out);

/* ---- a3: sector tables.  n_alpha = n_beta = -1: full 2^n space and
 * n_orb then means n_qubits.  Sector mode needs n_orb <= 32, 0 <= n_alpha, n_beta <= n_orb. */
int bs_sector_build(int n_orb, int n_alpha, int n_beta, void* cuda_stream, bs_sector_t* out);
int bs_sector_info(bs_sector_t s, int64_t* dim, int64_t* dim_alpha, int64_t* dim_beta);
/* alpha_strings [host] u64[dim_alpha], beta_strings [host] u64[dim_beta]: unrank tables. */
int bs_sector_export(bs_sector_t s, uint64_t* alpha_strings, uint64_t* beta_strings);
/* configs [host] u64[n] -> index_out [host] i64[n] (-1 outside the sector); ranks on the device
 * with the same lookup tables the apply kernels use.  Synchronises. */
int bs_sector_rank(bs_sector_t s, const uint64_t* configs, int64_t n, int64_t* index_out);
int bs_sector_destroy(bs_sector_t s);

/* ---- point-group symmetry blocking (Eq. 29-31) for Abelian point groups (D2h and subgroups).
 * orb_irrep [host] int[n_orb]: irrep label 0..7 of every spatial orbital; the irrep of a spin string is the XOR of the
 * labels of its occupied orbitals; the block holds the configurations of `parent` with irrep(t_a) ^ irrep(t_b) =
 * target_irrep (Eq. 30).  Blocked vector layout (Eq. 29): blocks r = 0..7 in order of the alpha irrep; block r pairs
 * the alpha strings of irrep r with the beta strings of irrep r ^ target_irrep, each in increasing numeric order,
 * index = offset_r + rank_alpha^r * D_beta^r + rank_beta^r.  `parent` must outlive the handle.
 * The blocking is a STORAGE layout: bs_sym_apply / bs_sym_expect embed the blocked vector into the sector layout
 * (zero in the other irreps), run bs_apply / bs_expect there and read the block back, using two sector-sized
 * scratch vectors owned by the handle (allocated at the first call).  They return P_block H P_block psi. */
int bs_symsector_build(bs_sector_t parent, const int* orb_irrep, int target_irrep, void* cuda_stream,
                       bs_symsector_t* out);
/* dim: amplitudes of the block; dim_alpha[r], dim_beta[r] [host] int64[8]: strings of irrep r (any pointer may be NULL) */
int bs_symsector_info(bs_symsector_t h, int64_t* dim, int64_t dim_alpha[8], int64_t dim_beta[8]);
int bs_symsector_destroy(bs_symsector_t h);
/* psi_blocked [device] complex128[dim of the block], psi_sector [device] complex128[dim of the parent sector] */
int bs_sym_scatter(bs_symsector_t h, const void* psi_blocked, void* psi_sector, void* cuda_stream);
int bs_sym_gather(bs_symsector_t h, const void* psi_sector, void* psi_blocked, void* cuda_stream);
int bs_sym_apply(bs_op_t op, bs_symsector_t h, const void* psi_in, void* psi_out, void* cuda_stream);
int bs_sym_expect(bs_op_t op, bs_symsector_t h, const void* psi, double result_reim[2], void* cuda_stream);

/* ---- a4: out = P_sector H P_sector psi  (Eq. 27).  psi_in, psi_out [device]
 * complex128[dim], distinct buffers.  The first call for a given (op, sector) pair builds and
 * caches sector-specific device tables (synchronises once); later calls only launch. */
int bs_apply(bs_op_t op, bs_sector_t s, const void* psi_in, void* psi_out, void* cuda_stream);
/* Same, for alpha rows [row_lo, row_hi) only (full-space mode: index range): writes
 * psi_out[row_lo*D_beta .. row_hi*D_beta) and nothing else.  This is the multi-GPU shard unit
 * (targets are independent). */
int bs_apply_rows(bs_op_t op, bs_sector_t s, const void* psi_in, void* psi_out, int64_t row_lo,
                  int64_t row_hi, void* cuda_stream);
/* out = alpha * (H psi_in) + beta * psi_in, and if acc != NULL additionally acc += out, fused into
 * the apply epilogue (the Taylor recurrence of PAPER.md:74-83, Eq. 6-7).  alpha, beta [host]
 * double[2] complex; acc [device] complex128[dim] or NULL. */
int bs_apply_axpby(bs_op_t op, bs_sector_t s, const void* psi_in, void* psi_out,
                   const double alpha_reim[2], const double beta_reim[2], void* acc,
                   void* cuda_stream);

/* ---- a5: <psi|H|psi> (Eq. 5), fused gather + dot, H psi is never stored.
 * result_reim [host] double[2]; deterministic two-stage reduction.  Synchronises the stream. */
int bs_expect(bs_op_t op, bs_sector_t s, const void* psi, double result_reim[2], void* cuda_stream);
/* <a|b> = sum conj(a_i) b_i over dim amplitudes, same deterministic reduction.  Synchronises. */
int bs_vdot(bs_sector_t s, const void* a, const void* b, double result_reim[2], void* cuda_stream);

/* ---- no-allocation variant of bs_vdot, for callers that cannot call cudaMalloc (CUDA graph capture, serving loops):
 * result_dev [device] double[2] <- sum_i conj(a_i) b_i over n amplitudes; a, b [device] complex128[n], 16-byte aligned.
 * The per-block partial sums live in a 128 KiB file-scope __device__ array (every GPU that loads the library holds it
 * until exit) instead of malloc'ed scratch: 8192 partials of 65,536 amplitudes each, so n <= bs_noalloc_max_dim() =
 * 536,870,912; longer vectors return BS_ERR_ARG.  The call allocates nothing, copies nothing to the host and does not
 * synchronise (two launches on cuda_stream).  bs_noalloc_setup takes the array's device address for the CURRENT device,
 * once per device; bs_vdot_noalloc calls it on first use, but under graph capture call it beforehand.  Every call on a
 * device shares the array: calls that overlap on the GPU (other streams, concurrent graph replays) race -- one stream
 * at a time.  Stale contents are harmless: a call reads only the partials it has just written.  Deterministic. */
int bs_noalloc_setup(void);
int64_t bs_noalloc_max_dim(void);
int bs_vdot_noalloc(const void* a, const void* b, int64_t n, void* result_dev, void* cuda_stream);

/* ---- a6: psi <- exp(theta_j A_j) psi for j = 0..n_rot-1 in order, A_j = group j of a
 * BS_MODE_SEQUENCE operator: anti-Hermitian (every c_k purely imaginary), one x, mutually
 * commuting strings (Eq. 39).  x = 0 (diagonal generator, e.g. exp(-i w Z_j Z_{j+1}) of
 * PAPER.md:469-473, Eq. 42) multiplies every amplitude by exp(theta F(t)).  thetas [host] double[n_rot], n_rot must
 * equal the operator's group count.  In place on disjoint pairs {t, t^x}.  Returns
 * BS_ERR_NOT_COMMUTING / BS_ERR_LEAVES_SECTOR instead of applying a non-unitary map.
 * The first call for a (generators, sector) pair runs a read-only leak check and synchronises; later
 * calls only enqueue n_rot launches. */
int bs_apply_pauli_rotations(bs_op_t generators, bs_sector_t s, const double* thetas,
                             int64_t n_rot, void* psi_inout, void* cuda_stream);

/* ---- a7: one step psi <- e^{-i E_s dt} sum_{k<=order} (-i dt)^k/k! (H - E_s)^k psi
 * (Eq. 6-7; reading U9).  work [device] complex128[2*dim] scratch. */
int bs_taylor_step(bs_op_t op, bs_sector_t s, void* psi_inout, void* work, double dt, int order,
                   double e_shift, void* cuda_stream);

/* Machine-readable facts about the cached (op, sector) plan (built if needed); info [host] int64[8]:
 *   [0] kernel path: 0 full space, 1 sector v1 (fallback), 2 row kernel v2, 3 v2 + light (few-group operators)
 *   [1] 1 if a v2 row plan could NOT be built (allocation failure or a size limit) and the much slower v1 kernel runs
 *   [2] 1 if beta-only groups run on the transposed problem   [3] 1 if alpha-beta groups run K-resolved
 *   [4] bytes of state-vector-sized library scratch this pair can allocate (0, or 3 x 16 x dim)
 *   [5] bytes of the K-resolution scratch (allocated at plan build)
 *   [6] largest number of V slots (keys = distinct beta Z masks) under one alpha mask   [7] plan groups in total */
int bs_plan_info(bs_op_t op, bs_sector_t s, int64_t info[8], void* cuda_stream);
/* The groups of the plan after the spin split (Eq. 28) and the exact phase factorisation
 * (Eq. 32-37): for group g, x[g] = its X mask (alpha bits | beta bits << n_orb) and nkeys[g] = the
 * number of distinct beta Z masks of its strings, i.e. the number of terms of F_g(t_a, t_b) = sum_j V_gj(t_a)
 * (-1)^{popc(zb_gj & t_b)} -- the exact counterpart of the paper's factorisation rank R_g (Table 1).
 * x, nkeys [host] arrays of capacity cap (may be NULL to query); *n_groups receives the group count.  Sector mode with
 * a v2 plan only (else BS_ERR_ARG). */
int bs_plan_groups(bs_op_t op, bs_sector_t s, uint64_t* x, int32_t* nkeys, int64_t cap, int64_t* n_groups,
                   void* cuda_stream);
/* Human-readable description of the cached (op, sector) plan (kernel path, table sizes, launch
 * geometry) written to buf [host] (at most n bytes, NUL terminated); builds the plan if needed. */
int bs_plan_describe(bs_op_t op, bs_sector_t s, char* buf, int64_t n, void* cuda_stream);

/* number of kernels this library has launched in this process (for bench.py's gpu_launches) */
int64_t bs_launch_count(void);
const char* bs_last_error(void);
const char* bs_version(void);

#ifdef __cplusplus
}
#endif
#endif /* BS_H_ */
