// a6 grouped Pauli rotations (section 2.5; Eq. 39).
//
// Generator A = sum_k c_k P_k, all strings sharing one x and mutually commuting, A^dag = -A (x = 0: k_rot_diag).
// With F(t) = sum_k w_k (-1)^{popc(z_k & t)} = <t|A|t^x> (target form, w_k = c_k (-i)^{ny_k}) the
// operator is block diagonal on the pairs {t, u = t^x}: A|u> = F(t)|t>, A|t> = F(u)|u>,
// F(u) = -conj F(t), A^2 = -|F|^2 on the pair, hence
//   exp(theta A) = cos(theta r) + A sin(theta r)/r,  r = |F(t)|,
//   psi'[t] = cos(theta r) psi[t] + sin(theta r)/r F(t) psi[u],
//   psi'[u] = cos(theta r) psi[u] - sin(theta r)/r conj(F(t)) psi[t].
// Routing (pairing) and phase accumulation are computed once per pair and group.
// The pair is owned by the thread of its smaller index, so the update is in place and race free.
#include <cooperative_groups.h>
#include <algorithm>

#include "bs_internal.cuh"

namespace {

__device__ __forceinline__ double flipd(double v, u32 par) {
    return __hiloint2double(__double2hiint(v) ^ (int)(par << 31), __double2loint(v));
}

__device__ __forceinline__ double2 phase_sum(const u64* __restrict__ z, const double2* __restrict__ w, int k0, int k1,
                                             u64 t) {
    double fr = 0.0, fi = 0.0;
    for (int k = k0; k < k1; ++k) {
        const u32 par = (u32)__popcll(__ldg(z + k) & t) & 1u;
        const double2 wk = __ldg(w + k);
        fr += flipd(wk.x, par);
        fi += flipd(wk.y, par);
    }
    return make_double2(fr, fi);
}

// sc1 = (sin theta, cos theta) precomputed on the host for the common case |F| = 1 (fermionic excitation
// generators: |f| is 0 or 1); other moduli take the sincos path.
__device__ __forceinline__ void rotate_pair(double2* __restrict__ psi, i64 it, i64 iu, double2 F, double theta,
                                            double2 sc1) {
    const double r2 = F.x * F.x + F.y * F.y;
    if (r2 == 0.0) return;
    double sn, cs;
    if (r2 == 1.0) {
        sn = sc1.x;
        cs = sc1.y;
    } else {
        const double r = hypot(F.x, F.y);
        sincos(theta * r, &sn, &cs);
        sn /= r;
    }
    const double2 a = psi[it], b = psi[iu];
    // psi'[t] = cs a + sn F b ; psi'[u] = cs b - sn conj(F) a
    psi[it] = make_double2(cs * a.x + sn * (F.x * b.x - F.y * b.y), cs * a.y + sn * (F.x * b.y + F.y * b.x));
    psi[iu] = make_double2(cs * b.x - sn * (F.x * a.x + F.y * a.y), cs * b.y - sn * (F.x * a.y - F.y * a.x));
}

__global__ void __launch_bounds__(256)
k_rot_sector(SpinTab A, SpinTab B, int n_orb, u64 x, const u64* __restrict__ z, const double2* __restrict__ w, int k0,
             int k1, double theta, double2 sc1, double2* __restrict__ psi) {
    // grid: x = column blocks, y = alpha rows (no 64-bit division); the alpha test is uniform per block
    const u32 row = blockIdx.y, col = blockIdx.x * blockDim.x + threadIdx.x;
    const u32 xa = (u32)(x & ((u64(1) << n_orb) - 1)), xb = (u32)(x >> n_orb);
    const u32 ta = A.str[row];
    if (2 * __popc(ta & xa) != __popc(xa)) return;  // partner outside the sector: F = 0 there (leak check)
    if (col >= B.D) return;
    const u32 tb = B.str[col];
    if (2 * __popc(tb & xb) != __popc(xb)) return;
    const u32 urow = xa ? spin_rank(A, ta ^ xa) : row;
    if (urow < row) return;  // the pair belongs to its smaller index (x != 0, so iu != i)
    const u32 ucol = xb ? spin_rank(B, tb ^ xb) : col;
    if (urow == row && ucol < col) return;
    const i64 i = (i64)row * B.D + col, iu = (i64)urow * B.D + ucol;
    rotate_pair(psi, i, iu, phase_sum(z, w, k0, k1, (u64)ta | ((u64)tb << n_orb)), theta, sc1);
}

// Row-list variant: the alpha side (validity, partner row, ownership) is precomputed per (generator, sector)
// on the host, so the grid holds only rows that own pairs and the kernel's dependent chain is
// beta string -> partner column -> amplitudes.
__global__ void __launch_bounds__(256)
k_rot_rows(SpinTab A, SpinTab B, int n_orb, u64 x, const uint2* __restrict__ pairs, const u64* __restrict__ z,
           const double2* __restrict__ w, int k0, int k1, double theta, double2 sc1, double2* __restrict__ psi) {
    const uint2 pr = __ldg(pairs + blockIdx.y);
    const u32 row = pr.x, urow = pr.y, col = blockIdx.x * blockDim.x + threadIdx.x;
    if (col >= B.D) return;
    const u32 xb = (u32)(x >> n_orb);
    const u32 ta = A.str[row], tb = B.str[col];
    if (2 * __popc(tb & xb) != __popc(xb)) return;
    const u32 ucol = xb ? spin_rank(B, tb ^ xb) : col;
    if (urow == row && ucol < col) return;  // x_a = 0: the pair belongs to its smaller column
    rotate_pair(psi, (i64)row * B.D + col, (i64)urow * B.D + ucol, phase_sum(z, w, k0, k1, (u64)ta | ((u64)tb << n_orb)),
                theta, sc1);
}

// Pair-list variant (the per-generator path at sector sizes whose cells do not fit shared memory, configs 4-5): both
// sides are precomputed per (generator, sector) -- owner (row, partner row) pairs and valid (column, partner column)
// pairs -- so every thread rotates one pair: no validity test, no rank lookup, no idle lanes; the strings are the
// z-reduced ones (see reduce_generators), typically 2 instead of 8 for a double excitation.
__global__ void __launch_bounds__(256)
k_rot_pairs(SpinTab A, SpinTab B, int n_orb, const uint2* __restrict__ rpairs, const uint2* __restrict__ cpairs, i64 n_cp,
            const u64* __restrict__ z, const double2* __restrict__ w, int k0, int k1, double theta, double2 sc1,
            double2* __restrict__ psi) {
    const i64 p = blockIdx.x * (i64)blockDim.x + threadIdx.x;
    if (p >= n_cp) return;
    const uint2 rp = __ldg(rpairs + blockIdx.y), cp = __ldg(cpairs + p);
    const u64 t = (u64)A.str[rp.x] | ((u64)B.str[cp.x] << n_orb);
    rotate_pair(psi, (i64)rp.x * B.D + cp.x, (i64)rp.y * B.D + cp.y, phase_sum(z, w, k0, k1, t), theta, sc1);
}

// Diagonal generator (x = 0, e.g. exp(-i w Z_j Z_{j+1}) of the layered TFIM ansatz, Eq. 42):
// A|t> = F(t)|t> with F purely imaginary for an anti-Hermitian A, so psi[t] *= exp(theta F(t)).
__global__ void __launch_bounds__(256)
k_rot_diag(SpinTab A, SpinTab B, int n_orb, int full, i64 D, const u64* __restrict__ z, const double2* __restrict__ w,
           int k0, int k1, double theta, double2* __restrict__ psi) {
    const i64 i = blockIdx.x * (i64)blockDim.x + threadIdx.x;
    if (i >= D) return;
    u64 t = (u64)i;
    if (!full) {
        const i64 row = i / B.D;
        t = (u64)A.str[row] | ((u64)B.str[i - row * B.D] << n_orb);
    }
    const double2 F = phase_sum(z, w, k0, k1, t);
    double sn, cs;
    sincos(theta * F.y, &sn, &cs);
    const double m = exp(theta * F.x);  // 1 for an anti-Hermitian generator
    const double2 a = psi[i];
    psi[i] = make_double2(m * (cs * a.x - sn * a.y), m * (cs * a.y + sn * a.x));
}

// ---- closed-cell batching -------------------------------------------------------------------------------
// A run of consecutive generators can share ONE launch when the index space splits into cells that are closed
// under every pairing t <-> t ^ x_j of the run and fit in shared memory; inside a cell the rotations are applied
// one after the other with __syncthreads() in between, outside they are independent:
//   * all x_a equal (0 or not): cell = the row (x_a = 0) or the row pair {row, partner row}   (k_rot_cell_rows)
//   * all x_b = 0:              cell = a few columns, all rows                                 (k_rot_cell_cols)
// With the generator order of DESIGN.md reading U10 the 1,818 UCCSD rotations of config 2 become 40 launches.
__device__ __forceinline__ void rotate_smem(double2& pa, double2& pb, double2 F, double theta, double2 sc1) {
    const double r2 = F.x * F.x + F.y * F.y;
    if (r2 == 0.0) return;
    double sn = sc1.x, cs = sc1.y;
    if (r2 != 1.0) {
        const double r = hypot(F.x, F.y);
        sincos(theta * r, &sn, &cs);
        sn /= r;
    }
    const double2 a = pa, b = pb;
    pa = make_double2(cs * a.x + sn * (F.x * b.x - F.y * b.y), cs * a.y + sn * (F.x * b.y + F.y * b.x));
    pb = make_double2(cs * b.x - sn * (F.x * a.x + F.y * a.y), cs * b.y - sn * (F.x * a.y - F.y * a.x));
}

// Generator data of a chunk of the run, staged in shared memory by the whole block in one pass (all loads in
// flight together) so that the serial generator loop never waits on global memory for its headers or strings.
constexpr int kGenChunk = 32;   // generators per chunk
constexpr int kStrChunk = 256;  // strings per chunk (a chunk ends early when they would not fit)
struct GenChunk {
    u64 z[kStrChunk];
    double2 w[kStrChunk];
    double2 sc[kGenChunk];
    double th[kGenChunk];
    u64 x[kGenChunk];
    int k0[kGenChunk + 1];  // string offsets relative to the chunk
    i64 p0[kGenChunk + 1];  // bounds of every generator's pair list (coff / roff): staged with the headers, so that a
                            // generator's loop does not start with a dependent global look-up
    int n;                  // generators in the chunk
};

// loads generators [j, ...) into G; every thread returns the same chunk length
__device__ __forceinline__ int load_chunk(GenChunk& G, i64 j, i64 j1, const u64* __restrict__ xg,
                                          const i64* __restrict__ offs, const u64* __restrict__ z,
                                          const double2* __restrict__ w, const double* __restrict__ thetas,
                                          const double2* __restrict__ sc, const i64* __restrict__ pair_off) {
    const i64 base = offs[j];
    int n = (int)min((i64)kGenChunk, j1 - j);
    while (n > 1 && offs[j + n] - base > kStrChunk) --n;  // uniform
    const int ns = (int)min((i64)kStrChunk, offs[j + n] - base);
    for (int i = threadIdx.x; i < n; i += blockDim.x) {
        G.x[i] = xg[j + i];
        G.th[i] = thetas[j + i];
        G.sc[i] = sc[j + i];
    }
    for (int i = threadIdx.x; i <= n; i += blockDim.x) {
        G.k0[i] = (int)(offs[j + i] - base);
        G.p0[i] = pair_off[j + i];
    }
    for (int i = threadIdx.x; i < ns; i += blockDim.x) {
        G.z[i] = z[base + i];
        G.w[i] = w[base + i];
    }
    if (threadIdx.x == 0) G.n = n;
    return n;
}

__device__ __forceinline__ double2 phase_sum_s(const GenChunk& G, int k0, int k1, u64 t) {
    double fr = 0.0, fi = 0.0;
    for (int k = k0; k < k1; ++k) {
        const u32 par = (u32)__popcll(G.z[k] & t) & 1u;
        fr += flipd(G.w[k].x, par);
        fi += flipd(G.w[k].y, par);
    }
    return make_double2(fr, fi);
}

// beta-only phase sum: the alpha half of every sign was folded into G.w for this block's row (see fold below)
__device__ __forceinline__ double2 phase_sum_b(const GenChunk& G, int k0, int k1, u32 tb) {
    double fr = 0.0, fi = 0.0;
    for (int k = k0; k < k1; ++k) {
        const u32 par = (u32)__popc((u32)G.z[k] & tb) & 1u;
        fr += flipd(G.w[k].x, par);
        fi += flipd(G.w[k].y, par);
    }
    return make_double2(fr, fi);
}

// cells = rows (R = 1, x_a = 0) or row pairs (R = 2, common x_a != 0); generators [j0, j1)
// GLOBAL: the cell does not fit shared memory (D_beta > 5,937: configs 4-5): the block works on its rows in place.
// One launch still covers the whole run, the rows of the ~300 blocks in flight (0.4 - 0.7 MB each) stay in the 126 MB
// L2 across the run's generators, so HBM sees each row once per run instead of once per generator.
template <int R, bool GLOBAL>
__global__ void __launch_bounds__(R == 2 ? 512 : 256)
k_rot_cell_rows(SpinTab A, SpinTab B, int n_orb, const uint2* __restrict__ pairs, const u64* __restrict__ xg,
                const i64* __restrict__ offs, const u64* __restrict__ z, const double2* __restrict__ w,
                const double* __restrict__ thetas, const double2* __restrict__ sc, const uint2* __restrict__ cpairs,
                const u32* __restrict__ cstr, const i64* __restrict__ coff, i64 j0, i64 j1, double2* __restrict__ psi) {
    extern __shared__ __align__(16) unsigned char smem_cell[];
    __shared__ GenChunk G;
    const u32 Db = (u32)B.D;
    u32 row0, row1;
    if (R == 2) {
        const uint2 pr = pairs[blockIdx.x];
        row0 = pr.x;
        row1 = pr.y;
    } else row0 = row1 = blockIdx.x;
    double2* s0 = GLOBAL ? psi + (i64)row0 * Db : reinterpret_cast<double2*>(smem_cell);
    double2* s1 = GLOBAL ? psi + (i64)row1 * Db : ((R == 2) ? s0 + Db : s0);
    if (!GLOBAL)
        for (u32 c = threadIdx.x; c < Db; c += blockDim.x) {
            s0[c] = psi[(i64)row0 * Db + c];
            if (R == 2) s1[c] = psi[(i64)row1 * Db + c];
        }
    const u32 ta = A.str[row0];
    for (i64 j = j0; j < j1;) {
        __syncthreads();  // previous chunk fully consumed (and the rows are loaded)
        const int n = load_chunk(G, j, j1, xg, offs, z, w, thetas, sc, coff);
        __syncthreads();
        // fold the alpha half of every sign into the weights (t_a is fixed for the block): the per-column phase
        // sum is then one 32-bit AND + POPC per string
        for (int i = threadIdx.x; i < min(G.k0[n], kStrChunk); i += blockDim.x) {
            const u64 zz = G.z[i];
            const u32 par = (u32)__popc((u32)(zz & ((u64(1) << n_orb) - 1)) & ta) & 1u;
            G.w[i] = make_double2(flipd(G.w[i].x, par), flipd(G.w[i].y, par));
            G.z[i] = zz >> n_orb;
        }
        __syncthreads();
        for (int g = 0; g < n; ++g) {
            // the valid (column, partner column) pairs of the generator's beta mask were listed at plan time (they do
            // not depend on the row): no validity test, no rank lookup, no idle lanes
            const int k0 = G.k0[g], k1 = min(G.k0[g + 1], kStrChunk);
            const i64 p0 = G.p0[g], p1 = G.p0[g + 1];
            // In place (amplitudes through L2) the list entries of this thread's next four pairs are fetched together: they
            // do not depend on the amplitudes, whose read-modify-writes stay one after the other (q32 1,288 -> 1,175 ms).
            // With the cell in shared memory a generator has fewer pairs than the block has threads and the unrolled
            // form only adds work (q24 2.23 -> 2.96 ms): depth 1 there, i.e. the plain loop.
            constexpr int kRotU = GLOBAL ? 4 : 1;
            for (i64 pb = p0 + threadIdx.x; pb < p1; pb += (i64)kRotU * blockDim.x) {
                uint2 cp[kRotU];
                u32 tb[kRotU];
                bool ok[kRotU];
#pragma unroll
                for (int u = 0; u < kRotU; ++u) {
                    const i64 p = pb + (i64)u * blockDim.x;
                    ok[u] = p < p1;
                    cp[u] = ok[u] ? __ldg(cpairs + p) : make_uint2(0u, 0u);
                    tb[u] = (ok[u] && cstr) ? __ldg(cstr + p) : 0u;   // the list copy: no dependent look-up
                }
#pragma unroll
                for (int u = 0; u < kRotU; ++u)
                    if (ok[u]) {
                        const u32 t = cstr ? tb[u] : B.str[cp[u].x];
                        rotate_smem(s0[cp[u].x], s1[cp[u].y], phase_sum_b(G, k0, k1, t), G.th[g], G.sc[g]);
                    }
            }
            __syncthreads();
        }
        j += n;
    }
    if (!GLOBAL)
        for (u32 c = threadIdx.x; c < Db; c += blockDim.x) {
            psi[(i64)row0 * Db + c] = s0[c];
            if (R == 2) psi[(i64)row1 * Db + c] = s1[c];
        }
}

// Row-pair cells whose two rows do not fit ONE block's shared memory (D_beta = 12,870 at configs[3]: 2 x 206 KB) but
// whose single row does: a thread-block cluster of two, one row per block, the partner amplitude of every pair reached
// through distributed shared memory (a generic pointer from map_shared_rank).  Same run, same pair lists and the same
// arithmetic per pair as k_rot_cell_rows<2, false>; the pair list is split over the 2 x 512 threads of the cluster and the
// barrier between generators is the cluster's.  Replaces the in-place (L2) form there, which moves 64 bytes per pair
// through L2 for every generator.
__global__ void __cluster_dims__(2, 1, 1) __launch_bounds__(512)
k_rot_cluster_rows(SpinTab A, SpinTab B, int n_orb, const uint2* __restrict__ pairs, const u64* __restrict__ xg,
                   const i64* __restrict__ offs, const u64* __restrict__ z, const double2* __restrict__ w,
                   const double* __restrict__ thetas, const double2* __restrict__ sc, const uint2* __restrict__ cpairs,
                   const u32* __restrict__ cstr, const i64* __restrict__ coff, i64 j0, i64 j1, double2* __restrict__ psi) {
    namespace cg = cooperative_groups;
    extern __shared__ __align__(16) unsigned char smem_cell[];
    __shared__ GenChunk G;
    cg::cluster_group cluster = cg::this_cluster();
    const unsigned rank = cluster.block_rank();            // 0 holds row0, 1 holds row1
    const u32 Db = (u32)B.D;
    const uint2 pr = pairs[blockIdx.x >> 1];
    const u32 my_row = rank ? pr.y : pr.x;
    double2* mine = reinterpret_cast<double2*>(smem_cell);
    for (u32 c = threadIdx.x; c < Db; c += blockDim.x) mine[c] = psi[(i64)my_row * Db + c];
    double2* s0 = rank == 0 ? mine : cluster.map_shared_rank(mine, 0);
    double2* s1 = rank == 1 ? mine : cluster.map_shared_rank(mine, 1);
    const u32 ta = A.str[pr.x];
    const u32 tid2 = rank * blockDim.x + threadIdx.x, stride2 = 2 * blockDim.x;
    cluster.sync();   // both rows are in shared memory before anyone reaches across
    for (i64 j = j0; j < j1;) {
        __syncthreads();  // this block's previous chunk fully consumed (G is per block)
        const int n = load_chunk(G, j, j1, xg, offs, z, w, thetas, sc, coff);
        __syncthreads();
        for (int i = threadIdx.x; i < min(G.k0[n], kStrChunk); i += blockDim.x) {
            const u64 zz = G.z[i];
            const u32 par = (u32)__popc((u32)(zz & ((u64(1) << n_orb) - 1)) & ta) & 1u;
            G.w[i] = make_double2(flipd(G.w[i].x, par), flipd(G.w[i].y, par));
            G.z[i] = zz >> n_orb;
        }
        __syncthreads();
        for (int g = 0; g < n; ++g) {
            const int k0 = G.k0[g], k1 = min(G.k0[g + 1], kStrChunk);
            const i64 p0 = G.p0[g], p1 = G.p0[g + 1];
            for (i64 p = p0 + tid2; p < p1; p += stride2) {
                const uint2 cp = __ldg(cpairs + p);
                const u32 tb = cstr ? __ldg(cstr + p) : B.str[cp.x];
                rotate_smem(s0[cp.x], s1[cp.y], phase_sum_b(G, k0, k1, tb), G.th[g], G.sc[g]);
            }
            cluster.sync();   // the next generator may pair these amplitudes with others, from either block
        }
        j += n;
    }
    // the last cluster.sync() above ordered every remote write before this read of the block's own row
    for (u32 c = threadIdx.x; c < Db; c += blockDim.x) psi[(i64)my_row * Db + c] = mine[c];
}

// cells = CC consecutive columns x all rows (x_b = 0 for every generator of the run); GLOBAL as above (in place, L2)
template <int CC, bool GLOBAL>
__global__ void __launch_bounds__(1024)
k_rot_cell_cols(SpinTab A, SpinTab B, int n_orb, const u64* __restrict__ xg, const i64* __restrict__ offs,
                const u64* __restrict__ z, const double2* __restrict__ w, const double* __restrict__ thetas,
                const double2* __restrict__ sc, const uint2* __restrict__ rpairs, const i64* __restrict__ roff, i64 j0,
                i64 j1, double2* __restrict__ psi) {
    extern __shared__ __align__(16) unsigned char smem_cell[];
    __shared__ GenChunk G;
    const u32 Da = (u32)A.D, Db = (u32)B.D;
    const u32 c0 = blockIdx.x * CC;
    const u32 ncol = min((u32)CC, Db - c0);
    // cell element (row r, column c0 + c): shared memory [Da][CC], or the state vector itself
    double2* sm = GLOBAL ? psi + c0 : reinterpret_cast<double2*>(smem_cell);
    const i64 rs = GLOBAL ? (i64)Db : (i64)CC;   // row stride of the cell
    if (!GLOBAL)
        for (u32 i = threadIdx.x; i < Da * CC; i += blockDim.x) {
            const u32 r = i / CC, c = i - r * CC;
            if (c < ncol) sm[i] = psi[(i64)r * Db + c0 + c];
        }
    for (i64 j = j0; j < j1;) {
        __syncthreads();
        const int n = load_chunk(G, j, j1, xg, offs, z, w, thetas, sc, roff);
        __syncthreads();
        for (int g = 0; g < n; ++g) {
            // owner (row, partner row) pairs of the generator were listed at plan time: one work item per (pair, column)
            const int k0 = G.k0[g], k1 = min(G.k0[g + 1], kStrChunk);
            const i64 p0 = G.p0[g];
            const u32 np = (u32)(G.p0[g + 1] - p0);
            for (u32 i = threadIdx.x; i < np * CC; i += blockDim.x) {
                const u32 q = i / CC, c = i - q * CC;
                if (c >= ncol) continue;
                const uint2 rp = __ldg(rpairs + p0 + q);
                const u32 ta = A.str[rp.x], tb = B.str[c0 + c];
                rotate_smem(sm[rp.x * rs + c], sm[rp.y * rs + c], phase_sum_s(G, k0, k1, (u64)ta | ((u64)tb << n_orb)),
                            G.th[g], G.sc[g]);
            }
            __syncthreads();
        }
        j += n;
    }
    if (!GLOBAL)
        for (u32 i = threadIdx.x; i < Da * CC; i += blockDim.x) {
            const u32 r = i / CC, c = i - r * CC;
            if (c < ncol) psi[(i64)r * Db + c0 + c] = sm[i];
        }
}

// ---- orbit cells: closed cells that stay small at any sector size -------------------------------------------------
// A SUB-RUN of consecutive generators with a common alpha mask whose beta masks together touch the orbital set U
// (|U| <= kOrbitUmax) only moves electrons inside U: the columns with one fixed occupation OUTSIDE U form an orbit of at most
// C(|U|, |U|/2) columns, closed under every pairing of the sub-run.  One warp owns one orbit of one row (x_a = 0) or
// row pair: it loads the orbit's amplitudes into its slice of shared memory, applies ALL generators of the sub-run
// (__syncwarp between them, no block barrier) and writes them back: one trip through L2 / HBM per sub-run instead
// of one per generator.  UCCSD order (reading U10): the alpha-beta doubles of one (i, a) come as j outer, b inner, so
// a sub-run collects all b of two beta occupied orbitals j (|U| = 10 at configs[3]: 16 generators per load).
// OPT-IN (BS_ROT_ORBIT=1): at configs[3] it is slower than the in-place cells -- every sub-run touches every amplitude of
// the valid rows with scattered 16-byte accesses, the in-place kernel only the 28 % that a generator rotates.
constexpr int kOrbitUmax = 10;
constexpr int kOrbitMax = 252;   // C(10, 5) columns

struct OrbitTab {
    const u32* pat;            // [n_pat] sub-masks of U at their real bit positions, grouped by popcount m, ascending
    const u32* outs;           // [n_out] occupations outside U that leave 0 <= m <= |U| electrons for U
    const unsigned short* pairs;     // per (generator, m) the valid owner pairs, compacted: i | q << 8, i and q = positions of
                                     // p and p ^ x_b within the m block (< 252)
    const int* pair_off;             // [n_gen][12]: pairs of (generator, m) are [pair_off[g][m], pair_off[g][m + 1])
    int pat_off[kOrbitUmax + 2];     // m block [pat_off[m], pat_off[m + 1])
    int n_pat, n_out, Nb;
};

template <int R>
__global__ void __launch_bounds__(256)
k_rot_orbit(SpinTab A, SpinTab B, int n_orb, const uint2* __restrict__ pairs, OrbitTab T, const i64* __restrict__ offs,
            const u64* __restrict__ z, const double2* __restrict__ w, const double* __restrict__ thetas,
            const double2* __restrict__ sc, i64 j0, i64 j1, double2* __restrict__ psi) {
    extern __shared__ __align__(16) unsigned char smem_cell[];
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    double2* s0 = reinterpret_cast<double2*>(smem_cell) + (size_t)warp * (R * kOrbitMax);
    double2* s1 = (R == 2) ? s0 + kOrbitMax : s0;
    u32* scol = reinterpret_cast<u32*>(smem_cell + (size_t)8 * R * kOrbitMax * 16) + warp * (2 * kOrbitMax);
    u32* spat = scol + kOrbitMax;   // the orbit's beta strings o | p
    u32 row0, row1;
    if (R == 2) {
        const uint2 pr = pairs[blockIdx.y];
        row0 = pr.x;
        row1 = pr.y;
    } else row0 = row1 = blockIdx.y;
    const u64 ta = A.str[row0];
    const i64 Db = B.D;
    double2* __restrict__ p0 = psi + (i64)row0 * Db;
    double2* __restrict__ p1 = psi + (i64)row1 * Db;
    for (int oi = blockIdx.x * 8 + warp; oi < T.n_out; oi += gridDim.x * 8) {
        const u32 o = __ldg(T.outs + oi);
        const int m = T.Nb - __popc(o);
        const int pb = T.pat_off[m], np = T.pat_off[m + 1] - pb;
        if (np < (R == 2 ? 1 : 2)) continue;   // warp-uniform (one column: only a row pair can still rotate, x_b = 0)
        for (int i = lane; i < np; i += 32) {
            const u32 tb = o | __ldg(T.pat + pb + i);
            const u32 col = spin_rank(B, tb);
            scol[i] = col;
            spat[i] = tb;
            s0[i] = p0[col];
            if (R == 2) s1[i] = p1[col];
        }
        __syncwarp();
        for (i64 g = j0; g < j1; ++g) {
            const int* __restrict__ po = T.pair_off + (size_t)(g - j0) * 12 + m;
            const int q0 = __ldg(po), q1 = __ldg(po + 1);
            if (q0 == q1) continue;   // warp-uniform: the generator pairs nothing in this occupation class
            const int k0 = (int)__ldg(offs + g), k1 = (int)__ldg(offs + g + 1);
            const double th = __ldg(thetas + g);
            const double2 sc1 = __ldg(sc + g);
            for (int idx = q0 + lane; idx < q1; idx += 32) {
                const u32 pq = __ldg(T.pairs + idx);
                const u32 i = pq & 255u, q = pq >> 8;
                rotate_smem(s0[i], s1[q], phase_sum(z, w, k0, k1, ta | ((u64)spat[i] << n_orb)), th, sc1);
            }
            __syncwarp();
        }
        for (int i = lane; i < np; i += 32) {
            const u32 col = scol[i];
            p0[col] = s0[i];
            if (R == 2) p1[col] = s1[i];
        }
        __syncwarp();
    }
}

// One-off validation of a generator list against a sector: for every generator (blockIdx.y) and
// every sector configuration t whose partner t^x lies outside the sector, F(t) must vanish;
// otherwise exp(theta A) would leak out of the sector and its restriction would not be unitary.
__global__ void __launch_bounds__(256)
k_rot_leak_check(SpinTab A, SpinTab B, int n_orb, const u64* __restrict__ xg, const i64* __restrict__ offs,
                 const u64* __restrict__ z, const double2* __restrict__ w, i64 gen_lo, int* __restrict__ leak_flag) {
    const i64 i = blockIdx.x * (i64)blockDim.x + threadIdx.x;
    if (i >= A.D * B.D) return;
    const i64 j = gen_lo + blockIdx.y;
    const u64 x = xg[j];
    const u32 row = (u32)(i / B.D), col = (u32)(i - (i64)row * B.D);
    const u32 ta = A.str[row], tb = B.str[col];
    const u32 xa = (u32)(x & ((u64(1) << n_orb) - 1)), xb = (u32)(x >> n_orb);
    if ((2 * __popc(ta & xa) == __popc(xa)) && (2 * __popc(tb & xb) == __popc(xb))) return;
    const double2 F = phase_sum(z, w, (int)offs[j], (int)offs[j + 1], (u64)ta | ((u64)tb << n_orb));
    if (hypot(F.x, F.y) > 1e-12) atomicExch(leak_flag, 1);
}

__global__ void __launch_bounds__(256)
k_rot_full(i64 D, u64 x, const u64* __restrict__ z, const double2* __restrict__ w, int k0, int k1, double theta,
           double2 sc1, double2* __restrict__ psi) {
    const i64 i = blockIdx.x * (i64)blockDim.x + threadIdx.x;
    if (i >= D) return;
    const i64 iu = i ^ (i64)x;
    if (iu < i) return;
    rotate_pair(psi, i, iu, phase_sum(z, w, k0, k1, (u64)i), theta, sc1);
}

}  // namespace

extern "C" int bs_apply_pauli_rotations(bs_op_t gen, bs_sector_t s, const double* thetas, int64_t n_rot,
                                        void* psi_inout, void* cuda_stream) {
    BS_REQUIRE(gen && s, BS_ERR_ARG, "bs_apply_pauli_rotations: NULL handle");
    BS_REQUIRE(gen->mode == BS_MODE_SEQUENCE, BS_ERR_ARG,
               "bs_apply_pauli_rotations: generators must be grouped with BS_MODE_SEQUENCE");
    BS_REQUIRE(gen->n_qubits == s->n_qubits, BS_ERR_MISMATCH, "generators have %d qubits, sector has %d", gen->n_qubits,
               s->n_qubits);
    BS_REQUIRE(n_rot == gen->G, BS_ERR_ARG, "bs_apply_pauli_rotations: n_rot (%lld) != generator count (%lld)",
               (long long)n_rot, (long long)gen->G);
    BS_REQUIRE(n_rot == 0 || thetas, BS_ERR_ARG, "bs_apply_pauli_rotations: thetas is NULL");
    BS_REQUIRE(psi_inout && (reinterpret_cast<uintptr_t>(psi_inout) & 15u) == 0, BS_ERR_ARG,
               "psi is NULL or not 16-byte aligned");
    // validation: anti-Hermitian (c purely imaginary), mutually commuting (equal ny parity)
    for (i64 j = 0; j < gen->G; ++j) {
        const u64 x = gen->h_xg[j];
        int par0 = -1;
        for (i64 k = gen->h_offs[j]; k < gen->h_offs[j + 1]; ++k) {
            const double re = gen->h_c[2 * k], im = gen->h_c[2 * k + 1];
            BS_REQUIRE(fabs(re) <= 1e-14 * fabs(im) || (re == 0.0), BS_ERR_ARG,
                       "generator %lld is not anti-Hermitian (coefficient %lld has a real part)", (long long)j,
                       (long long)k);
            const int par = __builtin_popcountll(x & gen->h_z[k]) & 1;
            if (par0 < 0) par0 = par;
            BS_REQUIRE(par == par0, BS_ERR_NOT_COMMUTING, "generator %lld: strings do not mutually commute",
                       (long long)j);
        }
    }
    cudaStream_t st = (cudaStream_t)cuda_stream;
    double2* psi = (double2*)psi_inout;
    const unsigned nb = (unsigned)((s->D + 255) / 256);
    if (!s->full && std::find(gen->validated_sectors.begin(), gen->validated_sectors.end(), s->id) ==
                        gen->validated_sectors.end()) {
        BS_CUDA(cudaMemsetAsync(s->d_flag.p, 0, 4, st));
        for (i64 j = 0; j < n_rot; j += 32768) {
            dim3 grid(nb, (unsigned)std::min<i64>(32768, n_rot - j));
            k_rot_leak_check<<<grid, 256, 0, st>>>(s->ta, s->tb, s->n_orb, gen->d_xg.p, gen->d_offs.p, gen->d_z.p,
                                                   gen->d_w.p, j, s->d_flag.p);
            BS_COUNT_LAUNCH(1);
        }
        int leak = 0;
        BS_CUDA(cudaMemcpyAsync(&leak, s->d_flag.p, 4, cudaMemcpyDeviceToHost, st));
        BS_CUDA(cudaStreamSynchronize(st));
        BS_REQUIRE(!leak, BS_ERR_LEAVES_SECTOR, "a generator maps the sector outside itself");
        gen->validated_sectors.push_back(s->id);
    }
    // owner-row lists of this (generators, sector) pair, built once on the host
    bs_op::RotRows* RR = nullptr;
    if (!s->full && (double)n_rot * (double)s->Da <= 5e8) {
        auto it = gen->rot_rows.find(s->id);
        if (it == gen->rot_rows.end()) {
            RR = new (std::nothrow) bs_op::RotRows;
            BS_REQUIRE(RR, BS_ERR_ALLOC, "bs_apply_pauli_rotations: host allocation failed");
            std::vector<uint2> pairs;
            RR->off.assign(n_rot + 1, 0);
            const u64 mask_a = (u64(1) << s->n_orb) - 1;
            for (i64 j = 0; j < n_rot; ++j) {
                const u64 xa = gen->h_xg[j] & mask_a;
                const int pxa = __builtin_popcountll(xa);
                for (i64 r = 0; r < s->Da; ++r) {
                    const u64 ta = s->h_sa[r];
                    if (2 * __builtin_popcountll(ta & xa) != pxa) continue;
                    const i64 ur = xa ? (i64)(std::lower_bound(s->h_sa.begin(), s->h_sa.end(), ta ^ xa) - s->h_sa.begin()) : r;
                    if (ur >= r) pairs.push_back(make_uint2((u32)r, (u32)ur));
                }
                RR->off[j + 1] = (i64)pairs.size();
            }
            // column pairs per generator (independent of the row): valid columns and their partners; for x_a = 0 the
            // pair lives in one row and is listed once (smaller column first)
            std::vector<uint2> cpairs;
            std::vector<u32> cstr;
            RR->coff.assign(n_rot + 1, 0);
            if ((double)n_rot * (double)s->Db <= 5e8) {
                for (i64 j = 0; j < n_rot; ++j) {
                    const u64 xa = gen->h_xg[j] & mask_a, xb = gen->h_xg[j] >> s->n_orb;
                    const int pxb = __builtin_popcountll(xb);
                    for (i64 c = 0; c < s->Db; ++c) {
                        const u64 tb = s->h_sb[c];
                        if (2 * __builtin_popcountll(tb & xb) != pxb) continue;
                        const i64 uc = xb ? (i64)(std::lower_bound(s->h_sb.begin(), s->h_sb.end(), tb ^ xb) - s->h_sb.begin()) : c;
                        if (xa == 0 && uc <= c) continue;
                        cpairs.push_back(make_uint2((u32)c, (u32)uc));
                        cstr.push_back((u32)tb);
                    }
                    RR->coff[j + 1] = (i64)cpairs.size();
                }
            }
            // z-reduction modulo x (exact on every valid target: z and z ^ x_s differ by the constant (-1)^{popc(x_s)/2}
            // there, cf. bs_plan.cu): strings that differ by x on a spin merge, 8 strings of a double excitation -> 2
            std::vector<u64> rz;
            std::vector<double2> rw;
            RR->roff.assign(n_rot + 1, 0);
            for (i64 j = 0; j < n_rot; ++j) {
                const u64 xa = gen->h_xg[j] & mask_a, xb = gen->h_xg[j] >> s->n_orb;
                const double sga = ((__builtin_popcountll(xa) / 2) & 1) ? -1.0 : 1.0;
                const double sgb = ((__builtin_popcountll(xb) / 2) & 1) ? -1.0 : 1.0;
                std::vector<std::pair<u64, double2>> v;
                for (i64 k = gen->h_offs[j]; k < gen->h_offs[j + 1]; ++k) {
                    u64 za = gen->h_z[k] & mask_a, zb = gen->h_z[k] >> s->n_orb;
                    double2 wk = make_double2(gen->h_w[2 * k], gen->h_w[2 * k + 1]);
                    if ((za ^ xa) < za) { za ^= xa; wk.x *= sga; wk.y *= sga; }
                    if ((zb ^ xb) < zb) { zb ^= xb; wk.x *= sgb; wk.y *= sgb; }
                    v.push_back({za | (zb << s->n_orb), wk});
                }
                std::stable_sort(v.begin(), v.end(), [](const std::pair<u64, double2>& a, const std::pair<u64, double2>& b) {
                    return a.first < b.first;
                });
                for (size_t k = 0; k < v.size();) {
                    double2 acc = v[k].second;
                    size_t e2 = k + 1;
                    for (; e2 < v.size() && v[e2].first == v[k].first; ++e2) {
                        acc.x += v[e2].second.x;
                        acc.y += v[e2].second.y;
                    }
                    if (acc.x != 0.0 || acc.y != 0.0) {
                        rz.push_back(v[k].first);
                        rw.push_back(acc);
                    }
                    k = e2;
                }
                RR->roff[j + 1] = (i64)rz.size();
            }
            // ---- orbit cells: sub-runs and their tables (see k_rot_orbit) ----------------------------------------------
            std::vector<u32> opat, oout;
            std::vector<unsigned short> opart;
            std::vector<int> opoff;
            if (s->n_orb <= 32 && (double)n_rot * 1024.0 * 2.0 <= 2e9) {
                const int n = s->n_orb, Nb = s->n_beta;
                const u32 full_b = n == 32 ? 0xFFFFFFFFu : ((1u << n) - 1u);
                std::map<u32, int> tab_of;   // orbital set U -> index in orbit_tabs
                auto table_for = [&](u32 U) {
                    auto f = tab_of.find(U);
                    if (f != tab_of.end()) return f->second;
                    bs_op::RotRows::OrbitU t{};
                    t.nU = __builtin_popcount(U);
                    t.pat_off = (i64)opat.size();
                    std::vector<std::vector<u32>> by_m(t.nU + 1);
                    for (u32 p2 = U;; p2 = (p2 - 1) & U) {   // all sub-masks of U
                        by_m[__builtin_popcount(p2)].push_back(p2);
                        if (p2 == 0) break;
                    }
                    int off = 0;
                    for (int m = 0; m <= t.nU; ++m) {
                        std::sort(by_m[m].begin(), by_m[m].end());
                        t.m_off[m] = off;
                        off += (int)by_m[m].size();
                        opat.insert(opat.end(), by_m[m].begin(), by_m[m].end());
                    }
                    for (int m = t.nU + 1; m < 12; ++m) t.m_off[m] = off;
                    t.n_pat = off;
                    t.out_off = (i64)oout.size();
                    const u32 outside = full_b & ~U;
                    for (u32 o = outside;; o = (o - 1) & outside) {   // occupations outside U
                        const int m = Nb - __builtin_popcount(o);
                        if (m >= 0 && m <= t.nU) oout.push_back(o);
                        if (o == 0) break;
                    }
                    t.n_out = (int)(oout.size() - t.out_off);
                    RR->orbit_tabs.push_back(t);
                    tab_of[U] = (int)RR->orbit_tabs.size() - 1;
                    return tab_of[U];
                };
                for (i64 j = 0; j < n_rot;) {
                    const u64 xa0 = gen->h_xg[j] & mask_a;
                    i64 e2 = j + 1;
                    if (gen->h_xg[j] != 0)
                        while (e2 < n_rot && gen->h_xg[e2] != 0 && (gen->h_xg[e2] & mask_a) == xa0) ++e2;
                    if (e2 - j < 2) {   // isolated generator: no run, no sub-run
                        j = e2;
                        continue;
                    }
                    for (i64 q = j; q < e2;) {   // greedy sub-runs: beta masks touching at most kOrbitUmax orbitals
                        u32 U = 0;
                        i64 q1 = q;
                        while (q1 < e2 && __builtin_popcount(U | (u32)(gen->h_xg[q1] >> n)) <= kOrbitUmax) U |= (u32)(gen->h_xg[q1++] >> n);
                        bs_op::RotRows::OrbitSub sub{q, std::max(q1, q + 1), -1, 0, 0};
                        if (q1 > q && U != 0) {
                            sub.tab = table_for(U);
                            const bs_op::RotRows::OrbitU& t = RR->orbit_tabs[sub.tab];
                            sub.part_off = (i64)opart.size();
                            sub.poff_off = (i64)opoff.size();
                            const u32* pat = opat.data() + t.pat_off;
                            for (i64 g = sub.j0; g < sub.j1; ++g) {
                                const u32 xb = (u32)(gen->h_xg[g] >> n);
                                const int pxb = __builtin_popcount(xb);
                                for (int m = 0; m < 12; ++m) {
                                    opoff.push_back((int)((i64)opart.size() - sub.part_off));
                                    if (m > t.nU) continue;
                                    for (int i = t.m_off[m]; i < t.m_off[m + 1]; ++i) {
                                        if (2 * __builtin_popcount(pat[i] & xb) != pxb) continue;
                                        const u32 pp = pat[i] ^ xb;
                                        const int li = i - t.m_off[m];
                                        const int qi = (int)(std::lower_bound(pat + t.m_off[m], pat + t.m_off[m + 1], pp) - (pat + t.m_off[m]));
                                        // x_a = 0: the pair lives in one row and belongs to its smaller column (columns of an
                                        // orbit are ordered like their patterns); x_a != 0: every valid pattern pairs row 0 with row 1
                                        if (xa0 != 0 || qi > li) opart.push_back((unsigned short)(li | (qi << 8)));
                                    }
                                }
                            }
                        }
                        RR->orbit_subs.push_back(sub);
                        q = sub.j1;
                    }
                    j = e2;
                }
            }
            cudaError_t e = RR->d_pairs.upload(pairs, st);
            if (e == cudaSuccess) e = RR->d_opat.upload(opat, st);
            if (e == cudaSuccess) e = RR->d_oout.upload(oout, st);
            if (e == cudaSuccess) e = RR->d_opart.upload(opart, st);
            if (e == cudaSuccess) e = RR->d_opoff.upload(opoff, st);
            if (e == cudaSuccess) e = RR->d_rz.upload(rz, st);
            if (e == cudaSuccess) e = RR->d_rw.upload(rw, st);
            if (e == cudaSuccess) e = RR->d_roff.upload(RR->roff, st);
            if (e == cudaSuccess) e = RR->d_cpairs.upload(cpairs, st);
            if (e == cudaSuccess) e = RR->d_cstr.upload(cstr, st);
            if (e == cudaSuccess) e = RR->d_off.upload(RR->off, st);
            if (e == cudaSuccess) e = RR->d_coff.upload(RR->coff, st);
            if (e == cudaSuccess) e = cudaStreamSynchronize(st);
            if (e != cudaSuccess) {
                delete RR;
                BS_CUDA(e);
            }
            gen->rot_rows[s->id] = RR;
        } else RR = it->second;
    }
    const dim3 sgrid((unsigned)((s->Db + 255) / 256), (unsigned)std::min<i64>(s->Da, 65535));
    BS_REQUIRE(s->full || s->Da <= 65535, BS_ERR_ARG, "bs_apply_pauli_rotations: more than 65535 alpha strings");
    // ---- closed-cell batching of runs of generators (see k_rot_cell_rows) -------------------------------------
    // one generator, one launch (isolated generators, cells too large for shared memory, full space)
    auto single = [&](i64 j) {
        const int k0 = (int)gen->h_offs[j], k1 = (int)gen->h_offs[j + 1];
        const double2 sc1 = make_double2(sin(thetas[j]), cos(thetas[j]));
        if (gen->h_xg[j] == 0)
            k_rot_diag<<<nb, 256, 0, st>>>(s->ta, s->tb, s->n_orb, s->full ? 1 : 0, s->D, gen->d_z.p, gen->d_w.p, k0, k1,
                                           thetas[j], psi);
        else if (s->full)
            k_rot_full<<<nb, 256, 0, st>>>(s->D, gen->h_xg[j], gen->d_z.p, gen->d_w.p, k0, k1, thetas[j], sc1, psi);
        else if (RR && RR->coff.back() > 0) {
            const i64 nr = RR->off[j + 1] - RR->off[j], ncp = RR->coff[j + 1] - RR->coff[j];
            for (i64 r0 = 0; r0 < nr && ncp > 0; r0 += 65535) {
                const dim3 rg((unsigned)((ncp + 255) / 256), (unsigned)std::min<i64>(65535, nr - r0));
                k_rot_pairs<<<rg, 256, 0, st>>>(s->ta, s->tb, s->n_orb, RR->d_pairs.p + RR->off[j] + r0,
                                                RR->d_cpairs.p + RR->coff[j], ncp, RR->d_rz.p, RR->d_rw.p,
                                                (int)RR->roff[j], (int)RR->roff[j + 1], thetas[j], sc1, psi);
            }
        } else if (RR) {
            const i64 nr = RR->off[j + 1] - RR->off[j];
            for (i64 r0 = 0; r0 < nr; r0 += 65535) {
                const dim3 rg(sgrid.x, (unsigned)std::min<i64>(65535, nr - r0));
                k_rot_rows<<<rg, 256, 0, st>>>(s->ta, s->tb, s->n_orb, gen->h_xg[j], RR->d_pairs.p + RR->off[j] + r0,
                                               gen->d_z.p, gen->d_w.p, k0, k1, thetas[j], sc1, psi);
            }
        } else
            k_rot_sector<<<sgrid, 256, 0, st>>>(s->ta, s->tb, s->n_orb, gen->h_xg[j], gen->d_z.p, gen->d_w.p, k0, k1,
                                                thetas[j], sc1, psi);
        BS_COUNT_LAUNCH(1);
    };
    // test hooks, read once per process (never on a launch path)
    static const bool env_per_launch = getenv("BS_ROT_PER_LAUNCH") != nullptr;
    static const bool in_place = getenv("BS_ROT_IN_PLACE") != nullptr;   // cells in place (L2) even when they fit shared memory
    // BS_ROT_ORBIT=1 (test hook): orbit cells (k_rot_orbit) for common-x_a runs at any sector size.  Not the default:
    // measured slower than the in-place cells at configs[3] (1.79 s vs 1.32 s for the UCCSD list)
    static const int orbit_mode = getenv("BS_ROT_ORBIT") ? atoi(getenv("BS_ROT_ORBIT")) : 0;
    // row pairs too large for one block's shared memory in a cluster of two blocks (k_rot_cluster_rows): opt-in
    // 1: where the pair does not fit one block; 2 (test hook): every row-pair run whose single row fits
    static const int cluster_rows = getenv("BS_ROT_CLUSTER") ? atoi(getenv("BS_ROT_CLUSTER")) : 0;
    // column strings read from the pair list (1) or from the sector's string table (0); test hook, default below
    static const int cstr_mode = getenv("BS_ROT_CSTR") ? atoi(getenv("BS_ROT_CSTR")) : -1;
    const bool batching = RR && RR->coff.back() > 0 && !env_per_launch;
    {
        const size_t smem_cap = 190 * 1024;  // + the static generator chunk (7.5 KB)
        const u64 mask_a = (u64(1) << s->n_orb) - 1;
        std::vector<double2> h_sc(batching ? n_rot : 0);
        if (batching) {
        for (i64 j = 0; j < n_rot; ++j) h_sc[j] = make_double2(sin(thetas[j]), cos(thetas[j]));
        if (RR->d_th.n < (size_t)n_rot) {
            BS_CUDA(RR->d_th.alloc(n_rot));
            BS_CUDA(RR->d_sc.alloc(n_rot));
        }
        BS_CUDA(cudaMemcpyAsync(RR->d_th.p, thetas, n_rot * 8, cudaMemcpyHostToDevice, st));
        BS_CUDA(cudaMemcpyAsync(RR->d_sc.p, h_sc.data(), n_rot * 16, cudaMemcpyHostToDevice, st));
        BS_CUDA(cudaStreamSynchronize(st));  // h_sc is a local
        }
        i64 j = 0;
        while (j < n_rot) {
            const u64 xa0 = gen->h_xg[j] & mask_a, xb0 = gen->h_xg[j] >> s->n_orb;
            i64 e = j + 1;
            int kind = 0;  // 1: common x_a (rows / row pairs), 2: all x_b = 0 (columns)
            bool launched = false;
            const bool diag0 = gen->h_xg[j] == 0;  // diagonal generators never join a run
            while (batching && !diag0 && e < n_rot && gen->h_xg[e] != 0 && (gen->h_xg[e] & mask_a) == xa0) ++e;
            if (e - j >= 2) kind = 1;
            else if (batching && !diag0 && xb0 == 0) {
                e = j + 1;
                while (e < n_rot && gen->h_xg[e] != 0 && (gen->h_xg[e] >> s->n_orb) == 0) ++e;
                if (e - j >= 2) kind = 2;
            }
            for (i64 q = j; q < e && kind; ++q)
                if (RR->roff[q + 1] - RR->roff[q] > 256) kind = 0;  // kStrChunk
#define BS_ROT_ARGS_ROWS s->ta, s->tb, s->n_orb, pr, gen->d_xg.p, RR->d_roff.p, RR->d_rz.p, RR->d_rw.p, RR->d_th.p, RR->d_sc.p, \
                         RR->d_cpairs.p, cstr_arg, RR->d_coff.p, j, e, psi
#define BS_ROT_ARGS_COLS s->ta, s->tb, s->n_orb, gen->d_xg.p, RR->d_roff.p, RR->d_rz.p, RR->d_rw.p, RR->d_th.p, RR->d_sc.p, \
                         RR->d_pairs.p, RR->d_off.p, j, e, psi
#define BS_ROT_SMEM(K)                                                                                              \
    {                                                                                                               \
        static const cudaError_t e_attr = cudaFuncSetAttribute(K, cudaFuncAttributeMaxDynamicSharedMemorySize, 200 * 1024); \
        BS_CUDA(e_attr);                                                                                            \
    }
            if (kind == 1) {
                const int R = xa0 ? 2 : 1;
                const size_t smem = (size_t)R * s->Db * 16;
                const i64 n_cells = xa0 ? RR->off[j + 1] - RR->off[j] : s->Da;
                const uint2* pr = RR->d_pairs.p + RR->off[j];
                // column strings: from the pair list where the amplitudes come through L2 (in place, cluster: one dependent
                // look-up fewer, q32 1,323 -> 1,260 ms), from the sector's table (hot in L1) where the cell is in shared
                // memory; BS_ROT_CSTR = 0 | 1 forces either
                const bool cells_in_smem = smem <= smem_cap && !in_place && orbit_mode != 1 && !(R == 2 && cluster_rows == 2);
                const u32* cstr_arg = (cstr_mode >= 0 ? cstr_mode != 0 : !cells_in_smem) ? RR->d_cstr.p : nullptr;
                if (n_cells == 0) {
                    launched = true;  // x_a never valid in this sector: identity
                } else if (smem <= smem_cap && !in_place && orbit_mode != 1 && !(R == 2 && cluster_rows == 2)) {
                    if (R == 2) {
                        BS_ROT_SMEM((k_rot_cell_rows<2, false>))
                        k_rot_cell_rows<2, false><<<(unsigned)n_cells, 512, smem, st>>>(BS_ROT_ARGS_ROWS);
                    } else {
                        BS_ROT_SMEM((k_rot_cell_rows<1, false>))
                        k_rot_cell_rows<1, false><<<(unsigned)n_cells, 256, smem, st>>>(BS_ROT_ARGS_ROWS);
                    }
                    BS_COUNT_LAUNCH(1);
                    launched = true;
                } else if (R == 2 && cluster_rows && !in_place && orbit_mode != 1 &&
                           (size_t)s->Db * 16 + sizeof(GenChunk) + 1024 <= (size_t)227 * 1024) {
                    // one row per block of a two-block cluster (the pair does not fit one block, a single row does)
                    static const cudaError_t e_attr = cudaFuncSetAttribute(
                        k_rot_cluster_rows, cudaFuncAttributeMaxDynamicSharedMemorySize, 227 * 1024 - 1024 - (int)sizeof(GenChunk));
                    BS_CUDA(e_attr);
                    k_rot_cluster_rows<<<(unsigned)(2 * n_cells), 512, (size_t)s->Db * 16, st>>>(BS_ROT_ARGS_ROWS);
                    BS_COUNT_LAUNCH(1);
                    launched = true;
                } else if (!RR->orbit_subs.empty() && orbit_mode == 1 && !in_place) {
                    // cells of {row (pair)} x {orbit of <= 252 columns}: one launch per SUB-RUN, the cell in shared memory
                    auto it2 = std::lower_bound(RR->orbit_subs.begin(), RR->orbit_subs.end(), j,
                                                [](const bs_op::RotRows::OrbitSub& a, i64 v) { return a.j0 < v; });
                    for (; it2 != RR->orbit_subs.end() && it2->j0 < e; ++it2) {
                        const i64 j = it2->j0, e = it2->j1;   // shadow the run bounds for the argument macros
                        if (it2->tab < 0) {   // a beta mask wider than the orbit limit: in place for this sub-run
                            if (R == 2) k_rot_cell_rows<2, true><<<(unsigned)n_cells, 512, 0, st>>>(BS_ROT_ARGS_ROWS);
                            else k_rot_cell_rows<1, true><<<(unsigned)n_cells, 256, 0, st>>>(BS_ROT_ARGS_ROWS);
                        } else {
                            const bs_op::RotRows::OrbitU& t = RR->orbit_tabs[it2->tab];
                            OrbitTab T;
                            T.pat = RR->d_opat.p + t.pat_off;
                            T.outs = RR->d_oout.p + t.out_off;
                            T.pairs = RR->d_opart.p + it2->part_off;
                            T.pair_off = RR->d_opoff.p + it2->poff_off;
                            for (int m = 0; m < kOrbitUmax + 2; ++m) T.pat_off[m] = t.m_off[m];
                            T.n_pat = t.n_pat;
                            T.n_out = t.n_out;
                            T.Nb = s->n_beta;
                            const size_t osmem = (size_t)8 * R * kOrbitMax * 16 + (size_t)8 * 2 * kOrbitMax * 4;
                            const dim3 og((unsigned)std::min<i64>((t.n_out + 7) / 8, 4096), (unsigned)n_cells);
                            if (R == 2) {
                                BS_ROT_SMEM((k_rot_orbit<2>))
                                k_rot_orbit<2><<<og, 256, osmem, st>>>(s->ta, s->tb, s->n_orb, pr, T, RR->d_roff.p, RR->d_rz.p,
                                                                       RR->d_rw.p, RR->d_th.p, RR->d_sc.p, j, e, psi);
                            } else {
                                BS_ROT_SMEM((k_rot_orbit<1>))
                                k_rot_orbit<1><<<og, 256, osmem, st>>>(s->ta, s->tb, s->n_orb, pr, T, RR->d_roff.p, RR->d_rz.p,
                                                                       RR->d_rw.p, RR->d_th.p, RR->d_sc.p, j, e, psi);
                            }
                        }
                        BS_COUNT_LAUNCH(1);
                    }
                    launched = true;
                } else {   // the cell stays in place (L2): still one launch per run
                    if (R == 2) k_rot_cell_rows<2, true><<<(unsigned)n_cells, 512, 0, st>>>(BS_ROT_ARGS_ROWS);
                    else k_rot_cell_rows<1, true><<<(unsigned)n_cells, 256, 0, st>>>(BS_ROT_ARGS_ROWS);
                    BS_COUNT_LAUNCH(1);
                    launched = true;
                }
            } else if (kind == 2) {
                const int CC = in_place ? 0 : ((size_t)s->Da * 8 * 16 <= smem_cap) ? 8 : (((size_t)s->Da * 2 * 16 <= smem_cap) ? 2 : 0);
                if (CC) {
                    const size_t smem = (size_t)s->Da * CC * 16;
                    const unsigned nblk = (unsigned)((s->Db + CC - 1) / CC);
                    if (CC == 8) {
                        BS_ROT_SMEM((k_rot_cell_cols<8, false>))
                        k_rot_cell_cols<8, false><<<nblk, 1024, smem, st>>>(BS_ROT_ARGS_COLS);
                    } else {
                        BS_ROT_SMEM((k_rot_cell_cols<2, false>))
                        k_rot_cell_cols<2, false><<<nblk, 1024, smem, st>>>(BS_ROT_ARGS_COLS);
                    }
                } else {   // in place: 2 columns (one 32-byte sector per row) x all rows per block
                    k_rot_cell_cols<2, true><<<(unsigned)((s->Db + 1) / 2), 1024, 0, st>>>(BS_ROT_ARGS_COLS);
                }
                BS_COUNT_LAUNCH(1);
                launched = true;
            }
#undef BS_ROT_ARGS_ROWS
#undef BS_ROT_ARGS_COLS
#undef BS_ROT_SMEM
            if (!launched)
                for (i64 q = j; q < e; ++q) single(q);  // in order: rotations do not commute
            j = e;
        }
    }
    BS_CUDA(cudaGetLastError());
    return BS_OK;
}
