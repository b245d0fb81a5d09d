// Point-group symmetry blocking of the sector vector (Eq. 29-31; "sDet" of Table 2)
// for Abelian point groups (D2h and its subgroups): every orbital carries an irrep label in 0..7, the irrep of a spin
// string is the XOR of the labels of its occupied orbitals (direct products of one-dimensional irreps), and the
// symmetry block of the wave function holds the configurations with irrep(t_a) ^ irrep(t_b) = target (Eq. 30).
//
// Blocked layout (Eq. 29): blocks r = 0..7 in order of the alpha irrep; block r pairs the alpha strings of irrep r with
// the beta strings of irrep r ^ target, both in increasing numeric order, index = rank_a^r * D_b^r + rank_b^r.
// This file keeps the STORAGE blocked (state vectors the caller holds are |G| times smaller) and maps to and from the
// (N_alpha, N_beta) sector layout around the apply kernels, which run unblocked: the scatter zero-fills the other
// irreps, the gather reads back the target block (what leaves it is dropped: P_sym H P_sym, as for the sector itself).
#include <algorithm>

#include "bs_internal.cuh"

struct bs_symsector {
    bs_sector* parent;
    int target;
    i64 dim;
    i64 da[8], db[8], off[9];     // strings per irrep, block offsets
    DevBuf<unsigned char> d_ia, d_ib;   // irrep of every alpha / beta string of the parent sector
    DevBuf<u32> d_ra, d_rb;             // rank of the string among the strings of its own irrep
    DevBuf<i64> d_off, d_db;            // [8] block offsets, beta count of the block's beta irrep
    DevBuf<double2> d_in, d_out;        // full-sector scratch of bs_sym_apply / bs_sym_expect (allocated on first use)
};

namespace {

// one thread per amplitude of the parent sector; GATHER: blocked[idx] = full[i], else full[i] = allowed ? blocked[idx] : 0
template <bool GATHER>
__global__ void __launch_bounds__(256)
k_sym_map(const unsigned char* __restrict__ ia, const unsigned char* __restrict__ ib, const u32* __restrict__ ra,
          const u32* __restrict__ rb, const i64* __restrict__ off, const i64* __restrict__ dbr, int target, i64 Db,
          const double2* __restrict__ src, double2* __restrict__ dst) {
    const u32 col = blockIdx.x * blockDim.x + threadIdx.x;
    const i64 row = blockIdx.y;
    if (col >= Db) return;
    const int ga = ia[row], gb = ib[col];
    const bool allowed = (ga ^ gb) == target;
    const i64 i = row * Db + col;
    const i64 idx = allowed ? off[ga] + (i64)ra[row] * dbr[ga] + rb[col] : 0;
    if (GATHER) {
        if (allowed) dst[idx] = src[i];
    } else dst[i] = allowed ? src[idx] : make_double2(0.0, 0.0);
}

int sym_map(bs_symsector* h, bool gather, const double2* src, double2* dst, cudaStream_t st) {
    const bs_sector* s = h->parent;
    for (i64 r0 = 0; r0 < s->Da; r0 += 65535) {
        const dim3 grid((unsigned)((s->Db + 255) / 256), (unsigned)std::min<i64>(65535, s->Da - r0));
        const double2* sp = gather ? src + r0 * s->Db : src;
        double2* dp = gather ? dst : dst + r0 * s->Db;
        if (gather)
            k_sym_map<true><<<grid, 256, 0, st>>>(h->d_ia.p + r0, h->d_ib.p, h->d_ra.p + r0, h->d_rb.p, h->d_off.p,
                                                  h->d_db.p, h->target, s->Db, sp, dp);
        else
            k_sym_map<false><<<grid, 256, 0, st>>>(h->d_ia.p + r0, h->d_ib.p, h->d_ra.p + r0, h->d_rb.p, h->d_off.p,
                                                   h->d_db.p, h->target, s->Db, sp, dp);
        BS_COUNT_LAUNCH(1);
    }
    BS_CUDA(cudaGetLastError());
    return BS_OK;
}

int ensure_scratch(bs_symsector* h) {
    if (!h->d_in.p) BS_CUDA(h->d_in.alloc(h->parent->D));
    if (!h->d_out.p) BS_CUDA(h->d_out.alloc(h->parent->D));
    return BS_OK;
}

}  // namespace

extern "C" int bs_symsector_build(bs_sector_t parent, const int* orb_irrep, int target_irrep, void* cuda_stream,
                                  bs_symsector_t* out) {
    BS_REQUIRE(parent && orb_irrep && out, BS_ERR_ARG, "bs_symsector_build: NULL argument");
    BS_REQUIRE(!parent->full, BS_ERR_ARG, "bs_symsector_build: needs an (N_alpha, N_beta) sector");
    BS_REQUIRE(target_irrep >= 0 && target_irrep < 8, BS_ERR_ARG, "bs_symsector_build: irreps are 0..7");
    for (int p = 0; p < parent->n_orb; ++p)
        BS_REQUIRE(orb_irrep[p] >= 0 && orb_irrep[p] < 8, BS_ERR_ARG, "bs_symsector_build: orbital %d has irrep %d", p,
                   orb_irrep[p]);
    cudaStream_t st = (cudaStream_t)cuda_stream;
    bs_symsector* h = new (std::nothrow) bs_symsector;
    BS_REQUIRE(h, BS_ERR_ALLOC, "bs_symsector_build: host allocation failed");
    h->parent = parent;
    h->target = target_irrep;
    auto label = [&](const std::vector<u64>& strs, std::vector<unsigned char>& irr, std::vector<u32>& rank, i64* cnt) {
        for (int g = 0; g < 8; ++g) cnt[g] = 0;
        irr.resize(strs.size());
        rank.resize(strs.size());
        for (size_t i = 0; i < strs.size(); ++i) {
            int g = 0;
            for (u64 w = strs[i]; w; w &= w - 1) g ^= orb_irrep[__builtin_ctzll(w)];
            irr[i] = (unsigned char)g;
            rank[i] = (u32)cnt[g]++;   // strings are in increasing numeric order
        }
    };
    std::vector<unsigned char> ia, ib;
    std::vector<u32> ra, rb;
    label(parent->h_sa, ia, ra, h->da);
    label(parent->h_sb, ib, rb, h->db);
    std::vector<i64> off(8), dbr(8);
    h->off[0] = 0;
    for (int r = 0; r < 8; ++r) {
        dbr[r] = h->db[r ^ target_irrep];
        off[r] = h->off[r];
        h->off[r + 1] = h->off[r] + h->da[r] * dbr[r];
    }
    h->dim = h->off[8];
    cudaError_t e = h->d_ia.upload(ia, st);
    if (e == cudaSuccess) e = h->d_ib.upload(ib, st);
    if (e == cudaSuccess) e = h->d_ra.upload(ra, st);
    if (e == cudaSuccess) e = h->d_rb.upload(rb, st);
    if (e == cudaSuccess) e = h->d_off.upload(off, st);
    if (e == cudaSuccess) e = h->d_db.upload(dbr, st);
    if (e == cudaSuccess) e = cudaStreamSynchronize(st);
    if (e != cudaSuccess) {
        delete h;
        BS_CUDA(e);
    }
    *out = h;
    return BS_OK;
}

extern "C" int bs_symsector_info(bs_symsector_t h, int64_t* dim, int64_t dim_alpha[8], int64_t dim_beta[8]) {
    BS_REQUIRE(h, BS_ERR_ARG, "bs_symsector_info: NULL handle");
    if (dim) *dim = h->dim;
    for (int r = 0; r < 8; ++r) {
        if (dim_alpha) dim_alpha[r] = h->da[r];
        if (dim_beta) dim_beta[r] = h->db[r];
    }
    return BS_OK;
}

extern "C" int bs_symsector_destroy(bs_symsector_t h) {
    delete h;
    return BS_OK;
}

extern "C" int bs_sym_scatter(bs_symsector_t h, const void* psi_blocked, void* psi_sector, void* cuda_stream) {
    BS_REQUIRE(h && psi_blocked && psi_sector, BS_ERR_ARG, "bs_sym_scatter: NULL argument");
    return sym_map(h, false, (const double2*)psi_blocked, (double2*)psi_sector, (cudaStream_t)cuda_stream);
}

extern "C" int bs_sym_gather(bs_symsector_t h, const void* psi_sector, void* psi_blocked, void* cuda_stream) {
    BS_REQUIRE(h && psi_blocked && psi_sector, BS_ERR_ARG, "bs_sym_gather: NULL argument");
    return sym_map(h, true, (const double2*)psi_sector, (double2*)psi_blocked, (cudaStream_t)cuda_stream);
}

extern "C" int bs_sym_apply(bs_op_t op, bs_symsector_t h, const void* psi_in, void* psi_out, void* cuda_stream) {
    BS_REQUIRE(op && h && psi_in && psi_out, BS_ERR_ARG, "bs_sym_apply: NULL argument");
    int rc = ensure_scratch(h);
    if (rc) return rc;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    if ((rc = sym_map(h, false, (const double2*)psi_in, h->d_in.p, st))) return rc;
    if ((rc = bs_apply(op, h->parent, h->d_in.p, h->d_out.p, cuda_stream))) return rc;
    return sym_map(h, true, h->d_out.p, (double2*)psi_out, st);
}

extern "C" int bs_sym_expect(bs_op_t op, bs_symsector_t h, const void* psi, double result_reim[2], void* cuda_stream) {
    BS_REQUIRE(op && h && psi && result_reim, BS_ERR_ARG, "bs_sym_expect: NULL argument");
    int rc = ensure_scratch(h);
    if (rc) return rc;
    if ((rc = sym_map(h, false, (const double2*)psi, h->d_in.p, (cudaStream_t)cuda_stream))) return rc;
    return bs_expect(op, h->parent, h->d_in.p, result_reim, cuda_stream);   // the embedded vector is zero outside the block
}
