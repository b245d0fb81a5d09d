// a1 canonical reduction + a2 X-mask grouping and phase fold (Eq. 24).
//
// Device pipeline for BS_MODE_CANONICAL:
//   1. stable LSD radix sort of the 128-bit key (x major, z minor): sort by z carrying the input
//      index, gather x through it, sort by x (cub::DeviceRadixSort is stable, so equal keys stay
//      in input order);
//   2. head flags of equal-key runs, inclusive scan -> run ids, run starts;
//   3. one thread per run sums its coefficients sequentially in input order (bit-reproducible);
//   4. drop |c| < eps_drop (scan + compaction);
//   5. head flags by x -> xg[G], offs[G+1];
//   6. fold w_k = c_k (-i)^{ny_k}, ny_k = popc(x_k & z_k) (exact: swap / negate of re, im).
// CUB is used as a library for the radix sort and the prefix sums only.
#include <cub/cub.cuh>

#include "bs_internal.cuh"

namespace {

__global__ void k_iota(u32* idx, i64 n) {
    i64 i = blockIdx.x * (i64)blockDim.x + threadIdx.x;
    if (i < n) idx[i] = (u32)i;
}

__global__ void k_gather_u64(const u64* __restrict__ src, const u32* __restrict__ idx, u64* __restrict__ dst, i64 n) {
    i64 i = blockIdx.x * (i64)blockDim.x + threadIdx.x;
    if (i < n) dst[i] = src[idx[i]];
}

// head[i] = 1 where a new (x,z) key starts
__global__ void k_key_heads(const u64* __restrict__ x, const u64* __restrict__ z, int* __restrict__ head, i64 n) {
    i64 i = blockIdx.x * (i64)blockDim.x + threadIdx.x;
    if (i < n) head[i] = (i == 0 || x[i] != x[i - 1] || z[i] != z[i - 1]) ? 1 : 0;
}

__global__ void k_x_heads(const u64* __restrict__ x, int* __restrict__ head, i64 n) {
    i64 i = blockIdx.x * (i64)blockDim.x + threadIdx.x;
    if (i < n) head[i] = (i == 0 || x[i] != x[i - 1]) ? 1 : 0;
}

// start[id-1] = i for every head (ids are the inclusive scan of the heads), start[n_runs] = n
__global__ void k_run_starts(const int* __restrict__ head, const int* __restrict__ id, i64* __restrict__ start,
                             i64 n, i64 n_runs) {
    i64 i = blockIdx.x * (i64)blockDim.x + threadIdx.x;
    if (i < n && head[i]) start[id[i] - 1] = i;
    if (i == 0) start[n_runs] = n;
}

// one thread per run of equal keys: sequential sum in input order, keep flag against eps_drop
__global__ void k_merge_runs(const i64* __restrict__ start, const u32* __restrict__ idx,
                             const double2* __restrict__ c_in, const u64* __restrict__ xs,
                             const u64* __restrict__ zs, u64* __restrict__ xu, u64* __restrict__ zu,
                             double2* __restrict__ cu, int* __restrict__ keep, i64 n_runs, double eps) {
    i64 r = blockIdx.x * (i64)blockDim.x + threadIdx.x;
    if (r >= n_runs) return;
    i64 b = start[r], e = start[r + 1];
    double re = 0.0, im = 0.0;
    for (i64 i = b; i < e; ++i) {
        double2 c = c_in[idx[i]];
        re += c.x;
        im += c.y;
    }
    xu[r] = xs[b];
    zu[r] = zs[b];
    cu[r] = make_double2(re, im);
    // drop |c| < eps_drop; a merged coefficient that is exactly zero is dropped even with eps_drop = 0
    const double a = hypot(re, im);
    keep[r] = (a < eps || !(a > 0.0)) ? 0 : 1;
}

__global__ void k_compact(const int* __restrict__ keep, const int* __restrict__ pos, const u64* __restrict__ xu,
                          const u64* __restrict__ zu, const double2* __restrict__ cu, u64* __restrict__ xc,
                          u64* __restrict__ zc, double2* __restrict__ cc, i64 n) {
    i64 i = blockIdx.x * (i64)blockDim.x + threadIdx.x;
    if (i < n && keep[i]) {
        int p = pos[i] - 1;
        xc[p] = xu[i];
        zc[p] = zu[i];
        cc[p] = cu[i];
    }
}

// group tables: xg[g] = x of the run, offs[g] = first string; offs[G] = M
__global__ void k_group_tables(const int* __restrict__ head, const int* __restrict__ id, const u64* __restrict__ x,
                               u64* __restrict__ xg, i64* __restrict__ offs, i64 n, i64 G) {
    i64 i = blockIdx.x * (i64)blockDim.x + threadIdx.x;
    if (i < n && head[i]) {
        xg[id[i] - 1] = x[i];
        offs[id[i] - 1] = i;
    }
    if (i == 0) offs[G] = n;
}

// w = c * (-i)^{ny}: ny&3 = 0: c; 1: (im, -re); 2: -c; 3: (-im, re)     (reading U2)
__global__ void k_fold_phase(const u64* __restrict__ x, const u64* __restrict__ z, const double2* __restrict__ c,
                             double2* __restrict__ w, i64 n) {
    i64 i = blockIdx.x * (i64)blockDim.x + threadIdx.x;
    if (i >= n) return;
    int ny = __popcll(x[i] & z[i]) & 3;
    double2 v = c[i], r;
    if (ny == 0) r = v;
    else if (ny == 1) r = make_double2(v.y, -v.x);
    else if (ny == 2) r = make_double2(-v.x, -v.y);
    else r = make_double2(-v.y, v.x);
    w[i] = r;
}

inline unsigned nblk(i64 n, int t = 256) { return (unsigned)((n + t - 1) / t); }

int finish_op(bs_op* op, const u64* d_x_per_string, const double2* d_c, cudaStream_t st) {
    // host mirrors
    i64 G = op->G, M = op->M;
    op->h_xg.resize(G);
    op->h_offs.resize(G + 1);
    op->h_z.resize(M);
    op->h_c.resize(2 * M);
    op->h_w.resize(2 * M);
    if (G) BS_CUDA(cudaMemcpyAsync(op->h_xg.data(), op->d_xg.p, G * 8, cudaMemcpyDeviceToHost, st));
    BS_CUDA(cudaMemcpyAsync(op->h_offs.data(), op->d_offs.p, (G + 1) * 8, cudaMemcpyDeviceToHost, st));
    if (M) {
        BS_CUDA(cudaMemcpyAsync(op->h_z.data(), op->d_z.p, M * 8, cudaMemcpyDeviceToHost, st));
        BS_CUDA(cudaMemcpyAsync(op->h_c.data(), d_c, M * 16, cudaMemcpyDeviceToHost, st));
        BS_CUDA(cudaMemcpyAsync(op->h_w.data(), op->d_w.p, M * 16, cudaMemcpyDeviceToHost, st));
    }
    (void)d_x_per_string;
    BS_CUDA(cudaStreamSynchronize(st));
    return BS_OK;
}

}  // namespace

// canonical reduction + grouping of raw terms that already live on the device (x0, z0, c0 [M0])
int bs_group_canonical_dev(bs_op* op, const u64* x0p, const u64* z0p, const double2* c0p, i64 M0, double eps,
                           cudaStream_t st) {
    const int nq = op->n_qubits;
    if (M0 == 0) {
        op->G = 0;
        op->M = 0;
        BS_CUDA(op->d_xg.alloc(0));
        BS_CUDA(op->d_z.alloc(0));
        BS_CUDA(op->d_w.alloc(0));
        BS_CUDA(op->d_offs.alloc(1));
        BS_CUDA(cudaMemsetAsync(op->d_offs.p, 0, 8, st));
        return finish_op(op, nullptr, nullptr, st);
    }
    struct View {
        const u64* p;
    };
    struct ViewC {
        const double2* p;
    };
    const View x0{x0p}, z0{z0p};
    const ViewC c0{c0p};
    DevBuf<u64> ka, kb;
    DevBuf<u32> ia, ib;
    BS_CUDA(ka.alloc(M0));
    BS_CUDA(kb.alloc(M0));
    BS_CUDA(ia.alloc(M0));
    BS_CUDA(ib.alloc(M0));

    // 1. stable sort by (x, z): LSD over the two 64-bit words
    size_t tmp_bytes = 0;
    BS_CUDA(cub::DeviceRadixSort::SortPairs(nullptr, tmp_bytes, z0.p, ka.p, ia.p, ib.p, (int)M0, 0, nq, st));
    DevBuf<char> tmp;
    BS_CUDA(tmp.alloc(tmp_bytes));
    k_iota<<<nblk(M0), 256, 0, st>>>(ia.p, M0);
    BS_CUDA(cub::DeviceRadixSort::SortPairs(tmp.p, tmp_bytes, z0.p, ka.p, ia.p, ib.p, (int)M0, 0, nq, st));
    k_gather_u64<<<nblk(M0), 256, 0, st>>>(x0.p, ib.p, kb.p, M0);           // kb = x in z order
    BS_CUDA(cub::DeviceRadixSort::SortPairs(tmp.p, tmp_bytes, kb.p, ka.p, ib.p, ia.p, (int)M0, 0, nq, st));
    // now ka = sorted x, ia = input index in (x,z) order
    k_gather_u64<<<nblk(M0), 256, 0, st>>>(z0.p, ia.p, kb.p, M0);           // kb = sorted z
    BS_COUNT_LAUNCH(3 + 3);

    // 2. runs of equal keys
    DevBuf<int> head, id;
    BS_CUDA(head.alloc(M0));
    BS_CUDA(id.alloc(M0));
    k_key_heads<<<nblk(M0), 256, 0, st>>>(ka.p, kb.p, head.p, M0);
    size_t scan_bytes = 0;
    BS_CUDA(cub::DeviceScan::InclusiveSum(nullptr, scan_bytes, head.p, id.p, (int)M0, st));
    DevBuf<char> stmp;
    BS_CUDA(stmp.alloc(scan_bytes));
    BS_CUDA(cub::DeviceScan::InclusiveSum(stmp.p, scan_bytes, head.p, id.p, (int)M0, st));
    int n_runs = 0;
    BS_CUDA(cudaMemcpyAsync(&n_runs, id.p + (M0 - 1), 4, cudaMemcpyDeviceToHost, st));
    BS_CUDA(cudaStreamSynchronize(st));
    DevBuf<i64> start;
    BS_CUDA(start.alloc(n_runs + 1));
    k_run_starts<<<nblk(M0), 256, 0, st>>>(head.p, id.p, start.p, M0, n_runs);

    // 3. + 4. merge in input order, drop
    DevBuf<u64> xu, zu;
    DevBuf<double2> cu;
    DevBuf<int> keep, pos;
    BS_CUDA(xu.alloc(n_runs));
    BS_CUDA(zu.alloc(n_runs));
    BS_CUDA(cu.alloc(n_runs));
    BS_CUDA(keep.alloc(n_runs));
    BS_CUDA(pos.alloc(n_runs));
    k_merge_runs<<<nblk(n_runs, 128), 128, 0, st>>>(start.p, ia.p, c0.p, ka.p, kb.p, xu.p, zu.p, cu.p, keep.p,
                                                   n_runs, eps);
    BS_CUDA(cub::DeviceScan::InclusiveSum(stmp.p, scan_bytes, keep.p, pos.p, n_runs, st));
    int M = 0;
    BS_CUDA(cudaMemcpyAsync(&M, pos.p + (n_runs - 1), 4, cudaMemcpyDeviceToHost, st));
    BS_CUDA(cudaStreamSynchronize(st));
    BS_COUNT_LAUNCH(6);
    op->M = M;
    DevBuf<u64> xc;
    DevBuf<double2> cc;
    BS_CUDA(xc.alloc(M));
    BS_CUDA(cc.alloc(M));
    BS_CUDA(op->d_z.alloc(M));
    BS_CUDA(op->d_w.alloc(M));
    if (M == 0) {
        op->G = 0;
        BS_CUDA(op->d_xg.alloc(0));
        BS_CUDA(op->d_offs.alloc(1));
        BS_CUDA(cudaMemsetAsync(op->d_offs.p, 0, 8, st));
        return finish_op(op, nullptr, nullptr, st);
    }
    k_compact<<<nblk(n_runs), 256, 0, st>>>(keep.p, pos.p, xu.p, zu.p, cu.p, xc.p, op->d_z.p, cc.p, n_runs);

    // 5. groups by x
    k_x_heads<<<nblk(M), 256, 0, st>>>(xc.p, head.p, M);
    BS_CUDA(cub::DeviceScan::InclusiveSum(stmp.p, scan_bytes, head.p, id.p, M, st));
    int G = 0;
    BS_CUDA(cudaMemcpyAsync(&G, id.p + (M - 1), 4, cudaMemcpyDeviceToHost, st));
    BS_CUDA(cudaStreamSynchronize(st));
    op->G = G;
    BS_CUDA(op->d_xg.alloc(G));
    BS_CUDA(op->d_offs.alloc(G + 1));
    k_group_tables<<<nblk(M), 256, 0, st>>>(head.p, id.p, xc.p, op->d_xg.p, op->d_offs.p, M, G);
    // 6. fold
    k_fold_phase<<<nblk(M), 256, 0, st>>>(xc.p, op->d_z.p, cc.p, op->d_w.p, M);
    BS_COUNT_LAUNCH(5);
    BS_CUDA(cudaGetLastError());
    return finish_op(op, xc.p, cc.p, st);
}

namespace {

int group_canonical(bs_op* op, const u64* hx, const u64* hz, const double* hc, i64 M0, double eps, cudaStream_t st) {
    DevBuf<u64> x0, z0;
    DevBuf<double2> c0;
    BS_CUDA(x0.alloc(M0));
    BS_CUDA(z0.alloc(M0));
    BS_CUDA(c0.alloc(M0));
    if (M0) {
        BS_CUDA(cudaMemcpyAsync(x0.p, hx, M0 * 8, cudaMemcpyHostToDevice, st));
        BS_CUDA(cudaMemcpyAsync(z0.p, hz, M0 * 8, cudaMemcpyHostToDevice, st));
        BS_CUDA(cudaMemcpyAsync(c0.p, hc, M0 * 16, cudaMemcpyHostToDevice, st));
    }
    return bs_group_canonical_dev(op, x0.p, z0.p, c0.p, M0, eps, st);  // synchronises before the buffers die
}

int group_sequence(bs_op* op, const u64* hx, const u64* hz, const double* hc, i64 M, const i64* seq, i64 n_seq,
                   cudaStream_t st) {
    BS_REQUIRE(seq && n_seq >= 0, BS_ERR_ARG, "bs_group_xmask: mode 1 needs seq_offsets");
    BS_REQUIRE(seq[0] == 0 && seq[n_seq] == M, BS_ERR_ARG, "bs_group_xmask: seq_offsets must span [0, M]");
    std::vector<u64> xg(n_seq), xs(M);
    for (i64 j = 0; j < n_seq; ++j) {
        BS_REQUIRE(seq[j + 1] > seq[j], BS_ERR_ARG, "bs_group_xmask: empty or decreasing run %lld", (long long)j);
        xg[j] = hx[seq[j]];
        for (i64 k = seq[j]; k < seq[j + 1]; ++k) {
            BS_REQUIRE(hx[k] == xg[j], BS_ERR_ARG, "bs_group_xmask: run %lld mixes x masks", (long long)j);
            xs[k] = hx[k];
        }
    }
    op->G = n_seq;
    op->M = M;
    DevBuf<u64> dx;
    DevBuf<double2> dc;
    BS_CUDA(dx.alloc(M));
    BS_CUDA(dc.alloc(M));
    BS_CUDA(op->d_xg.alloc(n_seq));
    BS_CUDA(op->d_offs.alloc(n_seq + 1));
    BS_CUDA(op->d_z.alloc(M));
    BS_CUDA(op->d_w.alloc(M));
    if (n_seq) BS_CUDA(cudaMemcpyAsync(op->d_xg.p, xg.data(), n_seq * 8, cudaMemcpyHostToDevice, st));
    BS_CUDA(cudaMemcpyAsync(op->d_offs.p, seq, (n_seq + 1) * 8, cudaMemcpyHostToDevice, st));
    if (M) {
        BS_CUDA(cudaMemcpyAsync(dx.p, xs.data(), M * 8, cudaMemcpyHostToDevice, st));
        BS_CUDA(cudaMemcpyAsync(op->d_z.p, hz, M * 8, cudaMemcpyHostToDevice, st));
        BS_CUDA(cudaMemcpyAsync(dc.p, hc, M * 16, cudaMemcpyHostToDevice, st));
        k_fold_phase<<<nblk(M), 256, 0, st>>>(dx.p, op->d_z.p, dc.p, op->d_w.p, M);
        BS_COUNT_LAUNCH(1);
        BS_CUDA(cudaGetLastError());
    }
    return finish_op(op, dx.p, dc.p, st);
}

}  // namespace

extern "C" int bs_group_xmask(const uint64_t* x, const uint64_t* z, const double* coeff_reim, int64_t M,
                              int n_qubits, double eps_drop, int mode, const int64_t* seq_offsets,
                              int64_t n_seq, void* cuda_stream, bs_op_t* out) {
    BS_REQUIRE(out, BS_ERR_ARG, "bs_group_xmask: out is NULL");
    BS_REQUIRE(M >= 0 && M < (i64(1) << 31), BS_ERR_ARG, "bs_group_xmask: M out of range");
    BS_REQUIRE(M == 0 || (x && z && coeff_reim), BS_ERR_ARG, "bs_group_xmask: NULL input array");
    BS_REQUIRE(n_qubits >= 1 && n_qubits <= 64, BS_ERR_ARG, "bs_group_xmask: n_qubits must be in [1, 64]");
    BS_REQUIRE(mode == BS_MODE_CANONICAL || mode == BS_MODE_SEQUENCE, BS_ERR_ARG, "bs_group_xmask: bad mode");
    BS_REQUIRE(mode == BS_MODE_SEQUENCE || seq_offsets == nullptr, BS_ERR_ARG,
               "bs_group_xmask: seq_offsets must be NULL in canonical mode");
    if (n_qubits < 64) {
        u64 lim = ~u64(0) << n_qubits;
        for (i64 k = 0; k < M; ++k)
            BS_REQUIRE(!((x[k] | z[k]) & lim), BS_ERR_ARG, "bs_group_xmask: string %lld has bits above n_qubits",
                       (long long)k);
    }
    int dev_count = 0;
    BS_CUDA(cudaGetDeviceCount(&dev_count));
    BS_REQUIRE(dev_count > 0, BS_ERR_CUDA, "no CUDA device (libbs has no CPU fallback)");
    cudaStream_t st = (cudaStream_t)cuda_stream;
    bs_op* op = new (std::nothrow) bs_op;
    BS_REQUIRE(op, BS_ERR_ALLOC, "bs_group_xmask: host allocation failed");
    op->id = bs_next_id();
    op->n_qubits = n_qubits;
    op->mode = mode;
    int rc = (mode == BS_MODE_CANONICAL) ? group_canonical(op, x, z, coeff_reim, M, eps_drop, st)
                                         : group_sequence(op, x, z, coeff_reim, M, seq_offsets, n_seq, st);
    if (rc != BS_OK) {
        delete op;
        return rc;
    }
    *out = op;
    return BS_OK;
}

extern "C" int bs_op_info(bs_op_t op, int64_t* n_groups, int64_t* n_terms, int* n_qubits) {
    BS_REQUIRE(op, BS_ERR_ARG, "bs_op_info: NULL handle");
    if (n_groups) *n_groups = op->G;
    if (n_terms) *n_terms = op->M;
    if (n_qubits) *n_qubits = op->n_qubits;
    return BS_OK;
}

extern "C" int bs_op_export(bs_op_t op, uint64_t* xg, int64_t* offs, uint64_t* z, double* c_reim, double* w_reim) {
    BS_REQUIRE(op, BS_ERR_ARG, "bs_op_export: NULL handle");
    if (xg && op->G) std::memcpy(xg, op->h_xg.data(), op->G * 8);
    if (offs) std::memcpy(offs, op->h_offs.data(), (op->G + 1) * 8);
    if (z && op->M) std::memcpy(z, op->h_z.data(), op->M * 8);
    if (c_reim && op->M) std::memcpy(c_reim, op->h_c.data(), op->M * 16);
    if (w_reim && op->M) std::memcpy(w_reim, op->h_w.data(), op->M * 16);
    return BS_OK;
}

extern "C" int bs_op_destroy(bs_op_t op) {
    if (!op) return BS_OK;
    bs_plan_purge(op->id, 0);
    delete op;
    return BS_OK;
}
