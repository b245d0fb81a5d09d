// Plan builder: turns the canonical group tables of an operator (a2) into the sector-specific
// layout the apply kernels stream (spin-split masks, z-reduction, per-row valid alpha masks).
// PAPER.md:227-231 (Eq. 28: X_g = (X_ga, X_gb), Z_k = (Z_ka, Z_kb)), PAPER.md:247 (factorised phase).
#include <cub/cub.cuh>

#include <algorithm>

#include "bs_k2.cuh"
#include "bs_kres.cuh"
#include "bs_plan.cuh"
#include "bs_rowplan.cuh"

namespace {

std::mutex g_plan_mu;
std::map<std::pair<u64, u64>, bs_plan*> g_plans;

// count / fill the valid alpha masks of every target alpha row: mask xa is valid for row string ta
// iff ta ^ xa has the same popcount, i.e. 2 popc(ta & xa) = popc(xa).  One thread per row walks
// the masks in ascending order, so the list order (and hence the summation order) is fixed.
__global__ void k_row_count(SpinTab A, const u32* __restrict__ xa, int n_xa, int* __restrict__ cnt) {
    i64 r = blockIdx.x * (i64)blockDim.x + threadIdx.x;
    if (r >= A.D) return;
    u32 ta = A.str[r];
    int c = 0;
    for (int i = 0; i < n_xa; ++i) {
        u32 m = __ldg(xa + i);
        c += (2 * __popc(ta & m) == __popc(m));
    }
    cnt[r] = c;
}

__global__ void k_row_fill(SpinTab A, const u32* __restrict__ xa, int n_xa, const i64* __restrict__ off,
                           uint2* __restrict__ ent) {
    i64 r = blockIdx.x * (i64)blockDim.x + threadIdx.x;
    if (r >= A.D) return;
    u32 ta = A.str[r];
    i64 o = off[r];
    for (int i = 0; i < n_xa; ++i) {
        u32 m = __ldg(xa + i);
        if (2 * __popc(ta & m) == __popc(m)) ent[o++] = make_uint2((u32)i, spin_rank(A, ta ^ m));
    }
}

// v2 row plans.  B groups (xa = 0, xb != 0) stay in the main plan (same-row gathers from the staged
// row) when they are few; when they are many (molecular Hamiltonians: all beta single and double
// excitations) they are applied as A groups of the transposed problem, where the gather becomes a
// coalesced row read.  Any failure (tables too large, ...) leaves the v1 kernel in charge.
void build_row_plans(bs_plan* P, const std::vector<HostGroup>& groups, bs_sector* S, cudaStream_t st) {
    const char* force = getenv("BS_KERNEL");
    if (force && std::string(force) == "v1") return;
    if (S->Da > 32767 || S->Db > 32767) return;
    size_t nB = 0;
    for (auto& g : groups) nB += (g.xa == 0 && g.xb != 0);
    const bool transposed_b = nB > 64 && !(force && std::string(force) == "v2inrow");
    std::vector<HostGroup> main_g, t_g;
    auto to_transposed = [&](u32 xb, const std::vector<HostStr>& strs) {
        HostGroup t;
        t.xa = xb;
        t.xb = 0;
        for (auto& s : strs) t.s.push_back(HostStr{s.zb, s.za, s.re, s.im});
        std::stable_sort(t.s.begin(), t.s.end(), [](const HostStr& a, const HostStr& b) {
            return a.zb < b.zb || (a.zb == b.zb && a.za < b.za);
        });
        t_g.push_back(std::move(t));
    };
    // Beta single hops (x_a = 0, x_b = {r, s}) of a two-body Hamiltonian carry two kinds of strings: the JW chain between
    // r and s, alone or with one ALPHA Z (alpha spectator densities: F depends on t_a, not on the other beta electrons),
    // and the chain with one more BETA Z and no alpha Z (beta spectators: F depends on t_b only).  The first kind is an
    // alpha-beta coupling with the identity as its alpha move: it joins the K-resolved kernel as one more entry per row
    // (G[s][r] = A_rs(t_a)).  The second kind is the same sparse matrix for every alpha row: on the transposed problem it
    // is a plain row axpy with one scalar per (t_b, hop).  Without the split the group is a 1 + n-key item per non-zero.
    const bool hop_split = transposed_b && !getenv("BS_NO_KRES") && !getenv("BS_NO_HOPSPLIT");
    bool any_split = false;
    for (auto& g : groups) {
        if (transposed_b && g.xa == 0 && g.xb != 0) {
            bool done = false;
            if (hop_split && __builtin_popcount(g.xb) == 2) {
                const int lo = __builtin_ctz(g.xb), hi = 31 - __builtin_clz(g.xb);
                const u32 between = ((1u << hi) - 1u) & ~((2u << lo) - 1u);
                std::vector<HostStr> part_a, part_b;
                bool ok = true;
                u32 zb_chain = 0;
                bool have_chain = false;
                for (auto& st_ : g.s)
                    if ((st_.zb & ~g.xb) == between && (!have_chain || st_.zb == zb_chain)) {
                        zb_chain = st_.zb;
                        have_chain = true;
                    }
                for (auto& st_ : g.s) {
                    if (have_chain && st_.zb == zb_chain) part_a.push_back(st_);
                    else {
                        part_b.push_back(st_);
                        ok &= st_.za == 0;
                    }
                    ok &= st_.im == 0.0;
                }
                if (ok && have_chain && !part_a.empty()) {
                    HostGroup a;
                    a.xa = 0;
                    a.xb = g.xb;
                    a.s = part_a;
                    main_g.push_back(std::move(a));
                    if (!part_b.empty()) to_transposed(g.xb, part_b);
                    done = any_split = true;
                }
            }
            if (!done) to_transposed(g.xb, g.s);
        } else main_g.push_back(g);
    }
    std::stable_sort(main_g.begin(), main_g.end(), [](const HostGroup& a, const HostGroup& b) {
        return a.xa < b.xa || (a.xa == b.xa && a.xb < b.xb);
    });
    std::stable_sort(t_g.begin(), t_g.end(), [](const HostGroup& a, const HostGroup& b) { return a.xa < b.xa; });
    // alpha-beta groups with JW chains: K-resolved kernel (bs_kres.cuh); what it takes leaves main_g
    bs_kres* kres = nullptr;
    if (bs_kres_build(main_g, S, st, &kres, any_split) != BS_OK) {
        cudaGetLastError();
        kres = nullptr;
        P->rows_fallback = 1;
        return;
    }
    // same-spin double excitations: dense blocks over (N - 2)-electron strings (bs_k2.cuh); what they take leaves the lists
    bs_k2 *k2m = nullptr, *k2t = nullptr;
    if (bs_k2_build(main_g, S->h_sa, S->n_orb, S->n_alpha, S->Db, st, &k2m) != BS_OK ||
        (!t_g.empty() && bs_k2_build(t_g, S->h_sb, S->n_orb, S->n_beta, S->Da, st, &k2t) != BS_OK)) {
        cudaGetLastError();
        delete kres;
        delete k2m;
        delete k2t;
        P->rows_fallback = 1;
        return;
    }
    bs_rowplan* m = new (std::nothrow) bs_rowplan;
    bs_rowplan* t = t_g.empty() ? nullptr : new (std::nothrow) bs_rowplan;
    bool ok = m && (t_g.empty() || t);
    if (ok) ok = bs_rowplan_build(m, main_g, S->ta, S->tb, st) == BS_OK;
    if (ok && t) ok = bs_rowplan_build(t, t_g, S->tb, S->ta, st) == BS_OK;
    if (!ok) {
        cudaGetLastError();
        bs_rowplan_free(m);
        bs_rowplan_free(t);
        delete kres;
        delete k2m;
        delete k2t;
        P->rows_fallback = 1;   // queryable: bs_plan_describe says "fallback=1"
        return;
    }
    if (!t && !kres && !k2m && bs_light_build(m, st) != BS_OK) cudaGetLastError();  // optional fast path; k_rows stays available
    P->rp_main = m;
    P->rp_t = t;
    P->kres = kres;
    P->k2_main = k2m;
    P->k2_t = k2t;
}

int build_sector_plan(bs_plan* P, bs_op* op, bs_sector* S, cudaStream_t st) {
    const int n = S->n_orb;
    const u64 mask_a = (n == 64) ? ~u64(0) : ((u64(1) << n) - 1);
    std::vector<HostGroup> groups;
    groups.reserve(op->G);
    bool real_w = true;
    for (i64 g = 0; g < op->G; ++g) {
        u64 x = op->h_xg[g];
        u32 xa = (u32)(x & mask_a), xb = (u32)(x >> n);
        int pa = __builtin_popcount(xa), pb = __builtin_popcount(xb);
        if ((pa & 1) || (pb & 1)) continue;  // can never conserve N_alpha / N_beta
        if (pa / 2 > std::min(S->n_alpha, n - S->n_alpha) || pb / 2 > std::min(S->n_beta, n - S->n_beta)) continue;
        HostGroup hg;
        hg.xa = xa;
        hg.xb = xb;
        double sga = ((pa / 2) & 1) ? -1.0 : 1.0, sgb = ((pb / 2) & 1) ? -1.0 : 1.0;
        for (i64 k = op->h_offs[g]; k < op->h_offs[g + 1]; ++k) {
            u64 z = op->h_z[k];
            HostStr s{(u32)(z & mask_a), (u32)(z >> n), op->h_w[2 * k], op->h_w[2 * k + 1]};
            // z-reduction modulo x (exact on valid targets, see bs_plan.cuh)
            if ((s.za ^ xa) < s.za) { s.za ^= xa; s.re *= sga; s.im *= sga; }
            if ((s.zb ^ xb) < s.zb) { s.zb ^= xb; s.re *= sgb; s.im *= sgb; }
            hg.s.push_back(s);
        }
        std::stable_sort(hg.s.begin(), hg.s.end(), [](const HostStr& a, const HostStr& b) {
            return a.zb < b.zb || (a.zb == b.zb && a.za < b.za);
        });
        std::vector<HostStr> m;
        for (auto& s : hg.s) {
            if (!m.empty() && m.back().za == s.za && m.back().zb == s.zb) {
                m.back().re += s.re;
                m.back().im += s.im;
            } else m.push_back(s);
        }
        hg.s.clear();
        for (auto& s : m)
            if (s.re != 0.0 || s.im != 0.0) {
                hg.s.push_back(s);
                if (s.im != 0.0) real_w = false;
            }
        if (!hg.s.empty()) groups.push_back(std::move(hg));
    }
    std::stable_sort(groups.begin(), groups.end(), [](const HostGroup& a, const HostGroup& b) {
        return a.xa < b.xa || (a.xa == b.xa && a.xb < b.xb);
    });
    build_row_plans(P, groups, S, st);
    P->real_w = real_w;
    if (P->rp_main) return BS_OK;  // the v1 tables below are only needed when the v2 row plan could not be built
    std::vector<u32> xa_list, ga_off;
    std::vector<uint4> hdr;
    std::vector<uint2> szab;
    std::vector<double2> sw;
    for (size_t g = 0; g < groups.size(); ++g) {
        if (g == 0 || groups[g].xa != groups[g - 1].xa) {
            xa_list.push_back(groups[g].xa);
            ga_off.push_back((u32)g);
        }
        hdr.push_back(make_uint4(groups[g].xb, (u32)szab.size(), (u32)groups[g].s.size(),
                                 (u32)__builtin_popcount(groups[g].xb)));
        for (auto& s : groups[g].s) {
            szab.push_back(make_uint2(s.za, s.zb));
            sw.push_back(make_double2(s.re, s.im));
        }
    }
    ga_off.push_back((u32)groups.size());
    P->real_w = real_w;
    P->n_xa = (int)xa_list.size();
    P->n_groups = (i64)groups.size();
    P->n_strings = (i64)szab.size();
    BS_CUDA(P->d_xa.upload(xa_list, st));
    BS_CUDA(P->d_ga_off.upload(ga_off, st));
    BS_CUDA(P->d_ghdr.upload(hdr, st));
    BS_CUDA(P->d_szab.upload(szab, st));
    BS_CUDA(P->d_sw.upload(sw, st));

    // per-row valid alpha masks
    const i64 Da = S->Da;
    DevBuf<int> cnt;
    DevBuf<i64> cnt64;
    BS_CUDA(cnt.alloc(Da));
    BS_CUDA(P->d_row_off.alloc(Da + 1));
    unsigned nb = (unsigned)((Da + 127) / 128);
    k_row_count<<<nb, 128, 0, st>>>(S->ta, P->d_xa.p, P->n_xa, cnt.p);
    std::vector<int> hcnt(Da);
    BS_CUDA(cudaMemcpyAsync(hcnt.data(), cnt.p, Da * 4, cudaMemcpyDeviceToHost, st));
    BS_CUDA(cudaStreamSynchronize(st));
    std::vector<i64> hoff(Da + 1, 0);
    int mx = 0;
    for (i64 r = 0; r < Da; ++r) {
        hoff[r + 1] = hoff[r] + hcnt[r];
        mx = std::max(mx, hcnt[r]);
    }
    P->n_row_ent = hoff[Da];
    P->max_row_ent = mx;
    BS_CUDA(cudaMemcpyAsync(P->d_row_off.p, hoff.data(), (Da + 1) * 8, cudaMemcpyHostToDevice, st));
    BS_CUDA(P->d_row_ent.alloc(P->n_row_ent));
    k_row_fill<<<nb, 128, 0, st>>>(S->ta, P->d_xa.p, P->n_xa, P->d_row_off.p, P->d_row_ent.p);
    BS_COUNT_LAUNCH(2);
    BS_CUDA(cudaGetLastError());
    BS_CUDA(cudaStreamSynchronize(st));
    return BS_OK;
}

int build_full_plan(bs_plan* P, bs_op* op, cudaStream_t st, int max_strings) {
    // fixed-size chunks over the string stream; a chunk may split a group (the kernel gathers the
    // source amplitude once per piece, which is linear and therefore exact).  Every group owns at
    // least one string, so a chunk touches at most max_strings groups.
    i64 M = op->M, G = op->G;
    bool real_w = true;
    for (i64 k = 0; k < M; ++k)
        if (op->h_w[2 * k + 1] != 0.0) real_w = false;
    P->real_w = real_w;
    i64 g = 0;
    for (i64 s = 0; s < M; s += max_strings) {   // max_strings is even: s0 stays 16-byte aligned
        i64 e = std::min(M, s + max_strings);
        while (op->h_offs[g + 1] <= s) ++g;
        i64 ge = g;
        while (ge + 1 < G && op->h_offs[ge + 1] < e) ++ge;
        P->h_chunks.push_back(FullChunk{(int)g, (int)ge, (int)s, (int)e});
    }
    P->n_chunks = (int)P->h_chunks.size();
    BS_CUDA(P->d_chunks.upload(P->h_chunks, st));
    BS_CUDA(cudaStreamSynchronize(st));
    return BS_OK;
}

}  // namespace

// full-space staging capacities (must match bs_apply.cu)
extern const int kFullChunkStrings = 512;

int bs_plan_get(bs_op* op, bs_sector* s, cudaStream_t st, bs_plan** out) {
    std::lock_guard<std::mutex> lk(g_plan_mu);
    auto key = std::make_pair(op->id, s->id);
    auto it = g_plans.find(key);
    if (it != g_plans.end()) {
        *out = it->second;
        return BS_OK;
    }
    BS_REQUIRE(op->n_qubits == s->n_qubits, BS_ERR_MISMATCH, "operator has %d qubits, sector has %d", op->n_qubits,
               s->n_qubits);
    bs_plan* P = new (std::nothrow) bs_plan;
    BS_REQUIRE(P, BS_ERR_ALLOC, "plan allocation failed");
    P->op_id = op->id;
    P->sector_id = s->id;
    P->full = s->full;
    int rc = s->full ? build_full_plan(P, op, st, kFullChunkStrings) : build_sector_plan(P, op, s, st);
    if (rc != BS_OK) {
        delete P;
        return rc;
    }
    g_plans[key] = P;
    *out = P;
    return BS_OK;
}

bs_plan::~bs_plan() {
    bs_rowplan_free(rp_main);
    bs_rowplan_free(rp_t);
    delete kres;
    delete k2_main;
    delete k2_t;
}
void bs_rowplan_free(bs_rowplan* R) { delete R; }

void bs_plan_purge(u64 op_id, u64 sector_id) {
    std::lock_guard<std::mutex> lk(g_plan_mu);
    for (auto it = g_plans.begin(); it != g_plans.end();) {
        if ((op_id && it->first.first == op_id) || (sector_id && it->first.second == sector_id)) {
            delete it->second;
            it = g_plans.erase(it);
        } else ++it;
    }
}

extern "C" int bs_plan_info(bs_op_t op, bs_sector_t s, int64_t info[8], void* cuda_stream) {
    BS_REQUIRE(op && s && info, BS_ERR_ARG, "bs_plan_info: bad argument");
    bs_plan* P = nullptr;
    int rc = bs_plan_get(op, s, (cudaStream_t)cuda_stream, &P);
    if (rc != BS_OK) return rc;
    for (int i = 0; i < 8; ++i) info[i] = 0;
    info[0] = P->full ? 0 : (!P->rp_main ? 1 : (P->rp_main->light && !P->rp_t && !P->kres ? 3 : 2));
    info[1] = P->rows_fallback;
    info[2] = P->rp_t ? 1 : 0;
    info[3] = P->kres ? 1 : 0;
    info[4] = (P->rp_t || P->kres || P->k2_main) ? 3 * 16 * s->D : 0;
    info[5] = P->kres ? (int64_t)P->kres->slab_rows * P->kres->n * P->kres->DKp * 16 : 0;
    for (const bs_k2* K2 : {P->k2_main, P->k2_t})
        if (K2) info[5] += (int64_t)K2->F * K2->P * K2->slab_cols * 16;
    if (P->rp_main) {
        info[6] = P->rp_main->max_keys;
        info[7] = P->rp_main->n_items + (P->rp_t ? P->rp_t->n_items : 0) + (P->kres ? P->kres->rp->n_items : 0) +
                  (P->k2_main ? P->k2_main->n_groups : 0) + (P->k2_t ? P->k2_t->n_groups : 0);
    }
    return BS_OK;
}

extern "C" int bs_plan_groups(bs_op_t op, bs_sector_t s, uint64_t* x, int32_t* nkeys, int64_t cap, int64_t* n_groups,
                              void* cuda_stream) {
    BS_REQUIRE(op && s && n_groups, BS_ERR_ARG, "bs_plan_groups: bad argument");
    bs_plan* P = nullptr;
    int rc = bs_plan_get(op, s, (cudaStream_t)cuda_stream, &P);
    if (rc != BS_OK) return rc;
    BS_REQUIRE(!P->full && P->rp_main, BS_ERR_ARG, "bs_plan_groups: needs a sector-mode v2 plan");
    int64_t n = 0;
    auto emit = [&](const bs_rowplan* R, bool transposed) {
        if (!R) return;
        for (size_t h = 0; h < R->h_hdrs.size(); ++h)
            for (u32 i = R->h_hdrs[h].item0; i < R->h_hdrs[h].item1; ++i) {
                const RowItem& it = R->h_items[i];
                const u64 xr = R->h_xa[h], xc = it.tkey == kTkeyIdent ? 0u : R->h_tkeys[it.tkey].x;   // row / column spin
                if (x && nkeys && n < cap) {
                    x[n] = transposed ? (xc | (xr << s->n_orb)) : (xr | (xc << s->n_orb));
                    nkeys[n] = (int32_t)it.nkeys;
                }
                ++n;
            }
    };
    emit(P->rp_main, false);
    emit(P->kres ? P->kres->rp : nullptr, false);
    emit(P->rp_t, true);
    for (const bs_k2* K2 : {P->k2_main, P->k2_t})   // same-spin doubles: one key each
        if (K2)
            for (u32 xr : K2->h_x) {
                if (x && nkeys && n < cap) {
                    x[n] = K2 == P->k2_t ? ((u64)xr << s->n_orb) : (u64)xr;
                    nkeys[n] = 1;
                }
                ++n;
            }
    *n_groups = n;
    return BS_OK;
}

extern "C" int bs_plan_describe(bs_op_t op, bs_sector_t s, char* buf, int64_t n, void* cuda_stream) {
    BS_REQUIRE(op && s && buf && n > 0, BS_ERR_ARG, "bs_plan_describe: bad argument");
    bs_plan* P = nullptr;
    int rc = bs_plan_get(op, s, (cudaStream_t)cuda_stream, &P);
    if (rc != BS_OK) return rc;
    if (P->full) {
        snprintf(buf, (size_t)n, "kernel=full chunks=%d real_w=%d", P->n_chunks, (int)P->real_w);
    } else if (P->rp_main) {
        const bs_rowplan* M = P->rp_main;
        const bs_rowplan* T = P->rp_t;
        int w = snprintf(buf, (size_t)n,
                         "kernel=rows_v2%s fallback=0 real_w=%d main{xa=%d items=%lld keys=%lld strings=%lld tkeys=%lld max_keys=%d "
                         "row_ent=%lld threads=%d cpt=%d chunk_cols=%d win_cols=%d n_win=%d smem=%zu listed=%d l_max=%d}",
                         M->light ? "+light" : "", (int)M->real_w, M->n_xa, (long long)M->n_items, (long long)M->n_keys, (long long)M->n_strings,
                         (long long)M->n_tkeys, M->max_keys, (long long)M->n_row_ent, M->threads, M->cpt, M->chunk_cols,
                         M->win_cols, M->n_win, M->smem, M->n_listed, M->l_max);
        if (P->kres && w > 0 && w < n) {
            const bs_kres* K = P->kres;
            w += snprintf(buf + w, (size_t)(n - w),
                          " kres{xa=%d keys=%lld DK=%lld KC=%d chunks=%d NP=%d smem=%zu stages=%d staged_rows=%.2f max_segs=%d slab_rows=%lld "
                          "scratch_MB=%.0f}",
                          K->rp->n_xa, (long long)K->rp->n_keys, (long long)K->DK, K->KC, K->n_chunks, K->NP, K->smem,
                          K->n_stages, K->staged_rows, K->max_segs, (long long)K->slab_rows,
                          (double)K->slab_rows * K->n * K->DKp * 16.0 / 1048576.0);
        }
        for (const bs_k2* K2 : {P->k2_main, P->k2_t})
            if (K2 && w > 0 && w < n)
                w += snprintf(buf + w, (size_t)(n - w),
                              " k2%s{groups=%lld families=%d P=%d tile=%d tiles=%d smem=%zu slab_cols=%lld scratch_MB=%.0f}",
                              K2 == P->k2_t ? "_t" : "", (long long)K2->n_groups, K2->F, K2->P, K2->rt, K2->n_tiles, K2->smem,
                              (long long)K2->slab_cols, (double)K2->F * K2->P * K2->slab_cols * 16.0 / 1048576.0);
        if (T && w > 0 && w < n)
            snprintf(buf + w, (size_t)(n - w),
                     " transposed{xa=%d items=%lld keys=%lld strings=%lld tkeys=%lld max_keys=%d row_ent=%lld threads=%d "
                     "cpt=%d chunk_cols=%d smem=%zu}",
                     T->n_xa, (long long)T->n_items, (long long)T->n_keys, (long long)T->n_strings, (long long)T->n_tkeys,
                     T->max_keys, (long long)T->n_row_ent, T->threads, T->cpt, T->chunk_cols, T->smem);
    } else {
        snprintf(buf, (size_t)n, "kernel=sector_v1 fallback=%d real_w=%d xa=%d groups=%lld strings=%lld row_ent=%lld",
                 P->rows_fallback, (int)P->real_w, P->n_xa, (long long)P->n_groups, (long long)P->n_strings,
                 (long long)P->n_row_ent);
    }
    return BS_OK;
}
