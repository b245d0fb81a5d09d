// Builder of the v2 row plan (bs_rowplan.cuh): items / keys / strings tables, per-column u16 source
// tables, per-row valid alpha-mask lists and the launch geometry.
// PAPER.md:227-231 (Eq. 28, spin-split masks), PAPER.md:247 and 253-265 (phase factorisation).
#include <algorithm>
#include <map>

#include "bs_plan.cuh"
#include "bs_rowplan.cuh"

namespace {

// Thread-blocked column table: slot (chunk*threads + tid)*cpt + c of row `key` describes column
// col = chunk*chunk_cols + tid + c*threads: rank_B(tb ^ xb) | parity(zb0 & tb) << 15, or 0xFFFF if the column is
// outside the chunk / the row, or tb ^ xb leaves the sector.
__global__ void k_fill_ttab(SpinTab B, const uint2* __restrict__ keys, i64 tstride, int threads, int cpt,
                            int chunk_cols, unsigned short* __restrict__ T) {
    const i64 slot = blockIdx.x * (i64)blockDim.x + threadIdx.x;
    if (slot >= tstride) return;
    const uint2 k = keys[blockIdx.y];  // {xb, zb0}
    const i64 per_chunk = (i64)threads * cpt;
    const i64 chunk = slot / per_chunk, r = slot - chunk * per_chunk;
    const i64 tid = r / cpt, c = r - tid * cpt;
    const i64 lc = tid + c * threads;
    const i64 col = chunk * chunk_cols + lc;
    unsigned short e = 0xFFFFu;
    if (lc < chunk_cols && col < B.D) {
        const u32 tb = B.str[col];
        if (2 * __popc(tb & k.x) == __popc(k.x))
            e = (unsigned short)(spin_rank(B, tb ^ k.x) | ((u32)(__popc(tb & k.y) & 1) << 15));
    }
    T[(i64)blockIdx.y * tstride + slot] = e;
}

// l_max == 0: count the valid listed tables of every slot; else write the padded list
// Only entries whose source column lies in [w0, w0 + wn) are taken (one list per source-row window).
__global__ void k_list_build(const unsigned short* __restrict__ T, i64 tstride, int n_listed, int l_max, u32 pad_src,
                             u32 w0, u32 wn, u32* __restrict__ L, int* __restrict__ cnt) {
    const i64 slot = blockIdx.x * (i64)blockDim.x + threadIdx.x;
    if (slot >= tstride) return;
    int j = 0;
    for (int t = 0; t < n_listed; ++t) {
        const u32 e = T[(i64)t * tstride + slot];
        if (e == 0xFFFFu || ((e & 0x7FFFu) - w0) >= wn) continue;
        if (l_max) L[(i64)j * tstride + slot] = e | ((u32)t << 16);
        ++j;
    }
    if (!l_max) cnt[slot] = j;
    else for (; j < l_max; ++j) L[(i64)j * tstride + slot] = pad_src | ((u32)n_listed << 16);
}

// per-column constant of the diagonal group: cdiag[col] = sum_s w_s (-1)^{popc(zb_s & t_b)} over its strings whose weight
// does not depend on the row (z_a = 0: pure column-spin Z strings, e.g. the C(n,2) Z_q Z_q' pairs of a two-body H)
__global__ void k_cdiag(SpinTab B, const u32* __restrict__ zb, const double* __restrict__ w, int n,
                        double* __restrict__ cdiag) {
    const i64 col = blockIdx.x * (i64)blockDim.x + threadIdx.x;
    if (col >= B.D) return;
    const u32 tb = B.str[col];
    double f = 0.0;
    for (int s = 0; s < n; ++s) f += (__popc(__ldg(zb + s) & tb) & 1) ? -__ldg(w + s) : __ldg(w + s);
    cdiag[col] = f;
}

__global__ void k_row_count2(SpinTab A, const u32* __restrict__ xa, int n_xa, int* __restrict__ cnt) {
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

__global__ void k_row_fill2(SpinTab A, const u32* __restrict__ xa, const XaHdr* __restrict__ hdr, int n_xa,
                            const i64* __restrict__ off, uint4* __restrict__ ent) {
    i64 r = blockIdx.x * (i64)blockDim.x + threadIdx.x;
    if (r >= A.D) return;
    u32 ta = A.str[r];
    i64 o = off[r];
    u32 koff = 0;
    for (int i = 0; i < n_xa; ++i) {
        u32 m = __ldg(xa + i);
        if (2 * __popc(ta & m) == __popc(m)) {
            const u32 nk = hdr[i].key1 - hdr[i].key0;
            ent[o++] = make_uint4((u32)i, spin_rank(A, ta ^ m), koff, nk | ((hdr[i].stage & 1u) << 31) | (hdr[i].simple << 30));
            koff += nk;
        }
    }
}

}  // namespace

// groups: already z-reduced, oriented (xa = row-spin mask, xb = column-spin mask), sorted by (xa, xb).
// with_tables = false: headers / items / keys / strings and the per-row alpha-mask lists only (the K-resolved alpha-beta
// kernel of bs_kres.cu brings its own column tables): no list mode, no column tables.
int bs_rowplan_build(bs_rowplan* R, const std::vector<HostGroup>& groups_in, const SpinTab& A, const SpinTab& B,
                     cudaStream_t st, bool with_tables) {
    const i64 Da = A.D, Db = B.D;
    // ---- list mode: which alpha masks serve their single-key x_b != 0 groups from the column list -------------
    auto listable = [](const HostGroup& g) { return g.xb != 0 && g.s.front().zb == g.s.back().zb; };
    std::map<u32, int> n_listable;  // per xa
    for (auto& g : groups_in) n_listable[g.xa] += listable(g) ? 1 : 0;
    std::map<std::pair<u32, u32>, u32> listed_id;  // (xb, zb0) -> table id, listed tables first
    std::map<u32, bool> list_mode;
    for (auto& kv : n_listable) list_mode[kv.first] = with_tables && kv.second >= 8;
    for (int pass = 0; pass < 2; ++pass) {
        listed_id.clear();
        for (auto& g : groups_in)
            if (listable(g) && list_mode[g.xa])
                listed_id.emplace(std::make_pair(g.xb, g.s.front().zb), (u32)listed_id.size());
        if (pass == 0)  // drop masks that use only a small part of the list (their padding would dominate)
            for (auto& kv : n_listable)
                list_mode[kv.first] = list_mode[kv.first] && 10 * kv.second >= 3 * (int)listed_id.size();
    }
    if (listed_id.size() > 1024) {
        listed_id.clear();
        for (auto& kv : list_mode) kv.second = false;
    }
    // within an alpha mask: dense items first, listed items last (stable)
    std::vector<HostGroup> groups = groups_in;
    std::stable_sort(groups.begin(), groups.end(), [&](const HostGroup& a, const HostGroup& b) {
        if (a.xa != b.xa) return a.xa < b.xa;
        const int la = list_mode[a.xa] && listable(a), lb = list_mode[b.xa] && listable(b);
        return la < lb;
    });
    BS_REQUIRE(Db <= 32767, BS_ERR_ARG, "row plan: column space too large for u16 tables");
    // Diagonal group (x = 0): keys whose strings all have z_a = 0 and z_b != 0 carry a row-independent weight; when they
    // are many (two-body H: the C(n,2) pairs Z_q Z_q' of the column spin, 378 of 407 keys at configs[4]) their sum is a
    // per-COLUMN constant, tabulated once (k_cdiag) and added by the kernel; the item keeps its row-dependent keys, which
    // are then single-bit masks (bit test instead of POPC).  Real weights only; BS_NO_CDIAG (test hook) switches it off.
    std::vector<u32> cd_zb;
    std::vector<double> cd_w;
    int cdiag_group = -1;
    if (with_tables && !getenv("BS_NO_CDIAG"))
        for (size_t g = 0; g < groups.size(); ++g) {
            HostGroup& hg = groups[g];
            if (hg.xa != 0 || hg.xb != 0 || hg.s.front().zb != 0) continue;
            bool real = true;
            for (auto& st_ : hg.s) real &= st_.im == 0.0;
            if (!real) break;
            std::map<u32, bool> row_indep;   // per zb key: every string has z_a = 0
            for (auto& st_ : hg.s) {
                auto f = row_indep.find(st_.zb);
                if (f == row_indep.end()) row_indep[st_.zb] = st_.za == 0;
                else f->second = f->second && st_.za == 0;
            }
            int n_const = 0;
            for (auto& kv : row_indep) n_const += kv.first != 0 && kv.second;
            if (n_const < 8) break;
            std::vector<HostStr> keep;
            for (auto& st_ : hg.s) {
                if (st_.zb != 0 && row_indep[st_.zb]) {
                    cd_zb.push_back(st_.zb);
                    cd_w.push_back(st_.re);
                } else keep.push_back(st_);
            }
            hg.s.swap(keep);
            cdiag_group = (int)g;
            break;
        }
    std::vector<u32> xa_list, key_dz, key_s0, s_za;
    std::vector<XaHdr> hdrs;
    std::vector<RowItem> items;
    std::vector<double2> s_w;
    std::vector<uint2> tkeys(listed_id.size());
    std::map<std::pair<u32, u32>, u32> tkey_id = listed_id;
    for (auto& kv : listed_id) tkeys[kv.second] = make_uint2(kv.first.first, kv.first.second);
    const int n_listed = (int)listed_id.size();
    bool real_w = true;
    int max_keys = 0;
    for (size_t g = 0; g < groups.size(); ++g) {
        const HostGroup& hg = groups[g];
        if (g == 0 || hg.xa != groups[g - 1].xa) {
            if (!hdrs.empty()) {
                hdrs.back().item1 = (u32)items.size();
                hdrs.back().key1 = (u32)key_dz.size();
            }
            XaHdr h{};
            h.item0 = (u32)items.size();
            h.key0 = (u32)key_dz.size();
            h.stage = 0;
            h.item_split = 0xFFFFFFFFu;
            hdrs.push_back(h);
            xa_list.push_back(hg.xa);
        }
        // strings arrive sorted by (zb, za): bucket by zb
        RowItem it{};
        it.key0 = (u32)key_dz.size();
        it.single = 1;
        const u32 zb0 = hg.s.front().zb;
        for (size_t k = 0; k < hg.s.size(); ++k) {
            if (k == 0 || hg.s[k].zb != hg.s[k - 1].zb) {
                const u32 dz = hg.s[k].zb ^ zb0;
                key_dz.push_back(dz);
                key_s0.push_back((u32)s_za.size());
                if (k && __builtin_popcount(dz) != 1) it.single = 0;
            }
            s_za.push_back(hg.s[k].za);
            s_w.push_back(make_double2(hg.s[k].re, hg.s[k].im));
            if (hg.s[k].im != 0.0) real_w = false;
        }
        it.nkeys = (u32)key_dz.size() - it.key0;
        if ((int)g == cdiag_group) it.single |= 2u;   // the kernel adds cdiag[col]
        if (hg.xb == 0 && zb0 == 0) it.tkey = kTkeyIdent;
        else {
            auto key = std::make_pair(hg.xb, zb0);
            auto f = tkey_id.find(key);
            if (f == tkey_id.end()) {
                f = tkey_id.emplace(key, (u32)tkeys.size()).first;
                tkeys.push_back(make_uint2(hg.xb, zb0));
            }
            it.tkey = f->second;
        }
        if (hg.xb != 0) hdrs.back().stage = 1;
        if (list_mode[hg.xa] && listable(hg) && hdrs.back().item_split == 0xFFFFFFFFu) {
            hdrs.back().item_split = (u32)items.size();
            hdrs.back().key_split = it.key0;
        }
        items.push_back(it);
    }
    if (!hdrs.empty()) {
        hdrs.back().item1 = (u32)items.size();
        hdrs.back().key1 = (u32)key_dz.size();
    }
    key_s0.push_back((u32)s_za.size());
    for (auto& h : hdrs)
        if (h.item_split == 0xFFFFFFFFu) {
            h.item_split = h.item1;
            h.key_split = h.key1;
        }
    // stage bit 1: every listed group has a single string with z_a = 0 and the same weight -- AND the header owns
    // every listed table: the column list is the union over all list-mode alpha masks, and the uniform pass ignores
    // table ids, so a header with only a subset of the tables must take the sVx path (foreign tables: V = 0)
    for (auto& h : hdrs) {
        if (h.item_split >= h.item1) continue;
        bool unif = (int)(h.item1 - h.item_split) == n_listed;
        const u32 s_first = key_s0[items[h.item_split].key0];
        for (u32 i = h.item_split; i < h.item1 && unif; ++i) {
            const u32 k = items[i].key0, sa = key_s0[k], sb = key_s0[k + 1];
            unif = (sb - sa == 1) && s_za[sa] == 0 && s_w[sa].x == s_w[s_first].x && s_w[sa].y == s_w[s_first].y;
        }
        if (unif) h.stage |= 2u;
    }
    // "simple" alpha masks: one group with x_b = 0, no beta sign and a single key (pad[0] = 1)
    for (auto& h : hdrs) {
        const RowItem& it = items[h.item0];
        h.simple = (h.item1 - h.item0 == 1 && !h.stage && it.tkey == kTkeyIdent && it.nkeys == 1) ? 1u : 0u;
    }
    bool any_stage = false;
    for (auto& h : hdrs) {
        max_keys = std::max(max_keys, (int)(h.key1 - h.key0));
        any_stage |= h.stage != 0;
    }
    R->real_w = real_w;
    R->n_xa = (int)xa_list.size();
    R->n_items = (i64)items.size();
    R->n_keys = (i64)key_dz.size();
    R->n_strings = (i64)s_za.size();
    R->n_tkeys = (i64)tkeys.size();
    R->max_keys = max_keys;
    R->any_stage = any_stage;
    // ---- launch geometry ---------------------------------------------------------------------
    // Shared memory: [mbarrier 16 B][V slots: vcap * 16 B][list V slots: (n_listed + 1) * 16 B][row window].
    const int vcap = std::max(max_keys, 512);
    const size_t fixed = 16 + (size_t)vcap * 16 + (size_t)(n_listed + 1) * 16;
    const size_t smem_max = 227 * 1024 - 1024;
    i64 win = Db;
    int n_win = 1;
    if (any_stage) {
        i64 cap = (i64)((smem_max - fixed) / 16) - 1;
        if (const char* w = getenv("BS_ROW_WIN")) cap = std::max<i64>(8, std::min<i64>(cap, atoll(w)));  // tests
        if (Db > cap) {
            n_win = (int)((Db + cap - 1) / cap);
            win = (((Db + n_win - 1) / n_win) + 7) & ~i64(7);
        }
    } else win = 0;
    R->win_cols = (int)win;
    R->n_win = n_win;
    R->smem = fixed + (size_t)win * 16 + 16;  // + the zero amplitude behind the row (list padding)
    // threads / columns per thread: small rows -> several blocks per SM; big rows -> 1024 threads
    int threads, cpt;
    if (R->smem > 110 * 1024) threads = 1024;
    else if (R->smem > 56 * 1024 || Db >= 2048) threads = 512;
    else threads = 256;
    if (const char* t = getenv("BS_ROW_THREADS")) threads = std::max(64, std::min(1024, atoi(t)) & ~31);  // tuning / tests
    const i64 per_block_max = (i64)threads * 4;
    int n_chunks = (int)((Db + per_block_max - 1) / per_block_max);
    i64 chunk = ((Db + n_chunks - 1) / n_chunks + 31) & ~i64(31);
    cpt = (int)((chunk + threads - 1) / threads);
    while (threads > 64 && chunk <= threads / 2) threads /= 2;  // tiny rows
    cpt = (int)((chunk + threads - 1) / threads);
    R->threads = threads;
    R->cpt = cpt <= 1 ? 1 : 4;
    R->n_chunks = n_chunks;
    R->chunk_cols = (int)chunk;
    R->tstride = (i64)R->n_chunks * R->threads * R->cpt;
    if (!with_tables) R->tstride = 1;
    BS_REQUIRE((double)R->n_tkeys * (double)R->tstride * 2.0 <= 8e9, BS_ERR_ALLOC, "row plan: column tables too large");
    BS_REQUIRE(max_keys <= 2048, BS_ERR_ARG, "row plan: too many keys under one alpha mask");
    BS_CUDA(R->d_xa.upload(xa_list, st));
    BS_CUDA(R->d_xa_hdr.upload(hdrs, st));
    BS_CUDA(R->d_items.upload(items, st));
    BS_CUDA(R->d_key_dz.upload(key_dz, st));
    BS_CUDA(R->d_key_s0.upload(key_s0, st));
    BS_CUDA(R->d_s_za.upload(s_za, st));
    BS_CUDA(R->d_s_w.upload(s_w, st));
    DevBuf<uint2> d_tkeys;
    BS_CUDA(d_tkeys.upload(tkeys, st));
    BS_CUDA(R->d_ttab.alloc((size_t)std::max<i64>(1, R->n_tkeys) * R->tstride));
    for (i64 k0 = 0; with_tables && k0 < R->n_tkeys; k0 += 32768) {
        dim3 grid((unsigned)((R->tstride + 255) / 256), (unsigned)std::min<i64>(32768, R->n_tkeys - k0));
        k_fill_ttab<<<grid, 256, 0, st>>>(B, d_tkeys.p + k0, R->tstride, R->threads, R->cpt, R->chunk_cols,
                                          R->d_ttab.p + k0 * R->tstride);
        BS_COUNT_LAUNCH(1);
    }
    R->has_cdiag = cdiag_group >= 0;
    if (R->has_cdiag) {
        DevBuf<u32> d_zb;
        DevBuf<double> d_w;
        BS_CUDA(d_zb.upload(cd_zb, st));
        BS_CUDA(d_w.upload(cd_w, st));
        BS_CUDA(R->d_cdiag.alloc(Db));
        k_cdiag<<<(unsigned)((Db + 255) / 256), 256, 0, st>>>(B, d_zb.p, d_w.p, (int)cd_zb.size(), R->d_cdiag.p);
        BS_COUNT_LAUNCH(1);
        BS_CUDA(cudaStreamSynchronize(st));   // the uploads' sources and device buffers die here
    }
    // column list: compaction of the listed tables over table ids
    R->n_listed = n_listed;
    R->h_hdrs = hdrs;
    R->h_items = items;
    R->h_tkeys = tkeys;
    R->h_xa = xa_list;
    R->h_key_dz = key_dz;
    if (!with_tables) {   // the K-resolved plan folds single-string keys into its own tables
        R->h_key_s0 = key_s0;
        R->h_s_za = s_za;
        R->h_s_w = s_w;
    }
    R->l_max = 0;
    if (n_listed > 0) {
        DevBuf<int> lcnt;
        BS_CUDA(lcnt.alloc(R->tstride));
        const unsigned lb = (unsigned)((R->tstride + 255) / 256);
        std::vector<int> hl(R->tstride);
        // With windowed source rows every window gets its own list (only the entries whose source lies in it), so a
        // window pass walks its own entries instead of the whole list with a window test per entry. Padding entries
        // point at the zero amplitude behind the staged window (column w0 + win_cols: must fit the 15-bit source field).
        const bool split = n_win > 1 && (i64)n_win * win <= 32767 && !getenv("BS_ROW_NO_SPLIT");
        const int n_lists = split ? n_win : 1;
        std::vector<int> woff(n_lists + 1, 0), wcnt;
        for (int w = 0; w < n_lists; ++w) {
            const u32 w0 = split ? (u32)(w * win) : 0u, wn = split ? (u32)win : 0xFFFFFFFFu;
            k_list_build<<<lb, 256, 0, st>>>(R->d_ttab.p, R->tstride, n_listed, 0, 0u, w0, wn, nullptr, lcnt.p);
            BS_CUDA(cudaMemcpyAsync(hl.data(), lcnt.p, R->tstride * 4, cudaMemcpyDeviceToHost, st));
            BS_CUDA(cudaStreamSynchronize(st));
            int m = 0;
            for (int v : hl) m = std::max(m, v);
            // slots a block of column chunk c has to walk in this window: the longest list among its own columns
            const i64 per_chunk = (i64)R->threads * R->cpt;
            for (int c = 0; c < R->n_chunks; ++c) {
                int mc = 0;
                for (i64 sl = c * per_chunk; sl < (c + 1) * per_chunk; ++sl) mc = std::max(mc, hl[sl]);
                wcnt.push_back(mc);
            }
            woff[w + 1] = woff[w] + m;
            R->l_max = std::max(R->l_max, m);
        }
        BS_CUDA(R->d_ltab.alloc((size_t)std::max(1, woff[n_lists]) * R->tstride));
        for (int w = 0; w < n_lists; ++w) {
            const int m = woff[w + 1] - woff[w];
            if (m == 0) continue;
            const u32 w0 = split ? (u32)(w * win) : 0u, wn = split ? (u32)win : 0xFFFFFFFFu;
            k_list_build<<<lb, 256, 0, st>>>(R->d_ttab.p, R->tstride, n_listed, m, split ? w0 + (u32)win : (u32)Db, w0, wn,
                                             R->d_ltab.p + (size_t)woff[w] * R->tstride, lcnt.p);
        }
        BS_COUNT_LAUNCH(2 * n_lists);
        if (split) {  // [window offsets (n_win + 1)][slots per (window, chunk)]
            woff.insert(woff.end(), wcnt.begin(), wcnt.end());
            BS_CUDA(R->d_lwoff.upload(woff, st));
        }
        R->l_split = split;
    }
    // per-row valid alpha masks
    DevBuf<int> cnt;
    BS_CUDA(cnt.alloc(Da));
    BS_CUDA(R->d_row_off.alloc(Da + 1));
    const unsigned nb = (unsigned)((Da + 127) / 128);
    k_row_count2<<<nb, 128, 0, st>>>(A, R->d_xa.p, R->n_xa, cnt.p);
    std::vector<int> hcnt(Da);
    BS_CUDA(cudaMemcpyAsync(hcnt.data(), cnt.p, Da * 4, cudaMemcpyDeviceToHost, st));
    BS_CUDA(cudaStreamSynchronize(st));
    std::vector<i64> hoff(Da + 1, 0);
    for (i64 r = 0; r < Da; ++r) hoff[r + 1] = hoff[r] + hcnt[r];
    R->n_row_ent = hoff[Da];
    BS_CUDA(cudaMemcpyAsync(R->d_row_off.p, hoff.data(), (Da + 1) * 8, cudaMemcpyHostToDevice, st));
    BS_CUDA(R->d_row_ent.alloc(std::max<i64>(1, R->n_row_ent)));
    k_row_fill2<<<nb, 128, 0, st>>>(A, R->d_xa.p, R->d_xa_hdr.p, R->n_xa, R->d_row_off.p, R->d_row_ent.p);
    BS_COUNT_LAUNCH(2);
    BS_CUDA(cudaGetLastError());
    BS_CUDA(cudaStreamSynchronize(st));  // host vectors go out of scope

    RowPlanDev& d = R->dev;
    d.A = A;
    d.B = B;
    d.row_off = R->d_row_off.p;
    d.row_ent = R->d_row_ent.p;
    d.xa_hdr = R->d_xa_hdr.p;
    d.items = R->d_items.p;
    d.key_dz = R->d_key_dz.p;
    d.key_s0 = R->d_key_s0.p;
    d.s_za = R->d_s_za.p;
    d.s_w = R->d_s_w.p;
    d.ttab = R->d_ttab.p;
    d.tstride = R->tstride;
    d.max_keys = vcap;
    d.win_cols = R->win_cols;
    d.n_win = R->n_win;
    d.chunk_cols = R->chunk_cols;
    d.ltab = R->d_ltab.p;
    d.l_max = R->l_max;
    d.l_woff = R->l_split ? R->d_lwoff.p : nullptr;
    d.l_nchunks = R->n_chunks;
    d.n_listed = n_listed;
    d.cdiag = R->has_cdiag ? R->d_cdiag.p : nullptr;
    return BS_OK;
}
