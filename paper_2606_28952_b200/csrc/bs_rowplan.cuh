// v2 "row plan": sector-specific tables of one (operator, sector) pair for the row kernel
// (bs_rowkernel.cu).  See DESIGN.md "Apply kernel v2".
//
// Groups are split by (xa, xb) = (alpha part, beta part) of their X mask (Eq. 28):
//   D  xa = 0, xb = 0   diagonal
//   B  xa = 0, xb != 0  source in the same row, another column
//   A  xa != 0, xb = 0  source in another row, same column (coalesced, no gather)
//   AB both             source in another row, another column
// Phase factorisation: within a group, strings are bucketed by their beta Z
// mask ("keys"): F_g(ta, tb) = sum_j V_gj(ta) (-1)^{popc(zb_gj & tb)},
// V_gj(ta) = sum_{k: zb_k = zb_gj} w_k (-1)^{popc(za_k & ta)}.  V is evaluated once per (row, group)
// into shared memory; the per-target work is one term per KEY, not per string.
// Column tables: for every distinct (xb, zb_g0) pair a u16 table T[col] = source column | sign << 15
// (0xFFFF: tb ^ xb leaves the sector) replaces the per-target validity test, rank and first POPC.
#pragma once
#include "bs_internal.cuh"

constexpr u32 kTkeyIdent = 0xFFFFFFFFu;  // xb = 0 and zb_g0 = 0: source column = target column, sign +

struct __align__(16) XaHdr {
    u32 item0, item1;  // items (groups) under this alpha mask
    u32 key0, key1;    // their keys, contiguous: V slot of key k is k - key0
    u32 stage;         // 1: some item has xb != 0 -> the source row is staged in shared memory
    u32 simple;        // 1: one group, x_b = 0, no beta sign, one key: a plain row axpy
    u32 item_split;    // items [item_split, item1) are single-key x_b != 0 groups served by the column LIST
    u32 key_split;     // first key of those items (they own one key each, in item order)
};
struct __align__(16) RowItem {
    u32 tkey;   // column table id or kTkeyIdent
    u32 key0;   // first key (global index)
    u32 nkeys;  // >= 1
    u32 single; // bit 0: every dz of keys 1.. has exactly one bit (bit test instead of POPC); bit 1: add cdiag[col]
};

// device view handed to the kernel by value
struct RowPlanDev {
    SpinTab A, B;               // row strings (A) and column strings (B); swapped in the transposed plan
    const i64* row_off;         // [Da + 1]
    const uint4* row_ent;       // {xa id, source row, V-slot offset within the row (prefix sum of key counts),
                                //  key count | stage << 31}
    const XaHdr* xa_hdr;
    const RowItem* items;
    const u32* key_dz;          // [n_keys] zb_key ^ zb_g0
    const u32* key_s0;          // [n_keys + 1] string range of each key
    const u32* s_za;            // [n_strings]
    const double2* s_w;         // [n_strings]
    const unsigned short* ttab; // [n_tkeys][tstride], thread-blocked: slot (chunk*threads + tid)*cpt + c holds
                                // column chunk*chunk_cols + tid + c*threads (0xFFFF beyond the chunk / row)
    i64 tstride;
    int max_keys;               // V slots in shared memory (>= max keys under one alpha mask)
    int win_cols;               // columns of a source row staged at once (>= Db: whole row)
    int n_win;                  // number of windows
    int chunk_cols;             // target columns per thread block
    // Column list (compaction of the listed column tables over table ids): entry j of slot s is
    // source column | sign << 15 | table id << 16; padded with (0, 0, n_listed) whose V slot is always 0.
    const u32* ltab;            // [l_max][tstride]; with l_woff: window w owns list slots [l_woff[w], l_woff[w + 1])
    const int* l_woff;          // nullptr: one list for all windows (entries carry a window test); then per (window, chunk) slot counts
    int l_nchunks;
    int l_max, n_listed;
    const double* cdiag;        // [Db] row-independent part of the diagonal group (items with single & 2), or nullptr
};

struct bs_rowplan {
    bool real_w = true;
    i64 n_items = 0, n_keys = 0, n_strings = 0, n_tkeys = 0, n_row_ent = 0;
    int n_xa = 0, max_keys = 0;
    bool any_stage = false;
    DevBuf<u32> d_xa;
    DevBuf<XaHdr> d_xa_hdr;
    DevBuf<RowItem> d_items;
    DevBuf<u32> d_key_dz, d_key_s0, d_s_za;
    DevBuf<double2> d_s_w;
    DevBuf<unsigned short> d_ttab;
    DevBuf<u32> d_ltab;
    DevBuf<double> d_cdiag;
    bool has_cdiag = false;
    DevBuf<int> d_lwoff;
    bool l_split = false;
    int l_max = 0, n_listed = 0;
    DevBuf<i64> d_row_off;
    DevBuf<uint4> d_row_ent;
    i64 tstride = 0;
    // launch geometry
    int threads = 256, cpt = 1, n_chunks = 1, chunk_cols = 0, win_cols = 0, n_win = 1;
    size_t smem = 0;
    RowPlanDev dev{};
    // host copies kept for the light-plan builder (bs_light.cu)
    std::vector<XaHdr> h_hdrs;
    std::vector<RowItem> h_items;
    std::vector<uint2> h_tkeys;  // {xb, zb0} of every column table, listed ones first
    std::vector<u32> h_xa;
    std::vector<u32> h_key_dz, h_key_s0, h_s_za;
    std::vector<double2> h_s_w;
    // ---- light path (bs_light.cu): few groups, HBM-bound operators such as lattice models ---------------------
    // One 1024-thread block per SM owns ALL columns of a strip of rows: the per-column hop list (u16 entries) lives
    // in shared memory for the whole launch, rows are double-buffered by TMA, and every phase factor V(t_a) is
    // precomputed per (row, key) at plan time, so the row loop has no V phase and no list traffic.
    bool light = false;
    int light_lmax = 0;
    size_t light_smem = 0;
    int light_threads = 1024, light_maxt = 1024, light_sms = 0;        // launch geometry, fixed at plan build
    int light_stream = 1, light_order = 3, light_lut_nq = 0, light_sign = 1;  // kernel switches (test hooks, read at plan build)
    DevBuf<unsigned short> d_llist;  // [light_lmax][4 T], T = light_threads; entry 4 t + k of a slot: column t + k T;
                                     // value = source column * 16 | sign
    DevBuf<double> d_vtab;           // V values, row after row
    DevBuf<i64> d_voff;              // [Da + 1]
};

struct LightDev {
    RowPlanDev P;
    const unsigned short* llist;
    const double* vtab;
    const i64* voff;
    int l_max;
    u32 item0, item_split, key0, key_split;  // of the x_a = 0 header
    int lut_nq;                              // nibble tables of the diagonal (0: generic key loop)
    int stream;                              // streaming (evict-first) stores of out / acc
    int order;                               // which warps run the alpha-hop (global) phase before the shared-memory phase
};
int bs_light_build(bs_rowplan* R, cudaStream_t st);
