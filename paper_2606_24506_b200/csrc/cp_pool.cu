// cp_pool.cu -- host side of libcrosspool: the C ABI of include/crosspool.h, the pool
// manager (page ownership against the page budget, per-request page lists: the software
// counterpart of the paper's KV-cache virtualizer), the tile planner that
// builds the device work list (hot-path step a1), and the kernel launch glue.
#include <cuda_runtime.h>
#include <algorithm>
#include <cmath>
#include <cstdint>
#include <cstring>
#include <new>
#include <vector>

#include "../../include/crosspool.h"
#include "cp_internal.h"
#include "cp_launch.h"
#include "cp_vmm.h"

using namespace cp;

namespace {

struct DevBuf {
    void *ptr = nullptr;
    size_t cap = 0;
    // grow (never shrink); contents are NOT preserved.  Slow path: synchronises the device
    // before freeing the old buffer so no in-flight kernel can still read it.
    cudaError_t ensure(size_t bytes)
    {
        if (bytes <= cap) return cudaSuccess;
        if (ptr) {
            cudaError_t e = cudaDeviceSynchronize();
            if (e != cudaSuccess) return e;
            cudaFree(ptr);
            ptr = nullptr;
            cap = 0;
        }
        size_t want = std::max(bytes, (size_t)256);
        want = (want * 3 / 2 + 255) & ~(size_t)255;
        cudaError_t e = cudaMalloc(&ptr, want);
        if (e != cudaSuccess) { ptr = nullptr; return e; }
        cap = want;
        return cudaSuccess;
    }
    void release() { if (ptr) cudaFree(ptr); ptr = nullptr; cap = 0; }
};

struct Request {
    bool live = false;
    int32_t model = -1;
    int32_t ctx = 0;
    std::vector<int32_t> pages;      // page-major page list
    size_t uploaded = 0;             // entries already in the device page table
};

struct KindPlan {
    std::vector<Group> groups;
    std::vector<Tile> tiles;
    std::vector<TileRec> tile_recs;
    std::vector<Combine> combines;       // CTA-sized combine units (generic kernel)
    std::vector<CombineUnit> cunits;     // warp-sized combine units (tensor-core kernels)
    int max_splits = 1;
    int max_dk = 0, max_dv = 0;
    int max_group = 0;
    bool all_fast = false;           // every group of this kind runs on the tensor-core kernel
    bool use_kvt = false;            // KV kind: the tcgen05 tokens-on-M kernel (else the mma.sync kernel)
    int grid = 0;                    // tcgen05 K/V kernel: CTAs the static tile lists were laid out for
    int n_static_slots = 0;          // ... and the length of the static section of tile_recs (rounds * grid)
    bool uploaded = false;
    int counter_set = 0;             // scheduler counter set the next launch uses (alternates)
    int extra_counters = 0;          // multi-stage plans: one completion counter per stage after the groups'
    // device copy: ONE buffer (one host -> device copy per new plan) holding groups | tiles | tile_recs | combines | cunits,
    // the p_* pointers into it, and the counters: [32] scheduler + [n_groups * kCounterStride], twice
    // Both exist twice: a new plan is copied into the pair the running launch does not use, on the pool's copy stream, so
    // the upload overlaps the previous kernel instead of standing between two kernels of the stream.
    DevBuf d_pack2[2], d_counters2[2];
    int buf = 0;                          // the pair the current plan lives in
    cudaEvent_t ev_users[2] = {nullptr, nullptr};   // [b]: every launch that read pair b so far (recorded when the plan moves away from b)
    cudaEvent_t ev_copied = nullptr;                // the copy stream has finished the current plan's upload
    void *p_counters = nullptr;
    bool users_recorded[2] = {false, false};
    // pinned staging, a ring of four: a pageable source would make cudaMemcpyAsync wait for the stream (the copy is
    // staged chunk by chunk behind the work already queued), i.e. synchronise host and device on every new plan
    struct PinBuf { void *ptr = nullptr; size_t cap = 0; cudaEvent_t ev = nullptr; bool used = false; } pin[4];
    unsigned pin_next = 0;
    void *p_groups = nullptr, *p_tiles = nullptr, *p_tile_recs = nullptr, *p_combines = nullptr, *p_cunits = nullptr;
};

}  // namespace

struct cp_pool {
    uint8_t *arena = nullptr;
    uint64_t arena_bytes = 0;
    uint32_t P = 0, page_bytes = 0, num_pages = 0;
    std::vector<cp_model_cfg> models;
    int32_t max_requests = 0, max_ppr = 0;

    std::vector<int32_t> owner;          // per physical page: owning request id or -1
    uint32_t n_free = 0;
    uint32_t alloc_cursor = 0;
    std::vector<Request> reqs;
    std::vector<int32_t> h_ctx;          // host mirror of the device ctx table
    int32_t ctx_dirty_lo = INT32_MAX, ctx_dirty_hi = -1;
    uint64_t topo_version = 1;           // bumps when any request's planned page count changes

    // CUDA-VMM arena: the library owns the arena; request r's pages are the contiguous ids
    // r * slot_pages .. and physical chunks are mapped as the request grows
    VmmArena *vmm = nullptr;
    uint32_t slot_pages = 0;
    int opt_vmm_table = 0;               // 1: decode kernels read the (identity) page table anyway
    int opt_host_zero_copy = 1;          // cp_decode_attention_host: access pinned host buffers in place
    const void *zc_host[3] = {nullptr, nullptr, nullptr};   // last q / out / lse host pointers looked up ...
    void *zc_dev[3] = {nullptr, nullptr, nullptr};           // ... and their device aliases (nullptr: not mapped)

    // options
    int opt_kernel = 0, opt_num_ctas = 0, opt_waves_x16 = 16, opt_min_tile_pages = 2;
    int opt_static_pct = 100;            // tcgen05 K/V kernel: share of every group's slices in the static (equal) pieces
    int opt_tail_slices = 2;             // ... and the length of the dynamically popped tiles that hold the rest

    // query tokens per request of the call in progress (cp_decode_attention_qlen), and of the cached plan
    int qlen = 1, plan_qlen = 1;
    bool plan_for_stages = false;        // build_plan is called for a multi-stage work list (mma.sync kernel)
    const uint16_t *step_k = nullptr, *step_v = nullptr;   // cp_decode_step in progress: new rows the decode launch itself writes
    bool step_ctx_on_device = false;     // ... and the launch advances the device context table itself
    int opt_timeline = 0;                // CP_OPT_TIMELINE: per-CTA globaltimer stamps of the next decode launches
    int timeline_ctas = 0;               // grid size of the last launch that wrote stamps
    int device = -1;                     // device of the arena (the compute calls require it to be current)

    // plan cache
    std::vector<int32_t> plan_batch;
    uint64_t plan_version = 0;
    bool plan_valid = false;
    KindPlan plan[2];
    uint64_t plan_ws_floats = 0;
    std::vector<int64_t> q_off, out_off, lse_off;   // per batch slot (packed offsets)
    std::vector<int64_t> app_k_off, app_v_off;      // per batch slot: element offsets into the packed k_new / v_new of an append
    int64_t q_elems = 0, out_floats = 0, lse_floats = 0;

    // device side (lazy)
    bool dev_ready = false;
    int n_sm = 148;
    DevBuf d_page_table, d_ctx, d_models, d_append, d_timeline;   // d_ctx: TWO context tables of max_requests ints
    int ctx_cur = 0;                     // the table launches read; a fused decode step lets its kernel write the other
                                         // one (every entry copied, the batch's + 1) and flips this: no upload per step
    alignas(64) unsigned char kv_tmap[128];   // CUtensorMap of the arena for the MQA/GQA kernel
    bool kv_tmap_ok = false;
    alignas(64) unsigned char mla_tmap[128];  // CUtensorMap of the arena for the MLA kernel
    bool mla_tmap_ok = false;
    alignas(64) unsigned char mla2_tmap9[128], mla2_tmap2[128];   // CTA-pair MLA kernel
    bool mla2_tmap_ok = false;

    // multi-stage plan (cp_decode_attention_stages)
    struct StagesPlan {
        std::vector<int32_t> key;        // n_stages, sizes, ids, deps
        uint64_t version = 0;
        bool valid = false, uploaded = false;
        KindPlan kp;
        std::vector<StageRec> stages;
        DevBuf d_stages, d_gate;
        uint64_t ws_floats = 0;
        int64_t q_elems = 0, out_floats = 0, lse_floats = 0;
    } splan;

    // stream the last compute call ran on: the scheduler state of a plan (work list, counter sets, page table, context
    // table) is reused from call to call, so a call on ANOTHER stream first waits for everything the previous stream
    // was given (adopt_stream); side stream + events for the second attention kind of a mixed batch
    cudaStream_t last_stream = nullptr;
    bool last_stream_valid = false;
    cudaEvent_t ev_switch = nullptr, ev_fork = nullptr, ev_join = nullptr;
    cudaStream_t side_stream = nullptr, copy_stream = nullptr;
    // page-table entries of GROWN requests go up on the copy stream from pinned staging (flush_tables)
    struct TabPin { void *ptr = nullptr; size_t cap = 0; cudaEvent_t ev = nullptr; bool used = false; } tab_pin[4];
    int tab_next = 0;
    cudaEvent_t ev_tab = nullptr;
    bool tab_recorded = false;
    int kind_ctas[2] = {0, 0};           // CTAs each attention kind of the cached plan was planned for

    // counters
    uint64_t n_launches = 0, n_plan_builds = 0, n_h2d_bytes = 0;
};

namespace {

inline int ceil_div(int a, int b) { return (a + b - 1) / b; }

bool model_supported(const cp_model_cfg &m, uint32_t P, uint32_t page_bytes)
{
    if (m.kind != CP_KIND_KV && m.kind != CP_KIND_MLA) return false;
    if (m.n_q_heads < 1 || m.n_kv_heads < 1 || m.n_q_heads % m.n_kv_heads != 0) return false;
    if (m.head_dim_qk < 8 || m.head_dim_v < 8 || m.head_dim_qk % 8 || m.head_dim_v % 8) return false;
    if (m.head_dim_qk > kMaxDk || m.head_dim_v > kMaxDv) return false;
    if (!(m.softmax_scale == m.softmax_scale)) return false;
    uint64_t need;
    if (m.kind == CP_KIND_MLA) {
        if (m.n_kv_heads != 1 || m.head_dim_v > m.head_dim_qk) return false;
        need = (uint64_t)P * m.head_dim_qk * 2;
    } else {
        need = (uint64_t)P * (m.head_dim_qk + m.head_dim_v) * 2;
    }
    return need <= page_bytes;
}


// ----------------------------------------------------------------------------- planner, tcgen05 K/V kernel
// Step a1 for the tokens-on-M kernel.  The unit of work is a 128-token slice.  Every (request, kv
// head) group gives its first static_pct % slices to the STATIC part: the groups' static slices,
// laid end to end, are cut into n_ctas * waves pieces of equal length (the boundaries ignore the
// groups, as in a stream-K decomposition of a GEMM), piece j goes to CTA j mod n_ctas, and a
// piece that spans several groups becomes several tiles that its CTA runs one after the other
// (the kernel overlaps a tile's epilogue with the next tile's stream, so a tile boundary costs
// no bandwidth).  Equal pieces take away the 10 % spread that "near-equal splits of every
// group" leave between the CTAs' byte counts (cfg2: 64..78 pages per tile).  What remains of a
// group forms short TAIL tiles of tail_slices slices that the CTAs pop from one counter when
// their static lists are done: the SMs' streaming rates differ by a few per cent, and the tail
// lets the fast ones take more.  Every tile is a fixed token range with its own split slot, so
// results do not depend on which CTA runs it (deterministic).
constexpr int KT_COMBINE_WARPS = 11;     // warps per CTA of the tcgen05 K/V kernel (all of them run combine units)

void build_plan_kvt(cp_pool *pool, const int32_t *ids, int n, KindPlan &kp, uint64_t &ws)
{
    const int P = (int)pool->P;
    const int pps = 128 / P;                                   // pages per slice
    const int n_ctas = std::max(1, std::min(pool->kind_ctas[CP_KIND_KV], pool->n_sm));
    struct GInfo { int b, c, n_lp, n_sl, s_static; };
    std::vector<GInfo> gi;
    for (int b = 0; b < n; ++b) {
        const Request &r = pool->reqs[ids[b]];
        const cp_model_cfg &m = pool->models[r.model];
        if (m.kind != CP_KIND_KV) continue;
        const int n_lp = ceil_div(r.ctx, P), n_sl = ceil_div(n_lp, pps);
        int st = (int)((int64_t)n_sl * pool->opt_static_pct / 100);
        if (n_sl - st < 1 || pool->opt_static_pct >= 100) st = n_sl;
        for (int c = 0; c < m.n_kv_heads; ++c) gi.push_back(GInfo{b, c, n_lp, n_sl, st});
        kp.max_dk = std::max(kp.max_dk, m.head_dim_qk);
        kp.max_dv = std::max(kp.max_dv, m.head_dim_v);
    }
    const int ng = (int)gi.size();
    int64_t S = 0;
    for (const GInfo &g : gi) S += g.s_static;
    const int min_sl = std::max(1, ceil_div(pool->opt_min_tile_pages, pps));
    int64_t want_pieces = std::max<int64_t>(1, (int64_t)n_ctas * pool->opt_waves_x16 / 16);

    struct T { int g, sl0, sl1, piece; };                      // tile: slices [sl0, sl1) of group g; piece < 0: tail tile
    std::vector<T> tl;
    std::vector<int> n_static_of(ng), n_tail_of(ng), tail_len(ng);
    for (;;) {
        tl.clear();
        std::fill(n_static_of.begin(), n_static_of.end(), 0);
        const int64_t n_pieces = std::max<int64_t>(1, std::min<int64_t>(want_pieces, S));
        // cut positions in static-slice coordinates, snapped to a group boundary when they would leave
        // a fragment shorter than the minimum tile
        std::vector<int64_t> cut(n_pieces + 1);
        {
            std::vector<int64_t> gstart(ng + 1, 0);
            for (int g = 0; g < ng; ++g) gstart[g + 1] = gstart[g] + gi[g].s_static;
            int g = 0;
            for (int64_t j = 0; j <= n_pieces; ++j) {
                int64_t c = S * j / n_pieces;
                while (g < ng && gstart[g + 1] <= c && g + 1 < ng) ++g;
                if (j > 0 && j < n_pieces) {
                    if (c - gstart[g] < min_sl) c = gstart[g];
                    else if (gstart[g + 1] - c < min_sl) c = gstart[g + 1];
                }
                cut[j] = j > 0 ? std::max(c, cut[j - 1]) : 0;
            }
            cut[n_pieces] = S;
        }
        {
            int g = 0;
            int64_t gs0 = 0;                                   // static coordinate of group g's first slice
            for (int64_t j = 0; j < n_pieces; ++j) {
                int64_t a = cut[j];
                const int64_t e = cut[j + 1];
                while (a < e) {
                    while (g < ng && gs0 + gi[g].s_static <= a) { gs0 += gi[g].s_static; ++g; }
                    const int64_t ge = gs0 + gi[g].s_static;
                    const int64_t stop = std::min(e, ge);
                    tl.push_back(T{g, (int)(a - gs0), (int)(stop - gs0), (int)j});
                    n_static_of[g]++;
                    a = stop;
                }
            }
        }
        bool ok = true;
        for (int g = 0; g < ng; ++g) {
            const int rest = gi[g].n_sl - gi[g].s_static;
            int tlen = std::max(pool->opt_tail_slices, 1);
            const int room = kMaxSplits - n_static_of[g];
            if (rest > 0 && room < 1) ok = false;
            else if (rest > 0) tlen = std::max(tlen, ceil_div(rest, room));
            tail_len[g] = tlen;
            n_tail_of[g] = rest > 0 ? ceil_div(rest, tlen) : 0;
            if (n_static_of[g] > kMaxSplits) ok = false;
        }
        if (ok || want_pieces == 1) break;
        want_pieces = std::max<int64_t>(1, want_pieces / 2);
    }
    const int n_static_tiles = (int)tl.size();
    for (int g = 0; g < ng; ++g)
        for (int t = 0; t < n_tail_of[g]; ++t) {
            const int a = gi[g].s_static + t * tail_len[g];
            tl.push_back(T{g, a, std::min(a + tail_len[g], gi[g].n_sl), -1});
        }

    // groups, split slots (in token order: static tiles, then tail tiles), combine units
    std::vector<int> split_base(ng, 0);
    kp.groups.reserve(ng);
    // what all tile records of a group share, filled once per group (a rebuild sits between two decode steps of a
    // serving loop: cfg5 rebuilds at 4 of 5 steps), and where the group's page ids are
    std::vector<TileRec> rec_of(ng);
    std::vector<const int32_t *> pages_of(ng);
    for (int g = 0; g < ng; ++g) {
        const GInfo &G = gi[g];
        const Request &r = pool->reqs[ids[G.b]];
        const cp_model_cfg &m = pool->models[r.model];
        const int hpk = m.n_q_heads / m.n_kv_heads;
        const int rows = hpk * pool->qlen;             // rows of the group: (query token, head), token-major
        const int ns = n_static_of[g] + n_tail_of[g];
        kp.max_splits = std::max(kp.max_splits, ns);
        Group gr;
        gr.req = ids[G.b]; gr.model = r.model; gr.kv_head = G.c; gr.n_splits = ns;
        gr.n_pages = G.n_lp; gr.batch_index = G.b;
        gr.q_off = pool->q_off[G.b] + (int64_t)G.c * hpk * m.head_dim_qk;
        gr.out_off = pool->out_off[G.b] + (int64_t)G.c * hpk * m.head_dim_v;
        gr.lse_off = pool->lse_off[G.b] + (int64_t)G.c * hpk;
        gr.part_off = 0;
        if (ns > 1) {
            gr.part_off = (int64_t)ws;
            ws += (uint64_t)part_group_floats(rows, ns, m.head_dim_v);
            const int zl = ns <= 8 ? 0 : (ns <= 32 ? 3 : (ns <= 128 ? 4 : 5));
            const int cols = 128 >> zl;
            CombineUnit cu;
            std::memset(&cu, 0, sizeof(cu));
            cu.split_stride = cols;
            cu.n_splits = ns;
            cu.zl_log2 = zl;
            cu.want = ns * 4;                               // one arrival per epilogue warp and tile
            cu.group = g;
            for (int h = 0; h < rows; ++h) {
                kp.combines.push_back(Combine{g, h});
                // row (t, hh) of the group is row t * Hq + hh of the request's output (q_len = 1: row h)
                const int64_t orow = (int64_t)(h / hpk) * m.n_q_heads + h % hpk;
                cu.ml_off = gr.part_off + part_ml_off(rows, h, 0, ns, m.head_dim_v);
                for (int c0 = 0; c0 < m.head_dim_v; c0 += cols) {
                    // partial layout of this kernel: [h][c0 / cols][s][cols] (the unit's 512-byte reads are contiguous)
                    cu.part_off = gr.part_off + (int64_t)h * ns * m.head_dim_v + (int64_t)(c0 / cols) * ns * cols;
                    cu.out_off = gr.out_off + orow * m.head_dim_v + c0;
                    cu.lse_off = c0 == 0 ? gr.lse_off + orow : -1;
                    kp.cunits.push_back(cu);
                }
            }
        }
        kp.groups.push_back(gr);
        TileRec &t = rec_of[g];
        std::memset(&t, 0, sizeof(t));
        t.group = g; t.req = gr.req; t.kv_head = gr.kv_head; t.n_kv_heads = m.n_kv_heads;
        t.n_splits = ns;
        t.gsize = rows; t.n_q_heads = m.n_q_heads;
        t.scale_log2 = (float)((double)m.softmax_scale * 1.4426950408889634);
        t.q_off = gr.q_off; t.out_off = gr.out_off; t.lse_off = gr.lse_off; t.part_off = gr.part_off;
        t.pad = (ns <= 8 ? 0 : (ns <= 32 ? 3 : (ns <= 128 ? 4 : 5))) << 8;   // bits 8..15: partial layout (zl of the group's units)
        // (one new row per kv head and request: the packed k_new / v_new of a step stay far below 2^31 elements)
        t.app_k_off = (int32_t)(pool->app_k_off[G.b] + (int64_t)gr.kv_head * m.head_dim_qk);
        t.app_v_off = (int32_t)(pool->app_v_off[G.b] + (int64_t)gr.kv_head * m.head_dim_v);
        pages_of[g] = r.pages.data() + gr.kv_head;        // page j of the group at [j * n_kv_heads]
    }
    auto make_rec = [&](const T &t, int split) {
        const GInfo &G = gi[t.g];
        TileRec r = rec_of[t.g];
        r.page_begin = t.sl0 * pps; r.n_pages = std::min(t.sl1 * pps, G.n_lp) - r.page_begin;
        r.split = split;
        // bit 0 of pad (set by the caller): another static record of the CTA follows; bit 1: the group's last planned page is here
        if (r.page_begin + r.n_pages == G.n_lp) r.pad |= 2;
        const int32_t *pg = pages_of[t.g] + (size_t)r.page_begin * r.n_kv_heads;
        for (int i = 0; i < 8 && i < r.n_pages && i < pps; ++i) r.first_pid[i] = pg[(size_t)i * r.n_kv_heads];
        return r;
    };
    // split index of a tile = its rank inside the group by position (tl is in that order per group)
    std::vector<int> split_of(tl.size());
    for (size_t i = 0; i < tl.size(); ++i) split_of[i] = split_base[tl[i].g]++;

    // device order: record b < grid = the first tile of CTA b's static list (n_pages = 0: it has none), then the rest of
    // every CTA's list, contiguous and chained through TileRec::next (a list of lists would leave the array as sparse
    // as its longest list: 2220 records for 523 tiles on cfg5, all of it cleared, copied and uploaded at every rebuild),
    // then the tail tiles, longest first
    const int64_t n_pieces_used = n_static_tiles ? tl[n_static_tiles - 1].piece + 1 : 0;
    int grid = (int)std::min<int64_t>(n_ctas, std::max<int64_t>(std::max<int64_t>(n_pieces_used, 1),
                                                                 ((int64_t)kp.cunits.size() + KT_COMBINE_WARPS - 1) / KT_COMBINE_WARPS));
    if (tl.size() > (size_t)n_static_tiles) grid = n_ctas;          // dynamic tiles: every CTA may take some
    // (tl holds the static tiles in piece order, so CTA b's list is b's tiles in tl order: two counting passes)
    std::vector<int> cnt(grid, 0), slot_of(n_static_tiles);
    for (int i = 0; i < n_static_tiles; ++i) slot_of[i] = cnt[tl[i].piece % grid]++;
    std::vector<int> cont(grid, 0);                  // where the rest of CTA b's list starts
    size_t n_static_recs = n_static_tiles ? (size_t)grid : 0;
    for (int b = 0; b < grid; ++b) { cont[b] = (int)n_static_recs; n_static_recs += (size_t)std::max(cnt[b] - 1, 0); }
    kp.tile_recs.resize(n_static_recs + (tl.size() - n_static_tiles));
    if (n_static_tiles)
        for (int b = 0; b < grid; ++b)
            if (cnt[b] == 0) std::memset(&kp.tile_recs[b], 0, sizeof(TileRec));
    for (int i = 0; i < n_static_tiles; ++i) {
        const int b = tl[i].piece % grid, j = slot_of[i];
        const int idx = j == 0 ? b : cont[b] + j - 1;
        TileRec &r = kp.tile_recs[idx];
        r = make_rec(tl[i], split_of[i]);
        if (j + 1 < cnt[b]) { r.pad |= 1; r.next = j == 0 ? cont[b] : idx + 1; }
    }
    std::vector<int> tails;
    for (size_t i = n_static_tiles; i < tl.size(); ++i) tails.push_back((int)i);
    std::stable_sort(tails.begin(), tails.end(), [&](int a, int b) {
        return (tl[a].sl1 - tl[a].sl0) > (tl[b].sl1 - tl[b].sl0);
    });
    for (size_t t = 0; t < tails.size(); ++t)
        kp.tile_recs[n_static_recs + t] = make_rec(tl[tails[t]], split_of[tails[t]]);
    // the real tiles in device order (reporting: cp_decode_plan)
    kp.tiles.reserve(tl.size());
    for (const TileRec &r : kp.tile_recs)
        if (r.n_pages > 0) kp.tiles.push_back(Tile{r.group, r.split, r.page_begin, r.page_begin + r.n_pages});
    kp.grid = grid;
    kp.n_static_slots = (int)n_static_recs;
}

// ----------------------------------------------------------------------------- planner
// Step a1: cut every (request, kv head) group into page-aligned KV splits of near-equal
// length so that the whole batch yields about n_ctas * waves tiles; tiles are ordered
// longest first (the persistent CTAs pop them in array order), combine units follow.
void build_plan(cp_pool *pool, const int32_t *ids, int n)
{
    const int P = (int)pool->P;
    for (int k = 0; k < 2; ++k) {
        KindPlan &kp = pool->plan[k];
        kp.groups.clear(); kp.tiles.clear(); kp.combines.clear(); kp.cunits.clear();
        kp.max_splits = 1; kp.max_dk = kp.max_dv = kp.max_group = 0; kp.uploaded = false;
    }
    pool->q_off.assign(n, 0); pool->out_off.assign(n, 0); pool->lse_off.assign(n, 0);
    pool->app_k_off.assign(n, 0); pool->app_v_off.assign(n, 0);
    int64_t qo = 0, oo = 0, lo = 0, ako = 0, avo = 0;
    int64_t total_pages[2] = {0, 0};
    for (int b = 0; b < n; ++b) {
        const Request &r = pool->reqs[ids[b]];
        const cp_model_cfg &m = pool->models[r.model];
        pool->q_off[b] = qo; pool->out_off[b] = oo; pool->lse_off[b] = lo;
        qo += (int64_t)pool->qlen * m.n_q_heads * m.head_dim_qk;
        oo += (int64_t)pool->qlen * m.n_q_heads * m.head_dim_v;
        lo += (int64_t)pool->qlen * m.n_q_heads;
        pool->app_k_off[b] = ako; pool->app_v_off[b] = avo;
        ako += (int64_t)m.n_kv_heads * m.head_dim_qk;
        if (m.kind != CP_KIND_MLA) avo += (int64_t)m.n_kv_heads * m.head_dim_v;
        total_pages[m.kind] += (int64_t)ceil_div(r.ctx, P) * m.n_kv_heads;
    }
    pool->q_elems = qo; pool->out_floats = oo; pool->lse_floats = lo;

    // (A batch with models of both attention kinds runs two persistent kernels, each planned for ALL CTAs: either
    // needs every SM to reach its own rate -- measured: splitting the SMs between them in proportion to their bytes
    // makes the step longer than running them one after the other -- but launched on two streams the second
    // kernel's CTAs move in as the first one's leave, which hides the first's tail and the second's start-up.)
    const int n_all = pool->opt_num_ctas > 0 ? pool->opt_num_ctas : pool->n_sm;
    pool->kind_ctas[0] = pool->kind_ctas[1] = n_all;
    uint64_t ws = 0;
    for (int k = 0; k < 2; ++k) {
        KindPlan &kp = pool->plan[k];
        if (total_pages[k] == 0) continue;
        // smallest tile length L (pages) for which the batch yields at most target_tiles tiles, so
        // that with waves = w every persistent CTA gets exactly w near-equal tiles (one tile more
        // on a few CTAs would cost a whole extra tile time at the end)
        // the tcgen05 MLA kernel runs every tile as two work items (value halves)
        bool mla_fast = k == CP_KIND_MLA && pool->opt_kernel != 1 && mla_fast_supported(P, pool->page_bytes);
        if (mla_fast)
            for (int b = 0; b < n; ++b) {
                const cp_model_cfg &m = pool->models[pool->reqs[ids[b]].model];
                if (m.kind == CP_KIND_MLA && !(m.head_dim_qk == 576 && m.head_dim_v == 512 && m.n_q_heads <= 128))
                    mla_fast = false;
            }
        const int n_ctas = pool->kind_ctas[k];
        const int64_t target_tiles =
            std::max<int64_t>(1, (int64_t)n_ctas * pool->opt_waves_x16 / 16 / (mla_fast ? 2 : 1));
        // which K/V kernel will run this plan: it fixes how many arrivals a finished tile makes on its
        // group's counter (tcgen05 tokens-on-M kernel: its 4 softmax warps; mma.sync kernel: one per M tile)
        kp.all_fast = k == CP_KIND_KV ? true : mla_fast;
        kp.max_group = 0;
        for (int b = 0; b < n; ++b) {
            const cp_model_cfg &m = pool->models[pool->reqs[ids[b]].model];
            if (m.kind != k) continue;
            const int g = m.n_q_heads / m.n_kv_heads * pool->qlen;
            if (k == CP_KIND_KV && !(m.head_dim_qk == 128 && m.head_dim_v == 128 && g <= 128)) kp.all_fast = false;
            kp.max_group = std::max(kp.max_group, g);
        }
        kp.use_kvt = k == CP_KIND_KV && kp.all_fast && (pool->opt_kernel == 0 || pool->opt_kernel == 2) &&
                     !pool->plan_for_stages && kvt_supported(P) && kvt_pad_rows(kp.max_group) > 0;
        // q_len > 1: the 32-row instantiation (three ring stages, twice the softmax work per byte) beats the warp-MMA
        // kernel only back to back on long contexts (cfg2, q_len 4: 62.0 vs 64.3 us; after a flush 75.8 vs 71.7; cfg5,
        // q_len 2: 135 vs 126 us), so by default only groups of up to 16 rows go to the tcgen05 kernel; CP_OPT_KERNEL = 2
        // asks for it up to 32 rows
        if (kp.use_kvt && pool->qlen > 1 && pool->opt_kernel == 0 && kp.max_group > 16) kp.use_kvt = false;
        if (kp.use_kvt) {
            kp.tile_recs.clear();
            build_plan_kvt(pool, ids, n, kp, ws);
            continue;
        }
        kp.grid = 0; kp.n_static_slots = 0;
        // splits per request (shared with the device-side planner of the request queue: plan_request_splits)
        std::vector<int> req_splits(n, 0);
        {
            std::vector<int> v_lp(n, 0), v_hkv(n, 0);
            for (int b = 0; b < n; ++b) {
                const Request &r = pool->reqs[ids[b]];
                const cp_model_cfg &m = pool->models[r.model];
                if (m.kind != k) continue;
                v_lp[b] = ceil_div(r.ctx, P);
                v_hkv[b] = m.n_kv_heads;
            }
            plan_request_splits(n, v_lp.data(), v_hkv.data(), target_tiles, pool->opt_min_tile_pages, kMaxSplits, req_splits.data());
        }
        for (int b = 0; b < n; ++b) {
            const Request &r = pool->reqs[ids[b]];
            const cp_model_cfg &m = pool->models[r.model];
            if (m.kind != k) continue;
            const int hpk = m.n_q_heads / m.n_kv_heads;       // query heads per kv head
            const int g = hpk * pool->qlen;                   // rows of a group: (query token, head), token-major
            const int n_lp = ceil_div(r.ctx, P);
            const int ns = req_splits[b];
            kp.max_splits = std::max(kp.max_splits, ns);
            kp.max_dk = std::max(kp.max_dk, m.head_dim_qk);
            kp.max_dv = std::max(kp.max_dv, m.head_dim_v);
            for (int c = 0; c < m.n_kv_heads; ++c) {
                Group gr;
                gr.req = ids[b]; gr.model = r.model; gr.kv_head = c; gr.n_splits = ns;
                gr.n_pages = n_lp; gr.batch_index = b;
                gr.q_off = pool->q_off[b] + (int64_t)c * hpk * m.head_dim_qk;
                gr.out_off = pool->out_off[b] + (int64_t)c * hpk * m.head_dim_v;
                gr.lse_off = pool->lse_off[b] + (int64_t)c * hpk;
                gr.part_off = 0;
                if (ns > 1) {
                    gr.part_off = (int64_t)ws;
                    ws += (uint64_t)part_group_floats(g, ns, m.head_dim_v);
                }
                const int gi = (int)kp.groups.size();
                kp.groups.push_back(gr);
                const int base = n_lp / ns, rem = n_lp % ns;
                int pb = 0;
                for (int s = 0; s < ns; ++s) {
                    const int len = base + (s < rem ? 1 : 0);
                    kp.tiles.push_back(Tile{gi, s, pb, pb + len});
                    pb += len;
                }
                if (ns > 1) {
                    for (int h = 0; h < g; ++h) kp.combines.push_back(Combine{gi, h});
                    // warp-sized units: split lanes ZL so that a lane holds <= 16 splits (8 for ZL = 1, 8)
                    // wide value rows (MLA, 512 columns): a unit costs a few L2 round trips whatever its
                    // width, so keep units few and wide (zl = 0: one float4 column per lane, 128 columns)
                    // (the MLA pair kernel's own combine relies on zl = 0 for 512-column rows)
                    const int zl = m.head_dim_v > 128 ? 0 : (ns <= 8 ? 0 : (ns <= 32 ? 3 : (ns <= 128 ? 4 : 5)));
                    const int cols = 128 >> zl;
                    const int mt = (g + 15) / 16;
                    int mtp = 1;
                    while (mtp < mt) mtp <<= 1;
                    for (int h = 0; h < g; ++h)
                        for (int c0 = 0; c0 < m.head_dim_v; c0 += cols) {
                            CombineUnit cu;
                            std::memset(&cu, 0, sizeof(cu));
                            cu.part_off = gr.part_off + part_o_off(h, 0, ns, m.head_dim_v) + c0;
                            cu.ml_off = gr.part_off + part_ml_off(g, h, 0, ns, m.head_dim_v);
                            // row h = query token h / hpk, head h % hpk; a token's rows are Hq apart
                            const int64_t row = (int64_t)(h / hpk) * m.n_q_heads + h % hpk;
                            cu.out_off = gr.out_off + row * m.head_dim_v + c0;
                            cu.lse_off = c0 == 0 ? gr.lse_off + row : -1;
                            cu.split_stride = m.head_dim_v;
                            cu.n_splits = ns;
                            cu.zl_log2 = zl;
                            // arrivals per finished tile: K/V tcgen05 kernel 4 (softmax warps), K/V mma.sync kernel one
                            // per padded M tile, MLA 8 (4 softmax warps x 2 value halves / CTAs)
                            cu.want = ns * (k == CP_KIND_KV ? (kp.use_kvt ? 4 : mtp) : 8);
                            cu.group = gi;
                            kp.cunits.push_back(cu);
                        }
                }
            }
        }
        std::stable_sort(kp.tiles.begin(), kp.tiles.end(), [](const Tile &a, const Tile &b) {
            return (a.page_end - a.page_begin) > (b.page_end - b.page_begin);
        });
        // combine units in the order in which their groups' last tiles are popped, so a CTA
        // that runs out of tiles first combines the groups that finish first
        kp.tile_recs.resize(kp.tiles.size());
        for (size_t i = 0; i < kp.tiles.size(); ++i) {
            const Tile &t = kp.tiles[i];
            const Group &gr = kp.groups[t.group];
            const cp_model_cfg &m = pool->models[gr.model];
            TileRec &r = kp.tile_recs[i];
            std::memset(&r, 0, sizeof(r));
            r.group = t.group; r.req = gr.req; r.kv_head = gr.kv_head; r.n_kv_heads = m.n_kv_heads;
            r.page_begin = t.page_begin; r.n_pages = t.page_end - t.page_begin; r.split = t.split;
            r.n_splits = gr.n_splits; r.gsize = m.n_q_heads / m.n_kv_heads * pool->qlen; r.n_q_heads = m.n_q_heads;
            r.pad = pool->qlen > 1 ? m.n_q_heads / m.n_kv_heads : 0;
            r.scale_log2 = (float)((double)m.softmax_scale * 1.4426950408889634);
            r.q_off = gr.q_off; r.out_off = gr.out_off; r.lse_off = gr.lse_off; r.part_off = gr.part_off;
            r.app_k_off = (int32_t)(pool->app_k_off[gr.batch_index] + (int64_t)gr.kv_head * m.head_dim_qk);
            r.app_v_off = (int32_t)(pool->app_v_off[gr.batch_index] + (int64_t)gr.kv_head * m.head_dim_v);
        }
        std::vector<int> last_pos(kp.groups.size(), 0);
        for (size_t i = 0; i < kp.tiles.size(); ++i) last_pos[kp.tiles[i].group] = (int)i;
        std::stable_sort(kp.combines.begin(), kp.combines.end(), [&](const Combine &a, const Combine &b) {
            return last_pos[a.group] < last_pos[b.group];
        });
        std::stable_sort(kp.cunits.begin(), kp.cunits.end(), [&](const CombineUnit &a, const CombineUnit &b) {
            return last_pos[a.group] < last_pos[b.group];
        });
    }
    pool->plan_ws_floats = ws;
    pool->plan_batch.assign(ids, ids + n);
    pool->plan_version = pool->topo_version;
    pool->plan_qlen = pool->qlen;
    pool->plan_valid = true;
    pool->n_plan_builds++;
}

cp_status check_batch(cp_pool *pool, const int32_t *ids, int n)
{
    if (!pool || !ids || n < 1) return CP_ERR_INVALID_ARG;
    for (int b = 0; b < n; ++b) {
        if (ids[b] < 0 || ids[b] >= pool->max_requests) return CP_ERR_INVALID_ARG;
        if (!pool->reqs[ids[b]].live) return CP_ERR_UNKNOWN_REQUEST;
    }
    // distinct ids (batches are small; O(n log n))
    std::vector<int32_t> s(ids, ids + n);
    std::sort(s.begin(), s.end());
    for (int b = 1; b < n; ++b)
        if (s[b] == s[b - 1]) return CP_ERR_INVALID_ARG;
    return CP_OK;
}

void ensure_plan(cp_pool *pool, const int32_t *ids, int n)
{
    if (pool->plan_valid && pool->plan_version == pool->topo_version && pool->plan_qlen == pool->qlen &&
        (int)pool->plan_batch.size() == n && std::equal(ids, ids + n, pool->plan_batch.begin()))
        return;
    build_plan(pool, ids, n);
}

// ------------------------------------------------------------------------ device state
cp_status ensure_device(cp_pool *pool)
{
    int dev = 0;
    if (cudaGetDevice(&dev) != cudaSuccess) { cudaGetLastError(); return CP_ERR_CUDA; }
    if (pool->dev_ready) return dev == pool->device ? CP_OK : CP_ERR_INVALID_ARG;   // the arena's device must be current
    int adev = dev;
    if (pool->vmm) {
        // the base of a reserved range has no backing until slot 0 is mapped: take the device from the arena object
        adev = pool->vmm->device;
    } else {
        cudaPointerAttributes attr;
        if (cudaPointerGetAttributes(&attr, pool->arena) != cudaSuccess || attr.type != cudaMemoryTypeDevice) {
            cudaGetLastError();
            return CP_ERR_INVALID_ARG;          // arena is not device memory
        }
        adev = attr.device;
    }
    if (adev != dev) return CP_ERR_INVALID_ARG; // metadata, streams and launches all live on the arena's device
    int sms = 0;
    if (cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, adev) != cudaSuccess)
        return CP_ERR_CUDA;
    if (pool->d_page_table.ensure((size_t)pool->max_requests * pool->max_ppr * 4) != cudaSuccess ||
        pool->d_ctx.ensure((size_t)pool->max_requests * 4 * 2) != cudaSuccess ||
        pool->d_models.ensure(pool->models.size() * sizeof(DevModel)) != cudaSuccess) {
        cudaGetLastError();
        return CP_ERR_CUDA;
    }
    std::vector<DevModel> dm(pool->models.size());
    for (size_t i = 0; i < dm.size(); ++i) {
        const cp_model_cfg &m = pool->models[i];
        dm[i].kind = m.kind; dm[i].n_q_heads = m.n_q_heads; dm[i].n_kv_heads = m.n_kv_heads;
        dm[i].d_k = m.head_dim_qk; dm[i].d_v = m.head_dim_v; dm[i].group = m.n_q_heads / m.n_kv_heads;
        dm[i].scale = m.softmax_scale;
        dm[i].scale_log2 = (float)((double)m.softmax_scale * 1.4426950408889634);
    }
    if (cudaMemcpy(pool->d_models.ptr, dm.data(), dm.size() * sizeof(DevModel),
                   cudaMemcpyHostToDevice) != cudaSuccess)
        return CP_ERR_CUDA;
    pool->ctx_cur = 0;
    if (cudaMemset(pool->d_ctx.ptr, 0, (size_t)pool->max_requests * 4 * 2) != cudaSuccess)
        return CP_ERR_CUDA;
    // TMA row coordinates are signed 32-bit: a tensor map is only used while every row index fits (a
    // CUDA-VMM pool reserves virtual space only and can exceed that; it then runs on the generic kernel)
    pool->kv_tmap_ok = false;
    if (kv_fast_supported((int)pool->P) && pool->page_bytes % 256 == 0 &&
        pool->page_bytes >= pool->P * 512u) {
        const uint64_t rows = (uint64_t)pool->num_pages * (pool->page_bytes / 256);
        pool->kv_tmap_ok = rows < (1ull << 31) &&
                           make_arena_tensor_map(pool->kv_tmap, pool->arena, rows, 128, 64, pool->P);
    }
    pool->mla_tmap_ok = false;
    pool->mla2_tmap_ok = false;
    if (mla_fast_supported((int)pool->P, pool->page_bytes)) {
        const uint64_t rows = (uint64_t)pool->num_pages * (pool->page_bytes / 1152);
        pool->mla_tmap_ok = rows < (1ull << 31) && make_mla_tensor_map(pool->mla_tmap, pool->arena, rows);
        // (the pair kernel loads the score operand of a slice PAIR, 64 tokens, with one box: pages of 64 k tokens)
        pool->mla2_tmap_ok = rows < (1ull << 31) && pool->P % 64 == 0 &&
                             make_mla2_tensor_maps(pool->mla2_tmap9, pool->mla2_tmap2, pool->arena, rows);
    }
    pool->n_sm = sms;
    pool->device = adev;
    pool->dev_ready = true;
    pool->plan_valid = false;               // the SM count feeds the planner
    pool->splan.valid = false;
    // everything mapped so far is dirty
    for (auto &r : pool->reqs) r.uploaded = 0;
    pool->ctx_dirty_lo = 0; pool->ctx_dirty_hi = pool->max_requests - 1;
    return CP_OK;
}

// Calls of one pool are stream-ordered by the caller in the common case (one stream).  A call on another stream than
// the previous one is made to wait for all work the previous stream holds -- the earlier launch may still be reading
// the work list, counters and tables this call is about to rewrite.  Costs nothing while the stream stays the same.
cp_status adopt_stream(cp_pool *pool, cudaStream_t s)
{
    if (pool->last_stream_valid && pool->last_stream != s) {
        if (!pool->ev_switch && cudaEventCreateWithFlags(&pool->ev_switch, cudaEventDisableTiming) != cudaSuccess) {
            cudaGetLastError();
            return CP_ERR_CUDA;
        }
        if (cudaEventRecord(pool->ev_switch, pool->last_stream) != cudaSuccess ||
            cudaStreamWaitEvent(s, pool->ev_switch, 0) != cudaSuccess) {
            cudaGetLastError();
            return CP_ERR_CUDA;
        }
    }
    pool->last_stream = s;
    pool->last_stream_valid = true;
    return CP_OK;
}

// Upload page-table rows and context lengths that changed since the last device call.
cp_status flush_tables(cp_pool *pool, cudaStream_t stream)
{
    // Entries a request GAINED (r.uploaded > 0: the request's earlier entries are on the device) lie beyond every page
    // a launch already enqueued reads, so they need no ordering behind those launches: they go up on the copy stream
    // from pinned staging while the previous step's kernel still runs, and `stream` only waits for an event.  Measured:
    // the same few bytes as a copy on the caller's stream in front of the kernel cost a decode loop 10-15 us of device
    // time per page boundary (cfg5: 138 us per iteration against 126 for the attention alone).  A request's FIRST upload
    // (or its re-upload after unmap + map) may overwrite entries that enqueued launches read: caller's stream, after
    // everything the copy stream was given.
    size_t grown = 0;
    bool first = false;
    for (int rid = 0; rid < pool->max_requests; ++rid) {
        const Request &r = pool->reqs[rid];
        if (!r.live || r.uploaded >= r.pages.size()) continue;
        if (r.uploaded > 0) grown += r.pages.size() - r.uploaded;
        else first = true;
    }
    if (first && pool->tab_recorded && cudaStreamWaitEvent(stream, pool->ev_tab, 0) != cudaSuccess) return CP_ERR_CUDA;
    if (grown) {
        if (!pool->copy_stream && cudaStreamCreateWithFlags(&pool->copy_stream, cudaStreamNonBlocking) != cudaSuccess) { cudaGetLastError(); return CP_ERR_CUDA; }
        if (!pool->ev_tab && cudaEventCreateWithFlags(&pool->ev_tab, cudaEventDisableTiming) != cudaSuccess) { cudaGetLastError(); return CP_ERR_CUDA; }
        cp_pool::TabPin &pb = pool->tab_pin[pool->tab_next++ % 4];
        if (pb.used && cudaEventSynchronize(pb.ev) != cudaSuccess) { cudaGetLastError(); return CP_ERR_CUDA; }
        if (pb.cap < grown * 4) {
            if (pb.ptr) cudaFreeHost(pb.ptr);
            pb.ptr = nullptr; pb.cap = 0;
            const size_t want = (grown * 4 * 2 + 4095) & ~(size_t)4095;
            if (cudaHostAlloc(&pb.ptr, want, cudaHostAllocDefault) != cudaSuccess) { cudaGetLastError(); pb.ptr = nullptr; return CP_ERR_CUDA; }
            pb.cap = want;
        }
        if (!pb.ev && cudaEventCreateWithFlags(&pb.ev, cudaEventDisableTiming) != cudaSuccess) { cudaGetLastError(); return CP_ERR_CUDA; }
        size_t off = 0;
        for (int rid = 0; rid < pool->max_requests; ++rid) {
            Request &r = pool->reqs[rid];
            if (!r.live || r.uploaded >= r.pages.size() || r.uploaded == 0) continue;
            const size_t n = r.pages.size() - r.uploaded;
            int32_t *src = (int32_t *)pb.ptr + off;
            std::memcpy(src, r.pages.data() + r.uploaded, n * 4);
            int32_t *dst = (int32_t *)pool->d_page_table.ptr + (size_t)rid * pool->max_ppr + r.uploaded;
            if (cudaMemcpyAsync(dst, src, n * 4, cudaMemcpyHostToDevice, pool->copy_stream) != cudaSuccess) return CP_ERR_CUDA;
            pool->n_h2d_bytes += n * 4;
            r.uploaded = r.pages.size();
            off += n;
        }
        if (cudaEventRecord(pb.ev, pool->copy_stream) != cudaSuccess || cudaEventRecord(pool->ev_tab, pool->copy_stream) != cudaSuccess ||
            cudaStreamWaitEvent(stream, pool->ev_tab, 0) != cudaSuccess)
            return CP_ERR_CUDA;
        pb.used = true;
        pool->tab_recorded = true;
    }
    for (int rid = 0; first && rid < pool->max_requests; ++rid) {
        Request &r = pool->reqs[rid];
        if (!r.live || r.uploaded >= r.pages.size()) continue;
        const size_t n = r.pages.size() - r.uploaded;
        int32_t *dst = (int32_t *)pool->d_page_table.ptr + (size_t)rid * pool->max_ppr + r.uploaded;
        if (cudaMemcpyAsync(dst, r.pages.data() + r.uploaded, n * 4, cudaMemcpyHostToDevice, stream) != cudaSuccess)
            return CP_ERR_CUDA;
        pool->n_h2d_bytes += n * 4;
        r.uploaded = r.pages.size();
    }
    if (pool->ctx_dirty_hi >= pool->ctx_dirty_lo) {
        const int lo = pool->ctx_dirty_lo, hi = pool->ctx_dirty_hi;
        if (cudaMemcpyAsync((int32_t *)pool->d_ctx.ptr + (size_t)pool->ctx_cur * pool->max_requests + lo, pool->h_ctx.data() + lo, (size_t)(hi - lo + 1) * 4,
                            cudaMemcpyHostToDevice, stream) != cudaSuccess)
            return CP_ERR_CUDA;
        pool->n_h2d_bytes += (size_t)(hi - lo + 1) * 4;
        pool->ctx_dirty_lo = INT32_MAX; pool->ctx_dirty_hi = -1;
    }
    return CP_OK;
}

cp_status upload_plan(cp_pool *pool, KindPlan &kp, cudaStream_t stream)
{
    if (kp.uploaded) return CP_OK;
    const size_t set_ints = 32 + (kp.groups.size() + kp.extra_counters) * (size_t)kCounterStride, nb = 2 * set_ints * 4;
    const void *src[5] = {kp.groups.data(), kp.tiles.data(), kp.tile_recs.data(), kp.combines.data(), kp.cunits.data()};
    const size_t bytes[5] = {kp.groups.size() * sizeof(Group), kp.tiles.size() * sizeof(Tile), kp.tile_recs.size() * sizeof(TileRec),
                             kp.combines.size() * sizeof(Combine), kp.cunits.size() * sizeof(CombineUnit)};
    size_t off[5], total = 0;
    for (int i = 0; i < 5; ++i) { off[i] = total; total += (bytes[i] + 255) & ~(size_t)255; }
    total = std::max(total, (size_t)256);
    const int t = 1 - kp.buf;                 // target pair: not the one the stream's queued launches read
    if (kp.d_pack2[t].ensure(total) != cudaSuccess || kp.d_counters2[t].ensure(nb) != cudaSuccess) {
        cudaGetLastError();
        return CP_ERR_CUDA;
    }
    if (!pool->copy_stream && cudaStreamCreateWithFlags(&pool->copy_stream, cudaStreamNonBlocking) != cudaSuccess) { cudaGetLastError(); return CP_ERR_CUDA; }
    for (int i = 0; i < 2; ++i)
        if (!kp.ev_users[i] && cudaEventCreateWithFlags(&kp.ev_users[i], cudaEventDisableTiming) != cudaSuccess) { cudaGetLastError(); return CP_ERR_CUDA; }
    if (!kp.ev_copied && cudaEventCreateWithFlags(&kp.ev_copied, cudaEventDisableTiming) != cudaSuccess) { cudaGetLastError(); return CP_ERR_CUDA; }
    KindPlan::PinBuf &pb = kp.pin[kp.pin_next++ % 4];
    if (pb.used && cudaEventSynchronize(pb.ev) != cudaSuccess) { cudaGetLastError(); return CP_ERR_CUDA; }   // its last copy (4 plans ago) is done
    if (pb.cap < total) {
        if (pb.ptr) cudaFreeHost(pb.ptr);
        pb.ptr = nullptr; pb.cap = 0;
        const size_t want = (total * 3 / 2 + 4095) & ~(size_t)4095;
        if (cudaHostAlloc(&pb.ptr, want, cudaHostAllocDefault) != cudaSuccess) { cudaGetLastError(); pb.ptr = nullptr; return CP_ERR_CUDA; }
        pb.cap = want;
    }
    if (!pb.ev && cudaEventCreateWithFlags(&pb.ev, cudaEventDisableTiming) != cudaSuccess) { cudaGetLastError(); return CP_ERR_CUDA; }
    for (int i = 0; i < 5; ++i)
        if (bytes[i]) std::memcpy((uint8_t *)pb.ptr + off[i], src[i], bytes[i]);
    // copy stream: wait for the launches that read pair t (all enqueued before the plan moved to the other pair: ev_users[t]
    // was recorded then), copy, clear the counters (two sets for alternate launches; a new plan starts from zero)
    cudaStream_t cs = pool->copy_stream;
    if ((kp.users_recorded[t] && cudaStreamWaitEvent(cs, kp.ev_users[t], 0) != cudaSuccess) ||
        cudaMemcpyAsync(kp.d_pack2[t].ptr, pb.ptr, total, cudaMemcpyHostToDevice, cs) != cudaSuccess ||
        cudaEventRecord(pb.ev, cs) != cudaSuccess ||
        cudaMemsetAsync(kp.d_counters2[t].ptr, 0, kp.d_counters2[t].cap, cs) != cudaSuccess ||
        cudaEventRecord(kp.ev_copied, cs) != cudaSuccess)
        return CP_ERR_CUDA;
    pb.used = true;
    // caller's stream: everything enqueued so far may read the old pair; the launches that follow wait for the copy
    if (cudaEventRecord(kp.ev_users[kp.buf], stream) != cudaSuccess || cudaStreamWaitEvent(stream, kp.ev_copied, 0) != cudaSuccess)
        return CP_ERR_CUDA;
    kp.users_recorded[kp.buf] = true;
    kp.buf = t;
    uint8_t *base = (uint8_t *)kp.d_pack2[t].ptr;
    kp.p_groups = base + off[0]; kp.p_tiles = base + off[1]; kp.p_tile_recs = base + off[2];
    kp.p_combines = base + off[3]; kp.p_cunits = base + off[4];
    kp.p_counters = kp.d_counters2[t].ptr;
    kp.counter_set = 0;
    pool->n_h2d_bytes += total;
    kp.uploaded = true;
    return CP_OK;
}

}  // namespace

// =========================================================================== C ABI
extern "C" {

const char *cp_status_string(cp_status s)
{
    switch (s) {
    case CP_OK: return "CP_OK";
    case CP_ERR_INVALID_ARG: return "CP_ERR_INVALID_ARG";
    case CP_ERR_NO_PAGES: return "CP_ERR_NO_PAGES";
    case CP_ERR_PAGE_RANGE: return "CP_ERR_PAGE_RANGE";
    case CP_ERR_PAGE_IN_USE: return "CP_ERR_PAGE_IN_USE";
    case CP_ERR_UNKNOWN_REQUEST: return "CP_ERR_UNKNOWN_REQUEST";
    case CP_ERR_UNSUPPORTED: return "CP_ERR_UNSUPPORTED";
    case CP_ERR_WORKSPACE: return "CP_ERR_WORKSPACE";
    case CP_ERR_CUDA: return "CP_ERR_CUDA";
    case CP_ERR_TOO_LARGE: return "CP_ERR_TOO_LARGE";
    default: return "CP_ERR_?";
    }
}

cp_status cp_pool_create(void *arena_dev, uint64_t arena_bytes, uint32_t page_tokens,
                         uint32_t page_bytes, uint32_t num_pages, const cp_model_cfg *models,
                         int32_t n_models, int32_t max_requests, int32_t max_pages_per_request,
                         cp_pool **out)
{
    if (!out) return CP_ERR_INVALID_ARG;
    *out = nullptr;
    if (!arena_dev || !models || n_models < 1 || max_requests < 1 || max_pages_per_request < 1)
        return CP_ERR_INVALID_ARG;
    if (page_tokens < 1 || page_tokens > 256 || page_bytes < 16 || page_bytes % 16 || num_pages < 1)
        return CP_ERR_INVALID_ARG;
    if (num_pages > (uint32_t)INT32_MAX) return CP_ERR_INVALID_ARG;
    if ((uint64_t)num_pages * page_bytes > arena_bytes) return CP_ERR_INVALID_ARG;
    if (((uintptr_t)arena_dev & 255u) != 0) return CP_ERR_INVALID_ARG;
    if ((uint64_t)max_requests * (uint64_t)max_pages_per_request > (1ull << 31)) return CP_ERR_INVALID_ARG;
    for (int i = 0; i < n_models; ++i)
        if (!model_supported(models[i], page_tokens, page_bytes)) return CP_ERR_UNSUPPORTED;
    cp_pool *p = new (std::nothrow) cp_pool();
    if (!p) return CP_ERR_INVALID_ARG;
    try {
        p->arena = (uint8_t *)arena_dev; p->arena_bytes = arena_bytes;
        p->P = page_tokens; p->page_bytes = page_bytes; p->num_pages = num_pages;
        p->models.assign(models, models + n_models);
        p->max_requests = max_requests; p->max_ppr = max_pages_per_request;
        p->owner.assign(num_pages, -1);
        p->n_free = num_pages;
        p->reqs.resize(max_requests);
        p->h_ctx.assign(max_requests, 0);
    } catch (...) {
        delete p;
        return CP_ERR_INVALID_ARG;
    }
    *out = p;
    return CP_OK;
}

cp_status cp_pool_create_vmm(uint64_t physical_budget_bytes, uint32_t page_tokens, uint32_t page_bytes,
                             const cp_model_cfg *models, int32_t n_models, int32_t max_requests,
                             int32_t max_pages_per_request, cp_pool **out)
{
    if (!out) return CP_ERR_INVALID_ARG;
    *out = nullptr;
    if (!models || n_models < 1 || max_requests < 1 || max_pages_per_request < 1 || physical_budget_bytes == 0)
        return CP_ERR_INVALID_ARG;
    if (page_tokens < 1 || page_tokens > 256 || page_bytes < 16 || page_bytes % 16) return CP_ERR_INVALID_ARG;
    for (int i = 0; i < n_models; ++i)
        if (!model_supported(models[i], page_tokens, page_bytes)) return CP_ERR_UNSUPPORTED;
    VmmArena *vmm = nullptr;
    const int rc = vmm_create(&vmm, (uint64_t)max_pages_per_request * page_bytes, max_requests, physical_budget_bytes,
                              page_bytes);
    if (rc != 0) return CP_ERR_CUDA;
    const uint64_t slot_pages = vmm->slot_bytes / page_bytes;
    const uint64_t num_pages = slot_pages * (uint64_t)max_requests;
    if (num_pages > (uint64_t)INT32_MAX || vmm->budget_chunks == 0) {
        vmm_destroy(vmm);
        return CP_ERR_INVALID_ARG;
    }
    cp_pool *p = nullptr;
    const cp_status st = cp_pool_create((void *)(uintptr_t)vmm->base, vmm->va_bytes, page_tokens, page_bytes,
                                        (uint32_t)num_pages, models, n_models, max_requests,
                                        max_pages_per_request, &p);
    if (st != CP_OK) {
        vmm_destroy(vmm);
        return st;
    }
    p->vmm = vmm;
    p->slot_pages = (uint32_t)slot_pages;
    *out = p;
    return CP_OK;
}

cp_status cp_pool_vmm_info(const cp_pool *pool, void **arena_dev, uint64_t *va_bytes, uint64_t *chunk_bytes,
                           uint32_t *slot_pages, uint32_t *chunks_mapped, uint32_t *chunks_budget)
{
    if (!pool || !pool->vmm) return CP_ERR_INVALID_ARG;
    if (arena_dev) *arena_dev = (void *)(uintptr_t)pool->vmm->base;
    if (va_bytes) *va_bytes = pool->vmm->va_bytes;
    if (chunk_bytes) *chunk_bytes = pool->vmm->chunk_bytes;
    if (slot_pages) *slot_pages = pool->slot_pages;
    if (chunks_mapped) *chunks_mapped = vmm_chunks_mapped(pool->vmm);
    if (chunks_budget) *chunks_budget = pool->vmm->budget_chunks;
    return CP_OK;
}

cp_status cp_pool_free(cp_pool *pool)
{
    if (!pool) return CP_OK;
    if (pool->dev_ready || pool->vmm) cudaDeviceSynchronize();
    if (pool->vmm) { vmm_destroy(pool->vmm); pool->vmm = nullptr; }
    if (pool->ev_switch) cudaEventDestroy(pool->ev_switch);
    if (pool->ev_fork) cudaEventDestroy(pool->ev_fork);
    if (pool->ev_join) cudaEventDestroy(pool->ev_join);
    if (pool->side_stream) cudaStreamDestroy(pool->side_stream);
    if (pool->copy_stream) cudaStreamDestroy(pool->copy_stream);
    if (pool->ev_tab) cudaEventDestroy(pool->ev_tab);
    for (auto &pb : pool->tab_pin) { if (pb.ptr) cudaFreeHost(pb.ptr); if (pb.ev) cudaEventDestroy(pb.ev); }
    pool->d_page_table.release(); pool->d_ctx.release(); pool->d_models.release(); pool->d_append.release(); pool->d_timeline.release();
    for (int k = 0; k < 2; ++k) {
        pool->plan[k].d_pack2[0].release(); pool->plan[k].d_pack2[1].release(); pool->plan[k].d_counters2[0].release(); pool->plan[k].d_counters2[1].release();
        for (auto &e : pool->plan[k].ev_users) if (e) cudaEventDestroy(e);
        if (pool->plan[k].ev_copied) cudaEventDestroy(pool->plan[k].ev_copied);
        for (auto &pb : pool->plan[k].pin) { if (pb.ptr) cudaFreeHost(pb.ptr); if (pb.ev) cudaEventDestroy(pb.ev); }
    }
    {
        KindPlan &kp = pool->splan.kp;
        kp.d_pack2[0].release(); kp.d_pack2[1].release(); kp.d_counters2[0].release(); kp.d_counters2[1].release();
        for (auto &e : kp.ev_users) if (e) cudaEventDestroy(e);
        if (kp.ev_copied) cudaEventDestroy(kp.ev_copied);
        pool->splan.d_stages.release(); pool->splan.d_gate.release();
        for (auto &pb : kp.pin) { if (pb.ptr) cudaFreeHost(pb.ptr); if (pb.ev) cudaEventDestroy(pb.ev); }
    }
    delete pool;
    return CP_OK;
}

cp_status cp_pool_map_pages(cp_pool *pool, int32_t request_id, int32_t model_id,
                            const int32_t *page_ids_host, int32_t n_page_ids, int32_t context_len)
{
    if (!pool || request_id < 0 || request_id >= pool->max_requests) return CP_ERR_INVALID_ARG;
    if (model_id < 0 || model_id >= (int)pool->models.size()) return CP_ERR_INVALID_ARG;
    if (n_page_ids < 0 || context_len < 1) return CP_ERR_INVALID_ARG;
    Request &r = pool->reqs[request_id];
    if (r.live && r.model != model_id) return CP_ERR_INVALID_ARG;
    if (r.live && context_len < r.ctx) return CP_ERR_INVALID_ARG;
    const cp_model_cfg &m = pool->models[model_id];
    if (n_page_ids % m.n_kv_heads != 0) return CP_ERR_UNSUPPORTED;
    const size_t have = r.live ? r.pages.size() : 0;
    const size_t total = have + (size_t)n_page_ids;
    if (total > (size_t)pool->max_ppr) return CP_ERR_INVALID_ARG;
    const uint64_t capacity_tokens = (uint64_t)(total / m.n_kv_heads) * pool->P;
    if ((uint64_t)context_len > capacity_tokens) return CP_ERR_INVALID_ARG;

    std::vector<int32_t> fresh;
    if (n_page_ids > 0) {
        fresh.resize(n_page_ids);
        if (pool->vmm) {
            // contiguous virtual KV: the ids are the next entries of the request's slot; the physical
            // chunks under them are mapped below, after every check has passed
            if (page_ids_host) return CP_ERR_INVALID_ARG;
            for (int i = 0; i < n_page_ids; ++i)
                fresh[i] = (int32_t)((size_t)request_id * pool->slot_pages + have + i);
            const int rc = vmm_back(pool->vmm, request_id, (uint64_t)total * pool->page_bytes);
            if (rc == 3) return CP_ERR_NO_PAGES;
            if (rc != 0) return CP_ERR_CUDA;
        } else if (page_ids_host) {
            for (int i = 0; i < n_page_ids; ++i) {
                const int32_t pid = page_ids_host[i];
                if (pid < 0 || (uint32_t)pid >= pool->num_pages) return CP_ERR_PAGE_RANGE;
                fresh[i] = pid;
            }
            for (int i = 0; i < n_page_ids; ++i)
                if (pool->owner[fresh[i]] != -1) return CP_ERR_PAGE_IN_USE;
            std::vector<int32_t> s(fresh);
            std::sort(s.begin(), s.end());
            for (int i = 1; i < n_page_ids; ++i)
                if (s[i] == s[i - 1]) return CP_ERR_PAGE_IN_USE;
        } else {
            if ((uint32_t)n_page_ids > pool->n_free) return CP_ERR_NO_PAGES;
            uint32_t cur = pool->alloc_cursor;
            for (int i = 0; i < n_page_ids;) {
                if (pool->owner[cur] == -1) fresh[i++] = (int32_t)cur;
                cur = (cur + 1) % pool->num_pages;
            }
            pool->alloc_cursor = cur;
        }
    }
    // commit (nothing below can fail)
    const int old_planned = r.live ? ceil_div(r.ctx, (int)pool->P) : -1;
    if (!r.live) {
        r.live = true; r.model = model_id; r.pages.clear(); r.uploaded = 0;
    }
    for (int32_t pid : fresh) pool->owner[pid] = request_id;
    pool->n_free -= (uint32_t)fresh.size();
    r.pages.insert(r.pages.end(), fresh.begin(), fresh.end());
    r.ctx = context_len;
    pool->h_ctx[request_id] = context_len;
    pool->ctx_dirty_lo = std::min(pool->ctx_dirty_lo, request_id);
    pool->ctx_dirty_hi = std::max(pool->ctx_dirty_hi, request_id);
    if (ceil_div(context_len, (int)pool->P) != old_planned) pool->topo_version++;
    return CP_OK;
}

cp_status cp_pool_unmap_request(cp_pool *pool, int32_t request_id)
{
    if (!pool || request_id < 0 || request_id >= pool->max_requests) return CP_ERR_INVALID_ARG;
    Request &r = pool->reqs[request_id];
    if (!r.live) return CP_ERR_UNKNOWN_REQUEST;
    for (int32_t pid : r.pages) pool->owner[pid] = -1;
    pool->n_free += (uint32_t)r.pages.size();
    if (pool->vmm) {
        // kernels that may still read the slot must have finished before its memory is unmapped
        cudaDeviceSynchronize();
        if (vmm_release_slot(pool->vmm, request_id) != 0) { cudaGetLastError(); }
    }
    r = Request();
    pool->topo_version++;
    return CP_OK;
}

cp_status cp_pool_request_info(const cp_pool *pool, int32_t request_id, int32_t *model_id,
                               int32_t *context_len, int32_t *n_page_ids,
                               int32_t *page_ids_out_host, int32_t cap)
{
    if (!pool || request_id < 0 || request_id >= pool->max_requests) return CP_ERR_INVALID_ARG;
    const Request &r = pool->reqs[request_id];
    if (!r.live) return CP_ERR_UNKNOWN_REQUEST;
    if (model_id) *model_id = r.model;
    if (context_len) *context_len = r.ctx;
    if (n_page_ids) *n_page_ids = (int32_t)r.pages.size();
    if (page_ids_out_host && cap > 0)
        std::memcpy(page_ids_out_host, r.pages.data(), sizeof(int32_t) * std::min<size_t>(cap, r.pages.size()));
    return CP_OK;
}

cp_status cp_pool_stats(const cp_pool *pool, uint32_t *free_pages, uint32_t *used_pages)
{
    if (!pool) return CP_ERR_INVALID_ARG;
    if (pool->vmm) {
        // physical terms: pages that the chunks still available could hold / pages mapped to requests
        if (free_pages) *free_pages = (uint32_t)((uint64_t)vmm_chunks_available(pool->vmm) * pool->vmm->chunk_bytes / pool->page_bytes);
        if (used_pages) *used_pages = pool->num_pages - pool->n_free;
        return CP_OK;
    }
    if (free_pages) *free_pages = pool->n_free;
    if (used_pages) *used_pages = pool->num_pages - pool->n_free;
    return CP_OK;
}

cp_status cp_pool_set_option(cp_pool *pool, int32_t key, int64_t value)
{
    if (!pool) return CP_ERR_INVALID_ARG;
    switch (key) {
    case CP_OPT_KERNEL:
        if (value < 0 || value > 3) return CP_ERR_INVALID_ARG;
        pool->opt_kernel = (int)value; break;
    case CP_OPT_NUM_CTAS:
        if (value < 0 || value > 65536) return CP_ERR_INVALID_ARG;
        pool->opt_num_ctas = (int)value; break;
    case CP_OPT_WAVES_X16:
        if (value < 1 || value > 4096) return CP_ERR_INVALID_ARG;
        pool->opt_waves_x16 = (int)value; break;
    case CP_OPT_MIN_TILE_PAGES:
        if (value < 1 || value > (1 << 20)) return CP_ERR_INVALID_ARG;
        pool->opt_min_tile_pages = (int)value; break;
    case CP_OPT_VMM_TABLE:
        if (value < 0 || value > 1) return CP_ERR_INVALID_ARG;
        pool->opt_vmm_table = (int)value; break;
    case CP_OPT_HOST_ZERO_COPY:
        if (value < 0 || value > 1) return CP_ERR_INVALID_ARG;
        pool->opt_host_zero_copy = (int)value; break;
    case CP_OPT_STATIC_PCT:
        if (value < 0 || value > 100) return CP_ERR_INVALID_ARG;
        pool->opt_static_pct = (int)value; break;
    case CP_OPT_TAIL_TILE_SLICES:
        if (value < 1 || value > 4096) return CP_ERR_INVALID_ARG;
        pool->opt_tail_slices = (int)value; break;
    case CP_OPT_TIMELINE:
        if (value < 0 || value > 1) return CP_ERR_INVALID_ARG;
        pool->opt_timeline = (int)value; return CP_OK;      // no effect on the plan
    default: return CP_ERR_INVALID_ARG;
    }
    pool->plan_valid = false;
    pool->splan.valid = false;
    return CP_OK;
}

cp_status cp_pool_counters(const cp_pool *pool, uint64_t *kernel_launches, uint64_t *plan_builds,
                           uint64_t *metadata_h2d_bytes)
{
    if (!pool) return CP_ERR_INVALID_ARG;
    if (kernel_launches) *kernel_launches = pool->n_launches;
    if (plan_builds) *plan_builds = pool->n_plan_builds;
    if (metadata_h2d_bytes) *metadata_h2d_bytes = pool->n_h2d_bytes;
    return CP_OK;
}

cp_status cp_pool_read_timeline(cp_pool *pool, uint64_t *stamps_out_host, int32_t cap_ctas, int32_t *n_ctas_out)
{
    if (!pool || cap_ctas < 0 || (cap_ctas > 0 && !stamps_out_host)) return CP_ERR_INVALID_ARG;
    if (n_ctas_out) *n_ctas_out = 0;
    if (!pool->d_timeline.ptr) return CP_OK;
    if (cudaDeviceSynchronize() != cudaSuccess) { cudaGetLastError(); return CP_ERR_CUDA; }
    const int n = std::min<int>(cap_ctas, pool->n_sm);
    if (n > 0 && cudaMemcpy(stamps_out_host, pool->d_timeline.ptr, (size_t)n * kTimelineSlots * sizeof(uint64_t),
                            cudaMemcpyDeviceToHost) != cudaSuccess) {
        cudaGetLastError();
        return CP_ERR_CUDA;
    }
    if (n_ctas_out) *n_ctas_out = pool->n_sm;
    return CP_OK;
}

cp_status cp_decode_plan(cp_pool *pool, const int32_t *request_ids_host, int32_t n_requests,
                         cp_tile_info *tiles_out, int32_t cap, int32_t *n_tiles_out,
                         int32_t *n_groups_out)
{
    cp_status st = check_batch(pool, request_ids_host, n_requests);
    if (st != CP_OK) return st;
    ensure_plan(pool, request_ids_host, n_requests);
    int nt = 0, ng = 0;
    for (int k = 0; k < 2; ++k) {
        const KindPlan &kp = pool->plan[k];
        for (const Tile &t : kp.tiles) {
            if (tiles_out && nt < cap) {
                const Group &g = kp.groups[t.group];
                tiles_out[nt] = cp_tile_info{g.batch_index, g.kv_head, t.split, g.n_splits,
                                             t.page_begin, t.page_end};
            }
            ++nt;
        }
        ng += (int)kp.groups.size();
    }
    if (n_tiles_out) *n_tiles_out = nt;
    if (n_groups_out) *n_groups_out = ng;
    return CP_OK;
}

cp_status cp_decode_workspace_bytes(cp_pool *pool, const int32_t *request_ids_host,
                                    int32_t n_requests, uint64_t *bytes_out)
{
    if (!bytes_out) return CP_ERR_INVALID_ARG;
    cp_status st = check_batch(pool, request_ids_host, n_requests);
    if (st != CP_OK) return st;
    ensure_plan(pool, request_ids_host, n_requests);
    *bytes_out = pool->plan_ws_floats * 4;
    return CP_OK;
}

cp_status cp_pool_gather_kv(cp_pool *pool, int32_t request_id, void *k_out_dev, void *v_out_dev,
                            void *stream)
{
    if (!pool || request_id < 0 || request_id >= pool->max_requests || !k_out_dev)
        return CP_ERR_INVALID_ARG;
    Request &r = pool->reqs[request_id];
    if (!r.live) return CP_ERR_UNKNOWN_REQUEST;
    if (((uintptr_t)k_out_dev & 15u) || ((uintptr_t)v_out_dev & 15u)) return CP_ERR_INVALID_ARG;
    cp_status st = ensure_device(pool);
    if (st != CP_OK) return st;
    cudaStream_t s = (cudaStream_t)stream;
    st = adopt_stream(pool, s);
    if (st != CP_OK) return st;
    st = flush_tables(pool, s);
    if (st != CP_OK) return st;
    const cp_model_cfg &m = pool->models[r.model];
    launch_gather(pool->arena, pool->P, pool->page_bytes,
                  (const int32_t *)pool->d_page_table.ptr + (size_t)request_id * pool->max_ppr,
                  m.kind, m.n_kv_heads, m.head_dim_qk, m.head_dim_v, r.ctx, k_out_dev, v_out_dev,
                  pool->n_sm, s);
    pool->n_launches++;
    if (cudaGetLastError() != cudaSuccess) return CP_ERR_CUDA;
    return CP_OK;
}

namespace {

// Host half of an append (cp_pool_append_kv, cp_decode_step): validate the whole batch first (all-or-nothing:
// capacity of the page lists, page budget), then commit -- new pages from the free list where a position opens
// a logical page, context lengths + 1 -- and describe the device half in recs.  grew[b] = pages added to
// request b (what append_rollback takes back).
cp_status append_host(cp_pool *pool, const int32_t *ids, int n, bool need_v_ptr, const void *v_new_dev,
                      std::vector<AppendRec> &recs, std::vector<int> &grew)
{
    const int P = (int)pool->P;
    uint32_t need_pages = 0, need_chunks = 0;
    bool any_v = false;
    for (int b = 0; b < n; ++b) {
        const Request &r = pool->reqs[ids[b]];
        const cp_model_cfg &m = pool->models[r.model];
        if (m.kind != CP_KIND_MLA) any_v = true;
        if (r.ctx == INT32_MAX) return CP_ERR_INVALID_ARG;
        const size_t have_lp = r.pages.size() / m.n_kv_heads;
        if ((size_t)(r.ctx / P) >= have_lp) {                 // position r.ctx opens a new logical page
            if (r.pages.size() + m.n_kv_heads > (size_t)pool->max_ppr) return CP_ERR_INVALID_ARG;
            need_pages += (uint32_t)m.n_kv_heads;
            if (pool->vmm)
                need_chunks += vmm_chunks_missing(pool->vmm, ids[b], (uint64_t)(r.pages.size() + m.n_kv_heads) * pool->page_bytes);
        }
    }
    if (need_v_ptr && any_v && !v_new_dev) return CP_ERR_INVALID_ARG;
    if (pool->vmm ? need_chunks > vmm_chunks_available(pool->vmm) : need_pages > pool->n_free) return CP_ERR_NO_PAGES;
    const cp_status st = ensure_device(pool);
    if (st != CP_OK) return st;
    recs.resize(n);
    grew.assign(n, 0);
    int64_t ko = 0, vo = 0;
    for (int b = 0; b < n; ++b) {
        const int rid = ids[b];
        Request &r = pool->reqs[rid];
        const cp_model_cfg &m = pool->models[r.model];
        if ((size_t)(r.ctx / P) >= r.pages.size() / m.n_kv_heads && pool->vmm) {
            const uint64_t total = r.pages.size() + m.n_kv_heads;
            if (vmm_back(pool->vmm, rid, total * pool->page_bytes) != 0) return CP_ERR_CUDA;   // budget checked above
            for (int i = 0; i < m.n_kv_heads; ++i) {
                const int32_t pid = (int32_t)((size_t)rid * pool->slot_pages + r.pages.size());
                pool->owner[pid] = rid; r.pages.push_back(pid);
            }
            pool->n_free -= (uint32_t)m.n_kv_heads;
            grew[b] = m.n_kv_heads;
        } else if ((size_t)(r.ctx / P) >= r.pages.size() / m.n_kv_heads) {
            uint32_t cur = pool->alloc_cursor;
            for (int i = 0; i < m.n_kv_heads;) {
                if (pool->owner[cur] == -1) { pool->owner[cur] = rid; r.pages.push_back((int32_t)cur); ++i; }
                cur = (cur + 1) % pool->num_pages;
            }
            pool->alloc_cursor = cur;
            pool->n_free -= (uint32_t)m.n_kv_heads;
            grew[b] = m.n_kv_heads;
        }
        recs[b].req = rid; recs[b].model = r.model; recs[b].pos = r.ctx; recs[b].pad = 0;
        recs[b].k_off = ko; recs[b].v_off = vo;
        ko += (int64_t)m.n_kv_heads * m.head_dim_qk;
        if (m.kind != CP_KIND_MLA) vo += (int64_t)m.n_kv_heads * m.head_dim_v;
        const int old_planned = ceil_div(r.ctx, P);
        r.ctx += 1;
        pool->h_ctx[rid] = r.ctx;
        pool->ctx_dirty_lo = std::min(pool->ctx_dirty_lo, rid);
        pool->ctx_dirty_hi = std::max(pool->ctx_dirty_hi, rid);
        if (ceil_div(r.ctx, P) != old_planned) pool->topo_version++;
    }
    return CP_OK;
}

// Take back what append_host committed (a cp_decode_step that finds its workspace too small): the token is not
// appended, the pages it opened return to the free list (a CUDA-VMM chunk mapped for them stays mapped, parked
// under the request's slot).  Nothing has been sent to the device yet.
void append_rollback(cp_pool *pool, const int32_t *ids, int n, const std::vector<int> &grew)
{
    for (int b = 0; b < n; ++b) {
        const int rid = ids[b];
        Request &r = pool->reqs[rid];
        for (int i = 0; i < grew[b]; ++i) {
            pool->owner[r.pages.back()] = -1;
            r.pages.pop_back();
        }
        pool->n_free += (uint32_t)grew[b];
        r.uploaded = std::min(r.uploaded, r.pages.size());
        r.ctx -= 1;
        pool->h_ctx[rid] = r.ctx;
        pool->ctx_dirty_lo = std::min(pool->ctx_dirty_lo, rid);
        pool->ctx_dirty_hi = std::max(pool->ctx_dirty_hi, rid);
    }
    pool->topo_version++;
}

cp_status launch_append_recs(cp_pool *pool, const std::vector<AppendRec> &recs, const void *k_new_dev, const void *v_new_dev,
                             cudaStream_t s)
{
    if (recs.empty()) return CP_OK;
    if (pool->d_append.ensure(recs.size() * sizeof(AppendRec)) != cudaSuccess) { cudaGetLastError(); return CP_ERR_CUDA; }
    if (cudaMemcpyAsync(pool->d_append.ptr, recs.data(), recs.size() * sizeof(AppendRec), cudaMemcpyHostToDevice, s) != cudaSuccess)
        return CP_ERR_CUDA;
    pool->n_h2d_bytes += recs.size() * sizeof(AppendRec);
    launch_append(pool->arena, pool->P, pool->page_bytes, (const int32_t *)pool->d_page_table.ptr, pool->max_ppr,
                  (const DevModel *)pool->d_models.ptr, (const AppendRec *)pool->d_append.ptr, (int)recs.size(),
                  (const uint16_t *)k_new_dev, (const uint16_t *)v_new_dev, s);
    pool->n_launches++;
    if (cudaGetLastError() != cudaSuccess) return CP_ERR_CUDA;
    return CP_OK;
}

}  // namespace

cp_status cp_pool_append_kv(cp_pool *pool, const int32_t *request_ids_host, int32_t n_requests,
                            const void *k_new_dev, const void *v_new_dev, void *stream)
{
    cp_status st = check_batch(pool, request_ids_host, n_requests);
    if (st != CP_OK) return st;
    if (!k_new_dev || ((uintptr_t)k_new_dev & 15u) || ((uintptr_t)v_new_dev & 15u)) return CP_ERR_INVALID_ARG;
    std::vector<AppendRec> recs;
    std::vector<int> grew;
    st = append_host(pool, request_ids_host, n_requests, true, v_new_dev, recs, grew);
    if (st != CP_OK) return st;
    cudaStream_t s = (cudaStream_t)stream;
    st = adopt_stream(pool, s);
    if (st != CP_OK) return st;
    st = flush_tables(pool, s);                            // new page ids (and context lengths) to the device
    if (st != CP_OK) return st;
    return launch_append_recs(pool, recs, k_new_dev, v_new_dev, s);
}

cp_status cp_decode_attention(cp_pool *pool, const int32_t *request_ids_host, int32_t n_requests,
                              const void *q_dev, float *out_dev, float *lse_dev,
                              void *workspace_dev, uint64_t workspace_bytes, void *stream)
{
    cp_status st = check_batch(pool, request_ids_host, n_requests);
    if (st != CP_OK) return st;
    if (!q_dev || !out_dev || !lse_dev) return CP_ERR_INVALID_ARG;
    if (((uintptr_t)q_dev & 15u) || ((uintptr_t)out_dev & 15u) || ((uintptr_t)lse_dev & 3u))
        return CP_ERR_INVALID_ARG;
    st = ensure_device(pool);
    if (st != CP_OK) return st;
    ensure_plan(pool, request_ids_host, n_requests);
    if (pool->plan_ws_floats * 4 > workspace_bytes) return CP_ERR_WORKSPACE;
    if (pool->plan_ws_floats && (!workspace_dev || ((uintptr_t)workspace_dev & 15u))) return CP_ERR_WORKSPACE;
    cudaStream_t s = (cudaStream_t)stream;
    st = adopt_stream(pool, s);
    if (st != CP_OK) return st;
    st = flush_tables(pool, s);
    if (st != CP_OK) return st;

    // A batch with both attention kinds: everything either launch reads is uploaded on the caller's stream first;
    // then the second kind's kernel runs beside the first on a stream of the pool's own (fork here, join below).
    const bool both_kinds = !pool->plan[0].tiles.empty() && !pool->plan[1].tiles.empty();
    cudaStream_t s_main = s;
    for (int k = 0; k < 2; ++k) {
        if (pool->plan[k].tiles.empty()) continue;
        st = upload_plan(pool, pool->plan[k], s_main);
        if (st != CP_OK) return st;
    }
    if (pool->opt_timeline) {
        const size_t tb = (size_t)pool->n_sm * kTimelineSlots * sizeof(unsigned long long);
        if (pool->d_timeline.ensure(tb) != cudaSuccess || cudaMemsetAsync(pool->d_timeline.ptr, 0, tb, s_main) != cudaSuccess) {
            cudaGetLastError();
            return CP_ERR_CUDA;
        }
    }
    if (both_kinds) {
        if ((!pool->side_stream && cudaStreamCreateWithFlags(&pool->side_stream, cudaStreamNonBlocking) != cudaSuccess) ||
            (!pool->ev_fork && cudaEventCreateWithFlags(&pool->ev_fork, cudaEventDisableTiming) != cudaSuccess) ||
            (!pool->ev_join && cudaEventCreateWithFlags(&pool->ev_join, cudaEventDisableTiming) != cudaSuccess) ||
            cudaEventRecord(pool->ev_fork, s_main) != cudaSuccess ||
            cudaStreamWaitEvent(pool->side_stream, pool->ev_fork, 0) != cudaSuccess) {
            cudaGetLastError();
            return CP_ERR_CUDA;
        }
    }
    for (int k = 0; k < 2; ++k) {
        KindPlan &kp = pool->plan[k];
        if (kp.tiles.empty()) continue;
        s = (both_kinds && k == 1) ? pool->side_stream : s_main;
        DecodeParams prm;
        std::memset(&prm, 0, sizeof(prm));            // every field a launch does not use is null / 0
        prm.arena = pool->arena; prm.page_tokens = pool->P; prm.page_bytes = pool->page_bytes;
        prm.page_table = (const int32_t *)pool->d_page_table.ptr; prm.max_ppr = pool->max_ppr;
        prm.slot_pages = (pool->vmm && !pool->opt_vmm_table) ? (int32_t)pool->slot_pages : 0;
        prm.req_ctx = (const int32_t *)pool->d_ctx.ptr + (size_t)pool->ctx_cur * pool->max_requests;
        prm.models = (const DevModel *)pool->d_models.ptr;
        prm.groups = (const Group *)kp.p_groups;
        prm.tiles = (const Tile *)kp.p_tiles;
        prm.tile_recs = (const TileRec *)kp.p_tile_recs;
        prm.combines = (const Combine *)kp.p_combines;
        prm.cunits = (const CombineUnit *)kp.p_cunits;
        prm.n_tiles = (int)kp.tiles.size(); prm.n_combines = (int)kp.combines.size();
        prm.n_static_slots = 0;
        prm.n_combine_units = prm.n_combines;
        prm.n_groups = (int)kp.groups.size();
        prm.q = (const uint16_t *)q_dev; prm.out = out_dev; prm.lse = lse_dev;
        prm.workspace = (float *)workspace_dev;
        const size_t set_ints = 32 + kp.groups.size() * (size_t)kCounterStride;
        prm.work_counter = (int32_t *)kp.p_counters + kp.counter_set * set_ints;
        prm.group_counters = prm.work_counter + 32;
        prm.reset_counters = (int32_t *)kp.p_counters + (1 - kp.counter_set) * set_ints;
        prm.stages = nullptr; prm.stage_done = nullptr; prm.n_stages = 0; prm.q_len = pool->qlen;
        prm.published = nullptr; prm.gate_flag = nullptr; prm.gate_timeout_us = 0;
        prm.timeline = nullptr;
        prm.app_k = pool->step_k; prm.app_v = pool->step_v;
        if (pool->step_ctx_on_device) {
            // fused decode step whose kernel advances the context table itself: it reads table ctx_cur (+ 1 for the
            // batch's requests) and writes the other one for the launches that follow
            prm.ctx_add = 1;
            prm.req_ctx_next = (int32_t *)pool->d_ctx.ptr + (size_t)(1 - pool->ctx_cur) * pool->max_requests;
            prm.max_requests = pool->max_requests;
        }
        if (pool->opt_timeline && !(both_kinds && k == 1)) prm.timeline = (unsigned long long *)pool->d_timeline.ptr;
        kp.counter_set ^= 1;
        const int n_ctas = pool->kind_ctas[k];
        cudaError_t e;
        if (k == CP_KIND_KV && kp.use_kvt && pool->kv_tmap_ok) {
            prm.n_combine_units = (int)kp.cunits.size();
            prm.n_tiles = (int)kp.tile_recs.size();          // static slots (some empty) + dynamic tiles
            prm.n_static_slots = kp.n_static_slots;
            e = launch_decode_kvt(prm, pool->kv_tmap, (int)(pool->page_bytes / 256), kp.grid, kp.max_group, s);
        } else if (k == CP_KIND_KV && kp.use_kvt) {
            return CP_ERR_UNSUPPORTED;      // planned for the tcgen05 kernel but no tensor map (cannot happen: same conditions)
        } else if (k == CP_KIND_KV && pool->opt_kernel != 1 && kp.all_fast && pool->kv_tmap_ok) {
            // warp-sized combine units, popped warp by warp after the tiles
            prm.n_combine_units = (int)kp.cunits.size();
            e = launch_decode_kv(prm, pool->kv_tmap, (int)(pool->page_bytes / 256),
                                 std::min(n_ctas, pool->n_sm), s);
        } else if (k == CP_KIND_MLA && pool->opt_kernel == 0 && kp.all_fast && pool->mla2_tmap_ok) {
            prm.n_combine_units = (int)kp.cunits.size();
            e = launch_decode_mla2(prm, pool->mla2_tmap9, pool->mla2_tmap2, (int)(pool->page_bytes / 1152),
                                   std::min(n_ctas, pool->n_sm), s);
        } else if (k == CP_KIND_MLA && pool->opt_kernel != 1 && kp.all_fast && pool->mla_tmap_ok) {
            prm.n_combine_units = (int)kp.cunits.size();
            e = launch_decode_mla(prm, pool->mla_tmap, (int)(pool->page_bytes / 1152),
                                  std::min(n_ctas, pool->n_sm), s);
        } else
            e = launch_decode_generic(prm, kp.max_dk, kp.max_dv, k == CP_KIND_KV, kp.max_splits,
                                      std::min(n_ctas, pool->n_sm), s);
        pool->n_launches++;
        if (e != cudaSuccess) return CP_ERR_CUDA;
    }
    if (both_kinds &&
        (cudaEventRecord(pool->ev_join, pool->side_stream) != cudaSuccess || cudaStreamWaitEvent(s_main, pool->ev_join, 0) != cudaSuccess)) {
        cudaGetLastError();
        return CP_ERR_CUDA;
    }
    return CP_OK;
}

// ------------------------------------------------------------------ append + attend in one call
cp_status cp_decode_step(cp_pool *pool, const int32_t *request_ids_host, int32_t n_requests,
                         const void *k_new_dev, const void *v_new_dev, const void *q_dev, float *out_dev,
                         float *lse_dev, void *workspace_dev, uint64_t workspace_bytes, void *stream)
{
    cp_status st = check_batch(pool, request_ids_host, n_requests);
    if (st != CP_OK) return st;
    if (!k_new_dev || ((uintptr_t)k_new_dev & 15u) || ((uintptr_t)v_new_dev & 15u)) return CP_ERR_INVALID_ARG;
    if (!q_dev || !out_dev || !lse_dev) return CP_ERR_INVALID_ARG;
    if (((uintptr_t)q_dev & 15u) || ((uintptr_t)out_dev & 15u) || ((uintptr_t)lse_dev & 3u)) return CP_ERR_INVALID_ARG;
    std::vector<AppendRec> recs;
    std::vector<int> grew;
    cudaStream_t s = (cudaStream_t)stream;
    st = ensure_device(pool);
    if (st != CP_OK) return st;
    st = adopt_stream(pool, s);
    if (st != CP_OK) return st;
    st = flush_tables(pool, s);                 // whatever earlier calls left pending: the device tables are current now
    if (st != CP_OK) return st;
    st = append_host(pool, request_ids_host, n_requests, true, v_new_dev, recs, grew);
    if (st != CP_OK) return st;
    // the plan of the grown contexts decides the workspace; too small: the append is taken back, nothing changed
    ensure_plan(pool, request_ids_host, n_requests);
    if (pool->plan_ws_floats * 4 > workspace_bytes ||
        (pool->plan_ws_floats && (!workspace_dev || ((uintptr_t)workspace_dev & 15u)))) {
        append_rollback(pool, request_ids_host, n_requests, grew);
        return CP_ERR_WORKSPACE;
    }
    // Requests whose attention kernel writes the new row itself (the tcgen05 K/V kernel: the tile that holds a
    // group's last page stores the row before it requests the page) need no launch of their own; the others
    // (MLA, generic shapes, CP_OPT_KERNEL = 1 / 3) get the append kernel first.
    const bool fused_kv = pool->plan[CP_KIND_KV].use_kvt && pool->kv_tmap_ok;
    std::vector<AppendRec> sep;
    for (int b = 0; b < n_requests; ++b)
        if (!(fused_kv && pool->models[recs[b].model].kind == CP_KIND_KV)) sep.push_back(recs[b]);
    // Every request fused: the kernel also advances the context table (reads the current one + 1, writes the other
    // one for later launches), so a decode iteration uploads nothing but the ids of newly opened pages.
    const bool ctx_on_device = fused_kv && sep.empty() && pool->plan[CP_KIND_MLA].tiles.empty();
    if (ctx_on_device) { pool->ctx_dirty_lo = INT32_MAX; pool->ctx_dirty_hi = -1; }     // the only dirty entries are this step's
    st = flush_tables(pool, s);
    if (st != CP_OK) return st;
    st = launch_append_recs(pool, sep, k_new_dev, v_new_dev, s);
    if (st != CP_OK) return st;
    pool->step_k = fused_kv ? (const uint16_t *)k_new_dev : nullptr;
    pool->step_v = fused_kv ? (const uint16_t *)v_new_dev : nullptr;
    pool->step_ctx_on_device = ctx_on_device;
    st = cp_decode_attention(pool, request_ids_host, n_requests, q_dev, out_dev, lse_dev, workspace_dev, workspace_bytes, stream);
    pool->step_k = pool->step_v = nullptr;
    pool->step_ctx_on_device = false;
    if (ctx_on_device) {
        if (st == CP_OK) pool->ctx_cur ^= 1;
        else {                                   // the launch did not happen: the host values must be uploaded after all
            for (int b = 0; b < n_requests; ++b) {
                pool->ctx_dirty_lo = std::min(pool->ctx_dirty_lo, request_ids_host[b]);
                pool->ctx_dirty_hi = std::max(pool->ctx_dirty_hi, request_ids_host[b]);
            }
        }
    }
    return st;
}

cp_status cp_decode_step_workspace_bytes(cp_pool *pool, const int32_t *request_ids_host, int32_t n_requests, uint64_t *bytes_out)
{
    if (!bytes_out) return CP_ERR_INVALID_ARG;
    cp_status st = check_batch(pool, request_ids_host, n_requests);
    if (st != CP_OK) return st;
    // plan of the contexts as they will be after the append (host arithmetic only; the cached plan is dropped)
    for (int b = 0; b < n_requests; ++b) {
        if (pool->reqs[request_ids_host[b]].ctx == INT32_MAX) return CP_ERR_INVALID_ARG;
        pool->reqs[request_ids_host[b]].ctx += 1;
    }
    build_plan(pool, request_ids_host, n_requests);
    *bytes_out = pool->plan_ws_floats * 4;
    for (int b = 0; b < n_requests; ++b) pool->reqs[request_ids_host[b]].ctx -= 1;
    pool->plan_valid = false;
    return CP_OK;
}

// ------------------------------------------------------------------ q_len > 1 (SURVEY 8(f) N4 variant)
namespace {

cp_status check_qlen(cp_pool *pool, const int32_t *ids, int n, int q_len)
{
    cp_status st = check_batch(pool, ids, n);
    if (st != CP_OK) return st;
    if (q_len < 1 || q_len > 128) return CP_ERR_INVALID_ARG;
    if (q_len == 1) return CP_OK;
    if (pool->opt_kernel == 1 || !kv_fast_supported((int)pool->P)) return CP_ERR_UNSUPPORTED;
    for (int b = 0; b < n; ++b) {
        const Request &r = pool->reqs[ids[b]];
        const cp_model_cfg &m = pool->models[r.model];
        if (r.ctx < q_len) return CP_ERR_INVALID_ARG;           // the query tokens are the context's last q_len
        if (m.kind != CP_KIND_KV || m.head_dim_qk != 128 || m.head_dim_v != 128 ||
            m.n_q_heads / m.n_kv_heads * q_len > 128)
            return CP_ERR_UNSUPPORTED;
    }
    return CP_OK;
}

}  // namespace

cp_status cp_decode_workspace_bytes_qlen(cp_pool *pool, const int32_t *request_ids_host, int32_t n_requests,
                                         int32_t q_len, uint64_t *bytes_out)
{
    if (!bytes_out) return CP_ERR_INVALID_ARG;
    const cp_status st = check_qlen(pool, request_ids_host, n_requests, q_len);
    if (st != CP_OK) return st;
    pool->qlen = q_len;
    ensure_plan(pool, request_ids_host, n_requests);
    pool->qlen = 1;
    *bytes_out = pool->plan_ws_floats * 4;
    return CP_OK;
}

cp_status cp_decode_attention_qlen(cp_pool *pool, const int32_t *request_ids_host, int32_t n_requests,
                                   int32_t q_len, const void *q_dev, float *out_dev, float *lse_dev,
                                   void *workspace_dev, uint64_t workspace_bytes, void *stream)
{
    cp_status st = check_qlen(pool, request_ids_host, n_requests, q_len);
    if (st != CP_OK) return st;
    if (q_len > 1) {
        st = ensure_device(pool);                               // the fast kernel needs its tensor map
        if (st != CP_OK) return st;
        if (!pool->kv_tmap_ok) return CP_ERR_UNSUPPORTED;
    }
    pool->qlen = q_len;
    st = cp_decode_attention(pool, request_ids_host, n_requests, q_dev, out_dev, lse_dev, workspace_dev,
                             workspace_bytes, stream);
    pool->qlen = 1;
    return st;
}

// ------------------------------------------------------------------ multi-stage launch
namespace {

cp_status build_stages_plan(cp_pool *pool, int32_t n_stages, const int32_t *sizes, const int32_t *ids,
                            const int32_t *deps, float alpha)
{
    if (!pool || n_stages < 1 || n_stages > 4096 || !sizes || !ids || !deps) return CP_ERR_INVALID_ARG;
    std::vector<int32_t> key;
    key.push_back(n_stages);
    int64_t total = 0;
    for (int s = 0; s < n_stages; ++s) {
        if (sizes[s] < 1) return CP_ERR_INVALID_ARG;
        total += sizes[s];
    }
    key.insert(key.end(), sizes, sizes + n_stages);
    key.insert(key.end(), ids, ids + total);
    key.insert(key.end(), deps, deps + n_stages);
    cp_pool::StagesPlan &sp = pool->splan;
    if (sp.valid && sp.version == pool->topo_version && sp.key == key) {
        if (alpha == alpha && alpha != sp.stages[0].alpha) {       // same work list, new residual weight
            for (StageRec &sr : sp.stages) sr.alpha = alpha;
            sp.uploaded = false;
        }
        return CP_OK;
    }

    if (pool->opt_kernel == 1 || !kv_fast_supported((int)pool->P)) return CP_ERR_UNSUPPORTED;
    const int32_t *p_ids = ids;
    for (int s = 0; s < n_stages; ++s) {
        const cp_status st = check_batch(pool, p_ids, sizes[s]);
        if (st != CP_OK) return st;
        if (deps[s] >= s) return CP_ERR_INVALID_ARG;
        if (deps[s] >= 0) {
            // the dependent stage reads its predecessor's output row by row: same batch shape
            if (sizes[deps[s]] != sizes[s]) return CP_ERR_INVALID_ARG;
            const int32_t *d_ids = ids;
            for (int t = 0; t < deps[s]; ++t) d_ids += sizes[t];
            for (int b = 0; b < sizes[s]; ++b)
                if (pool->reqs[p_ids[b]].model != pool->reqs[d_ids[b]].model) return CP_ERR_INVALID_ARG;
        }
        for (int b = 0; b < sizes[s]; ++b) {
            const cp_model_cfg &m = pool->models[pool->reqs[p_ids[b]].model];
            if (m.kind != CP_KIND_KV || m.head_dim_qk != 128 || m.head_dim_v != 128 || m.n_q_heads / m.n_kv_heads > 128)
                return CP_ERR_UNSUPPORTED;
        }
        p_ids += sizes[s];
    }

    KindPlan &kp = sp.kp;
    kp.groups.clear(); kp.tiles.clear(); kp.tile_recs.clear(); kp.combines.clear(); kp.cunits.clear();
    kp.uploaded = false; kp.all_fast = true; kp.extra_counters = n_stages;
    sp.stages.assign(n_stages, StageRec());
    sp.uploaded = false;
    std::vector<int64_t> out_base(n_stages);
    std::vector<int32_t> target(n_stages);
    int64_t qb = 0, ob = 0, lb = 0, wb = 0;
    p_ids = ids;
    for (int s = 0; s < n_stages; ++s) {
        pool->plan_for_stages = true;
        build_plan(pool, p_ids, sizes[s]);
        pool->plan_for_stages = false;
        const KindPlan &src = pool->plan[CP_KIND_KV];
        const int gb = (int)kp.groups.size();
        const int cb = (int)kp.cunits.size();
        for (Group g : src.groups) {
            g.q_off += qb; g.out_off += ob; g.lse_off += lb;
            if (g.n_splits > 1) g.part_off += wb;
            kp.groups.push_back(g);
        }
        int32_t direct = 0;
        for (size_t i = 0; i < src.tiles.size(); ++i) {
            Tile t = src.tiles[i];
            t.group += gb;
            kp.tiles.push_back(t);
            TileRec r = src.tile_recs[i];
            r.group += gb; r.q_off += qb; r.out_off += ob; r.lse_off += lb;
            if (r.n_splits > 1) r.part_off += wb;
            r.pad = s;
            kp.tile_recs.push_back(r);
            if (r.n_splits == 1) {              // its plane-0 warps (one per padded M tile) each signal once
                int mt = (r.gsize + 15) / 16, mtp = 1;
                while (mtp < mt) mtp <<= 1;
                direct += mtp;
            }
        }
        for (CombineUnit cu : src.cunits) {
            cu.part_off += wb; cu.ml_off += wb; cu.out_off += ob;
            if (cu.lse_off >= 0) cu.lse_off += lb;
            cu.group += gb;
            cu.pad[0] = s;
            kp.cunits.push_back(cu);
        }
        StageRec &sr = sp.stages[s];
        sr.dep = deps[s]; sr.dep_target = 0; sr.cu_begin = cb; sr.cu_end = (int)kp.cunits.size();
        sr.dep_out_delta = 0; sr.alpha = alpha == alpha ? alpha : 0.f; sr.pad = 0;
        target[s] = (sr.cu_end - sr.cu_begin) + direct;
        out_base[s] = ob;
        qb += pool->q_elems; ob += pool->out_floats; lb += pool->lse_floats; wb += (int64_t)pool->plan_ws_floats;
        p_ids += sizes[s];
    }
    for (int s = 0; s < n_stages; ++s)
        if (deps[s] >= 0) {
            sp.stages[s].dep_target = target[deps[s]];
            sp.stages[s].dep_out_delta = out_base[deps[s]] - out_base[s];
        }
    pool->plan_valid = false;                  // build_plan overwrote the single-step plan cache
    sp.q_elems = qb; sp.out_floats = ob; sp.lse_floats = lb; sp.ws_floats = (uint64_t)wb;
    sp.key.swap(key);
    sp.version = pool->topo_version;
    sp.valid = true;
    return CP_OK;
}

}  // namespace

cp_status cp_decode_stages_workspace_bytes(cp_pool *pool, int32_t n_stages, const int32_t *stage_sizes_host,
                                           const int32_t *request_ids_host, const int32_t *stage_dep_host,
                                           uint64_t *bytes_out)
{
    if (!bytes_out) return CP_ERR_INVALID_ARG;
    const cp_status st = build_stages_plan(pool, n_stages, stage_sizes_host, request_ids_host, stage_dep_host,
                                           std::nanf(""));          // NaN: leave the residual weight alone
    if (st != CP_OK) return st;
    *bytes_out = pool->splan.ws_floats * 4;
    return CP_OK;
}

static cp_status decode_stages_core(cp_pool *pool, int32_t n_stages, const int32_t *stage_sizes_host,
                                    const int32_t *request_ids_host, const int32_t *stage_dep_host, float alpha,
                                    const void *q_dev, float *out_dev, float *lse_dev, void *workspace_dev,
                                    uint64_t workspace_bytes, void *stream, const int32_t *published_dev,
                                    uint32_t timeout_ms)
{
    if (!pool || !q_dev || !out_dev || !lse_dev || !(alpha == alpha)) return CP_ERR_INVALID_ARG;
    if (((uintptr_t)q_dev & 15u) || ((uintptr_t)out_dev & 15u) || ((uintptr_t)lse_dev & 3u)) return CP_ERR_INVALID_ARG;
    cp_status st = build_stages_plan(pool, n_stages, stage_sizes_host, request_ids_host, stage_dep_host, alpha);
    if (st != CP_OK) return st;
    cp_pool::StagesPlan &sp = pool->splan;
    if (sp.ws_floats * 4 > workspace_bytes) return CP_ERR_WORKSPACE;
    if (sp.ws_floats && (!workspace_dev || ((uintptr_t)workspace_dev & 15u))) return CP_ERR_WORKSPACE;
    st = ensure_device(pool);
    if (st != CP_OK) return st;
    if (!pool->kv_tmap_ok) return CP_ERR_UNSUPPORTED;
    cudaStream_t s = (cudaStream_t)stream;
    st = adopt_stream(pool, s);
    if (st != CP_OK) return st;
    st = flush_tables(pool, s);
    if (st != CP_OK) return st;
    KindPlan &kp = sp.kp;
    st = upload_plan(pool, kp, s);
    if (st != CP_OK) return st;
    if (!sp.uploaded) {
        const size_t sb = sp.stages.size() * sizeof(StageRec);
        if (sp.d_stages.ensure(sb) != cudaSuccess ||
            cudaMemcpyAsync(sp.d_stages.ptr, sp.stages.data(), sb, cudaMemcpyHostToDevice, s) != cudaSuccess) {
            cudaGetLastError();
            return CP_ERR_CUDA;
        }
        pool->n_h2d_bytes += sb;
        sp.uploaded = true;
    }
    DecodeParams prm;
    std::memset(&prm, 0, sizeof(prm));
    prm.arena = pool->arena; prm.page_tokens = pool->P; prm.page_bytes = pool->page_bytes;
    prm.page_table = (const int32_t *)pool->d_page_table.ptr; prm.max_ppr = pool->max_ppr;
    prm.slot_pages = (pool->vmm && !pool->opt_vmm_table) ? (int32_t)pool->slot_pages : 0;
    prm.req_ctx = (const int32_t *)pool->d_ctx.ptr + (size_t)pool->ctx_cur * pool->max_requests;
    prm.models = (const DevModel *)pool->d_models.ptr;
    prm.groups = (const Group *)kp.p_groups;
    prm.tiles = (const Tile *)kp.p_tiles;
    prm.tile_recs = (const TileRec *)kp.p_tile_recs;
    prm.combines = (const Combine *)kp.p_combines;
    prm.cunits = (const CombineUnit *)kp.p_cunits;
    prm.n_tiles = (int)kp.tiles.size(); prm.n_combines = 0;
    prm.n_static_slots = 0;
    prm.n_combine_units = (int)kp.cunits.size();
    prm.n_groups = (int)kp.groups.size() + n_stages;           // counters the next launch's reset covers
    prm.q = (const uint16_t *)q_dev; prm.out = out_dev; prm.lse = lse_dev;
    prm.workspace = (float *)workspace_dev;
    const size_t set_ints = 32 + (kp.groups.size() + (size_t)n_stages) * (size_t)kCounterStride;
    prm.work_counter = (int32_t *)kp.p_counters + kp.counter_set * set_ints;
    prm.group_counters = prm.work_counter + 32;
    prm.reset_counters = (int32_t *)kp.p_counters + (1 - kp.counter_set) * set_ints;
    prm.stages = (const StageRec *)sp.d_stages.ptr;
    prm.stage_done = prm.group_counters + kp.groups.size() * (size_t)kCounterStride;
    prm.n_stages = n_stages; prm.q_len = 1;
    prm.published = nullptr; prm.gate_flag = nullptr; prm.gate_timeout_us = 0;
    prm.timeline = nullptr;
    prm.app_k = nullptr; prm.app_v = nullptr;
    if (published_dev) {
        if (sp.d_gate.ensure(16) != cudaSuccess || cudaMemsetAsync(sp.d_gate.ptr, 0, 16, s) != cudaSuccess) {
            cudaGetLastError();
            return CP_ERR_CUDA;
        }
        prm.published = published_dev; prm.gate_flag = (int32_t *)sp.d_gate.ptr;
        prm.gate_timeout_us = timeout_ms > 4000000u ? 4000000000u : timeout_ms * 1000u;
    }
    kp.counter_set ^= 1;
    const int n_ctas = pool->opt_num_ctas > 0 ? pool->opt_num_ctas : pool->n_sm;
    const cudaError_t e = launch_decode_kv(prm, pool->kv_tmap, (int)(pool->page_bytes / 256), std::min(n_ctas, pool->n_sm), s);
    pool->n_launches++;
    if (e != cudaSuccess) return CP_ERR_CUDA;
    return CP_OK;
}

cp_status cp_decode_attention_stages(cp_pool *pool, int32_t n_stages, const int32_t *stage_sizes_host,
                                     const int32_t *request_ids_host, const int32_t *stage_dep_host, float alpha,
                                     const void *q_dev, float *out_dev, float *lse_dev, void *workspace_dev,
                                     uint64_t workspace_bytes, void *stream)
{
    return decode_stages_core(pool, n_stages, stage_sizes_host, request_ids_host, stage_dep_host, alpha, q_dev, out_dev,
                              lse_dev, workspace_dev, workspace_bytes, stream, nullptr, 0);
}

cp_status cp_decode_attention_stages_gated(cp_pool *pool, int32_t n_stages, const int32_t *stage_sizes_host,
                                           const int32_t *request_ids_host, const int32_t *stage_dep_host,
                                           float alpha, const void *q_dev, float *out_dev, float *lse_dev,
                                           void *workspace_dev, uint64_t workspace_bytes, void *stream,
                                           const int32_t *published_dev, uint32_t timeout_ms)
{
    if (!published_dev || ((uintptr_t)published_dev & 3u) || timeout_ms == 0) return CP_ERR_INVALID_ARG;
    return decode_stages_core(pool, n_stages, stage_sizes_host, request_ids_host, stage_dep_host, alpha, q_dev, out_dev,
                              lse_dev, workspace_dev, workspace_bytes, stream, published_dev, timeout_ms);
}

cp_status cp_decode_stages_gate_status(cp_pool *pool, void *stream, int32_t *timed_out_host)
{
    if (!pool || !timed_out_host) return CP_ERR_INVALID_ARG;
    *timed_out_host = 0;
    if (!pool->splan.d_gate.ptr) return CP_OK;
    cudaStream_t s = (cudaStream_t)stream;
    if (cudaMemcpyAsync(timed_out_host, pool->splan.d_gate.ptr, 4, cudaMemcpyDeviceToHost, s) != cudaSuccess ||
        cudaStreamSynchronize(s) != cudaSuccess) {
        cudaGetLastError();
        return CP_ERR_CUDA;
    }
    return CP_OK;
}

static inline uint64_t align256(uint64_t x) { return (x + 255) & ~(uint64_t)255; }

cp_status cp_decode_workspace_bytes_host(cp_pool *pool, const int32_t *request_ids_host,
                                         int32_t n_requests, uint64_t *bytes_out)
{
    uint64_t ws = 0;
    cp_status st = cp_decode_workspace_bytes(pool, request_ids_host, n_requests, &ws);
    if (st != CP_OK) return st;
    *bytes_out = align256((uint64_t)pool->q_elems * 2) + align256((uint64_t)pool->out_floats * 4) +
                 align256((uint64_t)pool->lse_floats * 4) + ws;
    return CP_OK;
}

cp_status cp_decode_attention_host(cp_pool *pool, const int32_t *request_ids_host,
                                   int32_t n_requests, const void *q_host, float *out_host,
                                   float *lse_host, void *workspace_dev, uint64_t workspace_bytes,
                                   void *stream)
{
    if (!q_host || !out_host || !lse_host || !workspace_dev) return CP_ERR_INVALID_ARG;
    uint64_t need = 0;
    cp_status st = cp_decode_workspace_bytes_host(pool, request_ids_host, n_requests, &need);
    if (st != CP_OK) return st;
    if (need > workspace_bytes || ((uintptr_t)workspace_dev & 255u)) return CP_ERR_WORKSPACE;
    st = ensure_device(pool);
    if (st != CP_OK) return st;
    cudaStream_t s = (cudaStream_t)stream;
    uint8_t *w = (uint8_t *)workspace_dev;
    void *q_dev = w;                      w += align256((uint64_t)pool->q_elems * 2);
    // O and LSE staging back to back, so that one copy serves a caller whose two host buffers are adjacent
    float *o_dev = (float *)w;
    float *l_dev = o_dev + pool->out_floats;
    w += align256((uint64_t)pool->out_floats * 4) + align256((uint64_t)pool->lse_floats * 4);
    const uint64_t rest = workspace_bytes - (uint64_t)(w - (uint8_t *)workspace_dev);
    // Pinned (mapped) host buffers are accessed in place where that moves fewer bytes more directly:
    // results are written exactly once, so O / LSE always qualify; Q is re-read by every tile of its
    // group, so only when those re-reads stay small (K/V kernel, a few hundred KB per step).
    void *zq = nullptr, *zo = nullptr, *zl = nullptr;
    if (pool->opt_host_zero_copy) {
        const void *hp[3] = {q_host, out_host, lse_host};
        for (int i = 0; i < 3; ++i) {
            if (pool->zc_host[i] != hp[i]) {
                cudaPointerAttributes a;
                pool->zc_host[i] = hp[i];
                pool->zc_dev[i] = nullptr;
                if (cudaPointerGetAttributes(&a, hp[i]) == cudaSuccess && a.type == cudaMemoryTypeHost && a.devicePointer &&
                    ((uintptr_t)a.devicePointer & (i == 2 ? 3u : 15u)) == 0)
                    pool->zc_dev[i] = a.devicePointer;
                cudaGetLastError();
            }
        }
        const KindPlan &kv = pool->plan[CP_KIND_KV];
        uint64_t q_reread = 0;
        for (const TileRec &r : kv.tile_recs) q_reread += (uint64_t)r.gsize * 256u;
        if (pool->plan[CP_KIND_MLA].tiles.empty() && kv.all_fast && pool->opt_kernel != 1 && pool->kv_tmap_ok &&
            q_reread <= (1u << 20))
            zq = pool->zc_dev[0];
        if (pool->zc_dev[1] && pool->zc_dev[2]) { zo = pool->zc_dev[1]; zl = pool->zc_dev[2]; }
    }
    if (!zq && cudaMemcpyAsync(q_dev, q_host, (size_t)pool->q_elems * 2, cudaMemcpyHostToDevice, s) != cudaSuccess)
        return CP_ERR_CUDA;
    st = cp_decode_attention(pool, request_ids_host, n_requests, zq ? zq : q_dev, zo ? (float *)zo : o_dev,
                             zl ? (float *)zl : l_dev, w, rest, s);
    if (st != CP_OK) return st;
    if (zo) {
        // written in place by the kernel; visible to the host after the synchronisation below
    } else if (lse_host == out_host + pool->out_floats) {
        if (cudaMemcpyAsync(out_host, o_dev, (size_t)(pool->out_floats + pool->lse_floats) * 4, cudaMemcpyDeviceToHost, s) !=
            cudaSuccess)
            return CP_ERR_CUDA;
    } else if (cudaMemcpyAsync(out_host, o_dev, (size_t)pool->out_floats * 4, cudaMemcpyDeviceToHost, s) != cudaSuccess ||
               cudaMemcpyAsync(lse_host, l_dev, (size_t)pool->lse_floats * 4, cudaMemcpyDeviceToHost, s) != cudaSuccess)
        return CP_ERR_CUDA;
    if (cudaStreamSynchronize(s) != cudaSuccess) return CP_ERR_CUDA;
    return CP_OK;
}

}  // extern "C"

// ------------------------------------------------------------------ request queue of a persistent launch
struct cp_queue {
    cp_pool *pool = nullptr;
    int max_stages = 0, max_tiles = 0, max_units = 0, max_groups = 0;
    QueueEntry *h_ring = nullptr;        // mapped pinned memory: [max_stages + 1] entries ...
    int32_t *h_tail = nullptr;           // ... and the tail counter (its own 64-byte line behind them)
    void *d_ring = nullptr, *d_tail = nullptr;
    DevBuf d_recs, d_units, d_stages, d_state, d_counters, d_out_base, d_target, d_req_model;
    int pushed = 0;
    bool closed = false, launched = false;
    std::vector<std::vector<int32_t>> stage_models;     // per pushed stage: model of every request (shape check of dependents)
    int64_t rows_pushed = 0;
};

extern "C" {

cp_status cp_queue_create(cp_pool *pool, int32_t max_stages, cp_queue **out)
{
    if (!out) return CP_ERR_INVALID_ARG;
    *out = nullptr;
    if (!pool || max_stages < 1 || max_stages > 65536) return CP_ERR_INVALID_ARG;
    cp_status st = ensure_device(pool);
    if (st != CP_OK) return st;
    if (!pool->kv_tmap_ok) return CP_ERR_UNSUPPORTED;
    cp_queue *q = new (std::nothrow) cp_queue();
    if (!q) return CP_ERR_INVALID_ARG;
    q->pool = pool;
    q->max_stages = max_stages;
    q->max_tiles = max_stages * 256;
    q->max_units = max_stages * 2048;
    q->max_groups = max_stages * 96;
    const size_t ring_bytes = (size_t)(max_stages + 1) * sizeof(QueueEntry) + 64;
    void *h = nullptr;
    if (cudaHostAlloc(&h, ring_bytes, cudaHostAllocMapped) != cudaSuccess) { cudaGetLastError(); delete q; return CP_ERR_CUDA; }
    std::memset(h, 0, ring_bytes);
    q->h_ring = (QueueEntry *)h;
    q->h_tail = (int32_t *)((uint8_t *)h + (size_t)(max_stages + 1) * sizeof(QueueEntry));
    void *d = nullptr;
    if (cudaHostGetDevicePointer(&d, h, 0) != cudaSuccess) { cudaGetLastError(); cudaFreeHost(h); delete q; return CP_ERR_CUDA; }
    q->d_ring = d;
    q->d_tail = (uint8_t *)d + (size_t)(max_stages + 1) * sizeof(QueueEntry);
    const size_t counters = 64 + ((size_t)q->max_groups + (size_t)max_stages) * kCounterStride;
    if (q->d_recs.ensure((size_t)q->max_tiles * sizeof(TileRec)) != cudaSuccess ||
        q->d_units.ensure((size_t)q->max_units * sizeof(CombineUnit)) != cudaSuccess ||
        q->d_stages.ensure((size_t)max_stages * sizeof(StageRec)) != cudaSuccess ||
        q->d_state.ensure(256) != cudaSuccess || q->d_counters.ensure(counters * 4) != cudaSuccess ||
        q->d_out_base.ensure((size_t)max_stages * 8) != cudaSuccess || q->d_target.ensure((size_t)max_stages * 4) != cudaSuccess ||
        q->d_req_model.ensure((size_t)pool->max_requests * 4) != cudaSuccess) {
        cudaGetLastError();
        cp_queue_free(q);
        return CP_ERR_CUDA;
    }
    *out = q;
    return CP_OK;
}

cp_status cp_queue_free(cp_queue *q)
{
    if (!q) return CP_OK;
    cudaDeviceSynchronize();
    q->d_recs.release(); q->d_units.release(); q->d_stages.release(); q->d_state.release(); q->d_counters.release();
    q->d_out_base.release(); q->d_target.release(); q->d_req_model.release();
    if (q->h_ring) cudaFreeHost(q->h_ring);
    delete q;
    return CP_OK;
}

cp_status cp_queue_push(cp_queue *q, const int32_t *request_ids_host, int32_t n_requests, int32_t dep_stage, float alpha,
                        int32_t *stage_index_out)
{
    if (!q || q->closed || q->pushed >= q->max_stages || !(alpha == alpha)) return CP_ERR_INVALID_ARG;
    cp_pool *pool = q->pool;
    cp_status st = check_batch(pool, request_ids_host, n_requests);
    if (st != CP_OK) return st;
    if (n_requests > kQueueMaxReq || dep_stage >= q->pushed || dep_stage < -1) return CP_ERR_INVALID_ARG;
    std::vector<int32_t> models(n_requests);
    int64_t rows = 0;
    for (int b = 0; b < n_requests; ++b) {
        const Request &r = pool->reqs[request_ids_host[b]];
        const cp_model_cfg &m = pool->models[r.model];
        if (m.kind != CP_KIND_KV || m.head_dim_qk != 128 || m.head_dim_v != 128 || m.n_q_heads / m.n_kv_heads > 128)
            return CP_ERR_UNSUPPORTED;
        models[b] = r.model;
        rows += m.n_q_heads;
    }
    if (dep_stage >= 0 && q->stage_models[dep_stage] != models) return CP_ERR_INVALID_ARG;   // same batch shape as its predecessor
    QueueEntry e;
    std::memset(&e, 0, sizeof(e));
    e.n_req = n_requests; e.dep = dep_stage; e.alpha = alpha; e.close = 0;
    for (int b = 0; b < n_requests; ++b) e.ids[b] = request_ids_host[b];
    // entry first, then the tail (release): the planner warp acquires the tail at system scope
    std::memcpy((void *)&q->h_ring[q->pushed], &e, sizeof(e));
    __atomic_store_n(q->h_tail, q->pushed + 1, __ATOMIC_RELEASE);
    if (stage_index_out) *stage_index_out = q->pushed;
    q->stage_models.push_back(std::move(models));
    q->rows_pushed += rows;
    q->pushed++;
    return CP_OK;
}

cp_status cp_queue_close(cp_queue *q)
{
    if (!q) return CP_ERR_INVALID_ARG;
    if (q->closed) return CP_OK;
    QueueEntry e;
    std::memset(&e, 0, sizeof(e));
    e.close = 1;
    std::memcpy((void *)&q->h_ring[q->pushed], &e, sizeof(e));
    __atomic_store_n(q->h_tail, q->pushed + 1, __ATOMIC_RELEASE);
    q->closed = true;
    return CP_OK;
}

cp_status cp_queue_launch(cp_queue *q, const void *q_dev, float *out_dev, float *lse_dev, void *workspace_dev,
                          uint64_t workspace_bytes, uint32_t timeout_ms, void *stream)
{
    if (!q || q->launched || !q_dev || !out_dev || !lse_dev || timeout_ms == 0) return CP_ERR_INVALID_ARG;
    if (((uintptr_t)q_dev & 15u) || ((uintptr_t)out_dev & 15u) || ((uintptr_t)lse_dev & 3u) || ((uintptr_t)workspace_dev & 15u))
        return CP_ERR_INVALID_ARG;
    cp_pool *pool = q->pool;
    cp_status st = ensure_device(pool);
    if (st != CP_OK) return st;
    if (!pool->kv_tmap_ok) return CP_ERR_UNSUPPORTED;
    cudaStream_t s = (cudaStream_t)stream;
    st = adopt_stream(pool, s);
    if (st != CP_OK) return st;
    st = flush_tables(pool, s);
    if (st != CP_OK) return st;
    std::vector<int32_t> rm(pool->max_requests, -1);
    for (int i = 0; i < pool->max_requests; ++i)
        if (pool->reqs[i].live) rm[i] = pool->reqs[i].model;
    if (cudaMemcpyAsync(q->d_req_model.ptr, rm.data(), rm.size() * 4, cudaMemcpyHostToDevice, s) != cudaSuccess ||
        cudaMemsetAsync(q->d_state.ptr, 0, 256, s) != cudaSuccess ||
        cudaMemsetAsync(q->d_counters.ptr, 0, q->d_counters.cap, s) != cudaSuccess)
        return CP_ERR_CUDA;
    DecodeParams prm;
    std::memset(&prm, 0, sizeof(prm));
    prm.arena = pool->arena; prm.page_tokens = pool->P; prm.page_bytes = pool->page_bytes;
    prm.page_table = (const int32_t *)pool->d_page_table.ptr; prm.max_ppr = pool->max_ppr;
    prm.slot_pages = (pool->vmm && !pool->opt_vmm_table) ? (int32_t)pool->slot_pages : 0;
    prm.req_ctx = (const int32_t *)pool->d_ctx.ptr + (size_t)pool->ctx_cur * pool->max_requests;
    prm.models = (const DevModel *)pool->d_models.ptr;
    prm.tile_recs = (const TileRec *)q->d_recs.ptr;
    prm.cunits = (const CombineUnit *)q->d_units.ptr;
    prm.stages = (const StageRec *)q->d_stages.ptr;
    prm.n_tiles = 0; prm.n_stages = 0; prm.q_len = 1;
    prm.q = (const uint16_t *)q_dev; prm.out = out_dev; prm.lse = lse_dev; prm.workspace = (float *)workspace_dev;
    int32_t *ctr = (int32_t *)q->d_counters.ptr;
    prm.work_counter = ctr;                       // [0] next tile; [32..63] the other set's scheduler words (unused here)
    prm.reset_counters = ctr + 32; prm.n_groups = 0;
    prm.group_counters = ctr + 64;
    prm.stage_done = ctr + 64 + (size_t)q->max_groups * kCounterStride;
    prm.gate_timeout_us = timeout_ms > 4000000u ? 4000000000u : timeout_ms * 1000u;
    prm.queue = (const QueueEntry *)q->d_ring; prm.queue_tail = (const int32_t *)q->d_tail;
    prm.qstate = (QueueState *)q->d_state.ptr;
    prm.req_model = (const int32_t *)q->d_req_model.ptr;
    prm.q_out_base = (int64_t *)q->d_out_base.ptr; prm.q_target = (int32_t *)q->d_target.ptr;
    prm.q_max_stages = q->max_stages; prm.q_max_tiles = q->max_tiles; prm.q_max_units = q->max_units; prm.q_max_groups = q->max_groups;
    const int n_ctas = std::min(pool->opt_num_ctas > 0 ? pool->opt_num_ctas : pool->n_sm, pool->n_sm);
    prm.q_target_tiles = std::max(1, n_ctas * pool->opt_waves_x16 / 16);
    prm.q_min_tile_pages = pool->opt_min_tile_pages;
    prm.q_ws_floats_cap = (int64_t)(workspace_bytes / 4);
    const cudaError_t e = launch_decode_kv(prm, pool->kv_tmap, (int)(pool->page_bytes / 256), n_ctas, s);
    pool->n_launches++;
    if (e != cudaSuccess) return CP_ERR_CUDA;
    q->launched = true;
    return CP_OK;
}

cp_status cp_queue_status(cp_queue *q, void *stream, int32_t *stages_planned, int32_t *tiles_planned, int32_t *error)
{
    if (!q) return CP_ERR_INVALID_ARG;
    QueueState st;
    cudaStream_t s = (cudaStream_t)stream;
    if (cudaMemcpyAsync(&st, q->d_state.ptr, sizeof(st), cudaMemcpyDeviceToHost, s) != cudaSuccess ||
        cudaStreamSynchronize(s) != cudaSuccess) {
        cudaGetLastError();
        return CP_ERR_CUDA;
    }
    if (stages_planned) *stages_planned = st.planned_stages;
    if (tiles_planned) *tiles_planned = st.planned_tiles;
    if (error) *error = st.error;
    return CP_OK;
}

}  // extern "C"
