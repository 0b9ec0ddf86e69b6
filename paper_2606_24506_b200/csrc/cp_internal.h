// cp_internal.h -- structures shared by the host pool manager and the CUDA kernels of
// libcrosspool.  Private to paper_2606_24506_b200/csrc (the oracle shares nothing with it).
#pragma once
#include <cstdint>
#ifndef __CUDACC__
#define __host__
#define __device__
#endif

namespace cp {

// Split partials of one group in the workspace (float offsets from Group::part_off), g = heads of
// the group, ns = its splits:  O[h][s][d_v] (unnormalised), then ML[h][s] = (m in log2 units, l).
// Head-major, so the LSE combine of one head reads contiguous rows and a contiguous (m, l) vector.
__host__ __device__ inline int64_t part_o_off(int h, int s, int ns, int dv) { return ((int64_t)h * ns + s) * dv; }
__host__ __device__ inline int64_t part_ml_off(int g, int h, int s, int ns, int dv)
{
    return (int64_t)g * ns * dv + ((int64_t)h * ns + s) * 2;
}
__host__ __device__ inline int64_t part_group_floats(int g, int ns, int dv)
{
    return (((int64_t)g * ns * (dv + 2)) + 3) & ~(int64_t)3;
}
constexpr int kMaxDk = 576;
constexpr int kMaxDv = 512;
constexpr int kMaxSplits = 512;
constexpr int kCounterStride = 32;   // ints between group counters: one 128-byte line each (no false sharing under polling)
constexpr int kTimelineSlots = 16;   // globaltimer stamps per CTA (CP_OPT_TIMELINE)

// Device copy of a model description (cp_model_cfg plus derived values).
struct DevModel {
    int32_t kind;
    int32_t n_q_heads;
    int32_t n_kv_heads;
    int32_t d_k;
    int32_t d_v;
    int32_t group;          // g = Hq / Hkv
    float scale;            // sigma
    float scale_log2;       // sigma * log2(e): scores are kept in log2 units
};

// One (batch slot, kv head) group: the g query heads that stream the same KV pages.
struct Group {
    int32_t req;            // request id = row of the page table / ctx table
    int32_t model;
    int32_t kv_head;
    int32_t n_splits;
    int32_t n_pages;        // logical pages the plan covers (ceil(ctx / P) at plan time)
    int32_t batch_index;
    int64_t q_off;          // element offset of this group's first query row in packed Q
    int64_t out_off;        // float offset of this group's first output row in packed O
    int64_t lse_off;        // index of this group's first head in packed LSE
    int64_t part_off;       // float offset of this group's partials in the workspace
};

// One tile of the work list: a page range of one group.  Persistent CTAs pop tiles in
// array order (longest first), then combine units.
struct Tile {
    int32_t group;
    int32_t split;
    int32_t page_begin;
    int32_t page_end;
};

// Everything a producer warp needs to start a tile, in one 80-byte record (one level of loads
// after the pop instead of tile -> group -> model): same order as Tile[].
struct TileRec {
    int32_t group, req, kv_head, n_kv_heads;
    int32_t page_begin, n_pages, split, n_splits;
    int32_t gsize, n_q_heads;
    float scale_log2;
    int32_t pad;                   // bit 0: another static slot of this CTA follows (tcgen05 K/V kernel); bit 1: the tile
                                   // holds its group's LAST planned page (where a fused append writes); bits 8..15: zl
                                   // of the group's partial layout; other kernels: see their planner
    int64_t q_off, out_off, lse_off, part_off;
    int32_t app_k_off, app_v_off;  // element offsets of this group's new K / V row in the packed k_new / v_new of cp_decode_step
    int32_t next;                  // tcgen05 K/V kernel: index of the next record of this CTA's static list (valid with pad bit 0)
    int32_t pad2;
    int32_t first_pid[8];          // tcgen05 K/V kernel: physical ids of the tile's first pages (one 128-token slice: 128 / P <= 8),
                                   // so that the first TMA loads need no page-table round trip (ids of mapped pages never change)
};
static_assert(sizeof(TileRec) == 128, "TileRec is loaded as 16-byte vectors (five for the fields the older kernels use, eight in all)");

// One request of a cp_pool_append_kv batch.
struct AppendRec {
    int32_t req, model, pos, pad;
    int64_t k_off, v_off;          // element offsets of this request's rows in the packed k_new / v_new
};

// One unit of the LSE combine: one query head of a split group.
struct Combine {
    int32_t group;
    int32_t head;           // head index inside the group (0 .. g-1)
};

// One warp-sized unit of the LSE combine (tensor-core kernels): 128 >> zl_log2 output columns of
// one (group, head), with everything the warp needs in one 64-byte record (no pointer chasing).
struct CombineUnit {
    int64_t part_off;       // float offset in the workspace of (split 0, this head, first column)
    int64_t ml_off;         // float offset in the workspace of (m, l) of (split 0, this head); splits contiguous
    int64_t out_off;        // float offset in packed O of (this head, first column)
    int64_t lse_off;        // index in packed LSE of this head, or -1 if another unit writes it
    int32_t split_stride;   // floats between consecutive splits of this head's O rows (= d_v)
    int32_t n_splits;
    int32_t zl_log2;        // split lanes of the warp = 1 << zl_log2 (1, 8 or 32)
    int32_t want;           // arrivals on the group counter that mean "all splits published"
    int32_t group;          // index of the group counter
    int32_t pad[3];
};
static_assert(sizeof(CombineUnit) == 64, "CombineUnit is loaded as four 16-byte vectors");

// One stage of a multi-stage launch (cp_decode_attention_stages): one attention step
// = one layer of one in-flight batch.  A stage with dep >= 0 builds its queries from the output of
// stage dep (same batch shape): q = bf16(q_in + alpha * O_dep), and may only do so once dep_target
// completion signals of stage dep have been counted (its combine units and single-split tiles).
struct StageRec {
    int32_t dep;            // stage this one depends on, or -1
    int32_t dep_target;     // value of stage_done[dep] that means "stage dep is complete"
    int32_t cu_begin, cu_end;   // this stage's combine units
    int64_t dep_out_delta;  // out offset of stage dep minus out offset of this stage (floats)
    float alpha;
    int32_t pad;
};
static_assert(sizeof(StageRec) == 32, "StageRec is loaded as two 16-byte vectors");

// Splits per request of one tile plan (hot-path step a1) -- the arithmetic shared by the host planner
// (build_plan) and the device-side planner of the request queue (cp_queue_*), so that a stage
// planned on the GPU is cut exactly like the same batch planned on the host.  n_lp[b] = logical pages of
// request b, hkv[b] = its kv heads (groups).  Smallest tile length L (pages) for which the batch yields at most
// target_tiles tiles (searched in [L_bal, 2 L_bal]; a batch of many short requests cannot meet the target at
// all -- every group is at least one tile -- and keeps the balanced length L_bal); then the tiles still missing
// from the target go, one at a time, to the request whose tiles are longest.  Depends on the page counts only.
__host__ __device__ inline void plan_request_splits(int n, const int *n_lp, const int *hkv, int64_t target_tiles,
                                                    int min_tile_pages, int max_splits, int *splits)
{
    // (32-bit divisions and an integer comparison of the tile lengths: the device-side planner runs this on one
    // thread of a GPU whose 64-bit integer and floating-point division are slow)
    int64_t total = 0;
    for (int b = 0; b < n; ++b) total += (int64_t)n_lp[b] * hkv[b];
    if (total == 0) return;
    auto tiles_for = [&](int len) {
        int64_t t = 0;
        for (int b = 0; b < n; ++b) t += (int64_t)hkv[b] * ((n_lp[b] + len - 1) / len);
        return t;
    };
    int64_t L_bal64 = (total + target_tiles - 1) / target_tiles;
    if (L_bal64 < min_tile_pages) L_bal64 = min_tile_pages;
    if (L_bal64 > (1 << 29)) L_bal64 = 1 << 29;
    const int L_bal = (int)L_bal64;
    int L = L_bal;
    if (tiles_for(2 * L_bal) <= target_tiles) {
        int lo = L_bal, hi = 2 * L_bal;
        while (lo < hi) {
            const int mid = lo + (hi - lo) / 2;
            if (tiles_for(mid) <= target_tiles) hi = mid; else lo = mid + 1;
        }
        L = lo;
    }
    int64_t have = 0;
    for (int b = 0; b < n; ++b) {
        if (hkv[b] == 0) { splits[b] = 0; continue; }
        int sp = (n_lp[b] + L - 1) / L;
        if (sp > max_splits) sp = max_splits;
        splits[b] = sp;
        have += (int64_t)sp * hkv[b];
    }
    while (have < target_tiles) {
        // the request whose tiles are longest, n_lp / splits compared exactly as a fraction (first one wins a tie)
        int best = -1;
        for (int b = 0; b < n; ++b) {
            if (hkv[b] == 0 || have + hkv[b] > target_tiles) continue;
            if (splits[b] + 1 > max_splits || n_lp[b] / (splits[b] + 1) < min_tile_pages) continue;
            if (best < 0 || (int64_t)n_lp[b] * splits[best] > (int64_t)n_lp[best] * splits[b]) best = b;
        }
        if (best < 0) break;
        splits[best] += 1;
        have += hkv[best];
    }
}

// Request queue of a persistent launch (cp_queue_*; "persistent kernels repeatedly
// poll per-model request queues on GPUs, select the next ready batch ...").  One entry = one stage = one
// attention step of one batch.  Written by the HOST into mapped pinned memory after the kernel has started;
// the planner warp of CTA 0 polls `tail`, cuts the batch into tiles on arrival and publishes them in QueueState.
constexpr int kQueueMaxReq = 12;
struct QueueEntry {
    int32_t n_req;
    int32_t dep;            // stage whose output feeds this one's queries (same batch shape), or -1
    float alpha;
    int32_t close;          // 1: no further entries; the kernel drains and exits
    int32_t ids[kQueueMaxReq];
};
static_assert(sizeof(QueueEntry) == 64, "QueueEntry is one 64-byte record");
struct QueueState {         // device memory; planner (CTA 0) -> every CTA
    int32_t planned_tiles;  // tile records [0, planned_tiles) are complete
    int32_t planned_stages;
    int32_t closed;         // 1: planned_tiles / planned_stages are final
    int32_t error;          // 1 queue poll timed out, 2 a capacity (tiles / units / groups / workspace) was exceeded,
                            // 3 an entry was malformed (request not mapped, unsupported shape, dep)
    int32_t n_units, n_groups;
    int32_t pad[2];
    int64_t q_rows, ws_floats;        // running totals: query / output rows and workspace floats handed out
};

// Kernel arguments common to all decode kernels (passed by value).
struct DecodeParams {
    const uint8_t *arena;
    uint32_t page_tokens;
    uint32_t page_bytes;
    const int32_t *page_table;     // [max_requests][max_ppr]
    int32_t max_ppr;
    int32_t slot_pages;            // > 0: contiguous virtual KV (CUDA VMM arena): page idx of request r is
                                   // r * slot_pages + idx and the decode kernels read no page table
    const int32_t *req_ctx;        // [max_requests] current context length
    const DevModel *models;
    const Group *groups;
    const Tile *tiles;
    const TileRec *tile_recs;      // [n_tiles], same order as tiles
    const Combine *combines;
    const CombineUnit *cunits;     // [n_combine_units] (tensor-core kernels)
    int32_t n_tiles;
    int32_t n_static_slots;        // tcgen05 K/V kernel: records [0, n_static_slots) are the CTAs' static lists (slot j of CTA b
                                   // at index b < gridDim.x, TileRec::pad bit 0 = another one follows at TileRec::next), the rest is popped
    int32_t n_combines;            // work items after the tiles (CTA-sized combine items)
    int32_t n_combine_units;       // tensor-core kernels: warp-sized combine units; else = n_combines
    int32_t n_groups;
    const uint16_t *q;             // bf16 packed
    float *out;
    float *lse;
    float *workspace;              // split partials
    int32_t *work_counter;         // [0] next work item (tile); [1..3] spare
    int32_t *group_counters;       // [n_groups * kCounterStride] tile arrivals, counter g at g * kCounterStride
    int32_t *reset_counters;
    // multi-stage launches only (else nullptr / 0)
    int32_t q_len;                 // query tokens per request (1 except cp_decode_attention_qlen)
    const StageRec *stages;
    const int32_t *published;      // admission doorbell (gated multi-stage launch) or nullptr: stages admitted so far
    int32_t *gate_flag;            // set to 1 if a poll of the doorbell timed out
    uint32_t gate_timeout_us;
    int32_t *stage_done;           // [n_stages] completion counters, kCounterStride apart
    int32_t n_stages;
    unsigned long long *timeline;  // CP_OPT_TIMELINE: [grid][kTimelineSlots] globaltimer stamps, or nullptr
    // request queue (cp_queue_launch) only, else nullptr / 0
    const QueueEntry *queue;       // [q_max_stages] host-written entries (mapped pinned memory)
    const int32_t *queue_tail;     // entries pushed so far (mapped pinned memory)
    QueueState *qstate;
    const int32_t *req_model;      // [max_requests] model of every mapped request, -1 if none
    int64_t *q_out_base;           // [q_max_stages] first output row of every planned stage
    int32_t *q_target;             // [q_max_stages] completion signals that mean "stage complete"
    int32_t q_max_stages, q_max_tiles, q_max_units, q_max_groups;
    int32_t q_target_tiles, q_min_tile_pages;
    int64_t q_ws_floats_cap;
    int32_t *req_ctx_next;         // cp_decode_step on the tcgen05 K/V kernel: the OTHER context table, which the launch fills
                                   // (all max_requests entries copied, the batch's requests + ctx_add), or nullptr
    int32_t ctx_add;               // added to every context length the launch reads (1 during such a step, else 0)
    int32_t max_requests;
    const uint16_t *app_k, *app_v; // cp_decode_step: packed new K / V rows the launch writes at position
                                   // context_len - 1 of every request before the page that holds it is read, or nullptr
};

}  // namespace cp
