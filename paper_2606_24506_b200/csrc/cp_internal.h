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
    int64_t app_k_off, app_v_off;  // element offsets of this group's new K / V row in the packed k_new / v_new of cp_decode_step
};
static_assert(sizeof(TileRec) == 96, "TileRec is loaded as 16-byte vectors (five for the fields the older kernels use, six in all)");

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
                                   // at j * gridDim.x + b, TileRec::pad bit 0 = another slot follows), the rest is popped
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
    const uint16_t *app_k, *app_v; // cp_decode_step: packed new K / V rows the launch writes at position
                                   // context_len - 1 of every request before the page that holds it is read, or nullptr
};

}  // namespace cp
