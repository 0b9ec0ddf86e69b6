// cp_internal.h -- structures shared by the host pool manager and the CUDA kernels of
// libcrosspool.  Private to paper_2606_24506_b200/csrc (the oracle shares nothing with it).
#pragma once
#include <cstdint>

namespace cp {

constexpr int kPartPad = 4;          // partial row = d_v floats of O, then m, l, 2 pad floats
constexpr int kMaxDk = 576;
constexpr int kMaxDv = 512;
constexpr int kMaxSplits = 512;      // KV splits per group (bounds the combine's shared memory)

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

// One unit of the LSE combine: one query head of a split group.
struct Combine {
    int32_t group;
    int32_t head;           // head index inside the group (0 .. g-1)
};

// Kernel arguments common to all decode kernels (passed by value).
struct DecodeParams {
    const uint8_t *arena;
    uint32_t page_tokens;
    uint32_t page_bytes;
    const int32_t *page_table;     // [max_requests][max_ppr]
    int32_t max_ppr;
    const int32_t *req_ctx;        // [max_requests] current context length
    const DevModel *models;
    const Group *groups;
    const Tile *tiles;
    const Combine *combines;
    int32_t n_tiles;
    int32_t n_combines;            // work items after the tiles (CTA-sized combine items)
    int32_t n_combine_units;       // tensor-core kernels: warp-sized combine units; else = n_combines
    int32_t n_groups;
    const uint16_t *q;             // bf16 packed
    float *out;
    float *lse;
    float *workspace;              // split partials
    int32_t *work_counter;         // [0] next work item, [1] CTAs that finished
    int32_t *group_counters;       // [n_groups] tile arrivals
};

}  // namespace cp
