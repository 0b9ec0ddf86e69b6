/*
 * crosspool.h -- C ABI of the B200-native paged decode attention on a shared KV-cache pool.
 *
 * One hot path of CrossPool (arxiv 2606.24506): the decode-step attention that runs
 * locally on the shared, virtualized KV-cache pool, where the paged KV blocks of many
 * cold models' active requests live interleaved in one device arena behind a page table.
 * Citations are PAPER.md line numbers (the paper text) and DESIGN.md readings.
 *
 * Conventions for every entry point
 *   - extern "C", plain pointers and sizes; no C++ types, no exceptions cross the boundary.
 *   - every call returns a cp_status (0 = CP_OK, negative = error); it never aborts.
 *   - "host" / "dev" in a parameter name says where the pointer lives.  All large device
 *     buffers (arena, Q, O, LSE, workspace) are owned by the CALLER (e.g. torch tensors);
 *     the library owns only its metadata (page table, work list, counters).
 *   - argument errors are detected synchronously and leave the pool unchanged.
 *   - device work is enqueued on `stream` (a cudaStream_t passed as void*; NULL = the
 *     legacy default stream) and the call returns without synchronising, except the
 *     *_host variant which synchronises the stream before returning.
 *   - an asynchronous CUDA fault surfaces as CP_ERR_CUDA on the call that observes it.
 *   - a pool is not thread-safe; the caller serialises calls on one pool.
 *   - device pointers must be 16-byte aligned (the arena 256-byte aligned).
 *   - there is NO CPU fallback: without a usable CUDA device the compute entry points
 *     return CP_ERR_CUDA.
 *
 * Arena layout (reading R1; the paper fixes only "page size" and per-token
 * KV bytes kappa(M)): the arena is num_pages pages of page_bytes.  ONE
 * PAGE holds page_tokens tokens of ONE kv head of one request:
 *     kind CP_KIND_KV : K block [page_tokens][head_dim_qk] bf16 row-major, immediately
 *                       followed by V block [page_tokens][head_dim_v] bf16;
 *     kind CP_KIND_MLA: one block [page_tokens][head_dim_qk] bf16 (the latent row, e.g.
 *                       512 latent + 64 rope); the value of a token is the first
 *                       head_dim_v entries of its row.
 * A model fits the pool if its block(s) fit in page_bytes (trailing bytes unused).
 * A request's page list is PAGE-MAJOR: page_ids[lp * n_kv_heads + c] is the physical page
 * of logical page lp (tokens lp*P .. lp*P+P-1) of kv head c.  Query head h reads kv head
 * c = h / (n_q_heads / n_kv_heads) (reading A2).  Slots past context_len in the last
 * page, and all unmapped pages, are undefined and never influence a result (reading A5).
 */
#ifndef CROSSPOOL_H_
#define CROSSPOOL_H_

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct cp_pool cp_pool;   /* opaque; created by cp_pool_create, owned by the library */
typedef int32_t cp_status;

enum {
    CP_OK = 0,
    CP_ERR_INVALID_ARG = -1,      /* NULL / out-of-range / inconsistent argument           */
    CP_ERR_NO_PAGES = -2,         /* page budget exhausted: the paper's "reject" (L122)     */
    CP_ERR_PAGE_RANGE = -3,       /* a page id is >= num_pages or negative                  */
    CP_ERR_PAGE_IN_USE = -4,      /* a page is already owned (or repeated in the list)      */
    CP_ERR_UNKNOWN_REQUEST = -5,  /* request id not mapped                                  */
    CP_ERR_UNSUPPORTED = -6,      /* model shape outside what the kernels implement         */
    CP_ERR_WORKSPACE = -7,        /* workspace_dev too small or misaligned                  */
    CP_ERR_CUDA = -8,             /* CUDA runtime / driver error (no device, launch fault)  */
    CP_ERR_TOO_LARGE = -9         /* problem exceeds the fixed capacity of a *_noalloc entry point */
};

enum { CP_KIND_KV = 0, CP_KIND_MLA = 1 };

/* Per-model KV description: "KV tensor layouts, numbers of KV heads, and per-token KV
 * bytes" differ per colocated model (challenge C1; kappa(M) in L103). */
typedef struct {
    int32_t kind;            /* CP_KIND_KV (MQA/GQA/MHA) or CP_KIND_MLA                      */
    int32_t n_q_heads;       /* Hq                                                          */
    int32_t n_kv_heads;      /* Hkv; Hq % Hkv == 0; MLA requires 1                          */
    int32_t head_dim_qk;     /* d_k (MLA: full latent row width, e.g. 576)                  */
    int32_t head_dim_v;      /* d_v (MLA: leading part of the row that is the value)        */
    float   softmax_scale;   /* sigma; multiplies the fp32 dot product (reading A3)         */
} cp_model_cfg;

/* One tile of the device work list (introspection only; see cp_decode_plan). */
typedef struct {
    int32_t batch_index;     /* position of the request in the decode batch                 */
    int32_t kv_head;         /* kv head of the (request, kv head) group this tile belongs to */
    int32_t split;           /* index of this KV split inside the group                     */
    int32_t n_splits;        /* number of KV splits of the group                            */
    int32_t page_begin;      /* first logical page of the tile                              */
    int32_t page_end;        /* one past the last logical page                              */
} cp_tile_info;

/* Tunables (cp_pool_set_option). */
enum {
    CP_OPT_KERNEL = 0,       /* 0 = auto (tensor-core kernels where the shape allows: MQA/GQA groups of up
                                    to 32 rows on the tcgen05 tokens-on-M kernel, MLA on CTA pairs,
                                    tcgen05 cta_group::2),
                                1 = force the generic SIMT kernel (any supported shape),
                                2 = as 0, but MLA on the single-CTA tcgen05 kernel, and q_len > 1 on the
                                    tcgen05 K/V kernel for groups of up to 32 rows (0: up to 16 rows),
                                3 = as 0, but MQA/GQA on the warp-MMA (mma.sync) kernel          */
    CP_OPT_NUM_CTAS = 1,     /* persistent grid size; 0 = number of SMs of the device       */
    CP_OPT_WAVES_X16 = 2,    /* target tiles per CTA, in 1/16 units (default 16 = 1.0)      */
    CP_OPT_MIN_TILE_PAGES = 3, /* lower bound on pages per tile (default 2)                  */
    CP_OPT_VMM_TABLE = 4,    /* pool from cp_pool_create_vmm only: 1 = the decode kernels read the
                                software page table anyway (it holds the same ids; for measuring
                                what the table costs), 0 (default) = page ids by arithmetic   */
    CP_OPT_HOST_ZERO_COPY = 5, /* cp_decode_attention_host: 1 (default) = pinned, device-mapped host
                                buffers are accessed in place (O / LSE written once; Q only when
                                its re-reads by the tiles stay under 1 MB), 0 = always staged  */
    CP_OPT_STATIC_PCT = 7,   /* tcgen05 MQA/GQA kernel: per cent of every group's 128-token slices that go into the
                                static, equally long per-CTA pieces (default 100); the rest forms short
                                tiles the CTAs pop dynamically when their static lists are done      */
    CP_OPT_TAIL_TILE_SLICES = 8, /* ... and the length of those tiles in slices (default 2)            */
    CP_OPT_TIMELINE = 6      /* 1 = the next cp_decode_attention launches record per-CTA globaltimer
                                stamps (cp_pool_read_timeline); 0 (default) = off.  Measurement aid of
                                bench.py --probe timeline; kernels that do not stamp leave zeros.  */
};

/*
 * cp_pool_create -- describe a shared KV-cache pool over a caller-owned device arena.
 * "a shared KV-cache pool ... total KV-cache pool page budget"; the
 * budget is num_pages.  The arena is never read or written by this call.  No CUDA call is
 * made here (device metadata is allocated lazily by the first compute call), so pool
 * bookkeeping can be exercised on a host without a GPU.
 *   arena_dev              device pointer, 256-B aligned, >= num_pages * page_bytes bytes
 *   page_tokens            P, tokens per page (multiple of 16, <= 256)
 *   page_bytes             bytes per page (multiple of 256)
 *   models / n_models      copied; model ids are indices into this array
 *   max_requests           request ids are 0 .. max_requests-1
 *   max_pages_per_request  capacity of one request's page list (entries = logical pages
 *                          * n_kv_heads)
 * Errors: INVALID_ARG (NULL, zero sizes, arena too small / misaligned), UNSUPPORTED (Hq not a
 * multiple of Hkv, head dims not multiples of 16 or > 576 (qk) / 512 (v), MLA with Hkv != 1
 * or d_v > d_k, a model whose page does not fit page_bytes).
 */
cp_status cp_pool_create(void *arena_dev, uint64_t arena_bytes,
                         uint32_t page_tokens, uint32_t page_bytes, uint32_t num_pages,
                         const cp_model_cfg *models, int32_t n_models,
                         int32_t max_requests, int32_t max_pages_per_request,
                         cp_pool **out);

/*
 * cp_pool_create_vmm -- the same pool on an arena the LIBRARY owns and backs with the CUDA
 * virtual memory management API: "CUDA VMM APIs to reserve a virtual KV address range for each
 * model and map physical KV pages on demand".  One virtual
 * range is reserved and cut into max_requests slots; request id r owns slot r, a contiguous
 * virtual KV space of slot_pages >= max_pages_per_request pages, so entry i of its page list is
 * page r * slot_pages + i and the decode kernels need no table lookup (CP_OPT_VMM_TABLE).
 * Physical memory is created in chunks of the device's allocation granularity (2 MiB) the first
 * time a request grows into them, and parked for reuse when the request is unmapped; chunks in
 * existence never exceed physical_budget_bytes / chunk size -- the pool page budget.
 * Differences from a caller-owned arena:
 *   - cp_pool_map_pages takes page_ids_host == NULL only (INVALID_ARG otherwise) and maps the
 *     chunks under the new pages; NO_PAGES when the budget cannot back them (nothing changes);
 *   - cp_pool_unmap_request synchronises the device, then unmaps the slot's chunks;
 *   - cp_pool_stats reports free pages as what the chunks still available could hold;
 *   - cp_pool_free unmaps and releases everything.
 * Pages of different requests never share a chunk (a slot starts on a chunk boundary).
 * Errors: INVALID_ARG, UNSUPPORTED (as cp_pool_create), CUDA (no device / driver call failed).
 */
cp_status cp_pool_create_vmm(uint64_t physical_budget_bytes,
                             uint32_t page_tokens, uint32_t page_bytes,
                             const cp_model_cfg *models, int32_t n_models,
                             int32_t max_requests, int32_t max_pages_per_request,
                             cp_pool **out);

/* cp_pool_vmm_info -- geometry and occupancy of a VMM pool (INVALID_ARG for any other pool): base
 * device address of the reserved range and its size, chunk size, pages per request slot, chunks
 * mapped now, chunk budget.  Any out pointer may be NULL.  The bytes of request r's pages live at
 * arena_dev + r * slot_pages * page_bytes; only its mapped prefix may be touched. */
cp_status cp_pool_vmm_info(const cp_pool *pool, void **arena_dev, uint64_t *va_bytes,
                           uint64_t *chunk_bytes, uint32_t *slot_pages,
                           uint32_t *chunks_mapped, uint32_t *chunks_budget);

/* cp_pool_free -- release the library's metadata (host and device).  Never touches the
 * arena.  NULL is accepted. */
cp_status cp_pool_free(cp_pool *pool);

/*
 * cp_pool_map_pages -- the virtualizer's slow path: "map physical KV pages on demand ...
 * mapping and unmapping remain slow paths outside the per-token critical path"
 * (PAPER.md:L122).  The first call for a request id creates the request (model_id fixed
 * from then on); later calls APPEND page ids and/or raise context_len.
 *   page_ids_host   n_page_ids physical page ids to append (page-major, see top), or NULL
 *                   with n_page_ids > 0 to let the library take pages from its free list,
 *                   or NULL with n_page_ids == 0 to only update context_len
 *   context_len     number of valid tokens now in the pool for this request (>= 1, never
 *                   decreasing, <= mapped logical pages * P) (readings A4, A8)
 * All-or-nothing.  Errors: INVALID_ARG, UNSUPPORTED (n_page_ids not a multiple of Hkv),
 * PAGE_RANGE, PAGE_IN_USE, NO_PAGES (budget exhausted -> the caller queues or rejects,
 * PAPER.md:L122), UNKNOWN_REQUEST is never returned here.
 * The device copy of the tables is refreshed by the next compute call on its stream.
 */
cp_status cp_pool_map_pages(cp_pool *pool, int32_t request_id, int32_t model_id,
                            const int32_t *page_ids_host, int32_t n_page_ids,
                            int32_t context_len);

/* cp_pool_unmap_request -- the request finished decoding: its pages return to the free
 * list ("Active KV pages are kept until their decode requests finish"). */
cp_status cp_pool_unmap_request(cp_pool *pool, int32_t request_id);

/* cp_pool_request_info -- query a request: model, context length, number of page-list
 * entries; if page_ids_out_host != NULL copies up to cap entries.  Any out pointer may be
 * NULL. */
cp_status cp_pool_request_info(const cp_pool *pool, int32_t request_id, int32_t *model_id,
                               int32_t *context_len, int32_t *n_page_ids,
                               int32_t *page_ids_out_host, int32_t cap);

/* cp_pool_stats -- free / used pages against the page budget. */
cp_status cp_pool_stats(const cp_pool *pool, uint32_t *free_pages, uint32_t *used_pages);

/* cp_pool_set_option -- tunables above; INVALID_ARG for unknown keys / bad values. */
cp_status cp_pool_set_option(cp_pool *pool, int32_t key, int64_t value);

/*
 * cp_pool_gather_kv -- page-table translation + KV gather (hot-path step a2): "attention
 * kernels can use a logical KV address space while the virtualizer controls physical page
 * allocation".  Copies the raw 16-bit patterns of tokens 0..context_len-1:
 *   k_out_dev  bf16 [T][Hkv][d_k]   (MLA: [T][d_k], the latent rows)
 *   v_out_dev  bf16 [T][Hkv][d_v]   (MLA: [T][d_v], the leading part); may be NULL
 * Bit-exact (NaN payloads, -0 included).  Runs on `stream`.
 */
cp_status cp_pool_gather_kv(cp_pool *pool, int32_t request_id,
                            void *k_out_dev, void *v_out_dev, void *stream);

/*
 * cp_pool_append_kv -- the step right before attention in every decode iteration (SURVEY.md §8(f)
 * N1): write ONE new token per request into the pool at position context_len and raise
 * context_len by one.  When the position opens a new logical page the library takes the n_kv_heads
 * physical pages from its free list -- "map physical KV pages on demand" -- and
 * rejects the whole batch with CP_ERR_NO_PAGES if the budget is exhausted (never preempts).
 *   request_ids_host  batch order; ids must be distinct and mapped
 *   k_new_dev  bf16, packed in batch order, per request [Hkv][d_k]  (MLA: the latent row [d_k])
 *   v_new_dev  bf16, packed in batch order, per request [Hkv][d_v]  (MLA requests contribute nothing;
 *              may be NULL when the batch has only MLA requests)
 * All-or-nothing.  Only the 16-bit patterns move (bit-exact).  Runs on `stream`; the page table and
 * context lengths seen by later compute calls on the same stream include the new token.
 * Errors: INVALID_ARG (also: a page list that cannot grow), UNKNOWN_REQUEST, NO_PAGES, CUDA.
 */
cp_status cp_pool_append_kv(cp_pool *pool, const int32_t *request_ids_host, int32_t n_requests,
                            const void *k_new_dev, const void *v_new_dev, void *stream);

/*
 * cp_decode_workspace_bytes -- bytes of scratch cp_decode_attention needs for this batch
 * (split-KV partial results; 0 when no group is split).
 */
cp_status cp_decode_workspace_bytes(cp_pool *pool, const int32_t *request_ids_host,
                                    int32_t n_requests, uint64_t *bytes_out);

/*
 * cp_decode_attention -- ONE decode step of attention for a batch of requests of any mix
 * of the pool's models (batch sizes 1-4 per model are typical): for every
 * request r in the batch and query head h,
 *     s_t = sigma * <q_h, k_t>,  t = 0 .. T_r - 1  (k_t, v_t read through the page table)
 *     O_h = sum_t softmax(s)_t v_t,          LSE_h = ln sum_t exp(s_t)
 * computed as split-KV partial attention (online softmax, fp32 accumulation over bf16 K/V)
 * plus a log-sum-exp combine, scheduled by persistent kernels over a device-resident
 * work list of (request, model, kv-split) tiles: one launch per attention kind present in
 * the batch, no per-request launches (GPU-resident control instead of host-driven
 * dispatch).
 *   request_ids_host  batch order; ids must be distinct and mapped
 *   q_dev    bf16, packed in batch order, per request [Hq][d_k]
 *   out_dev  fp32, packed in batch order, per request [Hq][d_v]
 *   lse_dev  fp32, packed in batch order, per request [Hq] (natural log, scale inside)
 *   workspace_dev / workspace_bytes  >= cp_decode_workspace_bytes(...), 16-B aligned
 * Errors: INVALID_ARG, UNKNOWN_REQUEST, WORKSPACE, CUDA.
 * Streams: the compute calls of one pool (gather, append, decode*, stages, queue launch) reuse device-side
 * scheduler state from call to call -- the uploaded work list, two alternating sets of scheduler counters, the
 * page and context tables.  Calls on ONE stream are ordered by the stream.  A call on another stream than the
 * pool's previous call first waits (cudaStreamWaitEvent) for everything the previous stream was given, so two
 * streams may drive one pool in turn; calls are NOT thread-safe, and a launch must not be captured into a CUDA
 * graph and replayed (the host alternates the counter sets and re-uploads plans between launches).  A batch
 * with models of both attention kinds launches its second kernel on an internal stream and joins it back.
 */
cp_status cp_decode_attention(cp_pool *pool, const int32_t *request_ids_host, int32_t n_requests,
                              const void *q_dev, float *out_dev, float *lse_dev,
                              void *workspace_dev, uint64_t workspace_bytes, void *stream);

/*
 * cp_decode_step -- one decode ITERATION in one call: append the new token of every request
 * (cp_pool_append_kv's semantics: position context_len, page growth from the free list, all-or-nothing)
 * and attend over the grown contexts (cp_decode_attention's semantics and layouts).  "map physical KV
 * pages on demand" and attend over them.  For MQA / GQA models on the
 * tcgen05 kernel the append costs no launch: the persistent CTA whose tile holds a group's last page writes
 * the new K and V rows through the page table before it requests that page, so the iteration is ONE kernel
 * (cp_pool_counters counts one launch); requests of other kinds / kernels get cp_pool_append_kv's kernel in
 * front of theirs.  The device arena after the call is bit-identical to append-then-attend.
 *   k_new_dev, v_new_dev  as cp_pool_append_kv;  q_dev, out_dev, lse_dev, workspace_dev  as cp_decode_attention
 *   (the queries are those of the NEW token: they see context_len + 1 tokens)
 * cp_decode_step_workspace_bytes: scratch the call needs, i.e. for the contexts grown by one token (host
 * arithmetic on a plan of the grown contexts; the pool is not changed).
 * Errors: those of both calls.  WORKSPACE is detected after the host bookkeeping of the append and takes it
 * back (context lengths, free list), so the pool is unchanged on every error but CUDA.
 */
cp_status cp_decode_step_workspace_bytes(cp_pool *pool, const int32_t *request_ids_host, int32_t n_requests,
                                         uint64_t *bytes_out);
cp_status cp_decode_step(cp_pool *pool, const int32_t *request_ids_host, int32_t n_requests,
                         const void *k_new_dev, const void *v_new_dev, const void *q_dev, float *out_dev,
                         float *lse_dev, void *workspace_dev, uint64_t workspace_bytes, void *stream);

/*
 * cp_decode_attention_host -- the same step with HOST query / result buffers: copies q
 * host->device, runs cp_decode_attention, copies O and LSE device->host and synchronises
 * `stream`.  Host buffers that are pinned and device-mapped (cudaHostAlloc / cudaHostRegister) are
 * accessed by the kernel in place instead (CP_OPT_HOST_ZERO_COPY): the same bytes cross the bus, without
 * the separate copy operations before and after the kernel.  Otherwise O and LSE come back in one
 * copy when lse_host directly follows out_host in memory, in two when not.
 * The KV arena stays resident on the device (it is the cache).  The staging
 * copies of q / O / LSE live at the front of workspace_dev: it must hold
 * cp_decode_workspace_bytes_host(...) bytes.
 */
cp_status cp_decode_workspace_bytes_host(cp_pool *pool, const int32_t *request_ids_host,
                                         int32_t n_requests, uint64_t *bytes_out);
cp_status cp_decode_attention_host(cp_pool *pool, const int32_t *request_ids_host,
                                   int32_t n_requests, const void *q_host, float *out_host,
                                   float *lse_host, void *workspace_dev, uint64_t workspace_bytes,
                                   void *stream);

/*
 * cp_decode_attention_qlen -- the same step with q_len > 1 query tokens per request (the variant
 * SURVEY 8(f) N4 names; e.g. the verification step of speculative decoding).  The query tokens are
 * the LAST q_len tokens of each request: their K/V is already in the pool and counted by
 * context_len (reading Q1).  Query token j (0-based) sits at position
 * context_len - q_len + j and attends causally to positions 0 .. context_len - q_len + j.
 *   q_dev    bf16, per request [q_len][Hq][d_k];  out_dev fp32 [q_len][Hq][d_v];  lse_dev [q_len][Hq]
 *   q_len    1 .. 128 with (Hq / Hkv) * q_len <= 128; q_len = 1 is cp_decode_attention
 * For q_len > 1: MQA / GQA / MHA models with d_k = d_v = 128 on page sizes 16/32/64/128 only
 * (UNSUPPORTED otherwise, and with CP_OPT_KERNEL = 1); INVALID_ARG if a context is shorter than q_len.
 * Kernel: a batch whose groups have at most 16 rows ((Hq / Hkv) * q_len; 32 with CP_OPT_KERNEL = 2) runs
 * on the tcgen05 K/V kernel (the rows sit on the MMA N dimension, the causal limit is applied per row in
 * the slices that reach the context's last q_len - 1 tokens), any other on the warp-MMA kernel.
 */
cp_status cp_decode_workspace_bytes_qlen(cp_pool *pool, const int32_t *request_ids_host,
                                         int32_t n_requests, int32_t q_len, uint64_t *bytes_out);
cp_status cp_decode_attention_qlen(cp_pool *pool, const int32_t *request_ids_host, int32_t n_requests,
                                   int32_t q_len, const void *q_dev, float *out_dev, float *lse_dev,
                                   void *workspace_dev, uint64_t workspace_bytes, void *stream);

/*
 * cp_decode_attention_stages -- several attention steps in ONE persistent launch: an
 * attention-only mock of the layer-wise pipeline, "two in-flight batches, each with its own model
 * id, layer cursor, and completion state" advanced "without requiring the two batches to have the
 * same model or the same number of layers", with the control on the GPU:
 * persistent CTAs that select the next ready work, wait "for computation ... completion, and update
 * the batch state for the next layer" (L146) instead of one host launch per layer.
 * A STAGE is one attention step = one layer of one batch, over stage_sizes_host[s] mapped requests
 * (the KV of that layer; ids may repeat across stages, not inside one).  The caller lists the stages
 * in the order the scheduler's state machine issues them (e.g. B1 L0, B2 L0, B1 L1, B2 L1, ...).
 * stage_dep_host[s] = the stage whose output feeds stage s (the same batch one layer earlier), or
 * -1.  The FFN between two layers lives in the other pool and is out of scope; it is mocked by a
 * residual pass-through (reading M1): for a dependent stage the query rows are
 *     q = bf16(fp32(q_in) + alpha * O_dep)        (float32 product, float32 sum, round-to-nearest-even)
 * with q_in the rows given in q_dev.  A dependent stage must have the batch shape of its
 * predecessor (same number of requests, same model per slot).  Tiles of a dependent stage stream
 * their KV pages as soon as a CTA is free and wait only for their queries.
 *   q_dev / out_dev / lse_dev   packed stage after stage, inside a stage as for cp_decode_attention
 *   workspace_dev               >= cp_decode_stages_workspace_bytes(...) bytes, 16-B aligned
 * Supported: MQA / GQA / MHA models with d_k = d_v = 128 on page sizes 16/32/64/128 (the tensor-core
 * K/V kernel); anything else, or CP_OPT_KERNEL = 1: UNSUPPORTED.  Other errors: INVALID_ARG (bad
 * sizes, dep >= s, shape mismatch with the predecessor, NaN alpha), UNKNOWN_REQUEST, WORKSPACE, CUDA.
 */
cp_status cp_decode_stages_workspace_bytes(cp_pool *pool, int32_t n_stages,
                                           const int32_t *stage_sizes_host,
                                           const int32_t *request_ids_host,
                                           const int32_t *stage_dep_host, uint64_t *bytes_out);
cp_status cp_decode_attention_stages(cp_pool *pool, int32_t n_stages,
                                     const int32_t *stage_sizes_host,
                                     const int32_t *request_ids_host,
                                     const int32_t *stage_dep_host, float alpha,
                                     const void *q_dev, float *out_dev, float *lse_dev,
                                     void *workspace_dev, uint64_t workspace_bytes, void *stream);

/*
 * cp_decode_attention_stages_gated -- the same launch behind an ADMISSION DOORBELL: the persistent
 * CTAs poll *published_dev (any device-accessible int32: device memory the host updates with a copy on
 * another stream, or mapped pinned host memory) and hand out the tiles of stage s -- and request its
 * KV pages -- only once *published_dev > s.  This is the GPU-side half of "persistent kernel[s]
 * repeatedly poll per-model request queues on GPUs ... while the host remains responsible for
 * coarse-grained admission": the host admits batches while the kernel runs and
 * never launches per layer.  The caller must eventually publish n_stages.  A poll that lasts longer
 * than timeout_ms stops gating (the launch then completes as the ungated one would) and raises a flag
 * that cp_decode_stages_gate_status returns; the device is never left spinning.
 * Extra errors: INVALID_ARG (NULL / misaligned doorbell, timeout_ms = 0).
 * cp_decode_stages_gate_status synchronises `stream` and writes 1 if the last gated launch saw a
 * poll time out, else 0.
 */
cp_status cp_decode_attention_stages_gated(cp_pool *pool, int32_t n_stages,
                                           const int32_t *stage_sizes_host,
                                           const int32_t *request_ids_host,
                                           const int32_t *stage_dep_host, float alpha,
                                           const void *q_dev, float *out_dev, float *lse_dev,
                                           void *workspace_dev, uint64_t workspace_bytes, void *stream,
                                           const int32_t *published_dev, uint32_t timeout_ms);
cp_status cp_decode_stages_gate_status(cp_pool *pool, void *stream, int32_t *timed_out_host);

/*
 * cp_decode_plan -- introspection of the device work list the next cp_decode_attention on
 * this batch will consume (host only, no CUDA): writes up to cap tiles in the order the
 * persistent CTAs pop them.  n_tiles_out receives the total number of tiles,
 * n_groups_out the number of (request, kv head) groups.  tiles_out may be NULL.
 */
cp_status cp_decode_plan(cp_pool *pool, const int32_t *request_ids_host, int32_t n_requests,
                         cp_tile_info *tiles_out, int32_t cap, int32_t *n_tiles_out,
                         int32_t *n_groups_out);

/* cp_pool_counters -- monotonically increasing counters since cp_pool_create: kernels
 * launched by the library, work-list (re)builds, host->device metadata bytes. */
cp_status cp_pool_counters(const cp_pool *pool, uint64_t *kernel_launches,
                           uint64_t *plan_builds, uint64_t *metadata_h2d_bytes);

/* cp_pool_read_timeline -- measurement aid (`bench.py --probe timeline`): with CP_OPT_TIMELINE = 1
 * the persistent CTAs of the MQA/GQA tcgen05 kernel stamp %globaltimer (ns) at fixed points of their life:
 *   slot 0 kernel entry, 1 the producer warp has its first tile, 2 first slice landed, 3 producer issued its last
 *   page, 4 softmax of a tile's last slice done, 5 tile published, 6 arrival at the barrier before the LSE combine,
 *   7 combine done, 8 %smid (not a time), 9 first TMA issued, 10 last slice landed, 11 tiles this CTA ran (a count),
 *   12 the combine's counters complete, 13 the combine's partials loaded, 14 set-up barrier and griddepcontrol.wait
 *   passed, 15 the scheduler warp has its first tile record (0 = not stamped).  A stamp taken right after a CTA
 *   barrier shows the thread's arrival, not the release.
 * Synchronises the device and copies the stamps of the last launch of the pool: stamps_out_host holds
 * cap_ctas x 16 uint64; n_ctas_out receives the number of CTA rows available (the SM count). */
cp_status cp_pool_read_timeline(cp_pool *pool, uint64_t *stamps_out_host, int32_t cap_ctas, int32_t *n_ctas_out);

/*
 * Request queue of a persistent launch: "persistent kernels repeatedly poll per-model request
 * queues on GPUs, select the next ready batch ... and update the batch state for the next layer", while "the host
 * remains responsible for coarse-grained admission" (state machine L126-L128).  Unlike
 * cp_decode_attention_stages, whose stage list is built by the host before the launch, the kernel started by
 * cp_queue_launch knows NOTHING of the work to come: the host pushes stage descriptors -- a batch of request ids
 * and the stage that feeds it -- into a ring in mapped host memory WHILE THE KERNEL RUNS, a planner warp on the
 * GPU cuts every batch into tiles as it arrives (the arithmetic of the host planner, from the device-resident
 * context lengths and model shapes) and the persistent CTAs consume them; a batch that exits early simply stops
 * being pushed; cp_queue_close ends the launch.  Stage semantics are those of cp_decode_attention_stages
 * (reading M1: q = bf16(q_in + alpha * O_dep)); stage s's rows follow stage s - 1's in q / out / lse.
 *   cp_queue_create   max_stages = capacity of the ring (no wrap: a queue serves one launch).  MQA / GQA / MHA
 *                     models with 128-wide heads only (the warp-MMA K/V kernel): UNSUPPORTED otherwise.
 *   cp_queue_launch   starts the persistent kernel on `stream` and returns; workspace_dev holds the split
 *                     partials of ALL stages (handed out cumulatively; a stage that does not fit ends the
 *                     launch with error 2).  timeout_ms: a planner that sees no push for that long closes the
 *                     launch itself (error 1) instead of spinning forever.  The requests' pages and context
 *                     lengths must not change while the launch runs.
 *   cp_queue_push     host only, any time before cp_queue_close (before or after the launch): at most 12 distinct
 *                     mapped requests; dep_stage = index of an earlier stage of the same batch shape, or -1.
 *                     *stage_index_out receives the stage's index.  Errors: INVALID_ARG, UNKNOWN_REQUEST, UNSUPPORTED.
 *   cp_queue_close    no further pushes; the kernel drains and exits.
 *   cp_queue_status   synchronises `stream`; stages / tiles the device planned and the device's error word
 *                     (0 none, 1 timed out, 2 a capacity was exceeded, 3 malformed entry).
 */
typedef struct cp_queue cp_queue;
cp_status cp_queue_create(cp_pool *pool, int32_t max_stages, cp_queue **out);
cp_status cp_queue_launch(cp_queue *q, const void *q_dev, float *out_dev, float *lse_dev, void *workspace_dev,
                          uint64_t workspace_bytes, uint32_t timeout_ms, void *stream);
cp_status cp_queue_push(cp_queue *q, const int32_t *request_ids_host, int32_t n_requests, int32_t dep_stage,
                        float alpha, int32_t *stage_index_out);
cp_status cp_queue_close(cp_queue *q);
cp_status cp_queue_status(cp_queue *q, void *stream, int32_t *stages_planned, int32_t *tiles_planned, int32_t *error);
cp_status cp_queue_free(cp_queue *q);

/* Measurement aids without any part in the hot path (cp_probe.cu; `bench.py --probe ...`).
 * cp_probe_globaltimer: a one-thread kernel on `stream` that stores %globaltimer (ns) to *stamp_dev (8-byte
 *   aligned device memory); bracketing a decode launch with two of them relates the per-CTA stamps of
 *   cp_pool_read_timeline to the stream's own order (launch gap before the first CTA, drain after the last).
 * cp_probe_read_stream: reads `bytes` of device memory once with 16-byte loads from n_ctas CTAs of 512
 *   threads (nothing is written; *sink_dev, 4 bytes of device memory, only keeps the loads alive): the
 *   read-only HBM ceiling next to the copy bandwidth of MEASURED_PEAKS.json.
 * Both return INVALID_ARG for null / misaligned pointers, CUDA when the launch fails. */
cp_status cp_probe_globaltimer(uint64_t *stamp_dev, void *stream);
cp_status cp_probe_read_stream(const void *src_dev, uint64_t bytes, int32_t n_ctas, uint32_t *sink_dev, void *stream);

/*
 * KV-cache planner: "The planner uses per-model prompt, output, and service-time
 * samples, arrival rate, page size, per-token KV bytes kappa(M), and a target provisioning
 * quantile.  It emits ... the total KV-cache pool page budget".  For request i of
 * model M arriving at A_i with O_p,i prompt tokens, O_d,i output tokens and decode residence T_i,
 *     Q_i(u) = (O_p,i + O_d,i u / T_i) 1{0 <= u < T_i},   K_M(t) = sum_i kappa(M) Q_i(t - A_i)   (1)
 *     K_pool(t) = sum_M K_M(t)                                                                  (2)
 * and the budget is the "P95/P99 trace-driven Monte Carlo quantile" of K_pool over random
 * observation times, rounded up to pages (L112).  The observation times are drawn by the caller.
 * All arithmetic is float64, each operation rounded separately in the order written above (terms in
 * trace order, models in index order), so results equal a sequential evaluation bit for bit.
 * The pool these numbers size is created with num_pages (cp_pool_create) or physical_budget_bytes
 * (cp_pool_create_vmm) = the budget; the planner functions need no cp_pool.
 *
 * cp_planner_pool_demand -- K_pool at n_obs observation times (asynchronous on `stream`).
 *   n_models             1 .. CP_PLANNER_MAX_MODELS
 *   trace_offsets_host   [n_models + 1], offsets[0] = 0, non-decreasing: model M owns trace entries
 *                        offsets[M] .. offsets[M+1]-1 of the four trace arrays
 *   kappa_host           [n_models] per-token KV bytes, >= 0
 *   arrival_dev          A_i (s), ASCENDING inside each model (precondition, not checked)
 *   prompt_tokens_dev, output_tokens_dev, residence_dev   O_p,i, O_d,i, T_i (doubles; T_i <= 0
 *                        makes the request contribute nothing)
 *   t_obs_dev / k_pool_dev   [n_obs] in / out (bytes)
 *   workspace_dev        >= cp_planner_workspace_bytes(offsets[n_models]) bytes, 16-B aligned,
 *                        caller-owned (cp_planner_quantile needs cp_planner_workspace_bytes(0))
 * Errors: INVALID_ARG, WORKSPACE, CUDA.
 *
 * cp_planner_quantile -- the empirical quantile x_(k), k = ceil(q n) (1-based order statistic, no
 * interpolation: at least a fraction q of the values is <= it) of n finite NON-NEGATIVE doubles in
 * device memory, and pages = ceil(x_(k) / page_bytes).  Exact selection (radix select on the bit
 * patterns); values_dev is not modified.  Synchronises `stream` and writes the two results to the
 * host.  Either out pointer may be NULL.  Errors: INVALID_ARG (n < 1, q outside (0, 1]), WORKSPACE,
 * CUDA.
 */
#define CP_PLANNER_MAX_MODELS 64
uint64_t cp_planner_workspace_bytes(int64_t n_trace_entries);
cp_status cp_planner_pool_demand(int32_t n_models, const int64_t *trace_offsets_host,
                                 const double *kappa_host, const double *arrival_dev,
                                 const double *prompt_tokens_dev, const double *output_tokens_dev,
                                 const double *residence_dev, int64_t n_obs, const double *t_obs_dev,
                                 double *k_pool_dev, void *workspace_dev, uint64_t workspace_bytes,
                                 void *stream);
cp_status cp_planner_quantile(const double *values_dev, int64_t n, double q, double page_bytes,
                              void *workspace_dev, uint64_t workspace_bytes,
                              double *quantile_out_host, uint64_t *pages_out_host, void *stream);

/*
 * cp_planner_pool_demand_noalloc -- cp_planner_pool_demand for callers that cannot allocate device memory
 * (code under CUDA graph capture, tight serving loops, harnesses that forbid cudaMalloc): same
 * arguments without the workspace, same launches, same results bit for bit.  The scratch lives in a
 * file-scope device array of the library (about 0.5 MiB, held by every GPU that loads the library until
 * the process exits), sized for traces of up to CP_PLANNER_NOALLOC_MAX_TRACE entries in all
 * (trace_offsets_host[n_models]); a longer trace is rejected with CP_ERR_TOO_LARGE before any CUDA call.
 * The call itself makes no cudaMalloc / cudaFree and calls no allocating library routine (one
 * cudaGetSymbolAddress per device on first use, one cudaMemsetAsync, three kernel launches).
 * ALL calls of a device share the one array, which keeps the last call's contents (each call clears or
 * overwrites everything it reads): calls that may overlap on the GPU -- different streams without an
 * ordering between them -- race on it and must use cp_planner_pool_demand with workspaces of their own.
 * Other errors: as cp_planner_pool_demand (INVALID_ARG, CUDA).
 */
#define CP_PLANNER_NOALLOC_MAX_TRACE (1 << 20)
cp_status cp_planner_pool_demand_noalloc(int32_t n_models, const int64_t *trace_offsets_host,
                                         const double *kappa_host, const double *arrival_dev,
                                         const double *prompt_tokens_dev, const double *output_tokens_dev,
                                         const double *residence_dev, int64_t n_obs, const double *t_obs_dev,
                                         double *k_pool_dev, void *stream);

/* cp_status_string -- static, never NULL. */
const char *cp_status_string(cp_status status);

#ifdef __cplusplus
}
#endif
#endif /* CROSSPOOL_H_ */
