// cp_kernels_kv.cu -- the MQA / GQA fast path of libcrosspool (hot-path steps a2-a6 for
// kind CP_KIND_KV with d_k = d_v = 128): ONE persistent launch per decode step.
//
//   * 1 producer warp: pops work items (tiles, then combine units) from the device work
//     list with a global atomic, translates logical pages through the page table and
//     streams the pages into a ring of shared-memory stages with TMA
//     (cp.async.bulk.tensor, SWIZZLE_128B boxes, mbarrier complete_tx, L2 evict-first).
//   * 8 consumer warps: a page is cut into 16/32-token slices; (slice, 16-query-head M tile)
//     units are dealt round-robin to the warps, so all warps work on the oldest page of
//     the ring at once.  S = Q K^T and O += P V on warp-level tensor-core MMA (mma.sync
//     m16n8k16, bf16 in, fp32 accumulate; operands via conflict-free ldmatrix from the
//     swizzled stage), online softmax in fp32 in log2 units.  North-star keeps tcgen05/TMEM for the MLA
//     path; this path is HBM-bound and the MMA only keeps the FP32 ALUs off the critical
//     path.
//   * slice lanes merge their running (m, l, O) through shared memory at the end of a
//     tile (fixed tree => deterministic), then publish the split partial (or the final
//     result when the group has a single split) and bump the group's counter; combine
//     items (LSE combine, step a4: one warp per (group, head, 32 columns)) are popped
//     from the same work list.
//
// Paper anchors: paged KV interface PAPER.md:L101,L122; KV-head-limited attention under
// low concurrency PAPER.md:L21,L57; GPU-resident persistent control PAPER.md:L146.
#include <cuda.h>
#include <cuda_runtime.h>
#include <cstdint>
#include "cp_device_common.cuh"
#include "cp_ptx.cuh"
#include "cp_launch.h"

namespace cp {

constexpr int KV_CWARPS = 8;                       // consumer warps
constexpr int KV_CTHREADS = KV_CWARPS * 32;        // 256
constexpr int KV_THREADS = KV_CTHREADS + 32;       // + producer warp
constexpr int KV_D = 128;                          // head dim (qk and v)
constexpr int KV_TQ = 4;                           // tile-queue depth
constexpr int KV_MERGE_SLOT_FLOATS = 68 * 32;      // per sender warp: 64 O + m0,m1,l0,l1 per lane
constexpr int KV_MERGE_BYTES = 4 * KV_MERGE_SLOT_FLOATS * 4;
constexpr int KV_MAX_STAGES = 16;
constexpr int KV_LDSM_DEPTH = 4;                   // ldmatrix prefetch distance (register ring)
constexpr float KV_LAZY_LOG2 = 8.0f;               // lazy-rescale threshold (log2 units)
constexpr int KV_SMEM_LIMIT = 232448;              // 227 KB opt-in maximum per CTA

constexpr int KV_COMBINE_WARP_FLOATS = kMaxSplits;  // per-warp split weights of the LSE combine
static_assert(KV_CWARPS * KV_COMBINE_WARP_FLOATS * 4 <= KV_MERGE_BYTES, "combine scratch must fit the merge area");

__host__ __device__ constexpr int kv_stage_bytes(int P) { return P * 4 * KV_D; }   // K + V blocks
__host__ __device__ constexpr int kv_num_stages(int P)
{
    return (KV_SMEM_LIMIT - KV_MERGE_BYTES - 1024) / kv_stage_bytes(P) > KV_MAX_STAGES
               ? KV_MAX_STAGES
               : (KV_SMEM_LIMIT - KV_MERGE_BYTES - 1024) / kv_stage_bytes(P);
}
__host__ __device__ constexpr int kv_smem_bytes(int P)
{
    return kv_num_stages(P) * kv_stage_bytes(P) + KV_MERGE_BYTES + 1024;
}
__host__ __device__ inline int kv_mtiles(int g)     // 16-head M tiles, rounded to a power of two
{
    int mt = (g + 15) / 16, p = 1;
    while (p < mt) p <<= 1;
    return p;
}

// What the producer hands to the consumers for one work item (shared-memory tile queue), so
// that no consumer warp chases tile -> group -> model pointers through global memory.
struct TileDesc {
    int32_t item;            // work index; < 0: no more work
    int32_t group_idx;
    int32_t page_begin;
    int32_t npg;
    int32_t split;
    int32_t n_splits;
    int32_t ctx;
    int32_t gsize;           // query heads per kv head
    int32_t mt;              // 16-head M tiles (power of two)
    float scale_log2;
    int64_t q_off, out_off, lse_off, part_off;
    int32_t stage;           // multi-stage launches: the stage of this tile; q_len > 1: heads per kv head
    int32_t hq;              // query heads of the model (row stride of a query token)
};

// ----------------------------------------------------------------------------- PTX helpers (see also cp_ptx.cuh)
__device__ __forceinline__ void ldmatrix_x4(uint32_t &r0, uint32_t &r1, uint32_t &r2, uint32_t &r3, uint32_t addr)
{
    asm volatile("ldmatrix.sync.aligned.m8n8.x4.shared.b16 {%0,%1,%2,%3}, [%4];"
                 : "=r"(r0), "=r"(r1), "=r"(r2), "=r"(r3) : "r"(addr));
}
__device__ __forceinline__ void ldmatrix_x4_trans(uint32_t &r0, uint32_t &r1, uint32_t &r2, uint32_t &r3, uint32_t addr)
{
    asm volatile("ldmatrix.sync.aligned.m8n8.x4.trans.shared.b16 {%0,%1,%2,%3}, [%4];"
                 : "=r"(r0), "=r"(r1), "=r"(r2), "=r"(r3) : "r"(addr));
}
__device__ __forceinline__ void mma_bf16(float (&c)[4], const uint32_t (&a)[4], uint32_t b0, uint32_t b1)
{
    // not volatile: the compiler may schedule it freely after the (ordered) ldmatrix that feeds it
    asm("mma.sync.aligned.m16n8k16.row.col.f32.bf16.bf16.f32 {%0,%1,%2,%3}, {%4,%5,%6,%7}, {%8,%9}, {%0,%1,%2,%3};"
                 : "+f"(c[0]), "+f"(c[1]), "+f"(c[2]), "+f"(c[3])
                 : "r"(a[0]), "r"(a[1]), "r"(a[2]), "r"(a[3]), "r"(b0), "r"(b1));
}
__device__ __forceinline__ float ex2(float x)        // 2^x, flush-to-zero; ex2(-inf) = 0
{
    float r;
    asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x));
    return r;
}
__device__ __forceinline__ uint32_t pack_bf16(float lo, float hi)
{
    uint32_t r;
    asm("cvt.rn.bf16x2.f32 %0, %1, %2;" : "=r"(r) : "f"(hi), "f"(lo));
    return r;
}
__device__ __forceinline__ void consumer_bar()      // the 256 consumer threads only
{
    asm volatile("bar.sync 1, %0;" ::"n"(KV_CTHREADS) : "memory");
}

struct ConsumerSync {
    __device__ __forceinline__ void operator()() const { consumer_bar(); }
};

// ----------------------------------------------------------------------------- the kernel
// One work unit of a consumer warp: a slice of 8*NT tokens of the page in stage `sb` against the
// warp's 16-head M tile.  S (16 x 8NT) = Q K^T as NT independent accumulator chains (ILP for the
// tensor pipe), one online-softmax update per unit (log2 units), O (16 x 128) += P V.
// koff / vbase: per-lane swizzle constants (see the caller).
// QLEN (several query tokens per request): the two rows of a thread may belong to different query
// tokens, each with its own causal limit (valid - back0 / valid - back1); a row can then have no
// visible token in a slice, or none yet at all (m = -inf), which the single-token path never sees.
template <int P, int NT, bool QLEN = false>
__device__ __forceinline__ void kv_slice_unit(const uint32_t sb, const int tok0, const int valid,
                                              const uint32_t (&qf)[8][4], const float scale_log2,
                                              float (&o)[16][4], float (&m_run)[2], float (&l_run)[2],
                                              const int lane, const uint32_t (&koff)[2], const uint32_t vrow,
                                              const uint32_t vbase, const int back0 = 0, const int back1 = 0)
{
    constexpr int SUB = P * 128;                    // one swizzled sub-tile: P rows x 128 B
    const int cq = (lane & 3) * 2;
    const int valid0 = QLEN ? valid - back0 : valid, valid1 = QLEN ? valid - back1 : valid;
    // ---- S = Q K^T for 8*NT tokens
    float s[NT][4];
#pragma unroll
    for (int nt = 0; nt < NT; ++nt) { s[nt][0] = s[nt][1] = s[nt][2] = s[nt][3] = 0.f; }
    const uint32_t kb = sb + tok0 * 128;
    {
        // 4*NT ldmatrix.x4, each feeding 2 MMAs.  The loads are issued KV_LDSM_DEPTH steps ahead of
        // their use through a small register ring (ldmatrix is asm volatile, i.e. kept in program
        // order: without the explicit prefetch every MMA pair would wait a full shared-memory latency).
        constexpr int L = 4 * NT;
        uint32_t fr[KV_LDSM_DEPTH][4];
        // load i -> (kp = i / NT, nt = i % NT): row = tok0 + nt*8 + (lane & 7); 16-B chunk kp*4 + (lane >> 3)
#define KV_K_ADDR(i) (kb + ((i) % NT) * 8 * 128 + (((i) / NT) >> 1) * SUB + koff[((i) / NT) & 1])
#pragma unroll
        for (int i = 0; i < KV_LDSM_DEPTH; ++i)
            ldmatrix_x4(fr[i][0], fr[i][1], fr[i][2], fr[i][3], KV_K_ADDR(i));
#pragma unroll
        for (int i = 0; i < L; ++i) {
            const int kp = i / NT, nt = i % NT;
            mma_bf16(s[nt], qf[2 * kp], fr[i % KV_LDSM_DEPTH][0], fr[i % KV_LDSM_DEPTH][1]);
            mma_bf16(s[nt], qf[2 * kp + 1], fr[i % KV_LDSM_DEPTH][2], fr[i % KV_LDSM_DEPTH][3]);
            if (i + KV_LDSM_DEPTH < L)
                ldmatrix_x4(fr[i % KV_LDSM_DEPTH][0], fr[i % KV_LDSM_DEPTH][1], fr[i % KV_LDSM_DEPTH][2],
                            fr[i % KV_LDSM_DEPTH][3], KV_K_ADDR(i + KV_LDSM_DEPTH));
        }
#undef KV_K_ADDR
    }
    // ---- online softmax, rows r0 = lane / 4 and r0 + 8
    float mx0 = -INFINITY, mx1 = -INFINITY;
#pragma unroll
    for (int nt = 0; nt < NT; ++nt) {
        const int t = tok0 + nt * 8 + cq;
        s[nt][0] = (t < valid0) ? s[nt][0] * scale_log2 : -INFINITY;
        s[nt][1] = (t + 1 < valid0) ? s[nt][1] * scale_log2 : -INFINITY;
        s[nt][2] = (t < valid1) ? s[nt][2] * scale_log2 : -INFINITY;
        s[nt][3] = (t + 1 < valid1) ? s[nt][3] * scale_log2 : -INFINITY;
        mx0 = fmaxf(mx0, fmaxf(s[nt][0], s[nt][1]));
        mx1 = fmaxf(mx1, fmaxf(s[nt][2], s[nt][3]));
    }
    mx0 = fmaxf(mx0, __shfl_xor_sync(0xffffffffu, mx0, 1));
    mx1 = fmaxf(mx1, __shfl_xor_sync(0xffffffffu, mx1, 1));
    mx0 = fmaxf(mx0, __shfl_xor_sync(0xffffffffu, mx0, 2));
    mx1 = fmaxf(mx1, __shfl_xor_sync(0xffffffffu, mx1, 2));
    // Lazy reference update: the running reference m only moves when the slice maximum exceeds
    // it by more than 2^KV_LAZY_LOG2 (p <= 2^KV_LAZY_LOG2 stays exact enough in bf16/fp32 and cannot
    // overflow), so the O rescale below is rare instead of once per slice.  (m, l, O) stay
    // mutually consistent: any reference gives the same O / l and LSE = m + log2 l.
    // token tok0 is valid (the caller skips dead slices), so mn0 / mn1 are finite
    float mn0 = (mx0 > m_run[0] + KV_LAZY_LOG2) ? mx0 : m_run[0];
    float mn1 = (mx1 > m_run[1] + KV_LAZY_LOG2) ? mx1 : m_run[1];
    // QLEN: a row that has seen no token yet keeps m = -inf; the exponents below then use 0 as the
    // reference (2^(-inf - 0) = 0) instead of -inf - (-inf)
    const float mk0 = mn0, mk1 = mn1;
    if (QLEN) {
        mn0 = (mn0 == -INFINITY) ? 0.f : mn0;
        mn1 = (mn1 == -INFINITY) ? 0.f : mn1;
    }
    if (__any_sync(0xffffffffu, (mk0 != m_run[0]) || (mk1 != m_run[1]))) {
        const float a0 = ex2(m_run[0] - mn0), a1 = ex2(m_run[1] - mn1);
        l_run[0] *= a0; l_run[1] *= a1;
#pragma unroll
        for (int i = 0; i < 16; ++i) { o[i][0] *= a0; o[i][1] *= a0; o[i][2] *= a1; o[i][3] *= a1; }
        m_run[0] = mk0; m_run[1] = mk1;
    }
    uint32_t pf[NT * 2];
    float sum0 = 0.f, sum1 = 0.f;
#pragma unroll
    for (int nt = 0; nt < NT; ++nt) {
        const float p0 = ex2(s[nt][0] - mn0), p1 = ex2(s[nt][1] - mn0);
        const float p2 = ex2(s[nt][2] - mn1), p3 = ex2(s[nt][3] - mn1);
        sum0 += p0 + p1; sum1 += p2 + p3;
        pf[nt * 2 + 0] = pack_bf16(p0, p1);
        pf[nt * 2 + 1] = pack_bf16(p2, p3);
    }
    l_run[0] += sum0;
    l_run[1] += sum1;
    // ---- O += P V (NT/2 k-steps of 16 tokens, 16 d n-tiles): 4*NT ldmatrix.x4.trans, same ring
    {
        constexpr int L = 4 * NT;
        uint32_t fr[KV_LDSM_DEPTH][4];
        // load i -> (kk = i / 8, np = i % 8): row = tok0 + kk*16 + (lane & 7) + ((lane >> 3) & 1) * 8;
        // 16-B chunk np*2 + (lane >> 4)
        const uint32_t vb = sb + 2 * SUB + tok0 * 128 + vrow;
#define KV_V_ADDR(i) (vb + ((i) / 8) * 16 * 128 + ((((i) % 8)) >> 2) * SUB + ((vbase ^ (uint32_t)(2 * (((i) % 8) & 3))) << 4))
#pragma unroll
        for (int i = 0; i < KV_LDSM_DEPTH; ++i)
            ldmatrix_x4_trans(fr[i][0], fr[i][1], fr[i][2], fr[i][3], KV_V_ADDR(i));
#pragma unroll
        for (int i = 0; i < L; ++i) {
            const int kk = i / 8, np = i % 8;
            const uint32_t (&pa)[4] = *reinterpret_cast<const uint32_t (*)[4]>(&pf[kk * 4]);
            mma_bf16(o[2 * np], pa, fr[i % KV_LDSM_DEPTH][0], fr[i % KV_LDSM_DEPTH][1]);
            mma_bf16(o[2 * np + 1], pa, fr[i % KV_LDSM_DEPTH][2], fr[i % KV_LDSM_DEPTH][3]);
            if (i + KV_LDSM_DEPTH < L)
                ldmatrix_x4_trans(fr[i % KV_LDSM_DEPTH][0], fr[i % KV_LDSM_DEPTH][1], fr[i % KV_LDSM_DEPTH][2],
                                  fr[i % KV_LDSM_DEPTH][3], KV_V_ADDR(i + KV_LDSM_DEPTH));
        }
#undef KV_V_ADDR
    }
}

// Two query entries of a dependent stage: q = bf16(fp32(q_in) + alpha * O_prev), one rounded product
// and one rounded sum in float32, then round-to-nearest-even (reading M1).
__device__ __forceinline__ uint32_t stage_query2(uint32_t q_in, float2 o, float alpha)
{
    const float lo = __fadd_rn(__uint_as_float(q_in << 16), __fmul_rn(alpha, o.x));
    const float hi = __fadd_rn(__uint_as_float(q_in & 0xFFFF0000u), __fmul_rn(alpha, o.y));
    const uint32_t a = __float_as_uint(lo), b = __float_as_uint(hi);
    const uint32_t ra = (a + 0x7FFFu + ((a >> 16) & 1u)) >> 16;
    const uint32_t rb = (b + 0x7FFFu + ((b >> 16) & 1u)) >> 16;
    return ra | (rb << 16);
}

// ---------------------------------------------------------------------------------------
// Device-side tile planner of the request queue (cp_queue_*; the persistent
// kernel "repeatedly poll[s] per-model request queues on GPUs, select[s] the next ready batch ... and update[s]
// the batch state for the next layer").  Run by ONE warp (the planner warp of CTA 0) while the other warps of
// the grid stream KV: it waits for the host to push entry s into the mapped ring, cuts the batch into tiles with
// the same arithmetic as the host planner (plan_request_splits: a stage planned here is cut exactly like the
// same batch planned by cp_decode_attention), writes the stage's tile records, combine units and StageRec into
// the launch's work list and publishes them with a release; the producers of all CTAs acquire
// QueueState::planned_tiles before they take a tile.  Everything a stage needs is derived from device-resident
// tables (context lengths, request -> model, model shapes): the host sends request ids and a dependency only.
// ---------------------------------------------------------------------------------------
__device__ __noinline__ void queue_planner(const DecodeParams &p, const int lane)
{
    TileRec *recs = const_cast<TileRec *>(p.tile_recs);
    CombineUnit *units = const_cast<CombineUnit *>(p.cunits);
    StageRec *stages = const_cast<StageRec *>(p.stages);
    QueueState *qs = p.qstate;
    const int P = (int)p.page_tokens;
    int n_tiles = 0, n_units = 0, n_groups = 0, n_stages = 0, err = 0;
    int64_t rows = 0, ws = 0;
    for (int s = 0; s < p.q_max_stages && !err; ++s) {
        // ---- wait for entry s (system-scope acquire: the host wrote the entry, then the tail)
        int have = 0;
        if (lane == 0) {
            unsigned ns = 128;
            const unsigned long long t0 = global_timer_ns();
            while ((have = ld_acquire_sys(p.queue_tail)) <= s) {
                __nanosleep(ns);
                if (ns < 2048) ns <<= 1;
                if (global_timer_ns() - t0 > (unsigned long long)p.gate_timeout_us * 1000ull) { have = -1; break; }
            }
        }
        have = __shfl_sync(0xffffffffu, have, 0);
        if (have < 0) { err = 1; break; }
        int word = 0;
        if (lane < 16) asm volatile("ld.relaxed.sys.global.s32 %0, [%1];" : "=r"(word) : "l"(reinterpret_cast<const int32_t *>(p.queue + s) + lane) : "memory");
        const int n_req = __shfl_sync(0xffffffffu, word, 0);
        const int dep = __shfl_sync(0xffffffffu, word, 1);
        const float alpha = __int_as_float(__shfl_sync(0xffffffffu, word, 2));
        const int close = __shfl_sync(0xffffffffu, word, 3);
        if (close) break;
        if (n_req < 1 || n_req > kQueueMaxReq || dep >= s) { err = 3; break; }
        // ---- per request: model shape, pages (lane b = request b), then the splits (lane 0, sequential: <= 12 requests)
        const int my_req = __shfl_sync(0xffffffffu, word, 4 + (lane < n_req ? lane : 0));
        int my_lp = 0, my_hkv = 0, my_hpk = 0, my_hq = 0, bad = 0;
        float my_scale = 0.f;
        if (lane < n_req) {
            const int mid = my_req >= 0 ? __ldg(p.req_model + my_req) : -1;
            if (mid < 0) bad = 1;
            else {
                const DevModel m = p.models[mid];
                if (m.kind != 0 || m.d_k != KV_D || m.d_v != KV_D || m.group > 128) bad = 1;
                my_hkv = m.n_kv_heads; my_hpk = m.group; my_hq = m.n_q_heads; my_scale = m.scale_log2;
                my_lp = (__ldg(p.req_ctx + my_req) + P - 1) / P;
                if (my_lp < 1) bad = 1;
            }
        }
        if (__any_sync(0xffffffffu, bad)) { err = 3; break; }
        int my_splits = 0;
        {
            int v_lp[kQueueMaxReq], v_hkv[kQueueMaxReq], v_sp[kQueueMaxReq];
#pragma unroll
            for (int b = 0; b < kQueueMaxReq; ++b) {
                v_lp[b] = __shfl_sync(0xffffffffu, my_lp, b);
                v_hkv[b] = b < n_req ? __shfl_sync(0xffffffffu, my_hkv, b) : 0;
                if (b >= n_req) v_lp[b] = 0;
                v_sp[b] = 0;
            }
            if (lane == 0) plan_request_splits(n_req, v_lp, v_hkv, p.q_target_tiles, p.q_min_tile_pages, kMaxSplits, v_sp);
#pragma unroll
            for (int b = 0; b < kQueueMaxReq; ++b) {
                const int sp = __shfl_sync(0xffffffffu, v_sp[b], 0);
                if (lane == b) my_splits = sp;
            }
        }
        // ---- capacities
        int st_tiles = my_splits * my_hkv, st_groups = my_hkv, st_rows = my_hq;
        for (int o = 16; o > 0; o >>= 1) {
            st_tiles += __shfl_xor_sync(0xffffffffu, st_tiles, o);
            st_groups += __shfl_xor_sync(0xffffffffu, st_groups, o);
            st_rows += __shfl_xor_sync(0xffffffffu, st_rows, o);
        }
        if (n_tiles + st_tiles > p.q_max_tiles || n_groups + st_groups > p.q_max_groups) { err = 2; break; }
        // ---- emit, request by request, kv head by kv head (all lanes walk together; parameters by shuffle)
        const int cu_begin = n_units;
        int direct = 0;                  // completion signals of single-split tiles (one per padded M tile)
        int64_t row_b = 0;
        for (int b = 0; b < n_req && !err; ++b) {
            const int req = __shfl_sync(0xffffffffu, my_req, b), n_lp = __shfl_sync(0xffffffffu, my_lp, b);
            const int hkv = __shfl_sync(0xffffffffu, my_hkv, b), hpk = __shfl_sync(0xffffffffu, my_hpk, b);
            const int hq = __shfl_sync(0xffffffffu, my_hq, b), nsp = __shfl_sync(0xffffffffu, my_splits, b);
            const float scale = __shfl_sync(0xffffffffu, my_scale, b);
            int mtp = 1;
            while (mtp < (hpk + 15) / 16) mtp <<= 1;
            for (int c = 0; c < hkv && !err; ++c) {
                const int gi = n_groups++;
                const int64_t row0 = rows + row_b + (int64_t)c * hpk;
                int64_t part_off = 0;
                if (nsp > 1) {
                    part_off = ws;
                    ws += part_group_floats(hpk, nsp, KV_D);
                    if (ws > p.q_ws_floats_cap) { err = 2; break; }
                }
                // tiles: near-equal page-aligned splits, lane t writes tile t (six 16-byte stores)
                const int base = n_lp / nsp, rem = n_lp % nsp;
                for (int t0 = 0; t0 < nsp; t0 += 32) {
                    const int t = t0 + lane;
                    if (t < nsp) {
                        TileRec r;
                        r.group = gi; r.req = req; r.kv_head = c; r.n_kv_heads = hkv;
                        r.page_begin = t * base + min(t, rem); r.n_pages = base + (t < rem ? 1 : 0);
                        r.split = t; r.n_splits = nsp; r.gsize = hpk; r.n_q_heads = hq; r.scale_log2 = scale; r.pad = s;
                        r.q_off = row0 * KV_D; r.out_off = row0 * KV_D; r.lse_off = row0; r.part_off = part_off;
                        r.app_k_off = 0; r.app_v_off = 0;
#pragma unroll
                        for (int i = 0; i < 8; ++i) r.first_pid[i] = 0;
                        uint4 *dst = reinterpret_cast<uint4 *>(recs + n_tiles + t);
                        const uint4 *src = reinterpret_cast<const uint4 *>(&r);
#pragma unroll
                        for (int i = 0; i < 8; ++i) __stcg(dst + i, src[i]);
                    }
                }
                n_tiles += nsp;
                if (nsp == 1) direct += mtp;
                else {
                    // combine units: one per (head, column block), as the host planner lays them out
                    const int zl = nsp <= 8 ? 0 : (nsp <= 32 ? 3 : (nsp <= 128 ? 4 : 5));
                    const int cols = 128 >> zl, nb = KV_D / cols, nu = hpk * nb;
                    if (n_units + nu > p.q_max_units) { err = 2; break; }
                    for (int u0 = 0; u0 < nu; u0 += 32) {
                        const int u = u0 + lane;
                        if (u < nu) {
                            const int h = u / nb, c0 = (u % nb) * cols;
                            CombineUnit cu;
                            cu.part_off = part_off + part_o_off(h, 0, nsp, KV_D) + c0;
                            cu.ml_off = part_off + part_ml_off(hpk, h, 0, nsp, KV_D);
                            cu.out_off = (row0 + h) * KV_D + c0;
                            cu.lse_off = c0 == 0 ? row0 + h : -1;
                            cu.split_stride = KV_D; cu.n_splits = nsp; cu.zl_log2 = zl; cu.want = nsp * mtp;
                            cu.group = gi; cu.pad[0] = s; cu.pad[1] = 0; cu.pad[2] = 0;
                            uint4 *dst = reinterpret_cast<uint4 *>(units + n_units + u);
                            const uint4 *src = reinterpret_cast<const uint4 *>(&cu);
#pragma unroll
                            for (int i = 0; i < 4; ++i) __stcg(dst + i, src[i]);
                        }
                    }
                    n_units += nu;
                }
            }
            row_b += hq;
        }
        if (err) break;
        if (lane == 0) {
            StageRec sr;
            sr.dep = dep; sr.dep_target = dep >= 0 ? __ldcg(p.q_target + dep) : 0;
            sr.cu_begin = cu_begin; sr.cu_end = n_units;
            sr.dep_out_delta = dep >= 0 ? (__ldcg(p.q_out_base + dep) - rows) * KV_D : 0;
            sr.alpha = alpha; sr.pad = 0;
            uint4 *dst = reinterpret_cast<uint4 *>(stages + s);
            const uint4 *src = reinterpret_cast<const uint4 *>(&sr);
            __stcg(dst, src[0]);
            __stcg(dst + 1, src[1]);
            __stcg(p.q_target + s, (n_units - cu_begin) + direct);
            __stcg(p.q_out_base + s, rows);
        }
        rows += st_rows;
        n_stages = s + 1;
        // ---- publish: the stage's records happen-before the counters (cumulative release over the warp barrier)
        __syncwarp();
        if (lane == 0) {
            __threadfence();
            asm volatile("st.release.gpu.global.s32 [%0], %1;" ::"l"(&qs->planned_stages), "r"(n_stages) : "memory");
            asm volatile("st.release.gpu.global.s32 [%0], %1;" ::"l"(&qs->planned_tiles), "r"(n_tiles) : "memory");
        }
    }
    if (lane == 0) {
        qs->error = err; qs->n_units = n_units; qs->n_groups = n_groups; qs->q_rows = rows; qs->ws_floats = ws;
        __threadfence();
        asm volatile("st.release.gpu.global.s32 [%0], %1;" ::"l"(&qs->planned_stages), "r"(n_stages) : "memory");
        asm volatile("st.release.gpu.global.s32 [%0], %1;" ::"l"(&qs->closed), "r"(1) : "memory");
    }
}

// MULTI: the work list is the concatenation of several stages (cp_decode_attention_stages): a CTA
// runs its combine units of every earlier stage before it starts a tile of a later one, and a tile
// of a dependent stage waits for its predecessor's completion counter before it builds its queries
// from that stage's output.  Waits only ever target earlier entries of the list, so they terminate.
// QLEN: q_len > 1 query tokens per request (cp_decode_attention_qlen).  Row r of a group is query token
// r / g, head r % g of the kv head's g heads; its causal limit ends q_len - 1 - r / g tokens before the
// context's end.
template <int P, int MULTI, bool QLEN>      // MULTI: 0 one step, 1 host-built stage list, 2 request queue (stages planned on the device)
__global__ void __launch_bounds__(KV_THREADS + 32, 1)
cp_decode_kv_kernel(const DecodeParams p, const __grid_constant__ CUtensorMap tmap, int rows_per_page)
{
    constexpr int STAGE_BYTES = P * 4 * KV_D;
    constexpr int SUB = P * 128;                    // one swizzled sub-tile: P rows x 128 B
    constexpr int NT = P >= 32 ? 4 : 2;             // 8-token n-tiles per work unit
    constexpr int TU = 8 * NT;                      // tokens per work unit (slice)
    constexpr int SPP = P / TU;                     // slices per page
    constexpr int NS = kv_num_stages(P);

    extern __shared__ __align__(1024) uint8_t smem[];
    uint8_t *stage_base = smem;
    float *merge = reinterpret_cast<float *>(smem + (size_t)NS * STAGE_BYTES);
    uint64_t *bars = reinterpret_cast<uint64_t *>(smem + (size_t)NS * STAGE_BYTES + KV_MERGE_BYTES);
    // bars: full[NS], empty[NS], tq_full[TQ], tq_empty[TQ]; then the tile queue
    uint64_t *full_b = bars, *empty_b = bars + NS, *tqf_b = bars + 2 * NS, *tqe_b = bars + 2 * NS + KV_TQ;
    TileDesc *tq = reinterpret_cast<TileDesc *>(bars + 2 * NS + 2 * KV_TQ);

    const int tid = threadIdx.x;
    const int warp = tid >> 5;
    const int lane = tid & 31;
    if (tid == 0) {
        // full[s]: one arrive.expect_tx by the producer + the TMA transaction bytes.
        // empty[s]: EVERY consumer warp waits for every page in ring order and arrives on its
        // release, whether or not it owns a slice of the page: the barrier count is a constant
        // and no warp can run a phase ahead of a stage.
        for (int i = 0; i < NS; ++i) { mbar_init(smem_u32(full_b + i), 1); mbar_init(smem_u32(empty_b + i), KV_CWARPS); }
        for (int i = 0; i < KV_TQ; ++i) { mbar_init(smem_u32(tqf_b + i), 1); mbar_init(smem_u32(tqe_b + i), KV_CWARPS); }
        asm volatile("prefetch.tensormap [%0];" ::"l"(reinterpret_cast<uint64_t>(&tmap)) : "memory");
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
    }
    __syncthreads();
    asm volatile("griddepcontrol.wait;" ::: "memory");    // from here on: data the previous kernel may have written
    scheduler_reset_other_set(p);


    if (warp == KV_CWARPS) {
        // =========================================================== producer warp
        uint64_t policy;
        asm volatile("createpolicy.fractional.L2::evict_first.b64 %0, 1.0;" : "=l"(policy));
        uint32_t pc = 0;          // pages issued by this CTA (ring position)
        uint32_t qi = 0;          // work items pushed
        for (;;) {
            // the first tile of a CTA is static (its block index): no atomic round trip at start-up
            int work = 0;
            if (qi == 0) work = blockIdx.x;
            else {
                if (lane == 0) work = atomicAdd(p.work_counter, 1) + (int)gridDim.x;
                work = __shfl_sync(0xffffffffu, work, 0);
            }
            int item = work < p.n_tiles ? work : -1;      // tiles only; combine units are static
            int final_stages = p.n_stages;
            if constexpr (MULTI == 2) {
                // request queue: tile `work` exists once the planner (CTA 0) has published more than `work` tiles;
                // after the close marker the counts are final
                int pt = 0, cl = 0;
                if (lane == 0) {
                    unsigned ns = 64;
                    for (;;) {
                        pt = ld_acquire(&p.qstate->planned_tiles);
                        if (pt > work) break;
                        cl = ld_acquire(&p.qstate->closed);
                        if (cl) { pt = ld_acquire(&p.qstate->planned_tiles); break; }
                        __nanosleep(ns);
                        if (ns < 1024) ns <<= 1;
                    }
                    final_stages = cl ? ld_acquire(&p.qstate->planned_stages) : 0;
                }
                pt = __shfl_sync(0xffffffffu, pt, 0);
                final_stages = __shfl_sync(0xffffffffu, final_stages, 0);
                item = work < pt ? work : -1;
            }
            TileRec r;
            int ctx = 0, mt = 1;
            if (item >= 0) {
                const uint4 *src = reinterpret_cast<const uint4 *>(p.tile_recs + item);
                uint4 *dst = reinterpret_cast<uint4 *>(&r);
#pragma unroll
                for (int i = 0; i < 5; ++i) dst[i] = MULTI == 2 ? __ldcg(src + i) : __ldg(src + i);
                ctx = __ldg(p.req_ctx + r.req);
                mt = kv_mtiles(r.gsize);
            } else {
                r.group = 0; r.req = 0; r.kv_head = 0; r.n_kv_heads = 1; r.page_begin = 0; r.n_pages = 0;
                r.split = 0; r.n_splits = 1; r.gsize = 1; r.n_q_heads = 1; r.scale_log2 = 0.f;
                r.q_off = r.out_off = r.lse_off = r.part_off = 0; r.pad = 0;
            }
            if constexpr (MULTI) {
                // Admission doorbell (cp_decode_attention_stages_gated): the host -- "coarse-grained admission"
                // stays on the CPU, PAPER.md L146 -- raises *published as it admits batches; a tile is handed
                // to the consumers, and its pages are requested, only once its stage is admitted.  A poll
                // that outlasts the timeout stops gating and raises a flag instead of hanging the device.
                if (p.published != nullptr && item >= 0) {
                    // (once a poll has timed out the launch stops gating: later tiles do not wait again)
                    if (lane == 0 && ld_relaxed(p.gate_flag) == 0) {
                        unsigned ns = 256;
                        const unsigned long long t0 = global_timer_ns();
                        while (ld_acquire_sys(p.published) <= r.pad) {
                            __nanosleep(ns);
                            if (ns < 4096) ns <<= 1;
                            if (global_timer_ns() - t0 > (unsigned long long)p.gate_timeout_us * 1000ull) {
                                atomicExch(p.gate_flag, 1);
                                break;
                            }
                        }
                    }
                    __syncwarp();
                }
            }
            // push the descriptor to the tile queue
            const uint32_t qs = qi % KV_TQ;
            mbar_wait(smem_u32(tqe_b + qs), ((qi / KV_TQ) & 1) ^ 1);
            if (lane == 0) {
                TileDesc d;
                d.item = item; d.group_idx = r.group; d.page_begin = r.page_begin;
                d.npg = r.n_pages; d.split = r.split; d.n_splits = r.n_splits;
                d.ctx = ctx; d.gsize = r.gsize; d.mt = mt; d.scale_log2 = r.scale_log2;
                d.q_off = r.q_off; d.out_off = r.out_off; d.lse_off = r.lse_off; d.part_off = r.part_off;
                d.stage = item >= 0 ? r.pad : final_stages; d.hq = r.n_q_heads;
                tq[qs] = d;
                mbar_arrive(smem_u32(tqf_b + qs));     // release: consumers acquire via try_wait
            }
            ++qi;
            if (item < 0) break;

            const int npg = r.n_pages;
            const int hkv = r.n_kv_heads;
            for (int j0 = 0; j0 < npg; j0 += 32) {
                // translate up to 32 logical pages at once (step a2: one page-table entry per lane)
                int32_t pid = 0;
                if (j0 + lane < npg) pid = page_of(p, r.req, (int64_t)(r.page_begin + j0 + lane) * hkv + r.kv_head);
                const int nj = min(32, npg - j0);
                for (int j = 0; j < nj; ++j) {
                    const int32_t my = __shfl_sync(0xffffffffu, pid, j);
                    const uint32_t slot = pc % NS;
                    const uint32_t par = ((pc / NS) & 1) ^ 1;
                    mbar_wait(smem_u32(empty_b + slot), par);
                    if (elect_one()) {
                        const uint32_t fb = smem_u32(full_b + slot);
                        mbar_arrive_expect_tx(fb, STAGE_BYTES);
                        const uint32_t dst = smem_u32(stage_base + (size_t)slot * STAGE_BYTES);
                        const int row = my * rows_per_page;
                        tma_load_2d(dst, &tmap, 0, row, fb, policy);               // K, d 0..63
                        tma_load_2d(dst + SUB, &tmap, 64, row, fb, policy);        // K, d 64..127
                        tma_load_2d(dst + 2 * SUB, &tmap, 0, row + P, fb, policy); // V, d 0..63
                        tma_load_2d(dst + 3 * SUB, &tmap, 64, row + P, fb, policy);// V, d 64..127
                    }
                    ++pc;
                }
            }
        }
        // programmatic dependent launch: see cp_kernels_kvt.cu (the next kernel's set-up overlaps this one's tail;
        // said once every page of this CTA has been requested, not at the top)
        if (lane == 0) asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
    } else if (warp == KV_CWARPS + 1) {
        // =========================================================== planner warp (request queue; CTA 0 only)
        if constexpr (MULTI == 2) {
            if (blockIdx.x == 0) queue_planner(p, lane);
        }
    } else {
        // =========================================================== consumer warps
        uint32_t pc = 0;          // pages consumed by this CTA so far (ring position of tile start)
        uint32_t qi = 0;
        int cur_stage = 0;        // MULTI: stages whose combine units this CTA has run
        const int r0 = lane >> 2;             // fragment row (query head in the M tile), and r0 + 8
        const int cq = (lane & 3) * 2;        // fragment column pair
        // per-lane constants of the SWIZZLE_128B addressing (16-B chunk index ^ (row & 7), row & 7 = lane & 7)
        const uint32_t koff[2] = {(uint32_t)((lane & 7) * 128 + ((((lane >> 3)) ^ (lane & 7)) << 4)),
                                  (uint32_t)((lane & 7) * 128 + (((4 + (lane >> 3)) ^ (lane & 7)) << 4))};
        const uint32_t vrow = (uint32_t)(((lane & 7) + ((lane >> 3) & 1) * 8) * 128);
        const uint32_t vbase = (uint32_t)((lane >> 4) ^ (lane & 7));
        for (;;) {
            const uint32_t qs = qi % KV_TQ;
            mbar_wait(smem_u32(tqf_b + qs), (qi / KV_TQ) & 1);
            const TileDesc d = tq[qs];
            __syncwarp();
            if (lane == 0) mbar_arrive(smem_u32(tqe_b + qs));
            ++qi;
            if constexpr (MULTI) {
                // combine units of every stage before this tile's (all of them once the list is exhausted)
                const int upto = d.stage;           // the end marker carries the number of stages
                if (upto > cur_stage) {
                    consumer_bar();                 // the merge slots of the previous tile are free
                    for (int s = cur_stage; s < upto; ++s) {
                        const int2 cur = MULTI == 2 ? __ldcg(reinterpret_cast<const int2 *>(&p.stages[s].cu_begin))
                                                    : __ldg(reinterpret_cast<const int2 *>(&p.stages[s].cu_begin));
                        combine_units<8, true, MULTI == 2>(p, cur.x + blockIdx.x * KV_CWARPS + warp, gridDim.x * KV_CWARPS,
                                                           merge + warp * KV_COMBINE_WARP_FLOATS, lane, cur.y);
                    }
                    consumer_bar();                 // combine scratch is free before the next merge
                    cur_stage = upto;
                }
            }
            if (d.item < 0) break;
            const int mt = d.mt;
            const int NL = KV_CWARPS / mt;            // slice lanes per M tile
            const int mtile = warp % mt;
            const int plane = warp / mt;
            const int ctx = d.ctx;
            const int npg = d.npg;
            const int gsize = d.gsize;
            const float scale_log2 = d.scale_log2;
            const int h0 = mtile * 16 + r0, h1 = h0 + 8;     // heads (inside the group) of my two rows

            // ---- Q fragments (A operand, 16 heads x 128), rows beyond the group are zero
            uint32_t qf[8][4];
            int64_t row0 = h0, row1 = h1;        // row offsets (in rows of 128) of my two rows in Q / O / LSE
            int back0 = 0, back1 = 0;            // QLEN: tokens at the context's end my rows must not see
            {
                if constexpr (QLEN) {
                    const int g = d.stage;                       // heads per kv head
                    const int j0q = h0 / g, j1q = h1 / g;
                    row0 = (int64_t)j0q * d.hq + (h0 - j0q * g);
                    row1 = (int64_t)j1q * d.hq + (h1 - j1q * g);
                    back0 = h0 < gsize ? p.q_len - 1 - j0q : 0;
                    back1 = h1 < gsize ? p.q_len - 1 - j1q : 0;
                }
                const uint16_t *q0 = p.q + d.q_off + row0 * KV_D;
                const uint16_t *q1 = p.q + d.q_off + row1 * KV_D;
#pragma unroll
                for (int ks = 0; ks < 8; ++ks) {
                    const int k = ks * 16 + cq;
                    qf[ks][0] = h0 < gsize ? __ldg(reinterpret_cast<const uint32_t *>(q0 + k)) : 0u;
                    qf[ks][1] = h1 < gsize ? __ldg(reinterpret_cast<const uint32_t *>(q1 + k)) : 0u;
                    qf[ks][2] = h0 < gsize ? __ldg(reinterpret_cast<const uint32_t *>(q0 + k + 8)) : 0u;
                    qf[ks][3] = h1 < gsize ? __ldg(reinterpret_cast<const uint32_t *>(q1 + k + 8)) : 0u;
                }
                if constexpr (MULTI) {
                    const int4 s0 = MULTI == 2 ? __ldcg(reinterpret_cast<const int4 *>(p.stages + d.stage))
                                               : __ldg(reinterpret_cast<const int4 *>(p.stages + d.stage));
                    if (s0.x >= 0) {
                        // the predecessor's output is complete: all its combine units and single-split
                        // tiles have signalled (acquire; the other lanes follow through the __syncwarp)
                        if (lane == 0) wait_group(p.stage_done, s0.x, s0.y);
                        __syncwarp();
                        const int4 s1 = MULTI == 2 ? __ldcg(reinterpret_cast<const int4 *>(p.stages + d.stage) + 1)
                                                   : __ldg(reinterpret_cast<const int4 *>(p.stages + d.stage) + 1);
                        const int64_t delta = (int64_t)(uint32_t)s1.x | ((int64_t)s1.y << 32);
                        const float alpha = __int_as_float(s1.z);
                        const float *o0 = p.out + d.out_off + delta + (int64_t)h0 * KV_D;
                        const float *o1 = p.out + d.out_off + delta + (int64_t)h1 * KV_D;
#pragma unroll
                        for (int ks = 0; ks < 8; ++ks) {
                            const int k = ks * 16 + cq;
                            if (h0 < gsize) {
                                qf[ks][0] = stage_query2(qf[ks][0], __ldcg(reinterpret_cast<const float2 *>(o0 + k)), alpha);
                                qf[ks][2] = stage_query2(qf[ks][2], __ldcg(reinterpret_cast<const float2 *>(o0 + k + 8)), alpha);
                            }
                            if (h1 < gsize) {
                                qf[ks][1] = stage_query2(qf[ks][1], __ldcg(reinterpret_cast<const float2 *>(o1 + k)), alpha);
                                qf[ks][3] = stage_query2(qf[ks][3], __ldcg(reinterpret_cast<const float2 *>(o1 + k + 8)), alpha);
                            }
                        }
                    }
                }
            }
            float o[16][4];
#pragma unroll
            for (int i = 0; i < 16; ++i) { o[i][0] = o[i][1] = o[i][2] = o[i][3] = 0.f; }
            float m_run[2] = {-INFINITY, -INFINITY};
            float l_run[2] = {0.f, 0.f};              // per-thread partial row sums

            // Slices are dealt round-robin over the NL slice lanes in logical token order, so all
            // warps work on the oldest page(s) of the ring at once and a stage is released after a
            // fraction of the time one warp would need for a whole page.
            for (int j = 0; j < npg; ++j) {
                const uint32_t pidx = pc + (uint32_t)j;
                const uint32_t slot = pidx % NS;
                mbar_wait(smem_u32(full_b + slot), (pidx / NS) & 1);
                const uint32_t sb = smem_u32(stage_base + (size_t)slot * STAGE_BYTES);
                const int valid = ctx - (d.page_begin + j) * P;     // >= 1; < P only on the request's last page
#pragma unroll
                for (int s = 0; s < SPP; ++s) {
                    if (((j * SPP + s) & (NL - 1)) != plane) continue;
                    const int tok0 = s * TU;
                    if (tok0 >= valid) continue;                     // dead slice of the last page
                    if (valid < tok0 + TU) {
                        // zero the V rows of dead slots (they may hold NaN; 0 * NaN would poison O)
                        for (int i = lane; i < (tok0 + TU - valid) * 16; i += 32) {
                            const int row = valid + (i >> 4), ch = i & 15;
                            const uint32_t a = sb + 2 * SUB + (ch >> 3) * SUB + row * 128 + (((ch & 7) ^ (row & 7)) << 4);
                            asm volatile("st.shared.v4.b32 [%0], {%1,%1,%1,%1};" ::"r"(a), "r"(0u) : "memory");
                        }
                        // generic-proxy writes ordered before the next TMA write into this stage
                        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
                        __syncwarp();
                    }
                    kv_slice_unit<P, NT, QLEN>(sb, tok0, valid, qf, scale_log2, o, m_run, l_run, lane, koff, vrow, vbase, back0, back1);
                }
                __syncwarp();
                if (lane == 0) mbar_arrive(smem_u32(empty_b + slot));
            }
            pc += (uint32_t)npg;

            // ---- quad-reduce the row sums, then merge the slice lanes (fixed tree)
            l_run[0] += __shfl_xor_sync(0xffffffffu, l_run[0], 1);
            l_run[0] += __shfl_xor_sync(0xffffffffu, l_run[0], 2);
            l_run[1] += __shfl_xor_sync(0xffffffffu, l_run[1], 1);
            l_run[1] += __shfl_xor_sync(0xffffffffu, l_run[1], 2);
            for (int r = 1; r < NL; r <<= 1) {
                const bool sender = (plane % (2 * r)) == r;
                const bool receiver = (plane % (2 * r)) == 0 && plane + r < NL;
                // slot of a (sender lane, m-tile): senders in this round are lanes r, 3r, 5r, ...
                const int pair = plane / (2 * r);
                float *slotp = merge + (size_t)((pair * mt + mtile) % 4) * KV_MERGE_SLOT_FLOATS;
                if (sender) {
#pragma unroll
                    for (int i = 0; i < 16; ++i) {
                        slotp[(i * 4 + 0) * 32 + lane] = o[i][0];
                        slotp[(i * 4 + 1) * 32 + lane] = o[i][1];
                        slotp[(i * 4 + 2) * 32 + lane] = o[i][2];
                        slotp[(i * 4 + 3) * 32 + lane] = o[i][3];
                    }
                    slotp[64 * 32 + lane] = m_run[0];
                    slotp[65 * 32 + lane] = m_run[1];
                    slotp[66 * 32 + lane] = l_run[0];
                    slotp[67 * 32 + lane] = l_run[1];
                }
                consumer_bar();
                if (receiver) {
                    const float om0 = slotp[64 * 32 + lane], om1 = slotp[65 * 32 + lane];
                    const float ol0 = slotp[66 * 32 + lane], ol1 = slotp[67 * 32 + lane];
                    const float M0 = fmaxf(m_run[0], om0), M1 = fmaxf(m_run[1], om1);
                    // a lane that saw no slice has m = -inf, l = 0, O = 0: weight 0
                    const float wa0 = (m_run[0] == -INFINITY) ? 0.f : exp2f(m_run[0] - M0);
                    const float wa1 = (m_run[1] == -INFINITY) ? 0.f : exp2f(m_run[1] - M1);
                    const float wb0 = (om0 == -INFINITY) ? 0.f : exp2f(om0 - M0);
                    const float wb1 = (om1 == -INFINITY) ? 0.f : exp2f(om1 - M1);
#pragma unroll
                    for (int i = 0; i < 16; ++i) {
                        o[i][0] = o[i][0] * wa0 + slotp[(i * 4 + 0) * 32 + lane] * wb0;
                        o[i][1] = o[i][1] * wa0 + slotp[(i * 4 + 1) * 32 + lane] * wb0;
                        o[i][2] = o[i][2] * wa1 + slotp[(i * 4 + 2) * 32 + lane] * wb1;
                        o[i][3] = o[i][3] * wa1 + slotp[(i * 4 + 3) * 32 + lane] * wb1;
                    }
                    l_run[0] = l_run[0] * wa0 + ol0 * wb0;
                    l_run[1] = l_run[1] * wa1 + ol1 * wb1;
                    m_run[0] = M0; m_run[1] = M1;
                }
                consumer_bar();
            }

            // ---- publish (slice lane 0 of every M tile)
            if (plane == 0) {
                if (d.n_splits == 1) {
                    const float i0 = 1.f / l_run[0], i1 = 1.f / l_run[1];
                    float *d0 = p.out + d.out_off + row0 * KV_D + cq;
                    float *d1 = p.out + d.out_off + row1 * KV_D + cq;
#pragma unroll
                    for (int i = 0; i < 16; ++i) {
                        if (h0 < gsize) *reinterpret_cast<float2 *>(d0 + i * 8) = make_float2(o[i][0] * i0, o[i][1] * i0);
                        if (h1 < gsize) *reinterpret_cast<float2 *>(d1 + i * 8) = make_float2(o[i][2] * i1, o[i][3] * i1);
                    }
                    if ((lane & 3) == 0) {
                        if (h0 < gsize) p.lse[d.lse_off + row0] = (m_run[0] + log2f(l_run[0])) * 0.6931471805599453f;
                        if (h1 < gsize) p.lse[d.lse_off + row1] = (m_run[1] + log2f(l_run[1])) * 0.6931471805599453f;
                    }
                    if constexpr (MULTI) {          // a single-split group is complete with this tile
                        __syncwarp();
                        if (lane == 0) red_release_add(p.stage_done + (size_t)d.stage * kCounterStride, 1);
                    }
                } else {
                    float *ws = p.workspace + d.part_off;
                    float *d0 = ws + part_o_off(h0, d.split, d.n_splits, KV_D) + cq;
                    float *d1 = ws + part_o_off(h1, d.split, d.n_splits, KV_D) + cq;
#pragma unroll
                    for (int i = 0; i < 16; ++i) {
                        if (h0 < gsize) __stcg(reinterpret_cast<float2 *>(d0 + i * 8), make_float2(o[i][0], o[i][1]));
                        if (h1 < gsize) __stcg(reinterpret_cast<float2 *>(d1 + i * 8), make_float2(o[i][2], o[i][3]));
                    }
                    if ((lane & 3) == 0) {
                        if (h0 < gsize) __stcg(reinterpret_cast<float2 *>(ws + part_ml_off(gsize, h0, d.split, d.n_splits, KV_D)), make_float2(m_run[0], l_run[0]));
                        if (h1 < gsize) __stcg(reinterpret_cast<float2 *>(ws + part_ml_off(gsize, h1, d.split, d.n_splits, KV_D)), make_float2(m_run[1], l_run[1]));
                    }
                    // the warp's partial stores happen-before lane 0's gpu-scope release (cumulative
                    // over the __syncwarp), which the combine units acquire: no membar needed
                    __syncwarp();
                    if (lane == 0) red_release_add(p.group_counters + (size_t)d.group_idx * kCounterStride, 1);
                }
            }
        }
        // ---- LSE combine (step a4): no tile is left to pop; every consumer warp runs its
        // warp-sized units.  A unit only waits for tiles that are already running on some SM, so
        // the spin inside terminates.
        // Units are assigned statically (unit u -> consumer warp u mod #warps of the grid): popping
        // them from one counter would serialise thousands of same-address atomics at the L2.
        if constexpr (!MULTI)
            combine_units<8>(p, blockIdx.x * KV_CWARPS + warp, gridDim.x * KV_CWARPS, merge + warp * KV_COMBINE_WARP_FLOATS, lane);
    }
}

// ----------------------------------------------------------------------------- host side
typedef CUresult (*EncodeTiledFn)(CUtensorMap *, CUtensorMapDataType, cuuint32_t, void *, const cuuint64_t *,
                                  const cuuint64_t *, const cuuint32_t *, const cuuint32_t *,
                                  CUtensorMapInterleave, CUtensorMapSwizzle, CUtensorMapL2promotion,
                                  CUtensorMapFloatOOBfill);

static EncodeTiledFn get_encode_fn()
{
    static EncodeTiledFn fn = nullptr;
    if (fn) return fn;
    void *ptr = nullptr;
    cudaDriverEntryPointQueryResult qres;
    if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &ptr, cudaEnableDefault, &qres) != cudaSuccess ||
        qres != cudaDriverEntryPointSuccess)
        return nullptr;
    fn = reinterpret_cast<EncodeTiledFn>(ptr);
    return fn;
}

// 2-D view of the arena as rows of `row_elems` bf16; box = box_cols x box_rows, SWIZZLE_128B.
bool make_arena_tensor_map(void *out_map, const void *arena, uint64_t total_rows, uint32_t row_elems,
                           uint32_t box_cols, uint32_t box_rows)
{
    EncodeTiledFn fn = get_encode_fn();
    if (!fn) return false;
    cuuint64_t dims[2] = {row_elems, total_rows};
    cuuint64_t strides[1] = {(cuuint64_t)row_elems * 2};
    cuuint32_t box[2] = {box_cols, box_rows};
    cuuint32_t estr[2] = {1, 1};
    CUresult r = fn(reinterpret_cast<CUtensorMap *>(out_map), CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 2,
                    const_cast<void *>(arena), dims, strides, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE,
                    CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
                    CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    return r == CUDA_SUCCESS;
}


bool kv_fast_supported(int P) { return P == 16 || P == 32 || P == 64 || P == 128; }

template <int P, int MULTI, bool QLEN>
static cudaError_t launch_kv_tm(const DecodeParams &p, const CUtensorMap &tmap, int rows_per_page, int grid,
                                cudaStream_t stream)
{
    const int smem = kv_smem_bytes(P);
    static bool configured[64] = {};              // per device: the attribute belongs to the device's copy of the function
    int dev = 0;
    cudaError_t e0 = cudaGetDevice(&dev);
    if (e0 != cudaSuccess) return e0;
    if (dev < 0 || dev >= 64 || !configured[dev]) {
        cudaError_t e = cudaFuncSetAttribute(cp_decode_kv_kernel<P, MULTI, QLEN>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem);
        if (e != cudaSuccess) return e;
        if (dev >= 0 && dev < 64) configured[dev] = true;
    }
    // the request queue adds the planner warp (only CTA 0's does anything)
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3((unsigned)grid); cfg.blockDim = dim3(MULTI == 2 ? KV_THREADS + 32 : KV_THREADS); cfg.dynamicSmemBytes = (size_t)smem; cfg.stream = stream;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = attr; cfg.numAttrs = 1;
    return cudaLaunchKernelEx(&cfg, cp_decode_kv_kernel<P, MULTI, QLEN>, p, tmap, rows_per_page);
}

template <int P>
static cudaError_t launch_kv_t(const DecodeParams &p, const CUtensorMap &tmap, int rows_per_page, int grid,
                               cudaStream_t stream)
{
    if (p.queue != nullptr) return launch_kv_tm<P, 2, false>(p, tmap, rows_per_page, grid, stream);
    if (p.n_stages > 0) return launch_kv_tm<P, 1, false>(p, tmap, rows_per_page, grid, stream);
    if (p.q_len > 1) return launch_kv_tm<P, 0, true>(p, tmap, rows_per_page, grid, stream);
    return launch_kv_tm<P, 0, false>(p, tmap, rows_per_page, grid, stream);
}

cudaError_t launch_decode_kv(const DecodeParams &p, const void *tmap, int rows_per_page, int n_ctas,
                             cudaStream_t stream)
{
    const CUtensorMap &tm = *reinterpret_cast<const CUtensorMap *>(tmap);
    int grid = p.n_tiles > (p.n_combine_units + KV_CWARPS - 1) / KV_CWARPS
                   ? p.n_tiles : (p.n_combine_units + KV_CWARPS - 1) / KV_CWARPS;
    if (grid > n_ctas) grid = n_ctas;
    if (p.queue != nullptr) grid = n_ctas;          // the work is not known yet
    if (grid < 1) grid = 1;
    switch (p.page_tokens) {
    case 16: return launch_kv_t<16>(p, tm, rows_per_page, grid, stream);
    case 32: return launch_kv_t<32>(p, tm, rows_per_page, grid, stream);
    case 64: return launch_kv_t<64>(p, tm, rows_per_page, grid, stream);
    case 128: return launch_kv_t<128>(p, tm, rows_per_page, grid, stream);
    default: return cudaErrorInvalidValue;
    }
}

}  // namespace cp
