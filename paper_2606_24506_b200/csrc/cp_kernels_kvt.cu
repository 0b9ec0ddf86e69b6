// cp_kernels_kvt.cu -- the MQA / GQA fast path of libcrosspool on the 5th-generation tensor cores
// (hot-path steps a2-a6 for kind CP_KIND_KV with d_k = d_v = 128): ONE persistent launch per
// decode step, tcgen05.mma with the TOKENS on the MMA M dimension.
//
// A (request, kv head) group has g = Hq / Hkv query rows -- 8 to 32 here -- far fewer than the 128
// rows a tcgen05 tile wants, so the roles are swapped: a slice of 128 cached tokens is the M
// dimension and the group's rows (padded to N = 16 / 32) are the N dimension,
//     S^T[128 tok x N] = K_slice[128 tok x 128 d] . Q^T          8 x tcgen05.mma M128 N K16
//                        (A = the K blocks exactly as TMA lands them, K-major SWIZZLE_128B;
//                         B = the query rows, K-major SWIZZLE_128B)
//     O^T[128 d x N]  += V_slice^T[128 d x 128 tok] . P^T         8 x tcgen05.mma M128 N K16
//                        (A = the V blocks as landed, read MN-major; B = P^T written by the softmax
//                         threads as bf16, MN-major without swizzle),
// accumulators in tensor memory: two score buffers and TWO O^T buffers (4 N columns), so that the
// tile that follows starts its MMAs while the finished tile's O^T is still being written out.
// A softmax thread owns one TMEM lane = one token of the slice and N scores, one per query row.  It
// needs the row (= query head) maximum only as a REFERENCE for the exponent, not exactly: every
// thread keeps the same per-head reference m_ref[h] and computes p = 2^(s - m_ref[h]) with no
// cross-thread reduction; the reference moves (and O / l are rescaled) only when some score exceeds
// it by more than 2^8, which the 128 threads agree on with one barrier.red.or per slice (for the
// data at hand: once, on the first slice of a tile).  The row sums l[h] are per-thread partial sums
// reduced once per tile in a fixed shuffle tree, so results are deterministic.
//
// Why tcgen05 here although north_star keeps it "only on the MLA path": measured in round 1, eight
// mma.sync consumer warps sustain 3.4 TB/s-equivalent at g = 32 (cfg4) and their end-of-tile merge
// through shared memory costs ~3 us; with the tokens on M one elected thread issues 16 MMAs per 128
// tokens for ANY g <= N, and the tile result sits in ONE accumulator.
//
// Warp roles (352 threads, 1 CTA / SM):
//   warp 0      producer: pure TMA issue.  Takes tiles from the scheduler warp, translates the logical pages beyond
//               the first 32 through the page table (step a2) and streams the pages into a ring of 64 KB slice
//               stages [K d0-63 | K d64-127 | V d0-63 | V d64-127], each a [128 tok x 128 B] SWIZZLE_128B block
//               that the pages of the slice fill top to bottom.
//   warp 1      MMA issuer (one lane by elect.sync); the slices of consecutive tiles form one software
//               pipeline: S of slice j is issued before P.V of slice j - 1, across tile boundaries.
//   warps 2..5  softmax (thread = token of the slice).
//   warps 6..9  epilogue (thread = value column d): O^T from TMEM -> normalised output or split partial,
//               (m, l), release of the group's arrival counter (step a6).
//   warp 10     scheduler, the control plane (step a5): walks this CTA's static tile list, then pops the dynamic
//               one; fetches records, context lengths, first page ids; stages the query rows (cp.async); writes
//               the new K / V rows of a fused append (cp_decode_step); announces tiles up to three ahead.
//   all warps   LSE combine units after the CTA's last tile (step a4).
//
// Paper anchors: paged KV interface PAPER.md:L101,L122; KV-head-limited attention under low
// concurrency PAPER.md:L21,L57; GPU-resident persistent control PAPER.md:L146.
#include <cuda.h>
#include <cuda_runtime.h>
#include <cstdint>
#include "cp_device_common.cuh"
#include "cp_launch.h"
#include "cp_ptx.cuh"

namespace cp {

constexpr int KT_D = 128;                            // head dim (qk and v)
constexpr int KT_SLICE = 128;                        // tokens per slice = MMA M
constexpr int KT_SUBB = KT_SLICE * 128;              // one swizzled block: 128 rows x 128 B
constexpr int KT_STAGE_BYTES = 4 * KT_SUBB;          // 65536
constexpr int KT_TQ = 4;                             // tile-queue depth
constexpr int KT_WARPS = 11;
constexpr int KT_MQ = 3;                             // tile records the scheduler warp may run ahead of the producer
constexpr int KT_THREADS = 32 * KT_WARPS;
constexpr int KT_MISC_BYTES = 3072;
constexpr int KT_SMEM_LIMIT = 232448;                // 227 KB opt-in maximum per CTA
constexpr float KT_LAZY_LOG2 = 8.0f;                 // the reference moves when a score exceeds it by 2^8
constexpr int KT_NMAX = 32;

__host__ __device__ constexpr int kt_q_bytes(int N) { return 2 * N * 128; }          // one query buffer: 2 blocks [N x 128 B]
__host__ __device__ constexpr int kt_p_bytes(int N) { return (N / 8) * 2048; }       // one P^T buffer
__host__ __device__ constexpr int kt_fixed_bytes(int N) { return 2 * kt_q_bytes(N) + 2 * kt_p_bytes(N) + KT_MISC_BYTES; }
__host__ __device__ constexpr int kt_num_stages(int N) { return (KT_SMEM_LIMIT - kt_fixed_bytes(N)) / KT_STAGE_BYTES; }
__host__ __device__ constexpr int kt_smem_bytes(int N) { return kt_num_stages(N) * KT_STAGE_BYTES + kt_fixed_bytes(N); }
__host__ __device__ constexpr uint32_t kt_tmem_cols(int N) { return 4 * N <= 32 ? 32u : 4 * N <= 64 ? 64u : 4 * N <= 128 ? 128u : 4 * N <= 256 ? 256u : 512u; }

struct KtDesc {                  // what the producer hands to the other warps for one tile
    int32_t item;                // work index; < 0: no more work
    int32_t group_idx;
    int32_t n_slices;            // 128-token slices of the tile
    int32_t valid_last;          // valid tokens of the last slice (1..128)
    int32_t split, n_splits;
    int32_t gsize;               // query rows of the group
    float scale_log2;
    int32_t zl;                  // log2 of the split lanes of the group's combine units: fixes the partial layout
    int32_t q_len;               // query tokens per request (cp_decode_attention_qlen); row = (query token, head of the group)
    int32_t hpk;                 // query heads per K/V head = gsize / q_len
    int32_t n_q_heads;           // row (t, h) of the group is row t * n_q_heads + h of its request's Q / O / LSE
    int32_t rem0;                // context length - first token of the tile (q_len > 1: causal limit of the rows)
    int32_t pad;
    int64_t q_off, out_off, lse_off, part_off;
};

struct KtMeta {                  // what the scheduler warp hands to the producer for one tile
    int32_t item;                // < 0: no more work
    int32_t req, kv_head, n_kv_heads, page_begin, n_pages;
    int32_t pad[2];
    int32_t pid[8];              // the physical pages of the tile's first slice (from the tile record)
};
static_assert(sizeof(KtMeta) == 64, "KtMeta layout");

struct KtMisc {
    uint64_t full[4], empty[4];                  // slice ring: TMA -> MMA, MMA (commit) -> TMA
    uint64_t s_full[2], s_empty[2];              // score buffers in TMEM: MMA -> softmax -> MMA
    uint64_t p_full[2], p_done[2];               // P^T buffers: softmax -> MMA, MMA (commit) -> softmax
    uint64_t q_free[2];                          // query buffers: score MMAs of the tile that used it are complete
    uint64_t o_done[2];                          // O^T buffer: every value MMA of the tile is complete (MMA commit)
    uint64_t e_full[2];                          // tile's row sums / references are in red[] / mref[] (4 softmax warps)
    uint64_t o_free[2];                          // epilogue has read O^T, red[], mref[] of the tile (4 epilogue warps)
    uint64_t q_full[2];                          // query buffers: the tile's rows have landed (cp.async of the scheduler warp)
    uint64_t tq_full[KT_TQ], tq_empty[KT_TQ];    // tile descriptors: scheduler -> MMA, softmax, epilogue warps
    uint64_t meta_full[KT_MQ], meta_empty[KT_MQ];   // tile records: scheduler -> producer
    uint64_t app_done[KT_MQ];                    // the tile's LAST page may be requested (a fused append's row is in memory)
    KtDesc tq[KT_TQ];
    KtMeta meta[KT_MQ];
    uint32_t tmem_base;
    uint32_t pad[1];
    alignas(16) float redmax[4 * KT_NMAX];       // slice maxima when the reference moves: [row][warp]
    float red[2][4 * KT_NMAX];                   // per-tile row sums: [O buffer][row][warp]
    float mref[2][KT_NMAX];                      // per-tile exponent reference (log2 units): [O buffer][row]
};
static_assert(sizeof(KtMisc) <= KT_MISC_BYTES, "KtMisc must fit its reserved block");

__device__ __forceinline__ bool bar_red_or_softmax(bool pred)       // barrier 2, the 128 softmax threads
{
    uint32_t r;
    asm volatile("{\n\t.reg .pred p, q;\n\tsetp.ne.u32 q, %1, 0;\n\tbarrier.cta.red.or.pred p, 2, 128, q;\n\t"
                 "selp.u32 %0, 1, 0, p;\n\t}" : "=r"(r) : "r"((uint32_t)pred) : "memory");
    return r != 0;
}
__device__ __forceinline__ void bar_sync_softmax() { asm volatile("bar.sync 2, 128;" ::: "memory"); }
__device__ __forceinline__ void bar_sync_combine() { asm volatile("bar.sync 3, 352;" ::: "memory"); }

__device__ __forceinline__ void kt_stamp(const DecodeParams &p, int k)
{
    if (p.timeline) p.timeline[(size_t)blockIdx.x * kTimelineSlots + k] = global_timer_ns();
}

// Factor that moves an accumulator from exponent reference m_old to m_new >= m_old (log2 units).  A row that has seen
// no token yet has m_old = -inf and an accumulator of 0: the factor is 0; if it still sees none (q_len > 1: the whole
// slice is behind the row's causal limit) m_new is -inf too and the factor must not be 2^(NaN).
template <bool QL>
__device__ __forceinline__ float kt_rescale(float m_old, float m_new)
{
    return QL && m_new == -INFINITY ? 0.f : ex2_ftz(m_old - m_new);
}

struct OpAdd { __device__ __forceinline__ float operator()(float a, float b) const { return a + b; } };
struct OpMax { __device__ __forceinline__ float operator()(float a, float b) const { return fmaxf(a, b); } };

// Column reduction of a [32 lanes][CN] register tile over the warp's lanes in a fixed butterfly
// (recursive halving: CN - 1 + (CN < 32 ? 16 : 0) shuffles): afterwards lane L holds in v[0] the
// reduction of column (L mod CN).  The order of the operations depends on nothing but the lane
// numbers => deterministic.
template <int CN, class Op>
__device__ __forceinline__ float col_reduce(float (&v)[CN], const int lane, Op op)
{
    static_assert(CN == 16 || CN == 32, "column blocks of 16 or 32");
    if (CN == 16) {
#pragma unroll
        for (int i = 0; i < 16; ++i) v[i] = op(v[i], __shfl_xor_sync(0xffffffffu, v[i], 16));
    }
#pragma unroll
    for (int off = CN / 2; off >= 1; off >>= 1) {
        const bool up = (lane & off) != 0;
#pragma unroll
        for (int i = 0; i < off; ++i) {
            const float send = up ? v[i] : v[i + off];
            const float keep = up ? v[i + off] : v[i];
            v[i] = op(keep, __shfl_xor_sync(0xffffffffu, send, off));
        }
    }
    return v[0];
}

__device__ __forceinline__ TileRec load_tile_rec(const TileRec *recs, int item)
{
    TileRec r;
    const uint4 *src = reinterpret_cast<const uint4 *>(recs + item);
    uint4 *dst = reinterpret_cast<uint4 *>(&r);
#pragma unroll
    for (int i = 0; i < 8; ++i) dst[i] = __ldg(src + i);
    return r;
}

// ---------------------------------------------------------------------------------------
// LSE combine, kvt flavour (step a4).  Same arithmetic and the same fixed summation order as
// combine_units() of cp_device_common.cuh, restructured for latency -- it is the tail of the
// kernel: (1) ONE warp per CTA polls the arrival counters of the round's units (lane i for
// unit i; a few hundred pollers on one L2 line delay the very arrivals they wait for) and the
// CTA's warps pass a named barrier; (2) a lane loads the (m, l) pairs AND the O rows of its own
// splits z, z + ZL, ... in ONE round trip and needs no shared memory: weights are computed
// per lane, maxima and sums go through shuffles over the split-lane bits.
// ---------------------------------------------------------------------------------------
template <int KMAX>
__device__ __forceinline__ void combine_one_unit(const DecodeParams &p, const CombineUnit &cu, const int lane)
{
    const int ns = cu.n_splits;
    const int zl = cu.zl_log2;
    const int ZL = 1 << zl, CQ = 32 >> zl;
    const int z = lane >> (5 - zl), cq = lane & (CQ - 1);
    const float2 *mlp = reinterpret_cast<const float2 *>(p.workspace + cu.ml_off);
    const float *src = p.workspace + cu.part_off + cq * 4;
    const int ss = cu.split_stride;
    float2 ml[KMAX];
    float4 v[KMAX];
#pragma unroll
    for (int k = 0; k < KMAX; ++k) {
        const int s = z + k * ZL;
        ml[k] = make_float2(-INFINITY, 0.f);
        v[k] = make_float4(0.f, 0.f, 0.f, 0.f);
        if (s < ns) {
            // plain (weak) loads: strong gpu-scope loads complete one after the other (measured: 16 of them
            // take 1.5-2.4 us, 16 weak ones one L2 latency); the acquire fence of kt_combine orders them
            ml[k] = mlp[s];
            v[k] = *reinterpret_cast<const float4 *>(src + (size_t)s * ss);
        }
    }
    float M = -INFINITY;
#pragma unroll
    for (int k = 0; k < KMAX; ++k) M = fmaxf(M, ml[k].x);
    for (int o = CQ; o < 32; o <<= 1) M = fmaxf(M, __shfl_xor_sync(0xffffffffu, M, o));
    if (threadIdx.x == 0) kt_stamp(p, 13);
    float L = 0.f;
    float4 acc = make_float4(0.f, 0.f, 0.f, 0.f);
#pragma unroll
    for (int k = 0; k < KMAX; ++k) {
        const float w = ex2_ftz(ml[k].x - M);          // 0 for absent splits (m = -inf)
        L += w * ml[k].y;
        acc.x += w * v[k].x; acc.y += w * v[k].y; acc.z += w * v[k].z; acc.w += w * v[k].w;
    }
    for (int o = CQ; o < 32; o <<= 1) {                // warp-uniform trip count
        L += __shfl_xor_sync(0xffffffffu, L, o);
        acc.x += __shfl_xor_sync(0xffffffffu, acc.x, o);
        acc.y += __shfl_xor_sync(0xffffffffu, acc.y, o);
        acc.z += __shfl_xor_sync(0xffffffffu, acc.z, o);
        acc.w += __shfl_xor_sync(0xffffffffu, acc.w, o);
    }
    if (z == 0) {
        const float invL = 1.0f / L;
        *reinterpret_cast<float4 *>(p.out + cu.out_off + cq * 4) =
            make_float4(acc.x * invL, acc.y * invL, acc.z * invL, acc.w * invL);
    }
    if (cu.lse_off >= 0 && lane == 0) p.lse[cu.lse_off] = (M + log2f(L)) * 0.6931471805599453f;
}

// More than KMAX splits per lane: two passes (maximum, then weights and sums), same order.
__device__ __noinline__ void combine_one_unit_long(const DecodeParams &p, const CombineUnit &cu, const int lane)
{
    const int ns = cu.n_splits;
    const int zl = cu.zl_log2;
    const int ZL = 1 << zl, CQ = 32 >> zl;
    const int z = lane >> (5 - zl), cq = lane & (CQ - 1);
    const float2 *mlp = reinterpret_cast<const float2 *>(p.workspace + cu.ml_off);
    const float *src = p.workspace + cu.part_off + cq * 4;
    const int ss = cu.split_stride;
    float M = -INFINITY;
    for (int s = z; s < ns; s += ZL) M = fmaxf(M, mlp[s].x);
    for (int o = CQ; o < 32; o <<= 1) M = fmaxf(M, __shfl_xor_sync(0xffffffffu, M, o));
    float L = 0.f;
    float4 acc = make_float4(0.f, 0.f, 0.f, 0.f);
#pragma unroll 4
    for (int s = z; s < ns; s += ZL) {
        const float2 ml = mlp[s];
        const float4 v = *reinterpret_cast<const float4 *>(src + (size_t)s * ss);
        const float w = ex2_ftz(ml.x - M);
        L += w * ml.y;
        acc.x += w * v.x; acc.y += w * v.y; acc.z += w * v.z; acc.w += w * v.w;
    }
    for (int o = CQ; o < 32; o <<= 1) {
        L += __shfl_xor_sync(0xffffffffu, L, o);
        acc.x += __shfl_xor_sync(0xffffffffu, acc.x, o);
        acc.y += __shfl_xor_sync(0xffffffffu, acc.y, o);
        acc.z += __shfl_xor_sync(0xffffffffu, acc.z, o);
        acc.w += __shfl_xor_sync(0xffffffffu, acc.w, o);
    }
    if (z == 0) {
        const float invL = 1.0f / L;
        *reinterpret_cast<float4 *>(p.out + cu.out_off + cq * 4) =
            make_float4(acc.x * invL, acc.y * invL, acc.z * invL, acc.w * invL);
    }
    if (cu.lse_off >= 0 && lane == 0) p.lse[cu.lse_off] = (M + log2f(L)) * 0.6931471805599453f;
}

// Called by ALL threads of the CTA (named barrier 3).  Round r of CTA b holds the KT_WARPS consecutive
// units (r * gridDim.x + b) * KT_WARPS + warp; units are sorted by group, so a round polls one or two
// counters.  A unit only waits for tiles that are already running on some SM (every CTA reaches this
// point only after the tile lists are exhausted), so the polling terminates.
__device__ __forceinline__ void kt_combine(const DecodeParams &p, const int warp, const int lane)
{
    const int n = p.n_combine_units;
    for (int base = blockIdx.x * KT_WARPS; base < n; base += gridDim.x * KT_WARPS) {
        const int u = base + warp;
        CombineUnit cu;
        if (u < n) cu = load_combine_unit(p.cunits, u);
        if (warp == 0) {
            const int32_t *ctr = nullptr;
            int want = 0;
            if (lane < KT_WARPS && base + lane < n) {
                const int4 a = __ldg(reinterpret_cast<const int4 *>(&p.cunits[base + lane].split_stride));   // stride, n_splits, zl, want
                const int grp = __ldg(&p.cunits[base + lane].group);
                want = a.w;
                ctr = p.group_counters + (size_t)grp * kCounterStride;
            }
            // Relaxed gpu-scope polling, then ONE acquire fence (an acquire load would invalidate the L1 on every
            // iteration): the writers' release (stores, fence, red) and this fence order the partials before
            // the plain loads that follow the CTA barrier below.
            for (;;) {
                const bool ok = ctr == nullptr || ld_relaxed(ctr) >= want;
                if (__all_sync(0xffffffffu, ok)) break;
                __nanosleep(100);
            }
            __threadfence();
            if (lane == 0) kt_stamp(p, 12);
        }
        bar_sync_combine();
        if (u < n) {
            const int per_lane = (cu.n_splits + (1 << cu.zl_log2) - 1) >> cu.zl_log2;
            if (per_lane <= 8) combine_one_unit<8>(p, cu, lane);
            else combine_one_unit_long(p, cu, lane);
        }
    }
}

// QL: the instantiation for q_len > 1 (cp_decode_attention_qlen); the q_len = 1 instantiations carry none of its
// code -- a cold step fetches its instructions from HBM, and every line on the way to the first MMA counts.
template <int N, bool QL>
__global__ void __launch_bounds__(KT_THREADS, 1)
cp_decode_kvt_kernel(const DecodeParams p, const __grid_constant__ CUtensorMap tmap, int rows_per_page)
{
    constexpr int NS = kt_num_stages(N);
    constexpr int CN = N >= 32 ? 32 : 16;            // column block of the reductions
    constexpr int NB = N / CN;
    static_assert(NS >= 2 && NS <= 4, "slice ring depth");
    static_assert(N % 16 == 0 && N >= 16 && N <= KT_NMAX, "N = padded query rows of a group");

    extern __shared__ __align__(1024) uint8_t smem[];
    const uint32_t st_base = smem_u32(smem);
    const uint32_t q_base = st_base + NS * KT_STAGE_BYTES;
    const uint32_t p_base = q_base + 2 * kt_q_bytes(N);
    KtMisc *mi = reinterpret_cast<KtMisc *>(smem + NS * KT_STAGE_BYTES + 2 * kt_q_bytes(N) + 2 * kt_p_bytes(N));

    const int tid = threadIdx.x;
    const int warp = tid >> 5;
    const int lane = tid & 31;
    const int P = (int)p.page_tokens;
    const int pps = KT_SLICE / P;                    // pages per slice

    // the scheduler's first tile record is requested before anything else: its latency (the L2 is cold
    // at the start of a step) runs under the barrier / tensor-memory set-up
    TileRec r_next;
    bool has_next = false;
    if (warp == KT_WARPS - 1) {
        has_next = (int)blockIdx.x < p.n_static_slots;
        if (has_next) r_next = load_tile_rec(p.tile_recs, blockIdx.x);
    }
    if (tid == 0) {
        kt_stamp(p, 0);
        if (p.timeline) {
            uint32_t smid;
            asm volatile("mov.u32 %0, %%smid;" : "=r"(smid));
            p.timeline[(size_t)blockIdx.x * kTimelineSlots + 8] = smid;
        }
    }
    if (tid == 32) {
        for (int i = 0; i < NS; ++i) { mbar_init(smem_u32(&mi->full[i]), 1); mbar_init(smem_u32(&mi->empty[i]), 1); }
        for (int i = 0; i < 2; ++i) {
            mbar_init(smem_u32(&mi->s_full[i]), 1); mbar_init(smem_u32(&mi->s_empty[i]), 4);
            mbar_init(smem_u32(&mi->p_full[i]), 4); mbar_init(smem_u32(&mi->p_done[i]), 1);
            mbar_init(smem_u32(&mi->q_free[i]), 1); mbar_init(smem_u32(&mi->q_full[i]), 32);
            mbar_init(smem_u32(&mi->o_done[i]), 1); mbar_init(smem_u32(&mi->e_full[i]), 4); mbar_init(smem_u32(&mi->o_free[i]), 4);
        }
        for (int i = 0; i < KT_TQ; ++i) { mbar_init(smem_u32(&mi->tq_full[i]), 1); mbar_init(smem_u32(&mi->tq_empty[i]), 9); }
        for (int i = 0; i < KT_MQ; ++i) {
            mbar_init(smem_u32(&mi->meta_full[i]), 1); mbar_init(smem_u32(&mi->meta_empty[i]), 1);
            mbar_init(smem_u32(&mi->app_done[i]), 1);
        }
        asm volatile("prefetch.tensormap [%0];" ::"l"(reinterpret_cast<uint64_t>(&tmap)) : "memory");
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
        fence_proxy_async();
    }
    if (warp == 2) tmem_alloc(smem_u32(&mi->tmem_base), kt_tmem_cols(N));
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    const uint32_t tmem = mi->tmem_base;
    // Programmatic dependent launch: everything above (and the scheduler's first record, part of a plan uploaded
    // before the previous kernel even started) ran while the previous kernel of the stream was still finishing, on
    // the SMs its CTAs had already left.  From here on this launch touches what that kernel may have written
    // (queries, the arena of a fused append, counters, partials), so it waits for its completion.
    asm volatile("griddepcontrol.wait;" ::: "memory");
    if (tid == 0) kt_stamp(p, 14);

    if (warp == 0) {
        // =========================================================== producer warp: pure TMA issue
        uint64_t policy;
        asm volatile("createpolicy.fractional.L2::evict_first.b64 %0, 1.0;" : "=l"(policy));
        uint32_t gs = 0;          // slices issued by this CTA (ring position)
        uint32_t ti = 0;          // tiles taken from the scheduler
        for (;;) {
            const uint32_t ms = ti % KT_MQ;
            mbar_wait(smem_u32(&mi->meta_full[ms]), (ti / KT_MQ) & 1);
            const KtMeta *mt = &mi->meta[ms];
            const int item = mt->item;
            if (item < 0) break;
            if (lane == 0 && ti == 0) kt_stamp(p, 1);
            const int req = mt->req, hkv = mt->n_kv_heads, kvh = mt->kv_head, pb = mt->page_begin, npg = mt->n_pages;
            const int nf = min(pps, npg);                    // pages of the first slice: ids came with the tile record
            int32_t pid = lane < 8 ? mt->pid[lane] : 0;
            const uint32_t tph = (ti / KT_MQ) & 1;          // phase of this tile's use of slot ms (the slot is given back when
            ++ti;                                            // the tile's last page is out: app_done[ms] must not lap this warp)
            // translation of the pages behind them (step a2: one page-table entry per lane, 32 at a time) is
            // requested now -- it travels while the first slice is issued -- and one batch ahead from then on
            int32_t pid_nx = 0;
            if (nf + lane < npg) pid_nx = page_of(p, req, (int64_t)(pb + nf + lane) * hkv + kvh);
            for (int j0 = 0; j0 < npg;) {
                const int nj = j0 == 0 ? nf : min(32, npg - j0);
                for (int j = 0; j < nj; ++j) {
                    const int32_t my = __shfl_sync(0xffffffffu, pid, j);
                    const int jj = j0 + j;
                    const int pg = jj % pps;                 // position of the page inside its slice
                    const uint32_t slot = gs % NS;
                    if (pg == 0) mbar_wait(smem_u32(&mi->empty[slot]), ((gs / NS) & 1) ^ 1);
                    // the tile's last page is where a fused append writes: everything before it streams while the scheduler
                    // warp fetches and stores the row (non-append tiles: the barrier is complete at the hand-over)
                    if (jj == npg - 1) mbar_wait(smem_u32(&mi->app_done[ms]), tph);
                    if (elect_one()) {
                        const uint32_t fb = smem_u32(&mi->full[slot]);
                        if (pg == 0) mbar_arrive_expect_tx(fb, (uint32_t)min(pps, npg - jj) * (uint32_t)P * 512u);
                        const uint32_t dst = st_base + slot * KT_STAGE_BYTES + (uint32_t)pg * (uint32_t)P * 128u;
                        const int row = my * rows_per_page;
                        tma_load_2d(dst, &tmap, 0, row, fb, policy);                    // K, d 0..63
                        tma_load_2d(dst + KT_SUBB, &tmap, 64, row, fb, policy);         // K, d 64..127
                        tma_load_2d(dst + 2 * KT_SUBB, &tmap, 0, row + P, fb, policy);  // V, d 0..63
                        tma_load_2d(dst + 3 * KT_SUBB, &tmap, 64, row + P, fb, policy); // V, d 64..127
                        if (gs == 0 && pg == 0) kt_stamp(p, 9);
                    }
                    if (pg == pps - 1 || jj == npg - 1) {
                        ++gs;
                        // Cold start: after its very first slice the producer waits until the scheduler has announced
                        // the tile, i.e. until the context length (and, requested with it, the query rows) has come
                        // back.  Measured: otherwise 148 SMs put a whole ring (28 MB) in front of those two small loads
                        // whenever they lose the race by a few hundred ns, the MMA warp starts 5-8 us late and the
                        // step takes 37 instead of 31 us (cfg4).  (tq slot 0 is in its first phase for as long as the
                        // producer is on its first tile: the scheduler runs at most KT_MQ < KT_TQ tiles ahead.)
                        if (gs == 1) mbar_wait(smem_u32(&mi->tq_full[0]), 0);
                    }
                }
                j0 += nj;
                pid = pid_nx;
                pid_nx = 0;
                if (j0 + 32 + lane < npg) pid_nx = page_of(p, req, (int64_t)(pb + j0 + 32 + lane) * hkv + kvh);
            }
            __syncwarp();
            if (lane == 0) mbar_arrive(smem_u32(&mi->meta_empty[ms]));
        }
        if (lane == 0) {
            // The next kernel of the stream, if it was launched as a programmatic dependent, may now take the SMs this
            // grid's CTAs leave as they leave them (it waits for this grid's completion before it reads anything of
            // ours).  Said here, with every slice of this CTA requested, not at the top of the kernel: measured, the
            // instruction at the top delays the first slices of a cold start by 1.4 us (cfg4 32.0 vs 31.2 us).
            asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
            kt_stamp(p, 3);
            if (p.timeline) p.timeline[(size_t)blockIdx.x * kTimelineSlots + 11] = (unsigned long long)ti;
        }
    } else if (warp == KT_WARPS - 1) {
        // =========================================================== scheduler warp (step a5): the control plane.
        // Walks this CTA's static tile list, then pops the dynamic one; for every tile it fetches the record,
        // the context length and the first 32 page ids, stages the query rows in shared memory (cp.async) and
        // hands the tile to the producer (meta ring) and to the MMA / softmax / epilogue warps (tile queue),
        // up to KT_MQ tiles ahead of the producer -- a dependent global load takes microseconds while 148 SMs
        // stream at full rate, and none of them is on the producer's path.
        int item = has_next ? (int)blockIdx.x : -3;          // -3: no static slot at all, start with the dynamic list
        TileRec r = r_next;
        bool in_static = true;
        uint32_t ti = 0;
        bool have_pre = false;                               // the tile's context length / append operands were requested a tile ago
        int ctx_pre = 0;
        int32_t pid_pre = 0;
        uint4 row_pre = make_uint4(0u, 0u, 0u, 0u);
        for (;;) {
            if (item >= 0 && r.n_pages == 0) item = -2;      // empty static slot of this CTA: skip, go dynamic
            // ---- the tile after this one: the next static slot of this CTA, else a pop from the dynamic list
            // (the pop's result is looked at only after this tile's own loads have been issued)
            int nx_raw = -1;
            bool nx_pending = false;
            if (item != -1) {
                if (in_static && item >= 0 && (r.pad & 1)) nx_raw = r.next;
                else {
                    in_static = false;
                    if (lane == 0) nx_raw = atomicAdd(p.work_counter, 1) + p.n_static_slots;
                    nx_pending = true;
                }
            }
            int item_next = -1;
            auto resolve_next = [&]() {
                int nx = nx_raw;
                if (nx_pending) {
                    nx = __shfl_sync(0xffffffffu, nx_raw, 0);
                    if (nx >= p.n_tiles) nx = -1;
                }
                item_next = nx;
                if (nx >= 0) r_next = load_tile_rec(p.tile_recs, nx);
            };
            if (item <= -2) { resolve_next(); item = item_next; r = r_next; continue; }
            const uint32_t ms = ti % KT_MQ, qs = ti % KT_TQ;
            if (item == -1) {
                // ---- no more work: the end marker goes through both queues
                mbar_wait(smem_u32(&mi->meta_empty[ms]), ((ti / KT_MQ) & 1) ^ 1);
                mbar_wait(smem_u32(&mi->tq_empty[qs]), ((ti / KT_TQ) & 1) ^ 1);
                if (lane == 0) {
                    mi->meta[ms].item = -1;
                    mi->tq[qs].item = -1;
                    mbar_arrive(smem_u32(&mi->meta_full[ms]));
                    mbar_arrive(smem_u32(&mi->tq_full[qs]));
                }
                break;
            }
            // ---- (the ids of the first slice's pages came with the record; the producer translates the rest itself)
            const bool app = p.app_k != nullptr && (r.pad & 2);
            const int hpk = QL ? r.gsize / p.q_len : r.gsize;    // query heads per K/V head
            auto hand_to_producer = [&]() {
                mbar_wait(smem_u32(&mi->meta_empty[ms]), ((ti / KT_MQ) & 1) ^ 1);
                KtMeta *mt = &mi->meta[ms];
                if (lane < 8) mt->pid[lane] = r.first_pid[lane];
                if (lane == 0) {
                    mt->item = item; mt->req = r.req; mt->kv_head = r.kv_head; mt->n_kv_heads = r.n_kv_heads;
                    mt->page_begin = r.page_begin; mt->n_pages = r.n_pages;
                }
                __syncwarp();
                if (lane == 0) mbar_arrive(smem_u32(&mi->meta_full[ms]));   // release: the producer acquires via try_wait
            };
            if (lane == 0 && ti == 0) kt_stamp(p, 15);
            // The producer gets the tile as soon as the record is there (the first slice's page ids came with it).  A tile
            // that writes a fused append's row streams too: only its LAST page -- where the row goes -- waits (app_done).
            hand_to_producer();
            if (!app && lane == 0) mbar_arrive(smem_u32(&mi->app_done[ms]));
            // ---- one round trip: the context length (it decides only how many tokens of the tile's LAST slice are
            // valid: every planned page holds a valid token, contexts never shrink under a plan), the query rows
            // and, for a fused append, the new row and its page.  Volatile asm: issued here, not sunk to first use.
            // (Requested one tile AHEAD where there was a tile before this one, see the end of the loop: a list of short
            // tiles that all write an append row is otherwise bound by this warp -- round trip, store, fence: ~2 us per
            // tile against 2.6 us of streaming for two slices -- and cfg5's fused step ended 4 us late.)
            int ctx;
            if (have_pre) ctx = ctx_pre;
            else asm volatile("ld.global.nc.s32 %0, [%1];" : "=r"(ctx) : "l"(p.req_ctx + r.req));
            ctx += p.ctx_add;                    // a fused step reads the table of the step before (see req_ctx_next)
            // ---- fused append (cp_decode_step): the tile that holds its group's last page writes the
            // new token's K and V rows (position ctx - 1) before the producer may request that page (app_done), i.e. before
            // the page is requested.  Source row and the page's id travel in the same round trip.
            uint4 app_row = make_uint4(0u, 0u, 0u, 0u);
            int32_t app_pid = 0;
            if (app && have_pre) { app_row = row_pre; app_pid = pid_pre; }
            else if (app) {
                const uint16_t *src = lane < 16 ? p.app_k + r.app_k_off + lane * 8 : p.app_v + r.app_v_off + (lane - 16) * 8;
                asm volatile("ld.global.nc.v4.u32 {%0,%1,%2,%3}, [%4];" : "=r"(app_row.x), "=r"(app_row.y), "=r"(app_row.z), "=r"(app_row.w) : "l"(src));
                const int64_t idx = (int64_t)(r.page_begin + r.n_pages - 1) * r.n_kv_heads + r.kv_head;
                if (p.slot_pages > 0) app_pid = r.req * p.slot_pages + (int32_t)idx;
                else asm volatile("ld.global.nc.s32 %0, [%1];" : "=r"(app_pid) : "l"(p.page_table + (int64_t)r.req * p.max_ppr + idx));
            }
            if (app) {
                // the row goes in and the producer gets the tile BEFORE this warp waits for a free query buffer below:
                // with lists of short tiles that wait is what bounds the warp's lead over the producer
                const int slot = (ctx - 1) % P;
                uint8_t *dst = const_cast<uint8_t *>(p.arena) + (size_t)app_pid * p.page_bytes + (size_t)slot * (KT_D * 2) +
                               (lane < 16 ? (size_t)lane * 16 : (size_t)P * (KT_D * 2) + (size_t)(lane - 16) * 16);
                *reinterpret_cast<uint4 *>(dst) = app_row;
                // the row is read by TMA (async proxy) that another thread issues after the hand-over below
                __threadfence();
                fence_proxy_async_all();
                __syncwarp();
                if (lane == 0) mbar_arrive(smem_u32(&mi->app_done[ms]));      // release: the producer acquires via try_wait
            }
            // ---- the tile's query rows -> buffer (ti & 1), asynchronously: two K-major [N x 64] blocks, 128-byte
            // swizzle (16-B chunk index ^ (row & 7)); rows beyond the group are zero-filled.  The buffer is free
            // once the score MMAs of tile ti - 2 are complete; q_full counts the 32 lanes' copies.
            if (ti >= 2) mbar_wait(smem_u32(&mi->q_free[ti & 1]), ((ti >> 1) - 1) & 1);
            {
                const uint4 *qg = reinterpret_cast<const uint4 *>(p.q + r.q_off);
                const uint32_t qb = q_base + (ti & 1) * kt_q_bytes(N);
#pragma unroll
                for (int k = 0; k < N / 2; ++k) {
                    const int id = lane + 32 * k;
                    const int row = id >> 4, ch = id & 15;
                    const uint32_t a = qb + (ch >> 3) * (N * 128) + row * 128 + (((ch & 7) ^ (row & 7)) << 4);
                    const uint32_t nbytes = row < r.gsize ? 16u : 0u;
                    // q_len > 1: row (t, h) of the group (token-major) is row t * Hq + h of the request's queries
                    int src = row < r.gsize ? id : 0;
                    if (QL && row < r.gsize) src = ((row / hpk) * r.n_q_heads + row % hpk) * 16 + ch;
                    asm volatile("cp.async.cg.shared.global [%0], [%1], 16, %2;" ::"r"(a), "l"(qg + src), "r"(nbytes) : "memory");
                }
                asm volatile("cp.async.mbarrier.arrive.noinc.shared::cta.b64 [%0];" ::"r"(smem_u32(&mi->q_full[ti & 1])) : "memory");
            }
            resolve_next();
            mbar_wait(smem_u32(&mi->tq_empty[qs]), ((ti / KT_TQ) & 1) ^ 1);
            if (lane == 0) {
                const int t_begin = r.page_begin * P;
                const int t_end = min((r.page_begin + r.n_pages) * P, ctx);
                const int n_slices = (t_end - t_begin + KT_SLICE - 1) / KT_SLICE;
                KtDesc d;
                d.item = item; d.group_idx = r.group; d.n_slices = n_slices;
                d.valid_last = t_end - t_begin - (n_slices - 1) * KT_SLICE;
                d.split = r.split; d.n_splits = r.n_splits; d.gsize = r.gsize; d.scale_log2 = r.scale_log2;
                d.zl = (r.pad >> 8) & 0xff; d.pad = 0;
                d.q_len = p.q_len; d.hpk = hpk; d.n_q_heads = r.n_q_heads; d.rem0 = ctx - t_begin;
                d.q_off = r.q_off; d.out_off = r.out_off; d.lse_off = r.lse_off; d.part_off = r.part_off;
                mi->tq[qs] = d;
                mbar_arrive(smem_u32(&mi->tq_full[qs]));     // release: the consumers acquire via try_wait
            }
            __syncwarp();
            ++ti;
            // ---- the NEXT tile's context length (and append operands) are requested now: they travel while this warp
            // waits for queue slots, and the next round starts with them in registers
            have_pre = false;
            if (item_next >= 0 && r_next.n_pages > 0) {
                asm volatile("ld.global.nc.s32 %0, [%1];" : "=r"(ctx_pre) : "l"(p.req_ctx + r_next.req));
                if (p.app_k != nullptr && (r_next.pad & 2)) {
                    const uint16_t *src = lane < 16 ? p.app_k + r_next.app_k_off + lane * 8 : p.app_v + r_next.app_v_off + (lane - 16) * 8;
                    asm volatile("ld.global.nc.v4.u32 {%0,%1,%2,%3}, [%4];" : "=r"(row_pre.x), "=r"(row_pre.y), "=r"(row_pre.z), "=r"(row_pre.w) : "l"(src));
                    const int64_t idx = (int64_t)(r_next.page_begin + r_next.n_pages - 1) * r_next.n_kv_heads + r_next.kv_head;
                    if (p.slot_pages > 0) pid_pre = r_next.req * p.slot_pages + (int32_t)idx;
                    else asm volatile("ld.global.nc.s32 %0, [%1];" : "=r"(pid_pre) : "l"(p.page_table + (int64_t)r_next.req * p.max_ppr + idx));
                }
                have_pre = true;
            }
            item = item_next; r = r_next;
        }
    } else if (warp == 1) {
        // =========================================================== MMA issuer warp
        constexpr uint32_t IDESC_S = umma_idesc_bf16(KT_SLICE, N, 0, 0);      // K (K-major) x Q^T (K-major)
        constexpr uint32_t IDESC_PV = umma_idesc_bf16(KT_SLICE, N, 1, 1);     // V^T (MN-major) x P^T (MN-major)
        uint32_t gs = 0, qi = 0, tc = 0;
        // the value MMAs of the slice issued last, not yet issued themselves (software pipeline across tiles)
        bool pend = false;
        uint32_t pe_g = 0, pe_tc = 0;
        int pe_ksteps = 0;
        bool pe_first = false, pe_last = false;
        auto issue_pv = [&]() {
            // ---- O^T += V^T P^T of slice pe_g, 16 tokens per MMA; a tile's last slice stops after its last valid 16
            const uint32_t slot = pe_g % NS, b = pe_g & 1, ob = pe_tc & 1;
            mbar_wait(smem_u32(&mi->p_full[b]), (pe_g >> 1) & 1);
            if (pe_first && pe_tc >= 2) mbar_wait(smem_u32(&mi->o_free[ob]), ((pe_tc >> 1) - 1) & 1);   // epilogue of tile tc - 2
            tc_fence_after();
            if (elect_one()) {
                const uint32_t v0 = st_base + slot * KT_STAGE_BYTES + 2 * KT_SUBB;
                const uint32_t pb = p_base + b * kt_p_bytes(N);
                for (int k = 0; k < pe_ksteps; ++k) {
                    // V: 64-column blocks KT_SUBB apart (LBO), 8-token groups 1024 B apart (SBO)
                    const uint64_t ad = umma_smem_desc(v0 + k * 2048, KT_SUBB, 1024, 2);
                    // P^T: 8-token groups 128 B apart (LBO), 8-row groups 2048 B apart (SBO)
                    const uint64_t bd = umma_smem_desc(pb + k * 256, 128, 2048, 0);
                    umma_bf16_ss(tmem + (2 + ob) * N, ad, bd, IDESC_PV, (!pe_first) || (k > 0));
                }
                umma_commit(smem_u32(&mi->empty[slot]));      // slice consumed: the stage is free
                umma_commit(smem_u32(&mi->p_done[b]));        // P^T buffer free, O updated
                if (pe_last) umma_commit(smem_u32(&mi->o_done[ob]));
            }
            __syncwarp();
            pend = false;
        };
        for (;;) {
            const uint32_t qs = qi % KT_TQ;
            // never sit on finished work while waiting for the next tile
            if (pend && !mbar_try_wait(smem_u32(&mi->tq_full[qs]), (qi / KT_TQ) & 1)) issue_pv();
            mbar_wait(smem_u32(&mi->tq_full[qs]), (qi / KT_TQ) & 1);
            const KtDesc d = mi->tq[qs];
            __syncwarp();
            if (lane == 0) mbar_arrive(smem_u32(&mi->tq_empty[qs]));
            ++qi;
            if (d.item < 0) break;
            const uint32_t qb = q_base + (tc & 1) * kt_q_bytes(N);
            const int n = d.n_slices;
            // the tile's query rows (cp.async of the scheduler warp, generic proxy) must be visible to the tensor core
            mbar_wait(smem_u32(&mi->q_full[tc & 1]), (tc >> 1) & 1);
            fence_proxy_async();
            for (int i = 0; i < n; ++i) {
                // ---- S_i^T = K_i Q^T into score buffer (g & 1)
                const uint32_t g = gs + (uint32_t)i, slot = g % NS, b = g & 1;
                mbar_wait(smem_u32(&mi->full[slot]), (g / NS) & 1);
                if (lane == 0 && g == 0) kt_stamp(p, 2);
                if (lane == 0 && i == n - 1) kt_stamp(p, 10);
                mbar_wait(smem_u32(&mi->s_empty[b]), ((g >> 1) & 1) ^ 1);
                tc_fence_after();
                if (elect_one()) {
                    const uint32_t k0 = st_base + slot * KT_STAGE_BYTES;
#pragma unroll
                    for (int sb = 0; sb < 2; ++sb)
#pragma unroll
                        for (int j = 0; j < 4; ++j) {           // K = 16 per MMA: 32 bytes inside the swizzled row
                            const uint64_t ad = umma_smem_desc(k0 + sb * KT_SUBB + j * 32, 16, 1024, 2);
                            const uint64_t bd = umma_smem_desc(qb + sb * (N * 128) + j * 32, 16, 1024, 2);
                            umma_bf16_ss(tmem + b * N, ad, bd, IDESC_S, (sb | j) != 0);
                        }
                    umma_commit(smem_u32(&mi->s_full[b]));
                    if (i == n - 1) umma_commit(smem_u32(&mi->q_free[tc & 1]));
                }
                __syncwarp();
                if (pend) issue_pv();
                pend = true;
                pe_g = g; pe_tc = tc; pe_first = i == 0; pe_last = i == n - 1;
                pe_ksteps = (i == n - 1) ? (d.valid_last + 15) >> 4 : KT_SLICE / 16;
            }
            gs += (uint32_t)n;
            ++tc;
        }
        if (pend) issue_pv();
    } else if (warp < 6) {
        // =========================================================== softmax warps (thread = token of the slice)
        const int q4 = warp & 3;                          // TMEM lane quadrant this warp may access
        const int st = q4 * 32 + lane;                    // token of the slice
        const uint32_t tl = tmem + ((uint32_t)(q4 * 32) << 16);
        uint32_t gs = 0, qi = 0, tc = 0;
        for (;;) {
            const uint32_t qs = qi % KT_TQ;
            mbar_wait(smem_u32(&mi->tq_full[qs]), (qi / KT_TQ) & 1);
            const KtDesc d = mi->tq[qs];
            __syncwarp();
            if (lane == 0) mbar_arrive(smem_u32(&mi->tq_empty[qs]));
            ++qi;
            if (d.item < 0) break;
            const uint32_t ob = tc & 1;

            float m_ref[N], l_part[N];
#pragma unroll
            for (int h = 0; h < N; ++h) { m_ref[h] = -INFINITY; l_part[h] = 0.f; }
            const int n = d.n_slices;
            for (int i = 0; i < n; ++i) {
                const uint32_t g = gs + (uint32_t)i, b = g & 1;
                mbar_wait(smem_u32(&mi->s_full[b]), (g >> 1) & 1);
                tc_fence_after();
                uint32_t xr[N];
#pragma unroll
                for (int c = 0; c < N; c += 16)
                    tmem_ld16(tl + b * N + c, *reinterpret_cast<uint32_t (*)[16]>(&xr[c]));
                tmem_wait_ld();
                tc_fence_before();
                __syncwarp();
                if (lane == 0) mbar_arrive(smem_u32(&mi->s_empty[b]));       // score buffer free
                const int nvalid = (i == n - 1) ? d.valid_last : KT_SLICE;
                const bool tv = st < nvalid;
                float x[N];
                float ex = -INFINITY;
                // q_len > 1 (causal among the query tokens): row (t, h) sees positions < ctx - (q_len - 1 - t), i.e. this
                // thread's token, rem = ctx - position, is seen by the rows t >= q_len - rem: rows hmin .. N - 1.  Only the
                // slices that reach into the context's last q_len - 1 tokens take this path (CTA-uniform).
                const int rem_slice = d.rem0 - i * KT_SLICE;          // context length - first token of the slice
                const bool cmask = QL && rem_slice < KT_SLICE + d.q_len - 1;
                int hmin = 0;
                if (cmask) hmin = max(0, d.q_len - (rem_slice - st)) * d.hpk;
#pragma unroll
                for (int h = 0; h < N; ++h) x[h] = __uint_as_float(xr[h]) * d.scale_log2;
                if (cmask) {
#pragma unroll
                    for (int h = 0; h < N; ++h)
                        if (h < hmin) x[h] = -INFINITY;
                }
#pragma unroll
                for (int h = 0; h < N; ++h) ex = fmaxf(ex, x[h] - m_ref[h]);     // (-inf) - (-inf) = NaN never wins the maximum
                // NaN scores (NaN inputs) never trigger: they flow into P and O as in the definition
                if (bar_red_or_softmax(tv && ex > KT_LAZY_LOG2)) {
                    // ---- the reference moves: column maxima of the slice, rescale O and the partial sums
                    float mn[N];
#pragma unroll
                    for (int cb = 0; cb < NB; ++cb) {
                        float v[CN];
#pragma unroll
                        for (int h = 0; h < CN; ++h) v[h] = tv ? x[cb * CN + h] : -INFINITY;
                        const float cm = col_reduce<CN>(v, lane, OpMax());
                        if (lane < CN) mi->redmax[(cb * CN + lane) * 4 + q4] = cm;
                    }
                    bar_sync_softmax();
#pragma unroll
                    for (int h = 0; h < N; ++h) {
                        const float4 r4 = *reinterpret_cast<const float4 *>(&mi->redmax[h * 4]);
                        mn[h] = fmaxf(m_ref[h], fmaxf(fmaxf(r4.x, r4.y), fmaxf(r4.z, r4.w)));
                    }
                    if (i > 0) {
                        // O^T is rescaled in place (thread = value column, TMEM column = query row): the
                        // value MMAs of the previous slice must be complete
                        mbar_wait(smem_u32(&mi->p_done[(g - 1) & 1]), ((g - 1) >> 1) & 1);
                        tc_fence_after();
#pragma unroll
                        for (int c = 0; c < N; c += 16) {
                            uint32_t o[16];
                            tmem_ld16(tl + (2 + ob) * N + c, o);
                            tmem_wait_ld();
#pragma unroll
                            for (int j = 0; j < 16; ++j)
                                o[j] = __float_as_uint(__uint_as_float(o[j]) * kt_rescale<QL>(m_ref[c + j], mn[c + j]));
                            tmem_st16(tl + (2 + ob) * N + c, o);
                        }
                        tmem_wait_st();
                        tc_fence_before();
                    }
#pragma unroll
                    for (int h = 0; h < N; ++h) {
                        l_part[h] *= kt_rescale<QL>(m_ref[h], mn[h]);     // 2^(-inf) = 0 on the first slice (l_part is 0 there)
                        m_ref[h] = mn[h];
                    }
                    bar_sync_softmax();        // redmax[] may be rewritten only after every thread has read it
                }
                uint32_t pw[N / 2];
                if (!cmask) {
#pragma unroll
                    for (int h = 0; h < N; h += 2) {
                        const float p0 = tv ? ex2_ftz(x[h] - m_ref[h]) : 0.f;
                        const float p1 = tv ? ex2_ftz(x[h + 1] - m_ref[h + 1]) : 0.f;
                        l_part[h] += p0;
                        l_part[h + 1] += p1;
                        asm("cvt.rn.bf16x2.f32 %0, %1, %2;" : "=r"(pw[h >> 1]) : "f"(p1), "f"(p0));
                    }
                } else {
                    // a masked score (-inf) under a reference that is still -inf (a row that sees no token of the tile
                    // so far) would give 2^(NaN): such entries are 0 by the row test, not by the exponential
#pragma unroll
                    for (int h = 0; h < N; h += 2) {
                        const float p0 = tv && h >= hmin ? ex2_ftz(x[h] - m_ref[h]) : 0.f;
                        const float p1 = tv && h + 1 >= hmin ? ex2_ftz(x[h + 1] - m_ref[h + 1]) : 0.f;
                        l_part[h] += p0;
                        l_part[h + 1] += p1;
                        asm("cvt.rn.bf16x2.f32 %0, %1, %2;" : "=r"(pw[h >> 1]) : "f"(p1), "f"(p0));
                    }
                }
                // the P^T buffer is free once the value MMAs of slice g - 2 are complete
                mbar_wait(smem_u32(&mi->p_done[b]), ((g >> 1) & 1) ^ 1);
                // P^T[token][row]: 16-B chunk c (rows 8c..8c+7) of token t at c * 2048 + t * 16
                const uint32_t pb = p_base + b * kt_p_bytes(N) + st * 16;
#pragma unroll
                for (int c = 0; c < N / 8; ++c)
                    asm volatile("st.shared.v4.b32 [%0], {%1,%2,%3,%4};" ::"r"(pb + c * 2048), "r"(pw[4 * c]),
                                 "r"(pw[4 * c + 1]), "r"(pw[4 * c + 2]), "r"(pw[4 * c + 3]) : "memory");
                if ((nvalid & 15) != 0) {
                    // dead slots inside the last 16-token k-step may hold NaN: zero their value rows (0 * NaN)
                    const uint32_t vb = st_base + (g % NS) * KT_STAGE_BYTES + 2 * KT_SUBB;
                    const int nz = 16 - (nvalid & 15);
                    for (int e = st; e < nz * 16; e += 128) {
                        const int row = nvalid + (e >> 4), ch = e & 15;
                        asm volatile("st.shared.v4.b32 [%0], {%1,%1,%1,%1};"
                                     ::"r"(vb + (ch >> 3) * KT_SUBB + row * 128 + (((ch & 7) ^ (row & 7)) << 4)), "r"(0u) : "memory");
                    }
                }
                fence_proxy_async();
                tc_fence_before();
                __syncwarp();
                if (lane == 0) mbar_arrive(smem_u32(&mi->p_full[b]));
            }
            gs += (uint32_t)n;
            if (tid == 64) kt_stamp(p, 4);

            // ---- end of tile: row sums (fixed tree) and references into this O buffer's hand-over area,
            // which the epilogue of tile tc - 2 must have read
            if (tc >= 2) mbar_wait(smem_u32(&mi->o_free[ob]), ((tc >> 1) - 1) & 1);
#pragma unroll
            for (int cb = 0; cb < NB; ++cb) {
                float v[CN];
#pragma unroll
                for (int h = 0; h < CN; ++h) v[h] = l_part[cb * CN + h];
                const float s = col_reduce<CN>(v, lane, OpAdd());
                if (lane < CN) mi->red[ob][(cb * CN + lane) * 4 + q4] = s;
            }
            if (q4 == 0) {
                float mr = 0.f;
#pragma unroll
                for (int h = 0; h < N; ++h) mr = (h == lane) ? m_ref[h] : mr;
                if (lane < N) mi->mref[ob][lane] = mr;
            }
            __syncwarp();
            if (lane == 0) mbar_arrive(smem_u32(&mi->e_full[ob]));           // release; the epilogue warps acquire
            ++tc;
        }
    } else if (warp < 10) {
        // =========================================================== epilogue warps (thread = value column d)
        const int q4 = warp & 3;
        const int dcol = q4 * 32 + lane;
        const uint32_t tl = tmem + ((uint32_t)(q4 * 32) << 16);
        uint32_t qi = 0, tc = 0;
        // House-keeping of the last CTA, done by an epilogue warp because it has nothing to do until the first tile
        // ends (measured: the same lines between the set-up barrier and the role switch, where the scheduler and the
        // producer warp pass through them, cost cfg4 1.7 us of start-up).  (1) The other counter set is zeroed for
        // the next launch.  (2) Fused decode step: the context table of the launches that follow is filled -- every
        // entry copied, then the batch's requests set to + ctx_add (no launch reads the table it writes).
        if (warp == 9 && blockIdx.x == gridDim.x - 1) {
            for (int i = lane; i < p.n_groups; i += 32) p.reset_counters[32 + (size_t)i * kCounterStride] = 0;
            if (lane < 4) p.reset_counters[lane] = 0;
            if (p.req_ctx_next != nullptr) {
                for (int i = lane; i < p.max_requests; i += 32) p.req_ctx_next[i] = __ldg(p.req_ctx + i);
                __syncwarp();
                for (int g = lane; g < p.n_groups; g += 32) {
                    const Group gr = p.groups[g];
                    if (gr.kv_head == 0) p.req_ctx_next[gr.req] = __ldg(p.req_ctx + gr.req) + p.ctx_add;
                }
            }
        }
        for (;;) {
            const uint32_t qs = qi % KT_TQ;
            mbar_wait(smem_u32(&mi->tq_full[qs]), (qi / KT_TQ) & 1);
            const KtDesc d = mi->tq[qs];
            __syncwarp();
            if (lane == 0) mbar_arrive(smem_u32(&mi->tq_empty[qs]));
            ++qi;
            if (d.item < 0) break;
            const uint32_t ob = tc & 1, ph = (tc >> 1) & 1;
            mbar_wait(smem_u32(&mi->e_full[ob]), ph);        // row sums and references are there
            mbar_wait(smem_u32(&mi->o_done[ob]), ph);        // every value MMA of the tile is complete
            tc_fence_after();
            uint32_t o[N];
#pragma unroll
            for (int c = 0; c < N; c += 16)
                tmem_ld16(tl + (2 + ob) * N + c, *reinterpret_cast<uint32_t (*)[16]>(&o[c]));
            const bool final_out = d.n_splits == 1;
            // row sum of head h: the four softmax warps' parts in a fixed order
            float Lh = 1.f, mr = 0.f;
            if (dcol < d.gsize) {
                const float4 r4 = *reinterpret_cast<const float4 *>(&mi->red[ob][dcol * 4]);
                Lh = (r4.x + r4.y) + (r4.z + r4.w);
                mr = mi->mref[ob][dcol];
            }
            float inv[N];
            if (final_out) {
#pragma unroll
                for (int h = 0; h < N; ++h) {
                    const float4 r4 = *reinterpret_cast<const float4 *>(&mi->red[ob][h * 4]);
                    inv[h] = 1.0f / ((r4.x + r4.y) + (r4.z + r4.w));
                }
            }
            tmem_wait_ld();
            tc_fence_before();
            __syncwarp();
            if (lane == 0) mbar_arrive(smem_u32(&mi->o_free[ob]));           // O^T buffer and hand-over area are free
            if (final_out) {
                float *dst = p.out + d.out_off + dcol;
                if (!QL) {
#pragma unroll
                    for (int h = 0; h < N; ++h)
                        if (h < d.gsize) dst[h * KT_D] = __uint_as_float(o[h]) * inv[h];
                    if (dcol < d.gsize) p.lse[d.lse_off + dcol] = (mr + log2f(Lh)) * 0.6931471805599453f;
                } else {
                    // row (t, hh) of the group is row t * Hq + hh of the request's output
                    int t = 0, hh = 0;
#pragma unroll
                    for (int h = 0; h < N; ++h) {
                        if (h < d.gsize) dst[(size_t)(t * d.n_q_heads + hh) * KT_D] = __uint_as_float(o[h]) * inv[h];
                        if (++hh == d.hpk) { hh = 0; ++t; }
                    }
                    if (dcol < d.gsize)
                        p.lse[d.lse_off + (dcol / d.hpk) * d.n_q_heads + dcol % d.hpk] = (mr + log2f(Lh)) * 0.6931471805599453f;
                }
            } else {
                // O partial of head h, split s, column c: [h][c / (4 CQ)][s][(c / 4) % CQ][c % 4] with
                // CQ = 32 >> zl column quads per combine unit, so that the 32 lanes of a combine unit -- 2^zl
                // split lanes x CQ quads -- read 512 contiguous bytes
                const int cq_log2 = 5 - d.zl, quad = dcol >> 2;
                float *dst = p.workspace + d.part_off +
                             ((((int64_t)(quad >> cq_log2) * d.n_splits + d.split) << cq_log2) + (quad & ((1 << cq_log2) - 1))) * 4 + (dcol & 3);
                const int64_t hstride = (int64_t)d.n_splits * KT_D;
#pragma unroll
                for (int h = 0; h < N; ++h)
                    if (h < d.gsize) dst[h * hstride] = __uint_as_float(o[h]);
                // (m, l) of row dcol, written by the thread whose index is the row
                if (dcol < d.gsize)
                    *reinterpret_cast<float2 *>(p.workspace + d.part_off + part_ml_off(d.gsize, dcol, d.split, d.n_splits, KT_D)) =
                        make_float2(mr, Lh);
                // the warp's partial stores happen-before lane 0's gpu-scope release (cumulative over the
                // __syncwarp), which the combine acquires: no membar needed
                __syncwarp();
                if (lane == 0) red_release_add(p.group_counters + (size_t)d.group_idx * kCounterStride, 1);
            }
            if (tid == 192) kt_stamp(p, 5);
            ++tc;
        }
    }
    // ---- LSE combine (step a4): warp-sized units, statically assigned to ALL warps of every CTA
    __syncthreads();
    if (tid == 0) kt_stamp(p, 6);
    kt_combine(p, warp, lane);
    tc_fence_before();
    __syncthreads();
    if (tid == 0) kt_stamp(p, 7);
    if (warp == 2) tmem_dealloc(tmem, kt_tmem_cols(N));
}

// ----------------------------------------------------------------------------- host side
bool kvt_supported(int P) { return P == 16 || P == 32 || P == 64 || P == 128; }

int kvt_pad_rows(int g)          // N of the instantiation that serves groups of up to g rows (0: none)
{
    return g <= 16 ? 16 : g <= 32 ? 32 : 0;
}

template <int N, bool QL>
static cudaError_t launch_kvt_n(const DecodeParams &p, const CUtensorMap &tmap, int rows_per_page, int grid,
                                cudaStream_t stream)
{
    static bool configured[64] = {};
    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    if (dev < 0 || dev >= 64 || !configured[dev]) {
        e = cudaFuncSetAttribute(cp_decode_kvt_kernel<N, QL>, cudaFuncAttributeMaxDynamicSharedMemorySize, kt_smem_bytes(N));
        if (e != cudaSuccess) return e;
        if (dev >= 0 && dev < 64) configured[dev] = true;
    }
    // launched as a programmatic dependent of the stream's previous kernel (see griddepcontrol.wait in the kernel)
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3((unsigned)grid); cfg.blockDim = dim3(KT_THREADS); cfg.dynamicSmemBytes = (size_t)kt_smem_bytes(N); cfg.stream = stream;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = attr; cfg.numAttrs = 1;
    return cudaLaunchKernelEx(&cfg, cp_decode_kvt_kernel<N, QL>, p, tmap, rows_per_page);
}

// grid: the number of CTAs the plan's static tile lists were laid out for (slot j of CTA b is record
// b, the rest of its list is chained through TileRec::next); CTAs beyond the tiles still help with the combine units.
cudaError_t launch_decode_kvt(const DecodeParams &p, const void *tmap, int rows_per_page, int grid, int max_group,
                              cudaStream_t stream)
{
    const CUtensorMap &tm = *reinterpret_cast<const CUtensorMap *>(tmap);
    if (grid < 1) grid = 1;
    switch (kvt_pad_rows(max_group)) {
    case 16: return p.q_len > 1 ? launch_kvt_n<16, true>(p, tm, rows_per_page, grid, stream)
                                : launch_kvt_n<16, false>(p, tm, rows_per_page, grid, stream);
    case 32: return p.q_len > 1 ? launch_kvt_n<32, true>(p, tm, rows_per_page, grid, stream)
                                : launch_kvt_n<32, false>(p, tm, rows_per_page, grid, stream);
    default: return cudaErrorInvalidValue;
    }
}

}  // namespace cp
