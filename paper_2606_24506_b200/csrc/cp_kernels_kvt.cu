// cp_kernels_kvt.cu -- the MQA / GQA fast path of libcrosspool on the 5th-generation tensor cores
// (hot-path steps a2-a6 for kind CP_KIND_KV with d_k = d_v = 128): ONE persistent launch per
// decode step, tcgen05.mma with the TOKENS on the MMA M dimension.
//
// A (request, kv head) group has g = Hq / Hkv query rows -- 8 to 32 here -- far fewer than the 128
// rows a tcgen05 tile wants, so the roles are swapped: a slice of 128 cached tokens is the M
// dimension and the group's rows (padded to N = 16 / 32 / ...) are the N dimension,
//     S^T[128 tok x N] = K_slice[128 tok x 128 d] . Q^T          8 x tcgen05.mma M128 N K16
//                        (A = the K blocks exactly as TMA lands them, K-major SWIZZLE_128B;
//                         B = the query rows, K-major SWIZZLE_128B)
//     O^T[128 d x N]  += V_slice^T[128 d x 128 tok] . P^T         8 x tcgen05.mma M128 N K16
//                        (A = the V blocks as landed, read MN-major; B = P^T written by the softmax
//                         threads as bf16, MN-major without swizzle),
// both accumulators in tensor memory (2 score buffers + O = 3 N columns).  A softmax thread owns one
// TMEM lane = one token of the slice and N scores, one per query row.  It needs the row (= query
// head) maximum only as a REFERENCE for the exponent, not exactly: every thread keeps the same
// per-head reference m_ref[h] and computes p = 2^(s - m_ref[h]) with no cross-thread reduction;
// the reference moves (and O / l are rescaled) only when some score exceeds it by more than 2^8,
// which the 128 threads agree on with one barrier.red.or per slice (for the data at hand: once,
// on the first slice of a tile).  The row sums l[h] are per-thread partial sums that are reduced
// once per tile in a fixed shuffle tree, so results are deterministic.
//
// Why tcgen05 here although north_star keeps it "only on the MLA path": measured in round 1, eight
// mma.sync consumer warps sustain 3.4 TB/s-equivalent at g = 32 (cfg4) and their end-of-tile merge
// through shared memory costs ~3 us; with the tokens on M one elected thread issues 16 MMAs per 128
// tokens (~950 cycles against a 2800-cycle HBM budget per slice and SM), for ANY g <= N, and the
// tile result sits in ONE accumulator.
//
// Warp roles (256 threads, 1 CTA / SM):
//   warp 0      producer: pops tiles, translates logical pages through the page table (step a2) and
//               streams them with TMA into a ring of 64 KB slice stages [K d0-63 | K d64-127 |
//               V d0-63 | V d64-127], each a [128 tok x 128 B] SWIZZLE_128B block that the pages of
//               the slice fill top to bottom.
//   warp 1      MMA issuer (one lane by elect.sync); stages the tile's query rows into shared memory.
//   warps 2..5  softmax (thread = token of the slice), epilogue (thread = value column d).
//   warps 6..7  only help with the LSE combine units after the last tile.
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
constexpr int KT_WARPS = 8;
constexpr int KT_THREADS = 32 * KT_WARPS;
constexpr int KT_MISC_BYTES = 3072;
constexpr int KT_SMEM_LIMIT = 232448;                // 227 KB opt-in maximum per CTA
constexpr float KT_LAZY_LOG2 = 8.0f;                 // the reference moves when a score exceeds it by 2^8

__host__ __device__ constexpr int kt_q_bytes(int N) { return 2 * N * 128; }          // one query buffer: 2 blocks [N x 128 B]
__host__ __device__ constexpr int kt_p_bytes(int N) { return (N / 8) * 2048; }       // one P^T buffer
__host__ __device__ constexpr int kt_fixed_bytes(int N) { return 2 * kt_q_bytes(N) + 2 * kt_p_bytes(N) + KT_MISC_BYTES; }
__host__ __device__ constexpr int kt_num_stages(int N) { return (KT_SMEM_LIMIT - kt_fixed_bytes(N)) / KT_STAGE_BYTES; }
__host__ __device__ constexpr int kt_smem_bytes(int N) { return kt_num_stages(N) * KT_STAGE_BYTES + kt_fixed_bytes(N); }
__host__ __device__ constexpr uint32_t kt_tmem_cols(int N) { return 3 * N <= 32 ? 32u : 3 * N <= 64 ? 64u : 3 * N <= 128 ? 128u : 3 * N <= 256 ? 256u : 512u; }

struct KtDesc {                  // what the producer hands to the other warps for one tile
    int32_t item;                // work index; < 0: no more work
    int32_t group_idx;
    int32_t n_slices;            // 128-token slices of the tile
    int32_t valid_last;          // valid tokens of the last slice (1..128)
    int32_t split, n_splits;
    int32_t gsize;               // query rows of the group
    float scale_log2;
    int64_t q_off, out_off, lse_off, part_off;
};

struct KtMisc {
    uint64_t full[4], empty[4];                  // slice ring: TMA -> MMA, MMA (commit) -> TMA
    uint64_t s_full[2], s_empty[2];              // score buffers in TMEM: MMA -> softmax -> MMA
    uint64_t p_full[2], p_done[2];               // P^T buffers: softmax -> MMA, MMA (commit) -> softmax
    uint64_t q_free[2];                          // query buffers: score MMAs of the tile that used it are complete
    uint64_t tq_full[KT_TQ], tq_empty[KT_TQ];
    KtDesc tq[KT_TQ];
    uint32_t tmem_base;
    uint32_t pad[3];
    float red[4 * 128];                          // cross-warp reductions: [column][warp]
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

__device__ __forceinline__ void kt_stamp(const DecodeParams &p, int k)
{
    if (p.timeline) p.timeline[(size_t)blockIdx.x * kTimelineSlots + k] = global_timer_ns();
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

template <int N>
__global__ void __launch_bounds__(KT_THREADS, 1)
cp_decode_kvt_kernel(const DecodeParams p, const __grid_constant__ CUtensorMap tmap, int rows_per_page)
{
    constexpr int NS = kt_num_stages(N);
    constexpr int CN = N >= 32 ? 32 : 16;            // column block of the reductions
    constexpr int NB = N / CN;
    static_assert(NS >= 2 && NS <= 4, "slice ring depth");
    static_assert(N % 16 == 0 && N >= 16 && N <= 128, "N = padded query rows of a group");

    extern __shared__ __align__(1024) uint8_t smem[];
    const uint32_t st_base = smem_u32(smem);
    const uint32_t q_base = st_base + NS * KT_STAGE_BYTES;
    const uint32_t p_base = q_base + 2 * kt_q_bytes(N);
    KtMisc *mi = reinterpret_cast<KtMisc *>(smem + NS * KT_STAGE_BYTES + 2 * kt_q_bytes(N) + 2 * kt_p_bytes(N));

    const int tid = threadIdx.x;
    const int warp = tid >> 5;
    const int lane = tid & 31;
    if (tid == 0) kt_stamp(p, 0);
    scheduler_reset_other_set(p);

    if (tid == 0) {
        for (int i = 0; i < NS; ++i) { mbar_init(smem_u32(&mi->full[i]), 1); mbar_init(smem_u32(&mi->empty[i]), 1); }
        for (int i = 0; i < 2; ++i) {
            mbar_init(smem_u32(&mi->s_full[i]), 1); mbar_init(smem_u32(&mi->s_empty[i]), 4);
            mbar_init(smem_u32(&mi->p_full[i]), 4); mbar_init(smem_u32(&mi->p_done[i]), 1);
            mbar_init(smem_u32(&mi->q_free[i]), 1);
        }
        for (int i = 0; i < KT_TQ; ++i) { mbar_init(smem_u32(&mi->tq_full[i]), 1); mbar_init(smem_u32(&mi->tq_empty[i]), 5); }
        asm volatile("prefetch.tensormap [%0];" ::"l"(reinterpret_cast<uint64_t>(&tmap)) : "memory");
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
        fence_proxy_async();
    }
    if (warp == 1) tmem_alloc(smem_u32(&mi->tmem_base), kt_tmem_cols(N));
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    const uint32_t tmem = mi->tmem_base;
    const int P = (int)p.page_tokens;
    const int pps = KT_SLICE / P;                    // pages per slice

    if (warp == 0) {
        // =========================================================== producer warp
        uint64_t policy;
        asm volatile("createpolicy.fractional.L2::evict_first.b64 %0, 1.0;" : "=l"(policy));
        uint32_t gs = 0;          // slices issued by this CTA (ring position)
        uint32_t qi = 0;          // work items pushed
        for (;;) {
            // the first tile of a CTA is static (its block index): no atomic round trip at start-up
            int work = 0;
            if (qi == 0) work = blockIdx.x;
            else {
                if (lane == 0) work = atomicAdd(p.work_counter, 1) + (int)gridDim.x;
                work = __shfl_sync(0xffffffffu, work, 0);
            }
            const int item = work < p.n_tiles ? work : -1;
            TileRec r;
            int n_slices = 0, valid_last = KT_SLICE, npg = 0;
            if (item >= 0) {
                const uint4 *src = reinterpret_cast<const uint4 *>(p.tile_recs + item);
                uint4 *dst = reinterpret_cast<uint4 *>(&r);
#pragma unroll
                for (int i = 0; i < 5; ++i) dst[i] = __ldg(src + i);
                const int ctx = __ldg(p.req_ctx + r.req);
                const int t_begin = r.page_begin * P;
                const int t_end = min((r.page_begin + r.n_pages) * P, ctx);
                n_slices = (t_end - t_begin + KT_SLICE - 1) / KT_SLICE;
                valid_last = t_end - t_begin - (n_slices - 1) * KT_SLICE;
                npg = (t_end - t_begin + P - 1) / P;         // pages of the tile that hold at least one valid token
            } else {
                r.group = 0; r.req = 0; r.kv_head = 0; r.n_kv_heads = 1; r.page_begin = 0; r.n_pages = 0;
                r.split = 0; r.n_splits = 1; r.gsize = 1; r.n_q_heads = 1; r.scale_log2 = 0.f;
                r.q_off = r.out_off = r.lse_off = r.part_off = 0; r.pad = 0;
            }
            const uint32_t qs = qi % KT_TQ;
            mbar_wait(smem_u32(&mi->tq_empty[qs]), ((qi / KT_TQ) & 1) ^ 1);
            if (lane == 0) {
                KtDesc d;
                d.item = item; d.group_idx = r.group; d.n_slices = n_slices; d.valid_last = valid_last;
                d.split = r.split; d.n_splits = r.n_splits; d.gsize = r.gsize; d.scale_log2 = r.scale_log2;
                d.q_off = r.q_off; d.out_off = r.out_off; d.lse_off = r.lse_off; d.part_off = r.part_off;
                mi->tq[qs] = d;
                mbar_arrive(smem_u32(&mi->tq_full[qs]));     // release: the consumers acquire via try_wait
            }
            ++qi;
            if (item < 0) break;

            const int hkv = r.n_kv_heads;
            for (int j0 = 0; j0 < npg; j0 += 32) {
                // translate up to 32 logical pages at once (step a2: one page-table entry per lane)
                int32_t pid = 0;
                if (j0 + lane < npg) pid = page_of(p, r.req, (int64_t)(r.page_begin + j0 + lane) * hkv + r.kv_head);
                const int nj = min(32, npg - j0);
                for (int j = 0; j < nj; ++j) {
                    const int32_t my = __shfl_sync(0xffffffffu, pid, j);
                    const int jj = j0 + j;
                    const int pg = jj % pps;                 // position of the page inside its slice
                    const uint32_t slot = gs % NS;
                    if (pg == 0) mbar_wait(smem_u32(&mi->empty[slot]), ((gs / NS) & 1) ^ 1);
                    if (elect_one()) {
                        const uint32_t fb = smem_u32(&mi->full[slot]);
                        if (pg == 0) mbar_arrive_expect_tx(fb, (uint32_t)min(pps, npg - jj) * (uint32_t)P * 512u);
                        const uint32_t dst = st_base + slot * KT_STAGE_BYTES + (uint32_t)pg * (uint32_t)P * 128u;
                        const int row = my * rows_per_page;
                        tma_load_2d(dst, &tmap, 0, row, fb, policy);                    // K, d 0..63
                        tma_load_2d(dst + KT_SUBB, &tmap, 64, row, fb, policy);         // K, d 64..127
                        tma_load_2d(dst + 2 * KT_SUBB, &tmap, 0, row + P, fb, policy);  // V, d 0..63
                        tma_load_2d(dst + 3 * KT_SUBB, &tmap, 64, row + P, fb, policy); // V, d 64..127
                    }
                    if (pg == pps - 1 || jj == npg - 1) ++gs;
                }
            }
        }
        if (lane == 0) kt_stamp(p, 3);
    } else if (warp == 1) {
        // =========================================================== MMA issuer warp
        constexpr uint32_t IDESC_S = umma_idesc_bf16(KT_SLICE, N, 0, 0);      // K (K-major) x Q^T (K-major)
        constexpr uint32_t IDESC_PV = umma_idesc_bf16(KT_SLICE, N, 1, 1);     // V^T (MN-major) x P^T (MN-major)
        uint32_t gs = 0, qi = 0, tc = 0;
        for (;;) {
            const uint32_t qs = qi % KT_TQ;
            mbar_wait(smem_u32(&mi->tq_full[qs]), (qi / KT_TQ) & 1);
            const KtDesc d = mi->tq[qs];
            __syncwarp();
            if (lane == 0) mbar_arrive(smem_u32(&mi->tq_empty[qs]));
            ++qi;
            if (d.item < 0) break;
            if (lane == 0 && tc == 0) kt_stamp(p, 1);
            // ---- the tile's query rows -> buffer (tc & 1): two K-major [N x 64] blocks, 128-byte swizzle
            // (16-B chunk index ^ (row & 7)); rows beyond the group are zero.  The buffer is free once
            // the score MMAs of tile tc - 2 are complete.
            const uint32_t qb = q_base + (tc & 1) * kt_q_bytes(N);
            if (tc >= 2) mbar_wait(smem_u32(&mi->q_free[tc & 1]), ((tc >> 1) - 1) & 1);
            {
                const uint4 *qg = reinterpret_cast<const uint4 *>(p.q + d.q_off);
#pragma unroll 4
                for (int id = lane; id < N * 16; id += 32) {
                    const int r = id >> 4, ch = id & 15;
                    uint4 v = make_uint4(0u, 0u, 0u, 0u);
                    if (r < d.gsize) v = __ldg(qg + id);
                    const uint32_t a = qb + (ch >> 3) * (N * 128) + r * 128 + (((ch & 7) ^ (r & 7)) << 4);
                    asm volatile("st.shared.v4.b32 [%0], {%1,%2,%3,%4};" ::"r"(a), "r"(v.x), "r"(v.y), "r"(v.z), "r"(v.w) : "memory");
                }
                fence_proxy_async();
                __syncwarp();
            }
            const int n = d.n_slices;
            for (int i = 0; i <= n; ++i) {
                if (i < n) {
                    // ---- S_i^T = K_i Q^T into score buffer (g & 1)
                    const uint32_t g = gs + (uint32_t)i, slot = g % NS, b = g & 1;
                    mbar_wait(smem_u32(&mi->full[slot]), (g / NS) & 1);
                    if (lane == 0 && g == 0) kt_stamp(p, 2);
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
                }
                if (i >= 1) {
                    // ---- O^T += V_{i-1}^T P_{i-1}^T, 16 tokens per MMA; the last slice stops after its last valid 16
                    const uint32_t g = gs + (uint32_t)i - 1, slot = g % NS, b = g & 1;
                    mbar_wait(smem_u32(&mi->p_full[b]), (g >> 1) & 1);
                    tc_fence_after();
                    const int ksteps = (i == n) ? (d.valid_last + 15) >> 4 : KT_SLICE / 16;
                    if (elect_one()) {
                        const uint32_t v0 = st_base + slot * KT_STAGE_BYTES + 2 * KT_SUBB;
                        const uint32_t pb = p_base + b * kt_p_bytes(N);
                        for (int k = 0; k < ksteps; ++k) {
                            // V: 64-column blocks KT_SUBB apart (LBO), 8-token groups 1024 B apart (SBO)
                            const uint64_t ad = umma_smem_desc(v0 + k * 2048, KT_SUBB, 1024, 2);
                            // P^T: 8-token groups 128 B apart (LBO), 8-row groups 2048 B apart (SBO)
                            const uint64_t bd = umma_smem_desc(pb + k * 256, 128, 2048, 0);
                            umma_bf16_ss(tmem + 2 * N, ad, bd, IDESC_PV, (i > 1) || (k > 0));
                        }
                        umma_commit(smem_u32(&mi->empty[slot]));      // slice consumed: the stage is free
                        umma_commit(smem_u32(&mi->p_done[b]));        // P^T buffer free, O updated
                    }
                    __syncwarp();
                }
            }
            gs += (uint32_t)n;
            ++tc;
        }
    } else if (warp < 6) {
        // =========================================================== softmax warps (thread = token of the slice)
        const int q4 = warp & 3;                          // TMEM lane quadrant this warp may access
        const int st = q4 * 32 + lane;                    // token of the slice / value column of the epilogue
        const uint32_t tl = tmem + ((uint32_t)(q4 * 32) << 16);
        uint32_t gs = 0, qi = 0;
        for (;;) {
            const uint32_t qs = qi % KT_TQ;
            mbar_wait(smem_u32(&mi->tq_full[qs]), (qi / KT_TQ) & 1);
            const KtDesc d = mi->tq[qs];
            __syncwarp();
            if (lane == 0) mbar_arrive(smem_u32(&mi->tq_empty[qs]));
            ++qi;
            if (d.item < 0) break;

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
#pragma unroll
                for (int h = 0; h < N; ++h) {
                    x[h] = __uint_as_float(xr[h]) * d.scale_log2;
                    ex = fmaxf(ex, x[h] - m_ref[h]);
                }
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
                        if (lane < CN) mi->red[(cb * CN + lane) * 4 + q4] = cm;
                    }
                    bar_sync_softmax();
#pragma unroll
                    for (int h = 0; h < N; ++h) {
                        const float4 r4 = *reinterpret_cast<const float4 *>(&mi->red[h * 4]);
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
                            tmem_ld16(tl + 2 * N + c, o);
                            tmem_wait_ld();
#pragma unroll
                            for (int j = 0; j < 16; ++j)
                                o[j] = __float_as_uint(__uint_as_float(o[j]) * ex2_ftz(m_ref[c + j] - mn[c + j]));
                            tmem_st16(tl + 2 * N + c, o);
                        }
                        tmem_wait_st();
                        tc_fence_before();
                    }
#pragma unroll
                    for (int h = 0; h < N; ++h) {
                        l_part[h] *= ex2_ftz(m_ref[h] - mn[h]);       // 2^(-inf) = 0 on the first slice (l_part is 0 there)
                        m_ref[h] = mn[h];
                    }
                    bar_sync_softmax();        // red[] may be rewritten (end of tile) only after every thread has read it
                }
                uint32_t pw[N / 2];
#pragma unroll
                for (int h = 0; h < N; h += 2) {
                    const float p0 = tv ? ex2_ftz(x[h] - m_ref[h]) : 0.f;
                    const float p1 = tv ? ex2_ftz(x[h + 1] - m_ref[h + 1]) : 0.f;
                    l_part[h] += p0;
                    l_part[h + 1] += p1;
                    asm("cvt.rn.bf16x2.f32 %0, %1, %2;" : "=r"(pw[h >> 1]) : "f"(p1), "f"(p0));
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

            // ---- end of tile: row sums (fixed tree), then O^T from TMEM (thread = value column st)
#pragma unroll
            for (int cb = 0; cb < NB; ++cb) {
                float v[CN];
#pragma unroll
                for (int h = 0; h < CN; ++h) v[h] = l_part[cb * CN + h];
                const float s = col_reduce<CN>(v, lane, OpAdd());
                if (lane < CN) mi->red[(cb * CN + lane) * 4 + q4] = s;
            }
            bar_sync_softmax();
            {
                const uint32_t gl = gs - 1;
                mbar_wait(smem_u32(&mi->p_done[gl & 1]), (gl >> 1) & 1);      // all value MMAs of the tile are complete
                tc_fence_after();
            }
            const bool final_out = d.n_splits == 1;
            float *dst = final_out ? p.out + d.out_off + st
                                   : p.workspace + d.part_off + part_o_off(0, d.split, d.n_splits, KT_D) + st;
            const int64_t hstride = final_out ? KT_D : (int64_t)d.n_splits * KT_D;
#pragma unroll
            for (int c = 0; c < N; c += 16) {
                uint32_t o[16];
                tmem_ld16(tl + 2 * N + c, o);
                tmem_wait_ld();
#pragma unroll
                for (int j = 0; j < 16; ++j) {
                    const int h = c + j;
                    if (h < d.gsize) {
                        if (final_out) {
                            const float4 r4 = *reinterpret_cast<const float4 *>(&mi->red[h * 4]);
                            dst[h * hstride] = __uint_as_float(o[j]) / ((r4.x + r4.y) + (r4.z + r4.w));
                        } else {
                            __stcg(dst + h * hstride, __uint_as_float(o[j]));
                        }
                    }
                }
            }
            tc_fence_before();
            // (m, l) of row st, written by the thread whose index is the row
            if (st < d.gsize) {
                float mr = 0.f;
#pragma unroll
                for (int h = 0; h < N; ++h) mr = (h == st) ? m_ref[h] : mr;
                const float4 r4 = *reinterpret_cast<const float4 *>(&mi->red[st * 4]);
                const float L = (r4.x + r4.y) + (r4.z + r4.w);
                if (final_out)
                    p.lse[d.lse_off + st] = (mr + log2f(L)) * 0.6931471805599453f;
                else
                    __stcg(reinterpret_cast<float2 *>(p.workspace + d.part_off + part_ml_off(d.gsize, st, d.split, d.n_splits, KT_D)),
                           make_float2(mr, L));
            }
            if (!final_out) {
                // the warp's partial stores happen-before lane 0's gpu-scope release (cumulative over the
                // __syncwarp), which the combine units acquire: no membar needed
                __syncwarp();
                if (lane == 0) red_release_add(p.group_counters + (size_t)d.group_idx * kCounterStride, 1);
            }
            bar_sync_softmax();            // red[] is rewritten by the next tile's first slice
            if (tid == 64) kt_stamp(p, 5);
        }
    }
    // ---- LSE combine (step a4): warp-sized units, statically assigned to ALL warps of every CTA.  The
    // barrier orders it after this CTA's last tile (every slice consumed, every MMA complete), so the
    // slice stages can serve as the warps' scratch.  A unit only waits for tiles that are already
    // running on some SM, so the spin inside terminates.
    __syncthreads();
    if (tid == 0) kt_stamp(p, 6);
    {
        float *wsm = reinterpret_cast<float *>(smem) + warp * kMaxSplits;
        combine_units<8>(p, blockIdx.x * KT_WARPS + warp, gridDim.x * KT_WARPS, wsm, lane);
    }
    tc_fence_before();
    __syncthreads();
    if (tid == 0) kt_stamp(p, 7);
    if (warp == 1) tmem_dealloc(tmem, kt_tmem_cols(N));
}

// ----------------------------------------------------------------------------- host side
bool kvt_supported(int P) { return P == 16 || P == 32 || P == 64 || P == 128; }

int kvt_pad_rows(int g)          // N of the instantiation that serves groups of up to g rows (0: none)
{
    return g <= 16 ? 16 : g <= 32 ? 32 : 0;
}

template <int N>
static cudaError_t launch_kvt_n(const DecodeParams &p, const CUtensorMap &tmap, int rows_per_page, int grid,
                                cudaStream_t stream)
{
    static bool configured[64] = {};
    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    if (dev < 0 || dev >= 64 || !configured[dev]) {
        e = cudaFuncSetAttribute(cp_decode_kvt_kernel<N>, cudaFuncAttributeMaxDynamicSharedMemorySize, kt_smem_bytes(N));
        if (e != cudaSuccess) return e;
        if (dev >= 0 && dev < 64) configured[dev] = true;
    }
    cp_decode_kvt_kernel<N><<<grid, KT_THREADS, kt_smem_bytes(N), stream>>>(p, tmap, rows_per_page);
    return cudaGetLastError();
}

cudaError_t launch_decode_kvt(const DecodeParams &p, const void *tmap, int rows_per_page, int n_ctas, int max_group,
                              cudaStream_t stream)
{
    const CUtensorMap &tm = *reinterpret_cast<const CUtensorMap *>(tmap);
    int grid = p.n_tiles > (p.n_combine_units + KT_WARPS - 1) / KT_WARPS
                   ? p.n_tiles : (p.n_combine_units + KT_WARPS - 1) / KT_WARPS;
    if (grid > n_ctas) grid = n_ctas;
    if (grid < 1) grid = 1;
    switch (kvt_pad_rows(max_group)) {
    case 16: return launch_kvt_n<16>(p, tm, rows_per_page, grid, stream);
    case 32: return launch_kvt_n<32>(p, tm, rows_per_page, grid, stream);
    default: return cudaErrorInvalidValue;
    }
}

}  // namespace cp
