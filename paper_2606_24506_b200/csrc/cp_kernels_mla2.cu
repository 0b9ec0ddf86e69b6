// cp_kernels_mla2.cu -- MLA latent path on CTA PAIRS (cluster of 2 SMs, tcgen05 cta_group::2).
//
// Same computation as cp_kernels_mla.cu (hot-path steps a2, a3', a4-a6 for the 576/512 latent
// shape), but one tile is processed by a pair of CTAs that share every MMA:
//     S[128 x 32]   = Q[128 x 576] . C_slice^T     36 pair-MMAs M128 N32 K16
//     O[128 x 512] += P[128 x 32] . C_slice[:, :512]  2 k-steps x 2 pair-MMAs M128 N256 K16
// Each CTA holds 64 of the 128 heads (its rows of Q, S, P, O) and supplies half of every B
// operand from its own shared memory: its 16 tokens of the slice for the score MMA, its 128 of
// each 256 value columns for the value MMA.  With 64 rows per CTA the accumulator O[64 x 512]
// takes 128 lanes x 256 TMEM columns (2 x 2 layout: columns 0..127 of an N = 256 MMA in lanes
// 0..63, columns 128..255 in lanes 64..127), so all 512 value columns fit and QK^T is computed
// once per tile (the single-CTA kernel computes it once per value half).
//
// Shared memory of one CTA per slice stage: [S area: its 16 tokens x 9 column blocks, K-major]
// [PV area: for k-step kk in {0, 1} (tokens 16kk..16kk+15) and MMA j in {0, 1} its two 64-column
// blocks 4j + 2r, 4j + 2r + 1 (r = CTA rank), MN-major].  Both areas sit at the same offsets in both
// CTAs because one descriptor addresses both.
//
// Warp roles per CTA (192 threads): warp 0 TMA producer; warp 1 MMA issuer in the leader CTA
// (rank 0), relay of the "slice landed" barrier in the peer; warps 2..5 softmax: thread = TMEM
// lane = (head, token half), the two halves of a head exchange their row maximum through shared
// memory.  Tiles are assigned statically to pairs (tile = pair, pair + #pairs, ...).
//
// Paper anchors: paged KV interface PAPER.md:L101,L122; MLA among the KV-head-limited families
// PAPER.md:L21,L57; GPU-resident persistent control PAPER.md:L146.
#include <cuda.h>
#include <cuda_runtime.h>
#include <cstdint>
#include "cp_device_common.cuh"
#include "cp_launch.h"
#include "cp_ptx.cuh"

namespace cp {

constexpr int M2_DK = 576, M2_DV = 512;
constexpr int M2_TS = 32;                           // tokens per slice (16 per CTA for the score MMA)
constexpr int M2_KB = 9;                            // 64-column blocks of the latent row
constexpr int M2_STAGES = 4;                        // value ring: slices (32 tokens) in flight for the value MMAs
constexpr int M2_PF = 4;                            // L2 prefetch distance of the score producer, slice pairs
constexpr int M2_SR = 3;                            // score ring: slice PAIRS (64 tokens) in flight for the score MMAs
constexpr int M2_BLK = 16 * 128;                    // one [16 x 64] swizzled tile: 2048 bytes
constexpr int M2_SAREA = M2_KB * M2_BLK;            // 18432: this CTA's 16 tokens of one slice, 9 column blocks
constexpr int M2_SPAIR = 2 * M2_SAREA;              // 36864: score region of a slice pair, [column block][slice of the pair][16 tokens]
constexpr int M2_PVAREA = 2 * 2 * 2 * M2_BLK;       // 16384: [kk][j][2 blocks]
constexpr int M2_STAGE_BYTES = M2_PVAREA;           // one stage of the value ring
constexpr int M2_QBLK = 64 * 128;                   // one [64 x 64] K-major tile of this CTA's query rows
constexpr int M2_KB_TMEM = 6;                       // query column blocks 0..5 live in TMEM (A operand, TS mode)
constexpr int M2_Q_BYTES = (M2_KB - M2_KB_TMEM) * M2_QBLK;   // 24576: blocks 6..8 in shared memory
constexpr int M2_P_BYTES = 64 * M2_TS * 2;          // 4096 per P buffer (two buffers)
constexpr int M2_WARPS = 8;                         // producer, MMA issuer, 4 softmax warps, 2 that only help with the combine
constexpr int M2_THREADS = 32 * M2_WARPS;
constexpr int M2_SMEM_Q = 0;
constexpr int M2_SMEM_STAGE = M2_Q_BYTES;                    // value ring
constexpr int M2_SMEM_SRING = M2_SMEM_STAGE + M2_STAGES * M2_STAGE_BYTES;
constexpr int M2_SMEM_P = M2_SMEM_SRING + M2_SR * M2_SPAIR;
constexpr int M2_XPOSE_WARP = 32 * 36 * 4;                  // 4608: [32 rows][32 + 4 floats]
constexpr int M2_SMEM_XPOSE = M2_SMEM_P + 2 * M2_P_BYTES;   // epilogue transpose scratch of the 4 softmax warps
constexpr int M2_SMEM_MISC = M2_SMEM_XPOSE + 4 * M2_XPOSE_WARP;
constexpr int M2_SMEM_BYTES = M2_SMEM_MISC + 2048;
static_assert(M2_SMEM_BYTES <= 232448, "MLA pair kernel exceeds the 227 KB shared-memory limit");
constexpr uint32_t M2_TMEM_COLS = 512;
constexpr int M2_SB = 2;                            // score buffers, one slice PAIR each: the score issuer runs one pair ahead
constexpr uint32_t M2_TMEM_S = 256;                         // score buffer b at 256 + 32 b: 2 slices x 16 columns (2 x 2 layout)
constexpr uint32_t M2_TMEM_Q = 320;                         // 192 columns: Q[:, 0:384) as bf16 pairs, rows duplicated in lanes 64..127
static_assert(M2_TMEM_Q + M2_KB_TMEM * 32 <= M2_TMEM_COLS, "TMEM budget");
static_assert((M2_KB_TMEM * 32) % 96 == 0, "query staging batches");
constexpr float M2_LAZY_LOG2 = 8.0f;

struct M2Misc {
    uint64_t full[M2_STAGES];       // value ring: local TMA landed (this CTA's part of the slice)
    uint64_t full_peer[M2_STAGES];  // leader only: the peer's part landed (arrived by the peer's relay warp)
    uint64_t empty[M2_STAGES];      // pair-MMA commit (multicast): value stage free
    uint64_t sl_full[M2_SR];        // score ring: local TMA landed (this CTA's 16 tokens of each slice of the pair)
    uint64_t sl_full_peer[M2_SR];   // leader only: the peer's part landed
    uint64_t sl_empty[M2_SR];       // pair-MMA commit (multicast): score region free
    uint64_t s_full[M2_SB];         // pair-MMA commit (multicast): scores of a slice pair ready
    uint64_t s_empty[M2_SB];        // leader only: 8 softmax warps of the pair have read the scores of both slices
    uint64_t p_full[2];             // leader only: 8 softmax warps have written P buffer (slice & 1)
    uint64_t p_done[2];             // pair-MMA commit (multicast): value MMAs of the slice complete
    uint64_t q_full;                // leader only: 8 softmax warps have staged the query rows
    float xmax[2][128];             // row maxima exchanged between the two token halves of a head (by slice parity)
    float xsum[128];
    uint32_t tmem_base;
};
static_assert(sizeof(M2Misc) <= 2048, "M2Misc must fit its reserved block");

struct M2Item {                     // one tile, derived identically by every warp of the pair
    int32_t valid;                  // false: no more work
    int32_t group_idx, n_slices, valid_last, split, n_splits, n_heads, page_begin, req;
    float scale_log2;
    int64_t q_off, out_off, lse_off, part_off;
};

__device__ __forceinline__ M2Item m2_item(const DecodeParams &p, int tile_idx)
{
    M2Item it;
    it.valid = tile_idx < p.n_tiles;
    if (!it.valid) return it;
    TileRec r;
    const uint4 *src = reinterpret_cast<const uint4 *>(p.tile_recs + tile_idx);
    uint4 *dst = reinterpret_cast<uint4 *>(&r);
#pragma unroll
    for (int i = 0; i < 5; ++i) dst[i] = __ldg(src + i);
    const int ctx = __ldg(p.req_ctx + r.req);
    const int P = (int)p.page_tokens;
    const int t_begin = r.page_begin * P;
    const int t_end = min((r.page_begin + r.n_pages) * P, ctx);
    it.n_slices = (t_end - t_begin + M2_TS - 1) / M2_TS;
    it.valid_last = t_end - t_begin - (it.n_slices - 1) * M2_TS;
    it.group_idx = r.group; it.split = r.split; it.n_splits = r.n_splits; it.n_heads = r.n_q_heads;
    it.page_begin = r.page_begin; it.req = r.req; it.scale_log2 = r.scale_log2;
    it.q_off = r.q_off; it.out_off = r.out_off; it.lse_off = r.lse_off; it.part_off = r.part_off;
    return it;
}

// LSE combine of this kernel (step a4).  The plan's units are 128 value columns of one (group, head) each (zl = 0: a
// lane owns a float4 column and walks the splits in order), four per head; a warp takes TWO neighbouring units at once
// -- they share the head's (m, l) pairs and weights -- so that the 4 x 128 heads x 2 pairs of cfg3 are one round over
// the grid's warps instead of two (measured: a round is ~5 us of dependent L2 round trips at the very end of the
// kernel).  Same arithmetic and summation order as combine_units().
static __device__ __noinline__ void m2_combine(const DecodeParams &p, int w, const int stride, float *wsm, const int lane)
{
    constexpr int NPF = 12;                                // value rows requested before the weights are known
    const int n = p.n_combine_units >> 1;
    int done_group = -1;
    for (; w < n; w += stride) {
        const CombineUnit cu = load_combine_unit<false>(p.cunits, 2 * w);
        const int ns = cu.n_splits;
        if (cu.group != done_group) {
            // relaxed polling with a short back-off, then one acquire fence (as kt_combine of the K/V kernel)
            if (lane == 0) {
                const int32_t *c = p.group_counters + (size_t)cu.group * kCounterStride;
                unsigned nsl = 32;
                while (ld_relaxed(c) < cu.want) {
                    __nanosleep(nsl);
                    if (nsl < 256) nsl <<= 1;
                }
                __threadfence();
            }
            __syncwarp();
            done_group = cu.group;
        }
        const float2 *mlp = reinterpret_cast<const float2 *>(p.workspace + cu.ml_off);
        const float *src = p.workspace + cu.part_off + lane * 4;
        const int ss = cu.split_stride;
        // ONE round trip for the (m, l) pairs (splits lane, lane + 32, ... stay in registers) and the first NPF value rows
        float2 ml[8];
        const bool small = ns <= 256;
        if (small) {
#pragma unroll
            for (int k = 0; k < 8; ++k) {
                ml[k] = make_float2(-INFINITY, 0.f);
                if (lane + 32 * k < ns) ml[k] = __ldcg(mlp + lane + 32 * k);
            }
        }
        float4 va[NPF], vb[NPF];
#pragma unroll
        for (int s = 0; s < NPF; ++s) {
            va[s] = vb[s] = make_float4(0.f, 0.f, 0.f, 0.f);
            if (s < ns) { va[s] = ld_cg_f4(src + s * ss); vb[s] = ld_cg_f4(src + s * ss + 128); }
        }
        float M = -INFINITY, L = 0.f;
        if (small) {
#pragma unroll
            for (int k = 0; k < 8; ++k) M = fmaxf(M, ml[k].x);
            for (int o = 16; o > 0; o >>= 1) M = fmaxf(M, __shfl_xor_sync(0xffffffffu, M, o));
#pragma unroll
            for (int k = 0; k < 8; ++k) {
                const float wgt = ex2_ftz(ml[k].x - M);            // 0 for absent splits (m = -inf)
                if (lane + 32 * k < ns) wsm[lane + 32 * k] = wgt;
                L += wgt * ml[k].y;
            }
        } else {
#pragma unroll 8
            for (int s = lane; s < ns; s += 32) M = fmaxf(M, __ldcg(mlp + s).x);
            for (int o = 16; o > 0; o >>= 1) M = fmaxf(M, __shfl_xor_sync(0xffffffffu, M, o));
#pragma unroll 8
            for (int s = lane; s < ns; s += 32) {
                const float2 x = __ldcg(mlp + s);
                const float wgt = ex2_ftz(x.x - M);
                wsm[s] = wgt;
                L += wgt * x.y;
            }
        }
        for (int o = 16; o > 0; o >>= 1) L += __shfl_xor_sync(0xffffffffu, L, o);
        __syncwarp();
        float4 a = make_float4(0.f, 0.f, 0.f, 0.f), b = a;
#pragma unroll
        for (int s = 0; s < NPF; ++s)
            if (s < ns) {
                const float wgt = wsm[s];
                a.x += wgt * va[s].x; a.y += wgt * va[s].y; a.z += wgt * va[s].z; a.w += wgt * va[s].w;
                b.x += wgt * vb[s].x; b.y += wgt * vb[s].y; b.z += wgt * vb[s].z; b.w += wgt * vb[s].w;
            }
#pragma unroll 16
        for (int s = NPF; s < ns; ++s) {
            const float4 x = ld_cg_f4(src + s * ss), y = ld_cg_f4(src + s * ss + 128);
            const float wgt = wsm[s];
            a.x += wgt * x.x; a.y += wgt * x.y; a.z += wgt * x.z; a.w += wgt * x.w;
            b.x += wgt * y.x; b.y += wgt * y.y; b.z += wgt * y.z; b.w += wgt * y.w;
        }
        const float invL = 1.0f / L;
        float *dst = p.out + cu.out_off + lane * 4;
        *reinterpret_cast<float4 *>(dst) = make_float4(a.x * invL, a.y * invL, a.z * invL, a.w * invL);
        *reinterpret_cast<float4 *>(dst + 128) = make_float4(b.x * invL, b.y * invL, b.z * invL, b.w * invL);
        if (cu.lse_off >= 0 && lane == 0) p.lse[cu.lse_off] = (M + log2f(L)) * 0.6931471805599453f;
        __syncwarp();                                          // wsm is rewritten by the next unit pair
    }
}

__global__ void __cluster_dims__(2, 1, 1) __launch_bounds__(M2_THREADS, 1)
cp_decode_mla2_kernel(const DecodeParams p, const __grid_constant__ CUtensorMap tmap9,
                      const __grid_constant__ CUtensorMap tmap2, int rows_per_page)
{
    extern __shared__ __align__(1024) uint8_t smem[];
    M2Misc *mi = reinterpret_cast<M2Misc *>(smem + M2_SMEM_MISC);
    const int tid = threadIdx.x;
    const int warp = tid >> 5;
    const int lane = tid & 31;
    const uint32_t rank = cluster_ctarank();          // 0 = leader (issues the pair MMAs)
    const int pair = blockIdx.x >> 1, n_pairs = gridDim.x >> 1;
    const uint32_t q_base = smem_u32(smem + M2_SMEM_Q);
    const uint32_t st_base = smem_u32(smem + M2_SMEM_STAGE);
    const uint32_t sr_base = smem_u32(smem + M2_SMEM_SRING);
    const uint32_t p_base = smem_u32(smem + M2_SMEM_P);
    if (tid == 0) {
        for (int i = 0; i < M2_STAGES; ++i) {
            mbar_init(smem_u32(&mi->full[i]), 1); mbar_init(smem_u32(&mi->full_peer[i]), 1);
            mbar_init(smem_u32(&mi->empty[i]), 1);
        }
        for (int i = 0; i < M2_SR; ++i) {
            mbar_init(smem_u32(&mi->sl_full[i]), 1); mbar_init(smem_u32(&mi->sl_full_peer[i]), 1);
            mbar_init(smem_u32(&mi->sl_empty[i]), 1);
        }
        for (int i = 0; i < M2_SB; ++i) { mbar_init(smem_u32(&mi->s_full[i]), 1); mbar_init(smem_u32(&mi->s_empty[i]), 8); }
        for (int i = 0; i < 2; ++i) { mbar_init(smem_u32(&mi->p_full[i]), 8); mbar_init(smem_u32(&mi->p_done[i]), 1); }
        mbar_init(smem_u32(&mi->q_full), 8);
        asm volatile("prefetch.tensormap [%0];" ::"l"(reinterpret_cast<uint64_t>(&tmap9)) : "memory");
        asm volatile("prefetch.tensormap [%0];" ::"l"(reinterpret_cast<uint64_t>(&tmap2)) : "memory");
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
        fence_proxy_async();
    }
    if (warp == 1) tmem_alloc2(smem_u32(&mi->tmem_base), M2_TMEM_COLS);
    tc_fence_before();
    cluster_sync_all();                               // barriers of both CTAs initialised, TMEM allocated
    tc_fence_after();
    asm volatile("griddepcontrol.wait;" ::: "memory");    // from here on: data the previous kernel may have written
    scheduler_reset_other_set(p);
    const uint32_t tmem = mi->tmem_base;
    const int P = (int)p.page_tokens;
    const int spp = P / M2_TS;
    // leader's barriers as seen from this CTA (own address in the leader, mapped address in the peer)
    const uint32_t L_s_empty = mapa_u32(smem_u32(&mi->s_empty[0]), 0);      // + 8 b for buffer b
    const uint32_t L_p_full = mapa_u32(smem_u32(&mi->p_full[0]), 0), L_q_full = mapa_u32(smem_u32(&mi->q_full), 0);

    if (warp == 0) {
        // =========================================================== producer warp of the score ring (each CTA loads
        // its 16 tokens of every slice; the value ring has a producer of its own, warp 7: the two rings are filled at
        // their own pace -- a value stage is needed a softmax later than the score region of the same slice)
        uint64_t policy;
        asm volatile("createpolicy.fractional.L2::evict_normal.b64 %0, 1.0;" : "=l"(policy));
        uint32_t gp = 0;                                  // slice pairs issued so far (ring position)
        const int ppp = P / (2 * M2_TS);                  // slice pairs per page (pages hold 64 k tokens: a pair never straddles)
        for (int k = 0;; ++k) {
            const M2Item it = m2_item(p, pair + k * n_pairs);
            if (!it.valid) break;
            const int np = (it.n_slices + 1) >> 1;
            int32_t pid_nx = 0;                               // page ids one batch of 32 pairs ahead
            if (lane < np) pid_nx = page_of(p, it.req, it.page_begin + lane / ppp);
            for (int q0 = 0; q0 < np; q0 += 32) {
                const int32_t pid = pid_nx;
                pid_nx = 0;
                if (q0 + 32 + lane < np) pid_nx = page_of(p, it.req, it.page_begin + (q0 + 32 + lane) / ppp);
                const int nq = min(32, np - q0);
                for (int j = 0; j < nq; ++j) {
                    const int32_t my = __shfl_sync(0xffffffffu, pid, j);
                    const int i = q0 + j;                                  // pair of the tile
                    // The rings hold ~5 slices per CTA (every slice is staged twice: K-major for the scores, MN-major
                    // for the values) and an HBM round trip under load is ~2 us, which bounds a slice at ~0.48 us
                    // whatever the MMAs do.  So each CTA asks for its half of the tokens M2_PF pairs ahead to be
                    // brought into L2 (the rows are contiguous: one bulk prefetch per slice), and the TMA loads of both
                    // rings find their data at L2 latency.
                    {
                        const int t = j + M2_PF;
                        const int32_t pg = __shfl_sync(0xffffffffu, t < 32 ? pid : pid_nx, t & 31);
                        if (i + M2_PF < np && lane < 2) {
                            const int rowp = pg * rows_per_page + ((i + M2_PF) % ppp) * 2 * M2_TS + lane * M2_TS + 16 * (int)rank;
                            bulk_prefetch_l2(p.arena + (size_t)rowp * (M2_DK * 2), 16 * M2_DK * 2);
                        }
                    }
                    const uint32_t gq = gp + (uint32_t)i, reg = gq % M2_SR;
                    mbar_wait(smem_u32(&mi->sl_empty[reg]), ((gq / M2_SR) & 1) ^ 1);
                    if (elect_one()) {
                        // score region of the pair: this CTA's 16 tokens of each of the two slices, all 9 column blocks,
                        // with ONE 4-D box {64 columns, 16 tokens, 2 slices, 9 blocks}: block kb of slice h lands at
                        // kb * 4096 + h * 2048, i.e. the four 8-token groups of a block are 1024 B apart, which is what
                        // lets one N = 64 MMA take both slices.  (A tile's last pair may hold one slice: the second half
                        // of the page is loaded anyway and never looked at.)
                        const int row0 = my * rows_per_page + (i % ppp) * 2 * M2_TS;
                        const uint32_t sb = smem_u32(&mi->sl_full[reg]);
                        mbar_arrive_expect_tx(sb, M2_SPAIR);
                        tma_load_4d(sr_base + reg * M2_SPAIR, &tmap9, 0, row0 + 16 * (int)rank, 0, 0, sb, policy);
                    }
                }
            }
            gp += (uint32_t)np;
        }
        // programmatic dependent launch: see cp_kernels_kvt.cu (the next kernel's set-up overlaps this one's tail;
        // said once every slice of this CTA has been requested, not at the top)
        if (lane == 0) asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
    } else if (warp == 1 && rank != 0) {
        // =========================================================== peer: relay "my part of the slice landed"
        uint32_t gp = 0;
        for (int k = 0;; ++k) {
            const M2Item it = m2_item(p, pair + k * n_pairs);
            if (!it.valid) break;
            const int np = (it.n_slices + 1) >> 1;
            for (int i = 0; i < np; ++i) {
                const uint32_t gq = gp + (uint32_t)i, reg = gq % M2_SR;
                mbar_wait(smem_u32(&mi->sl_full[reg]), (gq / M2_SR) & 1);
                if (lane == 0) mbar_arrive_cluster(mapa_u32(smem_u32(&mi->sl_full_peer[reg]), 0));
                __syncwarp();
            }
            gp += (uint32_t)np;
        }
    } else if (warp == 6 && rank != 0) {
        // =========================================================== peer: relay "my part of the value stage landed"
        uint32_t gs = 0;
        for (int k = 0;; ++k) {
            const M2Item it = m2_item(p, pair + k * n_pairs);
            if (!it.valid) break;
            for (int i = 0; i < it.n_slices; ++i, ++gs) {
                const uint32_t slot = gs % M2_STAGES;
                mbar_wait(smem_u32(&mi->full[slot]), (gs / M2_STAGES) & 1);
                if (lane == 0) mbar_arrive_cluster(mapa_u32(smem_u32(&mi->full_peer[slot]), 0));
                __syncwarp();
            }
        }
    } else if (warp == 7) {
        // =========================================================== producer warp of the value ring
        uint64_t policy;
        asm volatile("createpolicy.fractional.L2::evict_normal.b64 %0, 1.0;" : "=l"(policy));
        uint32_t gs = 0;
        for (int k = 0;; ++k) {
            const M2Item it = m2_item(p, pair + k * n_pairs);
            if (!it.valid) break;
            for (int s0 = 0; s0 < it.n_slices; s0 += 32) {
                int32_t pid = 0;
                if (s0 + lane < it.n_slices) pid = page_of(p, it.req, it.page_begin + (s0 + lane) / spp);
                const int ns = min(32, it.n_slices - s0);
                for (int j = 0; j < ns; ++j, ++gs) {
                    const int32_t my = __shfl_sync(0xffffffffu, pid, j);
                    const int i = s0 + j;
                    const uint32_t slot = gs % M2_STAGES;
                    mbar_wait(smem_u32(&mi->empty[slot]), ((gs / M2_STAGES) & 1) ^ 1);
                    if (elect_one()) {
                        const int row0 = my * rows_per_page + (i % spp) * M2_TS;
                        // tokens 16kk.., this CTA's column blocks 4j + 2r, 4j + 2r + 1
                        const uint32_t fb = smem_u32(&mi->full[slot]);
                        mbar_arrive_expect_tx(fb, M2_STAGE_BYTES);
                        const uint32_t dst = st_base + slot * M2_STAGE_BYTES;
#pragma unroll
                        for (int kk = 0; kk < 2; ++kk)
#pragma unroll
                            for (int jj = 0; jj < 2; ++jj)
                                tma_load_3d(dst + (kk * 2 + jj) * 2 * M2_BLK, &tmap2, 0, row0 + 16 * kk,
                                            4 * jj + 2 * (int)rank, fb, policy);
                    }
                }
            }
        }
    } else if (warp == 1) {
        // =========================================================== leader: issuer of the score MMAs
        // One N = 64 MMA per k-step computes the scores of a PAIR of slices (measured: a score MMA costs ~19 cycles
        // whether N is 32 or 64 -- it is bound by the A operand, not by the arithmetic -- so pairing halves the 36
        // instructions per slice that used to pace the whole kernel).  Each CTA supplies 32 B rows: its 16 tokens of
        // slice 0, then of slice 1; D columns 0..15 (per lane half) are slice 0, 16..31 slice 1.  A tile's last
        // pair may hold one slice: the other half of the region is stale, its score columns are never read.
        constexpr uint32_t IDESC_S = umma_idesc_bf16(128, 2 * M2_TS, 0, 0);
        uint32_t gp = 0, qn = 0;
        int prev_group = -1;
        for (int k = 0;; ++k) {
            const M2Item it = m2_item(p, pair + k * n_pairs);
            if (!it.valid) break;
            if (it.group_idx != prev_group) { mbar_wait_cluster(smem_u32(&mi->q_full), qn & 1); ++qn; prev_group = it.group_idx; }
            const int np = (it.n_slices + 1) >> 1;
            for (int i = 0; i < np; ++i) {
                const uint32_t gq = gp + (uint32_t)i, reg = gq % M2_SR, b = gq % M2_SB;
                mbar_wait(smem_u32(&mi->sl_full[reg]), (gq / M2_SR) & 1);
                mbar_wait_cluster(smem_u32(&mi->sl_full_peer[reg]), (gq / M2_SR) & 1);
                mbar_wait_cluster(smem_u32(&mi->s_empty[b]), ((gq / M2_SB) & 1) ^ 1);
                tc_fence_after();
                if (elect_one()) {
                    const uint32_t c0 = sr_base + reg * M2_SPAIR;
                    const uint32_t dcol = tmem + M2_TMEM_S + 32 * b;
                    const uint64_t bd0 = umma_smem_desc(c0, 16, 1024, 2);
                    const uint64_t ad0 = umma_smem_desc(q_base, 16, 1024, 2);
#pragma unroll
                    for (int kb = 0; kb < M2_KB; ++kb)
#pragma unroll
                        for (int j = 0; j < 4; ++j) {
                            const uint64_t bd = bd0 + (uint64_t)((kb * 2 * M2_BLK + j * 32) >> 4);      // start-address field
                            if (kb < M2_KB_TMEM) {
                                umma2_bf16_ts(dcol, tmem + M2_TMEM_Q + kb * 32 + j * 8, bd, IDESC_S, (kb | j) != 0);
                            } else {
                                const uint64_t ad = ad0 + (uint64_t)(((kb - M2_KB_TMEM) * M2_QBLK + j * 32) >> 4);
                                umma2_bf16_ss(dcol, ad, bd, IDESC_S, 1);
                            }
                        }
                    umma2_commit(smem_u32(&mi->s_full[b]));
                    umma2_commit(smem_u32(&mi->sl_empty[reg]));
                }
                __syncwarp();
            }
            gp += (uint32_t)np;
        }
    } else if (warp == 6 && rank == 0) {
        // =========================================================== leader: issuer of the value MMAs
        // (a warp of its own: neither issuer waits for what only the other one needs, and a commit covers the MMAs of
        // the thread that makes it)
        constexpr uint32_t IDESC_PV = umma_idesc_bf16(128, 256, 0, 1);
        uint32_t gs = 0;
        for (int k = 0;; ++k) {
            const M2Item it = m2_item(p, pair + k * n_pairs);
            if (!it.valid) break;
            const int n = it.n_slices;
            for (int i = 0; i < n; ++i) {
                const uint32_t g = gs + (uint32_t)i, slot = g % M2_STAGES;
                mbar_wait(smem_u32(&mi->full[slot]), (g / M2_STAGES) & 1);
                mbar_wait_cluster(smem_u32(&mi->full_peer[slot]), (g / M2_STAGES) & 1);
                mbar_wait_cluster(smem_u32(&mi->p_full[g & 1]), (g >> 1) & 1);
                tc_fence_after();
                if (elect_one()) {
                    const uint32_t pv = st_base + slot * M2_STAGE_BYTES;
                    const uint64_t ad0 = umma_smem_desc(p_base + (g & 1) * M2_P_BYTES, 1024, 128, 0);
                    const uint64_t bd0 = umma_smem_desc(pv, M2_BLK, 1024, 2);
#pragma unroll
                    for (int kk = 0; kk < 2; ++kk)
#pragma unroll
                        for (int jj = 0; jj < 2; ++jj) {
                            // P: 8-token chunks of [64 rows x 16 B] 1024 B apart, 8-row groups 128 B apart
                            const uint64_t ad = ad0 + (uint64_t)((kk * 2048) >> 4);
                            // V: two 64-column blocks 2048 B apart, 8-token groups 1024 B apart
                            const uint64_t bd = bd0 + (uint64_t)(((kk * 2 + jj) * 2 * M2_BLK) >> 4);
                            umma2_bf16_ss(tmem + jj * 128, ad, bd, IDESC_PV, (i > 0) || (kk > 0));
                        }
                    umma2_commit(smem_u32(&mi->empty[slot]));
                    umma2_commit(smem_u32(&mi->p_done[g & 1]));
                }
                __syncwarp();
            }
            gs += (uint32_t)n;
        }
    } else {
        // =========================================================== softmax warps
        // thread = TMEM lane L: head (rank * 64 + L % 64), token half L / 64 of every slice
        const int q4 = warp & 3;
        const int L = q4 * 32 + lane;
        const int hrow = L & 63;                          // row inside this CTA
        const int head = (int)rank * 64 + hrow;
        const int th = L >> 6;                            // token half: tokens 16 th .. 16 th + 15 of a slice
        const uint32_t tl = tmem + ((uint32_t)(q4 * 32) << 16);
        const int st = tid - 64;
        uint32_t gs = 0, gp = 0;
        int prev_group = -1;
        for (int k = 0;; ++k) {
            const M2Item it = m2_item(p, pair + k * n_pairs);
            if (!it.valid) break;
            if (it.group_idx != prev_group) {
                // stage this CTA's 64 query rows.  Column blocks 0..5 go to tensor memory as the A operand of
                // the TS-mode score MMAs: lane = row, two bf16 per 32-bit column, and for a pair MMA the rows
                // are duplicated in lanes 64..127 -- exactly this thread layout (row = L % 64).  Blocks 6..8 go
                // to shared memory as K-major [64 x 64] tiles with the 128-byte swizzle.  Rows >= Hq are zero.
                prev_group = it.group_idx;
                {
                    const uint4 *qr = reinterpret_cast<const uint4 *>(p.q + it.q_off + (int64_t)head * M2_DK);
                    const bool live = head < it.n_heads;
                    for (int c0 = 0; c0 < M2_KB_TMEM * 32; c0 += 96) {    // 96 columns = 192 bf16 = 24 x 16 B in flight
                        uint4 v[24];
#pragma unroll
                        for (int i = 0; i < 24; ++i) {
                            v[i] = make_uint4(0u, 0u, 0u, 0u);
                            if (live) v[i] = __ldg(qr + c0 / 4 + i);
                        }
#pragma unroll
                        for (int b6 = 0; b6 < 6; ++b6) {
                            uint32_t w[16];
#pragma unroll
                            for (int v4 = 0; v4 < 4; ++v4) {
                                w[4 * v4] = v[4 * b6 + v4].x; w[4 * v4 + 1] = v[4 * b6 + v4].y;
                                w[4 * v4 + 2] = v[4 * b6 + v4].z; w[4 * v4 + 3] = v[4 * b6 + v4].w;
                            }
                            tmem_st16(tl + M2_TMEM_Q + c0 + b6 * 16, w);
                        }
                    }
                    tmem_wait_st();
                }
                {
                    constexpr int CPR = (M2_KB - M2_KB_TMEM) * 8;        // 16-B chunks per row in shared memory
                    const uint4 *qg = reinterpret_cast<const uint4 *>(p.q + it.q_off) + (int64_t)rank * 64 * (M2_DK / 8);
#pragma unroll 12
                    for (int id = st; id < 64 * CPR; id += 128) {
                        const int r = id / CPR, ch = id % CPR;
                        uint4 v = make_uint4(0u, 0u, 0u, 0u);
                        if ((int)rank * 64 + r < it.n_heads) v = __ldg(qg + r * (M2_DK / 8) + M2_KB_TMEM * 8 + ch);
                        const uint32_t a = q_base + (ch >> 3) * M2_QBLK + r * 128 + (((ch & 7) ^ (r & 7)) << 4);
                        asm volatile("st.shared.v4.b32 [%0], {%1,%2,%3,%4};" ::"r"(a), "r"(v.x), "r"(v.y), "r"(v.z), "r"(v.w) : "memory");
                    }
                }
                tc_fence_before();
                fence_proxy_async();
                __syncwarp();
                if (lane == 0) mbar_arrive_cluster(L_q_full);
            }
            float m_run = -INFINITY, l_run = 0.f;
            const int n = it.n_slices;
            for (int i = 0; i < n; ++i) {
                const uint32_t g = gs + (uint32_t)i, xb = g & 1;
                const uint32_t gq = gp + (uint32_t)(i >> 1), b = gq % M2_SB;       // the slice's pair and its score buffer
                if ((i & 1) == 0) mbar_wait(smem_u32(&mi->s_full[b]), (gq / M2_SB) & 1);
                tc_fence_after();
                uint32_t sr[16];
                tmem_ld16(tl + M2_TMEM_S + 32 * b + 16 * (i & 1), sr);
                tmem_wait_ld();
                tc_fence_before();
                __syncwarp();
                if (lane == 0 && ((i & 1) || i == n - 1)) mbar_arrive_cluster(L_s_empty + 8 * b);   // both slices read
                const int valid = ((i == n - 1) ? it.valid_last : M2_TS) - 16 * th;   // valid tokens of my half
                float mx = -INFINITY;
#pragma unroll
                for (int j = 0; j < 16; ++j) {
                    const float v = j < valid ? __uint_as_float(sr[j]) * it.scale_log2 : -INFINITY;
                    sr[j] = __float_as_uint(v);
                    mx = fmaxf(mx, v);
                }
                // the two token halves of a head agree on the row maximum through shared memory
                mi->xmax[xb][L] = mx;
                asm volatile("bar.sync 2, 128;" ::: "memory");
                mx = fmaxf(mx, mi->xmax[xb][L ^ 64]);
                const float m_new = (mx > m_run + M2_LAZY_LOG2) ? mx : m_run;
                const bool need = (m_new != m_run) && i > 0;
                const float a_resc = ex2_ftz(m_run - m_new);
                if (m_new != m_run) { l_run *= a_resc; m_run = m_new; }
                uint32_t pw[8];
                float sum = 0.f;
#pragma unroll
                for (int j = 0; j < 8; ++j) {
                    const float p0 = ex2_ftz(__uint_as_float(sr[2 * j]) - m_run), p1 = ex2_ftz(__uint_as_float(sr[2 * j + 1]) - m_run);
                    sum += p0 + p1;
                    asm("cvt.rn.bf16x2.f32 %0, %1, %2;" : "=r"(pw[j]) : "f"(p1), "f"(p0));
                }
                l_run += sum;
                mbar_wait(smem_u32(&mi->p_done[xb]), ((g >> 1) & 1) ^ 1);       // P buffer (slice & 1) free
                if (__any_sync(0xffffffffu, need)) {
                    // O is rescaled in place: the value MMAs of the previous slice must be complete
                    mbar_wait(smem_u32(&mi->p_done[(g - 1) & 1]), ((g - 1) >> 1) & 1);
                    tc_fence_after();
                    const float a = need ? a_resc : 1.f;
                    for (int c = 0; c < 256; c += 16) {
                        uint32_t o[16];
                        tmem_ld16(tl + c, o);
                        tmem_wait_ld();
#pragma unroll
                        for (int j = 0; j < 16; ++j) o[j] = __float_as_uint(__uint_as_float(o[j]) * a);
                        tmem_st16(tl + c, o);
                    }
                    tmem_wait_st();
                }
                // P[row][token] as 8-token chunks of [64 rows x 16 B]: chunk c at c * 1024 + row * 16
                asm volatile("st.shared.v4.b32 [%0], {%1,%2,%3,%4};" ::"r"(p_base + xb * M2_P_BYTES + (2 * th) * 1024 + hrow * 16), "r"(pw[0]), "r"(pw[1]), "r"(pw[2]), "r"(pw[3]) : "memory");
                asm volatile("st.shared.v4.b32 [%0], {%1,%2,%3,%4};" ::"r"(p_base + xb * M2_P_BYTES + (2 * th + 1) * 1024 + hrow * 16), "r"(pw[4]), "r"(pw[5]), "r"(pw[6]), "r"(pw[7]) : "memory");
                if (i == n - 1 && it.valid_last < M2_TS) {
                    // dead slots of the request's last slice may hold NaN: zero their value rows in the PV area
                    // (warp q4 clears the two 64-column blocks of MMA j = q4 & 1 for k-step kk = q4 >> 1)
                    const int kk = q4 >> 1, jj = q4 & 1;
                    const int vrows = min(16, max(0, it.valid_last - 16 * kk));        // valid rows of this k-step
                    const uint32_t blk = st_base + (g % M2_STAGES) * M2_STAGE_BYTES + (kk * 2 + jj) * 2 * M2_BLK;
                    for (int e = lane; e < (16 - vrows) * 16; e += 32) {
                        const int r = vrows + (e >> 4), ch = e & 15;
                        asm volatile("st.shared.v4.b32 [%0], {%1,%1,%1,%1};" ::"r"(blk + (ch >> 3) * M2_BLK + r * 128 + (((ch & 7) ^ (r & 7)) << 4)), "r"(0u) : "memory");
                    }
                }
                fence_proxy_async();
                tc_fence_before();
                __syncwarp();
                if (lane == 0) mbar_arrive_cluster(L_p_full + 8 * xb);
            }
            gs += (uint32_t)n;
            gp += (uint32_t)(n + 1) >> 1;

            // ---- end of tile: O rows from TMEM, publish
            {
                const uint32_t gl = gs - 1;
                mbar_wait(smem_u32(&mi->p_done[gl & 1]), (gl >> 1) & 1);
                tc_fence_after();
                mi->xsum[L] = l_run;
                asm volatile("bar.sync 2, 128;" ::: "memory");
                const float l_tot = th == 0 ? l_run + mi->xsum[L ^ 64] : mi->xsum[L ^ 64] + l_run;   // same order in both halves
                const bool final_out = it.n_splits == 1;
                const float inv = final_out ? 1.f / l_tot : 1.f;
                // Rows leave through a per-warp transpose in shared memory: a thread owns a row in TMEM, but 32 lanes storing 16 B each into 32 different
                // rows is the worst pattern for L2; after the transpose every store instruction writes
                // 8 rows x 64 contiguous bytes.
                const int head0 = (int)rank * 64 + (q4 & 1) * 32;            // first head of this warp's 32 rows
                const int64_t rstride = final_out ? M2_DV : (int64_t)it.n_splits * M2_DV;
                float *row0 = final_out ? p.out + it.out_off + (int64_t)head0 * M2_DV
                                        : p.workspace + it.part_off + part_o_off(head0, it.split, it.n_splits, M2_DV);
                const uint32_t scr = smem_u32(smem + M2_SMEM_XPOSE) + (uint32_t)(warp - 2) * M2_XPOSE_WARP;   // [32 rows][32 floats + 4 pad]
                for (int c = 0; c < 256; c += 32) {
                    // 32 columns per pass (two tcgen05.ld in flight, one wait): a pass is a chain of dependent TMEM,
                    // shared-memory and global accesses, and 16 passes of 16 columns took 3.4 us without any store
                    uint32_t o[32];
                    tmem_ld16(tl + c, *reinterpret_cast<uint32_t (*)[16]>(&o[0]));
                    tmem_ld16(tl + c + 16, *reinterpret_cast<uint32_t (*)[16]>(&o[16]));
                    tmem_wait_ld();
                    __syncwarp();                                            // previous pass fully read back
#pragma unroll
                    for (int j = 0; j < 32; j += 4)
                        asm volatile("st.shared.v4.f32 [%0], {%1,%2,%3,%4};" ::"r"(scr + lane * 144 + j * 4),
                                     "f"(__uint_as_float(o[j]) * inv), "f"(__uint_as_float(o[j + 1]) * inv),
                                     "f"(__uint_as_float(o[j + 2]) * inv), "f"(__uint_as_float(o[j + 3]) * inv) : "memory");
                    __syncwarp();
                    // TMEM column c of MMA jj = c / 128 holds value column 256 jj + 128 th + c % 128
                    const int col = 256 * (c >> 7) + 128 * th + (c & 127) + (lane & 7) * 4;
#pragma unroll
                    for (int r4 = 0; r4 < 8; ++r4) {
                        const int r = r4 * 4 + (lane >> 3);                   // a store instruction: 4 rows x 128 contiguous bytes
                        float4 v;
                        asm volatile("ld.shared.v4.f32 {%0,%1,%2,%3}, [%4];" : "=f"(v.x), "=f"(v.y), "=f"(v.z), "=f"(v.w)
                                     : "r"(scr + r * 144 + (lane & 7) * 16) : "memory");
                        if (head0 + r < it.n_heads) __stcg(reinterpret_cast<float4 *>(row0 + r * rstride + col), v);
                    }
                }
                tc_fence_before();
                if (th == 0 && head < it.n_heads) {
                    if (final_out)
                        p.lse[it.lse_off + head] = (m_run + log2f(l_tot)) * 0.6931471805599453f;
                    else
                        __stcg(reinterpret_cast<float2 *>(p.workspace + it.part_off +
                                                          part_ml_off(it.n_heads, head, it.split, it.n_splits, M2_DV)),
                               make_float2(m_run, l_tot));
                }
                if (!final_out) {
                    __syncwarp();
                    if (lane == 0) red_release_add(p.group_counters + (size_t)it.group_idx * kCounterStride, 1);
                }
            }
        }
    }
    // ---- LSE combine (step a4): warp-sized units, statically assigned to ALL warps of every CTA.
    // The barrier orders it after this CTA's last tile (every slice consumed, every MMA complete),
    // so the slice stages can serve as the warps' scratch.
    __syncthreads();
    {
        float *wsm = reinterpret_cast<float *>(smem + M2_SMEM_STAGE) + warp * kMaxSplits;
        m2_combine(p, blockIdx.x * M2_WARPS + warp, gridDim.x * M2_WARPS, wsm, lane);
    }
    tc_fence_before();
    cluster_sync_all();
    if (warp == 1) tmem_dealloc2(tmem, M2_TMEM_COLS);
}

// ----------------------------------------------------------------------------- host side
// Views of the arena as 64-column blocks of rows of 576 bf16.
bool make_mla2_tensor_maps(void *out_map9, void *out_map2, const void *arena, uint64_t total_rows)
{
    typedef CUresult (*EncodeTiledFn)(CUtensorMap *, CUtensorMapDataType, cuuint32_t, void *, const cuuint64_t *,
                                      const cuuint64_t *, const cuuint32_t *, const cuuint32_t *,
                                      CUtensorMapInterleave, CUtensorMapSwizzle, CUtensorMapL2promotion,
                                      CUtensorMapFloatOOBfill);
    void *ptr = nullptr;
    cudaDriverEntryPointQueryResult qres;
    if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &ptr, cudaEnableDefault, &qres) != cudaSuccess ||
        qres != cudaDriverEntryPointSuccess)
        return false;
    EncodeTiledFn fn = reinterpret_cast<EncodeTiledFn>(ptr);
    {
        // value operand: {64 columns, rows of 576 bf16, column blocks}, boxes of 16 tokens x 2 blocks
        cuuint64_t dims[3] = {64, total_rows, (cuuint64_t)M2_KB};
        cuuint64_t strides[2] = {(cuuint64_t)M2_DK * 2, 128};
        cuuint32_t estr[3] = {1, 1, 1};
        cuuint32_t box[3] = {64, 16, 2};
        CUresult r = fn(reinterpret_cast<CUtensorMap *>(out_map2), CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 3,
                        const_cast<void *>(arena), dims, strides, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE,
                        CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
        if (r != CUDA_SUCCESS) return false;
    }
    {
        // score operand: {64 columns, rows, slice of a pair (32 rows further), column blocks}, one box of
        // 16 tokens x 2 slices x 9 blocks per slice pair and CTA
        cuuint64_t dims[4] = {64, total_rows, 2, (cuuint64_t)M2_KB};
        cuuint64_t strides[3] = {(cuuint64_t)M2_DK * 2, (cuuint64_t)M2_TS * M2_DK * 2, 128};
        cuuint32_t estr[4] = {1, 1, 1, 1};
        cuuint32_t box[4] = {64, 16, 2, (cuuint32_t)M2_KB};
        CUresult r = fn(reinterpret_cast<CUtensorMap *>(out_map9), CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 4,
                        const_cast<void *>(arena), dims, strides, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE,
                        CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
        if (r != CUDA_SUCCESS) return false;
    }
    return true;
}

cudaError_t launch_decode_mla2(const DecodeParams &p, const void *tmap9, const void *tmap2, int rows_per_page,
                               int n_ctas, cudaStream_t stream)
{
    static bool configured[64] = {};              // per device: the attribute belongs to the device's copy of the function
    int dev = 0;
    if (cudaGetDevice(&dev) != cudaSuccess) return cudaGetLastError();
    if (dev < 0 || dev >= 64 || !configured[dev]) {
        cudaError_t e = cudaFuncSetAttribute(cp_decode_mla2_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                             M2_SMEM_BYTES);
        if (e != cudaSuccess) return e;
        if (dev >= 0 && dev < 64) configured[dev] = true;
    }
    int pairs = p.n_tiles;
    if (pairs < (p.n_combine_units + 7) / 8) pairs = (p.n_combine_units + 7) / 8;
    if (pairs > n_ctas / 2) pairs = n_ctas / 2;
    if (pairs < 1) pairs = 1;
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3((unsigned)(2 * pairs)); cfg.blockDim = dim3(M2_THREADS); cfg.dynamicSmemBytes = M2_SMEM_BYTES; cfg.stream = stream;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = attr; cfg.numAttrs = 1;
    return cudaLaunchKernelEx(&cfg, cp_decode_mla2_kernel, p, *reinterpret_cast<const CUtensorMap *>(tmap9),
                              *reinterpret_cast<const CUtensorMap *>(tmap2), rows_per_page);
}

}  // namespace cp
