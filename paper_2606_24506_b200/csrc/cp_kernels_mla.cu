// cp_kernels_mla.cu -- the MLA latent path of libcrosspool (hot-path steps a2, a3', a4-a6 for
// kind CP_KIND_MLA with a 576-wide latent row, value = its first 512 entries, Hq <= 128):
// ONE persistent launch per decode step, tcgen05 tensor-core MMA with accumulators in TMEM.
//
// 128 query heads against one shared latent row per token is a real dense contraction
// (241 flop per KV byte), so here -- and only here -- the 5th-generation tensor cores are used:
//     S[128 x 32]   = Q[128 x 576] . C_slice^T      36 x tcgen05.mma M128 N32  K16 (A, B K-major)
//     O[128 x 256] += P[128 x 32]  . C_slice[:, half]  2 x tcgen05.mma M128 N256 K16 (B MN-major)
// per 32-token slice of a page.  TMEM holds 512 fp32 columns per SM; O[128 x 512] alone would fill
// it, so one work item is (tile, value half): 256 O columns (TMEM columns 0..255), two score
// buffers (256.., 288..) and, in the remaining 192 columns, six of the nine 64-column blocks of Q
// as the A operand of TS-mode MMAs (measured: an SS-mode MMA re-reads its 4 KB A tile from shared
// memory, ~70 cycles whatever N is; A from tensor memory costs ~16 at N = 32).  The two halves of
// a tile are adjacent work items, popped by different CTAs at about the same time, so the second
// reader of a page hits L2 (DESIGN.md §6.3 states the cost: the QK^T part is computed twice).
//
// Warp roles (192 threads, 1 CTA/SM):
//   warp 0      producer: pops work items, translates logical pages through the page table
//               (step a2) and streams 32-token slices into a 4-stage ring with one 3-D TMA
//               box each (9 swizzled [32 x 64] tiles), mbarrier complete_tx.
//   warp 1      MMA issuer (one lane chosen by elect.sync): S_{i+1} is issued before P_i V_i so the tensor
//               pipe computes the next scores while the softmax warps work on the current ones.
//   warps 2..5  softmax: thread = one query head = one TMEM lane, so the row maximum and row
//               sum need no shuffles; online softmax in fp32 (log2 units) with a lazy reference
//               update; P is written as bf16 to shared memory for the second MMA; at the end
//               of a tile they read O from TMEM and publish the result or the split partial.
//               After the last tile the same warps run the LSE combine units (step a4).
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

constexpr int MLA_DK = 576;                         // latent row width (512 latent + 64 rope)
constexpr int MLA_DV = 512;                         // value = first 512 entries of the row
constexpr int MLA_HALF = 256;                       // value columns per work item
constexpr int MLA_M = 128;                          // query heads = MMA M = TMEM lanes
constexpr int MLA_TS = 32;                          // tokens per slice = MMA N of the score MMA
constexpr int MLA_KB = MLA_DK / 64;                 // 9 column blocks of 64 (128 B, one swizzle row)
constexpr int MLA_STAGES = 4;
constexpr int MLA_STAGE_BYTES = MLA_TS * MLA_DK * 2;        // 36864
constexpr int MLA_BLK_BYTES = MLA_TS * 128;                 // one [32 x 64] swizzled tile: 4096
constexpr int MLA_KB_TMEM = 6;                      // query column blocks 0..5 live in TMEM (A operand, TS mode)
constexpr int MLA_Q_BYTES = (MLA_KB - MLA_KB_TMEM) * MLA_M * 128;   // 49152: blocks 6..8 of [128 x 64] in shared memory
constexpr int MLA_QBLK_BYTES = MLA_M * 128;                 // 16384
constexpr int MLA_P_BYTES = MLA_M * MLA_TS * 2;             // 8192, one P buffer
constexpr int MLA_THREADS = 192;
constexpr int MLA_TQ = 2;                           // work-item queue depth
constexpr int MLA_SMEM_Q = 0;
constexpr int MLA_SMEM_STAGE = MLA_Q_BYTES;
constexpr int MLA_SMEM_P = MLA_SMEM_STAGE + MLA_STAGES * MLA_STAGE_BYTES;
constexpr int MLA_SMEM_MISC = MLA_SMEM_P + MLA_P_BYTES;         // barriers, queue, tmem address
constexpr int MLA_SMEM_BYTES = MLA_SMEM_MISC + 1024;
static_assert(MLA_SMEM_BYTES <= 232448, "MLA kernel exceeds the 227 KB shared-memory limit");
constexpr uint32_t MLA_TMEM_COLS = 512;
constexpr uint32_t MLA_TMEM_S0 = 256, MLA_TMEM_S1 = 288;       // two score buffers of MLA_TS columns
constexpr uint32_t MLA_TMEM_Q = 320;                           // 192 columns: Q[:, 0:384) as bf16 pairs
static_assert(MLA_TMEM_Q + MLA_KB_TMEM * 32 <= MLA_TMEM_COLS, "TMEM budget");
constexpr float MLA_LAZY_LOG2 = 8.0f;

// What the producer hands to the other warps for one work item.
struct MlaDesc {
    int32_t item;            // work index; < 0: no more work
    int32_t group_idx;
    int32_t n_slices;        // MLA_TS-token slices of the tile
    int32_t valid_last;      // valid tokens of the last slice (1..MLA_TS)
    int32_t split, n_splits;
    int32_t half;            // value half (0: columns 0..255, 1: 256..511)
    int32_t n_heads;         // Hq
    int32_t load_q;          // the query block differs from the one resident in shared memory
    float scale_log2;
    int64_t q_off, out_off, lse_off, part_off;
};

// Shared-memory bookkeeping block (at MLA_SMEM_MISC)
struct MlaMisc {
    uint64_t full[MLA_STAGES], empty[MLA_STAGES];       // slice ring: TMA -> MMA, MMA -> TMA
    uint64_t s_full[2], s_empty[2];                     // score buffers in TMEM: MMA -> softmax -> MMA
    uint64_t p_full, p_done;                            // P buffer in smem: softmax -> MMA; MMA done reading
    uint64_t q_full;                                    // query block staged (softmax warps -> MMA)
    uint64_t tq_full[MLA_TQ], tq_empty[MLA_TQ];         // work-item queue
    MlaDesc tq[MLA_TQ];
    uint32_t tmem_base;
};
static_assert(sizeof(MlaMisc) <= 1024, "MlaMisc must fit its reserved kilobyte");

__global__ void __launch_bounds__(MLA_THREADS, 1)
cp_decode_mla_kernel(const DecodeParams p, const __grid_constant__ CUtensorMap tmap, int rows_per_page)
{
    extern __shared__ __align__(1024) uint8_t smem[];
    MlaMisc *mi = reinterpret_cast<MlaMisc *>(smem + MLA_SMEM_MISC);
    const int tid = threadIdx.x;
    const int warp = tid >> 5;
    const int lane = tid & 31;
    const uint32_t q_base = smem_u32(smem + MLA_SMEM_Q);
    const uint32_t st_base = smem_u32(smem + MLA_SMEM_STAGE);
    const uint32_t p_base = smem_u32(smem + MLA_SMEM_P);
    scheduler_reset_other_set(p);

    if (tid == 0) {
        for (int i = 0; i < MLA_STAGES; ++i) { mbar_init(smem_u32(&mi->full[i]), 1); mbar_init(smem_u32(&mi->empty[i]), 1); }
        for (int i = 0; i < 2; ++i) {
            mbar_init(smem_u32(&mi->s_full[i]), 1); mbar_init(smem_u32(&mi->s_empty[i]), 4);
        }
        mbar_init(smem_u32(&mi->p_full), 4); mbar_init(smem_u32(&mi->p_done), 1);
        mbar_init(smem_u32(&mi->q_full), 4);
        for (int i = 0; i < MLA_TQ; ++i) { mbar_init(smem_u32(&mi->tq_full[i]), 1); mbar_init(smem_u32(&mi->tq_empty[i]), 5); }
        asm volatile("prefetch.tensormap [%0];" ::"l"(reinterpret_cast<uint64_t>(&tmap)) : "memory");
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
        fence_proxy_async();
    }
    if (warp == 1) tmem_alloc(smem_u32(&mi->tmem_base), MLA_TMEM_COLS);
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    const uint32_t tmem = mi->tmem_base;
    const int P = (int)p.page_tokens;
    const int spp = P / MLA_TS;                       // slices per page

    if (warp == 0) {
        // =========================================================== producer warp
        uint64_t policy;
        asm volatile("createpolicy.fractional.L2::evict_normal.b64 %0, 1.0;" : "=l"(policy));
        uint32_t gs = 0;          // slices issued by this CTA (ring position)
        uint32_t qi = 0;          // work items pushed
        int resident_group = -1;  // group whose query block is in shared memory
        const int n_work = 2 * p.n_tiles;             // (tile, value half)
        for (;;) {
            int work = 0;
            if (lane == 0) work = atomicAdd(p.work_counter, 1);
            work = __shfl_sync(0xffffffffu, work, 0);
            const int item = work < n_work ? work : -1;
            Tile tile = Tile{0, 0, 0, 0};
            Group g;
            g.req = 0; g.model = 0; g.kv_head = 0; g.n_splits = 1; g.n_pages = 0; g.batch_index = 0;
            g.q_off = g.out_off = g.lse_off = g.part_off = 0;
            int ctx = 0, nheads = 0;
            float scale_log2 = 0.f;
            int n_slices = 0, valid_last = MLA_TS;
            if (item >= 0) {
                tile = p.tiles[item >> 1];
                g = p.groups[tile.group];
                const DevModel m = p.models[g.model];
                nheads = m.n_q_heads; scale_log2 = m.scale_log2;
                ctx = __ldg(p.req_ctx + g.req);
                const int t_begin = tile.page_begin * P;
                const int t_end = min(tile.page_end * P, ctx);
                n_slices = (t_end - t_begin + MLA_TS - 1) / MLA_TS;
                valid_last = t_end - t_begin - (n_slices - 1) * MLA_TS;
            }
            const uint32_t qs = qi % MLA_TQ;
            mbar_wait(smem_u32(&mi->tq_empty[qs]), ((qi / MLA_TQ) & 1) ^ 1);
            if (lane == 0) {
                MlaDesc d;
                d.item = item; d.group_idx = tile.group; d.n_slices = n_slices; d.valid_last = valid_last;
                d.split = tile.split; d.n_splits = g.n_splits; d.half = item & 1; d.n_heads = nheads;
                d.load_q = (item >= 0 && tile.group != resident_group) ? 1 : 0;
                d.scale_log2 = scale_log2;
                d.q_off = g.q_off; d.out_off = g.out_off; d.lse_off = g.lse_off; d.part_off = g.part_off;
                mi->tq[qs] = d;
                mbar_arrive(smem_u32(&mi->tq_full[qs]));
            }
            ++qi;
            if (item < 0) break;
            resident_group = tile.group;

            for (int s0 = 0; s0 < n_slices; s0 += 32) {
                // translate (step a2): one page-table entry per lane; slice s -> page s / spp
                int32_t pid = 0;
                if (s0 + lane < n_slices) pid = page_of(p, g.req, tile.page_begin + (s0 + lane) / spp);
                const int ns = min(32, n_slices - s0);
                for (int j = 0; j < ns; ++j) {
                    const int32_t my = __shfl_sync(0xffffffffu, pid, j);
                    const uint32_t slot = gs % MLA_STAGES;
                    mbar_wait(smem_u32(&mi->empty[slot]), ((gs / MLA_STAGES) & 1) ^ 1);
                    if (elect_one()) {
                        const uint32_t fb = smem_u32(&mi->full[slot]);
                        mbar_arrive_expect_tx(fb, MLA_STAGE_BYTES);
                        const int row = my * rows_per_page + ((s0 + j) % spp) * MLA_TS;
                        // one 3-D box {64 columns, 32 rows, 9 column blocks} -> 9 swizzled [32 x 64] tiles
                        tma_load_3d(st_base + slot * MLA_STAGE_BYTES, &tmap, 0, row, 0, fb, policy);
                    }
                    ++gs;
                }
            }
        }
    } else if (warp == 1) {
        // =========================================================== MMA issuer warp
        constexpr uint32_t IDESC_S = umma_idesc_bf16(MLA_M, MLA_TS, 0, 0);      // Q (K-major) x C^T (K-major)
        constexpr uint32_t IDESC_PV = umma_idesc_bf16(MLA_M, MLA_HALF, 0, 1);   // P (K-major) x V (MN-major)
        uint32_t gs = 0, qi = 0, qn = 0;
        for (;;) {
            const uint32_t qs = qi % MLA_TQ;
            mbar_wait(smem_u32(&mi->tq_full[qs]), (qi / MLA_TQ) & 1);
            const MlaDesc d = mi->tq[qs];
            __syncwarp();
            if (lane == 0) mbar_arrive(smem_u32(&mi->tq_empty[qs]));
            ++qi;
            if (d.item < 0) break;
            if (d.load_q) { mbar_wait(smem_u32(&mi->q_full), qn & 1); ++qn; }
            const int n = d.n_slices;
            for (int i = 0; i <= n; ++i) {
                if (i < n) {
                    // ---- S_i = Q C_i^T into score buffer (g & 1)
                    const uint32_t g = gs + (uint32_t)i, slot = g % MLA_STAGES, b = g & 1;
                    mbar_wait(smem_u32(&mi->full[slot]), (g / MLA_STAGES) & 1);
                    mbar_wait(smem_u32(&mi->s_empty[b]), ((g >> 1) & 1) ^ 1);
                    tc_fence_after();
                    if (elect_one()) {
                        const uint32_t c0 = st_base + slot * MLA_STAGE_BYTES;
                        const uint32_t dcol = tmem + (b ? MLA_TMEM_S1 : MLA_TMEM_S0);
#pragma unroll
                        for (int kb = 0; kb < MLA_KB; ++kb) {
#pragma unroll
                            for (int j = 0; j < 4; ++j) {        // K = 16 per MMA: 32 bytes inside the swizzled row
                                const uint64_t bd = umma_smem_desc(c0 + kb * MLA_BLK_BYTES + j * 32, 16, 1024, 2);
                                if (kb < MLA_KB_TMEM) {          // A from tensor memory: 8 columns per K = 16
                                    umma_bf16_ts(dcol, tmem + MLA_TMEM_Q + kb * 32 + j * 8, bd, IDESC_S, (kb | j) != 0);
                                } else {
                                    const uint64_t ad = umma_smem_desc(q_base + (kb - MLA_KB_TMEM) * MLA_QBLK_BYTES + j * 32, 16, 1024, 2);
                                    umma_bf16_ss(dcol, ad, bd, IDESC_S, 1);
                                }
                            }
                        }
                        umma_commit(smem_u32(&mi->s_full[b]));
                    }
                    __syncwarp();
                }
                if (i >= 1) {
                    // ---- O += P_{i-1} V_{i-1} (value half of the work item)
                    const uint32_t g = gs + (uint32_t)i - 1, slot = g % MLA_STAGES;
                    mbar_wait(smem_u32(&mi->p_full), g & 1);
                    tc_fence_after();
                    if (elect_one()) {
#pragma unroll
                        for (int kk = 0; kk < MLA_TS / 16; ++kk) {    // K = 16 tokens per MMA
                            // P: no swizzle, core matrices of 8 rows x 16 B: 8-token chunks 2048 B apart, 8-row groups 128 B apart
                            const uint64_t ad = umma_smem_desc(p_base + kk * 4096, 2048, 128, 0);
                            // V: MN-major, 128-byte swizzle: 64-column blocks MLA_BLK_BYTES apart, 8-token groups 1024 B apart
                            const uint64_t bd = umma_smem_desc(st_base + slot * MLA_STAGE_BYTES + d.half * 4 * MLA_BLK_BYTES + kk * 2048,
                                                               MLA_BLK_BYTES, 1024, 2);
                            umma_bf16_ss(tmem, ad, bd, IDESC_PV, (i > 1) || (kk > 0));
                        }
                        umma_commit(smem_u32(&mi->empty[slot]));      // slice consumed: the stage is free
                        umma_commit(smem_u32(&mi->p_done));           // P buffer free, O updated
                    }
                    __syncwarp();
                }
            }
            gs += (uint32_t)n;
        }
    } else {
        // =========================================================== softmax warps (thread = query head)
        const int q4 = warp & 3;                          // TMEM lane quadrant this warp may access
        const int row = q4 * 32 + lane;                   // query head
        const uint32_t tl = tmem + ((uint32_t)(q4 * 32) << 16);
        const int st = tid - 64;                          // 0..127
        uint32_t gs = 0, qi = 0;
        for (;;) {
            const uint32_t qs = qi % MLA_TQ;
            mbar_wait(smem_u32(&mi->tq_full[qs]), (qi / MLA_TQ) & 1);
            const MlaDesc d = mi->tq[qs];
            __syncwarp();
            if (lane == 0) mbar_arrive(smem_u32(&mi->tq_empty[qs]));
            ++qi;
            if (d.item < 0) break;

            if (d.load_q) {
                // stage the query block [128 x 576] bf16.  Column blocks 0..5 go to tensor memory (this
                // thread's head = its TMEM lane; two bf16 per 32-bit column, memory order), where the
                // score MMAs read them as the A operand without shared-memory traffic; blocks 6..8 go
                // to shared memory as K-major [128 x 64] tiles with the 128-byte swizzle the MMA
                // descriptor expects (16-B chunk index ^ (row & 7)).  Rows >= Hq are zero.
                {
                    const uint4 *qr = reinterpret_cast<const uint4 *>(p.q + d.q_off + (int64_t)row * MLA_DK);
                    const bool live = row < d.n_heads;
                    for (int c0 = 0; c0 < MLA_KB_TMEM * 32; c0 += 64) {   // batches of 4 x 16 columns: 16 loads in flight
                        uint4 v[16];
#pragma unroll
                        for (int i = 0; i < 16; ++i) {
                            v[i] = make_uint4(0u, 0u, 0u, 0u);
                            if (live) v[i] = __ldg(qr + c0 / 4 + i);
                        }
#pragma unroll
                        for (int b4 = 0; b4 < 4; ++b4) {                  // 16 columns = 32 bf16 = 4 x 16 B
                            uint32_t w[16];
#pragma unroll
                            for (int v4 = 0; v4 < 4; ++v4) {
                                w[4 * v4] = v[4 * b4 + v4].x; w[4 * v4 + 1] = v[4 * b4 + v4].y;
                                w[4 * v4 + 2] = v[4 * b4 + v4].z; w[4 * v4 + 3] = v[4 * b4 + v4].w;
                            }
                            tmem_st16(tl + MLA_TMEM_Q + c0 + b4 * 16, w);
                        }
                    }
                    tmem_wait_st();
                }
                {
                    constexpr int CPR = (MLA_KB - MLA_KB_TMEM) * 8;      // 16-B chunks per row in shared memory
                    const uint4 *qg = reinterpret_cast<const uint4 *>(p.q + d.q_off);
#pragma unroll 8
                    for (int id = st; id < MLA_M * CPR; id += 128) {
                        const int r = id / CPR, ch = id % CPR;
                        uint4 v = make_uint4(0u, 0u, 0u, 0u);
                        if (r < d.n_heads) v = __ldg(qg + r * (MLA_DK / 8) + MLA_KB_TMEM * 8 + ch);
                        const uint32_t a = q_base + (ch >> 3) * MLA_QBLK_BYTES + r * 128 + (((ch & 7) ^ (r & 7)) << 4);
                        asm volatile("st.shared.v4.b32 [%0], {%1,%2,%3,%4};" ::"r"(a), "r"(v.x), "r"(v.y), "r"(v.z), "r"(v.w) : "memory");
                    }
                }
                tc_fence_before();
                fence_proxy_async();
                __syncwarp();
                if (lane == 0) mbar_arrive(smem_u32(&mi->q_full));
            }

            float m_run = -INFINITY, l_run = 0.f;
            const int n = d.n_slices;
            for (int i = 0; i < n; ++i) {
                const uint32_t g = gs + (uint32_t)i, b = g & 1, k = g >> 1;
                mbar_wait(smem_u32(&mi->s_full[b]), k & 1);
                tc_fence_after();
                uint32_t sr[MLA_TS];
#pragma unroll
                for (int c = 0; c < MLA_TS; c += 16)
                    tmem_ld16(tl + (b ? MLA_TMEM_S1 : MLA_TMEM_S0) + c, *reinterpret_cast<uint32_t (*)[16]>(&sr[c]));
                tmem_wait_ld();
                tc_fence_before();
                __syncwarp();
                if (lane == 0) mbar_arrive(smem_u32(&mi->s_empty[b]));       // score buffer free
                const int valid = (i == n - 1) ? d.valid_last : MLA_TS;
                float mx = -INFINITY;
#pragma unroll
                for (int j = 0; j < MLA_TS; ++j) {
                    const float v = j < valid ? __uint_as_float(sr[j]) * d.scale_log2 : -INFINITY;
                    sr[j] = __float_as_uint(v);
                    mx = fmaxf(mx, v);
                }
                // lazy reference update (see the MQA/GQA kernel): m only moves when it must
                const float m_new = (mx > m_run + MLA_LAZY_LOG2) ? mx : m_run;
                const bool need = (m_new != m_run) && i > 0;     // at i == 0 the MMA overwrites O
                const float a_resc = ex2_ftz(m_run - m_new);      // 1 when the reference stays
                if (m_new != m_run) { l_run *= a_resc; m_run = m_new; }
                uint32_t pw[MLA_TS / 2];
                float sum = 0.f;
#pragma unroll
                for (int j = 0; j < MLA_TS / 2; ++j) {
                    const float p0 = ex2_ftz(__uint_as_float(sr[2 * j]) - m_run), p1 = ex2_ftz(__uint_as_float(sr[2 * j + 1]) - m_run);
                    sum += p0 + p1;
                    asm("cvt.rn.bf16x2.f32 %0, %1, %2;" : "=r"(pw[j]) : "f"(p1), "f"(p0));
                }
                l_run += sum;
                // the P buffer (and O, if it must be rescaled) is free once P_{i-1} V_{i-1} has completed
                mbar_wait(smem_u32(&mi->p_done), (g & 1) ^ 1);
                if (__any_sync(0xffffffffu, need)) {
                    // rescale this warp's O rows in TMEM
                    tc_fence_after();
                    const float a = need ? a_resc : 1.f;
                    for (int c = 0; c < MLA_HALF; c += 16) {
                        uint32_t o[16];
                        tmem_ld16(tl + c, o);
                        tmem_wait_ld();
#pragma unroll
                        for (int j = 0; j < 16; ++j) o[j] = __float_as_uint(__uint_as_float(o[j]) * a);
                        tmem_st16(tl + c, o);
                    }
                    tmem_wait_st();
                }
                // P[row][token] as 8-token chunks: chunk c of row r at c * 2048 + r * 16
#pragma unroll
                for (int c = 0; c < MLA_TS / 8; ++c)
                    asm volatile("st.shared.v4.b32 [%0], {%1,%2,%3,%4};" ::"r"(p_base + c * 2048 + row * 16), "r"(pw[4 * c]),
                                 "r"(pw[4 * c + 1]), "r"(pw[4 * c + 2]), "r"(pw[4 * c + 3]) : "memory");
                if (valid < MLA_TS) {
                    // dead slots of the request's last slice may hold NaN: zero their value rows (0 * NaN);
                    // warp q4 clears column block half*4 + q4 of the stage
                    const uint32_t blk = st_base + (g % MLA_STAGES) * MLA_STAGE_BYTES + (d.half * 4 + q4) * MLA_BLK_BYTES;
                    for (int e = lane; e < (MLA_TS - valid) * 8; e += 32) {
                        const int r = valid + (e >> 3), ch = e & 7;
                        asm volatile("st.shared.v4.b32 [%0], {%1,%1,%1,%1};" ::"r"(blk + r * 128 + ((ch ^ (r & 7)) << 4)), "r"(0u) : "memory");
                    }
                }
                fence_proxy_async();
                tc_fence_before();
                __syncwarp();
                if (lane == 0) mbar_arrive(smem_u32(&mi->p_full));
            }
            gs += (uint32_t)n;

            // ---- end of tile: O (this value half) from TMEM, publish
            {
                const uint32_t gl = gs - 1;
                mbar_wait(smem_u32(&mi->p_done), gl & 1);
                tc_fence_after();
                const bool final_out = d.n_splits == 1;
                const float inv = final_out ? 1.f / l_run : 1.f;
                float *dst = final_out
                                 ? p.out + d.out_off + (int64_t)row * MLA_DV + d.half * MLA_HALF
                                 : p.workspace + d.part_off + part_o_off(row, d.split, d.n_splits, MLA_DV) + d.half * MLA_HALF;
                for (int c = 0; c < MLA_HALF; c += 16) {
                    uint32_t o[16];
                    tmem_ld16(tl + c, o);
                    tmem_wait_ld();
                    if (row < d.n_heads) {
#pragma unroll
                        for (int j = 0; j < 16; j += 4)
                            __stcg(reinterpret_cast<float4 *>(dst + c + j),
                                   make_float4(__uint_as_float(o[j]) * inv, __uint_as_float(o[j + 1]) * inv,
                                               __uint_as_float(o[j + 2]) * inv, __uint_as_float(o[j + 3]) * inv));
                    }
                }
                tc_fence_before();
                if (d.half == 0 && row < d.n_heads) {
                    if (final_out)
                        p.lse[d.lse_off + row] = (m_run + log2f(l_run)) * 0.6931471805599453f;
                    else
                        __stcg(reinterpret_cast<float2 *>(p.workspace + d.part_off +
                                                          part_ml_off(d.n_heads, row, d.split, d.n_splits, MLA_DV)),
                               make_float2(m_run, l_run));
                }
                if (!final_out) {
                    __syncwarp();
                    if (lane == 0) red_release_add(p.group_counters + (size_t)d.group_idx * kCounterStride, 1);
                }
            }
        }
        // ---- LSE combine (step a4): warp-sized units, statically assigned (see the MQA/GQA kernel)
        float *wsm = reinterpret_cast<float *>(smem + MLA_SMEM_P) + (warp - 2) * kMaxSplits;
        combine_units<16>(p, blockIdx.x * 4 + (warp - 2), gridDim.x * 4, wsm, lane);
    }
    tc_fence_before();
    __syncthreads();
    if (warp == 1) tmem_dealloc(tmem, MLA_TMEM_COLS);
}

// ----------------------------------------------------------------------------- host side
bool mla_fast_supported(int page_tokens, uint32_t page_bytes)
{
    return page_tokens >= MLA_TS && page_tokens % MLA_TS == 0 && page_bytes % (MLA_DK * 2) == 0;
}

// 3-D view of the arena: {64 columns, rows of 576 bf16 (1152 B apart), 9 column blocks (128 B apart)};
// one box = a 32-token slice as 9 consecutive 128-byte-swizzled [32 x 64] tiles in shared memory.
bool make_mla_tensor_map(void *out_map, const void *arena, uint64_t total_rows)
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
    cuuint64_t dims[3] = {64, total_rows, (cuuint64_t)MLA_KB};
    cuuint64_t strides[2] = {(cuuint64_t)MLA_DK * 2, 128};
    cuuint32_t box[3] = {64, (cuuint32_t)MLA_TS, (cuuint32_t)MLA_KB};
    cuuint32_t estr[3] = {1, 1, 1};
    CUresult r = fn(reinterpret_cast<CUtensorMap *>(out_map), CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 3,
                    const_cast<void *>(arena), dims, strides, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE,
                    CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    return r == CUDA_SUCCESS;
}

cudaError_t launch_decode_mla(const DecodeParams &p, const void *tmap, int rows_per_page, int n_ctas,
                              cudaStream_t stream)
{
    static bool configured[64] = {};              // per device: the attribute belongs to the device's copy of the function
    int dev = 0;
    if (cudaGetDevice(&dev) != cudaSuccess) return cudaGetLastError();
    if (dev < 0 || dev >= 64 || !configured[dev]) {
        cudaError_t e = cudaFuncSetAttribute(cp_decode_mla_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                             MLA_SMEM_BYTES);
        if (e != cudaSuccess) return e;
        if (dev >= 0 && dev < 64) configured[dev] = true;
    }
    int grid = 2 * p.n_tiles;
    if (grid < (p.n_combine_units + 3) / 4) grid = (p.n_combine_units + 3) / 4;
    if (grid > n_ctas) grid = n_ctas;
    if (grid < 1) grid = 1;
    cp_decode_mla_kernel<<<grid, MLA_THREADS, MLA_SMEM_BYTES, stream>>>(
        p, *reinterpret_cast<const CUtensorMap *>(tmap), rows_per_page);
    return cudaGetLastError();
}

}  // namespace cp
