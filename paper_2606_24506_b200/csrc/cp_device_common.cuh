// cp_device_common.cuh -- device helpers shared by the decode kernels: bf16 unpacking,
// acquire/release counters of the persistent scheduler, and the LSE combine unit
// (hot-path step a4).
#pragma once
#include <cuda_runtime.h>
#include <cstdint>
#include "cp_internal.h"

namespace cp {

__device__ __forceinline__ float bf16_lo(uint32_t w) { return __uint_as_float(w << 16); }
__device__ __forceinline__ float bf16_hi(uint32_t w) { return __uint_as_float(w & 0xFFFF0000u); }

__device__ __forceinline__ int ld_acquire(const int32_t *p)
{
    int v;
    asm volatile("ld.acquire.gpu.global.s32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
    return v;
}

__device__ __forceinline__ int ld_relaxed(const int32_t *p)
{
    int v;
    asm volatile("ld.relaxed.gpu.global.s32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
    return v;
}

__device__ __forceinline__ int ld_acquire_sys(const int32_t *p)
{
    int v;
    asm volatile("ld.acquire.sys.global.s32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
    return v;
}

__device__ __forceinline__ unsigned long long global_timer_ns()
{
    unsigned long long t;
    asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t) :: "memory");
    return t;
}

// Physical page of entry `idx` of request `req`'s page list.  Software table (PAPER.md, reading R1)
// or, on a CUDA-VMM arena, plain arithmetic on the request's contiguous virtual range.
__device__ __forceinline__ int32_t page_of(const DecodeParams &p, int req, int64_t idx)
{
    if (p.slot_pages > 0) return req * p.slot_pages + (int32_t)idx;
    return __ldg(p.page_table + (int64_t)req * p.max_ppr + idx);
}

// Wait until group counter `gi` has reached `want` (called by one lane).  Polls with exponential
// back-off: hundreds of warps polling one L2 line every few dozen ns would saturate its slice
// and delay the very arrivals they wait for.
__device__ __forceinline__ void wait_group(const int32_t *counters, int gi, int want)
{
    const int32_t *c = counters + (size_t)gi * kCounterStride;
    unsigned ns = 128;
    while (ld_acquire(c) < want) {
        __nanosleep(ns);
        if (ns < 1024) ns <<= 1;
    }
}

__device__ __forceinline__ void red_release_add(int32_t *p, int v)
{
    asm volatile("red.release.gpu.global.add.s32 [%0], %1;" ::"l"(p), "r"(v) : "memory");
}

__device__ __forceinline__ float4 ld_cg_f4(const float *p)
{
    return __ldcg(reinterpret_cast<const float4 *>(p));
}

// Byte offset of row `slot` of the K (is_v = false) or V block of a page, for a model.
__device__ __forceinline__ uint64_t row_byte_offset(const DecodeParams &p, const DevModel &m,
                                                    int32_t pid, uint32_t slot, bool is_v)
{
    uint64_t base = (uint64_t)pid * p.page_bytes;
    if (m.kind == 1 || !is_v) return base + (uint64_t)slot * m.d_k * 2u;
    return base + (uint64_t)p.page_tokens * m.d_k * 2u + (uint64_t)slot * m.d_v * 2u;
}

// ---------------------------------------------------------------------------------------
// LSE combine of one (group, head): waits until every split of the group has published
// its partial (acquire on the group counter), then
//     M = max_s m_s;  w_s = 2^(m_s - M);  L = sum_s w_s l_s;
//     O = (sum_s w_s O_s) / L;  LSE = (M + log2 L) * ln 2
// Every sum runs in a fixed order (strided lanes in split order, then a fixed tree), so
// the result does not depend on which CTA runs it or when (deterministic).
// Partials are unnormalised: O_s = sum_t 2^(s_t - m_s) v_t, l_s = sum_t 2^(s_t - m_s),
// scores in log2 units.  Called by all threads of a CTA (blockDim.x a multiple of 32,
// >= d_v / 4); smem_f is 16-B aligned and holds cp_combine_smem_bytes() bytes.
// ---------------------------------------------------------------------------------------
__host__ __device__ inline size_t cp_combine_smem_bytes(int max_splits, int threads)
{
    return ((size_t)4 * threads + 40 + 2 * (size_t)max_splits) * sizeof(float);
}

__host__ __device__ inline int mtiles_pow2(int g)    // 16-head M tiles rounded up to a power of two
{
    int mt = (g + 15) / 16, q = 1;
    while (q < mt) q <<= 1;
    return q;
}

struct BlockSync {
    __device__ __forceinline__ void operator()() const { __syncthreads(); }
};

// arrival_mode 0: one counter arrival per tile; 1: one per 16-head M tile (tensor-core KV path).
// tid / nthr / sync: the participating threads (a whole CTA, or the consumer warps only).
template <class Sync>
__device__ inline void combine_unit(const DecodeParams &p, const Combine cu, int arrival_mode,
                                    float *smem_f, const int tid, const int nthr, Sync sync)
{
    const Group g = p.groups[cu.group];
    const DevModel m = p.models[g.model];
    const int ns = g.n_splits;
    const int dv = m.d_v;

    // wait for all splits of the group (tiles are popped before combine units and never
    // block, so this spin terminates)
    if (tid == 0) {
        const int want = ns * (arrival_mode ? mtiles_pow2(m.group) : 1);
        wait_group(p.group_counters, cu.group, want);
    }
    sync();

    float4 *red4 = reinterpret_cast<float4 *>(smem_f);      // [nthr]
    float *red = smem_f + 4 * nthr;                         // [40]
    float *w_s = red + 40;                                  // [ns]
    float *l_s = w_s + ns;                                  // [ns]
    const float *part = p.workspace + g.part_off + part_o_off(cu.head, 0, ns, dv);
    const float *mlp = p.workspace + g.part_off + part_ml_off(m.group, cu.head, 0, ns, dv);
    const int64_t split_stride = dv;

    // pass 1: M = max m_s, weights, L
    float mloc = -INFINITY;
    for (int s = tid; s < ns; s += nthr) {
        const float2 ml = __ldcg(reinterpret_cast<const float2 *>(mlp + 2 * s));
        w_s[s] = ml.x;
        l_s[s] = ml.y;
        mloc = fmaxf(mloc, ml.x);
    }
    for (int o = 16; o > 0; o >>= 1) mloc = fmaxf(mloc, __shfl_xor_sync(0xffffffffu, mloc, o));
    if ((tid & 31) == 0) red[tid >> 5] = mloc;
    sync();
    float M = -INFINITY;
    for (int w = 0; w < (nthr >> 5); ++w) M = fmaxf(M, red[w]);
    sync();
    for (int s = tid; s < ns; s += nthr) w_s[s] = exp2f(w_s[s] - M);
    sync();
    if (tid < 32) {                      // warp 0: strided in-order sums, then a fixed tree
        float L = 0.f;
        for (int s = tid; s < ns; s += 32) L += w_s[s] * l_s[s];
        for (int o = 16; o > 0; o >>= 1) L += __shfl_xor_sync(0xffffffffu, L, o);
        if (tid == 0) red[32] = L;
    }
    sync();
    const float L = red[32];
    const float invL = 1.0f / L;

    // pass 2: O.  Thread -> (column quad cq, lane z); the lanes interleave the splits.
    const int nq = dv >> 2;                       // float4 columns
    const int lanes = nthr / nq;                  // >= 1 by contract
    float4 acc = make_float4(0.f, 0.f, 0.f, 0.f);
    const int cq = tid % nq;
    const int z = tid / nq;
    if (z < lanes) {
#pragma unroll 8
        for (int s = z; s < ns; s += lanes) {
            const float w = w_s[s];
            const float4 v = ld_cg_f4(part + s * split_stride + cq * 4);
            acc.x += w * v.x; acc.y += w * v.y; acc.z += w * v.z; acc.w += w * v.w;
        }
        red4[z * nq + cq] = acc;
    }
    sync();
    if (tid < nq) {
        float4 o = red4[tid];
        for (int zz = 1; zz < lanes; ++zz) {
            const float4 v = red4[zz * nq + tid];
            o.x += v.x; o.y += v.y; o.z += v.z; o.w += v.w;
        }
        o.x *= invL; o.y *= invL; o.z *= invL; o.w *= invL;
        float *dst = p.out + g.out_off + (int64_t)cu.head * dv + tid * 4;
        *reinterpret_cast<float4 *>(dst) = o;
    }
    if (tid == 0) p.lse[g.lse_off + cu.head] = (M + log2f(L)) * 0.6931471805599453f;
    sync();
}

// ---------------------------------------------------------------------------------------
// Warp-sized LSE combine unit (tensor-core kernels): ONE warp combines (128 >> zl) output
// columns of one (group, head) described by a CombineUnit record; units are assigned statically
// to the grid's warps, no CTA barrier.  The warp's lanes are (split lane z of ZL = 2^zl) x
// (column quad cq of 32 / ZL).  Same arithmetic as combine_unit; all sums run in a fixed order
// (s ascending per lane, then a fixed shuffle tree) => deterministic.
// wsm: this warp's shared-memory scratch, >= n_splits floats (n_splits <= kMaxSplits).
// ---------------------------------------------------------------------------------------
__device__ __forceinline__ float ex2_ftz(float x)     // 2^x; ex2(-inf) = 0
{
    float r;
    asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x));
    return r;
}

// Deliberately compact (short loops, 32-bit offsets): the code runs once per
// launch per warp, so its cost is dominated by cold instruction-cache misses, not by issue slots.
// CG: the records were written during this launch (request queue: the planner warp of CTA 0): read them from
// the L2 (ld.cg), not through the non-coherent path, whose lines may predate the write.
template <bool CG = false>
__device__ __forceinline__ CombineUnit load_combine_unit(const CombineUnit *units, int u)
{
    CombineUnit cu;
    const uint4 *src = reinterpret_cast<const uint4 *>(units + u);
    uint4 *dst = reinterpret_cast<uint4 *>(&cu);
#pragma unroll
    for (int i = 0; i < 4; ++i) dst[i] = CG ? __ldcg(src + i) : __ldg(src + i);
    return cu;
}

// Runs the units first, first + stride, ... of one warp.  U3 = loads in flight per lane in the O
// pass.  The record of the next unit is fetched while the current one is combined, and a group
// already seen complete is not polled again (units are sorted by group).
// STAGED (multi-stage launches): the units u < end of one stage; every finished unit is counted in
// the stage's completion counter (release), which the dependent stage's tiles acquire.
template <int U3, bool STAGED = false, bool CG = false>
static __device__ __noinline__ void combine_units(const DecodeParams &p, int u, const int stride, float *wsm, const int lane,
                                                  const int end = 0)
{
    const int n_end = STAGED ? end : p.n_combine_units;
    if (u >= n_end) return;
    CombineUnit cu = load_combine_unit<CG>(p.cunits, u);
    int done_group = -1;
    for (;;) {
        const int un = u + stride;
        const bool has_next = un < n_end;
        CombineUnit nx;
        if (has_next) nx = load_combine_unit<CG>(p.cunits, un);
        const int ns = cu.n_splits;
        const int zl = cu.zl_log2;
        const int ZL = 1 << zl, CQ = 32 >> zl;
        const int z = lane >> (5 - zl), cq = lane & (CQ - 1);
        if (cu.group != done_group) {
            if (lane == 0) wait_group(p.group_counters, cu.group, cu.want);
            __syncwarp();
            done_group = cu.group;
        }
        const float2 *mlp = reinterpret_cast<const float2 *>(p.workspace + cu.ml_off);
        const float *src = p.workspace + cu.part_off + cq * 4;
        const int ss = cu.split_stride;

        float M = -INFINITY, L = 0.f;
        if (ns <= 256) {
            // (m, l) of splits lane, lane + 32, ... stay in registers: one round trip for both passes
            float2 ml[8];
#pragma unroll
            for (int k = 0; k < 8; ++k) {
                ml[k] = make_float2(-INFINITY, 0.f);
                if (lane + 32 * k < ns) ml[k] = __ldcg(mlp + lane + 32 * k);
            }
#pragma unroll
            for (int k = 0; k < 8; ++k) M = fmaxf(M, ml[k].x);
            for (int o = 16; o > 0; o >>= 1) M = fmaxf(M, __shfl_xor_sync(0xffffffffu, M, o));
#pragma unroll
            for (int k = 0; k < 8; ++k) {
                const float w = ex2_ftz(ml[k].x - M);          // 0 for absent splits (m = -inf)
                if (lane + 32 * k < ns) wsm[lane + 32 * k] = w;
                L += w * ml[k].y;
            }
        } else {
            // pass 1: M = max_s m_s (lane-strided, then a fixed tree)
#pragma unroll 8
            for (int s = lane; s < ns; s += 32) M = fmaxf(M, __ldcg(mlp + s).x);
            for (int o = 16; o > 0; o >>= 1) M = fmaxf(M, __shfl_xor_sync(0xffffffffu, M, o));
            // pass 2: weights w_s = 2^(m_s - M) to shared memory, L = sum_s w_s l_s
#pragma unroll 8
            for (int s = lane; s < ns; s += 32) {
                const float2 ml = __ldcg(mlp + s);
                const float w = ex2_ftz(ml.x - M);
                wsm[s] = w;
                L += w * ml.y;
            }
        }
        for (int o = 16; o > 0; o >>= 1) L += __shfl_xor_sync(0xffffffffu, L, o);
        __syncwarp();
        // pass 3: O = sum_s w_s O_s over this lane's splits z, z + ZL, ... (in order), then the tree
        float4 acc = make_float4(0.f, 0.f, 0.f, 0.f);
#pragma unroll U3
        for (int s = z; s < ns; s += ZL) {
            const float4 v = ld_cg_f4(src + s * ss);
            const float w = wsm[s];
            acc.x += w * v.x; acc.y += w * v.y; acc.z += w * v.z; acc.w += w * v.w;
        }
        for (int o = CQ; o < 32; o <<= 1) {               // warp-uniform trip count
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
        __syncwarp();               // wsm is reused by this warp's next unit
        if (STAGED) {
            // the unit's O / LSE stores happen-before this release (cumulative over the __syncwarp)
            if (lane == 0) red_release_add(p.stage_done + (size_t)cu.pad[0] * kCounterStride, 1);
        }
        if (!has_next) break;
        cu = nx;
        u = un;
    }
}

// The scheduler counters come in two sets used by alternate launches of a plan.  A launch works on
// one set and, right at its start, one CTA clears the OTHER set -- dirty from the previous launch,
// which has completed (stream order) -- for the next launch.  Nothing has to be reset at the end
// of a kernel: no last-CTA election, no atomic round trip on the exit path.
__device__ inline void scheduler_reset_other_set(const DecodeParams &p)
{
    if (blockIdx.x != gridDim.x - 1) return;
    for (int i = threadIdx.x; i < p.n_groups; i += blockDim.x) p.reset_counters[32 + (size_t)i * kCounterStride] = 0;
    if (threadIdx.x < 4) p.reset_counters[threadIdx.x] = 0;
}

}  // namespace cp
