// cp_kernels_generic.cu -- shape-generic CUDA kernels of libcrosspool:
//   * cp_gather_kernel: page-table translation + KV gather (hot-path step a2), bit-exact;
//   * cp_decode_generic_kernel: persistent split-KV decode attention for ANY supported
//     model shape (KV kind or MLA kind, d_k <= 576, d_v <= 512, any group size) with
//     fp32 SIMT arithmetic.  It is the path for shapes the tensor-core kernels do not
//     cover, and an independent GPU cross-check of those kernels.  Same work list, same
//     partial format and same LSE combine as the fast kernels.
// Paper anchors: paged KV interface PAPER.md:L101,L122; persistent GPU-resident control
// PAPER.md:L146.  Arithmetic: DESIGN.md §3 (definition) and §6 (split-KV formulation).
#include <cuda_runtime.h>
#include <cstdint>
#include "cp_device_common.cuh"
#include "cp_launch.h"

namespace cp {

// ------------------------------------------------------------------------------ gather
// Grid-stride over 16-byte vectors; every thread moves four vectors per iteration (four independent
// translations + loads in flight before the first store), one page-table lookup per vector.
template <class Idx>
__device__ __forceinline__ void gather_addr(const uint8_t *arena, uint32_t page_tokens, uint32_t page_bytes,
                                            const int32_t *page_ids, int kind, int n_kv_heads, int d_k, int d_v,
                                            int kvec, int per_row, Idx i, uint8_t *k_out, uint8_t *v_out,
                                            const uint4 *&src, uint4 *&dst)
{
    const Idx row = i / (Idx)per_row;           // row = t * Hkv + c
    const int vec = (int)(i - row * (Idx)per_row);
    const int t = (int)(row / (Idx)n_kv_heads);
    const int c = (int)(row - (Idx)t * (Idx)n_kv_heads);
    const int lp = t / (int)page_tokens;
    const uint32_t slot = (uint32_t)(t - lp * (int)page_tokens);
    const int32_t pid = __ldg(page_ids + (int64_t)lp * n_kv_heads + c);
    const uint64_t base = (uint64_t)pid * page_bytes;
    if (vec < kvec) {
        src = reinterpret_cast<const uint4 *>(arena + base + (uint64_t)slot * d_k * 2 + vec * 16);
        dst = reinterpret_cast<uint4 *>(k_out + (uint64_t)row * d_k * 2 + vec * 16);
    } else {
        const int vv = vec - kvec;
        const uint64_t off = (kind == 1) ? (uint64_t)slot * d_k * 2
                                         : (uint64_t)page_tokens * d_k * 2 + (uint64_t)slot * d_v * 2;
        src = reinterpret_cast<const uint4 *>(arena + base + off + vv * 16);
        dst = reinterpret_cast<uint4 *>(v_out + (uint64_t)row * d_v * 2 + vv * 16);
    }
}

template <class Idx>      // uint32_t when the vector count fits (32-bit divisions), else uint64_t
__global__ void __launch_bounds__(256)
cp_gather_kernel(const uint8_t *__restrict__ arena, uint32_t page_tokens, uint32_t page_bytes,
                 const int32_t *__restrict__ page_ids, int kind, int n_kv_heads, int d_k, int d_v,
                 int context_len, uint8_t *__restrict__ k_out, uint8_t *__restrict__ v_out)
{
    const int kvec = d_k / 8;                       // 16-B vectors per K row
    const int vvec = v_out ? d_v / 8 : 0;
    const int per_row = kvec + vvec;
    const Idx total = (Idx)context_len * (Idx)n_kv_heads * (Idx)per_row;
    const Idx T = (Idx)gridDim.x * blockDim.x;
    for (Idx i0 = (Idx)blockIdx.x * blockDim.x + threadIdx.x; i0 < total; i0 += 4 * T) {
        const uint4 *src[4];
        uint4 *dst[4];
        uint4 val[4];
#pragma unroll
        for (int u = 0; u < 4; ++u)
            if (i0 + u * T < total)
                gather_addr<Idx>(arena, page_tokens, page_bytes, page_ids, kind, n_kv_heads, d_k, d_v, kvec, per_row,
                            i0 + u * T, k_out, v_out, src[u], dst[u]);
#pragma unroll
        for (int u = 0; u < 4; ++u)
            if (i0 + u * T < total) val[u] = __ldcs(src[u]);          // streamed once
#pragma unroll
        for (int u = 0; u < 4; ++u)
            if (i0 + u * T < total) __stcs(dst[u], val[u]);
    }
}

void launch_gather(const uint8_t *arena, uint32_t page_tokens, uint32_t page_bytes,
                   const int32_t *page_ids_dev, int kind, int n_kv_heads, int d_k, int d_v,
                   int context_len, void *k_out, void *v_out, int n_sm, cudaStream_t stream)
{
    const int64_t total = (int64_t)context_len * n_kv_heads * (d_k / 8 + (v_out ? d_v / 8 : 0));
    int64_t blocks = (total + 1023) / 1024;
    const int64_t cap = (int64_t)n_sm * 16;
    if (blocks > cap) blocks = cap;
    if (blocks < 1) blocks = 1;
    if (total + 4 * blocks * 256 < (int64_t)0xFFFFFFFFll)
        cp_gather_kernel<uint32_t><<<(unsigned)blocks, 256, 0, stream>>>(
            arena, page_tokens, page_bytes, page_ids_dev, kind, n_kv_heads, d_k, d_v, context_len,
            (uint8_t *)k_out, (uint8_t *)v_out);
    else
        cp_gather_kernel<uint64_t><<<(unsigned)blocks, 256, 0, stream>>>(
            arena, page_tokens, page_bytes, page_ids_dev, kind, n_kv_heads, d_k, d_v, context_len,
            (uint8_t *)k_out, (uint8_t *)v_out);
}

// ------------------------------------------------------------------------------ append
// One block per request: translate (request, logical page of `pos`, kv head) through the page
// table and copy the new token's K and V rows (16-byte vectors) into their slots.
__global__ void cp_append_kernel(uint8_t *__restrict__ arena, uint32_t page_tokens, uint32_t page_bytes,
                                 const int32_t *__restrict__ page_table, int max_ppr,
                                 const DevModel *__restrict__ models, const AppendRec *__restrict__ recs,
                                 const uint16_t *__restrict__ k_new, const uint16_t *__restrict__ v_new)
{
    const AppendRec r = recs[blockIdx.x];
    const DevModel m = models[r.model];
    const int lp = r.pos / (int)page_tokens;
    const uint32_t slot = (uint32_t)(r.pos - lp * (int)page_tokens);
    const int kvec = m.d_k / 8, vvec = m.kind == 1 ? 0 : m.d_v / 8;
    const int per_head = kvec + vvec;
    for (int i = threadIdx.x; i < m.n_kv_heads * per_head; i += blockDim.x) {
        const int c = i / per_head, vec = i - c * per_head;
        const int32_t pid = __ldg(page_table + (int64_t)r.req * max_ppr + (int64_t)lp * m.n_kv_heads + c);
        const uint64_t base = (uint64_t)pid * page_bytes;
        if (vec < kvec) {
            const uint4 v = *reinterpret_cast<const uint4 *>(k_new + r.k_off + (int64_t)c * m.d_k + vec * 8);
            *reinterpret_cast<uint4 *>(arena + base + (uint64_t)slot * m.d_k * 2 + vec * 16) = v;
        } else {
            const int vv = vec - kvec;
            const uint4 v = *reinterpret_cast<const uint4 *>(v_new + r.v_off + (int64_t)c * m.d_v + vv * 8);
            *reinterpret_cast<uint4 *>(arena + base + (uint64_t)page_tokens * m.d_k * 2 + (uint64_t)slot * m.d_v * 2 + vv * 16) = v;
        }
    }
}

void launch_append(uint8_t *arena, uint32_t page_tokens, uint32_t page_bytes, const int32_t *page_table,
                   int max_ppr, const DevModel *models, const AppendRec *recs, int n_requests,
                   const uint16_t *k_new, const uint16_t *v_new, cudaStream_t stream)
{
    cp_append_kernel<<<n_requests, 128, 0, stream>>>(arena, page_tokens, page_bytes, page_table, max_ppr, models,
                                                    recs, k_new, v_new);
}

// ---------------------------------------------------------------------- generic decode
constexpr int GEN_THREADS = 256;
constexpr int GEN_HB = 16;      // query heads per pass
constexpr int GEN_TC = 32;      // tokens per chunk (= warp width: one lane per token)
constexpr int GEN_PADE = 8;     // row padding in bf16 elements (16 B): conflict-free uint4 reads

struct GenSmem {
    // carved from dynamic shared memory by the kernel
    float *q;          // [GEN_HB][d_k]
    uint16_t *k;       // [GEN_TC][d_k + PAD]
    uint16_t *v;       // [GEN_TC][d_v + PAD]   (MLA: aliases k)
    float *p;          // [GEN_HB][GEN_TC]
    float *alpha;      // [GEN_HB]
    float *m;          // [GEN_HB]
    float *l;          // [GEN_HB]
};

size_t generic_smem_bytes(int max_dk, int max_dv, bool any_kv_kind, int max_splits)
{
    size_t b = (size_t)GEN_HB * max_dk * 4;
    b += (size_t)GEN_TC * (max_dk + GEN_PADE) * 2;
    if (any_kv_kind) b += (size_t)GEN_TC * (max_dv + GEN_PADE) * 2;
    b += (size_t)GEN_HB * GEN_TC * 4 + 3 * GEN_HB * 4 + 64;
    size_t c = cp_combine_smem_bytes(max_splits, GEN_THREADS);
    return (b > c ? b : c) + 16;
}

__global__ void __launch_bounds__(GEN_THREADS, 1)
cp_decode_generic_kernel(const DecodeParams p, int max_dk, int max_dv, int any_kv_kind)
{
    extern __shared__ __align__(16) uint8_t smem_raw[];
    __shared__ int s_work;
    const int tid = threadIdx.x;
    const int warp = tid >> 5;
    const int lane = tid & 31;

    // carve shared memory (sizes from the launch-wide maxima so every tile fits)
    GenSmem sm;
    {
        uint8_t *ptr = smem_raw;
        sm.q = reinterpret_cast<float *>(ptr);            ptr += (size_t)GEN_HB * max_dk * 4;
        sm.k = reinterpret_cast<uint16_t *>(ptr);         ptr += (size_t)GEN_TC * (max_dk + GEN_PADE) * 2;
        sm.v = sm.k;
        if (any_kv_kind) { sm.v = reinterpret_cast<uint16_t *>(ptr); ptr += (size_t)GEN_TC * (max_dv + GEN_PADE) * 2; }
        sm.p = reinterpret_cast<float *>(ptr);            ptr += (size_t)GEN_HB * GEN_TC * 4;
        sm.alpha = reinterpret_cast<float *>(ptr);        ptr += GEN_HB * 4;
        sm.m = reinterpret_cast<float *>(ptr);            ptr += GEN_HB * 4;
        sm.l = reinterpret_cast<float *>(ptr);
    }

    scheduler_reset_other_set(p);
    const int n_work = p.n_tiles + p.n_combines;
    for (;;) {
        if (tid == 0) s_work = atomicAdd(p.work_counter, 1);
        __syncthreads();
        const int work = s_work;
        __syncthreads();
        if (work >= n_work) break;

        if (work >= p.n_tiles) {        // ---- LSE combine unit (step a4)
            combine_unit(p, p.combines[work - p.n_tiles], 0, reinterpret_cast<float *>(smem_raw), tid, GEN_THREADS, BlockSync());
            continue;
        }

        // ---- split-KV partial attention of one tile (steps a2 + a3)
        const Tile tile = p.tiles[work];
        const Group g = p.groups[tile.group];
        const DevModel m = p.models[g.model];
        const int dk = m.d_k, dv = m.d_v, P = (int)p.page_tokens;
        const int krow = dk + GEN_PADE;
        const int vrow = (m.kind == 1) ? krow : dv + GEN_PADE;
        const uint16_t *vbuf = (m.kind == 1) ? sm.k : sm.v;
        const int ctx = __ldg(p.req_ctx + g.req);
        const int t_begin = tile.page_begin * P;
        const int t_end = min(tile.page_end * P, ctx);
        const int ncol = (dv + GEN_THREADS - 1) / GEN_THREADS;      // 1 or 2 columns per thread

        for (int h0 = 0; h0 < m.group; h0 += GEN_HB) {
            const int nh = min(GEN_HB, m.group - h0);
            // stage the query rows as fp32
            for (int i = tid; i < nh * dk; i += GEN_THREADS) {
                const int h = i / dk, e = i % dk;
                const uint16_t b = p.q[g.q_off + (int64_t)(h0 + h) * dk + e];
                sm.q[h * dk + e] = __uint_as_float(((uint32_t)b) << 16);
            }
            float acc[2][GEN_HB];
#pragma unroll
            for (int j = 0; j < 2; ++j)
#pragma unroll
                for (int h = 0; h < GEN_HB; ++h) acc[j][h] = 0.f;
            // warp w owns the softmax state of heads w and w + 8 (replicated over lanes)
            float m_run[2] = {-INFINITY, -INFINITY};
            float l_run[2] = {0.f, 0.f};
            __syncthreads();

            for (int t0 = t_begin; t0 < t_end; t0 += GEN_TC) {
                const int nt = min(GEN_TC, t_end - t0);
                // --- a2: translate + stage K (and V) rows of this chunk
                const int kvec = dk / 8;
                for (int i = tid; i < nt * kvec; i += GEN_THREADS) {
                    const int r = i / kvec, vch = i % kvec;
                    const int t = t0 + r;
                    const int32_t pid = page_of(p, g.req, (int64_t)(t / P) * m.n_kv_heads + g.kv_head);
                    const uint4 val = *reinterpret_cast<const uint4 *>(
                        p.arena + row_byte_offset(p, m, pid, (uint32_t)(t % P), false) + vch * 16);
                    *reinterpret_cast<uint4 *>(sm.k + (size_t)r * krow + vch * 8) = val;
                }
                if (m.kind == 0) {
                    const int vvec = dv / 8;
                    for (int i = tid; i < nt * vvec; i += GEN_THREADS) {
                        const int r = i / vvec, vch = i % vvec;
                        const int t = t0 + r;
                        const int32_t pid = page_of(p, g.req, (int64_t)(t / P) * m.n_kv_heads + g.kv_head);
                        const uint4 val = *reinterpret_cast<const uint4 *>(
                            p.arena + row_byte_offset(p, m, pid, (uint32_t)(t % P), true) + vch * 16);
                        *reinterpret_cast<uint4 *>(sm.v + (size_t)r * vrow + vch * 8) = val;
                    }
                }
                __syncthreads();

                // --- a3: scores.  thread = (token lane, heads warp and warp + 8)
                float s[2] = {-INFINITY, -INFINITY};
                if (lane < nt) {
                    float d0 = 0.f, d1 = 0.f;
                    const uint16_t *krp = sm.k + (size_t)lane * krow;
                    const float *q0 = sm.q + (size_t)warp * dk;
                    const float *q1 = sm.q + (size_t)(warp + 8) * dk;
                    const bool has0 = warp < nh, has1 = warp + 8 < nh;
                    for (int e = 0; e < dk; e += 8) {
                        const uint4 kk = *reinterpret_cast<const uint4 *>(krp + e);
                        const float kf[8] = {bf16_lo(kk.x), bf16_hi(kk.x), bf16_lo(kk.y), bf16_hi(kk.y),
                                             bf16_lo(kk.z), bf16_hi(kk.z), bf16_lo(kk.w), bf16_hi(kk.w)};
                        if (has0) {
#pragma unroll
                            for (int u = 0; u < 8; ++u) d0 = fmaf(q0[e + u], kf[u], d0);
                        }
                        if (has1) {
#pragma unroll
                            for (int u = 0; u < 8; ++u) d1 = fmaf(q1[e + u], kf[u], d1);
                        }
                    }
                    if (has0) s[0] = d0 * m.scale_log2;
                    if (has1) s[1] = d1 * m.scale_log2;
                }
                // online softmax per head (warp-wide over the chunk's tokens)
#pragma unroll
                for (int j = 0; j < 2; ++j) {
                    const int h = warp + 8 * j;
                    float mx = s[j];
                    for (int o = 16; o > 0; o >>= 1) mx = fmaxf(mx, __shfl_xor_sync(0xffffffffu, mx, o));
                    const float m_new = fmaxf(m_run[j], mx);
                    const bool live = (h < nh) && (m_new > -INFINITY);
                    const float a = live ? exp2f(m_run[j] - m_new) : 1.f;
                    const float pr = (live && lane < nt) ? exp2f(s[j] - m_new) : 0.f;
                    float sum = pr;
                    for (int o = 16; o > 0; o >>= 1) sum += __shfl_xor_sync(0xffffffffu, sum, o);
                    if (live) { l_run[j] = l_run[j] * a + sum; m_run[j] = m_new; }
                    sm.p[h * GEN_TC + lane] = pr;
                    if (lane == 0) sm.alpha[h] = a;
                }
                __syncthreads();

                // --- a3: O += P V.  thread = value column(s), all heads
#pragma unroll
                for (int j = 0; j < 2; ++j) {
                    const int c = tid + j * GEN_THREADS;
                    if (j < ncol && c < dv) {
#pragma unroll
                        for (int h = 0; h < GEN_HB; ++h) acc[j][h] *= sm.alpha[h];
                        for (int t = 0; t < nt; ++t) {      // masked slots never enter (no 0 * NaN)
                            const float vv = __uint_as_float(((uint32_t)vbuf[(size_t)t * vrow + c]) << 16);
#pragma unroll
                            for (int h = 0; h < GEN_HB; ++h) acc[j][h] = fmaf(sm.p[h * GEN_TC + t], vv, acc[j][h]);
                        }
                    }
                }
                __syncthreads();
            }

            // --- publish: final result (single split) or partial (step a6 / a4 input)
            if (lane == 0) {
                if (warp < nh) { sm.m[warp] = m_run[0]; sm.l[warp] = l_run[0]; }
                if (warp + 8 < nh) { sm.m[warp + 8] = m_run[1]; sm.l[warp + 8] = l_run[1]; }
            }
            __syncthreads();
            if (g.n_splits == 1) {
#pragma unroll
                for (int j = 0; j < 2; ++j) {
                    const int c = tid + j * GEN_THREADS;
                    if (j < ncol && c < dv)
                        for (int h = 0; h < nh; ++h)
                            p.out[g.out_off + (int64_t)(h0 + h) * dv + c] = acc[j][h] / sm.l[h];
                }
                if (tid < nh)
                    p.lse[g.lse_off + h0 + tid] = (sm.m[tid] + log2f(sm.l[tid])) * 0.6931471805599453f;
            } else {
                float *ws = p.workspace + g.part_off;
#pragma unroll
                for (int j = 0; j < 2; ++j) {
                    const int c = tid + j * GEN_THREADS;
                    if (j < ncol && c < dv)
                        for (int h = 0; h < nh; ++h) ws[part_o_off(h0 + h, tile.split, g.n_splits, dv) + c] = acc[j][h];
                }
                if (tid < nh) {
                    float *mlp = ws + part_ml_off(m.group, h0 + tid, tile.split, g.n_splits, dv);
                    mlp[0] = sm.m[tid];
                    mlp[1] = sm.l[tid];
                }
            }
            __syncthreads();
        }
        if (g.n_splits > 1) {
            // all partial stores of this CTA happen-before the release increment
            __threadfence();
            __syncthreads();
            if (tid == 0) red_release_add(p.group_counters + (size_t)tile.group * kCounterStride, 1);
        }
    }
}

cudaError_t launch_decode_generic(const DecodeParams &p, int max_dk, int max_dv, bool any_kv_kind,
                                  int max_splits, int n_ctas, cudaStream_t stream)
{
    const size_t smem = generic_smem_bytes(max_dk, max_dv, any_kv_kind, max_splits);
    cudaError_t e = cudaFuncSetAttribute(cp_decode_generic_kernel,
                                         cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    int grid = p.n_tiles + p.n_combines;
    if (grid > n_ctas) grid = n_ctas;
    if (grid < 1) grid = 1;
    cp_decode_generic_kernel<<<grid, GEN_THREADS, smem, stream>>>(p, max_dk, max_dv, any_kv_kind ? 1 : 0);
    return cudaGetLastError();
}

}  // namespace cp
