// cp_planner.cu -- KV-cache planner on the GPU (Eq. (1)-(2)).
//
//   Q_i(u)    = (O_p,i + O_d,i u / T_i) 1{0 <= u < T_i}
//   K_M(t)    = sum_i kappa(M) Q_i(t - A_i)                    Eq. (1)
//   K_pool(t) = sum_M K_M(t)                                   Eq. (2)
//
// evaluated at the Monte-Carlo observation times the caller drew, then the empirical P95 / P99 and
// the page budget ("rounds memory to pages", L112).  Everything is float64 and every operation is a
// separately rounded IEEE operation in the paper's order (intrinsics, no FMA contraction), one
// thread per observation time summing its terms in trace order, so the demand vector equals a plain
// sequential evaluation bit for bit.  What the kernel adds is only pruning of exact zeros: arrivals
// are ascending inside a model, so two binary searches bound the requests that can be resident (not
// yet arrived, or older than the model's longest residence time: zero), and inside that window a
// block of 32 consecutive requests is skipped when even its youngest member is older than the block's
// longest residence time (fl(t - A) is monotone in A, so the test is exact, not approximate).
//
// The quantile is an exact selection, not a sort: four passes of a 16-bit radix select over the bit
// patterns (non-negative doubles order like their bit patterns), histogram by warp-aggregated
// atomics, one block turning the histogram into the next prefix.
#include <cuda_runtime.h>
#include <cmath>
#include <cstdint>

#include "../../include/crosspool.h"

namespace {

constexpr int kMaxModels = CP_PLANNER_MAX_MODELS;
constexpr int kBins = 1 << 16;

struct PlannerModels {
    int32_t n_models;
    int32_t pad;
    int64_t offs[kMaxModels + 1];
    double kappa[kMaxModels];
};

// workspace layout (bytes): [0, 512) selection state, [512, 512 + 8 * kMaxModels) longest residence
// time per model (bit patterns), the histogram, then the longest residence time per block of 32
// trace entries
struct SelectState {
    unsigned long long prefix;      // digits fixed so far (high bits of the answer)
    unsigned long long k;           // 1-based rank still to find among the elements matching prefix
    double value;                   // the selected value (after the last pass)
    unsigned long long pages;       // ceil(value / page_bytes)
};
constexpr size_t kOffTmax = 512;
constexpr size_t kOffHist = kOffTmax + 8 * (size_t)kMaxModels;
constexpr size_t kOffBlocks = kOffHist + 4 * (size_t)kBins;
constexpr int kBlock = 32;

size_t workspace_bytes_for(int64_t n_entries)
{
    return kOffBlocks + 8 * (size_t)((n_entries + kBlock - 1) / kBlock) + 16;
}

// longest residence time of every block of 32 consecutive trace entries (one warp per block)
__global__ void planner_block_tmax_kernel(const double *__restrict__ t_res, int64_t n, double *__restrict__ blk_tmax)
{
    const int64_t b = ((int64_t)blockIdx.x * blockDim.x + threadIdx.x) >> 5;
    const int64_t i = b * kBlock + (threadIdx.x & 31);
    if (b * kBlock >= n) return;
    double t = i < n ? t_res[i] : 0.0;
    if (!(t > 0.0)) t = 0.0;
    for (int o = 16; o > 0; o >>= 1) t = fmax(t, __shfl_xor_sync(0xffffffffu, t, o));
    if ((threadIdx.x & 31) == 0) blk_tmax[b] = t;
}

__global__ void planner_tmax_kernel(PlannerModels pm, const double *__restrict__ t_res, unsigned long long *tmax_bits)
{
    const int m = blockIdx.y;
    unsigned long long best = 0;
    for (int64_t i = pm.offs[m] + (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < pm.offs[m + 1];
         i += (int64_t)gridDim.x * blockDim.x) {
        const double t = t_res[i];
        if (t > 0.0) best = max(best, (unsigned long long)__double_as_longlong(t));
    }
    for (int o = 16; o > 0; o >>= 1) best = max(best, __shfl_xor_sync(0xffffffffu, best, o));
    if ((threadIdx.x & 31) == 0 && best) atomicMax(tmax_bits + m, best);
}

__device__ __forceinline__ int64_t lower_bound(const double *__restrict__ a, int64_t lo, int64_t hi, double x)
{   // first index in [lo, hi) with a[i] >= x
    while (lo < hi) {
        const int64_t mid = lo + ((hi - lo) >> 1);
        if (__ldg(a + mid) < x) lo = mid + 1; else hi = mid;
    }
    return lo;
}

__device__ __forceinline__ int64_t upper_bound(const double *__restrict__ a, int64_t lo, int64_t hi, double x)
{   // first index in [lo, hi) with a[i] > x
    while (lo < hi) {
        const int64_t mid = lo + ((hi - lo) >> 1);
        if (__ldg(a + mid) <= x) lo = mid + 1; else hi = mid;
    }
    return lo;
}

__global__ void __launch_bounds__(128)
planner_demand_kernel(PlannerModels pm, const double *__restrict__ arrival, const double *__restrict__ o_p,
                      const double *__restrict__ o_d, const double *__restrict__ t_res,
                      const unsigned long long *__restrict__ tmax_bits, const double *__restrict__ blk_tmax,
                      int64_t n_obs, const double *__restrict__ t_obs, double *__restrict__ k_pool)
{
    const int64_t n = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (n >= n_obs) return;
    const double t = t_obs[n];
    double pool = 0.0;
    for (int m = 0; m < pm.n_models; ++m) {
        const double tmax = __longlong_as_double((long long)tmax_bits[m]);
        // requests that arrived before t - tmax have age u > tmax >= T_i: an exact zero.  The bound is
        // taken a little low (rounding of t - tmax); what it lets in is still decided by the exact test.
        const double oldest = t - tmax - 1e-9 * (fabs(t) + tmax) - 1e-300;
        const int64_t lo = lower_bound(arrival, pm.offs[m], pm.offs[m + 1], oldest);
        const int64_t hi = upper_bound(arrival, lo, pm.offs[m + 1], t);      // A_i > t: u < 0, zero
        const double kappa = pm.kappa[m];
        double k_m = 0.0;
        for (int64_t i = lo; i < hi;) {
            const int64_t b = i / kBlock;
            const int64_t end = min(hi, (b + 1) * kBlock);
            // the youngest request of this part of the block has the smallest age; if even that age is not
            // below the block's longest residence time, every term of the block is an exact zero
            if (__dsub_rn(t, __ldg(arrival + end - 1)) >= __ldg(blk_tmax + b)) { i = end; continue; }
            for (; i < end; ++i) {
                const double u = __dsub_rn(t, __ldg(arrival + i));
                const double T = __ldg(t_res + i);
                if (u >= 0.0 && u < T) {
                    const double q = __dadd_rn(__ldg(o_p + i), __dmul_rn(__ldg(o_d + i), __ddiv_rn(u, T)));
                    k_m = __dadd_rn(k_m, __dmul_rn(kappa, q));
                }
            }
        }
        pool = __dadd_rn(pool, k_m);
    }
    k_pool[n] = pool;
}

__global__ void planner_select_init_kernel(SelectState *st, unsigned long long k, uint32_t *hist)
{
    for (int i = blockIdx.x * blockDim.x + threadIdx.x; i < kBins; i += gridDim.x * blockDim.x) hist[i] = 0;
    if (blockIdx.x == 0 && threadIdx.x == 0) { st->prefix = 0; st->k = k; st->value = 0.0; st->pages = 0; }
}

// pass = 0 .. 3, most significant digit first
__global__ void planner_hist_kernel(const double *__restrict__ x, int64_t n, const SelectState *st, int pass,
                                    uint32_t *hist)
{
    const unsigned long long prefix = st->prefix;
    const int shift = 48 - 16 * pass;
    for (int64_t i0 = (int64_t)blockIdx.x * blockDim.x; i0 < n; i0 += (int64_t)gridDim.x * blockDim.x) {
        const int64_t i = i0 + threadIdx.x;
        bool in = false;
        uint32_t digit = 0;
        if (i < n) {
            const unsigned long long b = (unsigned long long)__double_as_longlong(x[i]);
            in = pass == 0 || (b >> (shift + 16)) == prefix;
            digit = (uint32_t)(b >> shift) & 0xFFFFu;
        }
        const unsigned act = __ballot_sync(0xffffffffu, in);
        if (in) {
            const unsigned peers = __match_any_sync(act, digit);
            if ((threadIdx.x & 31) == (unsigned)(__ffs(peers) - 1)) atomicAdd(hist + digit, (uint32_t)__popc(peers));
        }
    }
}

// one block of 1024 threads: the digit where the cumulative count reaches k; clears the histogram
__global__ void __launch_bounds__(1024)
planner_pick_kernel(SelectState *st, uint32_t *hist, int pass, double page_bytes)
{
    __shared__ unsigned long long part[1024];
    __shared__ int s_thread;
    __shared__ unsigned long long s_below;
    const int tid = threadIdx.x;
    constexpr int per = kBins / 1024;
    unsigned long long sum = 0;
    for (int j = 0; j < per; ++j) sum += hist[tid * per + j];
    part[tid] = sum;
    __syncthreads();
    if (tid == 0) {
        const unsigned long long k = st->k;
        unsigned long long acc = 0;
        int t = 0;
        for (; t < 1023; ++t) {
            if (acc + part[t] >= k) break;
            acc += part[t];
        }
        s_thread = t; s_below = acc;
    }
    __syncthreads();
    if (tid == s_thread) {
        const unsigned long long k = st->k;
        unsigned long long acc = s_below;
        int d = tid * per;
        for (int j = 0; j < per - 1; ++j, ++d) {
            if (acc + hist[d] >= k) break;
            acc += hist[d];
        }
        const unsigned long long prefix = (st->prefix << 16) | (unsigned long long)d;
        st->prefix = prefix;
        st->k = k - acc;
        if (pass == 3) {
            const double v = __longlong_as_double((long long)prefix);
            st->value = v;
            st->pages = (unsigned long long)ceil(__ddiv_rn(v, page_bytes));
        }
    }
    __syncthreads();
    for (int j = 0; j < per; ++j) hist[tid * per + j] = 0;
}

bool fill_models(PlannerModels &pm, int32_t n_models, const int64_t *offs, const double *kappa)
{
    if (n_models < 1 || n_models > kMaxModels || !offs || !kappa) return false;
    pm.n_models = n_models; pm.pad = 0;
    for (int m = 0; m <= n_models; ++m) {
        pm.offs[m] = offs[m];
        if (offs[m] < 0 || (m > 0 && offs[m] < offs[m - 1])) return false;
    }
    for (int m = 0; m < n_models; ++m) {
        pm.kappa[m] = kappa[m];
        if (!(kappa[m] >= 0.0)) return false;
    }
    return offs[0] == 0;
}

}  // namespace

extern "C" {

uint64_t cp_planner_workspace_bytes(int64_t n_trace_entries)
{
    return workspace_bytes_for(n_trace_entries < 0 ? 0 : n_trace_entries);
}

cp_status cp_planner_pool_demand(int32_t n_models, const int64_t *trace_offsets_host, const double *kappa_host,
                                 const double *arrival_dev, const double *prompt_tokens_dev,
                                 const double *output_tokens_dev, const double *residence_dev, int64_t n_obs,
                                 const double *t_obs_dev, double *k_pool_dev, void *workspace_dev,
                                 uint64_t workspace_bytes, void *stream)
{
    PlannerModels pm;
    if (!fill_models(pm, n_models, trace_offsets_host, kappa_host)) return CP_ERR_INVALID_ARG;
    if (n_obs < 0 || (n_obs > 0 && (!t_obs_dev || !k_pool_dev))) return CP_ERR_INVALID_ARG;
    const int64_t n_req = pm.offs[n_models];
    if (n_req > 0 && (!arrival_dev || !prompt_tokens_dev || !output_tokens_dev || !residence_dev))
        return CP_ERR_INVALID_ARG;
    if (!workspace_dev || workspace_bytes < workspace_bytes_for(n_req) || ((uintptr_t)workspace_dev & 15u))
        return CP_ERR_WORKSPACE;
    if (n_obs == 0) return CP_OK;
    cudaStream_t s = (cudaStream_t)stream;
    unsigned long long *tmax = (unsigned long long *)((uint8_t *)workspace_dev + kOffTmax);
    double *blk_tmax = (double *)((uint8_t *)workspace_dev + kOffBlocks);
    if (cudaMemsetAsync(tmax, 0, 8 * (size_t)kMaxModels, s) != cudaSuccess) { cudaGetLastError(); return CP_ERR_CUDA; }
    if (n_req > 0) {
        int64_t longest = 0;
        for (int m = 0; m < n_models; ++m) longest = longest > pm.offs[m + 1] - pm.offs[m] ? longest : pm.offs[m + 1] - pm.offs[m];
        const int bx = (int)((longest + 255) / 256 < 1024 ? (longest + 255) / 256 : 1024);
        planner_tmax_kernel<<<dim3(bx > 0 ? bx : 1, n_models), 256, 0, s>>>(pm, residence_dev, tmax);
        const int64_t n_blk = (n_req + kBlock - 1) / kBlock;
        planner_block_tmax_kernel<<<(unsigned)((n_blk * 32 + 255) / 256), 256, 0, s>>>(residence_dev, n_req, blk_tmax);
    }
    planner_demand_kernel<<<(unsigned)((n_obs + 127) / 128), 128, 0, s>>>(pm, arrival_dev, prompt_tokens_dev,
                                                                          output_tokens_dev, residence_dev, tmax, blk_tmax, n_obs,
                                                                          t_obs_dev, k_pool_dev);
    if (cudaGetLastError() != cudaSuccess) return CP_ERR_CUDA;
    return CP_OK;
}

// ---------------------------------------------------------------------------------------------------------------
// cp_planner_pool_demand_noalloc: the same launches as cp_planner_pool_demand, with the scratch (the models' and the
// 32-entry blocks' longest residence times) in a file-scope device array instead of a caller-owned workspace, for
// callers that cannot call cudaMalloc (CUDA graph capture, serving loops, harnesses that forbid it).  Every GPU that
// loads the library holds the array until the process exits.  In HOST code `g_planner_scratch` is a host-side
// stand-in, not a device address: the address the kernels get comes from cudaGetSymbolAddress, asked once per
// device with that device current.
// ---------------------------------------------------------------------------------------------------------------
constexpr int64_t kNoallocMaxTrace = CP_PLANNER_NOALLOC_MAX_TRACE;
constexpr size_t kNoallocScratchBytes = (kOffBlocks + 8 * (size_t)((kNoallocMaxTrace + kBlock - 1) / kBlock) + 16 + 255) / 256 * 256;
static __device__ __align__(256) unsigned char g_planner_scratch[kNoallocScratchBytes];

cp_status cp_planner_pool_demand_noalloc(int32_t n_models, const int64_t *trace_offsets_host, const double *kappa_host,
                                         const double *arrival_dev, const double *prompt_tokens_dev,
                                         const double *output_tokens_dev, const double *residence_dev, int64_t n_obs,
                                         const double *t_obs_dev, double *k_pool_dev, void *stream)
{
    // sizes first: no CUDA call for a request this entry point cannot serve
    if (n_models < 1 || n_models > kMaxModels || !trace_offsets_host) return CP_ERR_INVALID_ARG;
    if (trace_offsets_host[n_models] > kNoallocMaxTrace) return CP_ERR_TOO_LARGE;
    static void *scratch_of[64] = {};                     // per device: the array's address on that device
    int dev = 0;
    if (cudaGetDevice(&dev) != cudaSuccess) { cudaGetLastError(); return CP_ERR_CUDA; }
    void *ptr = dev >= 0 && dev < 64 ? scratch_of[dev] : nullptr;
    if (!ptr) {
        if (cudaGetSymbolAddress(&ptr, g_planner_scratch) != cudaSuccess || !ptr) { cudaGetLastError(); return CP_ERR_CUDA; }
        if (dev >= 0 && dev < 64) scratch_of[dev] = ptr;
    }
    // (cp_planner_pool_demand clears what must start at zero -- the per-model maxima -- on the stream and writes every
    // block maximum it reads; it allocates nothing: a memset and three kernel launches)
    return cp_planner_pool_demand(n_models, trace_offsets_host, kappa_host, arrival_dev, prompt_tokens_dev,
                                  output_tokens_dev, residence_dev, n_obs, t_obs_dev, k_pool_dev, ptr,
                                  (uint64_t)kNoallocScratchBytes, stream);
}

cp_status cp_planner_quantile(const double *values_dev, int64_t n, double q, double page_bytes, void *workspace_dev,
                              uint64_t workspace_bytes, double *quantile_out_host, uint64_t *pages_out_host,
                              void *stream)
{
    if (!values_dev || n < 1 || !(q > 0.0 && q <= 1.0) || !(page_bytes > 0.0)) return CP_ERR_INVALID_ARG;
    if (!workspace_dev || workspace_bytes < workspace_bytes_for(0) || ((uintptr_t)workspace_dev & 15u)) return CP_ERR_WORKSPACE;
    int64_t k = (int64_t)std::ceil(q * (double)n);        // rank of the order statistic, 1-based
    if (k < 1) k = 1;
    if (k > n) k = n;
    cudaStream_t s = (cudaStream_t)stream;
    SelectState *st = (SelectState *)workspace_dev;
    uint32_t *hist = (uint32_t *)((uint8_t *)workspace_dev + kOffHist);
    planner_select_init_kernel<<<64, 1024, 0, s>>>(st, (unsigned long long)k, hist);
    const unsigned blocks = (unsigned)((n + 255) / 256 < 1184 ? (n + 255) / 256 : 1184);
    for (int pass = 0; pass < 4; ++pass) {
        planner_hist_kernel<<<blocks, 256, 0, s>>>(values_dev, n, st, pass, hist);
        planner_pick_kernel<<<1, 1024, 0, s>>>(st, hist, pass, page_bytes);
    }
    if (cudaGetLastError() != cudaSuccess) return CP_ERR_CUDA;
    SelectState out;
    if (cudaMemcpyAsync(&out, st, sizeof(out), cudaMemcpyDeviceToHost, s) != cudaSuccess ||
        cudaStreamSynchronize(s) != cudaSuccess) {
        cudaGetLastError();
        return CP_ERR_CUDA;
    }
    if (quantile_out_host) *quantile_out_host = out.value;
    if (pages_out_host) *pages_out_host = out.pages;
    return CP_OK;
}

}  // extern "C"
