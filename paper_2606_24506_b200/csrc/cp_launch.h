// cp_launch.h -- host-callable launchers of the CUDA kernels (internal to libcrosspool).
#pragma once
#include <cuda_runtime.h>
#include <cstdint>
#include "cp_internal.h"

namespace cp {

void launch_gather(const uint8_t *arena, uint32_t page_tokens, uint32_t page_bytes,
                   const int32_t *page_ids_dev, int kind, int n_kv_heads, int d_k, int d_v,
                   int context_len, void *k_out, void *v_out, int n_sm, cudaStream_t stream);

size_t generic_smem_bytes(int max_dk, int max_dv, bool any_kv_kind, int max_splits);
cudaError_t launch_decode_generic(const DecodeParams &p, int max_dk, int max_dv, bool any_kv_kind,
                                  int max_splits, int n_ctas, cudaStream_t stream);

}  // namespace cp
