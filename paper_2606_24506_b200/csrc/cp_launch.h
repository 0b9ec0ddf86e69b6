// cp_launch.h -- host-callable launchers of the CUDA kernels (internal to libcrosspool).
#pragma once
#include <cuda_runtime.h>
#include <cstdint>
#include "cp_internal.h"

namespace cp {

void launch_gather(const uint8_t *arena, uint32_t page_tokens, uint32_t page_bytes,
                   const int32_t *page_ids_dev, int kind, int n_kv_heads, int d_k, int d_v,
                   int context_len, void *k_out, void *v_out, int n_sm, cudaStream_t stream);

void launch_append(uint8_t *arena, uint32_t page_tokens, uint32_t page_bytes, const int32_t *page_table,
                   int max_ppr, const DevModel *models, const AppendRec *recs, int n_requests,
                   const uint16_t *k_new, const uint16_t *v_new, cudaStream_t stream);

size_t generic_smem_bytes(int max_dk, int max_dv, bool any_kv_kind, int max_splits);
cudaError_t launch_decode_generic(const DecodeParams &p, int max_dk, int max_dv, bool any_kv_kind,
                                  int max_splits, int n_ctas, cudaStream_t stream);

// tensor-core MQA/GQA path (cp_kernels_kv.cu)
bool kv_fast_supported(int page_tokens);
bool make_arena_tensor_map(void *out_map, const void *arena, uint64_t total_rows, uint32_t row_elems,
                           uint32_t box_cols, uint32_t box_rows);
cudaError_t launch_decode_kv(const DecodeParams &p, const void *tmap, int rows_per_page, int n_ctas,
                             cudaStream_t stream);

// tcgen05 MQA/GQA path, tokens on the MMA M dimension (cp_kernels_kvt.cu)
bool kvt_supported(int page_tokens);
int kvt_pad_rows(int max_group);      // N of the instantiation for groups of up to max_group rows, 0 = none
cudaError_t launch_decode_kvt(const DecodeParams &p, const void *tmap, int rows_per_page, int n_ctas, int max_group,
                              cudaStream_t stream);

// tcgen05 MLA path (cp_kernels_mla.cu)
bool mla_fast_supported(int page_tokens, uint32_t page_bytes);
bool make_mla_tensor_map(void *out_map, const void *arena, uint64_t total_rows);
cudaError_t launch_decode_mla(const DecodeParams &p, const void *tmap, int rows_per_page, int n_ctas,
                              cudaStream_t stream);

// tcgen05 MLA path on CTA pairs (cp_kernels_mla2.cu)
bool make_mla2_tensor_maps(void *out_map9, void *out_map2, const void *arena, uint64_t total_rows);
cudaError_t launch_decode_mla2(const DecodeParams &p, const void *tmap9, const void *tmap2, int rows_per_page,
                               int n_ctas, cudaStream_t stream);

}  // namespace cp
