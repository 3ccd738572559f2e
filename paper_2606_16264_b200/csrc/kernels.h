// kernels.h -- internal launch interfaces between api.cu and the kernel translation units.
#pragma once
#include <cuda_runtime.h>
#include <stddef.h>
#include <stdint.h>

#include "common.cuh"

namespace tropical {

cudaError_t launch_kv_append(const PoolDesc& pool, const BatchDesc& b, const void* k_new, const void* v_new,
                             cudaStream_t stream);
cudaError_t launch_kv_append_rope(const PoolDesc& pool, const BatchDesc& b, const void* k_new, const void* v_new,
                                  const float* cos_t, const float* sin_t, cudaStream_t stream);
cudaError_t launch_kv_gather(const PoolDesc& pool, const BatchDesc& b, int req, int n_keys, void* k_dense,
                             void* v_dense, cudaStream_t stream);
// NEXT-3 KV migration (csrc/kv_migrate.cu): source pool through src_pt -> destination pool under dst_pt
struct MigrateArgs {
    int Hkv, D, num_reqs, src_stride, dst_stride;
    const int* kv_lens;
    const int* src_pt;
    const int* dst_pt;
    const uint16_t* k_src;
    const uint16_t* v_src;
    uint16_t* k_dst;
    uint16_t* v_dst;
};
cudaError_t launch_kv_migrate(const MigrateArgs& args, int max_kv_len, cudaStream_t stream, int* launches);
cudaError_t launch_validate_batch(const PoolDesc& pool, const BatchDesc& b, int* first_bad_dev, cudaStream_t stream);
cudaError_t launch_attention_simt(const PoolDesc& pool, const BatchDesc& b, const void* q, void* out, float* lse,
                                  float scale_log2, cudaStream_t stream);
// k_new / v_new != nullptr: the fused step (the rows are read from there and appended to the pool inside the kernel)
cudaError_t launch_mixed_attention(const PoolDesc& pool, const BatchDesc& b, const void* q, const void* k_new,
                                   const void* v_new, void* out, float* lse, float scale_log2, void* workspace,
                                   cudaStream_t stream, int* launches);
void set_debug_grid(int num_ctas);
void set_debug_split_pages(int pages);
void set_debug_fused(int mode);
int read_wait_profile(unsigned long long* cycles, unsigned long long* calls, int n, int reset);
size_t profile_offset_bytes();
int read_timeline_append(unsigned long long* out16, int reset);  // 0 unless built with -DTROPICAL_TIMELINE
int read_timeline_mixed(unsigned long long* out16, int reset);
size_t mixed_workspace_bytes(int Hq, int Hkv, int D, int num_reqs, int total_q);

}  // namespace tropical
