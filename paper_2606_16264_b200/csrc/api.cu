// api.cu -- the extern "C" boundary declared in include/tropical.h: argument validation,
// workspace carving, launches.  Every step of the path runs in this library's kernels.
#include <cuda_runtime.h>
#include <math.h>
#include <stdio.h>
#include <string.h>

#include <atomic>

#include "../../include/tropical.h"
#include "../../include/tropical_debug.h"
#include "kernels.h"

using namespace tropical;

namespace {

thread_local char g_cuda_err[256] = "";
thread_local int g_launches = 0;

int cuda_fail(cudaError_t e, const char* where) {
    snprintf(g_cuda_err, sizeof g_cuda_err, "%s: %s", where, cudaGetErrorString(e));
    return TROPICAL_ERR_CUDA;
}

int check_pool(const tropical_kv_pool_t* p) {
    if (p == nullptr || p->k_pool == nullptr || p->v_pool == nullptr) return TROPICAL_ERR_INVALID_ARG;
    if (p->num_q_heads <= 0 || p->num_kv_heads <= 0 || p->num_pages <= 0) return TROPICAL_ERR_INVALID_ARG;
    if (p->num_q_heads % p->num_kv_heads != 0) return TROPICAL_ERR_INVALID_ARG;
    if (p->head_dim != 64 && p->head_dim != 128) return TROPICAL_ERR_UNSUPPORTED;
    if (p->page_size != kPageSize) return TROPICAL_ERR_UNSUPPORTED;
    if (p->num_q_heads / p->num_kv_heads > 64) return TROPICAL_ERR_UNSUPPORTED;
    if (((uintptr_t)p->k_pool & 255) || ((uintptr_t)p->v_pool & 255)) return TROPICAL_ERR_INVALID_ARG;
    return TROPICAL_OK;
}

int check_scalars(const tropical_kv_pool_t* p, int num_reqs, int total_q, int max_kv_len, int stride) {
    if (num_reqs < 0 || total_q < 0 || max_kv_len < 0 || stride < 0) return TROPICAL_ERR_INVALID_ARG;
    if ((long long)stride * p->page_size < (long long)max_kv_len) return TROPICAL_ERR_INVALID_ARG;
    if (total_q > 0 && num_reqs == 0) return TROPICAL_ERR_INVALID_ARG;
    return TROPICAL_OK;
}

int check_batch(const tropical_kv_pool_t* p, const tropical_batch_t* b) {
    if (b == nullptr) return TROPICAL_ERR_INVALID_ARG;
    int rc = check_scalars(p, b->num_reqs, b->total_q, b->max_kv_len, b->page_table_stride);
    if (rc != TROPICAL_OK) return rc;
    if (b->num_reqs > 0 && (b->q_lens == nullptr || b->ctx_lens == nullptr || b->q_offsets == nullptr ||
                            b->page_table == nullptr))
        return TROPICAL_ERR_INVALID_ARG;
    return TROPICAL_OK;
}

PoolDesc to_pool(const tropical_kv_pool_t* p) {
    PoolDesc d;
    d.Hq = p->num_q_heads;
    d.Hkv = p->num_kv_heads;
    d.D = p->head_dim;
    d.num_pages = p->num_pages;
    d.k_pool = (const uint16_t*)p->k_pool;
    d.v_pool = (const uint16_t*)p->v_pool;
    return d;
}

BatchDesc to_batch(const tropical_batch_t* b) {
    BatchDesc d;
    d.num_reqs = b->num_reqs;
    d.total_q = b->total_q;
    d.max_kv_len = b->max_kv_len;
    d.stride = b->page_table_stride;
    d.q_lens = b->q_lens;
    d.ctx_lens = b->ctx_lens;
    d.q_offsets = b->q_offsets;
    d.page_table = b->page_table;
    return d;
}

size_t align_up(size_t x, size_t a) { return (x + a - 1) / a * a; }

// k_new / v_new != nullptr: the fused step
int mixed_attention_impl(const tropical_kv_pool_t* pool, const tropical_batch_t* batch, const void* q,
                         const void* k_new, const void* v_new, void* out, float* lse, float sm_scale, void* workspace,
                         size_t workspace_bytes, cudaStream_t stream, int* launches) {
    (void)workspace_bytes;
    const float scale = sm_scale > 0.f ? sm_scale : 1.0f / sqrtf((float)pool->head_dim);
    const float scale_log2 = scale * 1.4426950408889634f;
    cudaError_t e = launch_mixed_attention(to_pool(pool), to_batch(batch), q, k_new, v_new, out, lse, scale_log2,
                                           workspace, stream, launches);
    if (e != cudaSuccess) return cuda_fail(e, "mixed_attention");
    return TROPICAL_OK;
}


// ---- built-in scratch for tropical_mixed_attention_static (include/tropical.h) ----------------------------------
// The step's work lists and split-K partials normally live in a workspace the caller allocates.  A caller that may
// not allocate device memory gets this array instead: it is part of the loaded module, so every GPU that loads
// libtropical.so holds TROPICAL_STATIC_WORKSPACE_BYTES of it from module load until the process exits, used or not.
// In host code `g_static_ws` is only a handle for the runtime's symbol calls, never a device address: the address
// this device gave the array comes from cudaGetSymbolAddress, once per device, with that device current.
static __device__ __align__(256) unsigned char g_static_ws[TROPICAL_STATIC_WORKSPACE_BYTES];

constexpr int kStaticWsDevices = 64;
std::atomic<void*> g_static_ws_addr[kStaticWsDevices];  // per device: the array's address there, nullptr = not asked yet

// Address of g_static_ws on the current device (looked up on the first call per device, remembered afterwards).
int static_workspace(void** ws) {
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return cuda_fail(e, "mixed_attention_static: cudaGetDevice");
    const bool cached = dev >= 0 && dev < kStaticWsDevices;
    void* p = cached ? g_static_ws_addr[dev].load(std::memory_order_acquire) : nullptr;
    if (p == nullptr) {
        e = cudaGetSymbolAddress(&p, g_static_ws);
        if (e != cudaSuccess) return cuda_fail(e, "mixed_attention_static: cudaGetSymbolAddress");
        if (p == nullptr || ((uintptr_t)p & 255)) {
            snprintf(g_cuda_err, sizeof g_cuda_err, "mixed_attention_static: static workspace address %p unusable", p);
            return TROPICAL_ERR_CUDA;
        }
        if (cached) g_static_ws_addr[dev].store(p, std::memory_order_release);
    }
    *ws = p;
    return TROPICAL_OK;
}

}  // namespace

extern "C" {

int tropical_kv_append(const tropical_kv_pool_t* pool, const tropical_batch_t* batch, const void* k_new,
                       const void* v_new, void* cuda_stream) {
    g_launches = 0;
    int rc = check_pool(pool);
    if (rc != TROPICAL_OK) return rc;
    rc = check_batch(pool, batch);
    if (rc != TROPICAL_OK) return rc;
    if (batch->total_q == 0) return TROPICAL_OK;
    if (k_new == nullptr || v_new == nullptr) return TROPICAL_ERR_INVALID_ARG;
    cudaError_t e = launch_kv_append(to_pool(pool), to_batch(batch), k_new, v_new, (cudaStream_t)cuda_stream);
    if (e != cudaSuccess) return cuda_fail(e, "kv_append");
    g_launches = 1;
    return TROPICAL_OK;
}

int tropical_kv_append_rope(const tropical_kv_pool_t* pool, const tropical_batch_t* batch, const void* k_new,
                            const void* v_new, const float* cos_table, const float* sin_table, int32_t table_len,
                            void* cuda_stream) {
    g_launches = 0;
    int rc = check_pool(pool);
    if (rc != TROPICAL_OK) return rc;
    rc = check_batch(pool, batch);
    if (rc != TROPICAL_OK) return rc;
    if (table_len < 0 || table_len < batch->max_kv_len) return TROPICAL_ERR_INVALID_ARG;  // a row for every position
    if (batch->total_q == 0) return TROPICAL_OK;
    if (k_new == nullptr || v_new == nullptr || cos_table == nullptr || sin_table == nullptr) return TROPICAL_ERR_INVALID_ARG;
    if (((uintptr_t)cos_table & 15) || ((uintptr_t)sin_table & 15)) return TROPICAL_ERR_INVALID_ARG;
    cudaError_t e = launch_kv_append_rope(to_pool(pool), to_batch(batch), k_new, v_new, cos_table, sin_table,
                                          (cudaStream_t)cuda_stream);
    if (e != cudaSuccess) return cuda_fail(e, "kv_append_rope");
    g_launches = 1;
    return TROPICAL_OK;
}

int tropical_kv_gather(const tropical_kv_pool_t* pool, const tropical_batch_t* batch, int32_t req, int32_t n_keys,
                       void* k_dense, void* v_dense, void* cuda_stream) {
    g_launches = 0;
    int rc = check_pool(pool);
    if (rc != TROPICAL_OK) return rc;
    rc = check_batch(pool, batch);
    if (rc != TROPICAL_OK) return rc;
    if (req < 0 || req >= batch->num_reqs || n_keys < 0) return TROPICAL_ERR_INVALID_ARG;
    if ((long long)n_keys > (long long)batch->page_table_stride * pool->page_size) return TROPICAL_ERR_INVALID_ARG;
    if (n_keys == 0) return TROPICAL_OK;
    if (k_dense == nullptr || v_dense == nullptr) return TROPICAL_ERR_INVALID_ARG;
    cudaError_t e =
        launch_kv_gather(to_pool(pool), to_batch(batch), req, n_keys, k_dense, v_dense, (cudaStream_t)cuda_stream);
    if (e != cudaSuccess) return cuda_fail(e, "kv_gather");
    g_launches = 1;
    return TROPICAL_OK;
}

int tropical_kv_migrate(const tropical_kv_pool_t* src, const tropical_kv_pool_t* dst, const tropical_migration_t* mig,
                        void* cuda_stream) {
    g_launches = 0;
    int rc = check_pool(src);
    if (rc != TROPICAL_OK) return rc;
    rc = check_pool(dst);
    if (rc != TROPICAL_OK) return rc;
    if (src->num_kv_heads != dst->num_kv_heads || src->head_dim != dst->head_dim || src->page_size != dst->page_size)
        return TROPICAL_ERR_INVALID_ARG;
    if (mig == nullptr || mig->num_reqs < 0 || mig->max_kv_len < 0 || mig->src_page_table_stride < 0 ||
        mig->dst_page_table_stride < 0)
        return TROPICAL_ERR_INVALID_ARG;
    const long long need_pages = ((long long)mig->max_kv_len + kPageSize - 1) / kPageSize;
    if (mig->src_page_table_stride < need_pages || mig->dst_page_table_stride < need_pages) return TROPICAL_ERR_INVALID_ARG;
    if (mig->num_reqs == 0 || mig->max_kv_len == 0) return TROPICAL_OK;
    if (mig->kv_lens == nullptr || mig->src_page_table == nullptr || mig->dst_page_table == nullptr)
        return TROPICAL_ERR_INVALID_ARG;
    MigrateArgs a;
    a.Hkv = src->num_kv_heads;
    a.D = src->head_dim;
    a.num_reqs = mig->num_reqs;
    a.src_stride = mig->src_page_table_stride;
    a.dst_stride = mig->dst_page_table_stride;
    a.kv_lens = mig->kv_lens;
    a.src_pt = mig->src_page_table;
    a.dst_pt = mig->dst_page_table;
    a.k_src = (const uint16_t*)src->k_pool;
    a.v_src = (const uint16_t*)src->v_pool;
    a.k_dst = (uint16_t*)dst->k_pool;
    a.v_dst = (uint16_t*)dst->v_pool;
    int launches = 0;
    cudaError_t e = launch_kv_migrate(a, mig->max_kv_len, (cudaStream_t)cuda_stream, &launches);
    if (e != cudaSuccess) return cuda_fail(e, "kv_migrate");
    g_launches = launches;
    return TROPICAL_OK;
}

int tropical_enable_peer_access(int32_t peer_device) {
    int dev = 0, can = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return cuda_fail(e, "enable_peer_access");
    if (peer_device == dev) return TROPICAL_OK;
    e = cudaDeviceCanAccessPeer(&can, dev, peer_device);
    if (e != cudaSuccess) return cuda_fail(e, "enable_peer_access");
    if (!can) return TROPICAL_ERR_UNSUPPORTED;
    e = cudaDeviceEnablePeerAccess(peer_device, 0);
    if (e == cudaErrorPeerAccessAlreadyEnabled) {
        cudaGetLastError();  // clear the sticky-less error
        return TROPICAL_OK;
    }
    if (e != cudaSuccess) return cuda_fail(e, "enable_peer_access");
    return TROPICAL_OK;
}

int tropical_validate_batch(const tropical_kv_pool_t* pool, const tropical_batch_t* batch, int32_t* first_bad_request,
                            void* scratch, void* cuda_stream) {
    g_launches = 0;
    int rc = check_pool(pool);
    if (rc != TROPICAL_OK) return rc;
    rc = check_batch(pool, batch);
    if (rc != TROPICAL_OK) return rc;
    if (scratch == nullptr || ((uintptr_t)scratch & 3)) return TROPICAL_ERR_WORKSPACE;
    cudaStream_t stream = (cudaStream_t)cuda_stream;
    int* d_bad = (int*)scratch;  // caller-owned: the library allocates nothing
    int bad = 0x7fffffff;
    cudaError_t e = cudaMemcpyAsync(d_bad, &bad, sizeof bad, cudaMemcpyHostToDevice, stream);
    if (e == cudaSuccess) e = launch_validate_batch(to_pool(pool), to_batch(batch), d_bad, stream);
    if (e == cudaSuccess) e = cudaMemcpyAsync(&bad, d_bad, sizeof bad, cudaMemcpyDeviceToHost, stream);
    if (e == cudaSuccess) e = cudaStreamSynchronize(stream);
    if (e != cudaSuccess) return cuda_fail(e, "validate_batch");
    g_launches = 1;
    if (bad != 0x7fffffff) {
        if (first_bad_request != nullptr) *first_bad_request = bad;
        return TROPICAL_ERR_INVALID_ARG;
    }
    return TROPICAL_OK;
}

size_t tropical_workspace_bytes(const tropical_kv_pool_t* pool, int32_t num_reqs, int32_t total_q,
                                int32_t max_kv_len) {
    if (pool == nullptr || num_reqs < 0 || total_q < 0 || max_kv_len < 0) return 0;
    if (pool->num_q_heads <= 0 || pool->num_kv_heads <= 0 || pool->num_q_heads % pool->num_kv_heads) return 0;
    if (pool->head_dim != 64 && pool->head_dim != 128) return 0;
    (void)max_kv_len;  // split-K partials are bounded by the unit budget, not by the context length
    return mixed_workspace_bytes(pool->num_q_heads, pool->num_kv_heads, pool->head_dim, num_reqs, total_q);
}

int tropical_mixed_attention(const tropical_kv_pool_t* pool, const tropical_batch_t* batch, const void* q, void* out,
                             float* lse, float sm_scale, void* workspace, size_t workspace_bytes,
                             void* cuda_stream) {
    g_launches = 0;
    int rc = check_pool(pool);
    if (rc != TROPICAL_OK) return rc;
    rc = check_batch(pool, batch);
    if (rc != TROPICAL_OK) return rc;
    if (batch->total_q == 0) return TROPICAL_OK;
    if (q == nullptr || out == nullptr) return TROPICAL_ERR_INVALID_ARG;
    const size_t need = tropical_workspace_bytes(pool, batch->num_reqs, batch->total_q, batch->max_kv_len);
    if (workspace == nullptr || ((uintptr_t)workspace & 255) || workspace_bytes < need) return TROPICAL_ERR_WORKSPACE;
    return mixed_attention_impl(pool, batch, q, nullptr, nullptr, out, lse, sm_scale, workspace, workspace_bytes,
                                (cudaStream_t)cuda_stream, &g_launches);
}

int tropical_mixed_attention_static(const tropical_kv_pool_t* pool, const tropical_batch_t* batch, const void* q,
                                    void* out, float* lse, float sm_scale, void* cuda_stream) {
    g_launches = 0;
    int rc = check_pool(pool);
    if (rc != TROPICAL_OK) return rc;
    rc = check_batch(pool, batch);
    if (rc != TROPICAL_OK) return rc;
    if (batch->total_q == 0) return TROPICAL_OK;
    if (q == nullptr || out == nullptr) return TROPICAL_ERR_INVALID_ARG;
    // the size check comes before any CUDA call: a step that does not fit is refused, never run on a short array
    const size_t need = tropical_workspace_bytes(pool, batch->num_reqs, batch->total_q, batch->max_kv_len);
    if (need == 0 || need > (size_t)TROPICAL_STATIC_WORKSPACE_BYTES) {
        snprintf(g_cuda_err, sizeof g_cuda_err,
                 "mixed_attention_static: this step needs %zu bytes of scratch, the built-in array holds %zu "
                 "(TROPICAL_STATIC_WORKSPACE_BYTES); use tropical_mixed_attention with a caller workspace",
                 need, (size_t)TROPICAL_STATIC_WORKSPACE_BYTES);
        return TROPICAL_ERR_STATIC_CAPACITY;
    }
    void* ws = nullptr;
    rc = static_workspace(&ws);
    if (rc != TROPICAL_OK) return rc;
    // Nothing in the array has to be zero when the kernels start: the tile-directory kernel rewrites the header, both
    // ticket counters and every split group's arrival counter it will use, and the split-K partials are written by
    // the decode units before the combine reads them.  What the previous call left behind is never read.
    return mixed_attention_impl(pool, batch, q, nullptr, nullptr, out, lse, sm_scale, ws,
                                (size_t)TROPICAL_STATIC_WORKSPACE_BYTES, (cudaStream_t)cuda_stream, &g_launches);
}

int tropical_mixed_step(const tropical_kv_pool_t* pool, const tropical_batch_t* batch, const void* q, const void* k_new,
                        const void* v_new, void* out, float* lse, float sm_scale, void* workspace,
                        size_t workspace_bytes, void* cuda_stream) {
    g_launches = 0;
    int rc = check_pool(pool);
    if (rc != TROPICAL_OK) return rc;
    rc = check_batch(pool, batch);
    if (rc != TROPICAL_OK) return rc;
    if (batch->total_q == 0) return TROPICAL_OK;
    if (q == nullptr || out == nullptr || k_new == nullptr || v_new == nullptr) return TROPICAL_ERR_INVALID_ARG;
    if (((uintptr_t)k_new & 15) || ((uintptr_t)v_new & 15)) return TROPICAL_ERR_INVALID_ARG;  // TMA global address
    const size_t need = tropical_workspace_bytes(pool, batch->num_reqs, batch->total_q, batch->max_kv_len);
    if (workspace == nullptr || ((uintptr_t)workspace & 255) || workspace_bytes < need) return TROPICAL_ERR_WORKSPACE;
    return mixed_attention_impl(pool, batch, q, k_new, v_new, out, lse, sm_scale, workspace, workspace_bytes,
                                (cudaStream_t)cuda_stream, &g_launches);
}

size_t tropical_step_host_staging_bytes(const tropical_kv_pool_t* pool, int32_t num_reqs, int32_t total_q,
                                        int32_t page_table_stride) {
    if (pool == nullptr || num_reqs < 0 || total_q < 0 || page_table_stride < 0) return 0;
    const size_t row_q = (size_t)pool->num_q_heads * pool->head_dim * 2;
    const size_t row_kv = (size_t)pool->num_kv_heads * pool->head_dim * 2;
    size_t s = 0;
    s += align_up((size_t)total_q * row_q, 256) * 2;          // q, out
    s += align_up((size_t)total_q * row_kv, 256) * 2;         // k_new, v_new
    s += align_up((size_t)total_q * pool->num_q_heads * 4, 256);  // lse
    s += align_up((size_t)num_reqs * 4, 256) * 2;             // q_lens, ctx_lens
    s += align_up((size_t)(num_reqs + 1) * 4, 256);           // q_offsets
    s += align_up((size_t)num_reqs * page_table_stride * 4, 256);
    return s + 256;
}

int tropical_step_host(const tropical_kv_pool_t* pool, const tropical_host_batch_t* hb, const void* h_q,
                       const void* h_k_new, const void* h_v_new, void* h_out, float* h_lse, float sm_scale,
                       void* staging, size_t staging_bytes, void* workspace, size_t workspace_bytes,
                       void* cuda_stream) {
    g_launches = 0;
    int rc = check_pool(pool);
    if (rc != TROPICAL_OK) return rc;
    if (hb == nullptr) return TROPICAL_ERR_INVALID_ARG;
    rc = check_scalars(pool, hb->num_reqs, hb->total_q, hb->max_kv_len, hb->page_table_stride);
    if (rc != TROPICAL_OK) return rc;
    if (hb->total_q == 0) return TROPICAL_OK;
    if (!hb->q_lens || !hb->ctx_lens || !hb->q_offsets || !hb->page_table || !h_q || !h_k_new || !h_v_new || !h_out)
        return TROPICAL_ERR_INVALID_ARG;
    const size_t need = tropical_step_host_staging_bytes(pool, hb->num_reqs, hb->total_q, hb->page_table_stride);
    if (staging == nullptr || ((uintptr_t)staging & 255) || staging_bytes < need) return TROPICAL_ERR_WORKSPACE;
    const size_t ws_need = tropical_workspace_bytes(pool, hb->num_reqs, hb->total_q, hb->max_kv_len);
    if (workspace == nullptr || ((uintptr_t)workspace & 255) || workspace_bytes < ws_need)
        return TROPICAL_ERR_WORKSPACE;

    cudaStream_t stream = (cudaStream_t)cuda_stream;
    const int T = hb->total_q, n = hb->num_reqs;
    const size_t bq = (size_t)T * pool->num_q_heads * pool->head_dim * 2;
    const size_t bkv = (size_t)T * pool->num_kv_heads * pool->head_dim * 2;
    const size_t blse = (size_t)T * pool->num_q_heads * 4;
    char* p = (char*)staging;
    auto take = [&](size_t bytes) { char* r = p; p += align_up(bytes, 256); return r; };
    void* d_q = take(bq);
    void* d_out = take(bq);
    void* d_k = take(bkv);
    void* d_v = take(bkv);
    float* d_lse = (float*)take(blse);
    int* d_ql = (int*)take((size_t)n * 4);
    int* d_cl = (int*)take((size_t)n * 4);
    int* d_qo = (int*)take((size_t)(n + 1) * 4);
    int* d_pt = (int*)take((size_t)n * hb->page_table_stride * 4);

    cudaError_t e;
#define H2D(dst, src, bytes)                                                           \
    if ((bytes) > 0) {                                                                 \
        e = cudaMemcpyAsync(dst, src, bytes, cudaMemcpyHostToDevice, stream);          \
        if (e != cudaSuccess) return cuda_fail(e, "step_host H2D");                   \
    }
    H2D(d_ql, hb->q_lens, (size_t)n * 4);
    H2D(d_cl, hb->ctx_lens, (size_t)n * 4);
    H2D(d_qo, hb->q_offsets, (size_t)(n + 1) * 4);
    H2D(d_pt, hb->page_table, (size_t)n * hb->page_table_stride * 4);
    H2D(d_k, h_k_new, bkv);
    H2D(d_v, h_v_new, bkv);
    H2D(d_q, h_q, bq);
#undef H2D
    tropical_batch_t b;
    b.num_reqs = n;
    b.total_q = T;
    b.max_kv_len = hb->max_kv_len;
    b.page_table_stride = hb->page_table_stride;
    b.q_lens = d_ql;
    b.ctx_lens = d_cl;
    b.q_offsets = d_qo;
    b.page_table = d_pt;
    int launches = 0;
    rc = mixed_attention_impl(pool, &b, d_q, d_k, d_v, d_out, h_lse ? d_lse : nullptr, sm_scale, workspace,
                              workspace_bytes, stream, &launches);  // the fused step: append inside
    if (rc != TROPICAL_OK) return rc;
    e = cudaMemcpyAsync(h_out, d_out, bq, cudaMemcpyDeviceToHost, stream);
    if (e != cudaSuccess) return cuda_fail(e, "step_host D2H");
    if (h_lse) {
        e = cudaMemcpyAsync(h_lse, d_lse, blse, cudaMemcpyDeviceToHost, stream);
        if (e != cudaSuccess) return cuda_fail(e, "step_host D2H lse");
    }
    e = cudaStreamSynchronize(stream);
    if (e != cudaSuccess) return cuda_fail(e, "step_host sync");
    g_launches = launches;
    return TROPICAL_OK;
}

int tropical_last_launch_count(void) { return g_launches; }

const char* tropical_status_string(int s) {
    switch (s) {
        case TROPICAL_OK: return "ok";
        case TROPICAL_ERR_INVALID_ARG: return "invalid argument";
        case TROPICAL_ERR_UNSUPPORTED: return "unsupported shape";
        case TROPICAL_ERR_WORKSPACE: return "workspace missing, misaligned or too small";
        case TROPICAL_ERR_CUDA: return "CUDA failure";
        case TROPICAL_ERR_UNCALIBRATED: return "no cost-model coefficients for this shape";
        case TROPICAL_ERR_STATIC_CAPACITY:
            return "step needs more scratch than the built-in static workspace holds (TROPICAL_STATIC_WORKSPACE_BYTES)";
        default: return "unknown status";
    }
}

int tropical_debug_read_profile(const void* workspace, uint64_t* out_ns, void* cuda_stream) {
    if (workspace == nullptr || out_ns == nullptr) return TROPICAL_ERR_INVALID_ARG;
    cudaStream_t stream = (cudaStream_t)cuda_stream;
    cudaError_t e = cudaMemcpyAsync(out_ns, (const char*)workspace + profile_offset_bytes(), 4 * sizeof(uint64_t),
                                    cudaMemcpyDeviceToHost, stream);
    if (e == cudaSuccess) e = cudaStreamSynchronize(stream);
    if (e != cudaSuccess) return cuda_fail(e, "read_profile");
    return TROPICAL_OK;
}

void tropical_debug_set_grid(int num_ctas) { set_debug_grid(num_ctas); }

void tropical_debug_set_split_pages(int pages) { set_debug_split_pages(pages); }
void tropical_debug_set_fused(int mode) { set_debug_fused(mode); }

int tropical_debug_wait_profile(uint64_t* cycles, uint64_t* calls, int32_t n, int32_t reset) {
    if (cycles == nullptr || calls == nullptr || n <= 0) return TROPICAL_ERR_INVALID_ARG;
    const int got = read_wait_profile((unsigned long long*)cycles, (unsigned long long*)calls, n, reset);
    if (got < 0) return cuda_fail(cudaGetLastError(), "wait_profile");
    return got == 0 ? TROPICAL_ERR_UNSUPPORTED : TROPICAL_OK;
}

int tropical_debug_timeline(uint64_t* out_ns, int32_t reset) {
    unsigned long long a[16] = {0}, m[16] = {0};
    const int ra = read_timeline_append(out_ns ? a : nullptr, reset), rm = read_timeline_mixed(out_ns ? m : nullptr, reset);
    if (ra < 0 || rm < 0) return cuda_fail(cudaGetLastError(), "timeline");
    if (ra == 0 || rm == 0) return TROPICAL_ERR_UNSUPPORTED;
    if (out_ns != nullptr)
        for (int i = 0; i < 9; ++i) out_ns[i] = i < 2 ? a[i] : m[i];
    return TROPICAL_OK;
}

const char* tropical_last_cuda_error(void) { return g_cuda_err; }

const char* tropical_version(void) {
#ifdef TROPICAL_WHATIF_BUILD
    return "tropical-b200 0.2 (sm_100a) WHATIF measurement build: attention results are wrong by design";
#else
    return "tropical-b200 0.2 (sm_100a)";
#endif
}

}  // extern "C"

// Test hook: the CUDA-core kernel on its own (cross-check for the tile kernels).
extern "C" int tropical_debug_attention_simt(const tropical_kv_pool_t* pool, const tropical_batch_t* batch,
                                             const void* q, void* out, float* lse, float sm_scale,
                                             void* cuda_stream) {
    int rc = check_pool(pool);
    if (rc != TROPICAL_OK) return rc;
    rc = check_batch(pool, batch);
    if (rc != TROPICAL_OK) return rc;
    if (batch->total_q == 0) return TROPICAL_OK;
    if (q == nullptr || out == nullptr) return TROPICAL_ERR_INVALID_ARG;
    const float scale = sm_scale > 0.f ? sm_scale : 1.0f / sqrtf((float)pool->head_dim);
    cudaError_t e = launch_attention_simt(to_pool(pool), to_batch(batch), q, out, lse,
                                          scale * 1.4426950408889634f, (cudaStream_t)cuda_stream);
    if (e != cudaSuccess) return cuda_fail(e, "attention_simt");
    return TROPICAL_OK;
}
