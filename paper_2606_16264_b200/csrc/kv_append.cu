// kv_append.cu -- SURVEY.md 8(a) rows A1 (KV append) and A2 (page gather), bit-exact copies.
//
// A1: for t < q_i, pos = c_i + t: pool[page_table[i][pos/P]][h][pos%P][:] = new[q_off_i+t][h][:].
// HBM-bound and tiny: T*Hkv rows of 2*d bytes each for K and V.  One thread moves the 16-byte chunk
// `chunk` of every kv head of one (token, K|V); the d/8 threads of a row read and write 2*d contiguous
// bytes (fully coalesced on both sides -- a (page, head, slot) row of the HND pool is contiguous).
#include <atomic>

#include "common.cuh"
#include "kernels.h"

namespace tropical {

constexpr int kAppendStagedReqs = 2048;  // q_offsets kept in shared memory for the token -> request search

template <int D>
__global__ void __launch_bounds__(256) kv_append_kernel(PoolDesc pool, BatchDesc b,
                                                        const uint4* __restrict__ k_new,
                                                        const uint4* __restrict__ v_new, int hg) {
    constexpr int CH = D / 8;  // 16-byte chunks per row
    // Programmatic dependent launch: a following kernel that opted in (the tile-directory kernel of
    // tropical_mixed_attention, which reads only q_lens / ctx_lens) may start while this one is still copying; every
    // other kernel keeps normal stream order.  The launcher keeps the grid small enough for all of its blocks to be
    // resident at once (so that all of them trigger at once) with room left on every SM for the directory's blocks.
    asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
    if (threadIdx.x == 0) tl_mark(0, true);
    // token -> request: binary search over q_offsets, from shared memory when the batch fits (one coalesced load
    // instead of log2(n) dependent global loads per thread)
    __shared__ int s_off[kAppendStagedReqs + 1];
    const bool staged = b.num_reqs <= kAppendStagedReqs;
    if (staged) {
        for (int i = threadIdx.x; i <= b.num_reqs; i += blockDim.x) s_off[i] = __ldg(b.q_offsets + i);
        __syncthreads();
    }
    // One thread per (token, group of hg kv heads, K|V, 16-byte chunk): the request lookup and the (page, slot) of the
    // token are done once per thread and reused for its heads, whose rows are copied with several independent loads
    // in flight.  hg is chosen by the launcher: all heads for big steps, fewer when a step has few tokens.
    const int ngroups = (pool.Hkv + hg - 1) / hg;
    const long long total = (long long)b.total_q * ngroups * CH * 2;
    for (long long idx = blockIdx.x * (long long)blockDim.x + threadIdx.x; idx < total;
         idx += (long long)gridDim.x * blockDim.x) {
        const int chunk = (int)(idx % CH);
        long long r = idx / CH;
        const int which = (int)(r & 1);  // 0 = K, 1 = V
        r >>= 1;
        const int h_lo = (int)(r % ngroups) * hg, h_hi = min(pool.Hkv, h_lo + hg);
        const int tok = (int)(r / ngroups);
        int req, t;
        if (staged) {
            int lo = 0, hi = b.num_reqs;  // invariant: s_off[lo] <= tok < s_off[hi]
            while (hi - lo > 1) {
                const int mid = (lo + hi) >> 1;
                if (s_off[mid] <= tok) lo = mid; else hi = mid;
            }
            req = lo;
            t = tok - s_off[lo];
        } else {
            req = find_request(b.q_offsets, b.num_reqs, tok);
            t = tok - __ldg(b.q_offsets + req);
        }
        const int pos = __ldg(b.ctx_lens + req) + t;
        const int page = __ldg(b.page_table + (size_t)req * b.stride + pos / kPageSize);
        const int slot = pos % kPageSize;
        const uint4* src = (which == 0 ? k_new : v_new) + (size_t)tok * pool.Hkv * CH + chunk;
        uint4* dst = reinterpret_cast<uint4*>(const_cast<uint16_t*>(which == 0 ? pool.k_pool : pool.v_pool)) +
                     ((size_t)page * pool.Hkv * kPageSize + slot) * CH + chunk;
        int h = h_lo;
        for (; h + 4 <= h_hi; h += 4) {
            uint4 v[4];
#pragma unroll
            for (int k = 0; k < 4; ++k) v[k] = __ldg(src + (size_t)(h + k) * CH);
#pragma unroll
            for (int k = 0; k < 4; ++k) dst[(size_t)(h + k) * kPageSize * CH] = v[k];
        }
        for (; h < h_hi; ++h) dst[(size_t)h * kPageSize * CH] = __ldg(src + (size_t)h * CH);
    }
    if (threadIdx.x == 0) tl_mark(1, false);
}

// SURVEY 8(f) NEXT-4 "fuse RoPE+append": the same scatter with rotate-half rotary embedding applied to the K rows on the
// way (include/tropical.h tropical_kv_append_rope): channel c < d/2 pairs with c + d/2, the token at position pos uses
// row pos of the caller's fp32 tables cos, sin [table_len][d/2].  One thread per (token, kv head, 16-byte chunk c of the
// lower half): it reads chunks c and c + d/16 of the K row (the two halves of 8 pairs), 8 cos and 8 sin values, writes
// both rotated chunks, and copies the two V chunks.  fp32 arithmetic (fmaf), bf16 round-to-nearest-even.
__device__ __forceinline__ void rope8(const uint4& lo, const uint4& hi, const float4& c0, const float4& c1, const float4& s0,
                                      const float4& s1, uint4& out_lo, uint4& out_hi) {
    const uint32_t xl[4] = {lo.x, lo.y, lo.z, lo.w}, xh[4] = {hi.x, hi.y, hi.z, hi.w};
    const float cs[8] = {c0.x, c0.y, c0.z, c0.w, c1.x, c1.y, c1.z, c1.w};
    const float sn[8] = {s0.x, s0.y, s0.z, s0.w, s1.x, s1.y, s1.z, s1.w};
    uint32_t ol[4], oh[4];
#pragma unroll
    for (int j = 0; j < 4; ++j) {
        const float x0 = bf16_lo(xl[j]), x1 = bf16_hi(xl[j]), y0 = bf16_lo(xh[j]), y1 = bf16_hi(xh[j]);
        ol[j] = pack_bf16x2(fmaf(x0, cs[2 * j], -(y0 * sn[2 * j])), fmaf(x1, cs[2 * j + 1], -(y1 * sn[2 * j + 1])));
        oh[j] = pack_bf16x2(fmaf(y0, cs[2 * j], x0 * sn[2 * j]), fmaf(y1, cs[2 * j + 1], x1 * sn[2 * j + 1]));
    }
    out_lo = make_uint4(ol[0], ol[1], ol[2], ol[3]);
    out_hi = make_uint4(oh[0], oh[1], oh[2], oh[3]);
}

template <int D>
__global__ void __launch_bounds__(256) kv_append_rope_kernel(PoolDesc pool, BatchDesc b, const uint4* __restrict__ k_new,
                                                             const uint4* __restrict__ v_new,
                                                             const float4* __restrict__ cos_t,
                                                             const float4* __restrict__ sin_t) {
    constexpr int CH = D / 8;    // 16-byte chunks per row
    constexpr int HC = CH / 2;   // chunks of the lower half = threads per row
    asm volatile("griddepcontrol.launch_dependents;" ::: "memory");  // as kv_append_kernel: the tile directory may overlap
    const long long total = (long long)b.total_q * pool.Hkv * HC;
    for (long long idx = blockIdx.x * (long long)blockDim.x + threadIdx.x; idx < total;
         idx += (long long)gridDim.x * blockDim.x) {
        const int chunk = (int)(idx % HC);
        long long r = idx / HC;
        const int h = (int)(r % pool.Hkv);
        const int tok = (int)(r / pool.Hkv);
        const int req = find_request(b.q_offsets, b.num_reqs, tok);
        const int pos = __ldg(b.ctx_lens + req) + tok - __ldg(b.q_offsets + req);
        const int page = __ldg(b.page_table + (size_t)req * b.stride + pos / kPageSize);
        const size_t src = ((size_t)tok * pool.Hkv + h) * CH + chunk;
        const size_t dst = (((size_t)page * pool.Hkv + h) * kPageSize + pos % kPageSize) * CH + chunk;
        const size_t tab = (size_t)pos * (D / 8) + chunk * 2;  // float4 index: row pos of [table_len][D/2] floats
        const uint4 klo = __ldg(k_new + src), khi = __ldg(k_new + src + HC);
        const uint4 vlo = __ldg(v_new + src), vhi = __ldg(v_new + src + HC);
        const float4 c0 = __ldg(cos_t + tab), c1 = __ldg(cos_t + tab + 1), s0 = __ldg(sin_t + tab), s1 = __ldg(sin_t + tab + 1);
        uint4 olo, ohi;
        rope8(klo, khi, c0, c1, s0, s1, olo, ohi);
        uint4* kp = reinterpret_cast<uint4*>(const_cast<uint16_t*>(pool.k_pool));
        uint4* vp = reinterpret_cast<uint4*>(const_cast<uint16_t*>(pool.v_pool));
        kp[dst] = olo;
        kp[dst + HC] = ohi;
        vp[dst] = vlo;
        vp[dst + HC] = vhi;
    }
}

template <int D>
__global__ void __launch_bounds__(256) kv_gather_kernel(PoolDesc pool, BatchDesc b, int req, int n_keys,
                                                        uint4* __restrict__ k_dense, uint4* __restrict__ v_dense) {
    constexpr int CH = D / 8;
    const long long total = (long long)n_keys * pool.Hkv * CH * 2;
    for (long long idx = blockIdx.x * (long long)blockDim.x + threadIdx.x; idx < total;
         idx += (long long)gridDim.x * blockDim.x) {
        const int chunk = (int)(idx % CH);
        long long r = idx / CH;
        const int which = (int)(r & 1);
        r >>= 1;
        const int h = (int)(r % pool.Hkv);
        const int j = (int)(r / pool.Hkv);
        const int page = __ldg(b.page_table + (size_t)req * b.stride + j / kPageSize);
        const size_t src = (((size_t)page * pool.Hkv + h) * kPageSize + j % kPageSize) * CH + chunk;
        const size_t dst = ((size_t)j * pool.Hkv + h) * CH + chunk;
        if (which == 0)
            k_dense[dst] = __ldg(reinterpret_cast<const uint4*>(pool.k_pool) + src);
        else
            v_dense[dst] = __ldg(reinterpret_cast<const uint4*>(pool.v_pool) + src);
    }
}

// debug check of a batch's device arrays (tropical_validate_batch): lowest offending request index via atomicMin
__global__ void __launch_bounds__(256) validate_batch_kernel(BatchDesc b, int num_pages, int* first_bad) {
    for (int i = blockIdx.x * blockDim.x + threadIdx.x; i <= b.num_reqs; i += gridDim.x * blockDim.x) {
        bool bad = false;
        if (i == b.num_reqs) {
            bad = b.q_offsets[i] != b.total_q;
        } else {
            const int q = b.q_lens[i], c = b.ctx_lens[i];
            const long long L = (long long)q + c;
            bad = q < 0 || c < 0 || b.q_offsets[i + 1] - b.q_offsets[i] != q || (i == 0 && b.q_offsets[0] != 0) ||
                  L > b.max_kv_len || (L + kPageSize - 1) / kPageSize > b.stride;
            if (!bad && q > 0) {
                const int np = (int)((L + kPageSize - 1) / kPageSize);
                for (int p = 0; p < np; ++p) {
                    const int page = b.page_table[(size_t)i * b.stride + p];
                    if (page < 0 || page >= num_pages) bad = true;
                }
            }
        }
        if (bad) atomicMin(first_bad, i);
    }
}

cudaError_t launch_validate_batch(const PoolDesc& pool, const BatchDesc& b, int* first_bad_dev, cudaStream_t stream) {
    const int grid = (b.num_reqs + 1 + 255) / 256;
    validate_batch_kernel<<<grid < 1 ? 1 : grid, 256, 0, stream>>>(b, pool.num_pages, first_bad_dev);
    return cudaGetLastError();
}

static int grid_for(long long total_threads, int block, long long cap = 148LL * 8) {
    long long g = (total_threads + block - 1) / block;  // grid-stride beyond `cap` CTAs
    if (g > cap) g = cap;
    if (g < 1) g = 1;
    return (int)g;
}

cudaError_t launch_kv_append(const PoolDesc& pool, const BatchDesc& b, const void* k_new, const void* v_new,
                             cudaStream_t stream) {
    if (b.total_q == 0) return cudaSuccess;
    // heads per thread: as many as keep >= 64K threads in flight (all of them for steps with many new tokens)
    const long long chunks = (long long)b.total_q * pool.Hkv * (pool.D / 8) * 2;
    long long hg = chunks / 65536;
    if (hg < 1) hg = 1;
    if (hg > pool.Hkv) hg = pool.Hkv;
    const long long total = (long long)b.total_q * ((pool.Hkv + hg - 1) / hg) * (pool.D / 8) * 2;
    // at most 6 blocks per SM: all resident in one wave (they trigger their programmatic dependents together) and a
    // quarter of every SM's threads and registers stays free for the tile-directory kernel that overlaps this one.
    // Blocks of two kernels share an SM only when both run with the same shared-memory carve-out: every kernel of
    // the step asks for the maximum one, which the step kernel needs anyway.
    const int grid = grid_for(total, 256, 148LL * 6);
    {
        static std::atomic<int> carve[64];
        int dev = 0;
        cudaGetDevice(&dev);
        if (dev < 0 || dev >= 64) dev = 0;
        if (!carve[dev].load(std::memory_order_acquire)) {
            cudaFuncSetAttribute(kv_append_kernel<128>, cudaFuncAttributePreferredSharedMemoryCarveout, cudaSharedmemCarveoutMaxShared);
            cudaFuncSetAttribute(kv_append_kernel<64>, cudaFuncAttributePreferredSharedMemoryCarveout, cudaSharedmemCarveoutMaxShared);
            carve[dev].store(1, std::memory_order_release);
        }
    }
    if (pool.D == 128)
        kv_append_kernel<128><<<grid, 256, 0, stream>>>(pool, b, (const uint4*)k_new, (const uint4*)v_new, (int)hg);
    else
        kv_append_kernel<64><<<grid, 256, 0, stream>>>(pool, b, (const uint4*)k_new, (const uint4*)v_new, (int)hg);
    return cudaGetLastError();
}

cudaError_t launch_kv_append_rope(const PoolDesc& pool, const BatchDesc& b, const void* k_new, const void* v_new,
                                  const float* cos_t, const float* sin_t, cudaStream_t stream) {
    if (b.total_q == 0) return cudaSuccess;
    const long long total = (long long)b.total_q * pool.Hkv * (pool.D / 16);
    const int grid = grid_for(total, 256, 148LL * 6);
    if (pool.D == 128)
        kv_append_rope_kernel<128><<<grid, 256, 0, stream>>>(pool, b, (const uint4*)k_new, (const uint4*)v_new,
                                                             (const float4*)cos_t, (const float4*)sin_t);
    else
        kv_append_rope_kernel<64><<<grid, 256, 0, stream>>>(pool, b, (const uint4*)k_new, (const uint4*)v_new,
                                                            (const float4*)cos_t, (const float4*)sin_t);
    return cudaGetLastError();
}

cudaError_t launch_kv_gather(const PoolDesc& pool, const BatchDesc& b, int req, int n_keys, void* k_dense,
                             void* v_dense, cudaStream_t stream) {
    if (n_keys == 0) return cudaSuccess;
    const long long total = (long long)n_keys * pool.Hkv * (pool.D / 8) * 2;
    const int grid = grid_for(total, 256);
    if (pool.D == 128)
        kv_gather_kernel<128><<<grid, 256, 0, stream>>>(pool, b, req, n_keys, (uint4*)k_dense, (uint4*)v_dense);
    else
        kv_gather_kernel<64><<<grid, 256, 0, stream>>>(pool, b, req, n_keys, (uint4*)k_dense, (uint4*)v_dense);
    return cudaGetLastError();
}

// measurement builds (-DTROPICAL_TIMELINE): this translation unit's copy of the timestamps (slots 0, 1)
int read_timeline_append(unsigned long long* out16, int reset) {
#ifdef TROPICAL_TIMELINE
    return timeline_read(out16, reset);
#else
    (void)out16; (void)reset;
    return 0;
#endif
}

}  // namespace tropical
