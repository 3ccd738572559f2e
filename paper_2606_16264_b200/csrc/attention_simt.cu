// attention_simt.cu -- the plain CUDA-core attention kernel: one warp per (new token, q head) row,
// online softmax over 32-key chunks, keys spread over lanes for QK^T and head-dim spread over
// lanes for PV.  It is the first correct CUDA path and stays as the in-library cross-check for
// the tensor-core tile kernels: tests call it through tropical_debug_attention_simt
// (include/tropical_debug.h).  No product entry point ever routes here.
//
// Definition followed: SURVEY.md 8(c) phase 2 -- row (i, t, hq): keys j <= c_i + t of kv head
// hq / (Hq/Hkv), s_j = scale * q.k_j, out = softmax(s) V, lse = m + ln Z.
#include "common.cuh"
#include "kernels.h"

namespace tropical {

constexpr int kSimtWarps = 4;

template <int D>
__global__ void __launch_bounds__(kSimtWarps * 32) attention_simt_kernel(PoolDesc pool, BatchDesc b,
                                                                         const uint16_t* __restrict__ q,
                                                                         uint16_t* __restrict__ out,
                                                                         float* __restrict__ lse, float scale_log2) {
    constexpr int EPL = D / 32;  // output elements per lane (4 at d=128, 2 at d=64)
    __shared__ float q_s[kSimtWarps][D];
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const long long n_rows = (long long)b.total_q * pool.Hq;
    const int g = pool.Hq / pool.Hkv;

    for (long long row = (long long)blockIdx.x * kSimtWarps + warp; row < n_rows;
         row += (long long)gridDim.x * kSimtWarps) {
        const int tok = (int)(row / pool.Hq), hq = (int)(row % pool.Hq), hk = hq / g;
        const int req = find_request(b.q_offsets, b.num_reqs, tok);
        const int t = tok - __ldg(b.q_offsets + req);
        const int n = __ldg(b.ctx_lens + req) + t + 1;  // visible keys
        const int* pt = b.page_table + (size_t)req * b.stride;

        __syncwarp();
        for (int c = lane; c < D; c += 32) q_s[warp][c] = bf16_lo(q[row * D + c]);
        __syncwarp();

        float m = -INFINITY, l = 0.f, o[EPL];
#pragma unroll
        for (int e = 0; e < EPL; ++e) o[e] = 0.f;

        for (int j0 = 0; j0 < n; j0 += 32) {
            const int j = j0 + lane;
            int page = 0;
            float s = -INFINITY;
            if (j < n) {
                page = __ldg(pt + j / kPageSize);
                const uint4* krow = reinterpret_cast<const uint4*>(
                    pool.k_pool + (((size_t)page * pool.Hkv + hk) * kPageSize + j % kPageSize) * D);
                float acc = 0.f;
#pragma unroll
                for (int c = 0; c < D / 8; ++c) {
                    const uint4 kv = __ldg(krow + c);
                    const float* qq = &q_s[warp][c * 8];
                    acc = fmaf(qq[0], bf16_lo(kv.x), acc);
                    acc = fmaf(qq[1], bf16_hi(kv.x), acc);
                    acc = fmaf(qq[2], bf16_lo(kv.y), acc);
                    acc = fmaf(qq[3], bf16_hi(kv.y), acc);
                    acc = fmaf(qq[4], bf16_lo(kv.z), acc);
                    acc = fmaf(qq[5], bf16_hi(kv.z), acc);
                    acc = fmaf(qq[6], bf16_lo(kv.w), acc);
                    acc = fmaf(qq[7], bf16_hi(kv.w), acc);
                }
                s = acc * scale_log2;
            }
            float mx = s;
#pragma unroll
            for (int off = 16; off; off >>= 1) mx = fmaxf(mx, __shfl_xor_sync(0xffffffffu, mx, off));
            const float m_new = fmaxf(m, mx);  // finite: key j0 is always visible
            const float alpha = exp2f(m - m_new);
            const float p = (j < n) ? exp2f(s - m_new) : 0.f;
            float ps = p;
#pragma unroll
            for (int off = 16; off; off >>= 1) ps += __shfl_xor_sync(0xffffffffu, ps, off);
            l = l * alpha + ps;
            m = m_new;
#pragma unroll
            for (int e = 0; e < EPL; ++e) o[e] *= alpha;
            const int cnt = min(32, n - j0);
            for (int jj = 0; jj < cnt; ++jj) {
                const float pj = __shfl_sync(0xffffffffu, p, jj);
                const int pg = __shfl_sync(0xffffffffu, page, jj);
                const uint16_t* vrow =
                    pool.v_pool + (((size_t)pg * pool.Hkv + hk) * kPageSize + (j0 + jj) % kPageSize) * D + lane * EPL;
                if (EPL == 4) {
                    const uint2 vv = __ldg(reinterpret_cast<const uint2*>(vrow));
                    o[0] = fmaf(pj, bf16_lo(vv.x), o[0]);
                    o[1] = fmaf(pj, bf16_hi(vv.x), o[1]);
                    o[2] = fmaf(pj, bf16_lo(vv.y), o[2]);
                    o[3] = fmaf(pj, bf16_hi(vv.y), o[3]);
                } else {
                    const uint32_t vv = __ldg(reinterpret_cast<const uint32_t*>(vrow));
                    o[0] = fmaf(pj, bf16_lo(vv), o[0]);
                    o[1] = fmaf(pj, bf16_hi(vv), o[1]);
                }
            }
        }
        const float inv = 1.f / l;
        uint16_t* orow = out + row * D + lane * EPL;
        if (EPL == 4) {
            uint2 w;
            w.x = pack_bf16x2(o[0] * inv, o[1] * inv);
            w.y = pack_bf16x2(o[2] * inv, o[3] * inv);
            *reinterpret_cast<uint2*>(orow) = w;
        } else {
            *reinterpret_cast<uint32_t*>(orow) = pack_bf16x2(o[0] * inv, o[1] * inv);
        }
        if (lse != nullptr && lane == 0) lse[row] = (m + log2f(l)) * 0.6931471805599453f;
    }
}

cudaError_t launch_attention_simt(const PoolDesc& pool, const BatchDesc& b, const void* q, void* out, float* lse,
                                  float scale_log2, cudaStream_t stream) {
    const long long n_rows = (long long)b.total_q * pool.Hq;
    if (n_rows == 0) return cudaSuccess;
    long long grid = (n_rows + kSimtWarps - 1) / kSimtWarps;
    if (grid > 148LL * 64) grid = 148LL * 64;
    if (pool.D == 128)
        attention_simt_kernel<128><<<(int)grid, kSimtWarps * 32, 0, stream>>>(pool, b, (const uint16_t*)q,
                                                                              (uint16_t*)out, lse, scale_log2);
    else
        attention_simt_kernel<64><<<(int)grid, kSimtWarps * 32, 0, stream>>>(pool, b, (const uint16_t*)q,
                                                                             (uint16_t*)out, lse, scale_log2);
    return cudaGetLastError();
}

}  // namespace tropical
