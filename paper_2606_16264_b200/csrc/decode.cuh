// decode.cuh -- SURVEY.md 8(a) row A4: decode tiles (split-K flash decoding over pages).
//
// One WARP is one decode worker.  It pops a unit (request, kv head, head block, page range),
// streams the unit's K and V page-heads HBM -> shared memory with TMA (two 64-column
// SWIZZLE_128B boxes per 16 x d page-head, i.e. whole 4 KiB contiguous blocks of the HND pool,
// landed bank-conflict-free for ldmatrix) through a private NSTAGE-deep mbarrier ring, and
// consumes them with warp-level tensor-core MMAs whose M rows are the (up to 8) q heads of the
// kv group: S = Q K^T (m16n8k16, fp32), online softmax in registers (quad shuffles), O += P V.
// HBM-bound: each K/V byte is read once; arithmetic per byte is the same for MHA and GQA.
// Results: final bf16 row when the request has one split, else fp32 partial (m, l, o) for A5.
#pragma once
#include "common.cuh"
#include "plan.cuh"

namespace tropical {

template <int D>
struct DecodeCfg {
    static constexpr int CB = D / 64;                 // 64-column swizzle blocks per row
    static constexpr int HALF_BYTES = 16 * 128;       // one TMA box: 16 rows x 128 B
    static constexpr int PAGE_BYTES = CB * HALF_BYTES;  // K (or V) of one page-head
    static constexpr int STAGE_BYTES = 2 * PAGE_BYTES;  // K + V
};

struct DecodeArgs {
    PoolDesc pool;
    BatchDesc b;
    const uint16_t* q;
    uint16_t* out;
    float* lse;
    float scale_log2;
    const int* hdr;
    int* ticket;
    const int4* req_info;
    const int4* units;
    float2* part_ml;
    float* part_o;
};

// ring: this warp's NSTAGE * STAGE_BYTES bytes (1024-aligned); full: NSTAGE mbarriers (count 1);
// it: running stage counter of this warp (persists across units so barrier parities stay consistent).
template <int D, int NSTAGE>
__device__ __forceinline__ void decode_warp_worker(const DecodeArgs& A, const CUtensorMap* tm_k, const CUtensorMap* tm_v,
                                                   uint8_t* ring, uint64_t* full, uint32_t& it) {
    using C = DecodeCfg<D>;
    const int lane = threadIdx.x & 31;
    const int row = lane >> 2, cq = (lane & 3) * 2;
    const int g = A.pool.Hq / A.pool.Hkv;
    const int n_units = A.hdr[HDR_N_UNITS];
    const uint32_t ring_s = smem_u32(ring);
    // ldmatrix lane addressing (row within 8x8 matrix r8, matrix id mi)
    const int mi = lane >> 3, r8 = lane & 7;
    const int k_key = (mi >> 1) * 8 + r8, k_chunk_off = mi & 1;   // K: matrices (keys lo/hi) x (chunk, chunk+1)
    const int v_key = (mi & 1) * 8 + r8, v_chunk_off = mi >> 1;   // V (trans): (keys lo/hi) x (chunk, chunk+1)

    for (;;) {
        int u = 0;
        if (lane == 0) u = atomicAdd(A.ticket, 1);
        u = __shfl_sync(0xffffffffu, u, 0);
        if (u >= n_units) break;
        const int4 un = A.units[u];
        const int req = un.x, kvh = un.y & 0xffff, hb = un.y >> 16, p0 = un.z, np = un.w;
        const int L = __ldg(A.b.ctx_lens + req) + 1;
        const int tok = __ldg(A.b.q_offsets + req);
        const int h0 = kvh * g + hb * kHeadBlock;
        const int nh = min(kHeadBlock, g - hb * kHeadBlock);
        const int* pt = A.b.page_table + (size_t)req * A.b.stride + p0;

        // Q fragments (A operand rows = heads of the group; rows >= nh and rows 8..15 are zero)
        uint32_t qa[D / 16][2];
        {
            const uint16_t* qrow = A.q + ((size_t)tok * A.pool.Hq + h0 + row) * D;
#pragma unroll
            for (int ks = 0; ks < D / 16; ++ks) {
                qa[ks][0] = row < nh ? *reinterpret_cast<const uint32_t*>(qrow + ks * 16 + cq) : 0u;
                qa[ks][1] = row < nh ? *reinterpret_cast<const uint32_t*>(qrow + ks * 16 + 8 + cq) : 0u;
            }
        }
        float o[D / 8][4];
#pragma unroll
        for (int nt = 0; nt < D / 8; ++nt) o[nt][0] = o[nt][1] = o[nt][2] = o[nt][3] = 0.f;
        float m = -INFINITY, l = 0.f;

        int ptv = 0;
        uint32_t it_issue = it;
        auto issue = [&](int pi) {  // whole warp calls; lane 0 issues the TMA boxes of page pi of this unit
            if ((pi & 31) == 0) ptv = (pi + lane < np) ? __ldg(pt + pi + lane) : 0;
            const int page = __shfl_sync(0xffffffffu, ptv, pi & 31);
            if (lane == 0) {
                const int st = it_issue % NSTAGE;
                uint8_t* dst = ring + st * C::STAGE_BYTES;
                const int r0 = (page * A.pool.Hkv + kvh) * kPageSize;
                mbar_arrive_expect_tx(full + st, C::STAGE_BYTES);
#pragma unroll
                for (int cb = 0; cb < C::CB; ++cb) {
                    tma_load_2d(dst + cb * C::HALF_BYTES, tm_k, cb * 64, r0, full + st);
                    tma_load_2d(dst + C::PAGE_BYTES + cb * C::HALF_BYTES, tm_v, cb * 64, r0, full + st);
                }
            }
            ++it_issue;
        };
        const int pre = min(NSTAGE - 1, np);
        for (int i = 0; i < pre; ++i) issue(i);

        for (int p = 0; p < np; ++p) {
            if (p + NSTAGE - 1 < np) issue(p + NSTAGE - 1);
            const int st = it % NSTAGE;
            mbar_wait(full + st, (it / NSTAGE) & 1);
            ++it;
            const uint32_t kbase = ring_s + st * C::STAGE_BYTES;
            const uint32_t vbase = kbase + C::PAGE_BYTES;

            // S = Q K^T for the 16 keys of this page (two n-tiles of 8 keys)
            float s0[4] = {0.f, 0.f, 0.f, 0.f}, s1[4] = {0.f, 0.f, 0.f, 0.f};
#pragma unroll
            for (int ks = 0; ks < D / 16; ++ks) {
                const int chunk = (ks & 3) * 2 + k_chunk_off;
                const uint32_t addr = kbase + (ks >> 2) * C::HALF_BYTES + k_key * 128 + ((chunk ^ (k_key & 7)) << 4);
                uint32_t b00, b01, b10, b11;
                ldmatrix_x4(addr, b00, b01, b10, b11);
                mma_bf16_16816(s0, qa[ks][0], 0u, qa[ks][1], 0u, b00, b01);
                mma_bf16_16816(s1, qa[ks][0], 0u, qa[ks][1], 0u, b10, b11);
            }
            const int nvalid = L - (p0 + p) * kPageSize;  // >= 1 by construction of the unit
            float v00 = (cq < nvalid) ? s0[0] * A.scale_log2 : -INFINITY;
            float v01 = (cq + 1 < nvalid) ? s0[1] * A.scale_log2 : -INFINITY;
            float v10 = (cq + 8 < nvalid) ? s1[0] * A.scale_log2 : -INFINITY;
            float v11 = (cq + 9 < nvalid) ? s1[1] * A.scale_log2 : -INFINITY;
            float mx = fmaxf(fmaxf(v00, v01), fmaxf(v10, v11));
            mx = fmaxf(mx, __shfl_xor_sync(0xffffffffu, mx, 1));
            mx = fmaxf(mx, __shfl_xor_sync(0xffffffffu, mx, 2));
            const float m_new = fmaxf(m, mx);  // finite: key 0 of the page is valid
            const float alpha = fast_exp2(m - m_new);
            v00 = fast_exp2(v00 - m_new);
            v01 = fast_exp2(v01 - m_new);
            v10 = fast_exp2(v10 - m_new);
            v11 = fast_exp2(v11 - m_new);
            l = l * alpha + ((v00 + v01) + (v10 + v11));
            if (__any_sync(0xffffffffu, m_new > m)) {
#pragma unroll
                for (int nt = 0; nt < D / 8; ++nt) { o[nt][0] *= alpha; o[nt][1] *= alpha; }
            }
            m = m_new;
            const uint32_t pa0 = pack_bf16x2(v00, v01), pa2 = pack_bf16x2(v10, v11);

            if (nvalid < kPageSize) {  // ragged last page: unused slots may hold NaN bits; 0 * NaN = NaN in the MMA
                const int nz = (kPageSize - nvalid) * 8 * C::CB;
                for (int idx = lane; idx < nz; idx += 32) {
                    const int r = nvalid + idx / (8 * C::CB), rem = idx % (8 * C::CB);
                    const uint32_t a = vbase + (rem >> 3) * C::HALF_BYTES + r * 128 + ((rem & 7) << 4);
                    asm volatile("st.shared.v4.b32 [%0], {%1,%1,%1,%1};" ::"r"(a), "r"(0u) : "memory");
                }
                __syncwarp();
            }
            // O += P V
#pragma unroll
            for (int n2 = 0; n2 < D / 16; ++n2) {
                const int chunk = ((n2 * 2) & 7) + v_chunk_off;
                const uint32_t addr = vbase + ((n2 * 2) >> 3) * C::HALF_BYTES + v_key * 128 + ((chunk ^ (v_key & 7)) << 4);
                uint32_t b0, b1, b2, b3;
                ldmatrix_x4_trans(addr, b0, b1, b2, b3);
                mma_bf16_16816(o[2 * n2], pa0, 0u, pa2, 0u, b0, b1);
                mma_bf16_16816(o[2 * n2 + 1], pa0, 0u, pa2, 0u, b2, b3);
            }
            if (nvalid < kPageSize) fence_proxy_async();  // generic zero-fill before the next TMA refill
            __syncwarp();  // every lane is done with this stage before lane 0 refills it
        }

        l += __shfl_xor_sync(0xffffffffu, l, 1);
        l += __shfl_xor_sync(0xffffffffu, l, 2);
        const int nsplit = A.req_info[req].z;
        if (row < nh) {
            if (nsplit == 1) {
                const float inv = 1.f / l;
                uint16_t* orow = A.out + ((size_t)tok * A.pool.Hq + h0 + row) * D + cq;
#pragma unroll
                for (int nt = 0; nt < D / 8; ++nt)
                    *reinterpret_cast<uint32_t*>(orow + nt * 8) = pack_bf16x2(o[nt][0] * inv, o[nt][1] * inv);
                if (A.lse != nullptr && cq == 0)
                    A.lse[(size_t)tok * A.pool.Hq + h0 + row] = (m + log2f(l)) * 0.6931471805599453f;
            } else {
                float* prow = A.part_o + ((size_t)u * kHeadBlock + row) * D + cq;
#pragma unroll
                for (int nt = 0; nt < D / 8; ++nt) *reinterpret_cast<float2*>(prow + nt * 8) = make_float2(o[nt][0], o[nt][1]);
                if (cq == 0) A.part_ml[(size_t)u * kHeadBlock + row] = make_float2(m, l);
            }
        }
    }
}

// A5: combine the split partials of one (decode request, q head) in fixed split order.
struct CombineArgs {
    PoolDesc pool;
    BatchDesc b;
    uint16_t* out;
    float* lse;
    const int4* req_info;
    const float2* part_ml;
    const float* part_o;
};

template <int D>
__device__ __forceinline__ void combine_row(const CombineArgs& A, int req, int hq, int lane) {
    const int4 info = A.req_info[req];
    if (info.x != 1 || info.z <= 1) return;
    const int g = A.pool.Hq / A.pool.Hkv;
    const int HB = (g + kHeadBlock - 1) / kHeadBlock;
    const int kvh = hq / g, hb = (hq % g) / kHeadBlock, r = (hq % g) % kHeadBlock;
    const int nsplit = info.z;
    const size_t u0 = (size_t)info.y + ((size_t)kvh * nsplit) * HB + hb;
    float M = -INFINITY;
    for (int s = 0; s < nsplit; ++s) M = fmaxf(M, A.part_ml[(u0 + (size_t)s * HB) * kHeadBlock + r].x);
    constexpr int EPL = D / 32;
    float acc[EPL], l = 0.f;
#pragma unroll
    for (int e = 0; e < EPL; ++e) acc[e] = 0.f;
    for (int s = 0; s < nsplit; ++s) {
        const size_t u = u0 + (size_t)s * HB;
        const float2 ml = A.part_ml[u * kHeadBlock + r];
        const float w = exp2f(ml.x - M);
        l += ml.y * w;
        const float* po = A.part_o + (u * kHeadBlock + r) * D + lane * EPL;
#pragma unroll
        for (int e = 0; e < EPL; ++e) acc[e] = fmaf(po[e], w, acc[e]);
    }
    const float inv = 1.f / l;
    const int tok = A.b.q_offsets[req];
    uint16_t* orow = A.out + ((size_t)tok * A.pool.Hq + hq) * D + lane * EPL;
    if (EPL == 4) {
        uint2 w;
        w.x = pack_bf16x2(acc[0] * inv, acc[1] * inv);
        w.y = pack_bf16x2(acc[2] * inv, acc[3] * inv);
        *reinterpret_cast<uint2*>(orow) = w;
    } else {
        *reinterpret_cast<uint32_t*>(orow) = pack_bf16x2(acc[0] * inv, acc[1] * inv);
    }
    if (A.lse != nullptr && lane == 0) A.lse[(size_t)tok * A.pool.Hq + hq] = (M + log2f(l)) * 0.6931471805599453f;
}

}  // namespace tropical
