// decode.cuh -- SURVEY.md 8(a) row A4: decode tiles (split-K flash decoding over pages).
//
// One WARP is one decode worker.  It pops a unit (request, kv head, head block, page range) and
// streams the unit's K and V page-heads HBM -> shared memory with TMA (64-column SWIZZLE_128B
// boxes, i.e. whole 4 KiB contiguous page-head blocks of the HND pool, landed bank-conflict-free
// for ldmatrix) through a private ring of page-head sized stages -- K(p), V(p), K(p+1), V(p+1), ...,
// one mbarrier each -- that is kept full: a stage is refilled as soon as the warp has read it, so
// (ring - 1) page-heads are in flight per warp while one is consumed.
// The math runs on warp-level tensor-core MMAs in the TRANSPOSED orientation, so the 16 keys of a
// page are the M rows and the (up to 8) q heads of the kv group are the N columns:
//     S^T[16 keys x 8 heads] = K[16 x d] Q^T[d x 8]          (A = K page via ldmatrix, B = q registers)
//     O^T[d x 8 heads]      += V^T[d x 16 keys] P^T[16 x 8]  (A = V page via ldmatrix.trans,
//                                                             B = P^T via movmatrix of the S^T fragment)
// No accumulator row is padding (an m16n8k16 tile with heads as M would waste rows 8-15), which
// halves the MMA count and the accumulator registers.  Online softmax in registers, max over keys
// by shuffles across the 8 row groups.  HBM-bound: each K/V byte is read once; arithmetic per byte
// is the same for MHA and GQA.
// Results: final bf16 row when the request has one split, else fp32 partial (m, l, o) for A5.
#pragma once
#include "common.cuh"
#include "plan.cuh"

namespace tropical {

template <int D>
struct DecodeCfg {
    static constexpr int CB = D / 64;                 // 64-column swizzle blocks per row
    static constexpr int HALF_BYTES = 16 * 128;       // one TMA box: 16 rows x 128 B
    static constexpr int PAGE_BYTES = CB * HALF_BYTES;  // K (or V) of one page-head = one ring stage
};

constexpr int kMaxDecodeStages = 32;  // mbarriers reserved per decode warp

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
    int* group_cnt;   // per split group (request, kv head, head block): units finished so far; zeroed by the plan kernel
    // Fused step (tropical_mixed_step): this step's rows [T][Hkv][D], not yet in the pool -- the attention roles read them
    // from here and idle warps copy them into the pool meanwhile (append_worker).  nullptr: the rows are in the pool.
    const uint16_t* k_new;
    const uint16_t* v_new;
};

// Ring state of one decode warp; persists across units so barrier parities stay consistent.
struct DecodeRing {
    uint8_t* base;     // nst * PAGE_BYTES bytes, 1024-aligned
    uint64_t* full;    // nst mbarriers (count 1)
    int nst;           // stages
    int c_slot;        // next stage to consume (== next stage to fill when nothing is in flight)
    uint32_t c_phase;  // parity of c_slot's current use
    int i_slot;        // next stage to fill
};

// Fused step: the request's own new token is not in the pool yet.  Its K (or V) row replaces slot `slot` of the page-head
// that TMA has just landed in the stage at `stage_s` (SWIZZLE_128B layout: [half][16 slots][128 B], 16-byte chunk c of
// slot r at r * 128 + ((c ^ (r & 7)) << 4)).  `v` = this lane's 16-byte chunk of the row (lanes < D / 8).
template <int D>
__device__ __forceinline__ void patch_new_row(uint32_t stage_s, const uint4& v, int slot, int lane) {
    if (lane < D / 8) {
        const uint32_t a = stage_s + (lane >> 3) * DecodeCfg<D>::HALF_BYTES + slot * 128 + (((lane & 7) ^ (slot & 7)) << 4);
        asm volatile("st.shared.v4.b32 [%0], {%1,%2,%3,%4};" ::"r"(a), "r"(v.x), "r"(v.y), "r"(v.z), "r"(v.w) : "memory");
    }
    __syncwarp();
}

// Row A1 inside the step kernel (fused step): warps with nothing else to do -- warp 15 always, the decode workers once
// their queue is empty -- pop blocks of kAppendTokens new tokens and copy their K / V rows into the pool: lanes look up
// (page, slot) of the block's tokens, then the warp moves 16-byte chunks, 8 independent rows in flight per lane.  Same
// bit copy as kv_append_kernel.  Nobody reads these slots from the pool during this step.
constexpr int kAppendTokens = 2;
template <int D>
__device__ __noinline__ void append_worker(const DecodeArgs& A) {
    if (A.k_new == nullptr) return;
    constexpr int CH = D / 8;     // 16-byte chunks per row
    constexpr int RPW = 32 / CH;  // rows (kv heads) per warp pass
    constexpr int SEG = 2 * kAppendTokens;  // (token, K|V) segments of a block, all in flight together
    const int lane = threadIdx.x & 31;
    const int T = A.b.total_q, Hkv = A.pool.Hkv;
    const int n_tickets = (T + kAppendTokens - 1) / kAppendTokens;
    int* ticket = const_cast<int*>(A.hdr) + HDR_TICKET_APPEND;
    const uint4* src_kv[2] = {reinterpret_cast<const uint4*>(A.k_new), reinterpret_cast<const uint4*>(A.v_new)};
    uint4* dst_kv[2] = {reinterpret_cast<uint4*>(const_cast<uint16_t*>(A.pool.k_pool)),
                        reinterpret_cast<uint4*>(const_cast<uint16_t*>(A.pool.v_pool))};
    const int sub = lane / CH, chunk = lane % CH;
    for (;;) {
        // look before taking a ticket: at the end of a step every decode worker passes here, and ~1800 atomics on one
        // address would serialise the kernel's tail
        // Lane 0 alone looks and takes; the warp leaves on the broadcast value.  (Every lane reading the counter for
        // itself could see different values while other CTAs bump it, and lanes that left early would then be
        // missing from the full-mask shuffles below.)
        int tk = n_tickets;
        if (lane == 0 && *reinterpret_cast<volatile int*>(ticket) < n_tickets) tk = atomicAdd(ticket, 1);
        tk = __shfl_sync(0xffffffffu, tk, 0);
        if (tk >= n_tickets) break;
        const int t0 = tk * kAppendTokens, nt = min(kAppendTokens, T - t0);
        long long base = 0;  // lane i < nt: (page, head 0, slot) of token t0 + i, in 16-byte units
        if (lane < nt) {
            const int tok = t0 + lane;
            const int req = find_request(A.b.q_offsets, A.b.num_reqs, tok);
            const int pos = __ldg(A.b.ctx_lens + req) + tok - __ldg(A.b.q_offsets + req);
            const int page = __ldg(A.b.page_table + (size_t)req * A.b.stride + pos / kPageSize);
            base = ((long long)page * Hkv * kPageSize + pos % kPageSize) * CH;
        }
        // segment g = (token g / 2, K|V g % 2): this lane's chunk of kv head `sub`, then heads sub + RPW, ...
        const uint4* src[SEG];
        uint4* dst[SEG];
#pragma unroll
        for (int g = 0; g < SEG; ++g) {
            const int i = min(g >> 1, nt - 1);
            const long long b = __shfl_sync(0xffffffffu, base, i);
            src[g] = src_kv[g & 1] + ((size_t)(t0 + i) * Hkv + sub) * CH + chunk;
            dst[g] = dst_kv[g & 1] + b + (long long)sub * kPageSize * CH + chunk;
        }
        for (int h = sub; h < Hkv; h += RPW) {
            uint4 v[SEG];
#pragma unroll
            for (int g = 0; g < SEG; ++g) v[g] = __ldg(src[g]);
#pragma unroll
            for (int g = 0; g < SEG; ++g) {
                if ((g >> 1) < nt) *dst[g] = v[g];   // an odd last block: its second token's segments repeat the first's reads
                src[g] += RPW * CH;
                dst[g] += RPW * kPageSize * CH;
            }
        }
    }
}

__device__ __forceinline__ uint32_t movmatrix_trans(uint32_t a) {
    uint32_t d;
    asm volatile("movmatrix.sync.aligned.m8n8.trans.b16 %0, %1;" : "=r"(d) : "r"(a));
    return d;
}

// A5 (in-kernel): merge the split partials of the (up to 8) q heads of one split group, in split-index order -- the
// result does not depend on which unit finished last.  Called by the warp whose unit completed the group; the
// partials of the other units were published with __threadfence() before their counter increment, and are read
// through L2 (ld.global.cg) here.
template <int D>
__device__ __noinline__ void combine_group(const DecodeArgs& A, size_t u_first, int HB, int nsplit, int nh, int tok, int h0,
                                           int lane) {
    // lane -> (head r = lane / 4, quarter k = lane % 4); the lane owns the float4s j * 4 + k (j < D / 16) of its head's
    // row, so the 8 heads of the group are merged concurrently with D / 16 independent loads per split in flight
    constexpr int J = D / 16;
    const int r = lane >> 2, k = lane & 3;
    if (r >= nh) return;
    float M = -INFINITY;
#pragma unroll 4
    for (int s = 0; s < nsplit; ++s) M = fmaxf(M, __ldcg(&A.part_ml[(u_first + (size_t)s * HB) * kHeadBlock + r]).x);
    float4 acc[J];
    float l = 0.f;
#pragma unroll
    for (int j = 0; j < J; ++j) acc[j] = make_float4(0.f, 0.f, 0.f, 0.f);
#pragma unroll 2
    for (int s = 0; s < nsplit; ++s) {
        const size_t u = u_first + (size_t)s * HB;
        const float2 ml = __ldcg(&A.part_ml[u * kHeadBlock + r]);
        const float w = exp2f(ml.x - M);
        l += ml.y * w;
        const float4* po = reinterpret_cast<const float4*>(A.part_o + (u * kHeadBlock + r) * D) + k;
#pragma unroll
        for (int j = 0; j < J; ++j) {
            const float4 v = __ldcg(po + j * 4);
            acc[j].x = fmaf(v.x, w, acc[j].x);
            acc[j].y = fmaf(v.y, w, acc[j].y);
            acc[j].z = fmaf(v.z, w, acc[j].z);
            acc[j].w = fmaf(v.w, w, acc[j].w);
        }
    }
    const float inv = 1.f / l;
    uint2* orow = reinterpret_cast<uint2*>(A.out + ((size_t)tok * A.pool.Hq + h0 + r) * D) + k;
#pragma unroll
    for (int j = 0; j < J; ++j) {
        uint2 w;
        w.x = pack_bf16x2(acc[j].x * inv, acc[j].y * inv);
        w.y = pack_bf16x2(acc[j].z * inv, acc[j].w * inv);
        orow[j * 4] = w;
    }
    if (A.lse != nullptr && k == 0) A.lse[(size_t)tok * A.pool.Hq + h0 + r] = (M + log2f(l)) * 0.6931471805599453f;
}

// FUSED: the fused step (tropical_mixed_step with the append inside the kernel).  The plain variant compiles none of the
// new-row handling: every instruction in the page loop is paid 300 000 times per C5 step.
template <int D, bool FUSED>
__device__ __forceinline__ void decode_warp_worker(const DecodeArgs& A, const CUtensorMap* tm_k, const CUtensorMap* tm_v,
                                                   DecodeRing& R) {
    using C = DecodeCfg<D>;
    const int lane = threadIdx.x & 31;
    const int row = lane >> 2, cq = (lane & 3) * 2;
    const int g = A.pool.Hq / A.pool.Hkv;
    const int n_units = A.hdr[HDR_N_UNITS];
    const uint32_t ring_s = uni(smem_u32(R.base));
    const uint32_t full_s = uni(smem_u32(R.full));
    const int Hkv = uni(A.pool.Hkv);
    // ldmatrix lane addressing (row within 8x8 matrix r8, matrix id mi)
    const int mi = lane >> 3, r8 = lane & 7;
    const int k_key = (mi & 1) * 8 + r8, k_chunk_off = mi >> 1;  // K as A: (keys lo/hi) x (chunk, chunk+1)
    const int v_key = (mi >> 1) * 8 + r8, v_chunk_off = mi & 1;  // V^T as A (trans): (chunk, chunk+1) x (keys lo/hi)
    // Swizzled byte offset of this lane's ldmatrix row inside a stage.  Chunk c of row r sits at
    // r*128 + ((c ^ (r & 7)) << 4); c = 2*i + off with off in {0,1}, so (c ^ x) = (2*i) ^ (off ^ x): the
    // per-instruction part is an XOR with a compile-time constant on top of one per-lane register.
    const uint32_t k_lane = k_key * 128 + ((k_chunk_off ^ (k_key & 7)) << 4);
    const uint32_t v_lane = v_key * 128 + ((v_chunk_off ^ (v_key & 7)) << 4);

    for (;;) {
        int u = 0;
        if (lane == 0) u = atomicAdd(A.ticket, 1);
        u = __shfl_sync(0xffffffffu, u, 0);
        if (u >= n_units) break;
        const int4 un = A.units[u];
        const int req = un.x, kvh = un.y & 0xffff, hb = un.y >> 16, p0 = un.z, np = un.w;
        const int kvh_u = uni(kvh);
        const int L = __ldg(A.b.ctx_lens + req) + 1;
        const int tok = __ldg(A.b.q_offsets + req);
        const int h0 = kvh * g + hb * kHeadBlock;
        const int nh = min(kHeadBlock, g - hb * kHeadBlock);
        const int* pt = A.b.page_table + (size_t)req * A.b.stride + p0;

        // Q^T fragments (B operand: column = head of the group; heads >= nh are zero)
        uint32_t qb[D / 16][2];
        {
            const uint16_t* qrow = A.q + ((size_t)tok * A.pool.Hq + h0 + row) * D;
#pragma unroll
            for (int ks = 0; ks < D / 16; ++ks) {
                qb[ks][0] = row < nh ? *reinterpret_cast<const uint32_t*>(qrow + ks * 16 + cq) : 0u;
                qb[ks][1] = row < nh ? *reinterpret_cast<const uint32_t*>(qrow + ks * 16 + 8 + cq) : 0u;
            }
        }
        // Fused step: the unit that holds the request's last page takes the new token's K / V row from k_new / v_new
        // (fused step) page of this unit that holds the request's own new token, whose row is not in the pool yet: -1 = none
        const int p_patch = (FUSED && (p0 + np) * kPageSize >= L) ? np - 1 : -1;
        // O^T accumulators: o[db][0,1] = d row (db*16 + row) x heads (cq, cq+1); o[db][2,3] = d row + 8
        float o[D / 16][4];
#pragma unroll
        for (int db = 0; db < D / 16; ++db) o[db][0] = o[db][1] = o[db][2] = o[db][3] = 0.f;
        float m0 = -INFINITY, m1 = -INFINITY, l0 = 0.f, l1 = 0.f;  // heads cq, cq+1 (l: this lane's keys only)

        // ---- stage issue: sub-stage j = K (j even) or V (j odd) of page j >> 1
        const int n_sub = 2 * np;
        int issued = 0, ptv = 0;
        auto issue_one = [&]() {  // whole warp calls; one elected lane issues the boxes of sub-stage `issued`
            const int pi = issued >> 1;
            if ((issued & 63) == 0) ptv = (pi + lane < np) ? __ldg(pt + pi + lane) : 0;
            const int page = __shfl_sync(0xffffffffu, ptv, pi & 31);  // warp-uniform: no waterfall around UTMALDG
            const uint32_t dst = ring_s + R.i_slot * C::PAGE_BYTES;
            const uint32_t bar = full_s + R.i_slot * 8;
            const int r0 = (page * Hkv + kvh_u) * kPageSize;
            const CUtensorMap* tm = (issued & 1) ? tm_v : tm_k;
            if (elect_one()) {
                asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"((uint32_t)C::PAGE_BYTES) : "memory");
#pragma unroll
                for (int cb = 0; cb < C::CB; ++cb)
                    asm volatile(
                        "cp.async.bulk.tensor.2d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%3, %4}], [%2];"
                        ::"r"(dst + cb * C::HALF_BYTES), "l"(tm), "r"(bar), "r"(cb * 64), "r"(r0)
                        : "memory");
            }
            __syncwarp();
            R.i_slot = (R.i_slot + 1 == R.nst) ? 0 : R.i_slot + 1;
            ++issued;
        };
        auto consume_advance = [&]() {
            if (++R.c_slot == R.nst) { R.c_slot = 0; R.c_phase ^= 1; }
        };
        {
            const int pre = min(R.nst, n_sub);
            for (int i = 0; i < pre; ++i) issue_one();
        }

        for (int p = 0; p < np; ++p) {
            // ---------------- S^T = K Q^T for the 16 keys of this page
            const int nvalid = L - (p0 + p) * kPageSize;  // >= 1 by construction of the unit; <= 16 on the request's last page
            const bool patch = FUSED && p == p_patch;  // the page that holds this step's token (slot nvalid - 1)
            const size_t new_row = ((size_t)tok * Hkv + kvh) * (D / 8) + lane;  // this lane's 16-byte chunk of the new row
            uint4 kn = make_uint4(0u, 0u, 0u, 0u);
            if (patch && lane < D / 8) kn = __ldg(reinterpret_cast<const uint4*>(A.k_new) + new_row);  // in flight while the page lands
            mbar_wait(R.full + R.c_slot, R.c_phase, 201);
            const uint32_t kbase = ring_s + R.c_slot * C::PAGE_BYTES;
            if (patch) patch_new_row<D>(kbase, kn, nvalid - 1, lane);
            float sa[4] = {0.f, 0.f, 0.f, 0.f}, sb[4] = {0.f, 0.f, 0.f, 0.f};
#pragma unroll
            for (int ks = 0; ks < D / 16; ++ks) {
                const uint32_t addr = ((kbase + k_lane) ^ (uint32_t)((ks & 3) * 32)) + (ks >> 2) * C::HALF_BYTES;
                uint32_t a0, a1, a2, a3;
#ifdef TROPICAL_WHATIF_NO_DECODE_MATH
                if (ks > 0) continue;
#endif
                ldmatrix_x4(addr, a0, a1, a2, a3);
                if (ks & 1) mma_bf16_16816(sb, a0, a1, a2, a3, qb[ks][0], qb[ks][1]);
                else mma_bf16_16816(sa, a0, a1, a2, a3, qb[ks][0], qb[ks][1]);
            }
            if (patch) fence_proxy_async();  // generic write of the new row before a TMA refill of the stage
            __syncwarp();  // every lane has read the K stage
            consume_advance();
            if (issued < n_sub) issue_one();

            // sa/sb[0,1]: key `row`, heads cq, cq+1;  [2,3]: key row + 8.  Scores relative to the running reference
            // maximum m (shared by the 8 row groups of a head): x = s * scale - m.
            float s00 = sa[0] + sb[0], s01 = sa[1] + sb[1], s10 = sa[2] + sb[2], s11 = sa[3] + sb[3];
            if (nvalid < kPageSize) {  // ragged last page: mask by select (the score of an unused slot may be NaN)
                if (row >= nvalid) { s00 = -INFINITY; s01 = -INFINITY; }
                if (row + 8 >= nvalid) { s10 = -INFINITY; s11 = -INFINITY; }
            }
            float v00 = fmaf(s00, A.scale_log2, -m0), v01 = fmaf(s01, A.scale_log2, -m1);
            float v10 = fmaf(s10, A.scale_log2, -m0), v11 = fmaf(s11, A.scale_log2, -m1);
            // Lazy maximum: m is raised (shuffle reduction over the 16 keys, rescale of O and l) only when some score
            // of the page exceeds it by more than 2^8 -- always on the first page of a unit (m = -inf), rarely after.
            if (__any_sync(0xffffffffu, fmaxf(fmaxf(v00, v01), fmaxf(v10, v11)) > 8.f)) {
                float mx0 = fmaxf(s00, s10) * A.scale_log2, mx1 = fmaxf(s01, s11) * A.scale_log2;
#pragma unroll
                for (int off = 4; off < 32; off <<= 1) {
                    mx0 = fmaxf(mx0, __shfl_xor_sync(0xffffffffu, mx0, off));
                    mx1 = fmaxf(mx1, __shfl_xor_sync(0xffffffffu, mx1, off));
                }
                const float mn0 = fmaxf(m0, mx0), mn1 = fmaxf(m1, mx1);  // finite: key 0 of the page is valid
                const float al0 = fast_exp2(m0 - mn0), al1 = fast_exp2(m1 - mn1);
                l0 *= al0;
                l1 *= al1;
#pragma unroll
                for (int db = 0; db < D / 16; ++db) { o[db][0] *= al0; o[db][1] *= al1; o[db][2] *= al0; o[db][3] *= al1; }
                m0 = mn0;
                m1 = mn1;
                v00 = fmaf(s00, A.scale_log2, -m0);
                v01 = fmaf(s01, A.scale_log2, -m1);
                v10 = fmaf(s10, A.scale_log2, -m0);
                v11 = fmaf(s11, A.scale_log2, -m1);
            }
            v00 = fast_exp2(v00);
            v10 = fast_exp2(v10);
            v01 = fast_exp2(v01);
            v11 = fast_exp2(v11);
            l0 += v00 + v10;
            l1 += v01 + v11;
            // P^T as B operand: transpose the two 8x8 (key x head) bf16 blocks of the S^T fragment
            const uint32_t pb0 = movmatrix_trans(pack_bf16x2(v00, v01));
            const uint32_t pb1 = movmatrix_trans(pack_bf16x2(v10, v11));

            // ---------------- O^T += V^T P^T
            uint4 vn = make_uint4(0u, 0u, 0u, 0u);
            if (patch && lane < D / 8) vn = __ldg(reinterpret_cast<const uint4*>(A.v_new) + new_row);
            mbar_wait(R.full + R.c_slot, R.c_phase, 202);
            const uint32_t vbase = ring_s + R.c_slot * C::PAGE_BYTES;
            if (patch) patch_new_row<D>(vbase, vn, nvalid - 1, lane);
            if (nvalid < kPageSize) {  // ragged last page: unused slots may hold NaN bits; 0 * NaN = NaN in the MMA
                const int nz = (kPageSize - nvalid) * 8 * C::CB;
                for (int idx = lane; idx < nz; idx += 32) {
                    const int r = nvalid + idx / (8 * C::CB), rem = idx % (8 * C::CB);
                    const uint32_t a = vbase + (rem >> 3) * C::HALF_BYTES + r * 128 + ((rem & 7) << 4);
                    asm volatile("st.shared.v4.b32 [%0], {%1,%1,%1,%1};" ::"r"(a), "r"(0u) : "memory");
                }
                __syncwarp();
            }
#pragma unroll
            for (int db = 0; db < D / 16; ++db) {
                const uint32_t addr = ((vbase + v_lane) ^ (uint32_t)((db & 3) * 32)) + (db >> 2) * C::HALF_BYTES;
                uint32_t a0, a1, a2, a3;
#ifdef TROPICAL_WHATIF_NO_DECODE_MATH
                if (db > 0) continue;
#endif
                ldmatrix_x4_trans(addr, a0, a1, a2, a3);
                mma_bf16_16816(o[db], a0, a1, a2, a3, pb0, pb1);
            }
            if (nvalid < kPageSize || patch) fence_proxy_async();  // generic zero-fill / new row before the next TMA refill
            __syncwarp();  // every lane is done with the V stage
            consume_advance();
            if (issued < n_sub) issue_one();
        }

#pragma unroll
        for (int off = 4; off < 32; off <<= 1) {
            l0 += __shfl_xor_sync(0xffffffffu, l0, off);
            l1 += __shfl_xor_sync(0xffffffffu, l1, off);
        }
        const int nsplit = A.req_info[req].z;
        // this lane owns heads cq, cq+1 and d rows {db*16 + row, db*16 + row + 8}
        if (nsplit == 1) {
            const float i0 = 1.f / l0, i1 = 1.f / l1;
            __nv_bfloat16* ob = reinterpret_cast<__nv_bfloat16*>(A.out) + ((size_t)tok * A.pool.Hq + h0) * D;
#pragma unroll
            for (int db = 0; db < D / 16; ++db) {
                const int d0 = db * 16 + row;
                if (cq < nh) {
                    ob[(size_t)cq * D + d0] = __float2bfloat16_rn(o[db][0] * i0);
                    ob[(size_t)cq * D + d0 + 8] = __float2bfloat16_rn(o[db][2] * i0);
                }
                if (cq + 1 < nh) {
                    ob[(size_t)(cq + 1) * D + d0] = __float2bfloat16_rn(o[db][1] * i1);
                    ob[(size_t)(cq + 1) * D + d0 + 8] = __float2bfloat16_rn(o[db][3] * i1);
                }
            }
            if (A.lse != nullptr && row == 0) {
                if (cq < nh) A.lse[(size_t)tok * A.pool.Hq + h0 + cq] = (m0 + log2f(l0)) * 0.6931471805599453f;
                if (cq + 1 < nh) A.lse[(size_t)tok * A.pool.Hq + h0 + cq + 1] = (m1 + log2f(l1)) * 0.6931471805599453f;
            }
        } else {
            float* pb = A.part_o + (size_t)u * kHeadBlock * D;
#pragma unroll
            for (int db = 0; db < D / 16; ++db) {
                const int d0 = db * 16 + row;
                if (cq < nh) {
                    pb[cq * D + d0] = o[db][0];
                    pb[cq * D + d0 + 8] = o[db][2];
                }
                if (cq + 1 < nh) {
                    pb[(cq + 1) * D + d0] = o[db][1];
                    pb[(cq + 1) * D + d0 + 8] = o[db][3];
                }
            }
            if (row == 0) {
                if (cq < nh) A.part_ml[(size_t)u * kHeadBlock + cq] = make_float2(m0, l0);
                if (cq + 1 < nh) A.part_ml[(size_t)u * kHeadBlock + cq + 1] = make_float2(m1, l1);
            }
            // last unit of the split group to finish merges the group (A5)
            const int HB = (g + kHeadBlock - 1) / kHeadBlock;
            const int s_idx = ((u - A.req_info[req].y) / HB) % nsplit;
            const size_t u_first = (size_t)u - (size_t)s_idx * HB;
            __threadfence();
            __syncwarp();
            int done = 0;
            if (lane == 0) done = atomicAdd(A.group_cnt + u_first, 1);
            done = __shfl_sync(0xffffffffu, done, 0);
            if (done == nsplit - 1) {
                __threadfence();
                combine_group<D>(A, u_first, HB, nsplit, nh, tok, h0, lane);
            }
        }
    }
    if constexpr (FUSED) append_worker<D>(A);  // what is left of this step's rows to copy into the pool
}

}  // namespace tropical
