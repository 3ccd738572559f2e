// decode_tc.cuh -- SURVEY.md 8(a) row A4 on the 5th-gen tensor cores: decode tiles in the TRANSPOSED
// orientation, so that the keys of a 128-key block (8 pages) are the M rows of the MMA and the (up to 8) q
// heads of the kv group are its N columns:
//     S^T[128 keys x 16] = K[128 x d] Q^T[d x 16]            A = K block (smem, K-major SW128, the same TMA
//                                                            boxes as the prefill K tile), B = Q^T (smem)
//     P^T = exp2(S^T * scale*log2e - m)                      one thread per KEY (tcgen05.ld 32x32b.x8), bf16 to smem
//     O^T[d x 16]       += V^T[d x 128 keys] P^T[128 x 16]   A = V block (smem, MN-major SW128), B = P^T (smem)
// A unit (request, kv head, block of <= 8 q heads, page range) is a run of such blocks; the fp32 O^T accumulator
// lives in TMEM (d = TMEM lane), so the decode role needs ~60 registers per thread and ~600 instructions per
// 64 KiB of K/V instead of the ~3500 of a warp-level (mma.sync) formulation, and it queues on the tensor pipe
// behind the prefill MMAs instead of stalling warps on it (profiles/r1b_c5.md).
//
// Online softmax without per-block reductions: the running maximum m[h] is shared by all 128 key threads and
// is only raised when some key of a block exceeds it by more than 2^8 (one barrier.red.or per block decides);
// the first block of a unit always takes that path.  Raising m rescales O^T in TMEM and the per-thread l[h].
//
// Roles (persistent over the decode ticket queue, 2-deep mailbox like the prefill roles):
//   producer warp : TMA.  Q^T (8 heads x d of the request's token) and, per block, K then V into a ring of
//                   16 KiB units: K unit = 128 keys x 64 columns, V unit = (8192 / d) keys x d columns.
//   MMA warp      : one elected lane issues S^T(b+1) ahead of PV(b).
//   softmax WG    : 4 warps, thread r = key r of the block; in the unit epilogue thread r = row r of O^T.
// Unused slots of a last page may hold NaN: scores are masked by select, P of an invalid key is exactly 0 and
// the V rows past the last valid key of a unit are zeroed in shared memory before PV (0 * NaN).
#pragma once
#include <cuda.h>

#include "common.cuh"
#include "plan.cuh"

namespace tropical {

constexpr int kDecBlockKeys = 128;
constexpr int kDecBlockPages = kDecBlockKeys / kPageSize;
constexpr int kDecMaxUnits = 8;  // ring units (mbarrier pairs) reserved per pipe

template <int D>
struct DecTcCfg {
    static constexpr int CB = D / 64;
    static constexpr int UNIT_BYTES = 16384;
    static constexpr int V_KEYS = kDecBlockKeys / CB;        // keys per V unit
    static constexpr int V_PAGES = V_KEYS / kPageSize;
    static constexpr int QT_BYTES = CB * 2048;               // per 64-column half: 16 rows x 128 B (rows 8-15 unused)
    static constexpr int PT_BYTES = 2 * 2048;                // two 64-key halves: 16 rows x 128 B each
    static constexpr int TM_ST = 0, TM_OT = 32, TM_COLS = 64;  // S^T slots at +0, +16; O^T slots at +32, +48
};

struct DecBars {
    uint64_t unit_full[2], unit_empty[2];
    uint64_t qt_full[2], qt_empty[2];
    uint64_t ring_full[kDecMaxUnits], ring_empty[kDecMaxUnits];
    uint64_t s_full[2], p_full[2];
    uint64_t pv_done;
    uint64_t o_full[2], o_empty[2];
    int mailbox[2];
    float red[2][4][8];
    float lsum[4][8];
};

struct DecPipe {
    uint8_t* ring;     // nunits * 16 KiB, 1024-aligned
    int nunits;
    uint8_t* qt;       // 2 x QT_BYTES
    uint8_t* pt;       // 2 x PT_BYTES
    DecBars* B;
    uint32_t tm;       // TMEM base column of this pipe (absolute address, lane 0)
    int bar_id;        // named barrier of the softmax warpgroup
};

struct DecTcArgs {
    PoolDesc pool;
    BatchDesc b;
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

__device__ __forceinline__ void dec_init_bars(DecBars* B) {
    for (int i = 0; i < 2; ++i) {
        mbar_init(&B->unit_full[i], 1);
        mbar_init(&B->unit_empty[i], 6);  // lane 0 of the V producer, the MMA warp and each softmax warp
        mbar_init(&B->qt_full[i], 1);
        mbar_init(&B->qt_empty[i], 1);
        mbar_init(&B->s_full[i], 1);
        mbar_init(&B->p_full[i], 128);
        mbar_init(&B->o_full[i], 1);
        mbar_init(&B->o_empty[i], 128);
    }
    for (int i = 0; i < kDecMaxUnits; ++i) {
        mbar_init(&B->ring_full[i], 1);
        mbar_init(&B->ring_empty[i], 1);
    }
    mbar_init(&B->pv_done, 1);
}

struct DecUnit {
    int req, kvh, hb, p0, np;
    int nb;        // 128-key blocks
    int key_end;   // valid keys of the unit, relative to its first key
};

__device__ __forceinline__ DecUnit dec_load_unit_raw(const DecTcArgs& A, int u) {
    DecUnit U;
    const int4 un = A.units[u];
    U.req = un.x;
    U.kvh = un.y & 0xffff;
    U.hb = un.y >> 16;
    U.p0 = un.z;
    U.np = un.w;
    U.nb = (U.np + kDecBlockPages - 1) / kDecBlockPages;
    const int L = __ldg(A.b.ctx_lens + U.req) + 1;
    U.key_end = min(L, (U.p0 + U.np) * kPageSize) - U.p0 * kPageSize;
    return U;
}
// every field broadcast from lane 0: warp-uniform for the compiler (see uni())
__device__ __forceinline__ DecUnit dec_load_unit(const DecTcArgs& A, int u) {
    DecUnit U = dec_load_unit_raw(A, u);
    U.req = uni(U.req); U.kvh = uni(U.kvh); U.hb = uni(U.hb); U.p0 = uni(U.p0); U.np = uni(U.np);
    U.nb = uni(U.nb); U.key_end = uni(U.key_end);
    return U;
}

// ------------------------------------------------------------------------------------------------ producers
// Ring entries follow the MMA warp's consumption order K(0), K(1), V(0), K(2), V(1), ..., V(nb-1); the K producer
// (KIND 0: pops the unit tickets, loads Q^T and the K units) and the V producer (KIND 1) both walk that sequence and
// each fills the entries of its own kind.  One rolled loop over "steps" keeps a single copy of the issue code (the
// roles of an SM share a 32 KiB L1.5 instruction cache); boxes are issued lane-parallel (lane = page / half).  Page
// ids are read 32 at a time, one chunk ahead, so no global-load latency sits between two blocks.
template <int D, int KIND>
__device__ __noinline__ void dec_producer(const DecTcArgs& A, const DecPipe& P, const CUtensorMap* tm_qd,
                                          const CUtensorMap* tm_kv) {
    using C = DecTcCfg<D>;
    DecBars* B = P.B;
    const int lane = threadIdx.x & 31;
    const int n_units = uni(A.hdr[HDR_N_UNITS]);
    const int g = uni(A.pool.Hq / A.pool.Hkv), Hkv = uni(A.pool.Hkv);
    uint8_t* ring = P.ring;
    const int nunits = uni(P.nunits);
    uint32_t unit_it = 0;
    RingCursor cur = {0, 0};
    for (;;) {
        const int ms = unit_it & 1;
        const uint32_t par = (unit_it >> 1) & 1;
        int u = 0;
        if (KIND == 0) {
            mbar_wait(&B->unit_empty[ms], par ^ 1, 301);
            if (lane == 0) {
                u = atomicAdd(A.ticket, 1);
                B->mailbox[ms] = u;
                mbar_arrive(&B->unit_full[ms]);
            }
            u = __shfl_sync(0xffffffffu, u, 0);
        } else {
            mbar_wait(&B->unit_full[ms], par, 305);
            u = uni(B->mailbox[ms]);
            __syncwarp();
            if (lane == 0) mbar_arrive(&B->unit_empty[ms]);
        }
        if (u >= n_units) break;
        const DecUnit U = dec_load_unit(A, u);
        const int* pt = A.b.page_table + (size_t)U.req * A.b.stride + U.p0;
        int pg_cur = lane < U.np ? __ldg(pt + lane) : 0;
        int pg_next = 32 + lane < U.np ? __ldg(pt + 32 + lane) : 0;
        if (KIND == 0) {
            const int tok = uni(__ldg(A.b.q_offsets + U.req));
            const int h0 = U.kvh * g + U.hb * kHeadBlock;
            mbar_wait(&B->qt_empty[ms], par ^ 1, 302);
            if (elect_one()) {
                mbar_arrive_expect_tx(&B->qt_full[ms], C::CB * 1024);
#pragma unroll
                for (int cb = 0; cb < C::CB; ++cb)
                    tma_load_3d(P.qt + ms * C::QT_BYTES + cb * 2048, tm_qd, cb * 64, h0, tok, &B->qt_full[ms]);
            }
        }
        for (int s = 0; s <= U.nb; ++s) {
            const int b = KIND == 0 ? s : s - 1;  // the block this producer loads in step s
            int npb = 0;
            if (b >= 0 && b < U.nb) {
                npb = min(kDecBlockPages, U.np - b * kDecBlockPages);
                if (b > 0 && (b & 3) == 0) {
                    pg_cur = pg_next;
                    pg_next = b * kDecBlockPages + 32 + lane < U.np ? __ldg(pt + b * kDecBlockPages + 32 + lane) : 0;
                }
            }
            if (s < U.nb) {  // K units of block s: 128 keys x 64 columns each
                if (KIND == 0) {
                    const int page = __shfl_sync(0xffffffffu, pg_cur, ((b & 3) * kDecBlockPages + lane) & 31);
#pragma unroll 1
                    for (int cb = 0; cb < C::CB; ++cb) {
                        mbar_wait(&B->ring_empty[cur.slot], cur.phase ^ 1, 303);
                        if (lane == 0) mbar_arrive_expect_tx(&B->ring_full[cur.slot], npb * 2048);
                        __syncwarp();
                        if (lane < npb)
                            tma_load_2d(ring + cur.slot * C::UNIT_BYTES + lane * 2048, tm_kv, cb * 64,
                                        (page * Hkv + U.kvh) * kPageSize, &B->ring_full[cur.slot]);
                        cur.advance(nunits);
                    }
                } else {
                    for (int cb = 0; cb < C::CB; ++cb) cur.advance(nunits);
                }
            }
            if (s > 0) {  // V units of block s - 1: V_KEYS keys x d columns each
                const int npv = KIND == 0 ? min(kDecBlockPages, U.np - (s - 1) * kDecBlockPages) : npb;
                const int pp = lane / C::CB, cb = lane % C::CB;
#pragma unroll 1
                for (int j = 0; j < C::CB; ++j) {
                    const int npj = min(C::V_PAGES, npv - j * C::V_PAGES);
                    if (npj <= 0) break;
                    if (KIND == 1) {
                        const int page = __shfl_sync(0xffffffffu, pg_cur, ((b & 3) * kDecBlockPages + j * C::V_PAGES + pp) & 31);
                        mbar_wait(&B->ring_empty[cur.slot], cur.phase ^ 1, 304);
                        if (lane == 0) mbar_arrive_expect_tx(&B->ring_full[cur.slot], npj * C::CB * 2048);
                        __syncwarp();
                        if (lane < npj * C::CB)
                            tma_load_2d(ring + cur.slot * C::UNIT_BYTES + cb * (C::V_KEYS * 128) + pp * 2048, tm_kv, cb * 64,
                                        (page * Hkv + U.kvh) * kPageSize, &B->ring_full[cur.slot]);
                    }
                    cur.advance(nunits);
                }
            }
        }
        ++unit_it;
    }
}

// ------------------------------------------------------------------------------------------------ MMA issuer
template <int D>
__device__ __noinline__ void dec_mma(const DecTcArgs& A, const DecPipe& P) {
    using C = DecTcCfg<D>;
    DecBars* B = P.B;
    const int lane = threadIdx.x & 31;
    const int n_units = uni(A.hdr[HDR_N_UNITS]);
    const uint32_t ring_a = uni(smem_u32(P.ring)), qt_a = uni(smem_u32(P.qt)), pt_a = uni(smem_u32(P.pt));
    const uint32_t tm_base = uni(P.tm);
    const int nunits = uni(P.nunits);
    constexpr uint32_t IDESC_S = make_idesc_bf16(128, 16, false, false);
    constexpr uint32_t IDESC_O = make_idesc_bf16(128, 16, false, true);  // A = V^T: MN-major
    uint32_t unit_it = 0, blk_it = 0;
    RingCursor cur = {0, 0};

    for (;;) {
        const int ms = unit_it & 1;
        const uint32_t par = (unit_it >> 1) & 1;
        mbar_wait(&B->unit_full[ms], par, 311);
        const int u = uni(B->mailbox[ms]);
        __syncwarp();
        if (lane == 0) mbar_arrive(&B->unit_empty[ms]);
        if (u >= n_units) break;
        const DecUnit U = dec_load_unit(A, u);
        const uint32_t tm_o = tm_base + C::TM_OT + ms * 16;

        mbar_wait(&B->qt_full[ms], par, 313);
        // step s issues S^T(s) (ahead) and then PV(s - 1): one copy of each issue sequence
        for (int s = 0; s <= U.nb; ++s) {
            if (s < U.nb) {  // S^T(s) = K(s) Q^T into S^T slot (blk_it + s) & 1
                const int st = (blk_it + s) & 1;
#pragma unroll 1
                for (int cb = 0; cb < C::CB; ++cb) {
                    mbar_wait(&B->ring_full[cur.slot], cur.phase, 312);
                    tc_fence_after();
                    const uint32_t k_a = ring_a + cur.slot * C::UNIT_BYTES;
                    const uint32_t q_a = qt_a + ms * C::QT_BYTES + cb * 2048;
                    if (elect_one()) {
#pragma unroll
                        for (int k4 = 0; k4 < 4; ++k4)
                            tc_mma_ss(tm_base + C::TM_ST + st * 16, make_smem_desc_sw128(k_a + k4 * 32, 0, 1024),
                                      make_smem_desc_sw128(q_a + k4 * 32, 0, 1024), IDESC_S, (cb | k4) != 0);
                        tc_commit(&B->ring_empty[cur.slot]);
                    }
                    __syncwarp();
                    cur.advance(nunits);
                }
                if (elect_one()) {
                    tc_commit(&B->s_full[st]);
                    if (s + 1 == U.nb) tc_commit(&B->qt_empty[ms]);  // every S^T MMA of this unit has been issued
                }
                __syncwarp();
            }
            if (s == 0) continue;
            const int b = s - 1;
            const uint32_t gb = blk_it + b;
            const int st = gb & 1;
            const int npb = min(kDecBlockPages, U.np - b * kDecBlockPages);
            const int nvalid_blk = min(kDecBlockKeys, U.key_end - b * kDecBlockKeys);
            bool first = true;
#pragma unroll 1
            for (int j = 0; j < C::CB; ++j) {
                const int npj = min(C::V_PAGES, npb - j * C::V_PAGES);
                if (npj <= 0) break;
                mbar_wait(&B->ring_full[cur.slot], cur.phase, 314);
                const uint32_t v_a = ring_a + cur.slot * C::UNIT_BYTES;
                const int nv = min(C::V_KEYS, nvalid_blk - j * C::V_KEYS);  // >= 1: every page of a unit has a valid key
                if (nv < C::V_KEYS) {  // zero the rows past the last valid key (stale or poisoned smem)
                    const int nz = (C::V_KEYS - nv) * 8 * C::CB;
                    for (int idx = lane; idx < nz; idx += 32) {
                        const int r = nv + idx / (8 * C::CB), rem = idx % (8 * C::CB);
                        const uint32_t a = v_a + (rem >> 3) * (C::V_KEYS * 128) + r * 128 + ((rem & 7) << 4);
                        asm volatile("st.shared.v4.b32 [%0], {%1,%1,%1,%1};" ::"r"(a), "r"(0u) : "memory");
                    }
                    fence_proxy_async();
                    __syncwarp();
                }
                if (first) {
                    if (b == 0) mbar_wait(&B->o_empty[ms], par ^ 1, 315);  // epilogue of unit_it - 2 has read this O^T slot
                    mbar_wait(&B->p_full[st], (gb >> 1) & 1, 316);
                    first = false;
                }
                tc_fence_after();
                const uint32_t p_a = pt_a + st * C::PT_BYTES + ((j * C::V_KEYS) >> 6) * 2048 + (((j * C::V_KEYS) & 63) >> 4) * 32;
                if (elect_one()) {
#pragma unroll
                    for (int ks = 0; ks < C::V_KEYS / 16; ++ks) {
                        // 16 keys per MMA: +32 B inside a 64-key P^T half, next half after 4 steps
                        const uint32_t pk = p_a + (ks >> 2) * 2048 + (ks & 3) * 32;
                        tc_mma_ss(tm_o, make_smem_desc_sw128(v_a + ks * 2048, C::V_KEYS * 128, 1024),
                                  make_smem_desc_sw128(pk, 0, 1024), IDESC_O, (b | j | ks) != 0);
                    }
                    tc_commit(&B->ring_empty[cur.slot]);
                }
                __syncwarp();
                cur.advance(nunits);
            }
            if (elect_one()) {
                tc_commit(&B->pv_done);
                if (b + 1 == U.nb) tc_commit(&B->o_full[ms]);
            }
            __syncwarp();
        }
        blk_it += U.nb;
        ++unit_it;
    }
}

// ------------------------------------------------------------------------------------------------ softmax warpgroup
template <int D>
__device__ __noinline__ void dec_softmax(const DecTcArgs& A, const DecPipe& P, int wg_warp) {
    using C = DecTcCfg<D>;
    DecBars* B = P.B;
    const int lane = threadIdx.x & 31;
    const int r = wg_warp * 32 + lane;
    const int n_units = A.hdr[HDR_N_UNITS];
    const int g = A.pool.Hq / A.pool.Hkv;
    const uint32_t tm = P.tm + ((uint32_t)(wg_warp * 32) << 16);
    const float scale = A.scale_log2;
    // this thread's key column inside a P^T half: 16-byte chunk (r & 63) >> 3 (XOR-swizzled with the head row), element r & 7
    const uint32_t pt_key = smem_u32(P.pt) + (r >> 6) * 2048 + (r & 7) * 2;
    const uint32_t pt_chunk = (r & 63) >> 3;
    uint32_t unit_it = 0, blk_it = 0;

    for (;;) {
        const int ms = unit_it & 1;
        const uint32_t par = (unit_it >> 1) & 1;
        mbar_wait(&B->unit_full[ms], par, 321);
        const int u = B->mailbox[ms];
        __syncwarp();
        if (lane == 0) mbar_arrive(&B->unit_empty[ms]);
        if (u >= n_units) break;
        const DecUnit U = dec_load_unit(A, u);
        const int nh = min(kHeadBlock, g - U.hb * kHeadBlock);
        const uint32_t tm_o = tm + C::TM_OT + ms * 16;
        float m[8], l[8];
#pragma unroll
        for (int h = 0; h < 8; ++h) { m[h] = -INFINITY; l[h] = 0.f; }

        for (int b = 0; b < U.nb; ++b) {
            const uint32_t gb = blk_it + b;
            const int st = gb & 1;
            mbar_wait(&B->s_full[st], (gb >> 1) & 1, 322);
            tc_fence_after();
            uint32_t s[8];
            tmem_ld_32x32_x8(tm + C::TM_ST + st * 16, s);
            tc_wait_ld();
            const bool valid = b * kDecBlockKeys + r < U.key_end;
            float x[8];
            bool over = false;
#pragma unroll
            for (int h = 0; h < 8; ++h) {
                x[h] = (valid && h < nh) ? __uint_as_float(s[h]) * scale : -INFINITY;  // select: the score may be NaN
                over |= x[h] > m[h] + 8.f;
            }
            bool raise = true;  // first block of a unit: m is -inf
            if (b > 0) raise = named_bar_or(P.bar_id, 128, over);
            if (raise) {
                float* rb = &B->red[gb & 1][0][0];
#pragma unroll
                for (int h = 0; h < 8; ++h) {
                    const float w = warp_max_f32(x[h]);
                    if (lane == 0) rb[wg_warp * 8 + h] = w;
                }
                named_bar_sync(P.bar_id, 128);
                float alpha[8];
#pragma unroll
                for (int h = 0; h < 8; ++h) {
                    const float mx = fmaxf(fmaxf(rb[h], rb[8 + h]), fmaxf(rb[16 + h], rb[24 + h]));
                    const float mn = fmaxf(m[h], mx);
                    alpha[h] = (h < nh && b > 0) ? fast_exp2(m[h] - mn) : 1.f;
                    l[h] *= alpha[h];
                    m[h] = mn;
                }
                if (b > 0) {  // rescale O^T (this thread: d row r) once PV(b-1) has landed.  The parity wait is
                    // unambiguous although this warp does not observe every phase: s_full(gb) was seen, S^T(gb)
                    // was issued after PV(gb-2) and tcgen05 ops complete in issue order, so at least gb-1 phases
                    // of pv_done are complete; PV(gb) cannot be issued before p_full(gb) is posted below.
                    mbar_wait(&B->pv_done, (gb - 1) & 1, 323);
                    tc_fence_after();
                    uint32_t o[8];
                    tmem_ld_32x32_x8(tm_o, o);
                    tc_wait_ld();
#pragma unroll
                    for (int h = 0; h < 8; ++h) o[h] = __float_as_uint(__uint_as_float(o[h]) * alpha[h]);
                    tmem_st_32x32_x8(tm_o, o);
                    tc_wait_st();
                    tc_fence_before();
                }
            }
#pragma unroll
            for (int h = 0; h < 8; ++h) {
                if (h < nh) {
                    const float p = fast_exp2(x[h] - m[h]);  // invalid key: exp2(-inf) = 0 exactly
                    l[h] += p;
                    const uint32_t a = pt_key + st * C::PT_BYTES + h * 128 + ((pt_chunk ^ h) << 4);
                    asm volatile("st.shared.b16 [%0], %1;" ::"r"(a), "h"(__bfloat16_as_ushort(__float2bfloat16_rn(p))) : "memory");
                }
            }
            fence_proxy_async();
            mbar_arrive(&B->p_full[st]);
        }
        blk_it += U.nb;

        // ---- unit epilogue: thread r owns row r of O^T
        mbar_wait(&B->o_full[ms], par, 325);
        tc_fence_after();
        uint32_t o[8];
        tmem_ld_32x32_x8(tm_o, o);
        tc_wait_ld();
        tc_fence_before();
        mbar_arrive(&B->o_empty[ms]);
#pragma unroll
        for (int h = 0; h < 8; ++h) {
            float v = l[h];
#pragma unroll
            for (int off = 16; off > 0; off >>= 1) v += __shfl_xor_sync(0xffffffffu, v, off);
            if (lane == 0) B->lsum[wg_warp][h] = v;
        }
        named_bar_sync(P.bar_id, 128);
        float lt[8];
#pragma unroll
        for (int h = 0; h < 8; ++h) lt[h] = (B->lsum[0][h] + B->lsum[1][h]) + (B->lsum[2][h] + B->lsum[3][h]);
        const int tok = __ldg(A.b.q_offsets + U.req);
        const int h0 = U.kvh * g + U.hb * kHeadBlock;
        const int nsplit = A.req_info[U.req].z;
        if (nsplit == 1) {
            if (r < D) {
                __nv_bfloat16* ob = reinterpret_cast<__nv_bfloat16*>(A.out) + ((size_t)tok * A.pool.Hq + h0) * D + r;
#pragma unroll
                for (int h = 0; h < 8; ++h)
                    if (h < nh) ob[(size_t)h * D] = __float2bfloat16_rn(__uint_as_float(o[h]) / lt[h]);
            }
            if (A.lse != nullptr && r < nh) {
                float mm = 0.f, ll = 1.f;
#pragma unroll
                for (int h = 0; h < 8; ++h)
                    if (h == r) { mm = m[h]; ll = lt[h]; }
                A.lse[(size_t)tok * A.pool.Hq + h0 + r] = (mm + log2f(ll)) * 0.6931471805599453f;
            }
        } else {
            if (r < D) {
                float* pb = A.part_o + (size_t)u * kHeadBlock * D + r;
#pragma unroll
                for (int h = 0; h < 8; ++h)
                    if (h < nh) pb[h * D] = __uint_as_float(o[h]);
            }
            if (r < nh) {
                float mm = 0.f, ll = 1.f;
#pragma unroll
                for (int h = 0; h < 8; ++h)
                    if (h == r) { mm = m[h]; ll = lt[h]; }
                A.part_ml[(size_t)u * kHeadBlock + r] = make_float2(mm, ll);
            }
        }
        ++unit_it;
    }
}

}  // namespace tropical
