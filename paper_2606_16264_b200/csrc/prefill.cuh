// prefill.cuh -- SURVEY.md 8(a) row A3: prefill tiles on the 5th-gen tensor cores.
//
// Item = (request i, 128-row query tile qt, q head h).  For every 128-key KV tile kt that the
// item's rows can see (keys j <= c_i + t, bottom-right aligned causal mask):
//     S  = Q K^T          tcgen05.mma kind::f16, A = Q (smem, K-major SW128), B = K (smem, K-major
//                         SW128), fp32 accumulator in TMEM (two S slots, alternating per KV tile)
//     P  = exp2(S*scale*log2e - m)   one thread per query row (tcgen05.ld 32x32b), fp32 online
//                         softmax with lazy rescale of O, P written back to TMEM as packed bf16
//                         over the S slot it came from
//     O += P V            tcgen05.mma, A = P (TMEM), B = V (smem, MN-major SW128), fp32 in TMEM
// and finally out = O / l (bf16), lse = ln2 * (m + log2 l).
//
// Warp roles, all persistent over the item queue (tickets popped by the producer and
// handed to the other roles through a 2-deep shared-memory mailbox):
//   producer warps: TMA. Q tile (3-D map, 2 boxes) and, per KV tile, the 8 page-heads of K and of V
//                   (2-D map, one 64-col x 16-row SW128 box per page-head half) into ONE 3-slot ring
//                   filled in the order the MMA warp consumes tiles (K0, K1, V0, K2, V1, ...); one warp
//                   issues the K tiles, a second one the V tiles.  The HND pool makes every box one
//                   contiguous 2 KiB run of HBM/L2.
//   MMA warp      : one elected lane issues S(kt+1) ahead of PV(kt) so the tensor pipe works on
//                   the next scores while the softmax warps work on the current ones.
//   softmax warps : 4 warps, thread r owns query row r (TMEM lane r): no shuffles.
// Unused slots of a request's last page may hold NaN bit patterns: scores are masked by select,
// and the V rows past the last visible key of the last tile are zeroed in shared memory before
// PV is issued (0 * NaN would poison the whole accumulator column).
#pragma once
#include <cuda.h>

#include "common.cuh"
#include "plan.cuh"

namespace tropical {

template <int D>
struct PrefillCfg {
    static constexpr int CB = D / 64;                    // 64-column (128-byte) swizzle halves per row
    static constexpr int HALF_BYTES = kKvTile * 128;     // one half of a 128-row tile: 16 KiB
    static constexpr int TILE_BYTES = CB * HALF_BYTES;   // Q tile / K tile / V tile
    static constexpr int PAGE_BOX = kPageSize * 128;     // one TMA box: 16 rows x 128 B
    static constexpr int KV_SLOTS = 3;                   // one ring for K and V tiles, filled in consumption order
    static constexpr int SMEM_TILES = TILE_BYTES * (1 + KV_SLOTS);
    // TMEM columns: S slot 0 at 0, S slot 1 at 128, O at 256
    static constexpr uint32_t TM_S = 0, TM_O = 256, TM_COLS = 512;
};

// mbarriers of the prefill role set
struct PrefillBars {
    uint64_t item_full[2], item_empty[2];
    uint64_t q_full, q_empty;
    uint64_t kv_full[3], kv_empty[3];
    uint64_t s_full[2], p_full[2];
    uint64_t pv_done, o_empty;
    int mailbox[2];
    uint32_t tmem_base;
};

struct PrefillArgs {
    PoolDesc pool;
    BatchDesc b;
    uint16_t* out;
    float* lse;
    float scale_log2;
    const int* hdr;
    int* ticket;
    const int2* items;
};

struct PrefillItem {
    int req, qt, h, hk;
    int c, ql, tok0;   // context length, chunk length, first packed row of the request
    int l_tile;        // keys visible to the last row of the tile: c + min(ql, (qt+1)*128)
    int n_kt;          // KV tiles
};

__device__ __forceinline__ PrefillItem load_item(const PrefillArgs& A, int id) {
    PrefillItem it;
    const int2 v = A.items[id];
    it.req = v.x;
    it.qt = v.y >> 16;
    it.h = v.y & 0xffff;
    it.hk = it.h / (A.pool.Hq / A.pool.Hkv);
    it.c = __ldg(A.b.ctx_lens + it.req);
    it.ql = __ldg(A.b.q_lens + it.req);
    it.tok0 = __ldg(A.b.q_offsets + it.req);
    it.l_tile = it.c + min(it.ql, (it.qt + 1) * kQTile);
    it.n_kt = (it.l_tile + kKvTile - 1) / kKvTile;
    return it;
}

// the same item with every field broadcast from lane 0 (warp-uniform for the compiler: see uni())
__device__ __forceinline__ PrefillItem load_item_uniform(const PrefillArgs& A, int id) {
    PrefillItem it = load_item(A, id);
    it.req = uni(it.req); it.qt = uni(it.qt); it.h = uni(it.h); it.hk = uni(it.hk);
    it.c = uni(it.c); it.ql = uni(it.ql); it.tok0 = uni(it.tok0); it.l_tile = uni(it.l_tile); it.n_kt = uni(it.n_kt);
    return it;
}

__device__ __forceinline__ void prefill_init_bars(PrefillBars* B) {
    for (int i = 0; i < 2; ++i) {
        mbar_init(&B->item_full[i], 1);
        mbar_init(&B->item_empty[i], 6);  // lane 0 of: MMA warp, V producer warp, each softmax warp
        mbar_init(&B->s_full[i], 1);
        mbar_init(&B->p_full[i], 128);
    }
    for (int i = 0; i < 3; ++i) {
        mbar_init(&B->kv_full[i], 1);
        mbar_init(&B->kv_empty[i], 1);
    }
    mbar_init(&B->q_full, 1);
    mbar_init(&B->q_empty, 1);
    mbar_init(&B->pv_done, 1);
    mbar_init(&B->o_empty, 128);
}

// ------------------------------------------------------------------------------------------------
// producer warps.  Ring entries follow the MMA warp's consumption order K0, K1, V0, K2, V1, ..., K(n-1),
// V(n-2), V(n-1); both producers walk that sequence and each fills the entries of its own kind, so K and V
// tiles are issued in parallel (a 128-key tile is 16 TMA boxes: one warp issuing all 32 of an iteration was
// the prefill role's bottleneck).

// One KV tile (8 page-heads) of item `it` into the cursor's slot: lane -> (page p, half cb), one box per lane.
template <int D>
__device__ __forceinline__ void prefill_load_tile(const PrefillArgs& A, PrefillBars* B, uint8_t* ring,
                                                  const PrefillItem& it, const int* pt, int n_pages, int kt,
                                                  const CUtensorMap* tm, const RingCursor& cur, int lane) {
    using C = PrefillCfg<D>;
    const int np = min(8, n_pages - kt * 8);
    const int p = lane / C::CB, cb = lane % C::CB;
    const bool act = p < np && lane < 8 * C::CB;
    const int page = act ? __ldg(pt + kt * 8 + p) : 0;
    const int r0 = (page * A.pool.Hkv + it.hk) * kPageSize;
    const uint32_t off = cb * C::HALF_BYTES + p * C::PAGE_BOX;
    mbar_wait(&B->kv_empty[cur.slot], cur.phase ^ 1, 103);
    if (lane == 0) mbar_arrive_expect_tx(&B->kv_full[cur.slot], np * C::CB * C::PAGE_BOX);
    __syncwarp();
    if (act) tma_load_2d(ring + cur.slot * C::TILE_BYTES + off, tm, cb * 64, r0, &B->kv_full[cur.slot]);
}

// warp A: pops the item tickets, loads Q and the K tiles
template <int D>
__device__ __forceinline__ void prefill_producer(const PrefillArgs& A, PrefillBars* B, uint8_t* tiles,
                                                 const CUtensorMap* tm_q, const CUtensorMap* tm_k) {
    using C = PrefillCfg<D>;
    const int lane = threadIdx.x & 31;
    const int n_items = uni(A.hdr[HDR_N_ITEMS]);
    uint8_t* q_s = tiles;
    uint8_t* ring = tiles + C::TILE_BYTES;
    uint32_t item_it = 0;
    RingCursor cur = {0, 0};
    for (;;) {
        const int ms = item_it & 1;
        mbar_wait(&B->item_empty[ms], ((item_it >> 1) & 1) ^ 1, 101);
        int id = 0;
        if (lane == 0) {
            id = atomicAdd(A.ticket, 1);
            B->mailbox[ms] = id;
            mbar_arrive(&B->item_full[ms]);
        }
        id = __shfl_sync(0xffffffffu, id, 0);
        if (id >= n_items) break;
        const PrefillItem it = load_item_uniform(A, id);
        const int* pt = A.b.page_table + (size_t)it.req * A.b.stride;

        mbar_wait(&B->q_empty, (item_it & 1) ^ 1, 102);
        if (elect_one()) {
            mbar_arrive_expect_tx(&B->q_full, C::TILE_BYTES);
#pragma unroll
            for (int cb = 0; cb < C::CB; ++cb)
                tma_load_3d(q_s + cb * C::HALF_BYTES, tm_q, cb * 64, it.h, it.tok0 + it.qt * kQTile, &B->q_full);
        }
        const int n_pages = (it.l_tile + kPageSize - 1) / kPageSize;
        for (int s = 0; s <= it.n_kt; ++s) {  // ring order K0, K1, V0, K2, V1, ...: step s = K(s), then V(s-1)
            if (s < it.n_kt) {
                prefill_load_tile<D>(A, B, ring, it, pt, n_pages, s, tm_k, cur, lane);
                cur.advance(C::KV_SLOTS);
            }
            if (s > 0) cur.advance(C::KV_SLOTS);  // V(s-1): the other producer's entry
        }
        ++item_it;
    }
}

// warp B: the V tiles of the same item sequence (item ids come through the mailbox)
template <int D>
__device__ __forceinline__ void prefill_producer_v(const PrefillArgs& A, PrefillBars* B, uint8_t* tiles,
                                                   const CUtensorMap* tm_v) {
    using C = PrefillCfg<D>;
    const int lane = threadIdx.x & 31;
    const int n_items = uni(A.hdr[HDR_N_ITEMS]);
    uint8_t* ring = tiles + C::TILE_BYTES;
    uint32_t item_it = 0;
    RingCursor cur = {0, 0};
    for (;;) {
        const int ms = item_it & 1;
        mbar_wait(&B->item_full[ms], (item_it >> 1) & 1, 115);
        const int id = uni(B->mailbox[ms]);
        __syncwarp();
        if (lane == 0) mbar_arrive(&B->item_empty[ms]);
        if (id >= n_items) break;
        const PrefillItem it = load_item_uniform(A, id);
        const int* pt = A.b.page_table + (size_t)it.req * A.b.stride;
        const int n_pages = (it.l_tile + kPageSize - 1) / kPageSize;
        for (int s = 0; s <= it.n_kt; ++s) {
            if (s < it.n_kt) cur.advance(C::KV_SLOTS);  // K(s): the other producer's entry
            if (s > 0) {
                prefill_load_tile<D>(A, B, ring, it, pt, n_pages, s - 1, tm_v, cur, lane);
                cur.advance(C::KV_SLOTS);
            }
        }
        ++item_it;
    }
}

// ------------------------------------------------------------------------------------------------
// MMA warp.  All 32 lanes run the (warp-uniform) control flow; one elected lane issues the tcgen05 instructions.
template <int D>
__device__ __forceinline__ void prefill_mma(const PrefillArgs& A, PrefillBars* B, uint8_t* tiles) {
    using C = PrefillCfg<D>;
    const int lane = threadIdx.x & 31;
    const int n_items = uni(A.hdr[HDR_N_ITEMS]);
    const uint32_t q_a = uni(smem_u32(tiles));
    const uint32_t ring_a = q_a + C::TILE_BYTES;
    const uint32_t tm = uni(B->tmem_base);
    constexpr uint32_t IDESC_S = make_idesc_bf16(128, 128, false);
    constexpr uint32_t IDESC_O = make_idesc_bf16(128, D, true);
    uint32_t item_it = 0, kv_it = 0;
    int slot = 0;
    uint32_t phase = 0;
    auto advance = [&]() {
        if (++slot == C::KV_SLOTS) { slot = 0; phase ^= 1; }
    };

    for (;;) {
        const int ms = item_it & 1;
        mbar_wait(&B->item_full[ms], (item_it >> 1) & 1, 105, item_it);
        const int id = uni(B->mailbox[ms]);
        __syncwarp();
        if (lane == 0) mbar_arrive(&B->item_empty[ms]);
        if (id >= n_items) break;
        const PrefillItem it = load_item_uniform(A, id);

        mbar_wait(&B->q_full, item_it & 1, 106, item_it);
        // step s issues S(s) (ahead) and then PV(s - 1): the tensor pipe works on the next scores while the softmax
        // warps work on the current ones; one copy of each issue sequence (instruction-cache footprint)
        for (int s = 0; s <= it.n_kt; ++s) {
            if (s < it.n_kt) {  // S(g) = Q K^T into S slot g & 1; consumes the next ring tile (a K tile)
                const uint32_t g = kv_it + s;
                const int st = g & 1;
                mbar_wait(&B->kv_full[slot], phase, 104, item_it * 100000 + g * 100 + slot);
                tc_fence_after();
                const uint32_t k_a = ring_a + slot * C::TILE_BYTES;
                if (elect_one()) {
#pragma unroll
                    for (int cb = 0; cb < C::CB; ++cb)
#pragma unroll
                        for (int k4 = 0; k4 < 4; ++k4) {
                            const uint32_t o = cb * C::HALF_BYTES + k4 * 32;
                            tc_mma_ss(tm + C::TM_S + st * 128, make_smem_desc_sw128(q_a + o, 0, 1024),
                                      make_smem_desc_sw128(k_a + o, 0, 1024), IDESC_S, (cb | k4) != 0);
                        }
                    tc_commit(&B->s_full[st]);
                    tc_commit(&B->kv_empty[slot]);
                    if (s + 1 == it.n_kt) tc_commit(&B->q_empty);  // every S MMA of this item has been issued
                }
                __syncwarp();
                advance();
            }
            if (s == 0) continue;
            const int kt = s - 1;
            const uint32_t g = kv_it + kt;
            const int st = g & 1;
            mbar_wait(&B->kv_full[slot], phase, 107, item_it * 100000 + kt * 1000 + slot * 100 + it.n_kt);  // the next ring tile is V(kt)
            const uint32_t v_a = ring_a + slot * C::TILE_BYTES;
            if (kt + 1 == it.n_kt) {  // zero V rows past the last visible key (stale or poisoned smem)
                const int nvalid = it.l_tile - kt * kKvTile;
                const int nz = (kKvTile - nvalid) * 8 * C::CB;
                for (int idx = lane; idx < nz; idx += 32) {
                    const int r = nvalid + idx / (8 * C::CB), rem = idx % (8 * C::CB);
                    const uint32_t a = v_a + (rem >> 3) * C::HALF_BYTES + r * 128 + ((rem & 7) << 4);
                    asm volatile("st.shared.v4.b32 [%0], {%1,%1,%1,%1};" ::"r"(a), "r"(0u) : "memory");
                }
                fence_proxy_async();
                __syncwarp();
            }
            if (kt == 0) mbar_wait(&B->o_empty, (item_it & 1) ^ 1, 108, item_it * 100000 + id);  // previous item's epilogue has read O
            mbar_wait(&B->p_full[st], (g >> 1) & 1, 109, item_it * 100000 + kt * 1000 + it.n_kt);
            tc_fence_after();
            if (elect_one()) {
#pragma unroll
                for (int ks = 0; ks < 8; ++ks)  // 16 keys per MMA
                    tc_mma_ts(tm + C::TM_O, tm + C::TM_S + st * 128 + ks * 8,
                              make_smem_desc_sw128(v_a + ks * 2048, C::HALF_BYTES, 1024), IDESC_O, (kt | ks) != 0);
                tc_commit(&B->kv_empty[slot]);
                tc_commit(&B->pv_done);
            }
            __syncwarp();
            advance();
        }
        kv_it += it.n_kt;
        ++item_it;
    }
}

// ------------------------------------------------------------------------------------------------
// softmax warps (4 warps, 128 threads: thread r <-> query row r <-> TMEM lane r)
__device__ __forceinline__ float max4(float a, float b, float c, float d) { return fmaxf(fmaxf(a, b), fmaxf(c, d)); }

template <int D>
__device__ __forceinline__ void prefill_softmax(const PrefillArgs& A, PrefillBars* B, int wg_warp) {
    using C = PrefillCfg<D>;
    const int lane = threadIdx.x & 31;
    const int r = wg_warp * 32 + lane;
    const int n_items = A.hdr[HDR_N_ITEMS];
    const uint32_t tm = B->tmem_base + ((uint32_t)(wg_warp * 32) << 16);
    const float scale = A.scale_log2;
    uint32_t item_it = 0, kv_it = 0;

    for (;;) {
        const int ms = item_it & 1;
        mbar_wait(&B->item_full[ms], (item_it >> 1) & 1, 110, item_it);
        const int id = B->mailbox[ms];
        __syncwarp();
        if (lane == 0) mbar_arrive(&B->item_empty[ms]);
        if (id >= n_items) break;
        const PrefillItem it = load_item(A, id);
        const int t = it.qt * kQTile + r;
        const int limit = it.c + min(t, it.ql - 1);  // last visible key of this row (rows past the chunk mirror its last row)
        float m_used = -INFINITY, l = 0.f;  // the first chunk of the item raises m_used from -inf (grow_fix)

        for (int kt = 0; kt < it.n_kt; ++kt) {
            const uint32_t g = kv_it + kt;
            const int st = g & 1;
            mbar_wait(&B->s_full[st], (g >> 1) & 1, 111, item_it * 100000 + kt * 1000 + it.n_kt);
            tc_fence_after();
            // ONE pass over the tile in 32-column chunks, the TMEM load of the next chunk in flight while the current
            // one is exponentiated (two register buffers).  P = exp2(s*scale - m_used) is written with the running
            // maximum m_used of the PREVIOUS chunks; a chunk whose maximum exceeds m_used by more than 2^8 (rare after
            // the first chunk of an item) takes grow_fix(): raise m_used, rescale O, l and the P chunks already written.
            // Code size matters: the roles of an SM share a 32 KiB instruction cache (profiles/r1c_c5.md).
            const uint32_t s_col = tm + C::TM_S + st * 128;
            const int n_vis = limit - kt * kKvTile + 1;  // visible columns of this tile for this row
            const bool masked = __any_sync(0xffffffffu, n_vis < kKvTile);
            float sum0 = 0.f, sum1 = 0.f;

            auto grow_fix = [&](int c4, float cm) {  // cold path
                const float m_new = fmaxf(m_used, cm * scale);
                const float alpha = m_new == -INFINITY ? 1.f : fast_exp2(m_used - m_new);  // rows that do not grow: 1; first chunk of an item: 0
                if (kt > 0) {
                    mbar_wait(&B->pv_done, (g - 1) & 1, 112, item_it * 100000 + kt * 1000 + it.n_kt);  // O holds PV(g-1)
                    tc_fence_after();
#pragma unroll 1
                    for (int c = 0; c < D / 32; ++c) {
                        uint32_t o[32];
                        tmem_ld_32x32(tm + C::TM_O + c * 32, o);
                        tc_wait_ld();
#pragma unroll
                        for (int j = 0; j < 32; ++j) o[j] = __float_as_uint(__uint_as_float(o[j]) * alpha);
                        tmem_st_32x32(tm + C::TM_O + c * 32, o);
                    }
                }
#pragma unroll 1
                for (int c = 0; c < c4; ++c) {  // P chunks of this tile written with the old maximum
                    uint32_t pk[16];
                    tmem_ld_32x32_x16(s_col + c * 16, pk);
                    tc_wait_ld();
#pragma unroll
                    for (int j = 0; j < 16; ++j) pk[j] = pack_bf16x2(bf16_lo(pk[j]) * alpha, bf16_hi(pk[j]) * alpha);
                    tmem_st_32x32_x16(s_col + c * 16, pk);
                }
                l *= alpha;
                sum0 *= alpha;
                sum1 *= alpha;
                m_used = m_new;
            };
            auto process = [&](uint32_t (&s)[32], int c4) {
                if (masked) {
#pragma unroll
                    for (int j = 0; j < 32; ++j)
                        if (c4 * 32 + j >= n_vis) s[j] = 0xff800000u;  // -inf, by select: the score may be NaN
                }
                float cm = -INFINITY;
#pragma unroll
                for (int j = 0; j < 32; j += 4)
                    cm = fmaxf(cm, max4(__uint_as_float(s[j]), __uint_as_float(s[j + 1]), __uint_as_float(s[j + 2]),
                                        __uint_as_float(s[j + 3])));
                if (__any_sync(0xffffffffu, cm * scale > m_used + 8.f)) grow_fix(c4, cm);  // lazy: P stays <= 2^8
                uint32_t pk[16];
#pragma unroll
                for (int j = 0; j < 32; j += 2) {
                    const float p0 = fast_exp2(fmaf(__uint_as_float(s[j]), scale, -m_used));
                    const float p1 = fast_exp2(fmaf(__uint_as_float(s[j + 1]), scale, -m_used));
                    sum0 += p0;
                    sum1 += p1;
                    pk[j >> 1] = pack_bf16x2(p0, p1);
                }
                // P columns [16 c4, 16 c4 + 16) overwrite S columns this thread has already loaded
                tmem_st_32x32_x16(s_col + c4 * 16, pk);
            };
            {
                uint32_t sa[32], sb[32];
                tmem_ld_32x32(s_col, sa);
                tc_wait_ld();
#pragma unroll 1
                for (int h = 0; h < 2; ++h) {
                    tmem_ld_32x32(s_col + (2 * h + 1) * 32, sb);
                    process(sa, 2 * h);
                    tc_wait_ld();
                    if (h == 0) tmem_ld_32x32(s_col + 64, sa);
                    process(sb, 2 * h + 1);
                    if (h == 0) tc_wait_ld();
                }
            }
            l += sum0 + sum1;
            tc_wait_st();
            tc_fence_before();
            // Observe EVERY phase of pv_done in order (a parity wait is only safe when the waiter is at most one
            // phase behind): PV(g-1) here -- long complete, and PV(g) cannot start before P(g) is posted below --
            // and PV(last) in the epilogue.  Skipping phases let a short item's epilogue pass its wait on a
            // stale phase while the MMA warp was still waiting for that item's first V tile.
            if (kt > 0) mbar_wait(&B->pv_done, (g - 1) & 1, 114, item_it * 100000 + kt * 1000 + it.n_kt);
            mbar_arrive(&B->p_full[st]);
        }
        kv_it += it.n_kt;

        // epilogue: out = O / l
        mbar_wait(&B->pv_done, (kv_it - 1) & 1, 113, item_it * 100000 + id);
        tc_fence_after();
        const float inv = 1.f / l;
        const bool valid = t < it.ql;
        uint16_t* orow = A.out + ((size_t)(it.tok0 + t) * A.pool.Hq + it.h) * D;
#pragma unroll 1
        for (int c4 = 0; c4 < D / 32; ++c4) {
            uint32_t o[32];
            tmem_ld_32x32(tm + C::TM_O + c4 * 32, o);
            tc_wait_ld();
            if (valid) {
#pragma unroll
                for (int j = 0; j < 32; j += 8) {
                    uint4 w;
                    w.x = pack_bf16x2(__uint_as_float(o[j]) * inv, __uint_as_float(o[j + 1]) * inv);
                    w.y = pack_bf16x2(__uint_as_float(o[j + 2]) * inv, __uint_as_float(o[j + 3]) * inv);
                    w.z = pack_bf16x2(__uint_as_float(o[j + 4]) * inv, __uint_as_float(o[j + 5]) * inv);
                    w.w = pack_bf16x2(__uint_as_float(o[j + 6]) * inv, __uint_as_float(o[j + 7]) * inv);
                    *reinterpret_cast<uint4*>(orow + c4 * 32 + j) = w;
                }
            }
        }
        tc_fence_before();
        mbar_arrive(&B->o_empty);
        if (valid && A.lse != nullptr)
            A.lse[(size_t)(it.tok0 + t) * A.pool.Hq + it.h] = (m_used + log2f(l)) * 0.6931471805599453f;
        ++item_it;
    }
}

}  // namespace tropical
