// prefill.cuh -- SURVEY.md 8(a) row A3: prefill tiles on the 5th-gen tensor cores.
//
// Item = (request i, 128-row query tile qt, q head h [, q head h+1 of the same kv group]).  An item carries ONE or
// TWO query tiles ("A" and "B"): under GQA the heads of a kv group read the same K/V, so two of them share every
// K/V tile that TMA brings into shared memory -- half the L2 -> SM traffic per FLOP (the fused step is bound by L2
// throughput, profiles/r1c_c5.md) -- and the tensor pipe works on one tile while the other is exponentiated.  For every 128-key KV tile kt the item's rows can see (keys j <= c_i + t):
//     S_w  = Q_w K^T          tcgen05.mma kind::f16, A = Q_w (smem, K-major SW128), B = K (smem, K-major SW128),
//                             fp32 accumulator in TMEM (one S slot per query tile w)
//     P_w  = exp2(S_w*scale*log2e - m)   one thread per query row (tcgen05.ld 32x32b), fp32 online softmax with lazy
//                             rescale of O_w, P_w written back to TMEM as packed bf16 over S_w
//     O_w += P_w V            tcgen05.mma, A = P_w (TMEM), B = V (smem, MN-major SW128), fp32 in TMEM
// and finally out = O_w / l (bf16), lse = ln2 * (m + log2 l).
//
// Warp roles, all persistent over the item queue (tickets popped by the K producer and handed to the other roles
// through a 2-deep shared-memory mailbox):
//   producer warps: TMA.  Q tiles (3-D map, 2 boxes each) and, per KV tile, the 8 page-heads of K and of V (2-D map,
//                   one 64-col x 16-row SW128 box per page-head half) into ONE 3-slot ring filled in the order the
//                   MMA warp consumes tiles (K0, V0, K1, V1, ...); one warp issues the K tiles, a second one the V
//                   tiles.  The HND pool makes every box one contiguous 2 KiB run of HBM/L2.
//   MMA warp      : one elected lane issues, per KV tile, {PV_A(kt), S_A(kt+1)} when P_A(kt) is posted and then
//                   {PV_B(kt), S_B(kt+1)} when P_B(kt) is; all operands of the issue are warp-uniform (common.cuh uni()).
//   softmax WG    : 4 warps, thread r owns query row r (TMEM lane r) of BOTH query tiles: no shuffles.  It alternates
//                   between the tiles, so the tensor pipe runs PV_A(kt), S_A(kt+1) while it exponentiates S_B(kt).
//                   (Two warpgroups, one per tile, were measured: no faster -- each waits for its own S -- and they
//                   cost four warps that the decode role needs.)
// Unused slots of a request's last page may hold NaN bit patterns: scores are masked by select, and the V rows
// past the last visible key of the last tile are zeroed in shared memory before PV is issued (0 * NaN would
// poison the whole accumulator column).
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
    static constexpr int Q_TILES = 2;                    // query tiles per item (A, B)
    static constexpr int KV_SLOTS = 2;                   // K tiles and V tiles alternate (K0, V0, K1, V1, ...): a K slot and a V slot
    static constexpr int SMEM_TILES = TILE_BYTES * (Q_TILES + KV_SLOTS);
    // TMEM columns: S_A at 0, S_B at 128, O_A at 256, O_B at 384 (P_w aliases the first 64 columns of S_w)
    static constexpr uint32_t TM_S = 0, TM_O = 256, TM_COLS = 512;
};

// mbarriers of the prefill role set ([w] = per query tile)
struct PrefillBars {
    uint64_t item_full[2], item_empty[2];
    uint64_t q_full, q_empty;
    uint64_t kv_full[2], kv_empty[2];
    uint64_t s_full[2], p_full[2];
    uint64_t pv_done[2], o_empty[2];
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

// Tensor maps of one of K / V for the prefill producers: the pool as 16-slot boxes (one page-head half) and as single
// slots, and this step's rows [T][Hkv][D] as 16-token and single-token boxes (fused step only).
struct KvMaps {
    const CUtensorMap* pool16;
    const CUtensorMap* pool1;
    const CUtensorMap* new16;
    const CUtensorMap* new1;
};

struct PrefillItem {
    int req, qt, h, hk, nt;   // nt query tiles.  rows == 0: heads h .. h + nt - 1 (same kv head hk) at row tile qt;
    int rows;                 // rows == 1 (two-warpgroup variant only): row tiles qt .. qt + nt - 1 of head h
    int c, ql, tok0;          // context length, chunk length, first packed row of the request
    int l_tile;               // keys visible to the last row of the item's LAST tile: c + min(ql, (qt_last+1)*128)
    int n_kt;                 // KV tiles of the last tile (the item's K/V extent)
    int n_kt0;                // KV tiles of tile 0: n_kt, or one fewer when it is the earlier row tile of a pair
    __device__ __forceinline__ int head(int w) const { return h + (rows ? 0 : w); }
    __device__ __forceinline__ int row0(int w) const { return (qt + (rows ? w : 0)) * kQTile; }  // first row of tile w in the chunk
    __device__ __forceinline__ int kv_tiles(int w) const { return w == 0 ? n_kt0 : n_kt; }
};

// ROWS = false (the plain step kernel): row-pair items do not occur, `rows` folds to 0 and n_kt0 to n_kt at compile time
template <bool ROWS>
__device__ __forceinline__ PrefillItem load_item(const PrefillArgs& A, int id) {
    PrefillItem it;
    const int2 v = A.items[id];
    it.req = v.x;
    it.qt = v.y >> 16;
    it.nt = ((v.y >> 15) & 1) + 1;
    it.rows = ROWS ? (v.y >> 14) & 1 : 0;
    it.h = v.y & 0x3fff;
    it.hk = it.h / (A.pool.Hq / A.pool.Hkv);
    it.c = __ldg(A.b.ctx_lens + it.req);
    it.ql = __ldg(A.b.q_lens + it.req);
    it.tok0 = __ldg(A.b.q_offsets + it.req);
    const int qt_last = it.qt + (it.rows ? it.nt - 1 : 0);
    it.l_tile = it.c + min(it.ql, (qt_last + 1) * kQTile);
    it.n_kt = (it.l_tile + kKvTile - 1) / kKvTile;
    it.n_kt0 = ROWS ? (it.c + min(it.ql, (it.qt + 1) * kQTile) + kKvTile - 1) / kKvTile : it.n_kt;
    return it;
}

// the same item with every field broadcast from lane 0 (warp-uniform for the compiler: see uni())
template <bool ROWS>
__device__ __forceinline__ PrefillItem load_item_uniform(const PrefillArgs& A, int id) {
    PrefillItem it = load_item<ROWS>(A, id);
    it.req = uni(it.req); it.qt = uni(it.qt); it.h = uni(it.h); it.hk = uni(it.hk); it.nt = uni(it.nt);
    it.c = uni(it.c); it.ql = uni(it.ql); it.tok0 = uni(it.tok0); it.l_tile = uni(it.l_tile); it.n_kt = uni(it.n_kt);
    if (ROWS) { it.rows = uni(it.rows); it.n_kt0 = uni(it.n_kt0); } else { it.n_kt0 = it.n_kt; }
    return it;
}

__device__ __forceinline__ void prefill_init_bars(PrefillBars* B, int softmax_warps) {
    for (int i = 0; i < 2; ++i) {
        mbar_init(&B->item_full[i], 1);
        mbar_init(&B->item_empty[i], 2 + softmax_warps);  // lane 0 of: MMA warp, V producer warp, each softmax warp
        mbar_init(&B->s_full[i], 1);
        mbar_init(&B->p_full[i], 128);
        mbar_init(&B->pv_done[i], 1);
        mbar_init(&B->o_empty[i], 128);
        mbar_init(&B->kv_full[i], 1);
        mbar_init(&B->kv_empty[i], 1);
    }
    mbar_init(&B->q_full, 1);
    mbar_init(&B->q_empty, 1);
}

// ------------------------------------------------------------------------------------------------
// producer warps.  Ring entries follow the MMA warp's consumption order K0, V0, K1, V1, ...; both producers walk
// that sequence and each fills the entries of its own kind, so K and V tiles are issued in parallel (a 128-key
// tile is 16 TMA boxes).

// One KV tile (8 page-heads) of item `it` into the cursor's slot: lane -> (page p, half cb), one box per lane.
// Fused step: keys below the request's prior context c come from the pool, keys from c on are this step's rows and
// come from k_new / v_new (token row tok0 + key - c); the one page that holds both (c not a multiple of 16) is loaded
// slot by slot.  The bytes per tile are the same in every case.
template <int D, bool FUSED>
__device__ __forceinline__ void prefill_load_tile(const PrefillArgs& A, PrefillBars* B, uint8_t* ring,
                                                  const PrefillItem& it, const int* pt, int n_pages, int kt,
                                                  const KvMaps& tm, const RingCursor& cur, int lane) {
    using C = PrefillCfg<D>;
    const int np = min(8, n_pages - kt * 8);
    const int p = lane / C::CB, cb = lane % C::CB;
#ifdef TROPICAL_WHATIF_HALF_KV
    const bool act = p < np && lane < 8 * C::CB && (np < 8 || p < 4);
#else
    const bool act = p < np && lane < 8 * C::CB;
#endif
    const int page = act ? __ldg(pt + kt * 8 + p) : 0;
    const int r0 = (page * A.pool.Hkv + it.hk) * kPageSize;
    const uint32_t off = cb * C::HALF_BYTES + p * C::PAGE_BOX;
    mbar_wait(&B->kv_empty[cur.slot], cur.phase ^ 1, 103);
#ifdef TROPICAL_WHATIF_HALF_KV
    if (lane == 0) mbar_arrive_expect_tx(&B->kv_full[cur.slot], (np < 8 ? np : 4) * C::CB * C::PAGE_BOX);
#else
    if (lane == 0) mbar_arrive_expect_tx(&B->kv_full[cur.slot], np * C::CB * C::PAGE_BOX);
#endif
    __syncwarp();
    if (act) {
        uint8_t* dst = ring + cur.slot * C::TILE_BYTES + off;
        const int key0 = (kt * 8 + p) * kPageSize;
        if (!FUSED || key0 + kPageSize <= it.c) {
            tma_load_2d(dst, tm.pool16, cb * 64, r0, &B->kv_full[cur.slot]);
        } else if (key0 >= it.c) {
            tma_load_3d(dst, tm.new16, cb * 64, it.hk, it.tok0 + key0 - it.c, &B->kv_full[cur.slot]);
        } else {
#pragma unroll 1
            for (int r = 0; r < kPageSize; ++r) {  // rare (one page per chunk whose context is not a multiple of 16): keep it small
                if (key0 + r < it.c) tma_load_2d(dst + r * 128, tm.pool1, cb * 64, r0 + r, &B->kv_full[cur.slot]);
                else tma_load_3d(dst + r * 128, tm.new1, cb * 64, it.hk, it.tok0 + key0 + r - it.c, &B->kv_full[cur.slot]);
            }
        }
    }
}

// KIND 0: pops the item tickets, loads the Q tiles and the K tiles.  KIND 1: the V tiles of the same item sequence
// (item ids come through the mailbox).
template <int D, int KIND, bool FUSED>
__device__ __forceinline__ void prefill_producer(const PrefillArgs& A, PrefillBars* B, uint8_t* tiles,
                                                 const CUtensorMap* tm_q, const KvMaps tm_kv) {
    using C = PrefillCfg<D>;
    const int lane = threadIdx.x & 31;
    const int n_items = uni(A.hdr[HDR_N_ITEMS]);
    uint8_t* q_s = tiles;
    uint8_t* ring = tiles + C::Q_TILES * C::TILE_BYTES;
    uint32_t item_it = 0;
    RingCursor cur = {0, 0};
    for (;;) {
        const int ms = item_it & 1;
        int id = 0;
        if (KIND == 0) {
            mbar_wait(&B->item_empty[ms], ((item_it >> 1) & 1) ^ 1, 101);
            if (lane == 0) {
                id = atomicAdd(A.ticket, 1);
                B->mailbox[ms] = id;
                mbar_arrive(&B->item_full[ms]);
            }
            id = __shfl_sync(0xffffffffu, id, 0);
        } else {
            mbar_wait(&B->item_full[ms], (item_it >> 1) & 1, 115);
            id = uni(B->mailbox[ms]);
            __syncwarp();
            if (lane == 0) mbar_arrive(&B->item_empty[ms]);
        }
        if (id >= n_items) break;
        const PrefillItem it = load_item_uniform<FUSED>(A, id);
        const int* pt = A.b.page_table + (size_t)it.req * A.b.stride;
        if (KIND == 0) {
            mbar_wait(&B->q_empty, (item_it & 1) ^ 1, 102);
            if (elect_one()) {
                mbar_arrive_expect_tx(&B->q_full, it.nt * C::TILE_BYTES);
                for (int w = 0; w < it.nt; ++w)
#pragma unroll
                    for (int cb = 0; cb < C::CB; ++cb)
                        tma_load_3d(q_s + w * C::TILE_BYTES + cb * C::HALF_BYTES, tm_q, cb * 64, it.head(w),
                                    it.tok0 + it.row0(w), &B->q_full);
            }
        }
        const int n_pages = (it.l_tile + kPageSize - 1) / kPageSize;
        for (int kt = 0; kt < it.n_kt; ++kt) {  // ring entries 2 kt (K) and 2 kt + 1 (V)
            if (KIND == 0) prefill_load_tile<D, FUSED>(A, B, ring, it, pt, n_pages, kt, tm_kv, cur, lane);
            cur.advance(C::KV_SLOTS);
            if (KIND == 1) prefill_load_tile<D, FUSED>(A, B, ring, it, pt, n_pages, kt, tm_kv, cur, lane);
            cur.advance(C::KV_SLOTS);
        }
        ++item_it;
    }
}

// ------------------------------------------------------------------------------------------------
// MMA warp.  All 32 lanes run the (warp-uniform) control flow; one elected lane issues the tcgen05 instructions.
// Per KV tile kt and query tile w: PV_w(kt) as soon as P_w(kt) is posted, then S_w(kt+1) into the S slot PV_w(kt) has
// just read -- so while warpgroup A exponentiates S_A(kt+1) the tensor pipe runs PV_B(kt) and S_B(kt+1).
template <int D, bool ROWS>
__device__ __forceinline__ void prefill_mma(const PrefillArgs& A, PrefillBars* B, uint8_t* tiles) {
    using C = PrefillCfg<D>;
    const int lane = threadIdx.x & 31;
    const int n_items = uni(A.hdr[HDR_N_ITEMS]);
    const uint32_t q_a = uni(smem_u32(tiles));
    const uint32_t ring_a = q_a + C::Q_TILES * C::TILE_BYTES;
    const uint32_t tm = uni(B->tmem_base);
#ifdef TROPICAL_WHATIF_NO_MMA
    constexpr uint32_t IDESC_S = make_idesc_bf16(128, 16, false);
    constexpr uint32_t IDESC_O = make_idesc_bf16(128, 16, true);
#else
    constexpr uint32_t IDESC_S = make_idesc_bf16(128, 128, false);
    constexpr uint32_t IDESC_O = make_idesc_bf16(128, D, true);
#endif
    uint32_t item_it = 0;
    uint32_t g0 = 0, g1 = 0;      // S / P / PV iterations of query tile A, B so far (barrier phases)
    uint32_t cnt0 = 0, cnt1 = 0;  // items that carried tile A, B so far (o_empty phases)
    RingCursor cur = {0, 0};

    auto issue_s = [&](int w, int slot) {  // S_w = Q_w K^T, K tile in ring slot `slot`
        const uint32_t k_a = ring_a + slot * C::TILE_BYTES;
        const uint32_t qw_a = q_a + w * C::TILE_BYTES;
        if (elect_one()) {
#pragma unroll
            for (int cb = 0; cb < C::CB; ++cb)
#pragma unroll
                for (int k4 = 0; k4 < 4; ++k4) {
                    const uint32_t o = cb * C::HALF_BYTES + k4 * 32;
                    tc_mma_ss(tm + C::TM_S + w * 128, make_smem_desc_sw128(qw_a + o, 0, 1024),
                              make_smem_desc_sw128(k_a + o, 0, 1024), IDESC_S, (cb | k4) != 0);
                }
            tc_commit(&B->s_full[w]);
        }
        __syncwarp();
    };

    for (;;) {
        const int ms = item_it & 1;
        mbar_wait(&B->item_full[ms], (item_it >> 1) & 1, 105, item_it);
        const int id = uni(B->mailbox[ms]);
        __syncwarp();
        if (lane == 0) mbar_arrive(&B->item_empty[ms]);
        if (id >= n_items) break;
        const PrefillItem it = load_item_uniform<ROWS>(A, id);

        mbar_wait(&B->q_full, item_it & 1, 106, item_it);
        mbar_wait(&B->kv_full[cur.slot], cur.phase, 104, item_it);  // K(0)
        tc_fence_after();
#pragma unroll 1
        for (int w = 0; w < it.nt; ++w) issue_s(w, cur.slot);
        if (elect_one()) {
            tc_commit(&B->kv_empty[cur.slot]);
            if (it.n_kt == 1) tc_commit(&B->q_empty);  // every S MMA of this item has been issued
        }
        __syncwarp();
        cur.advance(C::KV_SLOTS);

        for (int kt = 0; kt < it.n_kt; ++kt) {
            const RingCursor vcur = cur;  // V(kt)
            cur.advance(C::KV_SLOTS);
            const RingCursor kcur = cur;  // K(kt+1)
            const bool has_next = kt + 1 < it.n_kt;
            if (has_next) cur.advance(C::KV_SLOTS);
            mbar_wait(&B->kv_full[vcur.slot], vcur.phase, 107, item_it * 100000 + kt * 1000 + it.n_kt);
            const uint32_t v_a = ring_a + vcur.slot * C::TILE_BYTES;
            if (!has_next) {  // zero V rows past the last visible key (stale or poisoned smem)
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
#pragma unroll 1
            for (int w = 0; w < it.nt; ++w) {
                if (ROWS && kt >= it.kv_tiles(w)) continue;  // the earlier row tile of a pair sees one KV tile fewer
                const uint32_t gw = w ? g1 : g0;
                if (kt == 0) mbar_wait(&B->o_empty[w], ((w ? cnt1 : cnt0) & 1) ^ 1, 108, item_it);  // previous epilogue has read O_w
                mbar_wait(&B->p_full[w], gw & 1, 109, item_it * 100000 + kt * 1000 + it.n_kt);
                tc_fence_after();
                if (elect_one()) {
#pragma unroll
                    for (int ks = 0; ks < 8; ++ks)  // 16 keys per MMA
                        tc_mma_ts(tm + C::TM_O + w * 128, tm + C::TM_S + w * 128 + ks * 8,
                                  make_smem_desc_sw128(v_a + ks * 2048, C::HALF_BYTES, 1024), IDESC_O, (kt | ks) != 0);
                    tc_commit(&B->pv_done[w]);
                }
                __syncwarp();
                if (ROWS ? kt + 1 < it.kv_tiles(w) : has_next) {
                    // K(kt+1): waited by the first tile that needs it (with row pairs tile 0 may not: a repeated wait on
                    // a completed phase returns at once)
                    if (ROWS || w == 0) {
                        mbar_wait(&B->kv_full[kcur.slot], kcur.phase, 104, item_it * 100000 + kt);
                        tc_fence_after();
                    }
                    issue_s(w, kcur.slot);
                }
                if (w) ++g1; else ++g0;
            }
            if (elect_one()) {
                tc_commit(&B->kv_empty[vcur.slot]);
                if (has_next) {
                    tc_commit(&B->kv_empty[kcur.slot]);
                    if (kt + 2 == it.n_kt) tc_commit(&B->q_empty);  // every S MMA of this item has been issued
                }
            }
            __syncwarp();
        }
        ++cnt0;
        if (it.nt > 1) ++cnt1;
        ++item_it;
    }
}

// ------------------------------------------------------------------------------------------------
// softmax warpgroup (4 warps, 128 threads: thread r <-> query row r <-> TMEM lane r, for both query tiles)
__device__ __forceinline__ float max4(float a, float b, float c, float d) { return fmaxf(fmaxf(a, b), fmaxf(c, d)); }
// NWG = 1: one warpgroup alternates between the item's two query tiles.  NWG = 2 (the variant for prefill-dominated
// steps): warpgroup `wg` owns tile wg -- two softmax warps per scheduler, so each hides the other's latencies.
template <int D, bool ROWS, int NWG>
__device__ __forceinline__ void prefill_softmax(const PrefillArgs& A, PrefillBars* B, int wg_warp, int wg) {
    using C = PrefillCfg<D>;
    const int lane = threadIdx.x & 31;
    const int r = wg_warp * 32 + lane;
    const int n_items = A.hdr[HDR_N_ITEMS];
    const uint32_t tm = B->tmem_base + ((uint32_t)(wg_warp * 32) << 16);
    const float scale = A.scale_log2;
    uint32_t item_it = 0;
    uint32_t gA = 0, gB = 0;  // S / P / PV iterations of query tile A, B so far (barrier phases)

    for (;;) {
        const int ms = item_it & 1;
        mbar_wait(&B->item_full[ms], (item_it >> 1) & 1, 110, item_it);
        const int id = B->mailbox[ms];
        __syncwarp();
        if (lane == 0) mbar_arrive(&B->item_empty[ms]);
        if (id >= n_items) break;
        const PrefillItem it = load_item<ROWS>(A, id);
        // row of this thread in tile w: t0 + w * t_step; its last visible key: c + min(t, ql - 1) (rows past the chunk
        // mirror its last row)
        const int t0 = it.qt * kQTile + r, t_step = it.rows ? kQTile : 0;
        const int w_begin = NWG == 2 ? wg : 0, w_end = NWG == 2 ? min(it.nt, wg + 1) : it.nt;
        // running maximum / sum of this row in query tile A and B; the first chunk raises m from -inf (grow_fix)
        float mA = -INFINITY, lA = 0.f, mB = -INFINITY, lB = 0.f;

        for (int kt = 0; kt < it.n_kt; ++kt) {
#pragma unroll 1
          for (int w = w_begin; w < w_end; ++w) {  // NWG = 1: the warpgroup alternates between the two query tiles: while
            // it works on S_B(kt) the tensor pipe runs PV_A(kt) and S_A(kt+1)
            if (ROWS && kt >= it.kv_tiles(w)) continue;  // the earlier row tile of a pair sees one KV tile fewer
            const int limit = it.c + min(t0 + w * t_step, it.ql - 1);
            const uint32_t s_col = tm + C::TM_S + w * 128, o_col = tm + C::TM_O + w * 128;
            float m_used = w ? mB : mA, l = w ? lB : lA;
            const uint32_t g = (w ? gB : gA) + kt;
            mbar_wait(&B->s_full[w], g & 1, 111, item_it * 100000 + kt * 1000 + it.n_kt);
            tc_fence_after();
            // ONE pass over the tile in 32-column chunks, the TMEM load of the next chunk in flight while the current
            // one is exponentiated (two register buffers).  P = exp2(s*scale - m_used) is written with the running
            // maximum m_used of the PREVIOUS chunks; a chunk whose maximum exceeds m_used by more than 2^8 (rare after
            // the first chunk of an item) takes grow_fix(): raise m_used, rescale O, l and the P chunks already written.
            // Code size matters: the roles of an SM share a 32 KiB instruction cache (profiles/r1c_c5.md).
            const int n_vis = limit - kt * kKvTile + 1;  // visible columns of this tile for this row
            const bool masked = __any_sync(0xffffffffu, n_vis < kKvTile);
            float sum0 = 0.f, sum1 = 0.f;

            auto grow_fix = [&](int c4, float cm) {  // cold path
                const float m_new = fmaxf(m_used, cm * scale);
                const float alpha = m_new == -INFINITY ? 1.f : fast_exp2(m_used - m_new);  // rows that do not grow: 1; first chunk of an item: 0
                if (kt > 0) {
                    mbar_wait(&B->pv_done[w], (g - 1) & 1, 112, item_it * 100000 + kt * 1000 + it.n_kt);  // O holds PV(g-1)
                    tc_fence_after();
#pragma unroll 1
                    for (int c = 0; c < D / 32; ++c) {
                        uint32_t o[32];
                        tmem_ld_32x32(o_col + c * 32, o);
                        tc_wait_ld();
#pragma unroll
                        for (int j = 0; j < 32; ++j) o[j] = __float_as_uint(__uint_as_float(o[j]) * alpha);
                        tmem_st_32x32(o_col + c * 32, o);
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
                // Exponentials with the CURRENT m_used (speculative) and the chunk maximum are independent instruction
                // streams: no branch between them, so the FMNMX tree fills the MUFU latency.  If the maximum then
                // turns out to exceed m_used by more than 2^8 (rare; always for the first chunk of an item, where
                // m_used is -inf and the speculative values are inf / NaN), the chunk is redone from its registers.
                uint32_t pk[16];
                const uint64_t sc2 = f32x2_pack(scale, scale);
                uint64_t nm2 = f32x2_pack(-m_used, -m_used);
                uint64_t cs2 = f32x2_pack(0.f, 0.f);
#pragma unroll
                for (int j = 0; j < 32; j += 2) {
                    float x0, x1;
                    f32x2_unpack(f32x2_fma(f32x2_pack(__uint_as_float(s[j]), __uint_as_float(s[j + 1])), sc2, nm2), x0, x1);
                    const float p0 = fast_exp2(x0), p1 = fast_exp2(x1);
                    cs2 = f32x2_add(cs2, f32x2_pack(p0, p1));
                    pk[j >> 1] = pack_bf16x2(p0, p1);
                }
                float cm = -INFINITY;
#pragma unroll
                for (int j = 0; j < 32; j += 4)
                    cm = fmaxf(cm, max4(__uint_as_float(s[j]), __uint_as_float(s[j + 1]), __uint_as_float(s[j + 2]),
                                        __uint_as_float(s[j + 3])));
                if (__any_sync(0xffffffffu, cm * scale > m_used + 8.f)) {  // lazy: P stays <= 2^8
                    grow_fix(c4, cm);
                    nm2 = f32x2_pack(-m_used, -m_used);
                    cs2 = f32x2_pack(0.f, 0.f);
#pragma unroll
                    for (int j = 0; j < 32; j += 2) {
                        float x0, x1;
                        f32x2_unpack(f32x2_fma(f32x2_pack(__uint_as_float(s[j]), __uint_as_float(s[j + 1])), sc2, nm2), x0, x1);
                        const float p0 = fast_exp2(x0), p1 = fast_exp2(x1);
                        cs2 = f32x2_add(cs2, f32x2_pack(p0, p1));
                        pk[j >> 1] = pack_bf16x2(p0, p1);
                    }
                }
                {
                    float c0, c1;
                    f32x2_unpack(cs2, c0, c1);
                    sum0 += c0;
                    sum1 += c1;
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
            if (kt > 0) mbar_wait(&B->pv_done[w], (g - 1) & 1, 114, item_it * 100000 + kt * 1000 + it.n_kt);
            mbar_arrive(&B->p_full[w]);
            if (w) { mB = m_used; lB = l; } else { mA = m_used; lA = l; }
          }
        }

        // epilogue: out = O / l
#pragma unroll 1
        for (int w = w_begin; w < w_end; ++w) {
        const int t = t0 + w * t_step;
        const bool valid = t < it.ql;
        const uint32_t o_col = tm + C::TM_O + w * 128;
        const float m_used = w ? mB : mA, l = w ? lB : lA;
        const int head = it.head(w);
        mbar_wait(&B->pv_done[w], ((w ? gB : gA) + it.kv_tiles(w) - 1) & 1, 113, item_it * 100000 + id);
        tc_fence_after();
        const float inv = 1.f / l;
        uint16_t* orow = A.out + ((size_t)(it.tok0 + t) * A.pool.Hq + head) * D;
#pragma unroll 1
        for (int c4 = 0; c4 < D / 32; ++c4) {
            uint32_t o[32];
            tmem_ld_32x32(o_col + c4 * 32, o);
            tc_wait_ld();
            if (valid) {
#pragma unroll
                for (int j = 0; j < 32; j += 8) {
                    uint4 v;
                    v.x = pack_bf16x2(__uint_as_float(o[j]) * inv, __uint_as_float(o[j + 1]) * inv);
                    v.y = pack_bf16x2(__uint_as_float(o[j + 2]) * inv, __uint_as_float(o[j + 3]) * inv);
                    v.z = pack_bf16x2(__uint_as_float(o[j + 4]) * inv, __uint_as_float(o[j + 5]) * inv);
                    v.w = pack_bf16x2(__uint_as_float(o[j + 6]) * inv, __uint_as_float(o[j + 7]) * inv);
                    *reinterpret_cast<uint4*>(orow + c4 * 32 + j) = v;
                }
            }
        }
        tc_fence_before();
        mbar_arrive(&B->o_empty[w]);
        if (valid && A.lse != nullptr)
            A.lse[(size_t)(it.tok0 + t) * A.pool.Hq + head] = (m_used + log2f(l)) * 0.6931471805599453f;
        }
        gA += it.n_kt0;
        if (it.nt > 1) gB += it.n_kt;
        ++item_it;
    }
}

}  // namespace tropical
