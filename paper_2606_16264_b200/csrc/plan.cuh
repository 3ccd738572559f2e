// plan.cuh -- SURVEY.md 8(a) row A0: the tile directory.  One small kernel turns the per-request
// (q_i, c_i) arrays into two explicit work lists in the workspace -- prefill items
// (request, 128-row q tile, q head) and decode units (request, kv head, head block, page range) --
// so that the persistent attention kernel only pops tickets.  No host sync, no host plan.
#pragma once
#include "common.cuh"

namespace tropical {

constexpr int kQTile = 128;          // query rows per prefill item
constexpr int kKvTile = 128;         // keys per prefill KV iteration (8 pages)
constexpr int kHeadBlock = 8;        // q heads of one kv group handled by one decode unit (MMA M rows used)
constexpr int kTargetUnits = 9472;   // ~8 decode units per resident decode warp (148 SMs x 8 warps x 8)
constexpr int kMinSplitPages = 8;    // never split finer than 128 tokens
constexpr int kSmallBatchSplitPages = 32;  // ... nor finer than 512 tokens when a request has at least 1024 (see plan_kernel)

enum { HDR_N_ITEMS = 0, HDR_N_UNITS = 1, HDR_SPLIT_PAGES = 2, HDR_TICKET_PREFILL = 3, HDR_TICKET_DECODE = 4,
       HDR_TICKET_APPEND = 5 /* fused step: blocks of new tokens whose rows are copied into the pool */,
       HDR_PROF = 16 /* 4 x u64: kernel start (min), prefill end, WG1 decode end, WG0 decode end (max) */,
       HDR_INTS = 64 };

// req_info[i] = {kind, unit_base, nsplit, item_base}; kind 0 skip, 1 decode, 2 prefill
struct WorkspaceLayout {
    size_t hdr, req_info, items, units, group_cnt, part_ml, part_o, total;
    int max_items, max_units;
};

__host__ __device__ inline size_t ws_align(size_t x) { return (x + 255) / 256 * 256; }

__host__ __device__ inline WorkspaceLayout make_layout(int Hq, int Hkv, int D, int num_reqs, int total_q) {
    WorkspaceLayout w;
    const int g = Hq / Hkv;
    const int HB = (g + kHeadBlock - 1) / kHeadBlock;
    w.max_items = (total_q / kQTile + num_reqs) * Hq;
    w.max_units = kTargetUnits + num_reqs * Hkv * HB;
    size_t off = 0;
    w.hdr = off;       off += ws_align(HDR_INTS * sizeof(int));
    w.req_info = off;  off += ws_align((size_t)(num_reqs > 0 ? num_reqs : 1) * sizeof(int4));
    w.items = off;     off += ws_align((size_t)(w.max_items > 0 ? w.max_items : 1) * sizeof(int2));
    w.units = off;     off += ws_align((size_t)w.max_units * sizeof(int4));
    w.group_cnt = off; off += ws_align((size_t)w.max_units * sizeof(int));
    w.part_ml = off;   off += ws_align((size_t)w.max_units * kHeadBlock * sizeof(float2));
    w.part_o = off;    off += ws_align((size_t)w.max_units * kHeadBlock * D * sizeof(float));
    w.total = off;
    return w;
}

struct PlanPtrs {
    int* hdr;
    int4* req_info;
    int2* items;   // {req, (qtile << 16) | (two << 15) | (rows << 14) | head}: two = the item carries a second query tile:
                   // head + 1 of the same kv group at the same rows (rows = 0), or the next 128 rows of the same head (rows = 1)
    int4* units;   // {req, kvh | (hb << 16), page_start, page_count}
    int* group_cnt;  // [n_units] zeroed here: finished units per split group (indexed by the group's first unit)
};

// largest i in [0, n) with base(i) <= e, base non-decreasing
template <int FIELD>
__device__ __forceinline__ int find_owner(const int4* __restrict__ info, int n, int e) {
    int lo = 0, hi = n;
    while (hi - lo > 1) {
        const int mid = (lo + hi) >> 1;
        const int4 v = info[mid];
        const int base = FIELD == 1 ? v.y : v.w;
        if (base <= e) lo = mid; else hi = mid;
    }
    return lo;
}

constexpr int kPlanThreads = 256;      // small blocks with few registers: they find room beside the append's blocks
constexpr int kPlanBlocks = 16;        // each block rebuilds the (cheap) per-request directory and writes a share of the lists
constexpr int kPlanStagedReqs = 1024;  // per-request bases kept in shared memory for the ticket -> request search

// block-wide exclusive scan of one int per thread (256 threads): returns the exclusive prefix, *total = block sum
__device__ __forceinline__ int plan_block_scan(int v, int* s_warp, int* total) {
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    int incl = v;
#pragma unroll
    for (int off = 1; off < 32; off <<= 1) {
        const int t = __shfl_up_sync(0xffffffffu, incl, off);
        if (lane >= off) incl += t;
    }
    __syncthreads();  // s_warp may still be read from a previous scan
    if (lane == 31) s_warp[warp] = incl;
    __syncthreads();
    int base = 0, sum = 0;
#pragma unroll
    for (int w = 0; w < kPlanThreads / 32; ++w) {
        const int t = s_warp[w];
        if (w < warp) base += t;
        sum += t;
    }
    *total = sum;
    return base + incl - v;
}

// block-wide maximum of one non-negative int per thread
__device__ __forceinline__ int plan_block_max(int v, int* s_warp) {
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
#pragma unroll
    for (int off = 16; off > 0; off >>= 1) v = max(v, __shfl_xor_sync(0xffffffffu, v, off));
    __syncthreads();  // s_warp may still be read from a previous scan
    if (lane == 0) s_warp[warp] = v;
    __syncthreads();
    int m = 0;
#pragma unroll
    for (int w = 0; w < kPlanThreads / 32; ++w) m = max(m, s_warp[w]);
    return m;
}

// INVARIANTS of the three-kernel chain append -> plan_kernel -> step kernel (checked only by
// tests/test_gpu_parity.py::test_append_then_attention_ordering_stress, so keep that test in the default suite):
//   1. EVERY exit path of plan_kernel executes griddepcontrol.wait (the early return of the extra blocks below and
//      the end of the kernel).  The step kernel's own griddepcontrol.wait covers only ITS prerequisite grid -- this
//      one -- so the append's writes reach the step kernel only because this grid does not complete before the
//      append has completed and flushed.  A return that skips the wait breaks that silently.
//   2. The step kernel's prologue (everything before its griddepcontrol.wait, csrc/mixed.cu) must not load from or
//      store to global memory: it may run while the append and this kernel are still writing.
__global__ void __launch_bounds__(kPlanThreads) plan_kernel(BatchDesc b, int Hq, int Hkv, PlanPtrs P, int forced_split,
                                                            int row_pairs) {
    // the step kernel (a programmatic dependent of this one) may start its prologue now; it waits for this kernel's
    // completion before it reads the workspace
    asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
    if (threadIdx.x == 0) tl_mark(2, true);
    __shared__ int s_warp[kPlanThreads / 32];
    __shared__ int s_ub[kPlanStagedReqs], s_ib[kPlanStagedReqs], s_ns[kPlanStagedReqs], s_pg[kPlanStagedReqs];
    const int tid = threadIdx.x;
    const int g = Hq / Hkv;
    const int HB = (g + kHeadBlock - 1) / kHeadBlock;
    const int n = b.num_reqs;
    // Prefill items.  Under GQA with an even group an item carries two heads of a kv group at the same 128 rows (`pair`):
    // they share every K/V tile in shared memory.  Otherwise (MHA, odd groups) an item is one head's tile -- or, with
    // row_pairs (the step kernel variant with two softmax warpgroups, csrc/mixed.cu), two consecutive row tiles of the
    // same head, paired from the top so that the lone tile of an odd count is the lightest one, tile 0.
    const int pair = (g % 2 == 0) ? 1 : 0;
    const int rowp = (!pair && row_pairs) ? 1 : 0;
    const int ipt = pair ? Hq / 2 : Hq;
    auto items_of = [&](int q) {
        const int ntile = (q + kQTile - 1) / kQTile;
        return (rowp ? (ntile + 1) / 2 : ntile) * ipt;
    };
    const int chunk = (n + kPlanThreads - 1) / kPlanThreads;  // requests per thread (contiguous: prefix sums)
    const int i0 = tid * chunk, i1 = min(n, i0 + chunk);

    int my_pages = 0, my_max = 0;
    for (int i = i0; i < i1; ++i)
        if (__ldg(b.q_lens + i) == 1) {
            const int pg = (__ldg(b.ctx_lens + i) + 1 + kPageSize - 1) / kPageSize;
            my_pages += pg;
            my_max = max(my_max, pg);
        }
    int total_pages;
    plan_block_scan(my_pages, s_warp, &total_pages);
    const int max_pages = plan_block_max(my_max, s_warp);  // pages of the longest decode request
    const long long page_heads = (long long)total_pages * Hkv * HB;
    int split = (int)((page_heads + kTargetUnits - 1) / kTargetUnits);
    if (split < kMinSplitPages) split = kMinSplitPages;
    split = (split + 7) / 8 * 8;  // whole 128-key blocks: only a request's last unit is ragged
    // Small batches: a unit pays ~2.5 us of start-up (first TMA round trip, partial write, its share of the combine) and
    // the combine of a split group is serial in its splits, so 8-page units (64 splits of an 8192-token request) cost
    // 20-45 % of such a step.  Units of up to kSmallBatchSplitPages pages, but at least two per request, are within
    // 1.5 % of the best forced split over the sweep in profiles/r2c_split_sweep.md; large batches keep the unit target.
    {
        int floor_split = max_pages / 2 / 8 * 8;
        floor_split = min(kSmallBatchSplitPages, max(kMinSplitPages, floor_split));
        if (split < floor_split) split = floor_split;
    }
    // test hook: coarser splits only -- make_layout's max_units bound holds for split >= the automatic value
    if (forced_split > split) split = forced_split;

    int my_units = 0, my_items = 0;
    for (int i = i0; i < i1; ++i) {
        const int q = __ldg(b.q_lens + i);
        if (q == 1) {
            const int pages = (__ldg(b.ctx_lens + i) + 1 + kPageSize - 1) / kPageSize;
            my_units += ((pages + split - 1) / split) * Hkv * HB;
        } else if (q > 1) {
            my_items += items_of(q);
        }
    }
    int n_units, n_items;
    int ubase = plan_block_scan(my_units, s_warp, &n_units);
    int ibase = plan_block_scan(my_items, s_warp, &n_items);
    for (int i = i0; i < i1; ++i) {
        const int q = __ldg(b.q_lens + i);
        int4 info = make_int4(0, ubase, 0, ibase);
        if (q == 1) {
            const int pages = (__ldg(b.ctx_lens + i) + 1 + kPageSize - 1) / kPageSize;
            info.x = 1;
            info.z = (pages + split - 1) / split;
            ubase += info.z * Hkv * HB;
        } else if (q > 1) {
            info.x = 2;
            ibase += items_of(q);
        }
        if (blockIdx.x == 0) P.req_info[i] = info;
        if (n <= kPlanStagedReqs) {  // every block keeps its own copy of the directory for the ticket search below
            s_ub[i] = info.y;
            s_ib[i] = info.w;
            s_ns[i] = info.z;
            // decode request: pages of its context; prefill request: its 128-row query tiles
            s_pg[i] = info.x == 1 ? (__ldg(b.ctx_lens + i) + 1 + kPageSize - 1) / kPageSize : (q + kQTile - 1) / kQTile;
        }
    }
    if (tid == 0 && blockIdx.x == 0) {
        P.hdr[HDR_N_ITEMS] = n_items;
        P.hdr[HDR_N_UNITS] = n_units;
        P.hdr[HDR_SPLIT_PAGES] = split;
        P.hdr[HDR_TICKET_PREFILL] = 0;
        P.hdr[HDR_TICKET_DECODE] = 0;
        P.hdr[HDR_TICKET_APPEND] = 0;
        unsigned long long* prof = reinterpret_cast<unsigned long long*>(P.hdr + HDR_PROF);
        prof[0] = ~0ull;
        prof[1] = prof[2] = prof[3] = 0ull;
    }
    const bool staged = n <= kPlanStagedReqs;
    if (!staged && gridDim.x > 1) {
        // the un-staged search reads req_info from global memory, which only block 0 writes: one block does it all
        if (blockIdx.x != 0) {
            asm volatile("griddepcontrol.wait;" ::: "memory");
            return;
        }
    }
    __syncthreads();  // the directory (shared memory, or block 0's global writes) is visible to the whole block

    // ticket -> request: binary search over the per-request bases, staged in shared memory when they fit; the blocks
    // of the grid (each with its own copy of the directory) share the two work lists
    const int nblk = staged ? gridDim.x : 1, blk = staged ? blockIdx.x : 0;
    auto owner = [&](const int* base_s, int field, int e) {
        if (!staged) return field == 1 ? find_owner<1>(P.req_info, n, e) : find_owner<3>(P.req_info, n, e);
        int lo = 0, hi = n;
        while (hi - lo > 1) {
            const int mid = (lo + hi) >> 1;
            if (base_s[mid] <= e) lo = mid; else hi = mid;
        }
        return lo;
    };
    for (int e = blk * kPlanThreads + tid; e < n_units; e += nblk * kPlanThreads) {
        const int i = owner(s_ub, 1, e);
        int ub, nsplit, pages;
        if (staged) {
            ub = s_ub[i]; nsplit = s_ns[i]; pages = s_pg[i];
        } else {
            const int4 info = P.req_info[i];
            ub = info.y; nsplit = info.z;
            pages = (b.ctx_lens[i] + 1 + kPageSize - 1) / kPageSize;
        }
        const int u = e - ub;
        const int hb = u % HB;
        const int s = (u / HB) % nsplit;
        const int kvh = u / (HB * nsplit);
        const int p0 = s * split;
        P.units[e] = make_int4(i, kvh | (hb << 16), p0, min(split, pages - p0));
        P.group_cnt[e] = 0;
    }
    for (int e = blk * kPlanThreads + tid; e < n_items; e += nblk * kPlanThreads) {
        const int i = owner(s_ib, 3, e);
        const int local = e - (staged ? s_ib[i] : P.req_info[i].w);
        const int ntile = staged ? s_pg[i] : (b.q_lens[i] + kQTile - 1) / kQTile;
        if (!rowp) {
            const int qt = ntile - 1 - local / ipt;  // heaviest (most KV tiles) first
            P.items[e] = make_int2(i, (qt << 16) | (pair << 15) | ((local % ipt) << pair));
        } else {
            const int hi = ntile - 1 - 2 * (local / ipt);  // tiles (hi - 1, hi), heaviest pair first; tile 0 alone if odd
            const int two = hi >= 1 ? 1 : 0;
            P.items[e] = make_int2(i, ((hi - two) << 16) | (two << 15) | (1 << 14) | (local % ipt));
        }
    }
    // Programmatic dependent launch: this kernel may have started while the kernel before it on the stream (the
    // append, which triggers at its first instruction) was still running.  The step kernel behind this one reads what
    // the append wrote, so completion of this kernel must imply completion and visibility of the append:
    // griddepcontrol.wait returns once every prerequisite grid has completed and its memory is flushed (PTX ISA,
    // griddepcontrol); it is a no-op when there is no programmatic dependency.
    if (threadIdx.x == 0) tl_mark(3, false);
    asm volatile("griddepcontrol.wait;" ::: "memory");
    if (threadIdx.x == 0) tl_mark(4, false);
}

}  // namespace tropical
