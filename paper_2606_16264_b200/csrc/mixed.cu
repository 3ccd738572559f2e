// mixed.cu -- tropical_mixed_attention: the plan launch (A0) and the fused persistent step kernel that runs the prefill
// tiles (A3), the decode tiles (A4) and the combine (A5) side by side.
#include <cuda.h>

#include <atomic>

#include "common.cuh"
#include "decode.cuh"
#include "kernels.h"
#include "plan.cuh"
#include "prefill.cuh"
#include "step_variant.h"
#include "tma_host.h"

namespace tropical {

__device__ __forceinline__ DecodeRing make_ring(uint8_t* base, uint64_t* bars, int nst) {
    DecodeRing R;
    R.base = base;
    R.full = bars;
    R.nst = nst;
    R.c_slot = 0;
    R.c_phase = 0;
    R.i_slot = 0;
    return R;
}

// role finish times (globaltimer ns) for the A/B evidence under profiles/: hdr[HDR_PROF ...] as u64; -DTROPICAL_ROLE_PROF builds
__device__ __forceinline__ unsigned long long global_ns() {
    unsigned long long t;
    asm volatile("mov.u64 %0, %globaltimer;" : "=l"(t));
    return t;
}
__device__ __forceinline__ void prof_mark(const int* hdr, int which, bool is_min) {
#ifndef TROPICAL_ROLE_PROF
    // Measurement builds only (-DTROPICAL_ROLE_PROF): the stamps -- a globaltimer read and a 64-bit atomic per softmax /
    // decode warp -- measured 0.6-0.8 % of the C5 step in the burst run (profiles/r3_small_items.md), so the product
    // kernel does not carry them.
    (void)hdr; (void)which; (void)is_min;
    return;
#endif
    unsigned long long* p = reinterpret_cast<unsigned long long*>(const_cast<int*>(hdr) + HDR_PROF) + which;
    if (is_min) atomicMin(p, global_ns()); else atomicMax(p, global_ns());
}

// ------------------------------------------------------------------------------------------------
// The fused step kernel: ONE persistent launch, one CTA per SM, 16 warps, every role compiled for <= 128 registers.
//   warps 0-3       : prefill softmax warpgroup (both query tiles of a two-tile item, alternately)
//   warps 8, 9, 10  : prefill K producer (TMA; pops the item tickets), tcgen05 MMA issuer, V producer
//   warps 4-7, 11-14: decode warp workers, a private TMA ring each (HBM streaming; csrc/decode.cuh)
//   warp 15         : FUSED variant only: copies this step's K / V rows into the pool (append_worker); else idle
// FUSED variant (prefill-dominated steps, where the decode warps have little to do): warps 4-7 are a SECOND softmax
// warpgroup -- warpgroup w owns query tile w of every item, so each scheduler has two softmax warps hiding one
// another's latencies -- and MHA items carry two row tiles of one head (csrc/plan.cuh) so that both always have work;
// they turn into decode workers when the prefill queue is empty, like warps 0-3.
// (Softmax on warps 12-15 -- the issue arbiter is said to prefer the highest warp id of a sub-partition -- was measured:
// no gain, profiles/r2e_fused_step.md.)
// Two variants: FUSED = false is the step kernel of tropical_mixed_attention (this step's rows are in the pool);
// FUSED = true is tropical_mixed_step's for prefill-dominated steps: the rows are read from k_new / v_new and appended here.
// Prefill items and decode units are popped from two ticket counters, so on every SM the tensor pipe (prefill) and
// the HBM stream (decode) are busy at the same time -- the paper's multiplexing at SM granularity.  When the prefill
// queue is empty the four softmax warps become decode workers too, with rings carved out of the (now idle) prefill
// tile memory: a decode-heavy step then streams with 12 workers and ~220 KiB of K/V in flight per SM.
constexpr int kMixedThreads = 512;

template <int D>
struct MixedCfg {
    static constexpr int DEC_WARPS = 8;
    static constexpr int DEC_RING = 12288;                                  // bytes of TMA ring per dedicated decode warp
    static constexpr int DEC_STAGES = DEC_RING / DecodeCfg<D>::PAGE_BYTES;
    static constexpr int LATE_WARPS = 4;                                    // the softmax warps, once the prefill queue is empty
    static constexpr int LATE_RING = PrefillCfg<D>::SMEM_TILES / LATE_WARPS / 1024 * 1024;
    static constexpr int LATE_STAGES = LATE_RING / DecodeCfg<D>::PAGE_BYTES;
    static constexpr int N_DEC_BARS = DEC_WARPS * DEC_STAGES + LATE_WARPS * LATE_STAGES;
    static constexpr int BAR_BYTES = 2048;
    static constexpr int SMEM = PrefillCfg<D>::SMEM_TILES + DEC_WARPS * DEC_RING + BAR_BYTES + 1024;
    static_assert(DEC_STAGES <= kMaxDecodeStages && LATE_STAGES <= kMaxDecodeStages, "stage barriers");
    static_assert(LATE_RING % 1024 == 0 && DEC_RING % 1024 == 0, "ring alignment");
    static_assert(sizeof(PrefillBars) + N_DEC_BARS * 8 <= BAR_BYTES, "barrier block");
    static_assert(SMEM <= 232448, "shared memory per CTA");
};

// Tensor maps of a step: Q, the K / V pools as page-head halves (16 slots) and single slots, and -- fused step only --
// this step's rows k_new / v_new as 16-token and single-token boxes.
struct StepMaps {
    CUtensorMap q, k16, v16, k1, v1, kn16, vn16, kn1, vn1;
};

template <int D, bool FUSED>
__global__ void __launch_bounds__(kMixedThreads, 1)
mixed_kernel(PrefillArgs PA, DecodeArgs DA, const __grid_constant__ StepMaps TM) {
    const CUtensorMap* const tm_q = &TM.q;
    const CUtensorMap* const tm_k = &TM.k16;
    const CUtensorMap* const tm_v = &TM.v16;
    using C = PrefillCfg<D>;
    using M = MixedCfg<D>;
    extern __shared__ uint8_t smem_raw[];
    uint8_t* tiles = reinterpret_cast<uint8_t*>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~uintptr_t(1023));
    uint8_t* rings = tiles + C::SMEM_TILES;
    PrefillBars* PB = reinterpret_cast<PrefillBars*>(rings + M::DEC_WARPS * M::DEC_RING);
    uint64_t* dec_full = reinterpret_cast<uint64_t*>(PB + 1);
    const int warp = uni((int)(threadIdx.x >> 5));
    if (threadIdx.x == 0) tl_mark(5, true);
    if (threadIdx.x == 0) {
        tma_prefetch_desc(tm_q);
        tma_prefetch_desc(tm_k);
        tma_prefetch_desc(tm_v);
        prefill_init_bars(PB, FUSED ? 8 : 4);
        for (int i = 0; i < M::N_DEC_BARS; ++i) mbar_init(dec_full + i, 1);
        fence_mbar_init();
    }
    if (warp == 0) {
        tmem_alloc(&PB->tmem_base, C::TM_COLS);
        tmem_relinquish();
    }
    // (Invariant 2 of csrc/plan.cuh: keep it that way -- no global load or store above this line.)
    // Programmatic dependent launch: everything above (barriers, TMEM, descriptor prefetch) touches no global memory
    // and overlaps the tile-directory kernel and the tail of the append.  From here on the workspace and the pool are
    // read: wait until the directory kernel has completed -- which, by its own final griddepcontrol.wait, implies
    // that the append before it has completed and is visible.
    if (threadIdx.x == 0) tl_mark(6, false);
    asm volatile("griddepcontrol.wait;" ::: "memory");
    if (threadIdx.x == 0) tl_mark(7, true);
    if (threadIdx.x == 0) prof_mark(PA.hdr, 0, true);
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    if (warp < (FUSED ? 8 : 4)) {
        // one code instance for both softmax warpgroups of the FUSED variant (they share the instruction cache)
        const int wg = FUSED ? warp >> 2 : 0, sw = warp & 3;  // warpgroup = query tile it owns; sw = TMEM lane quadrant
        prefill_softmax<D, FUSED, FUSED ? 2 : 1>(PA, PB, sw, wg);
        if ((threadIdx.x & 31) == 0 && wg == 0) prof_mark(PA.hdr, 1, false);
        // The terminating ticket was seen after the last item's final epilogue (of BOTH warpgroups in the two-warpgroup
        // variant): every prefill MMA has completed, so every TMA load into the tile memory has been consumed and the
        // producers issue nothing more.  Warpgroup 0 then streams decode units through rings carved out of the tile
        // memory, warpgroup 1 through the rings of the decode workers it replaced.
        named_bar_sync(1, FUSED ? 256 : 128);
        DecodeRing R = wg == 0 ? make_ring(tiles + sw * M::LATE_RING,
                                           dec_full + M::DEC_WARPS * M::DEC_STAGES + sw * M::LATE_STAGES, M::LATE_STAGES)
                               : make_ring(rings + sw * M::DEC_RING, dec_full + sw * M::DEC_STAGES, M::DEC_STAGES);
        decode_warp_worker<D, FUSED>(DA, tm_k, tm_v, R);
        if ((threadIdx.x & 31) == 0) prof_mark(PA.hdr, wg == 0 ? 3 : 2, false);
    } else if (warp == 8) {
        prefill_producer<D, 0, FUSED>(PA, PB, tiles, tm_q, KvMaps{&TM.k16, &TM.k1, &TM.kn16, &TM.kn1});
    } else if (warp == 9) {
        prefill_mma<D, FUSED>(PA, PB, tiles);
    } else if (warp == 10) {
        prefill_producer<D, 1, FUSED>(PA, PB, tiles, tm_q, KvMaps{&TM.v16, &TM.v1, &TM.vn16, &TM.vn1});
    } else if (warp != 15) {
        const int dw = warp < 8 ? warp - 4 : warp - 7;
        DecodeRing R = make_ring(rings + dw * M::DEC_RING, dec_full + dw * M::DEC_STAGES, M::DEC_STAGES);
        decode_warp_worker<D, FUSED>(DA, tm_k, tm_v, R);
        if ((threadIdx.x & 31) == 0) prof_mark(PA.hdr, 2, false);
    } else if (FUSED) {
        append_worker<D>(DA);  // warp 15: copies this step's rows into the pool beside the attention roles
    }
    tc_fence_before();
    __syncthreads();
    if (threadIdx.x == 0) tl_mark(8, false);
    if (warp == 0) tmem_dealloc(PB->tmem_base, C::TM_COLS);
}

// Per-device one-time state (cudaFuncSetAttribute and the SM count are properties of a device, not of the process).
constexpr int kMaxDevices = 64;
struct DeviceState {
    std::atomic<int> num_sms{0};
    std::atomic<int> smem_attr_set{0};  // bits 0, 1: mixed_kernel<128 / 64, plain>, bit 2: plan_kernel carve-out, bits 3, 4: fused variants
};
static DeviceState g_dev[kMaxDevices];

static DeviceState& device_state() {
    int dev = 0;
    cudaGetDevice(&dev);
    return g_dev[(dev >= 0 && dev < kMaxDevices) ? dev : 0];
}

static int num_sms(DeviceState& ds) {
    int n = ds.num_sms.load(std::memory_order_relaxed);
    if (n == 0) {
        int dev = 0;
        cudaGetDevice(&dev);
        if (cudaDeviceGetAttribute(&n, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess || n <= 0) n = 148;
        ds.num_sms.store(n, std::memory_order_relaxed);
    }
    return n;
}

size_t mixed_workspace_bytes(int Hq, int Hkv, int D, int num_reqs, int total_q) {
    return make_layout(Hq, Hkv, D, num_reqs, total_q).total;
}

size_t profile_offset_bytes() { return make_layout(1, 1, 64, 1, 1).hdr + HDR_PROF * sizeof(int); }

static std::atomic<int> g_grid_cap{0};     // test hook (include/tropical_debug.h): 0 = one CTA per SM
#ifdef TROPICAL_DEBUG_WAIT
static volatile int* g_stuck_host = nullptr;
static void debug_wait_setup() {
    if (g_stuck_host != nullptr) return;
    int* h = nullptr;
    if (cudaHostAlloc((void**)&h, 64 * sizeof(int), cudaHostAllocMapped) != cudaSuccess) return;
    for (int i = 0; i < 64; ++i) h[i] = 0;
    int* d = nullptr;
    if (cudaHostGetDevicePointer((void**)&d, h, 0) != cudaSuccess) return;
    cudaMemcpyToSymbol(g_wait_stuck, &d, sizeof d);
    g_stuck_host = h;
}
#endif

int read_wait_profile(unsigned long long* cycles, unsigned long long* calls, int n, int reset) {
#ifdef TROPICAL_WAIT_PROF
    if (n > 512) n = 512;
    if (cudaMemcpyFromSymbol(cycles, g_wait_cycles, n * sizeof(unsigned long long)) != cudaSuccess) return -1;
    if (cudaMemcpyFromSymbol(calls, g_wait_calls, n * sizeof(unsigned long long)) != cudaSuccess) return -1;
    if (reset) {
        static unsigned long long zeros[512];
        cudaMemcpyToSymbol(g_wait_cycles, zeros, sizeof zeros);
        cudaMemcpyToSymbol(g_wait_calls, zeros, sizeof zeros);
    }
    return n;
#elif defined(TROPICAL_DEBUG_WAIT)
    if (g_stuck_host != nullptr) {  // host-mapped: readable even after the kernel faulted
        for (int i = 0; i < n; ++i) { cycles[i] = 0; calls[i] = 0; }
        cycles[0] = (unsigned long long)g_stuck_host[48];
        for (int w = 0; w < 16 && 16 + w * 3 + 2 < n; ++w)
            for (int k = 0; k < 3; ++k) cycles[16 + w * 3 + k] = (unsigned long long)(long long)g_stuck_host[w * 3 + k];
        calls[0] = 1;
        if (reset) for (int i = 0; i < 64; ++i) g_stuck_host[i] = 0;
        return n;
    }
    // debug build: cycles[0] = abort flag, cycles[1..5] = tag, block, warp, parity, aux of the first stuck wait
    int flag = 0, info[8] = {0};
    if (cudaMemcpyFromSymbol(&flag, g_wait_abort, sizeof flag) != cudaSuccess) return -1;
    if (cudaMemcpyFromSymbol(info, g_wait_abort_info, sizeof info) != cudaSuccess) return -1;
    for (int i = 0; i < n; ++i) { cycles[i] = 0; calls[i] = 0; }
    cycles[0] = (unsigned long long)flag;
    for (int i = 0; i < 5 && i + 1 < n; ++i) cycles[i + 1] = (unsigned long long)(long long)info[i];
    calls[0] = 1;
    (void)0;
    if (reset) {
        const int zero = 0;
        cudaMemcpyToSymbol(g_wait_abort, &zero, sizeof zero);
    }
    return n;
#else
    (void)cycles; (void)calls; (void)n; (void)reset;
    return 0;
#endif
}

static std::atomic<int> g_split_pages{0};  // test hook: 0 = automatic
void set_debug_split_pages(int pages) { g_split_pages.store(pages > 0 ? (pages + 7) / 8 * 8 : 0); }
void set_debug_grid(int num_ctas) { g_grid_cap.store(num_ctas > 0 ? num_ctas : 0); }

static std::atomic<int> g_fused_mode{-1};  // test hook: -1 = the heuristic below, 0 = never fuse, 1 = always fuse
void set_debug_fused(int mode) { g_fused_mode.store(mode < 0 ? -1 : (mode ? 1 : 0)); }

// tropical_mixed_step: fuse the append into the step kernel, or run the append kernel in front of the plain one?
// Measured (profiles/r2e_fused_step.md): the fused variant takes the append off the critical path (C3, prefill-only:
// 62 -> 50 us) but its extra work in the hot loops -- the new-row patch of the decode page loop, the append warp --
// costs 1-4 % on steps that stream a large decode batch (C2 +0.4 %, C5 +4 %), where the separate append is 2 % of the
// step to begin with.  The host sees only the scalars of the batch, not its contexts: a step is taken as
// prefill-dominated when its requests carry at least kFusedMinTokensPerReq new tokens on average, i.e. when it has at
// most one decode request per ~64 prefill tokens.
// The rule itself lives in step_variant.h, shared with the step-cost model whose fits are keyed on it.
static bool choose_fused(const BatchDesc& b) {
    const int mode = g_fused_mode.load(std::memory_order_relaxed);
    if (mode >= 0) return mode == 1;
    return step_is_prefill_dominated(b.total_q, b.num_reqs);
}

template <int D, bool FUSED>
static cudaError_t launch_mixed_t(const PoolDesc& pool, const BatchDesc& b, const void* q, const void* k_new,
                                  const void* v_new, void* out, float* lse, float scale_log2, void* workspace,
                                  cudaStream_t stream, int* launches) {
    const WorkspaceLayout w = make_layout(pool.Hq, pool.Hkv, D, b.num_reqs, b.total_q);
    char* ws = (char*)workspace;
    PlanPtrs P;
    P.hdr = (int*)(ws + w.hdr);
    P.req_info = (int4*)(ws + w.req_info);
    P.items = (int2*)(ws + w.items);
    P.units = (int4*)(ws + w.units);
    P.group_cnt = (int*)(ws + w.group_cnt);
    // The plan reads only the step's metadata and writes only the workspace: launched with programmatic stream
    // serialization it overlaps a preceding tropical_kv_append (whose kernel triggers at once), and its last
    // statement is griddepcontrol.wait.  The step kernel behind it is a programmatic dependent of the directory kernel
    // in turn: it sets up its barriers and tensor memory early and executes griddepcontrol.wait before its first read
    // of the workspace or the pool, so it reads them only after the directory kernel -- hence the append -- has
    // completed.  After a kernel that never triggers, each of the two starts in normal stream order.  Contract for
    // callers (include/tropical.h): a preceding kernel that triggers early must not still be writing q_lens /
    // ctx_lens / q_offsets / page_table.
    DeviceState& ds = device_state();
    if (!(ds.smem_attr_set.load(std::memory_order_acquire) & 4)) {
        // same shared-memory carve-out as the append and the step kernel: its blocks can then share SMs with theirs
        cudaFuncSetAttribute(plan_kernel, cudaFuncAttributePreferredSharedMemoryCarveout, cudaSharedmemCarveoutMaxShared);
        ds.smem_attr_set.fetch_or(4, std::memory_order_release);
    }
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3(kPlanBlocks);  // see plan_kernel: the blocks share the work lists
    cfg.blockDim = dim3(kPlanThreads);
    cfg.dynamicSmemBytes = 0;
    cfg.stream = stream;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = attr;
    cfg.numAttrs = 1;
    cudaError_t e = cudaLaunchKernelEx(&cfg, plan_kernel, b, pool.Hq, pool.Hkv, P, g_split_pages.load(std::memory_order_relaxed),
                                       FUSED ? 1 : 0);  // row-pair items: only the variant with two softmax warpgroups reads them
    if (e != cudaSuccess) return e;
    ++*launches;

    StepMaps TM;
    const long long rows = (long long)pool.num_pages * pool.Hkv * kPageSize;
    constexpr bool fused = FUSED;
    if (!encode_pool_map(&TM.k16, pool.k_pool, rows, D) || !encode_pool_map(&TM.v16, pool.v_pool, rows, D) ||
        !encode_q_map(&TM.q, q, b.total_q, pool.Hq, D, 1, kQTile))
        return cudaErrorInvalidValue;
    if (fused) {
        if (!encode_pool_map(&TM.k1, pool.k_pool, rows, D, 1) || !encode_pool_map(&TM.v1, pool.v_pool, rows, D, 1) ||
            !encode_q_map(&TM.kn16, k_new, b.total_q, pool.Hkv, D, 1, kPageSize) ||
            !encode_q_map(&TM.vn16, v_new, b.total_q, pool.Hkv, D, 1, kPageSize) ||
            !encode_q_map(&TM.kn1, k_new, b.total_q, pool.Hkv, D, 1, 1) ||
            !encode_q_map(&TM.vn1, v_new, b.total_q, pool.Hkv, D, 1, 1))
            return cudaErrorInvalidValue;
    } else {  // never dereferenced
        TM.k1 = TM.kn16 = TM.kn1 = TM.k16;
        TM.v1 = TM.vn16 = TM.vn1 = TM.v16;
    }

    PrefillArgs PA;
    PA.pool = pool;
    PA.b = b;
    PA.out = (uint16_t*)out;
    PA.lse = lse;
    PA.scale_log2 = scale_log2;
    PA.hdr = P.hdr;
    PA.ticket = P.hdr + HDR_TICKET_PREFILL;
    PA.items = P.items;

    DecodeArgs A;
    A.pool = pool;
    A.b = b;
    A.q = (const uint16_t*)q;
    A.out = (uint16_t*)out;
    A.lse = lse;
    A.scale_log2 = scale_log2;
    A.hdr = P.hdr;
    A.ticket = P.hdr + HDR_TICKET_DECODE;
    A.req_info = P.req_info;
    A.units = P.units;
    A.part_ml = (float2*)(ws + w.part_ml);
    A.part_o = (float*)(ws + w.part_o);
    A.group_cnt = P.group_cnt;
    A.k_new = FUSED ? (const uint16_t*)k_new : nullptr;
    A.v_new = FUSED ? (const uint16_t*)v_new : nullptr;

#ifdef TROPICAL_DEBUG_WAIT
    debug_wait_setup();
#endif
    // A3 + A4 + A5 in one persistent launch
    const size_t smem = MixedCfg<D>::SMEM;
    const int attr_bit = (D == 128 ? 1 : 2) << (FUSED ? 3 : 0);  // bits 0, 1: plain variants; bits 3, 4: fused variants
    if (!(ds.smem_attr_set.load(std::memory_order_acquire) & attr_bit)) {
        e = cudaFuncSetAttribute(mixed_kernel<D, FUSED>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (e != cudaSuccess) return e;
        ds.smem_attr_set.fetch_or(attr_bit, std::memory_order_release);
    }
    const int cap = g_grid_cap.load(std::memory_order_relaxed), sms = num_sms(ds);
    cudaLaunchConfig_t mcfg = {};
    mcfg.gridDim = dim3((cap > 0 && cap < sms) ? cap : sms);
    mcfg.blockDim = dim3(kMixedThreads);
    mcfg.dynamicSmemBytes = smem;
    mcfg.stream = stream;
    mcfg.attrs = attr;  // programmatic stream serialization: its prologue overlaps the directory kernel (which triggers at once)
    mcfg.numAttrs = 1;
    e = cudaLaunchKernelEx(&mcfg, mixed_kernel<D, FUSED>, PA, A, TM);
    if (e != cudaSuccess) return e;
    ++*launches;

    return cudaSuccess;
}

cudaError_t launch_mixed_attention(const PoolDesc& pool, const BatchDesc& b, const void* q, const void* k_new,
                                   const void* v_new, void* out, float* lse, float scale_log2, void* workspace,
                                   cudaStream_t stream, int* launches) {
    if (k_new != nullptr && choose_fused(b)) {  // tropical_mixed_step, append inside the step kernel
        if (pool.D == 128)
            return launch_mixed_t<128, true>(pool, b, q, k_new, v_new, out, lse, scale_log2, workspace, stream, launches);
        return launch_mixed_t<64, true>(pool, b, q, k_new, v_new, out, lse, scale_log2, workspace, stream, launches);
    }
    if (k_new != nullptr) {  // tropical_mixed_step on a decode-heavy step: the append kernel in front of the plain variant
        const cudaError_t e = launch_kv_append(pool, b, k_new, v_new, stream);
        if (e != cudaSuccess) return e;
        ++*launches;
    }
    if (pool.D == 128)
        return launch_mixed_t<128, false>(pool, b, q, nullptr, nullptr, out, lse, scale_log2, workspace, stream, launches);
    return launch_mixed_t<64, false>(pool, b, q, nullptr, nullptr, out, lse, scale_log2, workspace, stream, launches);
}

// measurement builds (-DTROPICAL_TIMELINE): this translation unit's copy of the timestamps (slots 2 .. 8)
int read_timeline_mixed(unsigned long long* out16, int reset) {
#ifdef TROPICAL_TIMELINE
    return timeline_read(out16, reset);
#else
    (void)out16; (void)reset;
    return 0;
#endif
}

}  // namespace tropical
