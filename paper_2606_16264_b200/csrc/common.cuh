// common.cuh -- shared device helpers for the sm_100a kernels (PTX wrappers, bf16 packing).
// Not shared with oracle/ in any way.
#pragma once
#include <cuda_bf16.h>
#include <cuda_runtime.h>
#include <stdint.h>
#include <stdio.h>

namespace tropical {

// Measurement build only (-DTROPICAL_TIMELINE): global-timer stamps of the three kernels of a step (min over the
// blocks for a start, max for an end), one copy per translation unit, read back by tropical_debug_timeline:
//   0 append start, 1 append end, 2 directory start, 3 directory body end, 4 directory end (after its wait on the
//   append), 5 step kernel start, 6 its prologue end (last CTA), 7 its first CTA past griddepcontrol.wait, 8 its end.
#ifdef TROPICAL_TIMELINE
static __device__ unsigned long long g_tl[16];
__device__ __forceinline__ void tl_mark(int i, bool mn) {
    unsigned long long t;
    asm volatile("mov.u64 %0, %globaltimer;" : "=l"(t));
    if (mn) atomicMin(&g_tl[i], t); else atomicMax(&g_tl[i], t);
}
static inline int timeline_read(unsigned long long* out16, int reset) {
    if (cudaDeviceSynchronize() != cudaSuccess) return -1;
    if (out16 && cudaMemcpyFromSymbol(out16, g_tl, 16 * sizeof(unsigned long long)) != cudaSuccess) return -1;
    if (reset) {
        unsigned long long init[16];
        for (int i = 0; i < 16; ++i) init[i] = 0ull;
        init[0] = init[2] = init[5] = init[7] = ~0ull;  // starts are minima
        if (cudaMemcpyToSymbol(g_tl, init, sizeof init) != cudaSuccess) return -1;
    }
    return 16;
}
#else
__device__ __forceinline__ void tl_mark(int, bool) {}
#endif

// Measurement builds only, WRONG RESULTS by design (profiles/r2b_whatif.md: what each part of the fused step costs under
// the board's power limit): -DTROPICAL_WHATIF_NO_MMA issues the prefill MMAs with N = 16 (1/8 of the tensor work),
// -DTROPICAL_WHATIF_NO_EXP replaces the softmax exponentials by one FMA, -DTROPICAL_WHATIF_NO_DECODE_MATH keeps 1/8 of
// the decode ldmatrix + MMA work, -DTROPICAL_WHATIF_HALF_KV loads half of every full prefill K/V tile.
#if defined(TROPICAL_WHATIF_NO_MMA) || defined(TROPICAL_WHATIF_NO_EXP) || defined(TROPICAL_WHATIF_NO_DECODE_MATH) || \
    defined(TROPICAL_WHATIF_HALF_KV)
#define TROPICAL_WHATIF_BUILD 1
#endif

constexpr int kPageSize = 16;  // BASELINE.json: page size 16 in every config

struct PoolDesc {
    int Hq, Hkv, D, num_pages;
    const uint16_t* k_pool;
    const uint16_t* v_pool;
};

struct BatchDesc {
    int num_reqs, total_q, max_kv_len, stride;
    const int* q_lens;
    const int* ctx_lens;
    const int* q_offsets;
    const int* page_table;
};

// ---------------------------------------------------------------- small math / packing
__device__ __forceinline__ float bf16_lo(uint32_t v) { return __uint_as_float(v << 16); }
__device__ __forceinline__ float bf16_hi(uint32_t v) { return __uint_as_float(v & 0xffff0000u); }

__device__ __forceinline__ uint32_t pack_bf16x2(float lo, float hi) {
    // cvt.rn.bf16x2.f32 d, a, b : a -> upper half, b -> lower half
    uint32_t r;
    asm("cvt.rn.bf16x2.f32 %0, %1, %2;" : "=r"(r) : "f"(hi), "f"(lo));
    return r;
}

__device__ __forceinline__ float fast_exp2(float x) {
    float y;
    asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}

// packed fp32 pairs (FFMA2 / FADD2 on sm_100): half the issue slots of the softmax inner loop
__device__ __forceinline__ uint64_t f32x2_pack(float lo, float hi) {
    uint64_t r;
    asm("mov.b64 %0, {%1, %2};" : "=l"(r) : "f"(lo), "f"(hi));
    return r;
}
__device__ __forceinline__ void f32x2_unpack(uint64_t v, float& lo, float& hi) {
    asm("mov.b64 {%0, %1}, %2;" : "=f"(lo), "=f"(hi) : "l"(v));
}
__device__ __forceinline__ uint64_t f32x2_fma(uint64_t a, uint64_t b, uint64_t c) {
    uint64_t r;
    asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(r) : "l"(a), "l"(b), "l"(c));
    return r;
}
__device__ __forceinline__ uint64_t f32x2_add(uint64_t a, uint64_t b) {
    uint64_t r;
    asm("add.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(a), "l"(b));
    return r;
}

__device__ __forceinline__ uint32_t smem_u32(const void* p) {
    return static_cast<uint32_t>(__cvta_generic_to_shared(p));
}

// request owning packed token row `tok`: largest i with q_offsets[i] <= tok
__device__ __forceinline__ int find_request(const int* __restrict__ q_offsets, int num_reqs, int tok) {
    int lo = 0, hi = num_reqs;  // invariant: q_offsets[lo] <= tok < q_offsets[hi]
    while (hi - lo > 1) {
        int mid = (lo + hi) >> 1;
        if (__ldg(q_offsets + mid) <= tok) lo = mid; else hi = mid;
    }
    return lo;
}

// ---------------------------------------------------------------- mbarrier
__device__ __forceinline__ void mbar_init(uint64_t* bar, uint32_t count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count));
}
__device__ __forceinline__ void fence_mbar_init() {
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
}
__device__ __forceinline__ void mbar_arrive_expect_tx(uint64_t* bar, uint32_t bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes)
                 : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint64_t* bar) {
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ bool mbar_try_wait(uint64_t* bar, uint32_t parity) {
    uint32_t ok;
    asm volatile(
        "{\n\t.reg .pred p;\n\t"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\t"
        "selp.u32 %0, 1, 0, p;\n\t}"
        : "=r"(ok)
        : "r"(smem_u32(bar)), "r"(parity)
        : "memory");
    return ok != 0;
}
// try_wait with a suspend-time hint: the hardware may park the thread for up to `ns` nanoseconds before it reports
// "not yet" (PTX ISA, mbarrier.try_wait, suspendTimeHint); a parked warp issues nothing.
__device__ __forceinline__ bool mbar_try_wait_hint(uint64_t* bar, uint32_t parity, uint32_t ns) {
    uint32_t ok;
    asm volatile(
        "{\n\t.reg .pred p;\n\t"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2, %3;\n\t"
        "selp.u32 %0, 1, 0, p;\n\t}"
        : "=r"(ok)
        : "r"(smem_u32(bar)), "r"(parity), "r"(ns)
        : "memory");
    return ok != 0;
}
// Spin policy of mbar_wait's slow path (A/B record: profiles/r3_wait_spin.md):
//   0 = round 2: try_wait + clock64() + 64-bit compare on every iteration (9 SASS instructions per spin)
//   1 = no clock read in the loop: iterations are counted and the deadline is looked at every 2^14 of them
//   2 = 1 + suspend-time hint on the try_wait
//   3 = 2 + nanosleep back-off on the long waits (decode ring, producer slot, MMA waiting for P)
//   4 = 1 + one clock read per iteration, its value unused (policy 0's pacing without its compare); 5 = two reads
// Policy 0 stays the product's: every alternative measured 1-5 % SLOWER on C5, burst and sustained, although each
// raised the SM clock the board holds at its power limit (fewer instructions per spin, but more cycles per step).
#ifndef TROPICAL_WAIT_V
#define TROPICAL_WAIT_V 0
#endif
#ifndef TROPICAL_WAIT_HINT_NS
#define TROPICAL_WAIT_HINT_NS 2000
#endif

#ifdef TROPICAL_WAIT_PROF
// Measurement build only (-DTROPICAL_WAIT_PROF): cycles and calls of every mbar_wait, by tag (lane 0 of each warp).
static __device__ unsigned long long g_wait_cycles[512];
static __device__ unsigned long long g_wait_calls[512];
#endif

#ifdef TROPICAL_DEBUG_WAIT
// Debug build (-DTROPICAL_DEBUG_WAIT): a wait that times out records (tag, block, warp, parity, aux) of the FIRST
// stuck waiter, raises g_wait_abort so that every other wait falls through, and the kernel runs to its end with
// garbage results; tropical_debug_wait_profile(...) then reports the record (cycles[0..4]).
static __device__ int g_wait_abort;
static __device__ int g_wait_abort_info[8];
static __device__ int* g_wait_stuck;  // host-mapped [16][3] (readable after a fault): per warp of block 0, the wait it was in (tag, parity, aux)
#endif

// Bounded wait: a protocol bug traps (launch failure, TROPICAL_ERR_CUDA at the next call) instead of hanging the GPU.
__device__ __forceinline__ void mbar_wait(uint64_t* bar, uint32_t parity, int tag = 0, int aux = 0) {
#ifdef TROPICAL_WAIT_PROF
    const long long tp = clock64();
#endif
#if TROPICAL_WAIT_V >= 1 && !defined(TROPICAL_DEBUG_WAIT)
    if (!mbar_try_wait(bar, parity)) {
        // Most of a step's waits end here within a few tries, and the step is bound by board power: the loop holds
        // nothing but the try, a counter and the branch.  The deadline (a protocol bug traps instead of hanging the
        // GPU) costs a clock read once per 2^14 tries.
        long long t0 = 0;
        bool ok = false;
        do {
#pragma unroll 1
            for (uint32_t spins = 0; spins < 0x4000u; ++spins) {
#if TROPICAL_WAIT_V == 2 || TROPICAL_WAIT_V == 3
                ok = mbar_try_wait_hint(bar, parity, TROPICAL_WAIT_HINT_NS);
#else
                ok = mbar_try_wait(bar, parity);
#endif
                if (ok) break;
#if TROPICAL_WAIT_V == 3
                if ((tag == 201 || tag == 202 || tag == 103 || tag == 109) && spins >= 4) __nanosleep(64);
#endif
#if TROPICAL_WAIT_V == 4 || TROPICAL_WAIT_V == 5
                {   // policy 1 paced like policy 0: the clock read(s) without the compare
                    long long dummy;
                    asm volatile("mov.u64 %0, %%clock64;" : "=l"(dummy));
#if TROPICAL_WAIT_V == 5
                    asm volatile("mov.u64 %0, %%clock64;" : "=l"(dummy));
#endif
                }
#endif
            }
#ifndef TROPICAL_NO_WAIT_TRAP
            if (!ok) {
                // ~20 s at 1.9 GHz: far beyond any legitimate wait even under time-slicing or MPS (a step takes < 1 ms);
                // build with -DTROPICAL_NO_WAIT_TRAP to wait forever (debugger sessions)
                const long long now = clock64();
                if (t0 == 0) t0 = now;
                else if (now - t0 > 40000000000LL) __trap();
            }
#endif
        } while (!ok);
    }
#else
    if (!mbar_try_wait(bar, parity)) {
        long long t0 = clock64();
        while (!mbar_try_wait(bar, parity)) {
#ifdef TROPICAL_DEBUG_WAIT
            if (*(volatile int*)&g_wait_abort) {
                if ((threadIdx.x & 31) == 0 && blockIdx.x == 0 && g_wait_stuck != nullptr &&
                    g_wait_stuck[(threadIdx.x >> 5) * 3] == 0) {
                    g_wait_stuck[(threadIdx.x >> 5) * 3 + 1] = (int)parity;
                    g_wait_stuck[(threadIdx.x >> 5) * 3 + 2] = aux;
                    g_wait_stuck[(threadIdx.x >> 5) * 3] = tag;
                    __threadfence_system();
                }
                break;
            }
            if (clock64() - t0 > 400000000LL) {  // ~0.2 s
                if ((threadIdx.x & 31) == 0 && atomicCAS(&g_wait_abort, 0, 1) == 0) {
                    g_wait_abort_info[0] = tag;
                    g_wait_abort_info[1] = blockIdx.x;
                    g_wait_abort_info[2] = threadIdx.x >> 5;
                    g_wait_abort_info[3] = (int)parity;
                    g_wait_abort_info[4] = aux;
                    if (g_wait_stuck != nullptr && blockIdx.x == 0) {
                        g_wait_stuck[(threadIdx.x >> 5) * 3 + 1] = (int)parity;
                        g_wait_stuck[(threadIdx.x >> 5) * 3 + 2] = aux;
                        g_wait_stuck[(threadIdx.x >> 5) * 3] = tag;
                        g_wait_stuck[48] = 1;
                    }
                    __threadfence_system();
                }
                break;
            }
#else
#ifndef TROPICAL_NO_WAIT_TRAP
            // ~20 s at 1.9 GHz: far beyond any legitimate wait even under time-slicing or MPS (a step takes < 1 ms);
            // build with -DTROPICAL_NO_WAIT_TRAP to wait forever (debugger sessions)
            if (clock64() - t0 > 40000000000LL) __trap();
#endif
#endif
        }
    }
#endif  // TROPICAL_WAIT_V
#ifdef TROPICAL_WAIT_PROF
    if ((threadIdx.x & 31) == 0) {
        atomicAdd(&g_wait_cycles[tag & 511], (unsigned long long)(clock64() - tp));
        atomicAdd(&g_wait_calls[tag & 511], 1ull);
    }
#endif
    (void)tag;
    (void)aux;
}

// measurement builds: total lifetime of a role (same counters as the waits, tag = role id)
__device__ __forceinline__ long long prof_begin() {
#ifdef TROPICAL_WAIT_PROF
    return clock64();
#else
    return 0;
#endif
}
__device__ __forceinline__ void prof_end(int tag, long long t0) {
#ifdef TROPICAL_WAIT_PROF
    if ((threadIdx.x & 31) == 0) {
        atomicAdd(&g_wait_cycles[tag & 511], (unsigned long long)(clock64() - t0));
        atomicAdd(&g_wait_calls[tag & 511], 1ull);
    }
#else
    (void)tag; (void)t0;
#endif
}

// position in a ring of mbarrier-guarded shared-memory slots
struct RingCursor {
    int slot;
    uint32_t phase;  // parity of the current use of `slot`
    __device__ __forceinline__ void advance(int nslots) {
        if (++slot == nslots) { slot = 0; phase ^= 1; }
    }
};

__device__ __forceinline__ void fence_proxy_async() {
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
}

// ---------------------------------------------------------------- TMA (cp.async.bulk.tensor)
__device__ __forceinline__ void tma_load_2d(void* dst, const void* tmap, int c0, int c1, uint64_t* bar) {
    asm volatile(
        "cp.async.bulk.tensor.2d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%3, %4}], [%2];"
        ::"r"(smem_u32(dst)), "l"(tmap), "r"(smem_u32(bar)), "r"(c0), "r"(c1)
        : "memory");
}
__device__ __forceinline__ void tma_load_3d(void* dst, const void* tmap, int c0, int c1, int c2, uint64_t* bar) {
    asm volatile(
        "cp.async.bulk.tensor.3d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%3, %4, %5}], [%2];"
        ::"r"(smem_u32(dst)), "l"(tmap), "r"(smem_u32(bar)), "r"(c0), "r"(c1), "r"(c2)
        : "memory");
}
__device__ __forceinline__ void tma_prefetch_desc(const void* tmap) {
    asm volatile("prefetch.tensormap [%0];" ::"l"(tmap) : "memory");
}

// ---------------------------------------------------------------- legacy warp MMA + ldmatrix (decode tiles)
__device__ __forceinline__ void ldmatrix_x4(uint32_t addr, uint32_t& r0, uint32_t& r1, uint32_t& r2, uint32_t& r3) {
    asm volatile("ldmatrix.sync.aligned.m8n8.x4.shared.b16 {%0,%1,%2,%3}, [%4];"
                 : "=r"(r0), "=r"(r1), "=r"(r2), "=r"(r3) : "r"(addr));
}
__device__ __forceinline__ void ldmatrix_x4_trans(uint32_t addr, uint32_t& r0, uint32_t& r1, uint32_t& r2, uint32_t& r3) {
    asm volatile("ldmatrix.sync.aligned.m8n8.x4.trans.shared.b16 {%0,%1,%2,%3}, [%4];"
                 : "=r"(r0), "=r"(r1), "=r"(r2), "=r"(r3) : "r"(addr));
}
// D(16x8,f32) += A(16x16,bf16,row) * B(16x8,bf16,col)
__device__ __forceinline__ void mma_bf16_16816(float (&d)[4], uint32_t a0, uint32_t a1, uint32_t a2, uint32_t a3,
                                               uint32_t b0, uint32_t b1) {
    asm volatile(
        "mma.sync.aligned.m16n8k16.row.col.f32.bf16.bf16.f32 {%0,%1,%2,%3}, {%4,%5,%6,%7}, {%8,%9}, {%0,%1,%2,%3};"
        : "+f"(d[0]), "+f"(d[1]), "+f"(d[2]), "+f"(d[3])
        : "r"(a0), "r"(a1), "r"(a2), "r"(a3), "r"(b0), "r"(b1));
}

// ---------------------------------------------------------------- tcgen05 / TMEM (prefill tiles)
__device__ __forceinline__ void tmem_alloc(uint32_t* dst_smem, uint32_t ncols) {
    asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(smem_u32(dst_smem)), "r"(ncols)
                 : "memory");
}
__device__ __forceinline__ void tmem_relinquish() {
    asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
}
__device__ __forceinline__ void tmem_dealloc(uint32_t taddr, uint32_t ncols) {
    asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(taddr), "r"(ncols) : "memory");
}
__device__ __forceinline__ void tc_fence_before() { asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void tc_fence_after() { asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void tc_wait_ld() { asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory"); }
__device__ __forceinline__ void tc_wait_st() { asm volatile("tcgen05.wait::st.sync.aligned;" ::: "memory"); }

// D[tmem] (+)= A[smem desc] * B[smem desc]
__device__ __forceinline__ void tc_mma_ss(uint32_t d_tmem, uint64_t a_desc, uint64_t b_desc, uint32_t idesc, uint32_t accumulate) {
    asm volatile(
        "{\n\t.reg .pred p;\n\tsetp.ne.b32 p, %4, 0;\n\t"
        "tcgen05.mma.cta_group::1.kind::f16 [%0], %1, %2, %3, p;\n\t}"
        ::"r"(d_tmem), "l"(a_desc), "l"(b_desc), "r"(idesc), "r"(accumulate)
        : "memory");
}
// D[tmem] (+)= A[tmem] * B[smem desc]
__device__ __forceinline__ void tc_mma_ts(uint32_t d_tmem, uint32_t a_tmem, uint64_t b_desc, uint32_t idesc, uint32_t accumulate) {
    asm volatile(
        "{\n\t.reg .pred p;\n\tsetp.ne.b32 p, %4, 0;\n\t"
        "tcgen05.mma.cta_group::1.kind::f16 [%0], [%1], %2, %3, p;\n\t}"
        ::"r"(d_tmem), "r"(a_tmem), "l"(b_desc), "r"(idesc), "r"(accumulate)
        : "memory");
}
// mbarrier arrives once every tcgen05 op issued so far by this thread has completed
__device__ __forceinline__ void tc_commit(uint64_t* bar) {
    asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" ::"r"(smem_u32(bar))
                 : "memory");
}

// 32 lanes x 32 consecutive 32-bit columns: thread i of the warp reads lane (lane_base + i)
__device__ __forceinline__ void tmem_ld_32x32(uint32_t taddr, uint32_t (&r)[32]) {
    asm volatile(
        "tcgen05.ld.sync.aligned.32x32b.x32.b32 "
        "{%0,%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15,"
        "%16,%17,%18,%19,%20,%21,%22,%23,%24,%25,%26,%27,%28,%29,%30,%31}, [%32];"
        : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]), "=r"(r[7]),
          "=r"(r[8]), "=r"(r[9]), "=r"(r[10]), "=r"(r[11]), "=r"(r[12]), "=r"(r[13]), "=r"(r[14]), "=r"(r[15]),
          "=r"(r[16]), "=r"(r[17]), "=r"(r[18]), "=r"(r[19]), "=r"(r[20]), "=r"(r[21]), "=r"(r[22]), "=r"(r[23]),
          "=r"(r[24]), "=r"(r[25]), "=r"(r[26]), "=r"(r[27]), "=r"(r[28]), "=r"(r[29]), "=r"(r[30]), "=r"(r[31])
        : "r"(taddr)
        : "memory");
}
__device__ __forceinline__ void tmem_st_32x32(uint32_t taddr, const uint32_t (&r)[32]) {
    asm volatile(
        "tcgen05.st.sync.aligned.32x32b.x32.b32 [%0], "
        "{%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15,%16,"
        "%17,%18,%19,%20,%21,%22,%23,%24,%25,%26,%27,%28,%29,%30,%31,%32};"
        ::"r"(taddr),
          "r"(r[0]), "r"(r[1]), "r"(r[2]), "r"(r[3]), "r"(r[4]), "r"(r[5]), "r"(r[6]), "r"(r[7]),
          "r"(r[8]), "r"(r[9]), "r"(r[10]), "r"(r[11]), "r"(r[12]), "r"(r[13]), "r"(r[14]), "r"(r[15]),
          "r"(r[16]), "r"(r[17]), "r"(r[18]), "r"(r[19]), "r"(r[20]), "r"(r[21]), "r"(r[22]), "r"(r[23]),
          "r"(r[24]), "r"(r[25]), "r"(r[26]), "r"(r[27]), "r"(r[28]), "r"(r[29]), "r"(r[30]), "r"(r[31])
        : "memory");
}

__device__ __forceinline__ void tmem_ld_32x32_x16(uint32_t taddr, uint32_t (&r)[16]) {
    asm volatile(
        "tcgen05.ld.sync.aligned.32x32b.x16.b32 "
        "{%0,%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15}, [%16];"
        : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]), "=r"(r[7]),
          "=r"(r[8]), "=r"(r[9]), "=r"(r[10]), "=r"(r[11]), "=r"(r[12]), "=r"(r[13]), "=r"(r[14]), "=r"(r[15])
        : "r"(taddr)
        : "memory");
}
__device__ __forceinline__ void tmem_st_32x32_x16(uint32_t taddr, const uint32_t (&r)[16]) {
    asm volatile(
        "tcgen05.st.sync.aligned.32x32b.x16.b32 [%0], "
        "{%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15,%16};"
        ::"r"(taddr),
          "r"(r[0]), "r"(r[1]), "r"(r[2]), "r"(r[3]), "r"(r[4]), "r"(r[5]), "r"(r[6]), "r"(r[7]),
          "r"(r[8]), "r"(r[9]), "r"(r[10]), "r"(r[11]), "r"(r[12]), "r"(r[13]), "r"(r[14]), "r"(r[15])
        : "memory");
}

// ---------------------------------------------------------------- named barriers
__device__ __forceinline__ void named_bar_sync(int id, int nthreads) {
    asm volatile("barrier.cta.sync %0, %1;" ::"r"(id), "r"(nthreads) : "memory");
}
// K-major / MN-major SWIZZLE_128B shared-memory matrix descriptor (sm_100 format, version 1).
//   bits [0,14) start>>4, [16,30) LBO>>4, [32,46) SBO>>4, [46,48) version=1, [61,64) layout (2 = SW128)
__device__ __forceinline__ uint64_t make_smem_desc_sw128(uint32_t saddr, uint32_t lbo_bytes, uint32_t sbo_bytes) {
    uint64_t d = 0;
    d |= (uint64_t)((saddr & 0x3FFFF) >> 4);
    d |= (uint64_t)((lbo_bytes >> 4) & 0x3FFF) << 16;
    d |= (uint64_t)((sbo_bytes >> 4) & 0x3FFF) << 32;
    d |= (uint64_t)1 << 46;
    d |= (uint64_t)2 << 61;
    return d;
}
// kind::f16 instruction descriptor: bf16 x bf16 -> f32, M x N, A K-major, B K-major or MN-major
__host__ __device__ constexpr uint32_t make_idesc_bf16(int M, int N, bool b_mn_major, bool a_mn_major = false) {
    return (1u << 4)                       // c_format = F32
           | (1u << 7)                     // a_format = BF16
           | (1u << 10)                    // b_format = BF16
           | ((a_mn_major ? 1u : 0u) << 15)
           | ((b_mn_major ? 1u : 0u) << 16)
           | ((uint32_t)(N >> 3) << 17)
           | ((uint32_t)(M >> 4) << 24);
}

// Broadcast lane 0's value: tells the compiler the result is warp-uniform, so operands of the uniform-datapath
// instructions (UTCHMMA, UTCBAR, UTMALDG) built from it need no per-lane "waterfall" loop (ELECT / R2UR.BROADCAST /
// BRA.U.ANY around every instruction: ~150 cycles per tcgen05.mma, measured in profiles/r1c_c5.md).
__device__ __forceinline__ uint32_t uni(uint32_t v) { return __shfl_sync(0xffffffffu, v, 0); }
__device__ __forceinline__ int uni(int v) { return __shfl_sync(0xffffffffu, v, 0); }

__device__ __forceinline__ bool elect_one() {
    uint32_t pred;
    asm volatile(
        "{\n\t.reg .pred p;\n\telect.sync _|p, 0xffffffff;\n\tselp.u32 %0, 1, 0, p;\n\t}"
        : "=r"(pred));
    return pred != 0;
}

}  // namespace tropical
