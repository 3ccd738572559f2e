// kv_migrate.cu -- SURVEY.md 8(f) NEXT-3: KV migration of Path 1 (a request prefilled on a prefill worker
// re-enters through the decode queue and its KV cache moves to the multiplexing worker that decodes it
// "migration of KVCache"; P:171 P2P between GPUs).
//
//   for request m, j < kv_lens[m], h < Hkv:
//       dst_pool[dst_pt[m][j / 16]][h][j % 16][:] = src_pool[src_pt[m][j / 16]][h][j % 16][:]      (K and V)
//
// Gather through the source page table and scatter under the destination page table in ONE kernel, no dense staging
// buffer in HBM.  In the HND pool a page (all kv heads) is one contiguous run of Hkv * 16 * d * 2 bytes in both pools,
// so the move is a list of contiguous block copies: unit = (request, page, head group, K|V), <= 16 KiB.  A unit of a
// full page is ONE bulk-async copy global -> shared memory (TMA, mbarrier complete_tx) and ONE bulk-async copy shared
// memory -> global; the ragged last page of a request moves only its valid slots (one copy per head).  One warp per
// CTA drives a 4-stage ring with one elected lane; the lanes look up the page ids of 32 units at a time.  HBM-bound:
// 2 * 2 * Hkv * d * 2 bytes per token (read + write, K + V); the destination may be peer memory (NVLink), then the
// source GPU reads its HBM and pushes over the link.
#include <atomic>

#include "common.cuh"
#include "kernels.h"

namespace tropical {

constexpr int kMigStages = 4;
constexpr int kMigStageBytes = 16384;
constexpr int kMigLag = 2;            // units between the load and the store of a stage
constexpr int kMigMaxReqs = 1024;     // per launch (the launcher chunks longer lists)
constexpr int kMigSmem = kMigStages * kMigStageBytes + 1024;

__device__ __forceinline__ void bulk_load(uint32_t dst_s, const void* src, uint32_t bytes, uint32_t bar_s) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                 ::"r"(dst_s), "l"(src), "r"(bytes), "r"(bar_s) : "memory");
}
__device__ __forceinline__ void bulk_store(void* dst, uint32_t src_s, uint32_t bytes) {
    asm volatile("cp.async.bulk.global.shared::cta.bulk_group [%0], [%1], %2;" ::"l"(dst), "r"(src_s), "r"(bytes) : "memory");
}
__device__ __forceinline__ void bulk_commit() { asm volatile("cp.async.bulk.commit_group;" ::: "memory"); }
template <int N>
__device__ __forceinline__ void bulk_wait_read() { asm volatile("cp.async.bulk.wait_group.read %0;" ::"n"(N) : "memory"); }
__device__ __forceinline__ void bulk_wait_all() { asm volatile("cp.async.bulk.wait_group 0;" ::: "memory"); }

template <int D>
__global__ void __launch_bounds__(32) kv_migrate_kernel(MigrateArgs A) {
    constexpr int ROW = D * 2;                       // bytes of one (slot, head) row
    constexpr int PH = kPageSize * ROW;              // bytes of one page-head
    constexpr int HG = kMigStageBytes / PH;          // kv heads per unit
    extern __shared__ uint8_t smem_raw[];
    uint8_t* stages = reinterpret_cast<uint8_t*>((reinterpret_cast<uintptr_t>(smem_raw) + 127) & ~uintptr_t(127));
    __shared__ uint64_t full[kMigStages];
    __shared__ int s_base[kMigMaxReqs + 1];          // exclusive prefix sum of units per request
    const int lane = threadIdx.x;
    const int n = A.num_reqs;
    const int groups = (A.Hkv + HG - 1) / HG;
    const int upp = groups * 2;                      // units per page

    if (lane == 0) {
        for (int s = 0; s < kMigStages; ++s) mbar_init(&full[s], 1);
        fence_mbar_init();
    }
    {   // units per request -> exclusive scan (32 lanes, each a contiguous run of requests)
        const int per = (n + 31) / 32;
        const int i0 = lane * per, i1 = min(n, i0 + per);
        int mine = 0;
        for (int i = i0; i < i1; ++i) mine += ((__ldg(A.kv_lens + i) + kPageSize - 1) / kPageSize) * upp;
        int incl = mine;
#pragma unroll
        for (int off = 1; off < 32; off <<= 1) {
            const int v = __shfl_up_sync(0xffffffffu, incl, off);
            if (lane >= off) incl += v;
        }
        int run = incl - mine;
        for (int i = i0; i < i1; ++i) {
            s_base[i] = run;
            run += ((__ldg(A.kv_lens + i) + kPageSize - 1) / kPageSize) * upp;
        }
        if (lane == 31) s_base[n] = incl;
    }
    __syncwarp();
    const int total = s_base[n];
    const uint32_t stage_s = uni(smem_u32(stages));
    const uint32_t full_s = uni(smem_u32(full));

    // This CTA's units: rounds of 32 consecutive units, round r = blockIdx.x + r * gridDim.x.  Unit k of the CTA's own
    // sequence uses stage k % kMigStages; its store is issued kMigLag units after its load.
    long long k = 0;                                  // units loaded so far by this CTA
    // destination of the unit a stage holds (written by the elected lane at load time, read by it at store time)
    __shared__ long long s_dst[kMigStages];
    __shared__ int s_nh[kMigStages], s_rowbytes[kMigStages];

    auto store_unit = [&](long long j) {  // unit j of this CTA's sequence: stage j % kMigStages -> destination pool
        const int st = (int)(j % kMigStages);
        mbar_wait(&full[st], (uint32_t)((j / kMigStages) & 1), 301);
        if (elect_one()) {
            fence_proxy_async();
            const uint32_t src = stage_s + st * kMigStageBytes;
            uint8_t* dst = reinterpret_cast<uint8_t*>(s_dst[st]);
            const int nh_u = s_nh[st], rb = s_rowbytes[st];
            if (rb == PH) {
                bulk_store(dst, src, (uint32_t)(nh_u * PH));
            } else {
                for (int hh = 0; hh < nh_u; ++hh) bulk_store(dst + (size_t)hh * PH, src + hh * PH, (uint32_t)rb);
            }
            bulk_commit();
        }
        __syncwarp();
    };

    for (long long base = (long long)blockIdx.x * 32; base < total; base += (long long)gridDim.x * 32) {
        // lane -> unit base + lane: request (binary search over the prefix sums), page, head group, K|V, page ids
        const int u = (int)min((long long)total - 1, base + lane);
        int lo = 0, hi = n;
        while (hi - lo > 1) {
            const int mid = (lo + hi) >> 1;
            if (s_base[mid] <= u) lo = mid; else hi = mid;
        }
        const int m = lo, local = u - s_base[m];
        const int p = local / upp, r = local % upp;
        const int which = r & 1, h0 = (r >> 1) * HG;
        const int nh = min(HG, A.Hkv - h0);
        const int nvalid = min(kPageSize, __ldg(A.kv_lens + m) - p * kPageSize);
        const long long sp = __ldg(A.src_pt + (size_t)m * A.src_stride + p);
        const long long dp = __ldg(A.dst_pt + (size_t)m * A.dst_stride + p);
        const long long src_off = ((sp * A.Hkv + h0) * kPageSize) * (long long)ROW;
        const long long dst_off = ((dp * A.Hkv + h0) * kPageSize) * (long long)ROW;
        const long long l_src = (long long)(which ? A.v_src : A.k_src) + src_off;
        const long long l_dst = (long long)(which ? A.v_dst : A.k_dst) + dst_off;
        const int cnt = (int)min(32LL, (long long)total - base);

        for (int i = 0; i < cnt; ++i) {
            const long long u_src = __shfl_sync(0xffffffffu, l_src, i);
            const long long u_dst = __shfl_sync(0xffffffffu, l_dst, i);
            const int u_nh = __shfl_sync(0xffffffffu, nh, i);
            const int u_nv = __shfl_sync(0xffffffffu, nvalid, i);
            const int st = (int)(k % kMigStages);
            const int rowbytes = u_nv * ROW;                          // == PH for a full page
            const int bytes = u_nh * rowbytes;
            // the store that last read this stage (unit k - kMigStages) must be done reading: at most
            // kMigStages - kMigLag - 1 younger store groups may still be pending
            if (elect_one()) {
                bulk_wait_read<kMigStages - kMigLag - 1>();
                const uint32_t dst_s = stage_s + st * kMigStageBytes, bar = full_s + st * 8;
                asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"((uint32_t)bytes) : "memory");
                const uint8_t* src = reinterpret_cast<const uint8_t*>(u_src);
                s_dst[st] = u_dst; s_nh[st] = u_nh; s_rowbytes[st] = rowbytes;
                if (rowbytes == PH) {
                    bulk_load(dst_s, src, (uint32_t)bytes, bar);
                } else {
                    for (int hh = 0; hh < u_nh; ++hh) bulk_load(dst_s + hh * PH, src + (size_t)hh * PH, (uint32_t)rowbytes, bar);
                }
            }
            __syncwarp();
            ++k;
            if (k > kMigLag) store_unit(k - 1 - kMigLag);
        }
    }
    for (long long j = (k > kMigLag ? k - kMigLag : 0); j < k; ++j) store_unit(j);
    if (elect_one()) bulk_wait_all();  // shared memory must outlive the reads of the last stores
    __syncwarp();
}

cudaError_t launch_kv_migrate(const MigrateArgs& args, int max_kv_len, cudaStream_t stream, int* launches) {
    static std::atomic<int> attr_set[64];
    int dev = 0;
    cudaGetDevice(&dev);
    if (dev < 0 || dev >= 64) dev = 0;
    const int bit = args.D == 128 ? 1 : 2;
    if (!(attr_set[dev].load(std::memory_order_acquire) & bit)) {
        cudaError_t e = args.D == 128
            ? cudaFuncSetAttribute(kv_migrate_kernel<128>, cudaFuncAttributeMaxDynamicSharedMemorySize, kMigSmem)
            : cudaFuncSetAttribute(kv_migrate_kernel<64>, cudaFuncAttributeMaxDynamicSharedMemorySize, kMigSmem);
        if (e != cudaSuccess) return e;
        attr_set[dev].fetch_or(bit, std::memory_order_release);
    }
    int sms = 0;
    if (cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess || sms <= 0) sms = 148;
    const int ph = kPageSize * args.D * 2, hg = kMigStageBytes / ph;
    const int upp = ((args.Hkv + hg - 1) / hg) * 2;
    for (int r0 = 0; r0 < args.num_reqs; r0 += kMigMaxReqs) {
        MigrateArgs a = args;
        a.num_reqs = args.num_reqs - r0 < kMigMaxReqs ? args.num_reqs - r0 : kMigMaxReqs;
        a.kv_lens = args.kv_lens + r0;
        a.src_pt = args.src_pt + (size_t)r0 * args.src_stride;
        a.dst_pt = args.dst_pt + (size_t)r0 * args.dst_stride;
        // upper bound of the units of this launch (device lengths are not read on the host): 3 CTAs per SM at most
        const long long max_units = (long long)a.num_reqs * ((max_kv_len + kPageSize - 1) / kPageSize) * upp;
        long long grid = (max_units + 31) / 32;
        if (grid > 3LL * sms) grid = 3LL * sms;
        if (grid < 1) grid = 1;
        if (args.D == 128) kv_migrate_kernel<128><<<(int)grid, 32, kMigSmem, stream>>>(a);
        else kv_migrate_kernel<64><<<(int)grid, 32, kMigSmem, stream>>>(a);
        cudaError_t e = cudaGetLastError();
        if (e != cudaSuccess) return e;
        ++*launches;
    }
    return cudaSuccess;
}

}  // namespace tropical
