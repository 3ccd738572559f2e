/*
 * tropical.h -- C-ABI boundary of the B200-native multiplexed-iteration hot path.
 *
 * What is computed (citations: P:n = /root/reference/PAPER.md line n; BJ = BASELINE.json):
 *   Tropical's SLO-aware multiplexing co-schedules, in ONE worker iteration, a prefill (chunk)
 *   with the running decode batch.  The iteration's attention over the
 *   paged KV cache and the KV append are inherited from the substrate and
 *   defined by BJ:north_star: append this step's K/V rows into the paged bf16 pool, then
 *   out = softmax(Q K^T / sqrt(d) + causal mask) V over the gathered pages, bf16 in,
 *   fp32 accumulate, bf16 out.  The execution-time predictor the scheduler needs (P:143,
 *   P:157) is tropical_step_cost.
 *
 * Notation: request i has q_i new tokens this step (1 = decode token, >= 2 = prefill chunk,
 * 0 = skipped), c_i tokens already cached, L_i = c_i + q_i.  T = sum_i q_i.
 * Query row t of request i sees keys j <= c_i + t (causal, bottom-right aligned; it sees
 * itself).  GQA: q head hq reads kv head hq / (Hq/Hkv).
 *
 * General conventions
 *   - All pointers marked [device] are CUDA device pointers, [host] are host pointers.
 *   - bf16 tensors are raw 16-bit patterns (void*), row-major in the stated shape.
 *   - The library owns nothing: it allocates no device memory, frees nothing and keeps no
 *     pointer after a call returns.  Process-global state: per-device cached attributes
 *     (SM count, one-time cudaFuncSetAttribute), the resolved cuTensorMapEncodeTiled entry
 *     point.  Any number of devices per process; calls act on the current device.
 *     One exception to "owns nothing": the module carries a fixed scratch array of
 *     TROPICAL_STATIC_WORKSPACE_BYTES for tropical_mixed_attention_static (see there).
 *   - Test and measurement hooks live in tropical_debug.h, not here.
 *   - Device work is enqueued on the caller's stream (void* = cudaStream_t, NULL = legacy
 *     default stream).  No host synchronisation, no H2D/D2H inside the device-pointer calls;
 *     they are CUDA-graph capturable.  tropical_step_host is the exception (see there).
 *   - Return value: tropical_status_t as int, never an exception or abort.  Host-visible
 *     argument errors are detected before any launch.  CONTENTS of device arrays cannot be
 *     validated without a sync: out-of-range page ids, q_offsets inconsistent with q_lens, or
 *     two requests writing the same (page, slot) in one step are UNDEFINED BEHAVIOUR.
 *     Read-sharing of prior-context pages between requests is allowed.
 *   - There is no CPU fallback.  Without a CUDA device every device call returns
 *     TROPICAL_ERR_CUDA.
 */
#ifndef TROPICAL_H_
#define TROPICAL_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef enum {
    TROPICAL_OK = 0,
    TROPICAL_ERR_INVALID_ARG = 1,  /* null pointer, negative size, Hq % Hkv != 0, stride too small */
    TROPICAL_ERR_UNSUPPORTED = 2,  /* head_dim not in {64,128}, page_size != 16, Hq/Hkv > 64 */
    TROPICAL_ERR_WORKSPACE = 3,    /* workspace NULL / misaligned (256 B) / smaller than tropical_workspace_bytes */
    TROPICAL_ERR_CUDA = 4,         /* launch or runtime failure; see tropical_last_cuda_error */
    TROPICAL_ERR_UNCALIBRATED = 5, /* tropical_step_cost: no coefficients for this head shape */
    TROPICAL_ERR_STATIC_CAPACITY = 6 /* tropical_mixed_attention_static: the step needs more scratch than the built-in array holds */
} tropical_status_t;

/* Paged KV pool, caller-owned.  Layout "HND": one (page, kv_head) is a contiguous
 * page_size x head_dim bf16 block (4 KiB at d = 128), so a page-head is one TMA box and the
 * append scatters 2*d-byte rows.  K and V are separate allocations, 256-byte aligned. */
typedef struct {
    int32_t num_q_heads;   /* Hq  */
    int32_t num_kv_heads;  /* Hkv, divides Hq */
    int32_t head_dim;      /* d in {64, 128} */
    int32_t page_size;     /* P = 16 */
    int32_t num_pages;     /* pool capacity in pages */
    void *k_pool;          /* [device] bf16 [num_pages][Hkv][P][d] */
    void *v_pool;          /* [device] bf16 [num_pages][Hkv][P][d] */
} tropical_kv_pool_t;

/* One multiplexed iteration.  Host scalars are used for validation, grid and
 * workspace sizing; per-request arrays live on the device so a step needs no sync. */
typedef struct {
    int32_t num_reqs;           /* >= 0 */
    int32_t total_q;            /* T == sum(q_lens): rows of q / out / k_new / v_new */
    int32_t max_kv_len;         /* >= max_i (ctx_lens[i] + q_lens[i]) */
    int32_t page_table_stride;  /* >= ceil(max_kv_len / P) */
    const int32_t *q_lens;      /* [device] [num_reqs]   new tokens: 1 decode, >= 2 prefill chunk, 0 skip */
    const int32_t *ctx_lens;    /* [device] [num_reqs]   tokens cached BEFORE this step (never mutated) */
    const int32_t *q_offsets;   /* [device] [num_reqs+1] exclusive prefix sum of q_lens */
    const int32_t *page_table;  /* [device] [num_reqs][page_table_stride]; entries past ceil(L_i/P) are ignored */
} tropical_batch_t;

/* Row A1 of SURVEY.md 8(a): for t < q_i, pos = c_i + t:
 *   k_pool[page_table[i][pos / P]][h][pos % P][:] = k_new[q_offsets[i] + t][h][:]  (same for V).
 * Bit copy, no floating point.  k_new / v_new: [device] bf16 [T][Hkv][d].  One launch. */
int tropical_kv_append(const tropical_kv_pool_t *pool, const tropical_batch_t *batch,
                       const void *k_new, const void *v_new, void *cuda_stream);

/* SURVEY.md 8(f) NEXT-4 "fuse RoPE+append": tropical_kv_append with rotary position embedding applied to the K rows on
 * their way into the pool (V rows are copied).  The paper says nothing about positional encoding; the convention is the
 * "rotate-half" one of its model family [DESIGN.md, readings]: for pos = c_i + t and channel c < d/2,
 *   k'[c]       = k[c] * cos[pos][c] - k[c + d/2] * sin[pos][c]
 *   k'[c + d/2] = k[c + d/2] * cos[pos][c] + k[c] * sin[pos][c]        (fp32 arithmetic, bf16 round-to-nearest-even)
 *   cos_table, sin_table [device] fp32 [table_len][d/2], 16-byte aligned, caller-owned (angles are the caller's: any
 *   base / scaling); table_len >= batch->max_kv_len, else INVALID_ARG.  One launch; same stream ordering as
 * tropical_kv_append.  Queries are rotated by the caller (the attention calls take q as given), and tropical_mixed_step
 * appends k_new as given: pass it rows that are already rotated, or use this call + tropical_mixed_attention. */
int tropical_kv_append_rope(const tropical_kv_pool_t *pool, const tropical_batch_t *batch,
                            const void *k_new, const void *v_new, const float *cos_table,
                            const float *sin_table, int32_t table_len, void *cuda_stream);

/* Row A2 as a standalone check / migration building block: dense copy-out of the first n_keys
 * keys of request req through the page table: k_dense, v_dense [device] bf16 [n_keys][Hkv][d]. */
int tropical_kv_gather(const tropical_kv_pool_t *pool, const tropical_batch_t *batch, int32_t req,
                       int32_t n_keys, void *k_dense, void *v_dense, void *cuda_stream);

/* KV migration of Path 1 (a request prefilled on a prefill worker re-enters through
 * the decode queue and its KV cache moves to the multiplexing worker that will decode it; "migration of
 * KVCache"; P:171 P2P between GPUs).  For every request m of the list, token j < kv_lens[m], kv head h:
 *   dst_pool[dst_page_table[m][j / P]][h][j % P][:] = src_pool[src_page_table[m][j / P]][h][j % P][:]   (K and V)
 * Gather through the source table and scatter under the destination table fused in one kernel (bulk-async copies
 * through shared memory; no dense staging buffer).  Bit copy.  Token-granular: slots >= kv_lens[m] of a destination
 * page and every other destination page keep their bits; the source pools are only read.
 *   src_pool, dst_pool: same num_kv_heads, head_dim, page_size (num_q_heads is ignored); num_pages may differ.
 *     The call runs on the CURRENT device, which must own src_pool; dst_pool may live on a peer device whose memory
 *     is mapped here (tropical_enable_peer_access, cudaDeviceEnablePeerAccess or a VMM mapping): the source GPU then
 *     pushes over NVLink.  The two pools must not overlap in the pages the tables name.
 *     STATUS OF THE PEER CASE: UNVERIFIED ON HARDWARE.  Every box this library has run on had one GPU, so bulk
 *     stores into peer-mapped memory have never been compared with the oracle; the comparison is armed
 *     (tests/test_gpu_migrate.py, the tests that need two GPUs) and runs on the first box that has them.
 *   Two requests of the list naming the same destination (page, slot) are undefined behaviour; page ids are not
 *   validated (device data).  Up to 1024 requests per launch; longer lists are split into several launches.
 * Returns INVALID_ARG for null pointers / negative sizes / strides smaller than ceil(max_kv_len / P) / mismatched pool
 * shapes, UNSUPPORTED for head_dim not in {64, 128} or page_size != 16. */
typedef struct {
    int32_t num_reqs;               /* >= 0 */
    int32_t max_kv_len;             /* >= max_m kv_lens[m]: grid sizing and stride validation */
    int32_t src_page_table_stride;  /* >= ceil(max_kv_len / P) */
    int32_t dst_page_table_stride;  /* >= ceil(max_kv_len / P) */
    const int32_t *kv_lens;         /* [device] [num_reqs] tokens to move per request */
    const int32_t *src_page_table;  /* [device] [num_reqs][src_page_table_stride] */
    const int32_t *dst_page_table;  /* [device] [num_reqs][dst_page_table_stride] */
} tropical_migration_t;

int tropical_kv_migrate(const tropical_kv_pool_t *src_pool, const tropical_kv_pool_t *dst_pool,
                        const tropical_migration_t *migration, void *cuda_stream);

/* Maps the memory of peer_device into the current device's address space (cudaDeviceEnablePeerAccess; "already
 * enabled" counts as success) so that a pool allocated there can be the dst_pool of tropical_kv_migrate.
 * TROPICAL_ERR_UNSUPPORTED when the two devices have no peer path. */
int tropical_enable_peer_access(int32_t peer_device);

/* Upper bound of the scratch tropical_mixed_attention needs for any batch with these host
 * scalars (work lists, split-K partials, tickets).  Returns 0 on invalid arguments. */
size_t tropical_workspace_bytes(const tropical_kv_pool_t *pool, int32_t num_reqs, int32_t total_q,
                                int32_t max_kv_len);

/* Rows A0, A2-A5: attention of every new token over its request's pages (which must already
 * contain this step's rows: call tropical_kv_append first on the same stream).
 *   q    [device] bf16 [T][Hq][d]      out [device] bf16 [T][Hq][d]
 *   lse  [device, nullable] fp32 [T][Hq], natural-log sum-exp of the scaled scores
 *   sm_scale <= 0 selects 1/sqrt(d)
 *   workspace [device] 256-byte aligned, >= tropical_workspace_bytes(...); contents are scratch.
 * Never writes the pool.  Unused slots of a request's last page may hold any bits (NaN
 * included); the result does not depend on them.  Run-to-run deterministic.
 * Stream ordering: the first of its two launches (the tile directory) opts into programmatic dependent launch so that
 * it overlaps a preceding tropical_kv_append; it waits for that kernel's completion before the step kernel starts.
 * A caller kernel placed right before this call that itself triggers dependents early
 * (griddepcontrol.launch_dependents / cudaTriggerProgrammaticLaunchCompletion) must have finished writing q_lens,
 * ctx_lens, q_offsets and page_table before it triggers. */
int tropical_mixed_attention(const tropical_kv_pool_t *pool, const tropical_batch_t *batch,
                             const void *q, void *out, float *lse, float sm_scale,
                             void *workspace, size_t workspace_bytes, void *cuda_stream);

/* tropical_mixed_attention for callers that cannot provide a workspace because they cannot allocate device memory.
 *
 * Who that is: tropical_mixed_attention wants 20-60 MB of scratch from its caller (work lists, tickets, split-K
 * partials).  A serving worker that handed every free byte of HBM to its KV pool at start-up (the cache is
 * sized to the memory watermark) has nothing left to cudaMalloc when a step arrives, and would not want to: cudaMalloc
 * and cudaFree synchronise the whole device, which stalls every stream of a loop that runs once per decode iteration.
 * The same holds for a host program that embeds this library under a "no allocation after initialisation" rule, or
 * that reaches it from a context where it may only enqueue work (its own allocator is not reachable from there).
 *
 * What it does: exactly what tropical_mixed_attention does -- same kernels, same arguments except that workspace and
 * workspace_bytes are gone, same results -- with the scratch taken from an array that is part of the library image
 * (a file-scope __device__ array, 256-byte aligned, TROPICAL_STATIC_WORKSPACE_BYTES long).  The call allocates
 * nothing and frees nothing: no cudaMalloc / cudaFree / cudaMallocAsync, no allocating library routine.  The caller
 * still owns and passes every input and output (pool, batch metadata, q, out, lse).
 *
 * Cost and limit: every GPU on which the library's module is loaded keeps the TROPICAL_STATIC_WORKSPACE_BYTES (64 MiB)
 * from module load until the process exits, whether this entry point is ever called or not.  A step whose
 * tropical_workspace_bytes(pool, num_reqs, total_q, max_kv_len) exceeds that is refused with
 * TROPICAL_ERR_STATIC_CAPACITY before anything is launched (tropical_last_cuda_error() then says how many bytes were
 * needed); nothing is truncated.  64 MiB covers all five BASELINE.json configs (C4, the largest, needs 58.4 MB); at
 * d = 128 it is roughly num_reqs * Hkv * ceil(Hq / Hkv / 8) <= 6000 with total_q of a few thousand.
 *
 * First call on a device: the array's device address is looked up then (cudaGetSymbolAddress, once per device, with
 * that device current, remembered afterwards), and the kernels' one-time attributes are set as in every entry point.
 * Make that first call during start-up, outside any stream capture; later calls only enqueue the two launches.
 *
 * One array per GPU, shared by every call and every stream: two calls of this entry point that can overlap on the
 * same GPU (different streams, or different host threads without stream ordering between them) race on it and give
 * wrong results.  Order them on one stream, or give the second caller tropical_mixed_attention with its own
 * workspace.  The array keeps whatever the last call left in it; nothing in it needs to start at zero, because the
 * tile-directory kernel rewrites the header, the ticket counters and the split-group counters of each step before
 * the step kernel reads them, so no clearing pass is enqueued. */
#define TROPICAL_STATIC_WORKSPACE_BYTES (64u << 20)
int tropical_mixed_attention_static(const tropical_kv_pool_t *pool, const tropical_batch_t *batch,
                                    const void *q, void *out, float *lse, float sm_scale,
                                    void *cuda_stream);

/* One multiplexed iteration in ONE call -- rows A0-A5 with the KV append (A1) included: the same results as
 * tropical_kv_append followed by tropical_mixed_attention (pool bit-identical afterwards, out / lse bit-identical to that
 * pair's).  The library chooses how from the host scalars of the batch:
 *   - prefill-dominated steps (total_q >= 64 * num_reqs, i.e. at most one decode request per ~64 prefill tokens): the
 *     FUSED variant of the step kernel, two launches.  Its attention roles read this step's K / V rows directly from
 *     k_new / v_new (TMA boxes over [T][Hkv][d]; a decode request's own new row is patched into the page-head it has just
 *     loaded) while otherwise idle warps of the same persistent kernel copy the rows into their (page, slot) of the pool
 *     -- the append leaves the critical path; nothing reads those slots from the pool during the step.  Since such steps
 *     leave the decode warps idle, the variant runs two softmax warpgroups and pairs MHA query tiles by rows.
 *   - other (decode-heavy) steps: the append kernel in front of the plain step kernel, three launches, exactly what the
 *     two separate calls enqueue (the fused variant's extra work in the decode loop costs more there than it saves).
 *   k_new, v_new [device] bf16 [T][Hkv][d], 16-byte aligned; every other argument as in tropical_mixed_attention.
 * The pool IS written (exactly the rows tropical_kv_append would write).  Idempotent, graph-capturable.  A preceding
 * kernel on the stream must have completed its writes of the batch metadata, k_new and v_new before it triggers
 * programmatic dependents, if it does (see tropical_mixed_attention). */
int tropical_mixed_step(const tropical_kv_pool_t *pool, const tropical_batch_t *batch, const void *q,
                        const void *k_new, const void *v_new, void *out, float *lse, float sm_scale,
                        void *workspace, size_t workspace_bytes, void *cuda_stream);

/* Opt-in debug check of the DEVICE-resident contents of a batch, which the other calls cannot validate without a
 * sync (out-of-range page ids there are undefined behaviour): q_lens / ctx_lens >= 0, q_offsets the exclusive prefix
 * sum of q_lens with q_offsets[num_reqs] == total_q, ctx + q <= max_kv_len, ceil((ctx + q) / page_size) <=
 * page_table_stride, every page id a request can touch in [0, num_pages).  Runs one small kernel and synchronises
 * the stream (so it is not graph-capturable).  scratch: [device] >= 4 bytes, 4-byte aligned, caller-owned (the first
 * bytes of the attention workspace will do); its contents are overwritten.  Returns TROPICAL_OK, or
 * TROPICAL_ERR_INVALID_ARG with *first_bad_request [host, nullable] = the lowest offending request index (num_reqs
 * when only the final q_offsets entry is wrong). */
int tropical_validate_batch(const tropical_kv_pool_t *pool, const tropical_batch_t *batch,
                            int32_t *first_bad_request, void *scratch, void *cuda_stream);

/* End-to-end step from HOST buffers (what bench.py's "e2e" times): copies this step's inputs
 * host->device into caller-provided device staging, runs append + attention, copies out back,
 * (the fused tropical_mixed_step), and synchronises the stream before returning.  The KV pool stays device resident (it is the
 * worker's cache).  Host buffers should be pinned for the copies to be async.
 *   staging [device] >= tropical_step_host_staging_bytes(...), 256-byte aligned.
 *   h_*: [host] same shapes as the device-pointer API.  h_lse nullable. */
typedef struct {
    int32_t num_reqs, total_q, max_kv_len, page_table_stride;
    const int32_t *q_lens, *ctx_lens, *q_offsets, *page_table; /* [host] */
} tropical_host_batch_t;

size_t tropical_step_host_staging_bytes(const tropical_kv_pool_t *pool, int32_t num_reqs,
                                        int32_t total_q, int32_t page_table_stride);

int tropical_step_host(const tropical_kv_pool_t *pool, const tropical_host_batch_t *batch,
                       const void *h_q, const void *h_k_new, const void *h_v_new, void *h_out,
                       float *h_lse, float sm_scale, void *staging, size_t staging_bytes,
                       void *workspace, size_t workspace_bytes, void *cuda_stream);

/* Row A6: predicted microseconds of append + attention for a batch ("predicted
 * execution time", "offline profiling tools", P:159 decode-batch time).  Pure host
 * code, reentrant.  Form:
 *   t = t0 + max(a*F, b*B) + kappa*min(a*F, b*B) + e_p*N_p/n_sm + e_d*N_d/n_sm + e_c*N_c
 * with F FLOPs, B algorithmic bytes, N_p prefill (128-row x head) tiles weighted by their KV
 * iterations, N_d decode page-head units, N_c the KV iterations of the heaviest prefill item (the critical path when a
 * step has about as many items as the GPU has SMs; an item is two heads of a kv group at the top row tile, or -- MHA /
 * odd groups -- the top row tile, or the top TWO row tiles in the fused variant of tropical_mixed_step).  model == NULL selects the built-in fit measured on
 * B200 for (Hq, Hkv, d), else TROPICAL_ERR_UNCALIBRATED. */
typedef struct {
    double t0_us, a_us_per_flop, b_us_per_byte, kappa, e_prefill_iter_us, e_decode_unit_us;
    double n_sm;
    double e_prefill_crit_us; /* e_c: per KV iteration of the heaviest prefill item */
} tropical_cost_model_t;

typedef struct {
    double flops;          /* 4*d*Hq*sum_i [q_i*c_i + q_i(q_i+1)/2]                         */
    double bytes;          /* KV read once + new rows r/w + Q/O + page table */
    double t_tc_us;        /* a * flops */
    double t_hbm_us;       /* b * bytes */
    int64_t prefill_tiles; /* sum over prefill requests of ceil(q_i/128) * Hq                */
    int64_t prefill_iters; /* 128x128 KV iterations over those tiles                          */
    int64_t decode_units;  /* decode page-head units: sum ceil(L_i/P) * Hkv                   */
    int64_t prefill_critical_iters; /* N_c: KV iterations of the heaviest prefill item       */
} tropical_cost_breakdown_t;

int tropical_step_cost(const tropical_cost_model_t *model, int32_t num_q_heads,
                       int32_t num_kv_heads, int32_t head_dim, int32_t page_size, int32_t num_reqs,
                       const int32_t *q_lens_host, const int32_t *ctx_lens_host, double *out_us,
                       tropical_cost_breakdown_t *breakdown /* nullable */);

/* predicted microseconds of a WHOLE model iteration on one GPU of a worker (the toggle
 * predicts "the execution time of a prefill request" and of the decoding batch with offline profiling; TP = 2
 * inside a worker).  Pure host code, reentrant.  Per layer, on one GPU of a tp-way tensor-parallel group:
 *   attention + KV append : tropical_step_cost on this GPU's head shard (Hq/tp, Hkv/tp, d) -- the path shards by kv head
 *                           with no collective;
 *   linear layers         : QKV [d_model x (Hq+2Hkv)d/tp], O [Hq d/tp x d_model], (gate and) up [d_model x (1 or 2)
 *                           d_ffn/tp], down [d_ffn/tp x d_model] as bf16 GEMMs over the T new tokens of the batch:
 *                             W = sum_j K_j N_j,  F = 2 T W,  B = 2 W + 2 T sum_j (K_j + N_j)
 *                             t_lin = g0 + max(f F, w B) + kappa min(f F, w B)
 *                           (weights streamed once per layer, activations in and out; same overlap form as the step);
 *   all-reduce (tp > 1)   : two per layer over T d_model bf16 values: 2 (ar0 + ar_b * 2 T d_model).
 *   total = num_layers * (attention + linear + all-reduce).
 * linear == NULL selects the built-in fit of `python -m paper_2606_16264_b200.cost_fit measure-gemm | fit` (library
 * GEMMs on a B200; its all-reduce coefficients are 0: one GPU is all that could be measured, DESIGN.md section 7;
 * `python -m paper_2606_16264_b200.cost_fit measure-allreduce` on a box with two GPUs, then `... cost_fit fit`, fills them in).
 * attn == NULL selects the built-in step model of the SHARD shape, else TROPICAL_ERR_UNCALIBRATED.  No norms, RoPE,
 * sampling or embedding: the form is this build's (parity unpinned, like row A6).
 * INVALID_ARG: null shape, non-positive sizes, tp not dividing num_kv_heads / d_ffn, and whatever tropical_step_cost
 * rejects. */
typedef struct {
    int32_t d_model;     /* hidden size */
    int32_t d_ffn;       /* FFN inner size */
    int32_t gated_mlp;   /* 1: gate, up and down projections; 0: up and down */
    int32_t num_layers;  /* >= 1 */
    int32_t tp;          /* tensor-parallel degree >= 1: heads and FFN columns split tp ways */
} tropical_layer_shape_t;

typedef struct {
    double g0_us;           /* fixed cost of a layer's four GEMM launches */
    double f_us_per_flop;   /* library-GEMM tensor throughput */
    double w_us_per_byte;   /* streaming of weights and activations */
    double kappa;           /* how imperfectly the two overlap, in [0, 1] */
    double ar0_us;          /* per all-reduce: latency */
    double ar_us_per_byte;  /* per all-reduce: per byte of the reduced tensor */
} tropical_linear_model_t;

typedef struct {
    double attn_us;       /* one layer: append + attention of this GPU's head shard */
    double linear_us;     /* one layer: the four GEMMs of this GPU's shard */
    double allreduce_us;  /* one layer: its two all-reduces (0 when tp == 1) */
    double gemm_flops;    /* F above */
    double gemm_bytes;    /* B above */
    double total_us;      /* num_layers * (attn_us + linear_us + allreduce_us) */
} tropical_iter_breakdown_t;

int tropical_iter_cost(const tropical_cost_model_t *attn /* nullable */, const tropical_linear_model_t *linear /* nullable */,
                       const tropical_layer_shape_t *shape, int32_t num_q_heads, int32_t num_kv_heads,
                       int32_t head_dim, int32_t page_size, int32_t num_reqs, const int32_t *q_lens_host,
                       const int32_t *ctx_lens_host, double *out_us /* nullable */,
                       tropical_iter_breakdown_t *breakdown /* nullable */);

/* Number of kernel launches the last tropical_kv_append / tropical_mixed_attention /
 * tropical_step_host call on this thread enqueued (bench.py's gpu_launches). */
int tropical_last_launch_count(void);

const char *tropical_status_string(int status);
const char *tropical_last_cuda_error(void); /* thread-local text of the last CUDA failure */
const char *tropical_version(void);

#ifdef __cplusplus
}
#endif
#endif /* TROPICAL_H_ */
