/* tropical_sim.h -- SURVEY.md 8(f) NEXT-1: the paper's scheduler on top of the step-cost model.
 *
 * A deterministic discrete-event simulation of a pool of workers fed by the Tropical "multiplexing toggle"
 * (section IV) and of the two serving styles the paper compares against
 * (non-disaggregated; disaggregated).  Pure host code, reentrant, no GPU.  Iteration times
 * come from tropical_step_cost (row A6): this is what that prediction is for.
 *
 * MODEL (every rule cites the passage it restates; readings the paper leaves open are marked [R] and listed in
 * DESIGN.md section 9):
 *  - Request r = (arrival, prompt_len, output_len).  Its prefill produces the first token; the
 *    remaining output_len - 1 tokens are produced one per decode iteration of the worker that holds its KV cache.
 *  - Worker iteration: at its start it takes every resident decode request (1 token each)
 *    and, if its local prefill queue is not empty, the head request's next chunk (chunk_tokens > 0: at most that
 *    many prompt tokens; 0: the whole rest of the prompt).  Prefill workers of the disaggregated and
 *    multiplexed policies never chunk [R].  Duration = num_layers * step_cost(batch) + linear_us_per_token * new
 *    tokens + iter_overhead_us, with step_cost = tropical_step_cost(attn model) on (q_lens, ctx_lens) of the batch.
 *    A worker with nothing to run is idle; it is re-examined at every event.
 *  - TTFT_r = (end of the iteration that finishes r's prompt) - arrival.  TPOT_r = (finish - first token) /
 *    max(1, output_len - 1): total time spent generating divided by tokens generated, wall clock, so it contains
 *    interference and KV migration [R].  Attainment A = |{r: TTFT_r <= TTFT_SLO and TPOT_r <= TPOT_SLO}|
 *    / |R| (eq. 1-3; the denominator printed as R is read as |R|).
 *  - COLOCATED (non-disaggregated): an arriving request goes at once to the worker with the fewest unfinished
 *    tokens (remaining prompt + remaining output of everything it holds) and decodes where it prefilled.
 *  - DISAGGREGATED: workers [0, num_prefill_workers) only prefill (FIFO, one whole prompt per iteration); an
 *    arriving request goes to the prefill worker with the least predicted queue time; after its prefill the KV
 *    cache migrates (migrate_us_per_token * prompt_len) to the decode worker with the fewest
 *    unfinished tokens, which it joins at the first iteration that starts after the migration.
 *  - MULTIPLEXED (Tropical): workers [0, num_prefill_workers) are prefill workers, the others multiplexing
 *    workers.  Arrivals enter the toggle's prefill queue.  At every event the queue is scanned in FIFO
 *    order and each request is dispatched if a competent worker exists, else it stays queued:
 *      Path 2: multiplexing workers with an empty local prefill queue, fewest unfinished
 *        tokens first.  Competent iff (a) t_dec < decode_guard * TPOT_SLO, t_dec = predicted decode-only iteration
 *        of its resident batch (0 if none) -- "will not route ... when the execution time of the decoding batch is
 *        approaching the preset TPOT SLO"; (b) resident KV tokens + prompt_len <= hbm_watermark *
 *        kv_capacity_tokens -- "will not select a multiplexing worker if the HBM usage ... exceeds the threshold";
 *        (c) predicted interference sum over the request's chunks of (t(decodes + chunk_k) - t_dec) <= slack, where
 *        slack = min over resident decode requests of (tokens generated so far + 1) * TPOT_SLO - (now - first
 *        token time) -- the TPOT slack accumulated so far (Fig. 7), +inf for an empty worker [R].
 *      Path 1: prefill workers, least predicted queue time first.  Competent iff predicted execution
 *        + predicted queue time < TTFT_SLO - (now - arrival) -- "only when the addition of the predicted execution
 *        time and the predicted queuing time ... is less than the available slack to TTFT SLO".
 *      A request whose TTFT slack is already <= 0 goes to the prefill worker with the least predicted queue time
 *        (it cannot meet its SLO any more; it must not starve) [R].
 *    After a Path-1 prefill the request is placed like a disaggregated one (decode queue -> multiplexing worker with
 *    the fewest unfinished tokens, with migration).
 *  - Role transitions (role_transitions = 1, MULTIPLEXED only), checked at the start of every toggle scan [R]:
 *      prefill -> multiplexing: "when the watermark of all decode workers exceeds its threshold ... prefill workers can
 *        be directly assigned as multiplexing workers": if every multiplexing worker holds more than hbm_watermark *
 *        kv_capacity_tokens KV tokens and at least two prefill workers exist (one must remain for Path 1), the prefill
 *        worker with the least predicted queue time becomes a multiplexing worker on the spot: it keeps its local queue
 *        and the requests it finishes prefilling from then on stay resident on it.
 *      multiplexing -> prefill: "if prefill frequently encounters delays ... a transition from multiplexing workers
 *        back to prefill workers": a delayed prefill is one dispatched by the no-starvation rule; once delay_threshold
 *        of them have occurred since the last such transition and at least two multiplexing workers exist, the lowest-
 *        indexed multiplexing worker with no resident and no arriving decode request becomes a prefill worker (if none
 *        is free of decode state the transition waits); the counter restarts.
 *      At most one transition of each direction per scan; with role_transitions = 0 roles are fixed by index.
 *  - Determinism: events are processed in time order, ties by worker index, then by request index.
 */
#ifndef TROPICAL_SIM_H_
#define TROPICAL_SIM_H_

#include <stdint.h>

#include "tropical.h"

#ifdef __cplusplus
extern "C" {
#endif

typedef enum {
    TROPICAL_SIM_COLOCATED = 0,
    TROPICAL_SIM_DISAGGREGATED = 1,
    TROPICAL_SIM_MULTIPLEXED = 2
} tropical_sim_policy_t;

typedef struct {
    double arrival_us;
    int32_t prompt_len; /* >= 1 */
    int32_t output_len; /* >= 1, the first token included */
} tropical_sim_request_t;

typedef struct {
    int32_t policy;              /* tropical_sim_policy_t */
    int32_t num_workers;         /* >= 1 */
    int32_t num_prefill_workers; /* policies 1, 2: in [1, num_workers - 1]; ignored by policy 0 */
    int32_t chunk_tokens;        /* chunked prefill on colocated / multiplexing workers; 0 = whole prompt */
    double ttft_slo_us, tpot_slo_us;
    double decode_guard;         /* Path 2 refused when t_dec >= decode_guard * tpot_slo_us */
    double hbm_watermark;        /* Path 2 refused above this fraction of kv_capacity_tokens */
    int64_t kv_capacity_tokens;  /* per worker */
    double migrate_us_per_token; /* KV migration between workers */
    int32_t num_q_heads, num_kv_heads, head_dim, page_size, num_layers;
    tropical_cost_model_t attn;  /* coefficients of tropical_step_cost for one layer's append + attention; n_sm <= 0:
                                  * the built-in B200 fits (one set per kernel variant of the step), UNCALIBRATED if none */
    double linear_us_per_token;  /* the rest of an iteration, linear in its new tokens */
    double iter_overhead_us;
    /* NEXT-4: with layer.d_model > 0 an iteration lasts tropical_iter_cost(&attn, &linear, &layer, heads, batch) +
     * iter_overhead_us (attn then holds the coefficients of the head SHARD Hq/tp, Hkv/tp), and num_layers /
     * linear_us_per_token above are ignored. */
    tropical_layer_shape_t layer;
    tropical_linear_model_t linear;
    int32_t role_transitions;    /* 1: P:161 role transitions on (policy 2); 0: roles fixed by index */
    int32_t delay_threshold;     /* >= 1 when role_transitions: delayed prefills that trigger multiplexing -> prefill */
} tropical_sim_config_t;

typedef struct {
    double ttft_us, tpot_us, first_token_us, finish_us;
    int32_t prefill_worker, decode_worker;
    int32_t multiplexed; /* 1: its prefill ran on a multiplexing worker (Path 2) */
} tropical_sim_result_t;

typedef struct {
    double attainment;                 /* eq. (3) */
    double ttft_mean_us, ttft_p90_us;  /* P:173 metrics; p90 = value at index ceil(0.9 n) - 1 of the sorted list */
    double tpot_mean_us, tpot_p90_us;
    double makespan_us;
    int64_t iterations;
    int64_t multiplexed_prefills;
    int64_t to_multiplexing, to_prefill; /* role transitions performed */
} tropical_sim_summary_t;

/* Runs the simulation.  requests [host] must be sorted by arrival_us (ties keep their order); results [host,
 * nullable] receives one entry per request; summary [host, nullable].  Returns TROPICAL_OK,
 * TROPICAL_ERR_INVALID_ARG (null / unsorted / out-of-range arguments) or the status of tropical_step_cost. */
int tropical_sim_run(const tropical_sim_config_t *config, int32_t num_requests,
                     const tropical_sim_request_t *requests, tropical_sim_result_t *results,
                     tropical_sim_summary_t *summary);

#ifdef __cplusplus
}
#endif
#endif /* TROPICAL_SIM_H_ */
