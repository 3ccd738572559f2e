// sim.cpp -- tropical_sim_run: discrete-event simulation of the Tropical multiplexing toggle and of the two
// serving styles it is compared with (include/tropical_sim.h holds the model, rule by rule, with its citations
// of PAPER.md section II-A, IV-B, IV-C).  Host code only; iteration times come from tropical_step_cost (row A6).
#include <math.h>
#include <stdint.h>

#include <algorithm>
#include <limits>
#include <vector>

#include "../../include/tropical_sim.h"

namespace {

const double kInf = std::numeric_limits<double>::infinity();

struct Req {
    double arrival;
    int prompt, output;
    int done_prompt = 0, generated = 0;
    double first_token = -1, finish = -1;
    int prefill_worker = -1, decode_worker = -1, multiplexed = 0;
};

struct Pending {
    double available_at;
    int rid;
};

struct Worker {
    std::vector<int> local_q, resident, it_decodes;
    std::vector<Pending> pending;
    double busy_until = kInf;  // kInf = idle
    int it_prefill = -1, it_chunk = 0;
};

struct Sim {
    const tropical_sim_config_t& cfg;
    std::vector<Req> R;
    std::vector<Worker> W;
    std::vector<int> toggle_q;
    std::vector<int32_t> q_buf, c_buf;
    std::vector<char> prefill_role;  // 1: dedicated prefill worker (policies 1, 2); may change under P:161
    int delayed = 0;                 // prefills dispatched by the no-starvation rule since the last transition
    int64_t to_multiplexing = 0, to_prefill = 0;
    double now = 0;
    int64_t iterations = 0;
    int status = TROPICAL_OK;

    explicit Sim(const tropical_sim_config_t& c) : cfg(c), prefill_role(c.num_workers, 0) {
        if (c.policy != TROPICAL_SIM_COLOCATED)
            for (int w = 0; w < c.num_prefill_workers; ++w) prefill_role[w] = 1;
    }

    bool is_prefill_worker(int w) const { return prefill_role[w] != 0; }
    int count_role(char role) const { return (int)std::count(prefill_role.begin(), prefill_role.end(), role); }
    int remaining_output(int r) const { return R[r].output - 1 - R[r].generated; }

    // duration of an iteration over the batch currently in q_buf / c_buf
    double iter_time() {
        // attn.n_sm <= 0: the library's built-in fits, one coefficient set per kernel variant of the step
        const tropical_cost_model_t* attn = cfg.attn.n_sm > 0 ? &cfg.attn : nullptr;
        if (cfg.layer.d_model > 0) {  // NEXT-4: whole-iteration predictor (attention on the head shard + GEMMs + all-reduce)
            double it = 0;
            const int rc = tropical_iter_cost(attn, &cfg.linear, &cfg.layer, cfg.num_q_heads, cfg.num_kv_heads,
                                              cfg.head_dim, cfg.page_size, (int32_t)q_buf.size(), q_buf.data(),
                                              c_buf.data(), &it, nullptr);
            if (rc != TROPICAL_OK) status = rc;
            return it + cfg.iter_overhead_us;
        }
        double us = 0;
        const int rc = tropical_step_cost(attn, cfg.num_q_heads, cfg.num_kv_heads, cfg.head_dim, cfg.page_size,
                                          (int32_t)q_buf.size(), q_buf.data(), c_buf.data(), &us, nullptr);
        if (rc != TROPICAL_OK) status = rc;
        long long tokens = 0;
        for (int32_t q : q_buf) tokens += q;
        return cfg.num_layers * us + cfg.linear_us_per_token * (double)tokens + cfg.iter_overhead_us;
    }
    void batch_clear() { q_buf.clear(); c_buf.clear(); }
    void batch_add(int q, int c) { q_buf.push_back(q); c_buf.push_back(c); }
    void batch_add_decodes(int w) {
        for (int r : W[w].resident) batch_add(1, R[r].prompt + R[r].generated);
    }

    long long unfinished_tokens(int w) const {
        long long t = 0;
        for (int r : W[w].local_q) t += (R[r].prompt - R[r].done_prompt) + remaining_output(r);
        for (int r : W[w].resident) t += remaining_output(r);
        for (const Pending& p : W[w].pending) t += remaining_output(p.rid);
        return t;
    }
    long long resident_kv(int w) const {
        long long t = 0;
        for (int r : W[w].local_q) t += R[r].done_prompt + R[r].generated;
        for (int r : W[w].resident) t += R[r].done_prompt + R[r].generated;
        for (const Pending& p : W[w].pending) t += R[p.rid].done_prompt + R[p.rid].generated;
        return t;
    }
    double pred_exec(int r) {  // the rest of r's prompt as one iteration of its own
        batch_clear();
        batch_add(R[r].prompt - R[r].done_prompt, R[r].done_prompt);
        return iter_time();
    }
    double pred_queue(int w) {  // P:157 "queuing time when scheduling to the local worker"
        double t = 0;
        size_t first = 0;
        if (W[w].busy_until != kInf) {
            t += W[w].busy_until - now;
            if (W[w].it_prefill >= 0) first = 1;
        }
        for (size_t i = first; i < W[w].local_q.size(); ++i) t += pred_exec(W[w].local_q[i]);
        return t;
    }
    int least_queue_prefill_worker() {
        int best = -1;
        double bq = kInf;
        for (int w = 0; w < cfg.num_workers; ++w) {
            if (!is_prefill_worker(w)) continue;
            const double q = pred_queue(w);
            if (best < 0 || q < bq) { bq = q; best = w; }
        }
        return best;
    }
    // worker with the fewest unfinished tokens among all workers (role < 0) or those of one role
    int fewest_unfinished(int role) const {
        int best = -1;
        long long bt = 0;
        for (int w = 0; w < cfg.num_workers; ++w) {
            if (role >= 0 && prefill_role[w] != role) continue;
            const long long t = unfinished_tokens(w);
            if (best < 0 || t < bt) { bt = t; best = w; }
        }
        return best;
    }

    void finish_iteration(int w) {
        Worker& wk = W[w];
        for (int r : wk.it_decodes) {
            if (++R[r].generated == R[r].output - 1) {
                R[r].finish = now;
                wk.resident.erase(std::find(wk.resident.begin(), wk.resident.end(), r));
            }
        }
        const int r = wk.it_prefill;
        if (r >= 0) {
            R[r].done_prompt += wk.it_chunk;
            if (R[r].done_prompt == R[r].prompt) {
                wk.local_q.erase(wk.local_q.begin());
                R[r].first_token = now;
                if (R[r].output == 1) {
                    R[r].finish = now;
                    R[r].decode_worker = w;
                } else if (is_prefill_worker(w)) {  // P:155 decode queue, P:186 dispatch, P:58 migration
                    const int best = fewest_unfinished(0);
                    W[best].pending.push_back({now + cfg.migrate_us_per_token * R[r].prompt, r});
                    R[r].decode_worker = best;
                } else {
                    wk.resident.push_back(r);
                    R[r].decode_worker = w;
                }
            }
        }
        wk.busy_until = kInf;
        wk.it_decodes.clear();
        wk.it_prefill = -1;
        wk.it_chunk = 0;
    }

    void try_start(int w) {
        Worker& wk = W[w];
        std::vector<Pending> still;
        for (const Pending& p : wk.pending) {  // migrated caches that have arrived join the batch
            if (p.available_at <= now) wk.resident.push_back(p.rid);
            else still.push_back(p);
        }
        wk.pending.swap(still);
        batch_clear();
        if (!wk.local_q.empty()) {
            const int r = wk.local_q[0];
            const int rest = R[r].prompt - R[r].done_prompt;
            const int chunk = (cfg.chunk_tokens <= 0 || is_prefill_worker(w)) ? rest : std::min(rest, cfg.chunk_tokens);
            wk.it_prefill = r;
            wk.it_chunk = chunk;
            batch_add(chunk, R[r].done_prompt);
        }
        wk.it_decodes = wk.resident;
        batch_add_decodes(w);
        if (q_buf.empty()) return;
        wk.busy_until = now + iter_time();
        ++iterations;
    }

    // P:161 role transitions [R]: readings in include/tropical_sim.h
    void role_transitions() {
        // prefill -> multiplexing: "when the watermark of all decode workers exceeds its threshold"
        bool all_above = true;
        for (int w = 0; w < cfg.num_workers; ++w)
            if (!is_prefill_worker(w) && !((double)resident_kv(w) > cfg.hbm_watermark * (double)cfg.kv_capacity_tokens))
                all_above = false;
        if (all_above && count_role(1) >= 2) {
            prefill_role[least_queue_prefill_worker()] = 0;
            ++to_multiplexing;
        }
        // multiplexing -> prefill: "if prefill frequently encounters delays"
        if (delayed >= cfg.delay_threshold && count_role(0) >= 2) {
            for (int w = 0; w < cfg.num_workers; ++w) {
                if (is_prefill_worker(w) || !W[w].resident.empty() || !W[w].pending.empty()) continue;
                prefill_role[w] = 1;
                ++to_prefill;
                delayed = 0;
                break;
            }
        }
    }

    void toggle_scan() {
        if (cfg.role_transitions) role_transitions();
        const std::vector<int> snapshot = toggle_q;
        for (int r : snapshot) {
            const double waited = now - R[r].arrival;
            int target = -1, mux = 0;
            // Path 2: multiplexing workers with an empty local queue, fewest unfinished tokens first
            std::vector<std::pair<long long, int>> cands;
            for (int w = 0; w < cfg.num_workers; ++w)
                if (!is_prefill_worker(w) && W[w].local_q.empty()) cands.push_back({unfinished_tokens(w), w});
            std::sort(cands.begin(), cands.end());
            for (const auto& cw : cands) {
                const int w = cw.second;
                const bool has_decodes = !W[w].resident.empty();
                double t_dec = 0;
                if (has_decodes) {
                    batch_clear();
                    batch_add_decodes(w);
                    t_dec = iter_time();
                    if (!(t_dec < cfg.decode_guard * cfg.tpot_slo_us)) continue;  // P:159 decode batch near the TPOT SLO
                }
                if ((double)(resident_kv(w) + R[r].prompt) > cfg.hbm_watermark * (double)cfg.kv_capacity_tokens) continue;  // P:159 HBM
                double slack = kInf;  // TPOT slack accumulated so far by the tightest resident request (Fig. 7)
                for (int x : W[w].resident)
                    slack = std::min(slack, (R[x].generated + 1) * cfg.tpot_slo_us - (now - R[x].first_token));
                double interference = 0;
                for (int done = 0; done < R[r].prompt;) {
                    const int rest = R[r].prompt - done;
                    const int chunk = cfg.chunk_tokens <= 0 ? rest : std::min(rest, cfg.chunk_tokens);
                    batch_clear();
                    batch_add(chunk, done);
                    batch_add_decodes(w);
                    interference += iter_time() - t_dec;
                    done += chunk;
                }
                if (interference <= slack) {  // P:143 predicted execution time within the slack
                    target = w;
                    mux = 1;
                    break;
                }
            }
            if (target < 0) {  // Path 1, or the no-starvation rule once the TTFT slack is gone
                const int best = least_queue_prefill_worker();
                const double slack_ttft = cfg.ttft_slo_us - waited;
                // the no-starvation rule fires on the very expression the wake-up below is scheduled with: testing
                // `slack_ttft <= 0` instead can miss it by one rounding of (now - arrival)
                const bool slack_gone = now >= R[r].arrival + cfg.ttft_slo_us;
                if (slack_gone) {
                    target = best;
                    ++delayed;  // a delayed prefill
                } else if (pred_exec(r) + pred_queue(best) < slack_ttft) {
                    target = best;
                }
            }
            if (target >= 0) {
                toggle_q.erase(std::find(toggle_q.begin(), toggle_q.end(), r));
                W[target].local_q.push_back(r);
                R[r].prefill_worker = target;
                R[r].multiplexed = mux;
            }
        }
    }

    void run() {
        size_t next_arrival = 0;
        for (;;) {
            for (int w = 0; w < cfg.num_workers; ++w)
                if (W[w].busy_until <= now) finish_iteration(w);
            while (next_arrival < R.size() && R[next_arrival].arrival <= now) {
                const int r = (int)next_arrival++;
                if (cfg.policy == TROPICAL_SIM_COLOCATED) {
                    const int w = fewest_unfinished(-1);
                    W[w].local_q.push_back(r);
                    R[r].prefill_worker = w;
                } else if (cfg.policy == TROPICAL_SIM_DISAGGREGATED) {
                    const int w = least_queue_prefill_worker();
                    W[w].local_q.push_back(r);
                    R[r].prefill_worker = w;
                } else {
                    toggle_q.push_back(r);
                }
            }
            if (cfg.policy == TROPICAL_SIM_MULTIPLEXED) toggle_scan();
            for (int w = 0; w < cfg.num_workers; ++w)
                if (W[w].busy_until == kInf) try_start(w);
            if (status != TROPICAL_OK) return;
            double nxt = kInf;
            if (next_arrival < R.size()) nxt = std::min(nxt, R[next_arrival].arrival);
            for (int w = 0; w < cfg.num_workers; ++w) {
                if (W[w].busy_until != kInf) nxt = std::min(nxt, W[w].busy_until);
                else
                    for (const Pending& p : W[w].pending) nxt = std::min(nxt, p.available_at);
            }
            for (int r : toggle_q)  // the moment the no-starvation rule applies
                if (R[r].arrival + cfg.ttft_slo_us > now) nxt = std::min(nxt, R[r].arrival + cfg.ttft_slo_us);
            if (nxt == kInf) return;
            now = nxt;
        }
    }
};

}  // namespace

extern "C" int tropical_sim_run(const tropical_sim_config_t* cfg, int32_t n, const tropical_sim_request_t* reqs,
                                tropical_sim_result_t* results, tropical_sim_summary_t* summary) {
    if (cfg == nullptr || n < 0 || (n > 0 && reqs == nullptr)) return TROPICAL_ERR_INVALID_ARG;
    if (cfg->policy < 0 || cfg->policy > 2 || cfg->num_workers < 1 || cfg->num_layers < 1) return TROPICAL_ERR_INVALID_ARG;
    if (cfg->policy != TROPICAL_SIM_COLOCATED &&
        (cfg->num_prefill_workers < 1 || cfg->num_prefill_workers >= cfg->num_workers))
        return TROPICAL_ERR_INVALID_ARG;
    if (!(cfg->ttft_slo_us > 0) || !(cfg->tpot_slo_us > 0) || cfg->chunk_tokens < 0 || cfg->migrate_us_per_token < 0)
        return TROPICAL_ERR_INVALID_ARG;
    if (cfg->role_transitions != 0 && (cfg->role_transitions != 1 || cfg->delay_threshold < 1)) return TROPICAL_ERR_INVALID_ARG;
    Sim S(*cfg);
    S.R.resize(n);
    for (int i = 0; i < n; ++i) {
        if (reqs[i].prompt_len < 1 || reqs[i].output_len < 1 || !(reqs[i].arrival_us >= 0)) return TROPICAL_ERR_INVALID_ARG;
        if (i > 0 && reqs[i].arrival_us < reqs[i - 1].arrival_us) return TROPICAL_ERR_INVALID_ARG;
        S.R[i].arrival = reqs[i].arrival_us;
        S.R[i].prompt = reqs[i].prompt_len;
        S.R[i].output = reqs[i].output_len;
    }
    S.W.resize(cfg->num_workers);
    S.run();
    if (S.status != TROPICAL_OK) return S.status;
    std::vector<double> ttft(n), tpot(n);
    double makespan = 0;
    int64_t ok = 0, mux = 0;
    for (int i = 0; i < n; ++i) {
        const Req& x = S.R[i];
        // a request the run never served (cannot happen under the model's rules; kept as a guard) violates both SLOs
        ttft[i] = x.first_token < 0 ? kInf : x.first_token - x.arrival;
        tpot[i] = x.finish < 0 ? kInf : (x.finish - x.first_token) / (double)std::max(1, x.output - 1);
        if (ttft[i] <= cfg->ttft_slo_us && tpot[i] <= cfg->tpot_slo_us) ++ok;  // eq. (1)-(3)
        mux += x.multiplexed;
        makespan = std::max(makespan, x.finish);
        if (results != nullptr) {
            results[i].ttft_us = ttft[i];
            results[i].tpot_us = tpot[i];
            results[i].first_token_us = x.first_token;
            results[i].finish_us = x.finish;
            results[i].prefill_worker = x.prefill_worker;
            results[i].decode_worker = x.decode_worker;
            results[i].multiplexed = x.multiplexed;
        }
    }
    if (summary != nullptr) {
        tropical_sim_summary_t s = {};
        if (n > 0) {
            double st = 0, sp = 0;
            for (int i = 0; i < n; ++i) { st += ttft[i]; sp += tpot[i]; }
            std::sort(ttft.begin(), ttft.end());
            std::sort(tpot.begin(), tpot.end());
            const int p90 = (int)ceil(0.9 * n) - 1;
            s.attainment = (double)ok / n;
            s.ttft_mean_us = st / n;
            s.ttft_p90_us = ttft[p90];
            s.tpot_mean_us = sp / n;
            s.tpot_p90_us = tpot[p90];
            s.makespan_us = makespan;
        }
        s.iterations = S.iterations;
        s.multiplexed_prefills = mux;
        s.to_multiplexing = S.to_multiplexing;
        s.to_prefill = S.to_prefill;
        *summary = s;
    }
    return TROPICAL_OK;
}
