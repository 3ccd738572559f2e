// step_cost.cpp -- SURVEY.md 8(a) row A6: host-side execution-time prediction for one
// multiplexed iteration (PAPER.md:143 "predicted execution time", :157 "offline profiling
// tools", :159 predicted decode-batch time).  The paper gives no functional form; the form
// below is this build's (parity unpinned).  Pure host code.
#include <math.h>
#include <stdint.h>

#include "../../include/tropical.h"
#include "step_variant.h"

namespace {

// One coefficient set per head shape and kernel variant of the step: tropical_mixed_step runs prefill-dominated steps
// (at least kFusedMinTokensPerReq new tokens per request on average, csrc/step_variant.h) through its fused variant -- append
// inside, two softmax warpgroups -- whose prefill role is up to 35 % faster; one closed form cannot follow that switch.
struct BuiltinFit {
    int Hq, Hkv, d, fused;
    tropical_cost_model_t m;
};

// Coefficients fitted to measured step times by `python -m paper_2606_16264_b200.cost_fit fit` from the grid
// that `... cost_fit measure` wrote on a B200 (calibration/b200_grid.csv; provenance in DESIGN.md section 7).
const BuiltinFit kBuiltin[] = {
    {0, 0, 0, 0, {0, 0, 0, 0, 0, 0, 148, 0}},  // sentinel: never matches
#include "cost_model_fit.inc"
};

// Coefficients of the linear layers (NEXT-4), fitted by `cost_fit fit` to calibration/b200_gemm.csv.
const tropical_linear_model_t kBuiltinLinear =
#include "linear_model_fit.inc"
    ;

// fused: the step runs through the fused kernel variant (tropical_mixed_step's rule), whose MHA items are row pairs
void features(int Hq, int Hkv, int d, int P, int n, const int32_t* q, const int32_t* c, bool fused,
              tropical_cost_breakdown_t* f) {
    double qc = 0, pages = 0, T = 0, csum = 0;
    int64_t tiles = 0, iters = 0, units = 0, crit = 0;
    const bool head_pairs = (Hq / Hkv) % 2 == 0;  // two heads of a kv group per prefill item (csrc/plan.cuh)
    for (int i = 0; i < n; ++i) {
        const double qi = q[i], ci = c[i];
        if (q[i] <= 0) continue;
        qc += qi * ci + qi * (qi + 1) / 2;
        T += qi;
        csum += ci;
        const int64_t L = (int64_t)q[i] + c[i];
        pages += (double)((L + P - 1) / P);
        if (q[i] == 1) {
            units += ((L + P - 1) / P) * Hkv;
        } else {
            const int nt = (q[i] + 127) / 128;
            tiles += (int64_t)nt * Hq;
            int64_t kv_top = 0, kv_below = 0;  // KV tiles of the last row tile and of the one before it
            for (int ti = 0; ti < nt; ++ti) {
                const int64_t last = (int64_t)c[i] + ((ti + 1) * 128 < q[i] ? (ti + 1) * 128 : q[i]);
                iters += ((last + 127) / 128) * Hq;
                kv_below = kv_top;
                kv_top = (last + 127) / 128;
            }
            // the heaviest item of this request: two heads at the top tile, or (fused variant, MHA) the top two row
            // tiles of one head, or the top tile alone
            const int64_t item = head_pairs ? 2 * kv_top : (fused ? kv_top + kv_below : kv_top);
            if (item > crit) crit = item;
        }
    }
    f->flops = 4.0 * d * Hq * qc;
    f->bytes = 2.0 * 2 * Hkv * d * csum + 2.0 * (2.0 * 2 * Hkv * d * T) + 2.0 * (2.0 * Hq * d * T) + 4.0 * pages;
    f->prefill_tiles = tiles;
    f->prefill_iters = iters;
    f->decode_units = units;
    f->prefill_critical_iters = crit;
    f->t_tc_us = 0;
    f->t_hbm_us = 0;
}

}  // namespace

extern "C" int tropical_step_cost(const tropical_cost_model_t* model, int32_t Hq, int32_t Hkv, int32_t d,
                                  int32_t P, int32_t num_reqs, const int32_t* q_lens, const int32_t* ctx_lens,
                                  double* out_us, tropical_cost_breakdown_t* breakdown) {
    if (Hq <= 0 || Hkv <= 0 || d <= 0 || P <= 0 || num_reqs < 0 || Hq % Hkv != 0) return TROPICAL_ERR_INVALID_ARG;
    if (num_reqs > 0 && (q_lens == nullptr || ctx_lens == nullptr)) return TROPICAL_ERR_INVALID_ARG;
    if (out_us == nullptr && breakdown == nullptr) return TROPICAL_ERR_INVALID_ARG;
    for (int i = 0; i < num_reqs; ++i)
        if (q_lens[i] < 0 || ctx_lens[i] < 0) return TROPICAL_ERR_INVALID_ARG;
    long long T = 0;
    for (int i = 0; i < num_reqs; ++i) T += q_lens[i];
    const int fused = tropical::step_is_prefill_dominated(T, num_reqs) ? 1 : 0;
    tropical_cost_breakdown_t f;
    features(Hq, Hkv, d, P, num_reqs, q_lens, ctx_lens, fused != 0, &f);
    if (model == nullptr) {
        for (const BuiltinFit& b : kBuiltin)
            if (b.Hq == Hq && b.Hkv == Hkv && b.d == d && b.fused == fused) model = &b.m;
    }
    if (model != nullptr) {
        f.t_tc_us = model->a_us_per_flop * f.flops;
        f.t_hbm_us = model->b_us_per_byte * f.bytes;
    }
    if (breakdown != nullptr) *breakdown = f;
    if (model == nullptr) return out_us ? TROPICAL_ERR_UNCALIBRATED : TROPICAL_OK;
    if (out_us != nullptr) {
        const double hi = f.t_tc_us > f.t_hbm_us ? f.t_tc_us : f.t_hbm_us;
        const double lo = f.t_tc_us > f.t_hbm_us ? f.t_hbm_us : f.t_tc_us;
        const double nsm = model->n_sm > 0 ? model->n_sm : 148.0;
        *out_us = model->t0_us + hi + model->kappa * lo + model->e_prefill_iter_us * (double)f.prefill_iters / nsm +
                  model->e_decode_unit_us * (double)f.decode_units / nsm +
                  model->e_prefill_crit_us * (double)f.prefill_critical_iters;
    }
    return TROPICAL_OK;
}

extern "C" int tropical_iter_cost(const tropical_cost_model_t* attn, const tropical_linear_model_t* linear,
                                  const tropical_layer_shape_t* shape, int32_t Hq, int32_t Hkv, int32_t d, int32_t P,
                                  int32_t num_reqs, const int32_t* q_lens, const int32_t* ctx_lens, double* out_us,
                                  tropical_iter_breakdown_t* breakdown) {
    if (shape == nullptr || (out_us == nullptr && breakdown == nullptr)) return TROPICAL_ERR_INVALID_ARG;
    if (shape->d_model <= 0 || shape->d_ffn <= 0 || shape->num_layers < 1 || shape->tp < 1) return TROPICAL_ERR_INVALID_ARG;
    if (Hq <= 0 || Hkv <= 0 || d <= 0 || Hq % Hkv != 0) return TROPICAL_ERR_INVALID_ARG;
    const int tp = shape->tp;
    if (Hkv % tp != 0 || shape->d_ffn % tp != 0) return TROPICAL_ERR_INVALID_ARG;
    double attn_us = 0;
    const int rc = tropical_step_cost(attn, Hq / tp, Hkv / tp, d, P, num_reqs, q_lens, ctx_lens, &attn_us, nullptr);
    if (rc != TROPICAL_OK) return rc;
    if (linear == nullptr) linear = &kBuiltinLinear;
    double T = 0;
    for (int i = 0; i < num_reqs; ++i) T += q_lens[i];
    // (K, N) of the four weight matrices this GPU holds
    const double mats[4][2] = {{(double)shape->d_model, (double)(Hq + 2 * Hkv) * d / tp},
                               {(double)Hq * d / tp, (double)shape->d_model},
                               {(double)shape->d_model, (shape->gated_mlp ? 2.0 : 1.0) * shape->d_ffn / tp},
                               {(double)shape->d_ffn / tp, (double)shape->d_model}};
    double W = 0, act = 0;
    for (const auto& m : mats) {
        W += m[0] * m[1];
        act += m[0] + m[1];
    }
    tropical_iter_breakdown_t b;
    b.attn_us = attn_us;
    b.gemm_flops = 2.0 * T * W;
    b.gemm_bytes = 2.0 * W + 2.0 * T * act;
    b.linear_us = 0;
    b.allreduce_us = 0;
    if (T > 0) {
        const double tf = linear->f_us_per_flop * b.gemm_flops, tw = linear->w_us_per_byte * b.gemm_bytes;
        b.linear_us = linear->g0_us + (tf > tw ? tf : tw) + linear->kappa * (tf > tw ? tw : tf);
        if (tp > 1) b.allreduce_us = 2.0 * (linear->ar0_us + linear->ar_us_per_byte * 2.0 * T * shape->d_model);
    }
    b.total_us = shape->num_layers * (b.attn_us + b.linear_us + b.allreduce_us);
    if (breakdown != nullptr) *breakdown = b;
    if (out_us != nullptr) *out_us = b.total_us;
    return TROPICAL_OK;
}
