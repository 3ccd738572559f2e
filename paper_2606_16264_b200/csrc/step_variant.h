// step_variant.h -- the ONE statement of which kernel variant tropical_mixed_step runs, shared by the launcher
// (csrc/mixed.cu) and the predictor (csrc/step_cost.cpp): the built-in cost fits are keyed on this rule, so the two
// must not drift apart.  Host-only, no CUDA types.
#pragma once

namespace tropical {

// A step is taken as prefill-dominated -- fused variant: append inside the step kernel, two softmax warpgroups --
// when its requests carry at least this many new tokens on average (at most one decode request per ~64 prefill
// tokens).  Measured crossover: profiles/r2e_fused_step.md.
constexpr int kFusedMinTokensPerReq = 64;

inline bool step_is_prefill_dominated(long long total_q, long long num_reqs) {
    return num_reqs > 0 && total_q >= (long long)kFusedMinTokensPerReq * num_reqs;
}

}  // namespace tropical
