// fft_fast.cuh -- size-specialised register FFT passes (placeholder: not built yet, generic path only).
#pragma once
#include <string>
#include "mm_common.cuh"

namespace mm {

struct FastPlan {
    bool usable;
};

inline bool fast_plan_init(FastPlan& fp, const Geom&, std::string*) { fp.usable = false; return true; }
inline void fast_plan_destroy(FastPlan&) {}
inline bool launch_eval_fast(FastPlan&, const Geom&, cudaStream_t, float2*, float2*, const float*,
                             const EpiParams&, KTimer&) { return false; }

}  // namespace mm
