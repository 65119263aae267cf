// fused_kernels.cuh -- fused persistent forward / adjoint sweep kernels (one CTA per subdomain).
#pragma once
#include "common.cuh"
#include "model_math.cuh"

struct FusedPlan {
    int enabled = 0;
};
typedef void* (*fused_take_fn)(void* arena, size_t bytes);

inline bool fused_fits(const Sub*, int) { return false; }
inline void fused_plan_init(FusedPlan& fp, const Sub*, int, int) { fp.enabled = 0; }
inline void fused_plan_arrays(FusedPlan&, fused_take_fn, void*) {}
inline int fused_setup(cudaStream_t, FusedPlan&, const Sub*) { return 0; }
inline void fused_sweep(cudaStream_t, long long*, FusedPlan&, const Sub*, int, const int*, ModelP, CostP, GeoP,
                        const double*, const double*, const double*, const double*, double*, const double*,
                        const long long*, const int*, const double*, const double*, double*, double*, bool,
                        double*, double*) {}
inline void fused_adjoint(cudaStream_t, long long*, FusedPlan&, const Sub*, int, const int*, ModelP, CostP, GeoP,
                          const double*, const double*, const double*, const double*, double*, const double*,
                          const long long*, const int*, const double*, const double*, double*, double*) {}
