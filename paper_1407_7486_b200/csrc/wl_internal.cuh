// wl_internal.cuh -- declarations shared by the translation units of libwl.so.
// Product code (CUDA path).  Shares nothing with oracle/.
#pragma once

#include <cuda_runtime.h>
#include <stdint.h>

#include "wl.h"

struct wl_field {
    int profile;        // wl_profile
    double p0;          // UNIFORM: eB      SECH2: eB0
    double p1;          // UNIFORM: unused  SECH2, FLUXTUBE: lambda   (p0 of FLUXTUBE: script-F)
    int scalar;         // 1: W = cos(phase) (WL_SCALAR), 0: W = cos(phase) cosh(spin)
};

namespace wl {

constexpr int kMaxPpl = 8192;        // generator limit (one loop in shared memory as double2)

// ---- how wl_eval cuts the work (a function of the sizes only, never of the device) ----
struct EvalPlan {
    int n_grid;          // n_T * n_rho
    int P;               // grid points per thread (register tile): 1, 2 or 4
    int threads;         // threads per CTA
    int n_tiles;         // CTAs along the grid: ceil(n_grid / (threads * P))
    int loops_per_unit;  // consecutive loops one CTA sums before writing a partial
    int64_t n_units;     // n_loops / loops_per_unit
    int units_per_group; // (n_loops / n_groups) / loops_per_unit
    int chunk_points;    // loop points staged in shared memory at a time
};

EvalPlan make_eval_plan(int64_t n_loops, int n_ppl, int n_T, int n_rho, int n_groups, wl_dtype compute,
                        bool per_loop);

struct EvalArgs {
    const void* loops;          // [n_loops][n_ppl][2]
    int loops_are_f64;
    int64_t n_loops;
    int n_ppl;
    const double* T;            // [n_T]
    const double* rho;          // [n_rho]
    const double* phi;          // [n_rho] or null
    int n_T, n_rho;
    double p0, p1;              // field parameters
    int scalar;                 // W = cos(phase) only
    int disc;                   // discretisation estimate (three levels, generic kernel only)
    double* partial;            // [n_units][n_grid]
    double* phase_out;          // per-loop mode only, nullable
    double* spin_out;           // per-loop mode only, nullable
};

cudaError_t launch_wilson(const EvalPlan& plan, const EvalArgs& a, int profile, wl_dtype compute,
                          cudaStream_t s);
// FP32, sech^2, phi_cm == NULL: the packed-FP32 kernel of wl_wilson_sech2_f32.cu (plan.P >= 2).
cudaError_t launch_wilson_sech2_f32(const EvalPlan& plan, const EvalArgs& a, cudaStream_t s);
// FP32, flux tube (eq. (68)), phi_cm == NULL: the packed-FP32 kernel of wl_wilson_fluxtube_f32.cu (plan.P >= 2).
cudaError_t launch_wilson_fluxtube_f32(const EvalPlan& plan, const EvalArgs& a, cudaStream_t s);
// FP64, sech^2, phi_cm == NULL: the lean FP64 kernel of wl_wilson_sech2_f64.cu (plan.P = 1 or 2).
cudaError_t launch_wilson_sech2_f64(const EvalPlan& plan, const EvalArgs& a, cudaStream_t s);
cudaError_t launch_group_reduce(const double* partial, int64_t n_units, int units_per_group, int n_groups,
                                int n_grid, int64_t n_loops, double* group_sums, double* W_mean,
                                cudaStream_t s);
cudaError_t launch_finalize(const double* group_sums, int n_groups, int64_t n_loops, int n_grid,
                            double* mean, double* err, double* delete_one, cudaStream_t s);
cudaError_t launch_extrapolate(const double* levels3, int64_t n, double* W_inf, double* delta, cudaStream_t s);
cudaError_t launch_generate(void* loops, int storage_is_f64, int64_t loop_begin, int64_t n_loops, int n_ppl,
                            uint64_t seed, cudaStream_t s);

}  // namespace wl
