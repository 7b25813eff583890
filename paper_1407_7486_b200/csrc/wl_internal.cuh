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

constexpr int kMaxPplSeeded = 1 << 16;   // generator / seeded-evaluation limit on N (skeleton of <= kSkeletonMax points, wl_dloop_device.cuh)

// ---- how wl_eval cuts the work (a function of the sizes only, never of the device) ----
struct EvalPlan {
    int n_grid;          // n_T * n_rho
    int P;               // grid points per thread (register tile): 1, 2 or 4
    int threads;         // threads per CTA
    int n_tiles;         // CTAs along the grid: ceil(n_grid / (threads * P))
    int loops_per_unit;  // consecutive loops one CTA sums before writing a partial
    int64_t n_units;     // n_loops / loops_per_unit
    int64_t units_per_group; // (n_loops / n_groups) / loops_per_unit
};

// ensemble_loops > 0: n_loops is a shard (whole groups) of an ensemble of that many loops; the units are those
// of a call over the whole ensemble.
EvalPlan make_eval_plan(int64_t n_loops, int n_ppl, int n_T, int n_rho, int n_groups, wl_dtype compute,
                        bool per_loop, int64_t ensemble_loops = 0);

// The order in which k_wilson walks the (T, rho_cm) grid (wl_wilson_body.cuh): strips of kRhoStrip neighbouring
// rho_cm, within a strip rho_cm fastest, then the proper time; the last strip may be narrower.  Position v of the walk
// is grid point (*it, *ir).
constexpr int kRhoStrip = 8;
__host__ __device__ inline void walk_position(int v, int n_T, int n_rho, int* it, int* ir)
{
    const int nb = n_rho / kRhoStrip, rem = n_rho % kRhoStrip, full = nb * kRhoStrip * n_T;
    if (v < full) { const int blk = v / (kRhoStrip * n_T), w = v % (kRhoStrip * n_T); *it = w / kRhoStrip; *ir = blk * kRhoStrip + w % kRhoStrip; }
    else { const int w = v - full; *it = w / rem; *ir = nb * kRhoStrip + w % rem; }
}

struct EvalArgs {
    const void* loops;          // [n_loops][n_ppl][2]; unused when seeded
    int loops_are_f64;          // storage precision of the loop coordinates (also the rounding a seeded run emulates)
    int64_t n_loops;
    int n_ppl;
    const double* T;            // [n_T]
    const double* rho;          // [n_rho]
    const double* phi;          // [n_rho] or null
    int n_T, n_rho;
    double p0, p1;              // field parameters
    int scalar;                 // W = cos(phase) only
    int disc;                   // discretisation estimate (three levels)
    int quad;                   // Gauss-Legendre points in t for eq. (24): 1 (midpoint), 2, 3
    int seeded;                 // 1: regenerate every loop from (seed, loop_begin + loop) instead of reading `loops`
    int bulk;                   // 1: stage raw chunks by cp.async.bulk + mbarrier (measurement variant)
    uint64_t seed;
    int64_t loop_begin;
    double* partial;            // [n_units][n_grid]
    int partial_in_walk_order;  // 1: partial[unit][v], v = position in the grid walk (coalesced; k_group_reduce maps it back);
                                // 0: partial[unit][t * n_rho + r] (per-loop and shuffled paths: the array is an output)
    double* phase_out;          // per-loop mode only, nullable
    double* spin_out;           // per-loop mode only, nullable
};

cudaError_t launch_wilson(const EvalPlan& plan, const EvalArgs& a, int profile, wl_dtype compute,
                          cudaStream_t s);
// FP32, sech^2: the packed-FP32 kernels of wl_wilson_sech2_f32.cu.
cudaError_t launch_wilson_sech2_f32(const EvalPlan& plan, const EvalArgs& a, cudaStream_t s);
// FP32, flux tube (eq. (68)): the packed-FP32 kernels of wl_wilson_fluxtube_f32.cu.
cudaError_t launch_wilson_fluxtube_f32(const EvalPlan& plan, const EvalArgs& a, cudaStream_t s);
// FP64, sech^2: the lean FP64 kernels of wl_wilson_sech2_f64.cu (plan.P = 1 or 2).
cudaError_t launch_wilson_sech2_f64(const EvalPlan& plan, const EvalArgs& a, cudaStream_t s);
// Is (quadrature order, phi_cm, discretisation, staging) a combination the lean kernels are instantiated for?
bool lean_combination(const EvalArgs& a);

// partial is [n_units][n_grid] in WALK order (EvalArgs::partial_in_walk_order = 1); group_sums and W_mean are [t][r]
cudaError_t launch_group_reduce(const double* partial, int64_t units_per_group, int n_groups,
                                int n_T, int n_rho, int64_t n_loops, double* group_sums, double* W_mean,
                                cudaStream_t s);
cudaError_t launch_group_permutation(uint64_t seed, int64_t n_loops, int n_T, int32_t* perm, cudaStream_t s);
cudaError_t launch_group_reduce_shuffled(const double* W_loop, const int32_t* perm, int64_t n_loops, int n_T,
                                         int n_rho, int n_groups, double* group_sums, double* W_mean,
                                         cudaStream_t s);
cudaError_t launch_finalize(const double* group_sums, int n_groups, int64_t n_loops, int n_grid,
                            double* mean, double* err, double* delete_one, cudaStream_t s);
cudaError_t launch_extrapolate(const double* levels3, int64_t n, double* W_inf, double* delta, cudaStream_t s);
cudaError_t launch_generate(void* loops, int storage_is_f64, int64_t loop_begin, int64_t n_loops, int n_ppl,
                            uint64_t seed, cudaStream_t s);

}  // namespace wl
