// wl_eval_kernels.cu -- the generic k_wilson instantiations (wl_terms_generic.cuh), the evaluation plan, the
// dispatch between the Terms, and the reductions over loops: k_group_reduce, k_mean, and the shuffled-group
// variants k_group_permutation / k_group_reduce_shuffled.   CUDA path, sm_100a.
#include "wl_terms_generic.cuh"

namespace wl {

constexpr int kThreads = 256;

// S_g = sum over the units of group g, in unit order (eq. (60)).  One thread per
// (group, grid point); the group index is folded into blockIdx.x (any number of groups).  The partial sums come in
// the order k_wilson walks the grid (coalesced on both sides); the group sums go out as [t][r].
__global__ void k_group_reduce(const double* __restrict__ partial, int64_t units_per_group, int n_T, int n_rho,
                               int tiles, double* __restrict__ group_sums)
{
    const int n_grid = n_T * n_rho;
    const int v = (blockIdx.x % tiles) * blockDim.x + threadIdx.x;
    const int64_t g = blockIdx.x / tiles;
    if (v >= n_grid) return;
    const double* p = partial + g * units_per_group * n_grid + v;
    double S = 0.0;
    for (int64_t c = 0; c < units_per_group; ++c) S += p[c * n_grid];
    int it, ir;
    walk_position(v, n_T, n_rho, &it, &ir);
    group_sums[g * n_grid + it * n_rho + ir] = S;
}

// <W> = (sum_g S_g)/N_l in group order (eq. (61)-(62)).
__global__ void k_mean(const double* __restrict__ group_sums, int n_groups, int n_grid, double n_loops,
                       double* __restrict__ W_mean)
{
    const int k = blockIdx.x * blockDim.x + threadIdx.x;
    if (k >= n_grid) return;
    double total = 0.0;
    for (int g = 0; g < n_groups; ++g) total += group_sums[(int64_t)g * n_grid + k];
    W_mean[k] = total / n_loops;
}

// Shuffled group assignment (Sec. IV.B.3; reading A17): perm[t][i] = pi_t(i), a
// keyed bijection of [0, n_loops) per proper-time index t.  Balanced Feistel network, 6 rounds, on 2b bits
// (4^b >= n_loops), round function = word 0 of Philox4x32-10 with counter (R, round, t, 'SHFL') and key
// (seed_lo, seed_hi); cycle walking brings the image back below n_loops.  One thread per (t, i).
__global__ void k_group_permutation(uint64_t seed, int64_t n_loops, int n_T, int half_bits, int32_t* __restrict__ perm)
{
    const int64_t idx = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (idx >= n_loops * n_T) return;
    const uint32_t t = (uint32_t)(idx / n_loops);
    const uint32_t mask = (1u << half_bits) - 1u;
    uint64_t x = (uint64_t)(idx % n_loops);
    do {
        uint32_t L = (uint32_t)(x >> half_bits), R = (uint32_t)x & mask;
#pragma unroll 1
        for (uint32_t round = 0; round < 6; ++round) {
            uint32_t w[4];
            philox4x32_10(R, round, t, 0x5348464Cu, (uint32_t)seed, (uint32_t)(seed >> 32), w);
            const uint32_t nR = L ^ (w[0] & mask);
            L = R;
            R = nR;
        }
        x = ((uint64_t)L << half_bits) | R;
    } while (x >= (uint64_t)n_loops);
    perm[idx] = (int32_t)x;
}

// S_g[t][r] = sum_{i in block g} W[perm[t][i]][t][r], in the order of i (eq. (60) with the shuffled membership).
__global__ void k_group_reduce_shuffled(const double* __restrict__ W_loop, const int32_t* __restrict__ perm,
                                        int64_t n_loops, int64_t per_group, int n_rho, int n_grid, int tiles,
                                        double* __restrict__ group_sums)
{
    const int k = (blockIdx.x % tiles) * blockDim.x + threadIdx.x;
    const int64_t g = blockIdx.x / tiles;
    if (k >= n_grid) return;
    const int32_t* row = perm + (int64_t)(k / n_rho) * n_loops + g * per_group;
    double S = 0.0;
    for (int64_t i = 0; i < per_group; ++i) S += W_loop[(int64_t)row[i] * n_grid + k];
    group_sums[g * n_grid + k] = S;
}

// ------------------------------------------------------------------ host side: plan + dispatch

EvalPlan make_eval_plan(int64_t n_loops, int n_ppl, int n_T, int n_rho, int n_groups, wl_dtype compute,
                        bool per_loop, int64_t ensemble_loops)
{
    (void)n_ppl;
    EvalPlan p;
    p.n_grid = n_T * n_rho;
    p.threads = kThreads;
    const int p_max = (compute == WL_F32) ? 4 : 2;
    p.P = 1;
    while (p.P < p_max && p.n_grid >= kThreads * p.P * 2) p.P *= 2;
    p.n_tiles = (p.n_grid + kThreads * p.P - 1) / (kThreads * p.P);
    const int64_t per_group = n_loops / n_groups;
    const int64_t all_loops = ensemble_loops > 0 ? ensemble_loops : n_loops;
    // Largest divisor of the group size, at most 8, that still leaves enough CTAs to balance
    // a 148-SM part over many waves.  A function of the sizes only: the summation order, and
    // with it every bit of the result, is the same on any device.
    p.loops_per_unit = 1;
    const int64_t min_ctas = 16384;         // ~28 waves of 592 resident CTAs: the last, partial wave costs < 1 %
    if (!per_loop) {
        for (int d = 8; d > 1; --d)
            if (per_group % d == 0 && (all_loops / d) * p.n_tiles >= min_ctas) { p.loops_per_unit = d; break; }
    }
    p.n_units = n_loops / p.loops_per_unit;
    p.units_per_group = per_group / p.loops_per_unit;
    return p;
}

template <typename Real, template <typename> class Prof, bool HAS_PHI>
static cudaError_t launch_p(const EvalPlan& plan, const EvalArgs& a, cudaStream_t s)
{
    if (a.disc) {                                        // discretisation estimate: P <= 2 (three W per grid point)
        switch (plan.P) {
            case 1: return launch_term<GenericTerm<Real, Prof, HAS_PHI, 1>, true, false>(plan, a, s);
            case 2: return launch_term<GenericTerm<Real, Prof, HAS_PHI, 2>, true, false>(plan, a, s);
            default: return cudaErrorInvalidValue;
        }
    }
    switch (plan.P) {
        case 1: return launch_term<GenericTerm<Real, Prof, HAS_PHI, 1>, false, false>(plan, a, s);
        case 2: return launch_term<GenericTerm<Real, Prof, HAS_PHI, 2>, false, false>(plan, a, s);
        case 4: if (sizeof(Real) == 4) return launch_term<GenericTerm<Real, Prof, HAS_PHI, (sizeof(Real) == 4 ? 4 : 2)>, false, false>(plan, a, s);
        default: return cudaErrorInvalidValue;
    }
}

// Uniform field: UniformTerm.  Grids of at most 256 points run 128 threads x 2 grid points; larger ones 256 threads
// x plan.P.  The bulk-staging measurement variant exists for the config-2 shape (phi_cm given, small grid).
template <typename Real, bool HAS_PHI>
static cudaError_t launch_uniform_phi(const EvalPlan& plan, const EvalArgs& a, cudaStream_t s)
{
    if (a.disc) {
        if (plan.n_grid <= 256) return launch_term<UniformTerm<Real, HAS_PHI, 2, 128>, true, false>(plan, a, s);
        return plan.P >= 2 ? launch_term<UniformTerm<Real, HAS_PHI, 2, 256>, true, false>(plan, a, s)
                           : launch_term<UniformTerm<Real, HAS_PHI, 1, 256>, true, false>(plan, a, s);
    }
    if (plan.n_grid <= 256) {
        if (HAS_PHI && bulk_ok(a)) return launch_term<UniformTerm<Real, true, 2, 128>, false, true>(plan, a, s);
        return launch_term<UniformTerm<Real, HAS_PHI, 2, 128>, false, false>(plan, a, s);
    }
    switch (plan.P) {
        case 1: return launch_term<UniformTerm<Real, HAS_PHI, 1, 256>, false, false>(plan, a, s);
        case 2: return launch_term<UniformTerm<Real, HAS_PHI, 2, 256>, false, false>(plan, a, s);
        default: return launch_term<UniformTerm<Real, HAS_PHI, 4, 256>, false, false>(plan, a, s);
    }
}

template <typename Real>
static cudaError_t launch_uniform(const EvalPlan& plan, const EvalArgs& a, cudaStream_t s)
{
    return a.phi ? launch_uniform_phi<Real, true>(plan, a, s) : launch_uniform_phi<Real, false>(plan, a, s);
}

template <typename Real>
static cudaError_t launch_r(const EvalPlan& plan, const EvalArgs& a, int profile, cudaStream_t s)
{
    const bool phi = a.phi != nullptr;
    if (profile == WL_PROFILE_UNIFORM && a.quad >= 1) return launch_uniform<Real>(plan, a, s);   // g is constant: any Q is the same sum
    if (profile == WL_PROFILE_SECH2)
        return phi ? launch_p<Real, Sech2, true>(plan, a, s) : launch_p<Real, Sech2, false>(plan, a, s);
    if (profile == WL_PROFILE_FLUXTUBE)
        return phi ? launch_p<Real, FluxTube, true>(plan, a, s) : launch_p<Real, FluxTube, false>(plan, a, s);
    return cudaErrorInvalidValue;
}

bool lean_combination(const EvalArgs& a) { return a.quad == 1 || (a.phi == nullptr && !a.disc); }

cudaError_t launch_wilson(const EvalPlan& plan, const EvalArgs& a, int profile, wl_dtype compute, cudaStream_t s)
{
    // The lean sech^2 / flux-tube kernels carry squared radii scaled by 1/lambda^2; outside this range of
    // lambda they could overflow or flush, so the generic kernel (unscaled) serves it.
    const bool lambda_ok = a.p1 >= 1e-4 && a.p1 <= 1e4;
    const bool lean = lambda_ok && lean_combination(a);
    if (compute == WL_F32 && lean && (profile == WL_PROFILE_SECH2 || profile == WL_PROFILE_FLUXTUBE)) {
        EvalPlan p2 = plan;                              // grid points go in register pairs there
        if (p2.P < 2) p2.P = 2;
        if (a.disc && p2.P == 2 && p2.n_grid >= kThreads * 8) p2.P = 4;   // the discretisation plan caps P at 2 for the generic kernel
        return profile == WL_PROFILE_SECH2 ? launch_wilson_sech2_f32(p2, a, s) : launch_wilson_fluxtube_f32(p2, a, s);
    }
    if (compute == WL_F64 && lean && profile == WL_PROFILE_SECH2) return launch_wilson_sech2_f64(plan, a, s);
    return compute == WL_F32 ? launch_r<float>(plan, a, profile, s) : launch_r<double>(plan, a, profile, s);
}

cudaError_t launch_group_reduce(const double* partial, int64_t units_per_group, int n_groups,
                                int n_T, int n_rho, int64_t n_loops, double* group_sums, double* W_mean,
                                cudaStream_t s)
{
    const int n_grid = n_T * n_rho;
    const int tiles = (n_grid + 255) / 256;
    if ((int64_t)tiles * n_groups > 0x7fffffffLL) return cudaErrorInvalidConfiguration;
    k_group_reduce<<<(unsigned)(tiles * n_groups), 256, 0, s>>>(partial, units_per_group, n_T, n_rho, tiles, group_sums);
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return e;
    if (!W_mean) return cudaSuccess;
    k_mean<<<tiles, 256, 0, s>>>(group_sums, n_groups, n_grid, (double)n_loops, W_mean);
    return cudaGetLastError();
}

cudaError_t launch_group_permutation(uint64_t seed, int64_t n_loops, int n_T, int32_t* perm, cudaStream_t s)
{
    int b = 1;
    while ((1LL << (2 * b)) < n_loops) ++b;
    const int64_t blocks = (n_loops * n_T + 255) / 256;
    if (blocks > 0x7fffffffLL) return cudaErrorInvalidConfiguration;
    k_group_permutation<<<(unsigned)blocks, 256, 0, s>>>(seed, n_loops, n_T, b, perm);
    return cudaGetLastError();
}

cudaError_t launch_group_reduce_shuffled(const double* W_loop, const int32_t* perm, int64_t n_loops, int n_T,
                                         int n_rho, int n_groups, double* group_sums, double* W_mean,
                                         cudaStream_t s)
{
    const int n_grid = n_T * n_rho;
    const int tiles = (n_grid + 255) / 256;
    if ((int64_t)tiles * n_groups > 0x7fffffffLL) return cudaErrorInvalidConfiguration;
    k_group_reduce_shuffled<<<(unsigned)(tiles * n_groups), 256, 0, s>>>(W_loop, perm, n_loops, n_loops / n_groups, n_rho,
                                                                        n_grid, tiles, group_sums);
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return e;
    if (!W_mean) return cudaSuccess;
    k_mean<<<tiles, 256, 0, s>>>(group_sums, n_groups, n_grid, (double)n_loops, W_mean);
    return cudaGetLastError();
}

}  // namespace wl
