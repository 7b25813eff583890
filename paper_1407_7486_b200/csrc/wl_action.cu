// wl_action.cu -- effective-action integrals on the group sums:
// k_action_density (proper-time integral, eq. (12), (44)-(47), (70))
// and k_action_radial (eq. (12), radial integral), both per jackknife group: one warp per
// (group, rho) resp. per group, lanes over the Simpson nodes, a fixed butterfly over the lanes.
// CUDA path, sm_100a; shares nothing with oracle/.  The paper does these on the host after a D2H copy
// per integrand sample; here they run on the group sums where they lie.
#include "wl_internal.cuh"

namespace wl {

namespace {

// e B_z(rho) of the field profile (eq. (13), (15)), FP64.
__device__ double profile_eB(int profile, double p0, double p1, double rho)
{
    switch (profile) {
        case WL_PROFILE_UNIFORM: return p0;
        case WL_PROFILE_SECH2: {                          // B0 sech^2(rho/lambda) = B0 / cosh^2, cosh >= 1: no overflow of the quotient
            const double c = cosh(fmin(rho / p1, 350.0));
            return p0 / (c * c);
        }
        default: {                                        // flux tube, eq. (68): 2 F lambda^2/(lambda^2 + rho^2)^2
            const double q = p1 * p1 / (p1 * p1 + rho * rho);
            return 2.0 * p0 * q * q / (p1 * p1);
        }
    }
}

// Fixed-order sum over the 32 lanes of a warp (butterfly: every lane ends with the same total).
__device__ __forceinline__ double warp_total(double v)
{
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}

// eq. (47), first part: the expansion eq. (44) / (45) integrated term by term from 0 to a,
//   beta a^2 [ k1 + k2 (mu a) + a^2 (k3b b^2 + k3m mu^2) + a^3 mu (k4b b^2 + k4m mu^2) ],  beta = (eB)^4, mu = m^2,
// with the printed coefficients divided by the power of the integration:
//   fermion: -1/90, 1/135, 1/1890, -1/360, -4/9450, 7/9450;   scalar: 7/720, -7/1080, -31/60480, 147/60480, 31/75600, -49/75600.
__device__ double expansion_integral(double eB, double mu, double a, bool scalar)
{
    const double b2 = eB * eB, beta = b2 * b2;
    const double k1 = scalar ? 7.0 / 720.0 : -1.0 / 90.0;
    const double k2 = scalar ? -7.0 / 1080.0 : 1.0 / 135.0;
    const double k3 = scalar ? (147.0 * mu * mu - 31.0 * b2) / 60480.0 : b2 / 1890.0 - mu * mu / 360.0;
    const double k4 = scalar ? mu * (31.0 * b2 - 49.0 * mu * mu) / 75600.0 : mu * (7.0 * mu * mu - 4.0 * b2) / 9450.0;
    return beta * a * a * (k1 + a * (k2 * mu + a * (k3 + a * k4)));
}

// One WARP per (group, rho).  The proper-time integral from a to infinity is taken in x = 1/(1 + T/Tmax)
// (PAPER.md:472): with T = Tmax (1 - x)/x and dT = -Tmax dx/x^2 the integrand of eq. (12)/(70) becomes
//     e^{-m^2 T} [ <W>_g - 1 -+ ... ] x / (Tmax^2 (1 - x)^3)  dx      on (0, x_a],
// sampled at the n_T + 1 Simpson nodes x_k = k x_a/n_T; x_0 (T = infinity) contributes nothing.  Node k belongs
// to T index j = n_T - k.  Lane L takes the nodes k = L + 1, L + 33, ... in that order, then the lanes are added
// by a fixed butterfly, so the result does not depend on scheduling.
__global__ void __launch_bounds__(128)
k_action_density(const double* __restrict__ group_sums, int n_groups, double loops_per_group,
                 const double* __restrict__ T, int n_T, const double* __restrict__ rho, int n_rho,
                 int profile, double p0, double p1, int scalar, double m2, double a, double Tmax,
                 double* __restrict__ density)
{
    const int warp = (blockIdx.x * blockDim.x + threadIdx.x) >> 5, lane = threadIdx.x & 31;
    if (warp >= n_groups * n_rho) return;                       // whole warps leave together
    const int g = warp / n_rho, r = warp - g * n_rho;
    const double eB = profile_eB(profile, p0, p1, rho[r]);
    const double x_a = Tmax / (Tmax + a), dx = x_a / double(n_T);
    const double* S = group_sums + (int64_t)g * n_T * n_rho + r;
    double part = 0.0;
    for (int k = lane + 1; k <= n_T; k += 32) {
        const int j = n_T - k;
        const double x = dx * double(k), t = T[j], bt = eB * t;
        const double W = S[(int64_t)j * n_rho] / loops_per_group;                                // <W>_g, eq. (60)
        const double counter = scalar ? -(bt * bt) * (1.0 / 6.0) : (bt * bt) * (1.0 / 3.0);     // eq. (45) / eq. (12)
        const double omx = 1.0 - x;
        const double jac = x / (Tmax * Tmax * omx * omx * omx);
        const double simpson = (k == n_T) ? 1.0 : ((k & 1) ? 4.0 : 2.0);
        part = fma(simpson * jac, exp(-m2 * t) * ((W - 1.0) - counter), part);
    }
    const double total = warp_total(part);
    if (lane == 0) density[warp] = expansion_integral(eB, m2, a, scalar != 0) + total * (dx / 3.0);
}

// eq. (12): action[g] = (1/4 pi) int rho density_g d rho by Simpson's rule on the uniform grid; one WARP per
// group, lanes strided over the rho nodes, fixed butterfly.
__global__ void __launch_bounds__(128)
k_action_radial(const double* __restrict__ density, int n_groups, const double* __restrict__ rho, int n_rho,
                double* __restrict__ action)
{
    const int g = (blockIdx.x * blockDim.x + threadIdx.x) >> 5, lane = threadIdx.x & 31;
    if (g >= n_groups) return;
    double part = 0.0;
    for (int r = lane; r < n_rho; r += 32) {
        const double simpson = (r == 0 || r == n_rho - 1) ? 1.0 : ((r & 1) ? 4.0 : 2.0);
        part = fma(simpson * rho[r], density[(int64_t)g * n_rho + r], part);
    }
    const double total = warp_total(part);
    const double step = (rho[n_rho - 1] - rho[0]) / double(n_rho - 1);
    if (lane == 0) action[g] = total * step / (12.0 * 3.14159265358979323846);                  // (h/3) / (4 pi)
}

}  // namespace

cudaError_t launch_action_density(const double* group_sums, int n_groups, int64_t n_loops, const double* T, int n_T,
                                  const double* rho, int n_rho, int profile, double p0, double p1, int scalar,
                                  double m2, double a, double Tmax, double* density, cudaStream_t s)
{
    const int64_t warps = (int64_t)n_groups * n_rho;
    k_action_density<<<(unsigned)((warps + 3) / 4), 128, 0, s>>>(group_sums, n_groups, double(n_loops / n_groups), T, n_T,
                                                                rho, n_rho, profile, p0, p1, scalar, m2, a, Tmax, density);
    return cudaGetLastError();
}

cudaError_t launch_action_radial(const double* density, int n_groups, const double* rho, int n_rho, double* action,
                                 cudaStream_t s)
{
    k_action_radial<<<(n_groups + 3) / 4, 128, 0, s>>>(density, n_groups, rho, n_rho, action);
    return cudaGetLastError();
}

}  // namespace wl

using namespace wl;

extern "C" {

wl_status wl_proper_time_nodes(double a, double Tmax, int n_T, double* h_T)
{
    if (!h_T || !(a > 0.0) || !(Tmax > 0.0) || n_T < 2 || (n_T & 1)) return WL_ERR_INVALID_ARG;
    // Simpson nodes x_k = k x_a/n_T of x = 1/(1 + T/Tmax), stored by decreasing k: T = Tmax (1 - x)/x
    const double x_a = Tmax / (Tmax + a);
    for (int k = n_T; k >= 1; --k) {
        const double x = x_a * (double(k) / double(n_T));
        h_T[n_T - k] = Tmax * (1.0 - x) / x;
    }
    h_T[0] = a;                                  // x_a maps back to a exactly
    return WL_OK;
}

wl_status wl_action_density(const wl_field* field, const double* d_group_sums, int n_groups, int64_t n_loops,
                            const double* d_T, int n_T, const double* d_rho_cm, int n_rho, double m2, double a,
                            double Tmax, double* d_density, void* stream)
{
    if (!field || !d_group_sums || !d_T || !d_rho_cm || !d_density) return WL_ERR_INVALID_ARG;
    if (n_groups < 1 || n_loops < 1 || n_loops % n_groups != 0 || n_rho < 1) return WL_ERR_INVALID_ARG;
    if (n_T < 2 || n_T % 2 != 0 || !(a > 0.0) || !(Tmax > 0.0) || !(m2 >= 0.0)) return WL_ERR_INVALID_ARG;
    if ((int64_t)n_groups * n_rho > 0x1fffffffLL) return WL_ERR_INVALID_ARG;      // one warp each
    cudaError_t e = launch_action_density(d_group_sums, n_groups, n_loops, d_T, n_T, d_rho_cm, n_rho, field->profile,
                                          field->p0, field->p1, field->scalar, m2, a, Tmax, d_density,
                                          (cudaStream_t)stream);
    return e == cudaSuccess ? WL_OK : WL_ERR_CUDA;
}

wl_status wl_action_radial(const double* d_density, int n_groups, const double* d_rho_cm, int n_rho,
                           double* d_action, void* stream)
{
    if (!d_density || !d_rho_cm || !d_action) return WL_ERR_INVALID_ARG;
    if (n_groups < 1 || n_rho < 3 || n_rho % 2 != 1) return WL_ERR_INVALID_ARG;
    cudaError_t e = launch_action_radial(d_density, n_groups, d_rho_cm, n_rho, d_action, (cudaStream_t)stream);
    return e == cudaSuccess ? WL_OK : WL_ERR_CUDA;
}

}  // extern "C"
