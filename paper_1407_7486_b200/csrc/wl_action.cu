// wl_action.cu -- effective-action integrals on the group sums:
// k_action_density (proper-time integral, eq. (12), (44)-(47), (70))
// and k_action_radial (eq. (12), radial integral), both per jackknife group.
// CUDA path, sm_100a; shares nothing with oracle/.  The paper does these on the host after a D2H copy
// per integrand sample; here they run on the group sums where they lie.
#include "wl_internal.cuh"

namespace wl {

namespace {

// e B_z(rho) of the field profile (eq. (13), (15)), FP64.
__device__ double field_b(int profile, double p0, double p1, double rho)
{
    if (profile == WL_PROFILE_UNIFORM) return p0;
    if (profile == WL_PROFILE_SECH2) {
        const double E = exp(-2.0 * rho / p1);
        return p0 * 4.0 * E / ((1.0 + E) * (1.0 + E));
    }
    const double l2 = p1 * p1, D = l2 + rho * rho;            // flux tube, eq. (68)
    return 2.0 * p0 * l2 / (D * D);
}

// int_0^a of the small-T expansion eq. (44) (fermion) / eq. (45) (scalar), b = eB(r_cm): eq. (47).
__device__ double small_T_integral(double b, double m2, double a, int scalar)
{
    const double b2 = b * b, b4 = b2 * b2, b6 = b4 * b2, m4 = m2 * m2, m6 = m4 * m2;
    double c1, c2, c3, c4;
    if (!scalar) {
        c1 = -b4 / 45.0;
        c2 = b4 * m2 / 45.0;
        c3 = 2.0 * b6 / 945.0 - b4 * m4 / 90.0;
        c4 = (7.0 * b4 * m6 - 4.0 * b6 * m2) / 1890.0;
    } else {
        c1 = 7.0 * b4 / 360.0;
        c2 = -7.0 * b4 * m2 / 360.0;
        c3 = (147.0 * b4 * m4 - 31.0 * b6) / 15120.0;
        c4 = (31.0 * b6 * m2 - 49.0 * b4 * m6) / 15120.0;
    }
    const double a2 = a * a;
    return a2 * (c1 / 2.0 + a * (c2 / 3.0 + a * (c3 / 4.0 + a * (c4 / 5.0))));
}

// One thread per (group, rho).  Simpson's rule on n_T equal intervals of x in [0, x_a], x = 1/(1+T/Tmax)
// (PAPER.md:472); node j of the T array is x_k with k = n_T - j; x_0 = 0 (T = infinity) contributes 0.
__global__ void k_action_density(const double* __restrict__ group_sums, int n_groups, double per_group,
                                 const double* __restrict__ T, int n_T, const double* __restrict__ rho, int n_rho,
                                 int profile, double p0, double p1, int scalar, double m2, double a, double Tmax,
                                 double* __restrict__ density)
{
    const int idx = blockIdx.x * blockDim.x + threadIdx.x;
    if (idx >= n_groups * n_rho) return;
    const int g = idx / n_rho, r = idx % n_rho;
    const double b = field_b(profile, p0, p1, rho[r]);
    const double xa = 1.0 / (1.0 + a / Tmax), h = xa / double(n_T);
    double simpson = 0.0;
    for (int j = 0; j < n_T; ++j) {
        const int k = n_T - j;
        const double x = h * double(k), Tj = T[j];
        const double W = group_sums[((int64_t)g * n_T + j) * n_rho + r] / per_group;       // <W>_g, eq. (60)
        const double bT = b * Tj;
        const double bracket = scalar ? W - 1.0 + bT * bT / 6.0 : W - 1.0 - bT * bT / 3.0;
        const double I = exp(-m2 * Tj) / (Tj * Tj * Tj) * bracket;                          // eq. (70)
        const double weight = (k == n_T) ? 1.0 : ((k & 1) ? 4.0 : 2.0);
        simpson += weight * I * Tmax / (x * x);                                             // dT = Tmax dx / x^2
    }
    density[idx] = small_T_integral(b, m2, a, scalar) + simpson * h / 3.0;
}

// eq. (12): action[g] = (1/4 pi) int rho density_g d rho, Simpson on a uniform grid; one thread per group,
// serial in rho (fixed order).
__global__ void k_action_radial(const double* __restrict__ density, int n_groups, const double* __restrict__ rho,
                                int n_rho, double* __restrict__ action)
{
    const int g = blockIdx.x * blockDim.x + threadIdx.x;
    if (g >= n_groups) return;
    const double h = (rho[n_rho - 1] - rho[0]) / double(n_rho - 1);
    double s = 0.0;
    for (int r = 0; r < n_rho; ++r) {
        const double weight = (r == 0 || r == n_rho - 1) ? 1.0 : ((r & 1) ? 4.0 : 2.0);
        s += weight * rho[r] * density[(int64_t)g * n_rho + r];
    }
    action[g] = s * h / 3.0 / (4.0 * 3.14159265358979323846);
}

}  // namespace

cudaError_t launch_action_density(const double* group_sums, int n_groups, int64_t n_loops, const double* T, int n_T,
                                  const double* rho, int n_rho, int profile, double p0, double p1, int scalar,
                                  double m2, double a, double Tmax, double* density, cudaStream_t s)
{
    const int n = n_groups * n_rho;
    k_action_density<<<(n + 127) / 128, 128, 0, s>>>(group_sums, n_groups, double(n_loops / n_groups), T, n_T, rho,
                                                    n_rho, profile, p0, p1, scalar, m2, a, Tmax, density);
    return cudaGetLastError();
}

cudaError_t launch_action_radial(const double* density, int n_groups, const double* rho, int n_rho, double* action,
                                 cudaStream_t s)
{
    k_action_radial<<<(n_groups + 127) / 128, 128, 0, s>>>(density, n_groups, rho, n_rho, action);
    return cudaGetLastError();
}

}  // namespace wl

using namespace wl;

extern "C" {

wl_status wl_proper_time_nodes(double a, double Tmax, int n_T, double* h_T)
{
    if (!h_T || !(a > 0.0) || !(Tmax > 0.0) || n_T < 2 || n_T % 2 != 0) return WL_ERR_INVALID_ARG;
    const double xa = 1.0 / (1.0 + a / Tmax);
    for (int j = 0; j < n_T; ++j) {
        const double x = xa * double(n_T - j) / double(n_T);
        h_T[j] = Tmax * (1.0 / x - 1.0);
    }
    h_T[0] = a;
    return WL_OK;
}

wl_status wl_action_density(const wl_field* field, const double* d_group_sums, int n_groups, int64_t n_loops,
                            const double* d_T, int n_T, const double* d_rho_cm, int n_rho, double m2, double a,
                            double Tmax, double* d_density, void* stream)
{
    if (!field || !d_group_sums || !d_T || !d_rho_cm || !d_density) return WL_ERR_INVALID_ARG;
    if (n_groups < 1 || n_loops < 1 || n_loops % n_groups != 0 || n_rho < 1) return WL_ERR_INVALID_ARG;
    if (n_T < 2 || n_T % 2 != 0 || !(a > 0.0) || !(Tmax > 0.0) || !(m2 >= 0.0)) return WL_ERR_INVALID_ARG;
    if ((int64_t)n_groups * n_rho > 0x7fffffffLL) return WL_ERR_INVALID_ARG;
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
