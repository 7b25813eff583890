// wl_generate_finalize.cu -- k_generate_dloops (support subsystem a0) and k_jackknife_finalize (a6).
// CUDA path, sm_100a.  Shares nothing with oracle/.
#include "wl_internal.cuh"

namespace wl {

// Philox4x32-10 (Salmon, Moraes, Dror, Shaw, SC'11), from the published description: ten
// rounds; each multiplies counter words 0 and 2 by two fixed constants, crosses the high
// halves with words 1, 3 and the key, and the key advances by the two Weyl constants.
__device__ __forceinline__ void philox4x32_10(uint32_t c0, uint32_t c1, uint32_t c2, uint32_t c3,
                                              uint32_t k0, uint32_t k1, uint32_t out[4])
{
#pragma unroll
    for (int r = 0; r < 10; ++r) {
        const uint32_t hi0 = __umulhi(0xD2511F53u, c0), lo0 = 0xD2511F53u * c0;
        const uint32_t hi1 = __umulhi(0xCD9E8D57u, c2), lo1 = 0xCD9E8D57u * c2;
        c0 = hi1 ^ c1 ^ k0;
        c1 = lo1;
        c2 = hi0 ^ c3 ^ k1;
        c3 = lo0;
        k0 += 0x9E3779B9u;
        k1 += 0xBB67AE85u;
    }
    out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

// Two standard normals for (seed, loop, point): DESIGN.md reading A11.
__device__ __forceinline__ double2 normal_pair(uint64_t seed, uint64_t loop, uint32_t point)
{
    uint32_t w[4];
    philox4x32_10(point, (uint32_t)loop, (uint32_t)(loop >> 32), 0u, (uint32_t)seed, (uint32_t)(seed >> 32), w);
    const uint64_t a = ((uint64_t)w[1] << 32) | w[0];
    const uint64_t b = ((uint64_t)w[3] << 32) | w[2];
    const double u1 = __dmul_rn((double)((a >> 11) + 1), 0x1.0p-53);     // (0, 1]
    const double u2 = __dmul_rn((double)((b >> 11) + 1), 0x1.0p-53);
    const double r = sqrt(__dmul_rn(-2.0, log(u1)));
    double sn, cs;
    sincos(__dmul_rn(6.283185307179586476925286766559, u2), &sn, &cs);
    return make_double2(__dmul_rn(r, cs), __dmul_rn(r, sn));
}

// One CTA per loop; the loop lives in shared memory as double2[N].
//   pass 1: y_p = sigma_k n_p for every p in 1..N-1 (k = level of p: p is an odd multiple of
//           h = N/2^k, sigma_k^2 = 1/N_k = 2^-k per component: eq. (10) at k = 1, eq. (11) above)
//   pass 2: level by level, y_p += (y_{p-h} + y_{p+h})/2      (steps (2)-(3))
//   pass 3: subtract the centre of mass                        (step (5))
template <typename Store>
__global__ void __launch_bounds__(256)
k_generate_dloops(Store* __restrict__ out, int64_t loop_begin, int N, int log2N, uint64_t seed)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    double2* y = reinterpret_cast<double2*>(smem_raw);
    __shared__ double2 red[8];
    const int tid = threadIdx.x;
    const uint64_t loop = (uint64_t)(loop_begin + blockIdx.x);

    for (int p = tid; p < N; p += blockDim.x) {
        if (p == 0) { y[0] = make_double2(0.0, 0.0); continue; }          // step (1): y_N = 0
        const int k = log2N - (__ffs(p) - 1);
        const double sigma = ldexp((k & 1) ? 0.70710678118654752440 : 1.0, -(k / 2));
        const double2 n = normal_pair(seed, loop, (uint32_t)p);
        y[p] = make_double2(__dmul_rn(sigma, n.x), __dmul_rn(sigma, n.y));
    }
    __syncthreads();
    for (int k = 1; k <= log2N; ++k) {
        const int h = N >> k;
        const int count = 1 << (k - 1);
        for (int q = tid; q < count; q += blockDim.x) {
            const int p = h + 2 * h * q;
            const double2 lo = y[p - h], hi = y[(p + h) & (N - 1)];
            double2 v = y[p];
            v.x = __dadd_rn(__dmul_rn(0.5, __dadd_rn(lo.x, hi.x)), v.x);
            v.y = __dadd_rn(__dmul_rn(0.5, __dadd_rn(lo.y, hi.y)), v.y);
            y[p] = v;
        }
        __syncthreads();
    }
    // centre of mass: per-thread strided sums, then a fixed-order warp / CTA tree
    double sx = 0.0, sy = 0.0;
    for (int p = tid; p < N; p += blockDim.x) { sx += y[p].x; sy += y[p].y; }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        sx += __shfl_down_sync(0xffffffffu, sx, o);
        sy += __shfl_down_sync(0xffffffffu, sy, o);
    }
    if ((tid & 31) == 0) red[tid >> 5] = make_double2(sx, sy);
    __syncthreads();
    double mx = 0.0, my = 0.0;
    for (int w = 0; w < (int)(blockDim.x >> 5); ++w) { mx += red[w].x; my += red[w].y; }
    mx /= (double)N;
    my /= (double)N;
    Store* o = out + (int64_t)blockIdx.x * N * 2;
    for (int p = tid; p < N; p += blockDim.x) {
        o[2 * p] = (Store)(y[p].x - mx);
        o[2 * p + 1] = (Store)(y[p].y - my);
    }
}

cudaError_t launch_generate(void* loops, int storage_is_f64, int64_t loop_begin, int64_t n_loops, int n_ppl,
                            uint64_t seed, cudaStream_t s)
{
    int log2N = 0;
    while ((1 << log2N) < n_ppl) ++log2N;
    const size_t smem = sizeof(double2) * (size_t)n_ppl;
    cudaError_t e;
    // one launch per 2^30 loops at most (gridDim.x limit is 2^31-1)
    for (int64_t done = 0; done < n_loops;) {
        const int64_t n = (n_loops - done < (1LL << 30)) ? n_loops - done : (1LL << 30);
        if (storage_is_f64) {
            e = cudaFuncSetAttribute(k_generate_dloops<double>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
            if (e != cudaSuccess) return e;
            k_generate_dloops<double><<<(unsigned)n, 256, smem, s>>>(
                reinterpret_cast<double*>(loops) + done * n_ppl * 2, loop_begin + done, n_ppl, log2N, seed);
        } else {
            e = cudaFuncSetAttribute(k_generate_dloops<float>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
            if (e != cudaSuccess) return e;
            k_generate_dloops<float><<<(unsigned)n, 256, smem, s>>>(
                reinterpret_cast<float*>(loops) + done * n_ppl * 2, loop_begin + done, n_ppl, log2N, seed);
        }
        e = cudaGetLastError();
        if (e != cudaSuccess) return e;
        done += n;
    }
    return cudaSuccess;
}

// eq. (60)-(63); delete-one-group means (reading A7).
__global__ void k_jackknife_finalize(const double* __restrict__ group_sums, int n_groups, double n_loops,
                                     int n_grid, double* __restrict__ mean, double* __restrict__ err,
                                     double* __restrict__ delete_one)
{
    const int k = blockIdx.x * blockDim.x + threadIdx.x;
    if (k >= n_grid) return;
    const double G = (double)n_groups;
    const double per_group = n_loops / G;
    double total = 0.0;
    for (int g = 0; g < n_groups; ++g) total += group_sums[(int64_t)g * n_grid + k];
    const double m = total / n_loops;
    double ss = 0.0;
    for (int g = 0; g < n_groups; ++g) {
        const double S = group_sums[(int64_t)g * n_grid + k];
        const double d = S / per_group - m;                  // <W>_g - <W>, eq. (60)
        ss += d * d;
        if (delete_one) delete_one[(int64_t)g * n_grid + k] = (total - S) / (n_loops - per_group);
    }
    mean[k] = m;
    err[k] = sqrt(ss / (G * (G - 1.0)));                     // eq. (63)
}

// eq. (51)-(52): parabola in 1/N through the levels (N/4, N/2, N).
__global__ void k_extrapolate(const double* __restrict__ lev3, int64_t n, double* __restrict__ W_inf,
                              double* __restrict__ delta)
{
    const int64_t k = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (k >= n) return;
    const double w4 = lev3[k], w2 = lev3[n + k], w1 = lev3[2 * n + k];
    const double wi = 8.0 / 3.0 * w1 - 2.0 * w2 + 1.0 / 3.0 * w4;
    W_inf[k] = wi;
    if (delta) delta[k] = fabs(w1 - wi);
}

cudaError_t launch_extrapolate(const double* levels3, int64_t n, double* W_inf, double* delta, cudaStream_t s)
{
    const int64_t blocks = (n + 255) / 256;
    if (blocks > 0x7fffffffLL) return cudaErrorInvalidConfiguration;
    k_extrapolate<<<(unsigned)blocks, 256, 0, s>>>(levels3, n, W_inf, delta);
    return cudaGetLastError();
}

cudaError_t launch_finalize(const double* group_sums, int n_groups, int64_t n_loops, int n_grid,
                            double* mean, double* err, double* delete_one, cudaStream_t s)
{
    k_jackknife_finalize<<<(n_grid + 127) / 128, 128, 0, s>>>(group_sums, n_groups, (double)n_loops, n_grid,
                                                             mean, err, delete_one);
    return cudaGetLastError();
}

}  // namespace wl
