// wl_generate_finalize.cu -- k_generate_dloops (support subsystem a0) and k_jackknife_finalize (a6).
// CUDA path, sm_100a.  Shares nothing with oracle/.
#include "wl_dloop_device.cuh"
#include "wl_internal.cuh"

namespace wl {

// One CTA per loop, through the chunked generator of wl_dloop_device.cuh (the same device functions the
// Wilson-loop kernels use in seeded mode, so both produce the same bits):
//   pass A: every chunk once, to sum the centre of mass (step (5))
//   pass B: every chunk again, shifted by the centre of mass, rounded once to the storage type, stored.
template <typename Store>
__global__ void __launch_bounds__(256)
k_generate_dloops(Store* __restrict__ out, int64_t loop_begin, DLoopShape sh, uint64_t seed)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    double2* yraw = reinterpret_cast<double2*>(smem_raw);
    DLoopScratch* sc = reinterpret_cast<DLoopScratch*>(smem_raw + sizeof(double2) * (size_t)(sh.Cg + 1));
    const uint64_t loop = (uint64_t)(loop_begin + blockIdx.x);
    dloop_begin(seed, loop, sh, sc, yraw);
    const double2 m = sc->mean;
    Store* o = out + (int64_t)blockIdx.x * sh.N * 2;
    for (int c = 0; c < sh.n_sk; ++c) {
        dloop_chunk(seed, loop, sh, c, sc->skel, yraw);
        for (int i = threadIdx.x; i < sh.Cg; i += blockDim.x) {
            const int p = c * sh.Cg + i;
            o[2 * p] = (Store)(yraw[i].x - m.x);
            o[2 * p + 1] = (Store)(yraw[i].y - m.y);
        }
        __syncthreads();
    }
}

cudaError_t launch_generate(void* loops, int storage_is_f64, int64_t loop_begin, int64_t n_loops, int n_ppl,
                            uint64_t seed, cudaStream_t s)
{
    const DLoopShape sh = dloop_shape(n_ppl, 1024);
    const size_t smem = sizeof(double2) * (size_t)(sh.Cg + 1) + sizeof(DLoopScratch);
    cudaError_t e;
    // one launch per 2^30 loops at most (gridDim.x limit is 2^31-1)
    for (int64_t done = 0; done < n_loops;) {
        const int64_t n = (n_loops - done < (1LL << 30)) ? n_loops - done : (1LL << 30);
        if (storage_is_f64)
            k_generate_dloops<double><<<(unsigned)n, 256, smem, s>>>(
                reinterpret_cast<double*>(loops) + done * n_ppl * 2, loop_begin + done, sh, seed);
        else
            k_generate_dloops<float><<<(unsigned)n, 256, smem, s>>>(
                reinterpret_cast<float*>(loops) + done * n_ppl * 2, loop_begin + done, sh, seed);
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
