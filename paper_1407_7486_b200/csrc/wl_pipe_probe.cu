// wl_pipe_probe.cu -- measurement helper: instruction streams that saturate ONE pipe of the SM, so that bench.py can
// state the roofline denominators of k_wilson as numbers measured in the same run instead of lanes x clock
// (the method of profiles/r01_pipe_rates.md, now part of the library).  Not on the hot path.
//   pipe 0: scalar FFMA      -- the FP32 non-tensor issue roofline (nominal 128 lanes/clk/SM)
//   pipe 1: MUFU.EX2         -- the special-function (XU) pipe that binds Sech2PackedF32 (nominal 16)
//   pipe 2: DFMA             -- the FP64 pipe that binds Sech2LeanF64 (nominal 64)
// Every thread runs kChains independent dependency chains, kUnroll times per loop iteration; the values are
// irrelevant (they may run to infinity: the pipes' rates do not depend on them).  CUDA path, sm_100a.
#include "wl_internal.cuh"

namespace wl {

constexpr int kProbeThreads = 256;
constexpr int kProbeCtasPerSm = 4;
constexpr int kChains = 16;
constexpr int kUnroll = 8;

template <int PIPE>
__global__ void __launch_bounds__(kProbeThreads) k_pipe_probe(int64_t iters, float* __restrict__ sink)
{
    float a[kChains];
    double d[kChains];
#pragma unroll
    for (int j = 0; j < kChains; ++j) { a[j] = 1e-3f * (float)(threadIdx.x + j); d[j] = 1e-3 * (double)(threadIdx.x + j); }
    const float c1 = 0.999f, c2 = 1e-4f;
    const double e1 = 0.999, e2 = 1e-4;
    for (int64_t i = 0; i < iters; ++i) {
#pragma unroll
        for (int u = 0; u < kUnroll; ++u) {
#pragma unroll
            for (int j = 0; j < kChains; ++j) {
                if (PIPE == 0) asm volatile("fma.rn.f32 %0, %0, %1, %2;" : "+f"(a[j]) : "f"(c1), "f"(c2));
                if (PIPE == 1) asm volatile("ex2.approx.ftz.f32 %0, %0;" : "+f"(a[j]));
                if (PIPE == 2) asm volatile("fma.rn.f64 %0, %0, %1, %2;" : "+d"(d[j]) : "d"(e1), "d"(e2));
            }
        }
    }
    float s = 0.f;
#pragma unroll
    for (int j = 0; j < kChains; ++j) s += a[j] + (float)d[j];
    if (s == 12345.678f) sink[0] = s;                      // keeps the chains alive; practically never true
}

}  // namespace wl

using namespace wl;

extern "C" wl_status wl_pipe_probe(int pipe, int64_t iters, float* d_sink, void* stream, int64_t* lane_ops, int* n_sms)
{
    if (pipe < 0 || pipe > 2 || iters < 1 || iters > (1LL << 32) || !d_sink) return WL_ERR_INVALID_ARG;
    int dev = 0, sms = 0;
    if (cudaGetDevice(&dev) != cudaSuccess || cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess
        || sms < 1) {
        cudaGetLastError();
        return WL_ERR_CUDA;
    }
    const unsigned ctas = (unsigned)(sms * kProbeCtasPerSm);
    cudaStream_t s = (cudaStream_t)stream;
    if (pipe == 0) k_pipe_probe<0><<<ctas, kProbeThreads, 0, s>>>(iters, d_sink);
    if (pipe == 1) k_pipe_probe<1><<<ctas, kProbeThreads, 0, s>>>(iters, d_sink);
    if (pipe == 2) k_pipe_probe<2><<<ctas, kProbeThreads, 0, s>>>(iters, d_sink);
    if (cudaGetLastError() != cudaSuccess) return WL_ERR_CUDA;
    if (lane_ops) *lane_ops = (int64_t)ctas * kProbeThreads * iters * (kChains * kUnroll);
    if (n_sms) *n_sms = sms;
    return WL_OK;
}
