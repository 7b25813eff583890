// bench_pipe_rates.cu -- micro-benchmarks of the SM pipes the Wilson-loop kernels are bound by.
// Not part of libwl.so.  It measures the denominators DESIGN.md section 5 uses for the roofline of
// k_wilson: lanes per clock per SM of the FP32 FMA pipe (scalar FFMA and packed FFMA2), of the
// special-function (XU) pipe (MUFU.EX2 / RSQ / SQRT / LG2), of the FP64 pipe, of the F32->F64
// conversion, and what MIXES of special-function and FMA work cost per warp instruction.
//
//   nvcc -gencode arch=compute_100a,code=sm_100a -O3 -o bench_pipe_rates \
//        paper_1407_7486_b200/csrc/bench_pipe_rates.cu && ./bench_pipe_rates
//
// Output of the B200 run is kept in profiles/r01_pipe_rates.md.
#include <cstdio>
#include <cuda_runtime.h>

typedef unsigned long long u64;
__device__ __forceinline__ u64 pack(float a, float b) { u64 r; asm("mov.b64 %0, {%1, %2};" : "=l"(r) : "f"(a), "f"(b)); return r; }
__device__ __forceinline__ void unpack(u64 v, float& a, float& b) { asm("mov.b64 {%0, %1}, %2;" : "=f"(a), "=f"(b) : "l"(v)); }
__device__ __forceinline__ u64 ffma2(u64 a, u64 b, u64 c) { u64 r; asm volatile("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(r) : "l"(a), "l"(b), "l"(c)); return r; }
#define MUFU(op, x) asm volatile(op ".approx.ftz.f32 %0, %0;" : "+f"(x))

enum { FFMA3 = 0, FFMA2X, FFMA2_2VAR, FFMA2_3VAR, EX2, RSQRT, SQRT, LG2, DFMA, F2F_DADD, MIX_SCALAR, MIX_PACKED, MIX_LDS };

// One loop iteration issues, per warp:
//   FFMA3: 32 three-register FFMA      FFMA2X: 16 FFMA2 (= 32 FMAs)      EX2..LG2: 32 MUFU
//   DFMA: 32 DFMA                      F2F_DADD: 4 x (F2F.F64.F32 + DADD)
//   MIX_SCALAR: M MUFU.EX2 + F FFMA    MIX_PACKED: M MUFU.EX2 + F FFMA2 + A FMNMX
//   FFMA2_2VAR / FFMA2_3VAR: 16 FFMA2 whose sources are two / three different, changing register pairs
//   MIX_LDS: M MUFU.EX2 + F FFMA2 + A broadcast LDS.128 (every lane reads the same address)
template <int KIND, int M, int F, int A>
__global__ void k(float* out, int iters, float s1, float s2)
{
    __shared__ float4 sm[256];
    sm[threadIdx.x] = make_float4(s1, s2, s1, s2);
    __syncthreads();
    float a[8];
    u64 p[4];
    double d[4];
    float lds_acc = 0.0f;
    float b = s1 + threadIdx.x * 1e-9f, c = s2;
    const u64 bb = pack(b, b), cc = pack(c, c);
#pragma unroll
    for (int i = 0; i < 8; ++i) a[i] = s1 + i + threadIdx.x;
#pragma unroll
    for (int i = 0; i < 4; ++i) { p[i] = pack(a[2 * i] * 0.5f, a[2 * i + 1] * 0.25f); d[i] = a[i]; }
    for (int it = 0; it < iters; ++it) {
        if (KIND == FFMA3) {
#pragma unroll
            for (int r = 0; r < 32; ++r) a[r & 7] = fmaf(a[r & 7], b, c);
        } else if (KIND == FFMA2X) {
#pragma unroll
            for (int r = 0; r < 16; ++r) p[r & 3] = ffma2(p[r & 3], bb, cc);
        } else if (KIND == FFMA2_2VAR) {
#pragma unroll
            for (int r = 0; r < 16; ++r) p[r & 3] = ffma2(p[r & 3], p[(r + 1) & 3], cc);
        } else if (KIND == FFMA2_3VAR) {
#pragma unroll
            for (int r = 0; r < 16; ++r) p[r & 3] = ffma2(p[r & 3], p[(r + 1) & 3], p[(r + 2) & 3]);
        } else if (KIND == EX2) {
#pragma unroll
            for (int r = 0; r < 32; ++r) MUFU("ex2", a[r & 7]);
        } else if (KIND == RSQRT) {
#pragma unroll
            for (int r = 0; r < 32; ++r) MUFU("rsqrt", a[r & 7]);
        } else if (KIND == SQRT) {
#pragma unroll
            for (int r = 0; r < 32; ++r) MUFU("sqrt", a[r & 7]);
        } else if (KIND == LG2) {
#pragma unroll
            for (int r = 0; r < 32; ++r) MUFU("lg2", a[r & 7]);
        } else if (KIND == DFMA) {
#pragma unroll
            for (int r = 0; r < 32; ++r) d[r & 3] = fma(d[r & 3], 1.0001, 0.5);
        } else if (KIND == F2F_DADD) {
#pragma unroll
            for (int r = 0; r < 4; ++r) { d[r] += (double)a[r]; a[r] += 1.0f; }
        } else if (KIND == MIX_SCALAR) {
#pragma unroll
            for (int m = 0; m < M; ++m) {
                MUFU("ex2", a[m & 7]);
#pragma unroll
                for (int f = 0; f < F / M; ++f) { const int q = (m + 1 + f) & 7; a[q] = fmaf(a[q], b, c); }
            }
        } else if (KIND == MIX_PACKED) {
#pragma unroll
            for (int m = 0; m < M; ++m) {
                MUFU("ex2", a[m & 7]);
#pragma unroll
                for (int f = 0; f < F / M; ++f) { const int q = (m + f) & 3; p[q] = ffma2(p[q], bb, cc); }
            }
#pragma unroll
            for (int x = 0; x < A; ++x) a[7 - (x & 1)] = fmaxf(a[7 - (x & 1)], b);
        } else if (KIND == MIX_LDS) {
#pragma unroll
            for (int m = 0; m < M; ++m) {
                MUFU("ex2", a[m & 7]);
#pragma unroll
                for (int f = 0; f < F / M; ++f) { const int q = (m + f) & 3; p[q] = ffma2(p[q], bb, cc); }
            }
#pragma unroll
            for (int x = 0; x < A; ++x) {
                float4 v;
                const unsigned addr = (unsigned)__cvta_generic_to_shared(&sm[(it * A + x) & 255]);
                asm volatile("ld.shared.v4.f32 {%0,%1,%2,%3}, [%4];" : "=f"(v.x), "=f"(v.y), "=f"(v.z), "=f"(v.w) : "r"(addr));
                lds_acc += v.x;
            }
        }
    }
    float s = c + lds_acc;
    for (int i = 0; i < 8; ++i) s += a[i];
    for (int i = 0; i < 4; ++i) { float x, y; unpack(p[i], x, y); s += x + y + (float)d[i]; }
    out[blockIdx.x * blockDim.x + threadIdx.x] = s;
}

static double g_ghz = 1.965;

template <int KIND, int M, int F, int A>
static void run(const char* name, double lane_ops_per_iter, const char* note)
{
    float* out;
    cudaMalloc(&out, 148 * 3 * 256 * sizeof(float));
    const int iters = 20000, threads = 256, blocks = 148 * 3;
    cudaEvent_t e0, e1;
    cudaEventCreate(&e0);
    cudaEventCreate(&e1);
    k<KIND, M, F, A><<<blocks, threads>>>(out, 200, 1.0f, 0.5f);
    cudaEventRecord(e0);
    k<KIND, M, F, A><<<blocks, threads>>>(out, iters, 1.0f, 0.5f);
    cudaEventRecord(e1);
    cudaEventSynchronize(e1);
    float ms;
    cudaEventElapsedTime(&ms, e0, e1);
    const double warp_iters_per_smsp = (double)blocks * (threads / 32) * iters / (148.0 * 4.0);
    const double clk = ms * 1e-3 * g_ghz * 1e9;
    printf("| %-34s | %8.3f | %10.2f | %10.2f | %s |\n", name, ms, clk / warp_iters_per_smsp,
           lane_ops_per_iter > 0 ? lane_ops_per_iter * 32.0 * warp_iters_per_smsp * 4.0 / clk : 0.0, note);
    cudaFree(out);
}

int main()
{
    cudaDeviceProp prop;
    cudaGetDeviceProperties(&prop, 0);
    int khz = 0;
    cudaDeviceGetAttribute(&khz, cudaDevAttrClockRate, 0);
    if (khz > 0) g_ghz = khz * 1e-6;
    printf("device: %s, %d SMs, clock used for the conversion: %.3f GHz\n\n", prop.name, prop.multiProcessorCount, g_ghz);
    printf("| test (per warp per loop iteration) | ms | clk / iter / sub-partition | lanes / clk / SM | note |\n|---|---|---|---|---|\n");
    run<FFMA3, 0, 0, 0>("32 FFMA (3 registers)", 32, "FP32 FMA pipe, scalar");
    run<FFMA2X, 0, 0, 0>("16 FFMA2 (= 32 FMAs)", 32, "packed: same FMA rate, half the issue slots");
    run<FFMA2_2VAR, 0, 0, 0>("16 FFMA2, 2 varying source pairs", 32, "register reads start to cost");
    run<FFMA2_3VAR, 0, 0, 0>("16 FFMA2, 3 varying source pairs", 32, "six registers per lane: 3 clk per FFMA2");
    run<EX2, 0, 0, 0>("32 MUFU.EX2", 32, "XU pipe");
    run<RSQRT, 0, 0, 0>("32 MUFU.RSQ", 32, "XU pipe");
    run<SQRT, 0, 0, 0>("32 MUFU.SQRT", 32, "XU pipe");
    run<LG2, 0, 0, 0>("32 MUFU.LG2", 32, "XU pipe");
    run<DFMA, 0, 0, 0>("32 DFMA", 32, "FP64 pipe");
    run<F2F_DADD, 0, 0, 0>("4 x (F2F.F64.F32 + DADD)", 4, "the conversion runs at the XU rate");
    run<MIX_SCALAR, 6, 12, 0>("6 MUFU + 12 FFMA", 0, "XU bound = 48");
    run<MIX_SCALAR, 6, 30, 0>("6 MUFU + 30 FFMA", 0, "XU bound = 48, issue 36 (+6: a MUFU costs 2 slots)");
    run<MIX_SCALAR, 6, 36, 0>("6 MUFU + 36 FFMA", 0, "XU bound = 48, issue 42 (+6)");
    run<MIX_SCALAR, 6, 42, 0>("6 MUFU + 42 FFMA", 0, "XU bound = 48, issue 48 (+6)");
    run<MIX_SCALAR, 5, 35, 0>("5 MUFU + 35 FFMA", 0, "XU bound = 40, issue 40 (+5)");
    run<MIX_PACKED, 6, 18, 0>("6 MUFU + 18 FFMA2 (36 FMAs)", 0, "XU bound = 48, FMA pipe 36");
    run<MIX_PACKED, 6, 24, 0>("6 MUFU + 24 FFMA2 (48 FMAs)", 0, "XU bound = 48, FMA pipe 48");
    run<MIX_PACKED, 5, 15, 0>("5 MUFU + 15 FFMA2 (30 FMAs)", 0, "XU bound = 40, FMA pipe 30");
    run<MIX_PACKED, 5, 20, 0>("5 MUFU + 20 FFMA2 (40 FMAs)", 0, "XU bound = 40, FMA pipe 40");
    run<MIX_PACKED, 5, 15, 6>("5 MUFU + 15 FFMA2 + 6 FMNMX", 0, "ALU-pipe work is nearly free");
    run<MIX_PACKED, 4, 16, 0>("4 MUFU + 16 FFMA2 (32 FMAs)", 0, "XU bound = 32, FMA pipe 32");
    run<MIX_LDS, 5, 15, 1>("5 MUFU + 15 FFMA2 + 1 LDS.128", 0, "shared-memory loads return through the XU's queue");
    run<MIX_LDS, 5, 15, 2>("5 MUFU + 15 FFMA2 + 2 LDS.128", 0, "");
    run<MIX_LDS, 5, 15, 4>("5 MUFU + 15 FFMA2 + 4 LDS.128", 0, "about 4 clk per LDS.128");
    run<MIX_LDS, 5, 15, 8>("5 MUFU + 15 FFMA2 + 8 LDS.128", 0, "");
    return 0;
}
