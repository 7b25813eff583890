// wl_dloop_device.cuh -- the d-loop generator as device functions (CUDA path; shares nothing with oracle/).
//
// One implementation serves both users, so that they produce the same bits:
//   * k_generate_dloops (wl_generate_finalize.cu): writes an ensemble to HBM            [wl_loops_generate]
//   * the Wilson-loop kernels in seeded mode (wl_wilson_body.cuh): regenerate every loop in shared memory
//     instead of reading it (Appendix 2: "generating the loops on-the-fly directly on the GPU
//     device itself without storing the entire loop in memory"; the device-memory ceiling that
//     forces the N_l-vs-N_ppl trade-off)                                                  [wl_eval_seeded]
//
// d-loops, steps (1)-(5), eq. (10)-(11), readings A1/A11: y_0 = 0; level k = 1..log2 N
// sets the odd multiples of h = N/2^k to y_p = (y_{p-h} + y_{p+h})/2 + sigma_k n_p, sigma_k^2 = 2^-k per component,
// n_p two standard normals from Philox4x32-10 with counter (p, loop_lo, loop_hi, 0) and key (seed_lo, seed_hi);
// finally the centre of mass is subtracted.
//
// The loop is produced CHUNK BY CHUNK (Cg = min(N, chunk capacity) points, a power of two): the "skeleton"
// = the points at multiples of Cg (levels with h >= Cg) is built first; chunk c then only needs its two skeleton
// end points and the normals of its own interior points (levels with h < Cg).  The centre of mass needs the
// whole loop, so a first pass generates every chunk once and sums; its summation order is fixed and does not
// depend on the number of threads (256 residue classes of the point index, then a fixed tree).
#pragma once

#include <cuda_runtime.h>
#include <stdint.h>

namespace wl {

constexpr int kSkeletonMax = 256;      // skeleton points per loop: N / Cg <= 65536 / 256 (the shortest chunk any Term stages)
constexpr int kClasses = 256;          // residue classes of the centre-of-mass sum

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

// sigma_k = 2^(-k/2): eq. (10) at k = 1, eq. (11) above.
__device__ __forceinline__ double level_sigma(int k)
{
    return ldexp((k & 1) ? 0.70710678118654752440 : 1.0, -(k / 2));
}

// y_p <- (y_lo + y_hi)/2 + y_p, the level update (steps (2)-(3)); explicit roundings so that
// every user computes the same bits.
__device__ __forceinline__ double2 level_update(double2 lo, double2 hi, double2 v)
{
    v.x = __dadd_rn(__dmul_rn(0.5, __dadd_rn(lo.x, hi.x)), v.x);
    v.y = __dadd_rn(__dmul_rn(0.5, __dadd_rn(lo.y, hi.y)), v.y);
    return v;
}

struct DLoopShape {
    int N, log2N;      // points per loop (a power of two)
    int Cg, n_sk;      // chunk length (a power of two dividing N), number of chunks = skeleton points
};

__host__ __device__ inline DLoopShape dloop_shape(int N, int chunk_capacity)
{
    DLoopShape s;
    s.N = N;
    s.log2N = 0;
    while ((1 << s.log2N) < N) ++s.log2N;
    s.Cg = N < chunk_capacity ? N : chunk_capacity;
    s.n_sk = N / s.Cg;
    return s;
}

// Shared memory the chunked generator needs beside the chunk buffer yraw[Cg + 1].
struct DLoopScratch {
    double2 skel[kSkeletonMax];     // un-shifted y at the multiples of Cg
    double2 cls[kClasses];          // residue-class sums of the centre-of-mass pass
    double2 mean;                   // centre of mass of the current loop
};

// Skeleton: y at p = 0, Cg, 2 Cg, ... (all levels with h >= Cg).  All threads of the CTA call it.
__device__ __forceinline__ void dloop_skeleton(uint64_t seed, uint64_t loop, const DLoopShape& sh, double2* skel)
{
    const int tid = threadIdx.x, bd = blockDim.x;
    for (int j = tid; j < sh.n_sk; j += bd) {
        if (j == 0) { skel[0] = make_double2(0.0, 0.0); continue; }            // step (1): y_N = y_0 = 0
        const int p = j * sh.Cg;
        const int k = sh.log2N - (__ffs(p) - 1);
        const double sigma = level_sigma(k);
        const double2 n = normal_pair(seed, loop, (uint32_t)p);
        skel[j] = make_double2(__dmul_rn(sigma, n.x), __dmul_rn(sigma, n.y));
    }
    __syncthreads();
    for (int hs = sh.n_sk >> 1; hs >= 1; hs >>= 1) {                            // h = hs * Cg, in skeleton units
        const int count = sh.n_sk / (2 * hs);
        for (int q = tid; q < count; q += bd) {
            const int j = hs + 2 * hs * q;
            skel[j] = level_update(skel[j - hs], skel[(j + hs) & (sh.n_sk - 1)], skel[j]);
        }
        __syncthreads();
    }
}

// Chunk c: un-shifted y at p = c Cg .. (c + 1) Cg (both ends included; the right end of the last chunk is
// y_N = y_0) into yraw[0 .. Cg].  All threads of the CTA call it; it ends with a barrier.
__device__ __forceinline__ void dloop_chunk(uint64_t seed, uint64_t loop, const DLoopShape& sh, int c,
                                            const double2* skel, double2* yraw)
{
    const int tid = threadIdx.x, bd = blockDim.x;
    for (int i = tid; i <= sh.Cg; i += bd) {
        if (i == 0) { yraw[0] = skel[c]; continue; }
        if (i == sh.Cg) { yraw[i] = skel[(c + 1 == sh.n_sk) ? 0 : c + 1]; continue; }
        const int k = sh.log2N - (__ffs(i) - 1);                                // ctz(c Cg + i) = ctz(i) for 0 < i < Cg
        const double sigma = level_sigma(k);
        const double2 n = normal_pair(seed, loop, (uint32_t)(c * sh.Cg + i));
        yraw[i] = make_double2(__dmul_rn(sigma, n.x), __dmul_rn(sigma, n.y));
    }
    __syncthreads();
    for (int h = sh.Cg >> 1; h >= 1; h >>= 1) {
        const int count = sh.Cg / (2 * h);
        for (int q = tid; q < count; q += bd) {
            const int i = h + 2 * h * q;
            yraw[i] = level_update(yraw[i - h], yraw[i + h], yraw[i]);
        }
        __syncthreads();
    }
}

// Fixed-order total of the 256 residue-class sums: lane L of warp 0 adds classes L, L + 32, ..., L + 224 in
// that order, then a shuffle-down tree over the 32 lanes.  The result lands in *out for every thread.
// All threads call it; cls[] must be complete (a barrier has been passed) on entry.
__device__ __forceinline__ void class_sum_total(const double2* cls, double2* out)
{
    if (threadIdx.x < 32) {
        double sx = 0.0, sy = 0.0;
#pragma unroll
        for (int m = 0; m < kClasses / 32; ++m) {
            sx = __dadd_rn(sx, cls[threadIdx.x + 32 * m].x);
            sy = __dadd_rn(sy, cls[threadIdx.x + 32 * m].y);
        }
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) {
            sx = __dadd_rn(sx, __shfl_down_sync(0xffffffffu, sx, o));
            sy = __dadd_rn(sy, __shfl_down_sync(0xffffffffu, sy, o));
        }
        if (threadIdx.x == 0) *out = make_double2(sx, sy);
    }
    __syncthreads();
}

// Step (5): the centre of mass of loop `loop`, (1/N) sum_p y_p, with the sum taken per residue
// class of p mod 256 in increasing p and the classes combined by class_sum_total.  Generates every chunk once
// (yraw is scratch).  blockDim.x must be 128 or 256.  On return sc->skel holds the loop's skeleton and
// sc->mean its centre of mass.
__device__ __forceinline__ void dloop_begin(uint64_t seed, uint64_t loop, const DLoopShape& sh, DLoopScratch* sc,
                                            double2* yraw)
{
    const int tid = threadIdx.x, bd = blockDim.x;
    dloop_skeleton(seed, loop, sh, sc->skel);
    double ax[2] = {0.0, 0.0}, ay[2] = {0.0, 0.0};             // classes tid (and tid + 128 when bd == 128)
    for (int c = 0; c < sh.n_sk; ++c) {
        dloop_chunk(seed, loop, sh, c, sc->skel, yraw);
        int m = 0;
        for (int i = tid; i < sh.Cg; i += bd, ++m) {
            const int w = (bd == kClasses) ? 0 : (m & 1);      // class of point c Cg + i is (i mod 256)
            ax[w] = __dadd_rn(ax[w], yraw[i].x);
            ay[w] = __dadd_rn(ay[w], yraw[i].y);
        }
        __syncthreads();                                        // yraw is overwritten by the next chunk
    }
    sc->cls[tid] = make_double2(ax[0], ay[0]);
    if (bd < kClasses) sc->cls[tid + bd] = make_double2(ax[1], ay[1]);
    __syncthreads();
    class_sum_total(sc->cls, &sc->mean);
    if (tid == 0) {
        const double2 s = sc->mean;
        sc->mean = make_double2(s.x / (double)sh.N, s.y / (double)sh.N);
    }
    __syncthreads();
}

}  // namespace wl
