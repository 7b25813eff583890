// wl_block_bounds.cuh -- "far blocks": how a sech^2 Term of k_wilson (wl_wilson_body.cuh) learns, for a whole warp and a
// whole block of staged segments at once, how close to the flux tube's axis the loop can come.  CUDA path, sm_100a.
//
// While a chunk is staged every warp records the bounding box (unit-loop coordinates) of the 32 segments it stages;
// kBlock / 32 such boxes make the box of a block of kBlock staged segments.  Before a block is walked every thread
// bounds rho_i^2(t) (times k^2: w') from below over that box for each of its grid points, the warp takes the minimum,
// and the Term picks an instantiation of its walk by it ("tier"): clear of the axis no near-axis polynomial, select
// or guard is needed, and E = 2^(-u') <= 2^(-sqrt(w'_min)) lets a shorter polynomial reach the accuracy of the full
// one.  The bound is conservative: the box holds every point of every segment (so every node of any quadrature rule),
// and the margins below cover the rounding of the kernels' own w' and of this test.  The tier is a function of the
// loop, the grid and the tile shape only: results stay bit-reproducible.
#pragma once

#include <cuda_runtime.h>

namespace wl {

template <int CHUNK, int BLOCK>
struct BlockBounds {
    static_assert(BLOCK % 32 == 0 && CHUNK % BLOCK == 0, "a warp's 32 staged segments lie in one block");
    static constexpr int kBlocks = CHUNK / BLOCK, kSlots = BLOCK / 32;
    static constexpr size_t kBytes = sizeof(float4) * kBlocks * kSlots;

    // floats <-> integers with the same order (for redux.sync min / max)
    __device__ __forceinline__ static int ordered(float f) { const int i = __float_as_int(f); return i ^ ((i >> 31) & 0x7fffffff); }
    __device__ __forceinline__ static float unordered(int i) { return __int_as_float(i ^ ((i >> 31) & 0x7fffffff)); }

    // EVERY thread of the CTA, once per staging step.  ib = first staged index of the step (a multiple of the CTA size),
    // valid = this thread staged a segment, (y, z) = its end points.  `base` = where the kBytes of boxes live.
    __device__ __forceinline__ static void note(unsigned char* base, int ib, bool valid, double yx, double yy, double zx, double zy)
    {
        const float inf = __int_as_float(0x7f800000);
        const float x0 = valid ? fminf(float(yx), float(zx)) : inf, x1 = valid ? fmaxf(float(yx), float(zx)) : -inf;
        const float y0 = valid ? fminf(float(yy), float(zy)) : inf, y1 = valid ? fmaxf(float(yy), float(zy)) : -inf;
        const float bx0 = unordered(__reduce_min_sync(0xffffffffu, ordered(x0))), bx1 = unordered(__reduce_max_sync(0xffffffffu, ordered(x1)));
        const float by0 = unordered(__reduce_min_sync(0xffffffffu, ordered(y0))), by1 = unordered(__reduce_max_sync(0xffffffffu, ordered(y1)));
        const int i0 = ib + (int)(threadIdx.x & ~31u);                 // first staged index of this warp's 32 segments
        if ((threadIdx.x & 31u) == 0 && i0 < CHUNK) reinterpret_cast<float4*>(base)[i0 / 32] = make_float4(bx0, bx1, by0, by1);
    }

    // box of the block that starts at staged index i0 (a multiple of BLOCK): (x_min, x_max, y_min, y_max)
    __device__ __forceinline__ static float4 box(const unsigned char* base, int i0)
    {
        const float4* bb = reinterpret_cast<const float4*>(base) + (i0 / BLOCK) * kSlots;
        float4 b = bb[0];
#pragma unroll
        for (int k = 1; k < kSlots; ++k) {
            const float4 c = bb[k];
            b.x = fminf(b.x, c.x); b.y = fmaxf(b.y, c.y); b.z = fminf(b.z, c.z); b.w = fmaxf(b.w, c.w);
        }
        return b;
    }
    __device__ __forceinline__ static float extent2(const float4& b)    // max |y|^2 over the box
    {
        return fmaxf(b.x * b.x, b.y * b.y) + fmaxf(b.z * b.z, b.w * b.w);
    }

    // Lower bound of w' = R2 + ax y_x + ay y_y + Tt |y|^2 over the box for ONE grid point, given the kernels' scaled
    // constants (R2 = k^2 rho^2, (ax, ay) = 2 k^2 sqrt(T) x_cm, Tt = k^2 T): with k x_cm = (ax, ay)/(2 sqrt(Tt)) and
    // k sqrt(T) = sqrt(Tt) the node is k x_cm + k sqrt(T) y, and its distance from the origin is at least the
    // distance of the scaled box.  0.999 and 1e-5 (R2 + Tt max|y|^2) are the margins; anything that is not a
    // non-negative number (NaN grids) counts as 0 = "on the axis".
    __device__ __forceinline__ static float w_low(const float4& b, float ext2, float R2, float ax, float ay, float Tt)
    {
        float t;
        asm("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(t) : "f"(Tt));
        const float ks = Tt * t, cx = 0.5f * ax * t, cy = 0.5f * ay * t;
        const float dx = fmaxf(fmaxf(fmaf(ks, b.x, cx), -fmaf(ks, b.y, cx)), 0.0f);
        const float dy = fmaxf(fmaxf(fmaf(ks, b.z, cy), -fmaf(ks, b.w, cy)), 0.0f);
        const float w = fmaf(fmaf(dx, dx, dy * dy), 0.999f, -1e-5f * fmaf(Tt, ext2, R2));
        return (w >= 0.0f) ? w : 0.0f;
    }
    // minimum over the warp (non-negative floats order like their bit patterns)
    __device__ __forceinline__ static float warp_min(float w) { return __int_as_float(__reduce_min_sync(0xffffffffu, __float_as_int(w))); }
};

}  // namespace wl
