// wl_field_device.cuh -- per-term field arithmetic of the Wilson-loop kernels (CUDA path).
//
// For one loop point (squared radius wp) and one segment midpoint (squared radius wm) a
// profile returns
//     bt : e B(rho_p)            up to the constant factor  Profile::b_scale()
//     gt : g(rho_m) = e A_phi/rho up to the constant factor  Profile::g_scale()
// (eq. (13)-(15), (23)).  The constant factors are applied once per
// (loop, grid point) in the FP64 epilogue.  Everything is written in rho^2, as the paper
// advises, but the sech^2 profile needs rho itself, hence one rsqrt.
//
// sech^2 profile, u = rho/lambda, E = exp(-2u) = 2^t, t = -2 u log2(e):
//     sech^2 u = 4 E/(1+E)^2
//     h(u) = [u tanh u - ln cosh u]/u^2 = ln2 [ (1 - log2(1+E)) + t E/(1+E) ] / u^2
// so that g = eB0 h (BASELINE.json config 1: Phi = 2 pi B0 [lambda rho tanh - lambda^2 ln cosh]).
// Near the axis the bracket cancels (it tends to u^2/2), so for u^2 below a threshold a
// polynomial in u^2 replaces it (coefficients from gen_h_poly.py, Chebyshev interpolation).
// Both are always evaluated and one is selected: lanes hold different grid points, a branch
// would diverge.
#pragma once

#include <cuda_runtime.h>

namespace wl {

__device__ __forceinline__ float mufu_rsqrt(float x) { float y; asm("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x)); return y; }
__device__ __forceinline__ float mufu_ex2(float x)   { float y; asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x)); return y; }
__device__ __forceinline__ float mufu_lg2(float x)   { float y; asm("lg2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x)); return y; }
__device__ __forceinline__ float mufu_rcp(float x)   { float y; asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x)); return y; }

template <typename Real> struct Uniform;
template <typename Real> struct Sech2;
template <typename Real> struct FluxTube;

// ---------------------------------------------------------------- uniform field
// g = eB/2, b = eB: the terms are the bare cross product and 1.
template <typename Real>
struct Uniform {
    static constexpr bool kNeedsRadius = false;
    double eB;
    __device__ explicit Uniform(double p0, double) : eB(p0) {}
    __device__ __forceinline__ void terms(Real, Real, Real& bt, Real& gt) const { bt = Real(1); gt = Real(1); }
    __device__ double b_scale() const { return eB; }
    __device__ double g_scale() const { return 0.5 * eB; }
};

// ---------------------------------------------------------------- sech^2, FP32
template <>
struct Sech2<float> {
    static constexpr bool kNeedsRadius = true;
    double eB0, lambda;
    float c1;        // -2 log2(e)/lambda
    float il2;       // 1/lambda^2
    float hc;        // ln2 lambda^2
    __device__ explicit Sech2(double p0, double p1) : eB0(p0), lambda(p1)
    {
        c1 = (float)(-2.0 * 1.4426950408889634074 / p1);
        il2 = (float)(1.0 / (p1 * p1));
        hc = (float)(0.69314718055994530942 * p1 * p1);
    }
    // 6 special-function ops: 2 rsqrt, 2 ex2, 1 lg2 and ONE rcp shared by the point and the
    // midpoint (1/(Dp Dm), Dp, Dm in [1,2]).
    __device__ __forceinline__ void terms(float wp, float wm, float& bt, float& gt) const
    {
        wp = fmaxf(wp, 1e-30f);
        wm = fmaxf(wm, 1e-30f);
        const float rp = mufu_rsqrt(wp);
        const float rm = mufu_rsqrt(wm);
        const float Ep = mufu_ex2(c1 * (wp * rp));
        const float t = c1 * (wm * rm);
        const float Em = mufu_ex2(t);
        const float Dp = 1.0f + Ep, Dm = 1.0f + Em;
        const float i12 = mufu_rcp(Dp * Dm);
        const float ip = i12 * Dm, im = i12 * Dp;
        const float q = Ep * ip;
        bt = q * ip;                                         // E/(1+E)^2 ; b_scale has the 4
        const float L = mufu_lg2(Dm);
        const float br = fmaf(t, Em * im, 1.0f - L);         // (1 - log2(1+E)) + t E/(1+E)
        const float hE = br * (hc * (rm * rm));              // ln2 lambda^2 / rho^2 * bracket
        const float w = wm * il2;                            // u^2
        float hP = -0.00032671079f;
        hP = fmaf(hP, w, 0.0021024490f);
        hP = fmaf(hP, w, -0.0072330751f);
        hP = fmaf(hP, w, 0.019300118f);
        hP = fmaf(hP, w, -0.047129907f);
        hP = fmaf(hP, w, 0.11109993f);
        hP = fmaf(hP, w, -0.24999948f);
        hP = fmaf(hP, w, 0.5f);
        gt = (w < 1.0f) ? hP : hE;
    }
    __device__ double b_scale() const { return 4.0 * eB0; }
    __device__ double g_scale() const { return eB0; }
};

// ---------------------------------------------------------------- sech^2, FP64
template <>
struct Sech2<double> {
    static constexpr bool kNeedsRadius = true;
    double eB0, lambda, il;
    __device__ explicit Sech2(double p0, double p1) : eB0(p0), lambda(p1), il(1.0 / p1) {}
    __device__ __forceinline__ void terms(double wp, double wm, double& bt, double& gt) const
    {
        const double up = sqrt(fmax(wp, 0.0)) * il;
        const double um = sqrt(fmax(wm, 0.0)) * il;
        const double Ep = exp(-2.0 * up);
        const double Em = exp(-2.0 * um);
        const double ip = 1.0 / (1.0 + Ep);
        const double im = 1.0 / (1.0 + Em);
        bt = Ep * ip * ip;
        const double w = um * um;
        const double hE = (0.69314718055994530942 - log1p(Em) - 2.0 * um * Em * im) / w;   // NaN at w = 0: not selected
        double hP = 0.00049741560165003009825;
        hP = fma(hP, w, -0.0013579858215890325492);
        hP = fma(hP, w, 0.0033351186608907291509);
        hP = fma(hP, w, -0.0081246168738242320088);
        hP = fma(hP, w, 0.019682539344289231951);
        hP = fma(hP, w, -0.047222222218121683809);
        hP = fma(hP, w, 0.11111111111108618644);
        hP = fma(hP, w, -0.24999999999999994163);
        hP = fma(hP, w, 0.5);
        gt = (w < 0.0625) ? hP : hE;
    }
    __device__ double b_scale() const { return 4.0 * eB0; }
    __device__ double g_scale() const { return eB0; }
};

// ---------------------------------------------------------------- flux tube, eq. (68)
// f_lambda = rho^2/(lambda^2+rho^2):  g = script-F/(lambda^2+rho^2),  b = 2 script-F lambda^2/(lambda^2+rho^2)^2
// (eq. (14), (15), (17)).  With a = 1 + w/lambda^2:  g = (script-F/lambda^2)/a_m,
// b = (2 script-F/lambda^2)/a_p^2.  No square root: the profile is a function of rho^2.
template <typename Real>
struct FluxTube {
    static constexpr bool kNeedsRadius = true;
    double F, lambda;
    Real il2;
    __device__ explicit FluxTube(double p0, double p1) : F(p0), lambda(p1), il2(Real(1.0 / (p1 * p1))) {}
    __device__ __forceinline__ void terms(float wp, float wm, float& bt, float& gt) const
    {
        const float ap = fmaf(wp, il2, 1.0f), am = fmaf(wm, il2, 1.0f);
        const float r = mufu_rcp(ap * am);                   // one reciprocal for point and midpoint
        const float ip = r * am;
        gt = r * ap;
        bt = ip * ip;
    }
    __device__ __forceinline__ void terms(double wp, double wm, double& bt, double& gt) const
    {
        const double ip = 1.0 / fma(wp, (double)il2, 1.0);
        gt = 1.0 / fma(wm, (double)il2, 1.0);
        bt = ip * ip;
    }
    __device__ double b_scale() const { return 2.0 * F / (lambda * lambda); }
    __device__ double g_scale() const { return F / (lambda * lambda); }
};

}  // namespace wl
