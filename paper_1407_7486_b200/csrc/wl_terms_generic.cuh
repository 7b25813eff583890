// wl_terms_generic.cuh -- GenericTerm<Real, Profile, HAS_PHI, P>: the Term of k_wilson (wl_wilson_body.cuh) for
// every case the lean Terms do not cover: the uniform field (terms reduce to the bare cross product), the
// flux-tube profile in FP64, sech^2 with lambda outside the lean kernels' range, and the rarer option
// combinations.  Scalar arithmetic in Real through the profile structs of wl_field_device.cuh (libdevice
// exp / log1p / sqrt / division in FP64); the quadrature order of eq. (24) is a run-time loop here.
//
// Staged per point i, as Vec4<Real> arrays:  cr = (dy_y, dy_x, y_i x y_{i+1}, -),  pt = (y_x, y_y, |y|^2, -),
// node[q] = (y(t_q)_x, y(t_q)_y, |y(t_q)|^2, -) for q < Q  (pt and node only if the profile needs radii).
#pragma once

#include "wl_field_device.cuh"
#include "wl_wilson_body.cuh"

namespace wl {

template <typename Real> struct alignas(4 * sizeof(Real)) Vec4 { Real a, b, c, d; };

template <typename Real, template <typename> class Prof, bool HAS_PHI, int P_>
struct GenericTerm {
    static constexpr int kP = P_, kThreads = 256, kMinBlocks = 1, kSumBlock = 32, kUnroll = 2;
    static constexpr int kChunk = sizeof(Real) == 4 ? 512 : 256;
    static constexpr bool kHasPhi = HAS_PHI;
    static constexpr bool kRadius = Prof<Real>::kNeedsRadius;
    __host__ __device__ static constexpr size_t stage_bytes(int quad)
    {
        return sizeof(Vec4<Real>) * (size_t)kChunk * (kRadius ? 2 + (quad < 1 ? 1 : quad) : 1);
    }

    Prof<Real> prof;
    int Q;
    Real wq[3];
    __device__ explicit GenericTerm(const EvalArgs& a) : prof(a.p0, a.p1), Q(a.quad < 1 ? 1 : a.quad)
    {
        for (int q = 0; q < 3; ++q) wq[q] = Real(gl_weight(Q, q));
    }
    struct Grid {
        Real R2[P_], ax[P_], Tt[P_], scx[P_];
        Real ay[HAS_PHI ? P_ : 1], scy[HAS_PHI ? P_ : 1];
        __device__ __forceinline__ void load(const GenericTerm&, const double (&T)[P_], const double (&rho)[P_],
                                             const double (&cx)[P_], const double (&cy)[P_])
        {
#pragma unroll
            for (int j = 0; j < P_; ++j) {
                const double s = sqrt(T[j]);
                R2[j] = Real(rho[j] * rho[j]);
                ax[j] = Real(2.0 * s * cx[j]);
                Tt[j] = Real(T[j]);
                scx[j] = Real(s * cx[j]);
                if (HAS_PHI) { ay[j] = Real(2.0 * s * cy[j]); scy[j] = Real(s * cy[j]); }
            }
        }
    };
    struct Acc {
        Real ph[P_], sp[P_];
        __device__ __forceinline__ void zero()
        {
#pragma unroll
            for (int j = 0; j < P_; ++j) { ph[j] = Real(0); sp[j] = Real(0); }
        }
        __device__ __forceinline__ void flush(const Grid&, double (&dph)[P_], double (&dsp)[P_]) const
        {
#pragma unroll
            for (int j = 0; j < P_; ++j) { dph[j] += double(ph[j]); dsp[j] += double(sp[j]); }
        }
    };
    __device__ double g_scale() const { return prof.g_scale(); }
    __device__ double b_scale() const { return prof.b_scale(); }

    __device__ __forceinline__ void stage(unsigned char* s, int i, double yx, double yy, double zx, double zy) const
    {
        Vec4<Real>* sCr = reinterpret_cast<Vec4<Real>*>(s);
        Vec4<Real> cr; cr.a = Real(zy - yy); cr.b = Real(zx - yx); cr.c = Real(yx * zy - yy * zx); cr.d = Real(0);
        sCr[i] = cr;
        if (kRadius) {
            Vec4<Real> pt; pt.a = Real(yx); pt.b = Real(yy); pt.c = Real(yx * yx + yy * yy); pt.d = Real(0);
            sCr[kChunk + i] = pt;
            for (int q = 0; q < Q; ++q) {
                double nx, ny, n2;
                segment_node(yx, yy, zx, zy, gl_node(Q, q), nx, ny, n2);
                Vec4<Real> nd; nd.a = Real(nx); nd.b = Real(ny); nd.c = Real(n2); nd.d = Real(0);
                sCr[(2 + q) * kChunk + i] = nd;
            }
        }
    }

    __device__ __forceinline__ void point(const unsigned char* s, int i, const Grid& g, Acc& acc) const
    {
        const Vec4<Real>* sCr = reinterpret_cast<const Vec4<Real>*>(s);
        const Vec4<Real> cr = sCr[i];
        if (!kRadius) {
#pragma unroll
            for (int j = 0; j < P_; ++j) {
                Real c = g.scx[j] * cr.a;
                if (HAS_PHI) c = fma(-g.scy[j], cr.b, c);
                c = fma(g.Tt[j], cr.c, c);                               // x_i x x_{i+1}, eq. (24)
                Real bt, gt;
                prof.terms(Real(0), Real(0), bt, gt);
                acc.ph[j] = fma(gt, c, acc.ph[j]);
                acc.sp[j] += bt;
            }
            return;
        }
        const Vec4<Real> pt = sCr[kChunk + i];
        Real wp[P_], c[P_], gs[P_], bt[P_];
#pragma unroll
        for (int j = 0; j < P_; ++j) {
            c[j] = g.scx[j] * cr.a;
            if (HAS_PHI) c[j] = fma(-g.scy[j], cr.b, c[j]);
            c[j] = fma(g.Tt[j], cr.c, c[j]);
            wp[j] = fma(g.ax[j], pt.a, g.R2[j]);
            if (HAS_PHI) wp[j] = fma(g.ay[j], pt.b, wp[j]);
            wp[j] = fma(g.Tt[j], pt.c, wp[j]);                           // |x_i|^2
            gs[j] = Real(0);
        }
        for (int q = 0; q < Q; ++q) {
            const Vec4<Real> nd = sCr[(2 + q) * kChunk + i];
#pragma unroll
            for (int j = 0; j < P_; ++j) {
                Real wm = fma(g.ax[j], nd.a, g.R2[j]);
                if (HAS_PHI) wm = fma(g.ay[j], nd.b, wm);
                wm = fma(g.Tt[j], nd.c, wm);                             // rho_i^2(t_q), eq. (25)
                Real gt;
                prof.terms(wp[j], wm, bt[j], gt);
                gs[j] = (Q == 1) ? gt : fma(wq[q], gt, gs[j]);
            }
        }
#pragma unroll
        for (int j = 0; j < P_; ++j) {
            acc.ph[j] = fma(gs[j], c[j], acc.ph[j]);
            acc.sp[j] += bt[j];
        }
    }
};

}  // namespace wl

namespace wl {

// UniformTerm<Real, HAS_PHI, P, THREADS>: the constant field B_z = B, A = (B/2)(-y, x) (config 2 of BASELINE.json).
// g = eB/2 and b = eB are constants, so a point-eval is the bare cross product of eq. (24),
//     x_i x x_{i+1} = s (c x dy_i) + T (y_i x y_{i+1}),
// three (two without phi_cm) FMAs that accumulate straight into the phase sum; the spin sum is the number of
// terms.  One staged Vec4 (dy_y, dy_x, y_i x y_{i+1}, -) per point feeds 3 P FMAs per thread.  The generic
// kernel spent 11 warp instructions per point-eval on this (issue-bound, profiles/r02_offtarget.md).
template <typename Real, bool HAS_PHI, int P_, int THREADS_>
struct UniformTerm {
    static constexpr int kP = P_, kThreads = THREADS_, kMinBlocks = 1, kUnroll = 4;
    static constexpr int kSumBlock = sizeof(Real) == 4 ? 128 : 0;      // FP64: straight accumulation
    static constexpr int kChunk = sizeof(Real) == 4 ? 1024 : 512;
    static constexpr bool kHasPhi = HAS_PHI;
    __host__ __device__ static constexpr size_t stage_bytes(int) { return sizeof(Vec4<Real>) * (size_t)kChunk; }

    double eB;
    __device__ explicit UniformTerm(const EvalArgs& a) : eB(a.p0) {}
    struct Grid {
        Real Tt[P_], scx[P_];
        Real nscy[HAS_PHI ? P_ : 1];
        __device__ __forceinline__ void load(const UniformTerm&, const double (&T)[P_], const double (&)[P_],
                                             const double (&cx)[P_], const double (&cy)[P_])
        {
#pragma unroll
            for (int j = 0; j < P_; ++j) {
                const double s = sqrt(T[j]);
                Tt[j] = Real(T[j]);
                scx[j] = Real(s * cx[j]);
                if (HAS_PHI) nscy[j] = Real(-(s * cy[j]));
            }
        }
    };
    struct Acc {
        Real ph[P_];
        int n;                                                       // terms in this block: the spin sum of a constant field
        __device__ __forceinline__ void zero()
        {
            n = 0;
#pragma unroll
            for (int j = 0; j < P_; ++j) ph[j] = Real(0);
        }
        __device__ __forceinline__ void flush(const Grid&, double (&dph)[P_], double (&dsp)[P_]) const
        {
#pragma unroll
            for (int j = 0; j < P_; ++j) { dph[j] += double(ph[j]); dsp[j] += double(n); }
        }
    };
    __device__ double g_scale() const { return 0.5 * eB; }
    __device__ double b_scale() const { return eB; }

    __device__ __forceinline__ static void stage(unsigned char* s, int i, double yx, double yy, double zx, double zy)
    {
        Vec4<Real> cr; cr.a = Real(zy - yy); cr.b = Real(zx - yx); cr.c = Real(yx * zy - yy * zx); cr.d = Real(0);
        reinterpret_cast<Vec4<Real>*>(s)[i] = cr;
    }
    __device__ __forceinline__ static void point(const unsigned char* s, int i, const Grid& g, Acc& acc)
    {
        const Vec4<Real> cr = reinterpret_cast<const Vec4<Real>*>(s)[i];
        ++acc.n;
#pragma unroll
        for (int j = 0; j < P_; ++j) {
            Real p = fma(g.scx[j], cr.a, acc.ph[j]);
            if (HAS_PHI) p = fma(g.nscy[j], cr.b, p);
            acc.ph[j] = fma(g.Tt[j], cr.c, p);                       // x_i x x_{i+1}, eq. (24)
        }
    }
};

}  // namespace wl
