// wl_terms_sech2_f64.cuh -- Sech2LeanF64: the FP64 Term of k_wilson (wl_wilson_body.cuh) for the sech^2 profile:
// configs 1 and 4 (FP64 variant) of BASELINE.json.  CUDA path, sm_100a.
// Every elementary function is written out branch-free for the FP64 pipe (64 lanes/clk/SM, DFMA
// = 2 clk per warp instruction per sub-partition, profiles/r01_pipe_rates.md) instead of calling the
// general-purpose exp / log1p / sqrt / division sequences (~200 FP64-pipe instructions per point-eval
// with slow-path branches):
//
//   sqrt, 1/w : MUFU.RSQ64H seed + two coupled Newton (Goldschmidt) steps + one residual correction
//   2^(-u)    : round-to-nearest split u = n + f via the 1.5*2^52 trick, degree-10 polynomial in f,
//               exponent adjusted with integer adds (E = exp(-2 rho/lambda) = 2^(-u'), u' = sqrt(w'))
//   1/((1+E_p) prod_q (1+E_q)) : ONE MUFU.RCP64H seed + two Newton steps, shared by the point and the nodes
//   1 - log2(1+E_q)    : degree-20 polynomial in E_q in [0,1]
//   near the axis (u^2 < 1/16): degree-7 polynomial in w' for the cancelling bracket (reading A4)
// about 100 FP64-pipe instructions per point-eval at Q = 1.  Coefficients: gen_h_poly.py (E2 10, L 20, hs 0.0625 7).
// Far blocks (wl_block_bounds.cuh): where a whole warp stays clear of the axis over a block of 128 staged segments,
// the near-axis polynomial and its select are left out and 1 - log2(1+E) needs degree 19 / 13 / 8 / 6 / 3 instead of
// 20 for the same 2e-17 (E <= 2^(-u'_min)): 97 -> 73 FP64-pipe instructions per point-eval in the farthest tier.
// Scaling as in wl_terms_packed_f32.cuh: all squared radii carried as w' = (2 log2(e)/lambda)^2 w.
// Sums round the loop are accumulated straight in FP64 (kSumBlock = 0).
#pragma once

#include "wl_block_bounds.cuh"
#include "wl_wilson_body.cuh"

namespace wl {

namespace f64lean {

__device__ __forceinline__ double xu_rsqrt64(double x) { double y; asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(x)); return y; }
__device__ __forceinline__ double xu_rcp64(double x) { double y; asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(x)); return y; }

// s = sqrt(w), ir = 1/sqrt(w) for w > 0 (w >= 1e-300): seed ~2^-22, two coupled steps -> ~2^-88, then
// one residual step on s.  9 FP64-pipe instructions + 1 MUFU.
__device__ __forceinline__ void sqrt_rsqrt(double w, double& s, double& ir)
{
    const double r0 = xu_rsqrt64(w);
    double g = w * r0;                 // -> sqrt(w)
    double h = 0.5 * r0;               // -> 1/(2 sqrt(w))
    double e = fma(-g, h, 0.5);
    g = fma(g, e, g);
    h = fma(h, e, h);
    e = fma(-g, h, 0.5);
    g = fma(g, e, g);
    h = fma(h, e, h);
    const double d = fma(-g, g, w);    // residual
    s = fma(d, h, g);
    ir = h + h;
}

// 1/D for D in [1, 16]: MUFU.RCP64H seed + two Newton steps.
__device__ __forceinline__ double rcp_newton(double D)
{
    double r = xu_rcp64(D);
    double e = fma(-D, r, 1.0);
    r = fma(r, e, r);
    e = fma(-D, r, 1.0);
    return fma(r, e, r);
}

// Polynomial coefficients live in constant memory: a DFMA takes one constant-bank operand directly, whereas
// a 64-bit literal costs two uniform-register moves per use (74 extra instructions per two point-evals).
__constant__ double kExp2[11] = {   // 2^(-f), |f| <= 1/2: gen_h_poly.py E2 10 (rel. error 3e-16), highest degree first
    7.0725859492692236999e-9, -1.0208690299958305835e-7, 1.3215442587921689653e-6, -0.000015252657260200837064,
    0.00015403530441736050155, -0.0013333558230164973899, 0.0096181291076068885273, -0.055504108664447719166,
    0.2402265069591009822, -0.69314718055994998286, 1.0};
__constant__ double kLog[21] = {    // 1 - log2(1+E), E in [0,1]: gen_h_poly.py L 20 (abs. error 2e-17), highest degree first
    0.000037716935465554877791, -0.00043656761569165172581, 0.0024001133617501894281, -0.0083829321823817315509,
    0.021049247229017102326, -0.040925999935882766517, 0.065142917694358537062, -0.089143555615740867799,
    0.10983761672477964967, -0.12712681926472003036, 0.14301332675890233011, -0.15998872460281850448,
    0.1802769786868982234, -0.20609048918280538869, 0.24044821605097346373, -0.28853893413338524963,
    0.360673756378019119, -0.4808983468401831136, 0.72134752044239441043, -1.4426950408889492514,
    0.99999999999999998397};
// 1 - log2(1+E) on the shorter ranges of E of the far-block tiers (all with abs. error < 3e-17)
// tier 1: u'^2 >= 0.53, E <= 0.604339, degree 19 (gen_h_poly.py Lw 0.53 19), highest degree first
__constant__ double kLogT1[20] = {
    -0.00064514930333626290451, 0.0045895602541965166215, -0.015814655553587231033, 0.035650269233658460794,
    -0.060293062553543541339, 0.083747101331824058093, -0.10258474311829583756, 0.11729639389379667497,
    -0.13033931384191816844, 0.1440901295174673664, -0.16026853583065484814, 0.18033277016488465521,
    -0.20609887840964535806, 0.2404491429405142745, -0.2885390065809844017, 0.36067376016643174925,
    -0.48089834696179172708, 0.72134752044446810222, -1.4426950408889633458, 0.99999999999999999995};
// tier 2: u'^2 >= 4, E <= 0.25025, degree 13 (gen_h_poly.py Lw 4 13)
__constant__ double kLogT2[14] = {
    -0.024887795416740174128, 0.070805936631926537284, -0.11175940373492745721, 0.13895587644456733789,
    -0.15926583799129985004, 0.18019309440597068775, -0.20608503470749155641, 0.24044818065772084687,
    -0.28853896099078533499, 0.36067375876335164926, -0.4808983469358815821, 0.72134752044421818009,
    -1.4426950408889623958, 0.99999999999999999935};
// tier 3: u'^2 >= 16, E <= 0.0625625, degree 8 (gen_h_poly.py Lw 16 8)
__constant__ double kLogT3[9] = {
    0.14118450783592787991, -0.201724835842929911, 0.24017898255855308115, -0.28852918283846478497,
    0.3606735492527275989, -0.48089834441051835446, 0.72134752042897980711, -1.4426950408889271023,
    0.99999999999999998598};
// tier 4: u'^2 >= 36, E <= 0.0156406, degree 6 (gen_h_poly.py Lw 36 6)
__constant__ double kLogT4[7] = {
    0.22948746423295850135, -0.28830549115279959543, 0.36067128126186996788, -0.48089833342659964874,
    0.72134752040924565814, -1.4426950408889289874, 0.99999999999999999451};
// tier 5: u'^2 >= 144, E <= 0.000244385, degree 3 (gen_h_poly.py Lw 144 3)
__constant__ double kLogT5[4] = {
    -0.4807221079967332697, 0.72134749352789418958, -1.44269504088764785, 0.99999999999999998995};
__constant__ double kHPoly[8] = {   // h(w)/(4 log2 e) in w', w = u^2 < 1/16: gen_h_poly.py hs 0.0625 7, highest degree first
    -7.7102839224224163556e-11, 1.7289132522207449606e-9, -3.519550981355539808e-8, 7.0992077974390822073e-7,
    -0.000014180275863490838682, 0.00027778246137776088779, -0.0052035101873268705174, 0.086643397569993163057};

// 2^(-u) for u >= 0.  u = n + f, n = rint(u), |f| <= 1/2; 2^(-f) by a degree-10 polynomial; 2^(-n) by
// subtracting n from the exponent field (n clamped to 1000: the result is then < 1e-301).
__device__ __forceinline__ double exp2_neg(double u)
{
    const double kMagic = 6755399441055744.0;            // 1.5 * 2^52
    const double t = u + kMagic;
    const double f = u - (t - kMagic);
    double p = kExp2[0];
#pragma unroll
    for (int i = 1; i < 11; ++i) p = fma(p, f, kExp2[i]);
    const int n = min(__double2loint(t), 1000);
    return __hiloint2double(__double2hiint(p) - (n << 20), __double2loint(p));
}

// (1 - log2(1+E)) - u E/(1+E) for E in [0,1], im = 1/(1+E).  With the polynomial 1 - log2(1+E) = c0 + E L'(E) the
// second term joins the last Horner step: c0 + E (L'(E) - u im).  TIER > 0: E is known to be small (far blocks).
template <int TIER> struct LogTable;
template <> struct LogTable<0> { static constexpr int kDeg = 20; __device__ __forceinline__ static double c(int i) { return kLog[i]; } };
template <> struct LogTable<1> { static constexpr int kDeg = 19; __device__ __forceinline__ static double c(int i) { return kLogT1[i]; } };
template <> struct LogTable<2> { static constexpr int kDeg = 13; __device__ __forceinline__ static double c(int i) { return kLogT2[i]; } };
template <> struct LogTable<3> { static constexpr int kDeg = 8; __device__ __forceinline__ static double c(int i) { return kLogT3[i]; } };
template <> struct LogTable<4> { static constexpr int kDeg = 6; __device__ __forceinline__ static double c(int i) { return kLogT4[i]; } };
template <> struct LogTable<5> { static constexpr int kDeg = 3; __device__ __forceinline__ static double c(int i) { return kLogT5[i]; } };

template <int TIER>
__device__ __forceinline__ double bracket(double E, double u, double im)
{
    typedef LogTable<TIER> Tb;
    double L = Tb::c(0);
#pragma unroll
    for (int i = 1; i < Tb::kDeg; ++i) L = fma(L, E, Tb::c(i));
    return fma(fma(-u, im, L), E, Tb::c(Tb::kDeg));
}

}  // namespace f64lean

// Staged record of point i (doubles; C = 2 values per position without phi_cm, 3 with), as double2 arrays:
//     [ y_x, (y_y), |y|^2 ]  [ y(t_q)_x, (y(t_q)_y), |y(t_q)|^2 ] x Q  [ dy_y/2, (dy_x/2), y_i x y_{i+1} ]
template <int P_, bool HAS_PHI, int Q_>
struct Sech2LeanF64 {
    static_assert(Q_ >= 1 && Q_ <= 3, "1-, 2- or 3-point Gauss-Legendre rule");
    static constexpr int kP = P_, kThreads = 256, kMinBlocks = 2, kChunk = 512, kSumBlock = 0, kUnroll = 1;
    static constexpr bool kHasPhi = HAS_PHI;
    static constexpr int C = HAS_PHI ? 3 : 2;
    static constexpr int NF = C * (2 + Q_), NV2 = (NF + 1) / 2, NFP = 2 * NV2;
    static constexpr int iPT = 0, iNODE = C, iCR = C * (1 + Q_);
    // far blocks: boxes of blocks of kBoundsBlock staged segments behind the staged records
    static constexpr bool kBlockBounds = true;
    static constexpr int kBoundsBlock = 128, kTiers = 6;
    typedef BlockBounds<kChunk, kBoundsBlock> Bounds;
    __host__ __device__ static constexpr size_t record_bytes() { return (size_t)16 * NV2 * kChunk; }
    __host__ __device__ static constexpr size_t stage_bytes(int) { return record_bytes() + Bounds::kBytes; }
    __device__ __forceinline__ void note_bounds(unsigned char* s, int ib, bool valid, double yx, double yy, double zx, double zy) const
    {
        Bounds::note(s + record_bytes(), ib, valid, yx, yy, zx, zy);
    }
    // tier k > 0 holds when w' >= tier_w(k) for every node of the block and every grid point of the warp
    __host__ __device__ static constexpr float tier_w(int k) { return k == 1 ? 0.53f : k == 2 ? 4.0f : k == 3 ? 16.0f : k == 4 ? 36.0f : 144.0f; }

    double eB0, lambda, k2;
    __device__ explicit Sech2LeanF64(const EvalArgs& a) : eB0(a.p0), lambda(a.p1)
    {
        const double k = 2.0 * 1.4426950408889634074 / lambda;
        k2 = k * k;
    }
    struct Grid {
        double R2[P_], ax[P_], Tt[P_];
        double ay[HAS_PHI ? P_ : 1];
        __device__ __forceinline__ void load(const Sech2LeanF64& t, const double (&T)[P_], const double (&rho)[P_],
                                             const double (&cx)[P_], const double (&cy)[P_])
        {
#pragma unroll
            for (int j = 0; j < P_; ++j) {
                R2[j] = t.k2 * rho[j] * rho[j];
                ax[j] = t.k2 * 2.0 * sqrt(T[j]) * cx[j];
                Tt[j] = t.k2 * T[j];
                if (HAS_PHI) ay[j] = t.k2 * 2.0 * sqrt(T[j]) * cy[j];
            }
        }
    };
    struct Acc {
        double ph[P_], sp[P_];
        __device__ __forceinline__ void zero()
        {
#pragma unroll
            for (int j = 0; j < P_; ++j) { ph[j] = 0.0; sp[j] = 0.0; }
        }
        __device__ __forceinline__ void flush(const Grid&, double (&dph)[P_], double (&dsp)[P_]) const
        {
#pragma unroll
            for (int j = 0; j < P_; ++j) { dph[j] += ph[j]; dsp[j] += sp[j]; }
        }
    };
    __device__ double g_scale() const
    {
        return eB0 * lambda * lambda * 0.69314718055994530942 * (Q_ == 2 ? 0.5 : (Q_ == 3 ? 5.0 / 18.0 : 1.0));
    }
    __device__ double b_scale() const { return 4.0 * eB0; }

    __device__ __forceinline__ static void stage(unsigned char* s, int i, double yx, double yy, double zx, double zy)
    {
        double v[NFP];
#pragma unroll
        for (int k = 0; k < NFP; ++k) v[k] = 0.0;
        v[iPT] = yx;
        if (HAS_PHI) v[iPT + 1] = yy;
        v[iPT + C - 1] = yx * yx + yy * yy;
#pragma unroll
        for (int q = 0; q < Q_; ++q) {
            double nx, ny, n2;
            segment_node(yx, yy, zx, zy, gl_node(Q_, q), nx, ny, n2);
            v[iNODE + C * q] = nx;
            if (HAS_PHI) v[iNODE + C * q + 1] = ny;
            v[iNODE + C * q + C - 1] = n2;
        }
        v[iCR] = 0.5 * (zy - yy);
        if (HAS_PHI) v[iCR + 1] = 0.5 * (zx - yx);
        v[iCR + C - 1] = yx * zy - yy * zx;
#pragma unroll
        for (int k = 0; k < NV2; ++k) reinterpret_cast<double2*>(s)[k * kChunk + i] = make_double2(v[2 * k], v[2 * k + 1]);
    }

    __device__ __forceinline__ static double radius2(const Grid& g, int j, const double (&v)[NFP], int at)
    {
        double w = fma(g.ax[j], v[at], g.R2[j]);
        if (HAS_PHI) w = fma(g.ay[j], v[at + 1], w);
        return fma(g.Tt[j], v[at + C - 1], w);
    }

    // near-axis polynomial (tier 0 only) or br/w' for one node
    template <int TIER>
    __device__ __forceinline__ static double g_node(double wm, double irm, double um, double Em, double im)
    {
        constexpr double kPolyBelow = 0.52034224525;         // w' < this  <=>  u^2 < 1/16
        const double br = f64lean::bracket<TIER>(Em, um, im);   // (1 - log2(1+E_m)) - u' E_m/(1+E_m)
        const double hE = br * (irm * irm);                  // br / w'
        if constexpr (TIER > 0) return hE;
        // h(w)/(4 log2 e) in w', w = u^2 < 1/16 (gen_h_poly.py hs 0.0625 7)
        double hP = f64lean::kHPoly[0];
#pragma unroll
        for (int i = 1; i < 8; ++i) hP = fma(hP, wm, f64lean::kHPoly[i]);
        return (wm < kPolyBelow) ? hP : hE;
    }

    template <int TIER>
    __device__ __forceinline__ void walk(const unsigned char* s, int i0, int ie, const Grid& g, Acc& acc) const
    {
        for (int i = i0; i < ie; ++i) point<TIER>(s, i, g, acc);
    }
    // one block of at most kBoundsBlock staged points, [i0, ie)
    __device__ __forceinline__ void block(const unsigned char* s, int i0, int ie, const Grid& g, Acc& acc) const
    {
        const float4 b = Bounds::box(s + record_bytes(), i0);
        const float ext2 = Bounds::extent2(b);
        float wlow = 1e30f;
#pragma unroll
        for (int j = 0; j < P_; ++j)
            wlow = fminf(wlow, Bounds::w_low(b, ext2, float(g.R2[j]), float(g.ax[j]), HAS_PHI ? float(g.ay[j]) : 0.0f, float(g.Tt[j])));
        const float wwarp = Bounds::warp_min(wlow);
        int tier = 0;
#pragma unroll
        for (int k = 1; k < kTiers; ++k) tier = (wwarp >= tier_w(k)) ? k : tier;
        switch (tier) {
            case 0: walk<0>(s, i0, ie, g, acc); break;
            case 1: walk<1>(s, i0, ie, g, acc); break;
            case 2: walk<2>(s, i0, ie, g, acc); break;
            case 3: walk<3>(s, i0, ie, g, acc); break;
            case 4: walk<4>(s, i0, ie, g, acc); break;
            default: walk<5>(s, i0, ie, g, acc); break;
        }
    }

    template <int TIER = 0>
    __device__ __forceinline__ void point(const unsigned char* s, int i, const Grid& g, Acc& acc) const
    {
        using namespace f64lean;
        double v[NFP];
#pragma unroll
        for (int k = 0; k < NV2; ++k) {
            const double2 d = reinterpret_cast<const double2*>(s)[k * kChunk + i];
            v[2 * k] = d.x; v[2 * k + 1] = d.y;
        }
        constexpr double kTiny = 1e-300;
#pragma unroll
        for (int j = 0; j < P_; ++j) {
            // |x_i|^2 and rho_i^2(t_q) (times k^2): eq. (8), (25)-(28)
            const double wp = fabs(radius2(g, j, v, iPT)) + kTiny;
            double up, irp;
            sqrt_rsqrt(wp, up, irp);
            (void)irp;
            const double Ep = exp2_neg(up);
            const double Dp = 1.0 + Ep;
            double wm[Q_], um[Q_], irm[Q_], Em[Q_], Dm[Q_];
#pragma unroll
            for (int n = 0; n < Q_; ++n) {
                wm[n] = fabs(radius2(g, j, v, iNODE + C * n)) + kTiny;
                sqrt_rsqrt(wm[n], um[n], irm[n]);
                Em[n] = exp2_neg(um[n]);
                Dm[n] = 1.0 + Em[n];
            }
            double ip, im[Q_];
            if constexpr (Q_ == 1) {
                const double r = rcp_newton(Dp * Dm[0]);                  // 1/((1+E_p)(1+E_m))
                ip = r * Dm[0];
                im[0] = r * Dp;
            } else if constexpr (Q_ == 2) {
                const double PD = Dm[0] * Dm[1];
                const double r = rcp_newton(Dp * PD);
                ip = r * PD;
                const double rDp = r * Dp;
                im[0] = rDp * Dm[1];
                im[1] = rDp * Dm[0];
            } else {
                const double D01 = Dm[0] * Dm[1];
                const double PD = D01 * Dm[2];
                const double r = rcp_newton(Dp * PD);
                ip = r * PD;
                const double rDp = r * Dp;
                im[2] = rDp * D01;
                const double t = rDp * Dm[2];
                im[0] = t * Dm[1];
                im[1] = t * Dm[0];
            }
            acc.sp[j] = fma(Ep * ip, ip, acc.sp[j]);                      // E_p/(1+E_p)^2 = sech^2/4
            double gt = g_node<TIER>(wm[0], irm[0], um[0], Em[0], im[0]);
            if constexpr (Q_ == 2) gt += g_node<TIER>(wm[1], irm[1], um[1], Em[1], im[1]);
            if constexpr (Q_ == 3) {                                      // 5/18 [ g_0 + g_2 + (8/5) g_1 ]
                gt += g_node<TIER>(wm[2], irm[2], um[2], Em[2], im[2]);
                gt = fma(g_node<TIER>(wm[1], irm[1], um[1], Em[1], im[1]), 1.6, gt);
            }
            // k^2 x_i x x_{i+1}, eq. (24)
            double cr = g.Tt[j] * v[iCR + C - 1];
            if (HAS_PHI) cr = fma(-g.ay[j], v[iCR + 1], cr);
            cr = fma(g.ax[j], v[iCR], cr);
            acc.ph[j] = fma(gt, cr, acc.ph[j]);
        }
    }
};

}  // namespace wl
