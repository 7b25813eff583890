// wl_wilson_sech2_f64.cu -- k_wilson_sech2_f64: the FP64 hot loop for the sech^2 profile with x_cm on
// the x axis (phi_cm = NULL): configs 1 and 4 (FP64 variant) of BASELINE.json.  CUDA path, sm_100a.
// Same mapping, summation order and epilogue as the generic k_wilson<double, Sech2, ...>; what differs is
// that every elementary function is written out branch-free for the FP64 pipe (64 lanes/clk/SM, DFMA
// = 2 clk per warp instruction per sub-partition, profiles/r01_pipe_rates.md) instead of calling the
// general-purpose exp / log1p / sqrt / division sequences (~200 FP64-pipe instructions per point-eval
// with slow-path branches):
//
//   sqrt, 1/w : MUFU.RSQ64H seed + two coupled Newton (Goldschmidt) steps + one residual correction
//   2^(-u)    : round-to-nearest split u = n + f via the 1.5*2^52 trick, degree-10 polynomial in f,
//               exponent adjusted with integer adds (E = exp(-2 rho/lambda) = 2^(-u'), u' = sqrt(w'))
//   1/((1+E_p)(1+E_m)) : ONE MUFU.RCP64H seed + two Newton steps, shared by point and midpoint
//   1 - log2(1+E_m)    : degree-20 polynomial in E_m in [0,1]
//   near the axis (u^2 < 1/16): degree-7 polynomial in w' for the cancelling bracket (reading A4)
// about 100 FP64-pipe instructions per point-eval.  Coefficients: gen_h_poly.py (E2 10, L 20, hs 0.0625 7).
// Scaling as in wl_wilson_sech2_f32.cu: all squared radii carried as w' = (2 log2(e)/lambda)^2 w.
#include "wl_internal.cuh"

namespace wl {

namespace {

constexpr int kThreads = 256;
constexpr int kChunk = 512;        // loop points staged in shared memory at a time (48 B each)

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

// (1 - log2(1+E)) - u E/(1+E) for E in [0,1], im = 1/(1+E).  With the degree-20 polynomial
// 1 - log2(1+E) = c0 + E L'(E) the second term joins the last Horner step: c0 + E (L'(E) - u im).
__device__ __forceinline__ double bracket(double E, double u, double im)
{
    double L = kLog[0];
#pragma unroll
    for (int i = 1; i < 20; ++i) L = fma(L, E, kLog[i]);
    return fma(fma(-u, im, L), E, kLog[20]);
}

}  // namespace

// DISC = true: the discretisation estimate (eq. (48)-(50)); the two passes, the three levels and the
// partial-sum layout are those of k_wilson<..., DISC = true> in wl_eval_kernels.cu.
template <int P, bool DISC>
__global__ void __launch_bounds__(kThreads, 2)
k_wilson_sech2_f64(EvalArgs a, int n_grid, int n_tiles, int loops_per_unit, int64_t n_units)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    double2* sPt = reinterpret_cast<double2*>(smem_raw);      // (y_x, |y|^2)
    double2* sMid = sPt + kChunk;                             // (ybar_x, |ybar|^2)
    double2* sCr = sMid + kChunk;                             // (dy_y/2, y_i x y_{i+1})

    const int tid = threadIdx.x;
    const int tile = blockIdx.x % n_tiles;
    const int64_t unit = blockIdx.x / n_tiles;
    const int N = a.n_ppl;
    const double eB0 = a.p0, lambda = a.p1;
    const double k = 2.0 * 1.4426950408889634074 / lambda;
    const double k2 = k * k;

    double R2[P], ax[P], Tt[P];
    int gp[P];
#pragma unroll
    for (int j = 0; j < P; ++j) {
        gp[j] = tile * (kThreads * P) + j * kThreads + tid;
        const int g = min(gp[j], n_grid - 1);
        const double T = a.T[g / a.n_rho];
        const double rho = a.rho[g % a.n_rho];
        R2[j] = k2 * rho * rho;
        ax[j] = k2 * 2.0 * sqrt(T) * rho;
        Tt[j] = k2 * T;
    }
    constexpr double kTiny = 1e-300;
    constexpr double kPolyBelow = 0.52034224525;         // w' < this  <=>  u^2 < 1/16

    constexpr int kLevels = DISC ? 3 : 1;
    double Wsum[kLevels][P];
#pragma unroll
    for (int v = 0; v < kLevels; ++v)
#pragma unroll
        for (int j = 0; j < P; ++j) Wsum[v][j] = 0.0;

    for (int ll = 0; ll < loops_per_unit; ++ll) {
        const int64_t loop = unit * loops_per_unit + ll;
        const double2* L64 = reinterpret_cast<const double2*>(a.loops) + loop * N;
        const float2* L32 = reinterpret_cast<const float2*>(a.loops) + loop * N;
        double ph[P], sp[P];
#pragma unroll
        for (int j = 0; j < P; ++j) { ph[j] = 0.0; sp[j] = 0.0; }
        double S2[DISC ? P : 1], B2[DISC ? P : 1];       // pass-0 sums (DISC only)

      const int Nv = DISC ? N / 2 : N;                  // terms per pass
      for (int pass = 0; pass < (DISC ? 2 : 1); ++pass) {
        if (DISC && pass == 1) {
#pragma unroll
            for (int j = 0; j < P; ++j) { S2[j] = ph[j]; B2[j] = sp[j]; ph[j] = 0.0; sp[j] = 0.0; }
        }
        for (int c0 = 0; c0 < Nv; c0 += kChunk) {
            const int cn = min(kChunk, Nv - c0);
            __syncthreads();                                  // the previous chunk has been consumed
            for (int i = tid; i < cn; i += kThreads) {        // stage: derived unit-loop quantities
                int n = c0 + i;
                int n1 = (n + 1 == N) ? 0 : n + 1;            // closed loop, i+1 mod N
                if (DISC) {                                   // sub-worldline: every 2nd / 4th point, closed on itself
                    n = pass + 2 * (c0 + i);
                    n1 = n + (pass ? 4 : 2);
                    if (n1 >= N) n1 -= N;
                }
                double yx, yy, zx, zy;
                if (a.loops_are_f64) {
                    const double2 u = L64[n], v = L64[n1];
                    yx = u.x; yy = u.y; zx = v.x; zy = v.y;
                } else {
                    const float2 u = L32[n], v = L32[n1];
                    yx = u.x; yy = u.y; zx = v.x; zy = v.y;
                }
                const double mx = 0.5 * (yx + zx), my = 0.5 * (yy + zy);
                sPt[i] = make_double2(yx, yx * yx + yy * yy);
                sMid[i] = make_double2(mx, mx * mx + my * my);
                sCr[i] = make_double2(0.5 * (zy - yy), yx * zy - yy * zx);
            }
            __syncthreads();

            for (int i = 0; i < cn; ++i) {
                const double2 pt = sPt[i];
                const double2 md = sMid[i];
                const double2 cx = sCr[i];
#pragma unroll
                for (int j = 0; j < P; ++j) {
                    // |x_i|^2 and |m_i|^2 (times k^2): eq. (8), (25)-(28)
                    const double wp = fabs(fma(Tt[j], pt.y, fma(ax[j], pt.x, R2[j]))) + kTiny;
                    const double wm = fabs(fma(Tt[j], md.y, fma(ax[j], md.x, R2[j]))) + kTiny;
                    double up, irp, um, irm;
                    sqrt_rsqrt(wp, up, irp);
                    sqrt_rsqrt(wm, um, irm);
                    (void)irp;
                    const double Ep = exp2_neg(up), Em = exp2_neg(um);
                    const double Dp = 1.0 + Ep, Dm = 1.0 + Em;
                    const double DD = Dp * Dm;
                    double r = xu_rcp64(DD);                                  // 1/((1+E_p)(1+E_m))
                    double e = fma(-DD, r, 1.0);
                    r = fma(r, e, r);
                    e = fma(-DD, r, 1.0);
                    r = fma(r, e, r);
                    const double ip = r * Dm, im = r * Dp;
                    sp[j] = fma(Ep * ip, ip, sp[j]);                          // E_p/(1+E_p)^2 = sech^2/4
                    const double br = bracket(Em, um, im);                    // (1 - log2(1+E_m)) - u' E_m/(1+E_m)
                    const double hE = br * (irm * irm);                       // br / w'
                    // h(w)/(4 log2 e) in w', w = u^2 < 1/16 (gen_h_poly.py hs 0.0625 7)
                    double hP = kHPoly[0];
#pragma unroll
                    for (int i = 1; i < 8; ++i) hP = fma(hP, wm, kHPoly[i]);
                    const double gt = (wm < kPolyBelow) ? hP : hE;
                    const double cr = fma(ax[j], cx.x, Tt[j] * cx.y);         // k^2 (m x d), eq. (24)
                    ph[j] = fma(gt, cr, ph[j]);
                }
            }
        }

      }   // pass

        // ---- W = cos(phase) cosh(spin), FP64, once per (loop, grid point): eq. (18), PAPER.md:121 ----
        const double g_scale = eB0 * lambda * lambda * 0.69314718055994530942;
        const double b_scale = 4.0 * eB0;
#pragma unroll
        for (int j = 0; j < P; ++j) {
            const int g = min(gp[j], n_grid - 1);
            const double T = a.T[g / a.n_rho];
            if (!DISC) {
                const double phase = g_scale * ph[j];
                const double spin = b_scale * (T / double(N)) * sp[j];
                const double W = a.scalar ? cos(phase) : cos(phase) * cosh(spin);
                Wsum[0][j] += W;
                if (gp[j] < n_grid) {
                    if (a.phase_out) a.phase_out[loop * n_grid + gp[j]] = phase;
                    if (a.spin_out) a.spin_out[loop * n_grid + gp[j]] = spin;
                }
            } else {
                const double S4 = ph[j], B4 = sp[j], c = b_scale * (T / double(N));
                const double phase[3] = {g_scale * (0.5 * S4), g_scale * S2[j], g_scale * (0.5 * S2[j] + 0.25 * S4)};   // eq. (48)-(50)
                const double spin[3] = {2.0 * c * B4, 2.0 * c * B2[j], c * (B2[j] + B4)};
#pragma unroll
                for (int v = 0; v < 3; ++v)
                    Wsum[v][j] += a.scalar ? cos(phase[v]) : cos(phase[v]) * cosh(spin[v]);
            }
        }
    }
#pragma unroll
    for (int v = 0; v < kLevels; ++v)
#pragma unroll
        for (int j = 0; j < P; ++j)
            if (gp[j] < n_grid) a.partial[((int64_t)v * n_units + unit) * n_grid + gp[j]] = Wsum[v][j];
}

cudaError_t launch_wilson_sech2_f64(const EvalPlan& plan, const EvalArgs& a, cudaStream_t s)
{
    const size_t smem = 3 * sizeof(double2) * (size_t)kChunk;
    const int64_t n_ctas = plan.n_units * plan.n_tiles;
    if (n_ctas > 0x7fffffffLL) return cudaErrorInvalidConfiguration;
    const unsigned g = (unsigned)n_ctas;
#define WL_LAUNCH(PP, DD) k_wilson_sech2_f64<PP, DD><<<g, kThreads, smem, s>>>(a, plan.n_grid, plan.n_tiles, plan.loops_per_unit, plan.n_units)
    if (a.disc) {
        switch (plan.P) {
            case 1: WL_LAUNCH(1, true); break;
            case 2: WL_LAUNCH(2, true); break;
            default: return cudaErrorInvalidValue;
        }
    } else {
        switch (plan.P) {
            case 1: WL_LAUNCH(1, false); break;
            case 2: WL_LAUNCH(2, false); break;
            default: return cudaErrorInvalidValue;
        }
    }
#undef WL_LAUNCH
    return cudaGetLastError();
}

}  // namespace wl
