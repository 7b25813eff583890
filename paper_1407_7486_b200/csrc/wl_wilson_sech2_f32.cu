// wl_wilson_sech2_f32.cu -- k_wilson_sech2_f32: the FP32 hot loop for the sech^2 profile with x_cm on
// the x axis (phi_cm = NULL), i.e. the kernel configs 3, 4 and 5 of BASELINE.json are timed on.
// CUDA path, sm_100a only.  Same mapping, summation order and epilogue as the generic k_wilson
// (wl_eval_kernels.cu); what differs is the per-term arithmetic, which is arranged for the two
// resources that bound it on B200 (profiles/r01_pipe_rates.md):
//
//   * the special-function (XU) pipe, 16 lanes/clk/SM: one warp instruction per 8 clk per
//     sub-partition, and each MUFU also costs two issue slots;
//   * the issue slots, 1 warp instruction/clk/sub-partition.
//
// So (i) the plain FP32 work is issued as PACKED fma/mul/add.f32x2 (FFMA2: two grid points per
// instruction, one issue slot), every thread owning P grid points as P/2 register pairs; (ii) the
// staged loop values enter FFMA2 as both-halves scalar operands, so a staged point costs one LDS.128 and
// one LDS.64 (shared-memory loads return through the same queue as the special-function results: every
// 4 bytes per lane cost about one XU-pipe clock, profiles/r01_pipe_rates.md); (iii) the special-function count per point-eval is 5 or 6:
//       sqrt(|x_i|^2), 2^(-u_p), rsqrt(|m_i|^2), 2^(-u_m), ONE reciprocal 1/((1+E_p)(1+E_m))
//   and log2(1+E_m), the last either on the XU pipe (LOGPOLY = false) or as a degree-8 polynomial
//   in E_m in [0,1] on the FMA pipe (LOGPOLY = true).
//
// Scaling.  With k = 2 log2(e)/lambda all squared radii are carried as w' = k^2 w, so that
// u' = sqrt(w') = 2 log2(e) rho/lambda and E = exp(-2 rho/lambda) = 2^(-u') need no multiply, and
//   h(u)    = ln2 [ (1 - log2(1+E)) - u' E/(1+E) ] / u^2  = 4 log2(e) * br / w'
//   m x d   = (k^2 s c) dy + (k^2 T) (y_i x y_{i+1})       = k^2 (m x d)
// hence phase = eB0 * lambda^2 ln2 * sum_i [br/w'](i) * [k^2 m x d](i): the constants leave the loop.
// Near the axis (w = u^2 < 1/8) the bracket cancels and a degree-3 polynomial in w' replaces br/w'
// (coefficients: gen_h_poly.py hs 0.125 3, relative error 8e-8).
#include "wl_internal.cuh"

namespace wl {

namespace {

constexpr int kThreads = 256;
constexpr int kSumBlock = 32;      // FP32 partial sums span this many terms before they go to FP64
constexpr int kChunk = 1024;       // loop points staged in shared memory at a time (24 B each)

typedef unsigned long long u64;    // two packed floats (lo, hi)

__device__ __forceinline__ u64 pk(float lo, float hi) { u64 r; asm("mov.b64 %0, {%1, %2};" : "=l"(r) : "f"(lo), "f"(hi)); return r; }
__device__ __forceinline__ void upk(u64 v, float& lo, float& hi) { asm("mov.b64 {%0, %1}, %2;" : "=f"(lo), "=f"(hi) : "l"(v)); }
__device__ __forceinline__ u64 fma2(u64 a, u64 b, u64 c) { u64 r; asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(r) : "l"(a), "l"(b), "l"(c)); return r; }
__device__ __forceinline__ u64 mul2(u64 a, u64 b) { u64 r; asm("mul.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(a), "l"(b)); return r; }
__device__ __forceinline__ u64 sub2(u64 a, u64 b) { u64 r; asm("sub.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(a), "l"(b)); return r; }

// XU-pipe instructions; abs / neg become free operand modifiers of MUFU.
__device__ __forceinline__ float xu_sqrt_abs(float x) { float y; asm("sqrt.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(fabsf(x))); return y; }
__device__ __forceinline__ float xu_rsqrt(float x) { float y; asm("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x)); return y; }
__device__ __forceinline__ float xu_ex2_neg(float x) { float y; asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(-x)); return y; }
__device__ __forceinline__ float xu_rcp(float x) { float y; asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x)); return y; }
__device__ __forceinline__ float xu_lg2_abs(float x) { float y; asm("lg2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(fabsf(x))); return y; }

}  // namespace

// DISC = true: the discretisation estimate (eq. (48)-(50)); the two passes, the three levels and the
// partial-sum layout are those of k_wilson<..., DISC = true> in wl_eval_kernels.cu.
template <int P, int THREADS, bool LOGPOLY, int MINB, int UNROLL, int SUMBLOCK, bool DISC>
__global__ void __launch_bounds__(THREADS, MINB)
k_wilson_sech2_f32(EvalArgs a, int n_grid, int n_tiles, int loops_per_unit, int64_t n_units)
{
    static_assert(P % 2 == 0, "grid points are processed as register pairs");
    constexpr int Q = P / 2;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    float4* sPM = reinterpret_cast<float4*>(smem_raw);             // (y_x, |y|^2, ybar_x, |ybar|^2)
    float2* sCr = reinterpret_cast<float2*>(sPM + kChunk);         // (dy_y/2, y_i x y_{i+1})

    const int tid = threadIdx.x;
    const int tile = blockIdx.x % n_tiles;
    const int64_t unit = blockIdx.x / n_tiles;
    const int N = a.n_ppl;
    const double eB0 = a.p0, lambda = a.p1;
    const double k = 2.0 * 1.4426950408889634074 / lambda;
    const double k2 = k * k;

    // ---- per-thread grid-point constants: pair q holds grid points gp[2q] (lo) and gp[2q+1] (hi) ----
    u64 R2p[Q], axp[Q], Ttp[Q];
    int gp[P];
    {
        float R2[P], ax[P], Tt[P];
#pragma unroll
        for (int j = 0; j < P; ++j) {
            gp[j] = tile * (THREADS * P) + j * THREADS + tid;
            const int g = min(gp[j], n_grid - 1);
            const double T = a.T[g / a.n_rho];
            const double rho = a.rho[g % a.n_rho];
            R2[j] = float(k2 * rho * rho);
            ax[j] = float(k2 * 2.0 * sqrt(T) * rho);
            Tt[j] = float(k2 * T);
        }
#pragma unroll
        for (int q = 0; q < Q; ++q) {
            R2p[q] = pk(R2[2 * q], R2[2 * q + 1]);
            axp[q] = pk(ax[2 * q], ax[2 * q + 1]);
            Ttp[q] = pk(Tt[2 * q], Tt[2 * q + 1]);
        }
    }
    const u64 one2 = pk(1.0f, 1.0f), mone2 = pk(-1.0f, -1.0f);
    constexpr float kTiny = 1e-36f;                 // rsqrt(kTiny)^2 is still finite
    constexpr float kPolyBelow = 1.0406844905f;     // w' < this  <=>  u^2 < 1/8
    // h(w)/(4 log2 e) in w' (gen_h_poly.py hs 0.125 3, rel. error 8e-8)
    const u64 h0 = pk(0.086643391691228f, 0.086643391691228f), h1 = pk(-0.0052033291295960f, -0.0052033291295960f),
              h2 = pk(0.00027690498335525f, 0.00027690498335525f), h3 = pk(-1.2801479229129e-5f, -1.2801479229129e-5f);

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
        double dph[P], dsp[P];
#pragma unroll
        for (int j = 0; j < P; ++j) { dph[j] = 0.0; dsp[j] = 0.0; }
        double S2[DISC ? P : 1], B2[DISC ? P : 1];       // pass-0 sums (DISC only)

      const int Nv = DISC ? N / 2 : N;                  // terms per pass
      for (int pass = 0; pass < (DISC ? 2 : 1); ++pass) {
        if (DISC && pass == 1) {
#pragma unroll
            for (int j = 0; j < P; ++j) { S2[j] = dph[j]; B2[j] = dsp[j]; dph[j] = 0.0; dsp[j] = 0.0; }
        }
        for (int c0 = 0; c0 < Nv; c0 += kChunk) {
            const int cn = min(kChunk, Nv - c0);
            __syncthreads();                                  // the previous chunk has been consumed
            for (int i = tid; i < cn; i += THREADS) {         // stage: derived unit-loop quantities, FP64 -> FP32
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
                const float f_yx = float(yx), f_y2 = float(yx * yx + yy * yy);
                const float f_mx = float(mx), f_m2 = float(mx * mx + my * my);
                const float f_hdy = float(0.5 * (zy - yy)), f_cr = float(yx * zy - yy * zx);
                sPM[i] = make_float4(f_yx, f_y2, f_mx, f_m2);
                sCr[i] = make_float2(f_hdy, f_cr);
            }
            __syncthreads();

            for (int i0 = 0; i0 < cn; i0 += SUMBLOCK) {
                u64 ph[Q], sp[Q];
#pragma unroll
                for (int q = 0; q < Q; ++q) { ph[q] = 0ull; sp[q] = 0ull; }       // (+0.0f, +0.0f)
                const int ie = min(i0 + SUMBLOCK, cn);
#pragma unroll UNROLL
                for (int i = i0; i < ie; ++i) {
                    // one LDS.128 + one LDS.64 per staged point (a broadcast: every lane reads the same address);
                    // each scalar feeds FFMA2 as a both-halves operand (SASS: Rn.F32), no duplication in memory
                    const float4 pm = sPM[i];
                    const float2 cs = sCr[i];
                    const ulonglong2 pt = make_ulonglong2(pk(pm.x, pm.x), pk(pm.y, pm.y));
                    const ulonglong2 md = make_ulonglong2(pk(pm.z, pm.z), pk(pm.w, pm.w));
                    const ulonglong2 cx = make_ulonglong2(pk(cs.x, cs.x), pk(cs.y, cs.y));
#pragma unroll
                    for (int q = 0; q < Q; ++q) {
                        // |x_i|^2 and |m_i|^2 (times k^2): eq. (8), (25)-(28)
                        const u64 wp = fma2(Ttp[q], pt.y, fma2(axp[q], pt.x, R2p[q]));
                        u64 wm = fma2(Ttp[q], md.y, fma2(axp[q], md.x, R2p[q]));
                        float wp0, wp1, wm0, wm1;
                        upk(wp, wp0, wp1);
                        upk(wm, wm0, wm1);
                        const float Ep0 = xu_ex2_neg(xu_sqrt_abs(wp0)), Ep1 = xu_ex2_neg(xu_sqrt_abs(wp1));
                        wm0 = fmaxf(wm0, kTiny);
                        wm1 = fmaxf(wm1, kTiny);
                        wm = pk(wm0, wm1);
                        const u64 rm = pk(xu_rsqrt(wm0), xu_rsqrt(wm1));
                        const u64 um = mul2(wm, rm);                              // u' = sqrt(w')
                        float um0, um1;
                        upk(um, um0, um1);
                        const u64 Em = pk(xu_ex2_neg(um0), xu_ex2_neg(um1));
                        const u64 Ep = pk(Ep0, Ep1);
                        const u64 Dp = fma2(Ep, one2, one2);                      //   1 + E_p
                        const u64 Dmn = fma2(Em, mone2, mone2);                   // -(1 + E_m)
                        float dd0, dd1;
                        upk(mul2(Dp, Dmn), dd0, dd1);
                        const u64 i12n = pk(xu_rcp(dd0), xu_rcp(dd1));            // -1/((1+E_p)(1+E_m))
                        const u64 ip = mul2(i12n, Dmn);                           //  1/(1+E_p)
                        const u64 imn = mul2(i12n, Dp);                           // -1/(1+E_m)
                        sp[q] = fma2(mul2(Ep, ip), ip, sp[q]);                    // E_p/(1+E_p)^2 = sech^2/4
                        u64 br;                                                   // (1 - log2(1+E_m)) - u' E_m/(1+E_m)
                        if (LOGPOLY) {
                            // 1 - log2(1+E), E in [0,1]: gen_h_poly.py L 8, abs. error 6e-8
                            u64 L = pk(0.00866569930832f, 0.00866569930832f);
                            L = fma2(L, Em, pk(-0.0494333683912f, -0.0494333683912f));
                            L = fma2(L, Em, pk(0.13314692741f, 0.13314692741f));
                            L = fma2(L, Em, pk(-0.238041983614f, -0.238041983614f));
                            L = fma2(L, Em, pk(0.345429336575f, 0.345429336575f));
                            L = fma2(L, Em, pk(-0.478176441505f, -0.478176441505f));
                            L = fma2(L, Em, pk(0.721095768202f, 0.721095768202f));
                            L = fma2(L, Em, pk(-1.44268585129f, -1.44268585129f));
                            // last Horner step folded with the second term: 1 - log2(1+E) = c0 + E L'(E) and
                            // -u' E/(1+E) = E (u' imn), so br = c0 + E (L' + u' imn): one instruction fewer
                            br = fma2(fma2(um, imn, L), Em, pk(0.999999943578f, 0.999999943578f));
                        } else {
                            float dm0, dm1;
                            upk(Dmn, dm0, dm1);
                            br = sub2(fma2(um, mul2(Em, imn), one2), pk(xu_lg2_abs(dm0), xu_lg2_abs(dm1)));
                        }
                        const u64 hE = mul2(br, mul2(rm, rm));                    // br / w'
                        u64 hP = fma2(h3, wm, h2);
                        hP = fma2(hP, wm, h1);
                        hP = fma2(hP, wm, h0);
                        float hE0, hE1, hP0, hP1;
                        upk(hE, hE0, hE1);
                        upk(hP, hP0, hP1);
                        const u64 gt = pk(wm0 < kPolyBelow ? hP0 : hE0, wm1 < kPolyBelow ? hP1 : hE1);
                        const u64 cr = fma2(axp[q], cx.x, mul2(Ttp[q], cx.y));    // k^2 (m x d), eq. (24)
                        ph[q] = fma2(gt, cr, ph[q]);
                    }
                }
#pragma unroll
                for (int q = 0; q < Q; ++q) {
                    float p0, p1, s0, s1;
                    upk(ph[q], p0, p1);
                    upk(sp[q], s0, s1);
                    dph[2 * q] += double(p0); dph[2 * q + 1] += double(p1);
                    dsp[2 * q] += double(s0); dsp[2 * q + 1] += double(s1);
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
                const double phase = g_scale * dph[j];
                const double spin = b_scale * (T / double(N)) * dsp[j];
                const double W = a.scalar ? cos(phase) : cos(phase) * cosh(spin);
                Wsum[0][j] += W;
                if (gp[j] < n_grid) {
                    if (a.phase_out) a.phase_out[loop * n_grid + gp[j]] = phase;
                    if (a.spin_out) a.spin_out[loop * n_grid + gp[j]] = spin;
                }
            } else {
                const double S4 = dph[j], B4 = dsp[j], c = b_scale * (T / double(N));
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

// plan.P grid points per thread; P = 1 (tiny grids) runs as a half-empty pair.
cudaError_t launch_wilson_sech2_f32(const EvalPlan& plan, const EvalArgs& a, cudaStream_t s)
{
    const size_t smem = (sizeof(float4) + sizeof(float2)) * (size_t)kChunk;
    // Grids of at most 256 points: 128 threads x 2 grid points, so that no thread of the tile idles.
    const bool small = plan.n_grid <= 256;
    const int n_tiles = small ? 1 : plan.n_tiles;
    const int64_t n_ctas = plan.n_units * n_tiles;
    if (n_ctas > 0x7fffffffLL) return cudaErrorInvalidConfiguration;
    const unsigned g = (unsigned)n_ctas;
    // 256 threads x P = 4, 4 CTAs/SM (64 registers), inner loop unrolled by 2: the fastest of the
    // combinations measured (profiles/r01_variants.md).
#define WL_LAUNCH(PP, TH, DD) k_wilson_sech2_f32<PP, TH, true, 4, 2, kSumBlock, DD><<<g, TH, smem, s>>>(a, plan.n_grid, n_tiles, plan.loops_per_unit, plan.n_units)
    if (a.disc) {
        if (small) WL_LAUNCH(2, 128, true);
        else if (plan.P == 2) WL_LAUNCH(2, kThreads, true);
        else if (plan.P == 4) WL_LAUNCH(4, kThreads, true);
        else return cudaErrorInvalidValue;
    } else {
        if (small) WL_LAUNCH(2, 128, false);
        else if (plan.P == 2) WL_LAUNCH(2, kThreads, false);
        else if (plan.P == 4) WL_LAUNCH(4, kThreads, false);
        else return cudaErrorInvalidValue;
    }
#undef WL_LAUNCH
    return cudaGetLastError();
}

}  // namespace wl
