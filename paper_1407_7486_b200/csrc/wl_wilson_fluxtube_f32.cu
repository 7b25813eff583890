// wl_wilson_fluxtube_f32.cu -- k_wilson_fluxtube_f32: the FP32 hot loop for the paper's own validation
// profile f_lambda = rho^2/(lambda^2+rho^2) (eq. (68); Fig. 11, 12) with x_cm on the x axis
// (phi_cm = NULL).  CUDA path, sm_100a only.  Same mapping, staging, summation order and epilogue as
// k_wilson_fluxtube_f32 (wl_wilson_sech2_f32.cu); the per-term arithmetic is
//     g = script-F/(lambda^2 + |m|^2),   b = 2 script-F lambda^2/(lambda^2 + |x|^2)^2      (eq. (14), (15), (17))
// With all squared radii carried as a = 1 + w/lambda^2 (the "+1" sits in the grid-point constant):
//     g = (script-F/lambda^2)/a_m,   b = (2 script-F/lambda^2)/a_p^2,   m x d carried as (m x d)/lambda^2
// so a point-eval is 11.5 packed FMA-pipe instructions and ONE special-function op (the reciprocal of
// a_p a_m, shared by point and midpoint): the kernel is FMA-pipe bound, not XU bound.  No square root:
// the profile is a function of rho^2, as PAPER.md:149 advises.
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

// XU-pipe instruction.
__device__ __forceinline__ float xu_rcp(float x) { float y; asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x)); return y; }

}  // namespace

// DISC = true: the discretisation estimate (eq. (48)-(50)); the two passes, the three levels and the
// partial-sum layout are those of k_wilson<..., DISC = true> in wl_eval_kernels.cu.
template <int P, int THREADS, int MINB, int UNROLL, int SUMBLOCK, bool DISC>
__global__ void __launch_bounds__(THREADS, MINB)
k_wilson_fluxtube_f32(EvalArgs a, int n_grid, int n_tiles, int loops_per_unit, int64_t n_units)
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
    const double F = a.p0, lambda = a.p1;             // script-F = eF/2pi (eq. (17)), lambda
    const double k2 = 1.0 / (lambda * lambda);

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
            R2[j] = float(1.0 + k2 * rho * rho);         // a = 1 + w/lambda^2
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
                        // a_p = 1 + |x_i|^2/lambda^2, a_m = 1 + |m_i|^2/lambda^2: eq. (8), (25)-(28)
                        const u64 ap = fma2(Ttp[q], pt.y, fma2(axp[q], pt.x, R2p[q]));
                        const u64 am = fma2(Ttp[q], md.y, fma2(axp[q], md.x, R2p[q]));
                        float d0, d1;
                        upk(mul2(ap, am), d0, d1);
                        const u64 r = pk(xu_rcp(d0), xu_rcp(d1));                 // 1/(a_p a_m): one reciprocal for both
                        const u64 ip = mul2(r, am);                               // 1/a_p
                        const u64 gt = mul2(r, ap);                               // 1/a_m          -> g
                        sp[q] = fma2(ip, ip, sp[q]);                              // 1/a_p^2        -> b
                        const u64 cr = fma2(axp[q], cx.x, mul2(Ttp[q], cx.y));    // (m x d)/lambda^2, eq. (24)
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
        const double g_scale = F;                       // (F/lambda^2) x lambda^2 from the scaled cross term
        const double b_scale = 2.0 * F * k2;
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
cudaError_t launch_wilson_fluxtube_f32(const EvalPlan& plan, const EvalArgs& a, cudaStream_t s)
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
#define WL_LAUNCH(PP, TH, DD) k_wilson_fluxtube_f32<PP, TH, 4, 2, kSumBlock, DD><<<g, TH, smem, s>>>(a, plan.n_grid, n_tiles, plan.loops_per_unit, plan.n_units)
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
