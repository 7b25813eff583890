// wl_eval_kernels.cu -- k_wilson (the hot loop), k_group_reduce, k_mean.   CUDA path, sm_100a.
//
// Mapping.  One CTA = (one unit of `loops_per_unit` consecutive loops)
// x (one tile of kThreads*P grid points).  LANES RUN OVER GRID POINTS, each thread owns P
// grid points in registers; the loop is staged chunk by chunk in shared memory as derived
// per-point / per-segment quantities of the UNIT loop, and every thread walks the staged
// points serially: all lanes of a warp read the same shared-memory address (a broadcast),
// and every sum round the loop is taken by one thread in index order.  No shuffles, no
// atomics: the result does not depend on how CTAs are scheduled.
//
// Algebra (eq. (8), (21)-(24)), with c = x_cm, s = sqrt(T), unit-loop
// point y_i, midpoint ybar_i = (y_i + y_{i+1})/2, step dy_i = y_{i+1} - y_i:
//     |x_i|^2 = |c|^2 + 2 s (c . y_i)    + T |y_i|^2
//     |m_i|^2 = |c|^2 + 2 s (c . ybar_i) + T |ybar_i|^2
//     m_i x d_i = s (c x dy_i) + T (y_i x y_{i+1})
// so per term the grid point contributes (|c|^2, 2 s c, T, s c) and the loop contributes
// (y_i, |y_i|^2, ybar_i, |ybar_i|^2, dy_i, y_i x y_{i+1}), the latter computed once per
// staged point in FP64.  With phi_cm = 0 (c on the x axis) half of those drop out.
#include "wl_field_device.cuh"
#include "wl_internal.cuh"

namespace wl {

constexpr int kThreads = 256;
constexpr int kSumBlock = 32;     // FP32 partial sums span this many terms before they go to FP64

template <typename Real> struct alignas(16) Vec4 { Real a, b, c, d; };
template <typename Real> struct alignas(2 * sizeof(Real)) Vec2 { Real a, b; };

// DISC = true: the discretisation estimate of Sec. IV.A (eq. (48)-(50)).  Each loop is
// walked as two VIRTUAL loops of N/2 terms: pass 0 = the even points with neighbour +2 (the "circle"
// sub-worldline, N/2 points), pass 1 = the odd points with neighbour +4 (the "box" and "triangle"
// sub-worldlines, N/4 points each, summed together).  With S2, S4 the phase sums and B2, B4 the spin
// sums of the two passes, the three levels are
//   N/4: phase = S4/2,          spin = 2 (T/N) B4      (mean of the two N/4 sub-worldlines)
//   N/2: phase = S2,            spin = 2 (T/N) B2
//   N  : phase = S2/2 + S4/4,   spin = (T/N)(B2 + B4)
// and the partial sums are written level-major: partial[level][unit][grid].
template <typename Real, template <typename> class Prof, bool HAS_PHI, int P, bool DISC>
__global__ void __launch_bounds__(kThreads)
k_wilson(EvalArgs a, int n_grid, int n_tiles, int loops_per_unit, int chunk_points, int64_t n_units)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    Vec4<Real>* sSeg = reinterpret_cast<Vec4<Real>*>(smem_raw);            // (ybar_x, |ybar|^2, dy_y, y_i x y_{i+1})
    Vec2<Real>* sPt = reinterpret_cast<Vec2<Real>*>(sSeg + chunk_points);  // (y_x, |y|^2)
    Vec4<Real>* sExt = reinterpret_cast<Vec4<Real>*>(sPt + chunk_points);  // (ybar_y, dy_x, y_y, -)   HAS_PHI only

    const int tid = threadIdx.x;
    const int tile = blockIdx.x % n_tiles;
    const int64_t unit = blockIdx.x / n_tiles;
    const int N = a.n_ppl;
    const Prof<Real> prof(a.p0, a.p1);

    // ---- per-thread grid-point constants (FP64 on the way in, then the compute type) ----
    Real R2[P], ax[P], Tt[P], scx[P];
    Real ay[HAS_PHI ? P : 1], scy[HAS_PHI ? P : 1];
    int gp[P];
#pragma unroll
    for (int j = 0; j < P; ++j) {
        gp[j] = tile * (kThreads * P) + j * kThreads + tid;
        const int g = min(gp[j], n_grid - 1);
        const double T = a.T[g / a.n_rho];
        const double rho = a.rho[g % a.n_rho];
        const double s = sqrt(T);
        double cx = rho, cy = 0.0;
        if (HAS_PHI) { const double ph = a.phi[g % a.n_rho]; cx = rho * cos(ph); cy = rho * sin(ph); }
        R2[j] = Real(rho * rho);
        ax[j] = Real(2.0 * s * cx);
        Tt[j] = Real(T);
        scx[j] = Real(s * cx);
        if (HAS_PHI) { ay[j] = Real(2.0 * s * cy); scy[j] = Real(s * cy); }
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
        double S2[DISC ? P : 1], B2[DISC ? P : 1];       // pass-0 sums (DISC only)
#pragma unroll
        for (int j = 0; j < P; ++j) { dph[j] = 0.0; dsp[j] = 0.0; }

      const int Nv = DISC ? N / 2 : N;                  // terms per pass
      for (int pass = 0; pass < (DISC ? 2 : 1); ++pass) {
        if (DISC && pass == 1) {
#pragma unroll
            for (int j = 0; j < P; ++j) { S2[j] = dph[j]; B2[j] = dsp[j]; dph[j] = 0.0; dsp[j] = 0.0; }
        }
        for (int c0 = 0; c0 < Nv; c0 += chunk_points) {
            const int cn = min(chunk_points, Nv - c0);
            __syncthreads();                                  // the previous chunk has been consumed
            for (int i = tid; i < cn; i += kThreads) {        // stage: derived unit-loop quantities, FP64
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
                Vec4<Real> sg; sg.a = Real(mx); sg.b = Real(mx * mx + my * my); sg.c = Real(zy - yy); sg.d = Real(yx * zy - yy * zx);
                Vec2<Real> pt; pt.a = Real(yx); pt.b = Real(yx * yx + yy * yy);
                sSeg[i] = sg;
                sPt[i] = pt;
                if (HAS_PHI) { Vec4<Real> ex; ex.a = Real(my); ex.b = Real(zx - yx); ex.c = Real(yy); ex.d = Real(0); sExt[i] = ex; }
            }
            __syncthreads();

            for (int i0 = 0; i0 < cn; i0 += kSumBlock) {
                Real ph[P], sp[P];
#pragma unroll
                for (int j = 0; j < P; ++j) { ph[j] = Real(0); sp[j] = Real(0); }
                const int ie = min(i0 + kSumBlock, cn);
#pragma unroll 2
                for (int i = i0; i < ie; ++i) {
                    const Vec4<Real> sg = sSeg[i];
                    const Vec2<Real> pt = sPt[i];
                    Vec4<Real> ex;
                    if (HAS_PHI) ex = sExt[i];
#pragma unroll
                    for (int j = 0; j < P; ++j) {
                        Real cr = scx[j] * sg.c;
                        if (HAS_PHI) cr = fma(-scy[j], ex.b, cr);
                        cr = fma(Tt[j], sg.d, cr);                       // m x d
                        Real bt, gt;
                        if (Prof<Real>::kNeedsRadius) {
                            Real wp = fma(ax[j], pt.a, R2[j]);
                            Real wm = fma(ax[j], sg.a, R2[j]);
                            if (HAS_PHI) { wp = fma(ay[j], ex.c, wp); wm = fma(ay[j], ex.a, wm); }
                            wp = fma(Tt[j], pt.b, wp);                   // |x_i|^2
                            wm = fma(Tt[j], sg.b, wm);                   // |m_i|^2
                            prof.terms(wp, wm, bt, gt);
                        } else {
                            prof.terms(Real(0), Real(0), bt, gt);
                        }
                        ph[j] = fma(gt, cr, ph[j]);
                        sp[j] += bt;
                    }
                }
#pragma unroll
                for (int j = 0; j < P; ++j) { dph[j] += double(ph[j]); dsp[j] += double(sp[j]); }
            }
        }

      }   // pass

        // ---- W = cos(phase) cosh(spin), FP64, once per (loop, grid point): eq. (18), PAPER.md:121 ----
#pragma unroll
        for (int j = 0; j < P; ++j) {
            const int g = min(gp[j], n_grid - 1);
            const double T = a.T[g / a.n_rho];
            if (!DISC) {
                const double phase = prof.g_scale() * dph[j];
                const double spin = prof.b_scale() * (T / double(N)) * dsp[j];
                const double W = a.scalar ? cos(phase) : cos(phase) * cosh(spin);
                Wsum[0][j] += W;
                if (gp[j] < n_grid) {
                    if (a.phase_out) a.phase_out[loop * n_grid + gp[j]] = phase;
                    if (a.spin_out) a.spin_out[loop * n_grid + gp[j]] = spin;
                }
            } else {
                const double S4 = dph[j], B4 = dsp[j];
                const double gs = prof.g_scale(), c = prof.b_scale() * (T / double(N));
                const double phase[3] = {gs * (0.5 * S4), gs * S2[j], gs * (0.5 * S2[j] + 0.25 * S4)};   // eq. (48)-(50)
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

// S_g = sum over the units of group g, in unit order (eq. (60)).
__global__ void k_group_reduce(const double* __restrict__ partial, int units_per_group, int n_grid,
                               double* __restrict__ group_sums)
{
    const int k = blockIdx.x * blockDim.x + threadIdx.x;
    const int g = blockIdx.y;
    if (k >= n_grid) return;
    const double* p = partial + (int64_t)g * units_per_group * n_grid + k;
    double S = 0.0;
    for (int c = 0; c < units_per_group; ++c) S += p[(int64_t)c * n_grid];
    group_sums[(int64_t)g * n_grid + k] = S;
}

// <W> = (sum_g S_g)/N_l in group order (eq. (61)-(62)).
__global__ void k_mean(const double* __restrict__ group_sums, int n_groups, int n_grid, double n_loops,
                       double* __restrict__ W_mean)
{
    const int k = blockIdx.x * blockDim.x + threadIdx.x;
    if (k >= n_grid) return;
    double total = 0.0;
    for (int g = 0; g < n_groups; ++g) total += group_sums[(int64_t)g * n_grid + k];
    W_mean[k] = total / n_loops;
}

// ------------------------------------------------------------------ host side: plan + dispatch

EvalPlan make_eval_plan(int64_t n_loops, int n_ppl, int n_T, int n_rho, int n_groups, wl_dtype compute,
                        bool per_loop)
{
    EvalPlan p;
    p.n_grid = n_T * n_rho;
    p.threads = kThreads;
    const int p_max = (compute == WL_F32) ? 4 : 2;
    p.P = 1;
    while (p.P < p_max && p.n_grid >= kThreads * p.P * 2) p.P *= 2;
    p.n_tiles = (p.n_grid + kThreads * p.P - 1) / (kThreads * p.P);
    const int64_t per_group = n_loops / n_groups;
    // Largest divisor of the group size, at most 8, that still leaves enough CTAs to balance
    // a 148-SM part over many waves.  A function of the sizes only: the summation order, and
    // with it every bit of the result, is the same on any device.
    p.loops_per_unit = 1;
    if (!per_loop) {
        for (int d = 8; d > 1; --d)
            if (per_group % d == 0 && (n_loops / d) * p.n_tiles >= 4096) { p.loops_per_unit = d; break; }
    }
    p.n_units = n_loops / p.loops_per_unit;
    p.units_per_group = (int)(per_group / p.loops_per_unit);
    p.chunk_points = (compute == WL_F32) ? 1024 : 512;
    if (p.chunk_points > n_ppl) p.chunk_points = (n_ppl + kSumBlock - 1) / kSumBlock * kSumBlock;
    return p;
}

template <typename Real, template <typename> class Prof, bool HAS_PHI, int P, bool DISC>
static cudaError_t launch_one(const EvalPlan& plan, const EvalArgs& a, cudaStream_t s)
{
    const size_t per_point = sizeof(Vec4<Real>) + sizeof(Vec2<Real>) + (HAS_PHI ? sizeof(Vec4<Real>) : 0);
    const size_t smem = per_point * (size_t)plan.chunk_points;
    const int64_t n_ctas = plan.n_units * plan.n_tiles;
    if (n_ctas > 0x7fffffffLL) return cudaErrorInvalidConfiguration;
    k_wilson<Real, Prof, HAS_PHI, P, DISC><<<(unsigned)n_ctas, kThreads, smem, s>>>(
        a, plan.n_grid, plan.n_tiles, plan.loops_per_unit, plan.chunk_points, plan.n_units);
    return cudaGetLastError();
}

template <typename Real, template <typename> class Prof, bool HAS_PHI>
static cudaError_t launch_p(const EvalPlan& plan, const EvalArgs& a, cudaStream_t s)
{
    if (a.disc) {                                        // discretisation estimate: P <= 2 (three W per grid point)
        switch (plan.P) {
            case 1: return launch_one<Real, Prof, HAS_PHI, 1, true>(plan, a, s);
            case 2: return launch_one<Real, Prof, HAS_PHI, 2, true>(plan, a, s);
            default: return cudaErrorInvalidValue;
        }
    }
    switch (plan.P) {
        case 1: return launch_one<Real, Prof, HAS_PHI, 1, false>(plan, a, s);
        case 2: return launch_one<Real, Prof, HAS_PHI, 2, false>(plan, a, s);
        case 4: if (sizeof(Real) == 4) return launch_one<Real, Prof, HAS_PHI, (sizeof(Real) == 4 ? 4 : 2), false>(plan, a, s);
        default: return cudaErrorInvalidValue;
    }
}

template <typename Real>
static cudaError_t launch_r(const EvalPlan& plan, const EvalArgs& a, int profile, cudaStream_t s)
{
    const bool phi = a.phi != nullptr;
    if (profile == WL_PROFILE_UNIFORM)
        return phi ? launch_p<Real, Uniform, true>(plan, a, s) : launch_p<Real, Uniform, false>(plan, a, s);
    if (profile == WL_PROFILE_SECH2)
        return phi ? launch_p<Real, Sech2, true>(plan, a, s) : launch_p<Real, Sech2, false>(plan, a, s);
    if (profile == WL_PROFILE_FLUXTUBE)
        return phi ? launch_p<Real, FluxTube, true>(plan, a, s) : launch_p<Real, FluxTube, false>(plan, a, s);
    return cudaErrorInvalidValue;
}

cudaError_t launch_wilson(const EvalPlan& plan, const EvalArgs& a, int profile, wl_dtype compute, cudaStream_t s)
{
    // The lean sech^2 kernels carry squared radii scaled by (2 log2(e)/lambda)^2; outside this range of
    // lambda the FP32 one could overflow or flush, so the generic kernel (unscaled) serves it.
    const bool lambda_ok = a.p1 >= 1e-4 && a.p1 <= 1e4;
    if (compute == WL_F32 && profile == WL_PROFILE_SECH2 && a.phi == nullptr && lambda_ok) {
        EvalPlan p2 = plan;                              // grid points go in register pairs there
        if (p2.P < 2) { p2.P = 2; p2.n_tiles = (p2.n_grid + kThreads * 2 - 1) / (kThreads * 2); }
        if (a.disc && p2.P == 2 && p2.n_grid >= kThreads * 8) {   // the discretisation plan caps P at 2 for the generic kernel
            p2.P = 4;
            p2.n_tiles = (p2.n_grid + kThreads * 4 - 1) / (kThreads * 4);
        }
        return launch_wilson_sech2_f32(p2, a, s);
    }
    if (compute == WL_F32 && profile == WL_PROFILE_FLUXTUBE && a.phi == nullptr && lambda_ok) {
        EvalPlan p2 = plan;
        if (p2.P < 2) { p2.P = 2; p2.n_tiles = (p2.n_grid + kThreads * 2 - 1) / (kThreads * 2); }
        if (a.disc && p2.P == 2 && p2.n_grid >= kThreads * 8) {
            p2.P = 4;
            p2.n_tiles = (p2.n_grid + kThreads * 4 - 1) / (kThreads * 4);
        }
        return launch_wilson_fluxtube_f32(p2, a, s);
    }
    if (compute == WL_F64 && profile == WL_PROFILE_SECH2 && a.phi == nullptr)
        return launch_wilson_sech2_f64(plan, a, s);
    return compute == WL_F32 ? launch_r<float>(plan, a, profile, s) : launch_r<double>(plan, a, profile, s);
}

cudaError_t launch_group_reduce(const double* partial, int64_t n_units, int units_per_group, int n_groups,
                                int n_grid, int64_t n_loops, double* group_sums, double* W_mean,
                                cudaStream_t s)
{
    (void)n_units;
    const dim3 grid((n_grid + 255) / 256, n_groups);
    k_group_reduce<<<grid, 256, 0, s>>>(partial, units_per_group, n_grid, group_sums);
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return e;
    if (!W_mean) return cudaSuccess;
    k_mean<<<(n_grid + 255) / 256, 256, 0, s>>>(group_sums, n_groups, n_grid, (double)n_loops, W_mean);
    return cudaGetLastError();
}

}  // namespace wl
