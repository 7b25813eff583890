// wl_terms_packed_f32.cuh -- the packed-FP32 Terms of k_wilson (wl_wilson_body.cuh): Sech2PackedF32 (the kernel
// configs 3, 4 and 5 of BASELINE.json are timed on) and FluxTubePackedF32 (the paper's validation profile,
// eq. (68)).  CUDA path, sm_100a only.  The per-term arithmetic is arranged for the two resources that bound
// it on B200 (profiles/r01_pipe_rates.md, profiles/r03_wilson_f32_ncu.md, "Tried"):
//
//   * the special-function (XU) pipe, 16 lanes/clk/SM: one warp instruction per 8 clk per sub-partition;
//   * the FMA pipe: one packed FFMA2 per 2 clk per sub-partition, and next to a stream of FMA-pipe work every MUFU
//     also takes 2-3 of that pipe's issue cycles.
//
// So (i) the plain FP32 work is issued as PACKED fma/mul/add.f32x2 (FFMA2: two grid points per
// instruction, one issue slot), every thread owning P grid points as P/2 register pairs; (ii) the
// staged loop values enter FFMA2 as both-halves scalar operands, so a staged point costs one LDS.128 and
// one LDS.64 (shared-memory loads return through the same queue as the special-function results: every
// 4 bytes per lane cost about one XU-pipe clock, profiles/r01_pipe_rates.md); (iii) the special-function
// count per point-eval of the sech^2 profile is 2 + 2Q + 1/P (Q = Gauss-Legendre points of eq. (24); 4.25 at Q = 1, P = 4):
//       sqrt(|x_i|^2), 2^(-u_p), [rsqrt(rho_i^2(t_q)), 2^(-u_q)] x Q, and ONE reciprocal per staged point and THREAD
//   (the product of the denominators (1+E_p) prod_q (1+E_q) of all P grid points is inverted once);
//   log2(1+E_q) is a polynomial in E_q on the FMA pipe (degree 8 on [0,1], lower in the far-block tiers);
//   (iv) blocks of staged points that stay clear of the axis for a whole warp run shorter code (far blocks, below).
//
// Staged record of a point i (floats; C = 2 values per position without phi_cm, 3 with):
//     [ y_x, (y_y), |y|^2 ]  [ y(t_q)_x, (y(t_q)_y), |y(t_q)|^2 ] x Q  [ dy_y/2, (dy_x/2), y_i x y_{i+1} ]
//   laid out as NV4 float4 arrays followed by one float2 array (Q = 1 without phi_cm: exactly one LDS.128 + one LDS.64).
#pragma once

#include "wl_block_bounds.cuh"
#include "wl_wilson_body.cuh"

namespace wl {

typedef unsigned long long u64;    // two packed floats (lo, hi)

__device__ __forceinline__ u64 pk(float lo, float hi) { u64 r; asm("mov.b64 %0, {%1, %2};" : "=l"(r) : "f"(lo), "f"(hi)); return r; }
__device__ __forceinline__ u64 pk1(float x) { return pk(x, x); }
__device__ __forceinline__ void upk(u64 v, float& lo, float& hi) { asm("mov.b64 {%0, %1}, %2;" : "=f"(lo), "=f"(hi) : "l"(v)); }
__device__ __forceinline__ u64 fma2(u64 a, u64 b, u64 c) { u64 r; asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(r) : "l"(a), "l"(b), "l"(c)); return r; }
__device__ __forceinline__ u64 mul2(u64 a, u64 b) { u64 r; asm("mul.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(a), "l"(b)); return r; }
__device__ __forceinline__ u64 add2(u64 a, u64 b) { u64 r; asm("add.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(a), "l"(b)); return r; }

// XU-pipe instructions; abs / neg become free operand modifiers of MUFU.
__device__ __forceinline__ float xu_sqrt_abs(float x) { float y; asm("sqrt.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(fabsf(x))); return y; }
__device__ __forceinline__ float xu_rsqrt(float x) { float y; asm("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x)); return y; }
__device__ __forceinline__ float xu_ex2_neg(float x) { float y; asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(-x)); return y; }
__device__ __forceinline__ float xu_rcp(float x) { float y; asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x)); return y; }
__device__ __forceinline__ u64 xu_rcp2(u64 d) { float d0, d1; upk(d, d0, d1); return pk(xu_rcp(d0), xu_rcp(d1)); }

// ------------------------------------------------------------------------------------------------------------
// What the two packed Terms share: the staged record, the grid-point register pairs, the FP32 -> FP64 hand-over.
// ------------------------------------------------------------------------------------------------------------
template <int P_, int THREADS_, bool HAS_PHI, int Q_, int MINB_>
struct PackedF32Base {
    static_assert(P_ % 2 == 0, "grid points are processed as register pairs");
    static_assert(Q_ >= 1 && Q_ <= 3, "1-, 2- or 3-point Gauss-Legendre rule");
    static constexpr int kP = P_, kThreads = THREADS_, kMinBlocks = MINB_, kChunk = 1024, kSumBlock = 128, kUnroll = 2;
    static constexpr bool kHasPhi = HAS_PHI;
    static constexpr int kQ = Q_;
    static constexpr int NP = P_ / 2;                         // register pairs per thread
    static constexpr int C = HAS_PHI ? 3 : 2;                 // staged floats per position
    static constexpr int NF = C * (2 + Q_);                   // point, Q nodes, cross record
    static constexpr int NV4 = NF / 4, NV2 = (NF % 4 + 1) / 2;
    static constexpr int NFP = 4 * NV4 + 2 * NV2;             // padded record length
    static constexpr int iPT = 0, iNODE = C, iCR = C * (1 + Q_);
    __host__ __device__ static constexpr size_t stage_bytes(int) { return (size_t)(16 * NV4 + 8 * NV2) * kChunk; }

    // pair q holds grid points gp[2q] (lo) and gp[2q+1] (hi)
    struct Grid {
        u64 R2[NP], ax[NP], Tt[NP];
        u64 ay[HAS_PHI ? NP : 1];
    };

    // the staged record of point i -> v[]
    __device__ __forceinline__ static void load_record(const unsigned char* s, int i, float (&v)[NFP])
    {
#pragma unroll
        for (int k = 0; k < NV4; ++k) {
            const float4 f = reinterpret_cast<const float4*>(s)[k * kChunk + i];
            v[4 * k] = f.x; v[4 * k + 1] = f.y; v[4 * k + 2] = f.z; v[4 * k + 3] = f.w;
        }
        if (NV2) {
            const float2 f = reinterpret_cast<const float2*>(s + (size_t)16 * NV4 * kChunk)[i];
            v[4 * NV4] = f.x; v[4 * NV4 + 1] = f.y;
        }
    }
    __device__ __forceinline__ static void store_record(unsigned char* s, int i, const float (&v)[NFP])
    {
#pragma unroll
        for (int k = 0; k < NV4; ++k)
            reinterpret_cast<float4*>(s)[k * kChunk + i] = make_float4(v[4 * k], v[4 * k + 1], v[4 * k + 2], v[4 * k + 3]);
        if (NV2) reinterpret_cast<float2*>(s + (size_t)16 * NV4 * kChunk)[i] = make_float2(v[4 * NV4], v[4 * NV4 + 1]);
    }

    // derive the record of point y and its neighbour z (FP64 -> FP32 once)
    __device__ __forceinline__ static void stage(unsigned char* s, int i, double yx, double yy, double zx, double zy)
    {
        float v[NFP];
#pragma unroll
        for (int k = 0; k < NFP; ++k) v[k] = 0.0f;
        v[iPT] = float(yx);
        if (HAS_PHI) v[iPT + 1] = float(yy);
        v[iPT + C - 1] = float(yx * yx + yy * yy);
#pragma unroll
        for (int q = 0; q < Q_; ++q) {
            double nx, ny, n2;
            segment_node(yx, yy, zx, zy, gl_node(Q_, q), nx, ny, n2);
            v[iNODE + C * q] = float(nx);
            if (HAS_PHI) v[iNODE + C * q + 1] = float(ny);
            v[iNODE + C * q + C - 1] = float(n2);
        }
        v[iCR] = float(0.5 * (zy - yy));
        if (HAS_PHI) v[iCR + 1] = float(0.5 * (zx - yx));
        v[iCR + C - 1] = float(yx * zy - yy * zx);
        store_record(s, i, v);
    }

    // squared radius (scaled) of staged position `at` for pair q: R2 + ax x + [ay y] + Tt r2
    __device__ __forceinline__ static u64 radius2(const Grid& g, int q, const float (&v)[NFP], int at)
    {
        u64 w = fma2(g.ax[q], pk1(v[at]), g.R2[q]);
        if (HAS_PHI) w = fma2(g.ay[q], pk1(v[at + 1]), w);
        return fma2(g.Tt[q], pk1(v[at + C - 1]), w);
    }
    // FP32 partial sums of one block of kSumBlock = 128 terms (reading A8).  The phase sum is kept as C
    // sums  sum_i g_i dy_y/2, [sum_i g_i dy_x/2], sum_i g_i (y_i x y_{i+1})  and the grid-point factors (ax, ay, Tt)
    // of the cross product, eq. (24), are applied once per block in FP64: two two-source FFMA2 per pair instead of
    // FMUL2 + FFMA2 + a three-source FFMA2 (3 clk on the FMA pipe, profiles/r01_pipe_rates.md).
    struct Acc {
        u64 ph[NP][C], sp[NP];
        __device__ __forceinline__ void zero()
        {
#pragma unroll
            for (int q = 0; q < NP; ++q) {
                sp[q] = 0ull;                                                   // (+0.0f, +0.0f)
#pragma unroll
                for (int k = 0; k < C; ++k) ph[q][k] = 0ull;
            }
        }
        __device__ __forceinline__ void add_phase(int q, u64 gt, const float (&v)[NFP])
        {
#pragma unroll
            for (int k = 0; k < C; ++k) ph[q][k] = fma2(gt, pk1(v[iCR + k]), ph[q][k]);
        }
        __device__ __forceinline__ void flush(const Grid& g, double (&dph)[P_], double (&dsp)[P_]) const
        {
#pragma unroll
            for (int q = 0; q < NP; ++q) {
                float s0, s1, a0, a1, t0, t1, y0, y1, c0, c1;
                upk(sp[q], s0, s1);
                dsp[2 * q] += double(s0); dsp[2 * q + 1] += double(s1);
                upk(g.ax[q], a0, a1);
                upk(g.Tt[q], t0, t1);
                upk(ph[q][0], y0, y1);
                upk(ph[q][C - 1], c0, c1);
                double d0 = double(a0) * double(y0) + double(t0) * double(c0);
                double d1 = double(a1) * double(y1) + double(t1) * double(c1);
                if (HAS_PHI) {
                    float b0, b1, x0, x1;
                    upk(g.ay[q], b0, b1);
                    upk(ph[q][HAS_PHI ? 1 : 0], x0, x1);
                    d0 -= double(b0) * double(x0);
                    d1 -= double(b1) * double(x1);
                }
                dph[2 * q] += d0; dph[2 * q + 1] += d1;
            }
        }
    };

    // grid constants scaled by k2 (and R2 offset by `one`): the common part of Grid::load
    __device__ __forceinline__ static void load_grid(Grid& g, double k2, double one, const double (&T)[P_],
                                                     const double (&rho)[P_], const double (&cx)[P_], const double (&cy)[P_])
    {
        float R2[P_], ax[P_], ay[P_], Tt[P_];
#pragma unroll
        for (int j = 0; j < P_; ++j) {
            R2[j] = float(one + k2 * rho[j] * rho[j]);
            ax[j] = float(k2 * 2.0 * sqrt(T[j]) * cx[j]);
            ay[j] = float(k2 * 2.0 * sqrt(T[j]) * cy[j]);
            Tt[j] = float(k2 * T[j]);
        }
#pragma unroll
        for (int q = 0; q < NP; ++q) {
            g.R2[q] = pk(R2[2 * q], R2[2 * q + 1]);
            g.ax[q] = pk(ax[2 * q], ax[2 * q + 1]);
            g.Tt[q] = pk(Tt[2 * q], Tt[2 * q + 1]);
            if (HAS_PHI) g.ay[q] = pk(ay[2 * q], ay[2 * q + 1]);
        }
    }
};

// ------------------------------------------------------------------------------------------------------------
// sech^2 profile.  Scaling: with k = 2 log2(e)/lambda all squared radii are carried as w' = k^2 w, so that
// u' = sqrt(w') = 2 log2(e) rho/lambda and E = exp(-2 rho/lambda) = 2^(-u') need no multiply, and
//   h(u)    = ln2 [ (1 - log2(1+E)) - u' E/(1+E) ] / u^2  = 4 log2(e) * br / w'
//   x_i x x_{i+1} carried times k^2 (through ax, ay, Tt at the end of every block)
// hence phase = eB0 * lambda^2 ln2 * sum_i [sum_q w_q br/w'](i) * [k^2 x_i x x_{i+1}](i): the constants leave the loop.
// Near the axis (w = u^2 < 1/8) the bracket cancels and a degree-3 polynomial in w' replaces br/w'
// (coefficients: gen_h_poly.py hs 0.125 3, relative error 8e-8).
// ------------------------------------------------------------------------------------------------------------
// SCALAR_ = true (scalar QED, W = cos(phase)): the spin sum is not needed, so the point's
// sqrt and 2^x are skipped and the reciprocal is that of the nodes alone: 2 + 1/P MUFU per point-eval at Q = 1.
template <int P_, int THREADS_, bool HAS_PHI, int Q_, int MINB_ = 4, bool SCALAR_ = false>
struct Sech2PackedF32 : PackedF32Base<P_, THREADS_, HAS_PHI, Q_, MINB_> {
    static_assert(!SCALAR_ || Q_ == 1, "the scalar-only variant is compiled for the midpoint rule");
    typedef PackedF32Base<P_, THREADS_, HAS_PHI, Q_, MINB_> B;
    using typename B::Acc;
    using B::NP; using B::NFP; using B::C; using B::iPT; using B::iNODE;
    double eB0, lambda, k2;

    __device__ explicit Sech2PackedF32(const EvalArgs& a) : eB0(a.p0), lambda(a.p1)
    {
        const double k = 2.0 * 1.4426950408889634074 / lambda;
        k2 = k * k;
    }
    struct Grid : B::Grid {
        __device__ __forceinline__ void load(const Sech2PackedF32& t, const double (&T)[P_], const double (&rho)[P_],
                                             const double (&cx)[P_], const double (&cy)[P_])
        {
            B::load_grid(*this, t.k2, 0.0, T, rho, cx, cy);
        }
    };
    // sum_q w_q g_q carries 1/2 (Q = 2) or 5/18 (Q = 3) outside the loop
    __device__ double g_scale() const
    {
        return eB0 * lambda * lambda * 0.69314718055994530942 * (Q_ == 2 ? 0.5 : (Q_ == 3 ? 5.0 / 18.0 : 1.0));
    }
    __device__ double b_scale() const { return 4.0 * eB0; }

    // ---- far blocks (wl_block_bounds.cuh) ------------------------------------------------------------------------
    // The near-axis polynomial, its select and the guard of rsqrt are needed only where a node can come within
    // u^2 < 1/8 of the axis, and the bound that rules this out for a whole warp and block also limits E = 2^(-u') from
    // above: on a shorter range of E the polynomial for 1 - log2(1+E) reaches the same 6e-8 with a lower degree.
    // kTiers instantiations of the walk; tier 0 is the full code.
    static constexpr bool kBlockBounds = true;
    static constexpr int kBoundsBlock = B::kSumBlock;
    typedef BlockBounds<B::kChunk, kBoundsBlock> Bounds;
    __host__ __device__ static constexpr size_t stage_bytes(int q) { return B::stage_bytes(q) + Bounds::kBytes; }
    __device__ __forceinline__ void note_bounds(unsigned char* s, int ib, bool valid, double yx, double yy, double zx, double zy) const
    {
        Bounds::note(s + B::stage_bytes(0), ib, valid, yx, yy, zx, zy);
    }
    static constexpr int kTiers = 6;
    __device__ __forceinline__ static int block_tier(const unsigned char* s, int i0, const Grid& g)
    {
        const float4 b = Bounds::box(s + B::stage_bytes(0), i0);
        const float ext2 = Bounds::extent2(b);
        float wlow = 1e30f;
#pragma unroll
        for (int q = 0; q < NP; ++q) {
            float R2[2], ax[2], Tt[2], ay[2] = {0.0f, 0.0f};
            upk(g.R2[q], R2[0], R2[1]);
            upk(g.ax[q], ax[0], ax[1]);
            upk(g.Tt[q], Tt[0], Tt[1]);
            if (HAS_PHI) upk(g.ay[q], ay[0], ay[1]);
#pragma unroll
            for (int h = 0; h < 2; ++h) wlow = fminf(wlow, Bounds::w_low(b, ext2, R2[h], ax[h], ay[h], Tt[h]));
        }
        const float wwarp = Bounds::warp_min(wlow);
        int tier = 0;
#pragma unroll
        for (int k = 1; k < kTiers; ++k) tier = (wwarp >= tier_w(k)) ? k : tier;
        return tier;
    }
    // tier k > 0 holds when w' >= tier_w(k) for every node: E = 2^(-u') <= 2^(-sqrt(tier_w)), and 1 - log2(1+E) needs
    // only degree tier_deg(k) there for the same 6e-8 (gen_h_poly.py Lw <tier_w> <degree>)
    __host__ __device__ static constexpr float tier_w(int k) { return k == 1 ? 1.05f : k == 2 ? 9.0f : k == 3 ? 16.0f : k == 4 ? 36.0f : 144.0f; }
    __host__ __device__ static constexpr int tier_deg(int k) { return k == 0 ? 8 : k == 1 ? 6 : k == 2 ? 4 : k == 3 ? 3 : k == 4 ? 2 : 1; }
    __host__ __device__ static constexpr float tier_coef(int k, int i)
    {
        constexpr float c0[9] = {0.999999943578f, -1.44268585129f, 0.721095768202f, -0.478176441505f, 0.345429336575f,
                                 -0.238041983614f, 0.13314692741f, -0.0494333683912f, 0.00866569930832f};   // L 8
        constexpr float c1[7] = {0.999999951917f, -1.44268542229f, 0.72102782158f, -0.476826061169f, 0.33512281736f,
                                 -0.20083019495f, 0.0676755895834f};                                            // Lw 1.05 6
        constexpr float c2[5] = {0.999999986538f, -1.44268965027f, 0.720999117524f, -0.472913355165f, 0.283761002847f};  // Lw 9 4
        constexpr float c3[4] = {0.999999960862f, -1.44267499105f, 0.719731652215f, -0.438694041338f};         // Lw 16 3
        constexpr float c4[3] = {0.999999943498f, -1.44262997327f, 0.710212211046f};                           // Lw 36 2
        constexpr float c5[2] = {0.999999994616f, -1.44251877967f};                                            // Lw 144 1
        return k == 0 ? c0[i] : k == 1 ? c1[i] : k == 2 ? c2[i] : k == 3 ? c3[i] : k == 4 ? c4[i] : c5[i];
    }

    // 1/t for a positive, normal t on the FMA pipe: the integer seed 0x7EF311C7 - bits(t) is within 12.6 %, three Newton
    // steps r <- r (2 - t r) bring that to 6e-8 (the accuracy of MUFU.RCP).  Six scalar FMA-pipe instructions and one
    // integer subtraction per thread and staged point instead of a special-function op: the XU pipe is the kernel's bound.
    // (measured: 139.7 -> 135.4 ms on config 3.  Kept on the MUFU where the FMA pipe or latency binds instead: the
    // scalar-only variant with its 2.25 special-function ops per point-eval (83.0 against 87.8 ms), the phi_cm variant with
    // its third component per radius and phase sum (41.9 against 42.7 ms on 4096 loops), and the 128-thread variant of
    // grids of at most 256 points, whose launches are too short to hide the longer dependent chain (config 1: 0.099
    // against 0.104 ms).)
    static constexpr bool kFmaRcp = !SCALAR_ && !HAS_PHI && THREADS_ >= 256;
    __device__ __forceinline__ static float fma_rcp(float t)
    {
        float r = __int_as_float(0x7EF311C7 - __float_as_int(t));
        r = r * fmaf(-t, r, 2.0f);
        r = r * fmaf(-t, r, 2.0f);
        return r * fmaf(-t, r, 2.0f);
    }
    // 1/den[q] for every pair from ONE reciprocal per thread: the product of all 2 NP lanes' denominators is inverted
    // once and each lane's inverse is recovered by multiplying the others back in (every denominator is a product of
    // at most four factors in [1, 2] with a common sign per Term, so the product of all is positive and below 2^16).
    __device__ __forceinline__ static void shared_inverse(const u64 (&den)[NP], u64 (&inv)[NP])
    {
        static_assert(NP <= 2, "written for one or two register pairs");
        if constexpr (NP == 1) {
            float a, b;
            upk(den[0], a, b);
            const float r = kFmaRcp ? fma_rcp(a * b) : xu_rcp(a * b);
            inv[0] = pk(r * b, r * a);
        } else {
            float a, b;
            upk(mul2(den[0], den[1]), a, b);
            const float r = kFmaRcp ? fma_rcp(a * b) : xu_rcp(a * b);
            const u64 iq = pk(r * b, r * a);
            inv[0] = mul2(iq, den[1]);
            inv[1] = mul2(iq, den[0]);
        }
    }

    // g-term of one node from (w' clamped, 1/sqrt(w'), u', E, -1/(1+E)):  br/w' or, in tier 0, the near-axis polynomial
    template <int TIER>
    __device__ __forceinline__ static u64 g_node(u64 wm, u64 rm, u64 um, u64 Em, u64 imn)
    {
        constexpr float kPolyBelow = 1.0406844905f;     // w' < this  <=>  u^2 < 1/8
        // 1 - log2(1+E) = c0 + E L'(E), abs. error 6e-8 on the tier's range of E
        constexpr int D = tier_deg(TIER);
        u64 L = pk1(tier_coef(TIER, D));
#pragma unroll
        for (int k = D - 1; k >= 1; --k) L = fma2(L, Em, pk1(tier_coef(TIER, k)));
        // last Horner step folded with the second term: -u' E/(1+E) = E (u' imn), so br = c0 + E (L' + u' imn)
        const u64 br = fma2(fma2(um, imn, L), Em, pk1(tier_coef(TIER, 0)));    // (1 - log2(1+E)) - u' E/(1+E)
        const u64 hE = mul2(br, mul2(rm, rm));                                  // br / w'
        if constexpr (TIER > 0) return hE;
        // h(w)/(4 log2 e) in w' (gen_h_poly.py hs 0.125 3, rel. error 8e-8)
        u64 hP = fma2(pk1(-1.2801479229129e-5f), wm, pk1(0.00027690498335525f));
        hP = fma2(hP, wm, pk1(-0.0052033291295960f));
        hP = fma2(hP, wm, pk1(0.086643391691228f));
        float wm0, wm1, hE0, hE1, hP0, hP1;
        upk(wm, wm0, wm1);
        upk(hE, hE0, hE1);
        upk(hP, hP0, hP1);
        return pk(wm0 < kPolyBelow ? hP0 : hE0, wm1 < kPolyBelow ? hP1 : hE1);
    }

    template <int TIER = 0>
    __device__ __forceinline__ void point(const unsigned char* s, int i, const Grid& g, Acc& acc) const
    {
        // one LDS.128 + one LDS.64 per staged point at Q = 1 (a broadcast: every lane reads the same address);
        // each scalar feeds FFMA2 as a both-halves operand (SASS: Rn.F32), no duplication in memory
        float v[NFP];
        B::load_record(s, i, v);
        const u64 one2 = pk1(1.0f), mone2 = pk1(-1.0f);
        constexpr float kTiny = 1e-36f;                 // rsqrt(kTiny)^2 is still finite
        u64 Ep[NP], Dp[NP], wm[NP][Q_], rm[NP][Q_], um[NP][Q_], Em[NP][Q_], Dmn[NP][Q_], den[NP], inv[NP], PD[NP], D01[NP];
#pragma unroll
        for (int q = 0; q < NP; ++q) {
            // |x_i|^2 and rho_i^2(t_q) (times k^2): eq. (8), (25)-(28)
            Ep[q] = 0ull;
            if constexpr (!SCALAR_) {
                float wp0, wp1;
                upk(B::radius2(g, q, v, iPT), wp0, wp1);
                Ep[q] = pk(xu_ex2_neg(xu_sqrt_abs(wp0)), xu_ex2_neg(xu_sqrt_abs(wp1)));
            }
#pragma unroll
            for (int n = 0; n < Q_; ++n) {
                float w0, w1, u0, u1;
                upk(B::radius2(g, q, v, iNODE + C * n), w0, w1);
                if constexpr (TIER == 0) {
                    w0 = fmaxf(w0, kTiny);
                    w1 = fmaxf(w1, kTiny);
                }
                wm[q][n] = pk(w0, w1);
                rm[q][n] = pk(xu_rsqrt(w0), xu_rsqrt(w1));
                um[q][n] = mul2(wm[q][n], rm[q][n]);                          // u' = sqrt(w')
                upk(um[q][n], u0, u1);
                Em[q][n] = pk(xu_ex2_neg(u0), xu_ex2_neg(u1));
                Dmn[q][n] = fma2(Em[q][n], mone2, mone2);                     // -(1 + E_q)
            }
            Dp[q] = fma2(Ep[q], one2, one2);                                  //   1 + E_p
            // the denominator the point and all nodes share
            if constexpr (SCALAR_) den[q] = Dmn[q][0];
            else if constexpr (Q_ == 1) den[q] = mul2(Dp[q], Dmn[q][0]);
            else if constexpr (Q_ == 2) { PD[q] = mul2(Dmn[q][0], Dmn[q][1]); den[q] = mul2(Dp[q], PD[q]); }
            else { D01[q] = mul2(Dmn[q][0], Dmn[q][1]); PD[q] = mul2(D01[q], Dmn[q][2]); den[q] = mul2(Dp[q], PD[q]); }
        }
        shared_inverse(den, inv);                                             // ONE reciprocal per staged point and thread
#pragma unroll
        for (int q = 0; q < NP; ++q) {
            // imn[n] = -1/(1 + E_n), ip = 1/(1 + E_p)
            const u64 r = inv[q];
            u64 ip = 0ull, imn[Q_];
            if constexpr (SCALAR_) {
                imn[0] = r;                                                   // -1/(1+E_m)
            } else if constexpr (Q_ == 1) {
                ip = mul2(r, Dmn[q][0]);                                      // r = -1/((1+E_p)(1+E_m))
                imn[0] = mul2(r, Dp[q]);
            } else if constexpr (Q_ == 2) {
                ip = mul2(r, PD[q]);                                          // r, PD (+)
                const u64 rDp = mul2(r, Dp[q]);
                imn[0] = mul2(rDp, Dmn[q][1]);
                imn[1] = mul2(rDp, Dmn[q][0]);
            } else {
                ip = mul2(r, PD[q]);                                          // r, PD (-); D01 (+)
                const u64 rDp = mul2(r, Dp[q]);                               // (-)
                imn[2] = mul2(rDp, D01[q]);                                   // (-)
                const u64 t = mul2(rDp, Dmn[q][2]);                           // (+)
                imn[0] = mul2(t, Dmn[q][1]);
                imn[1] = mul2(t, Dmn[q][0]);
            }
            if constexpr (!SCALAR_) acc.sp[q] = fma2(mul2(Ep[q], ip), ip, acc.sp[q]);   // E_p/(1+E_p)^2 = sech^2/4
            u64 gt = g_node<TIER>(wm[q][0], rm[q][0], um[q][0], Em[q][0], imn[0]);
            if constexpr (Q_ == 2) gt = add2(gt, g_node<TIER>(wm[q][1], rm[q][1], um[q][1], Em[q][1], imn[1]));
            if constexpr (Q_ == 3) {                                          // 5/18 [ g_0 + g_2 + (8/5) g_1 ]
                gt = add2(gt, g_node<TIER>(wm[q][2], rm[q][2], um[q][2], Em[q][2], imn[2]));
                gt = fma2(g_node<TIER>(wm[q][1], rm[q][1], um[q][1], Em[q][1], imn[1]), pk1(1.6f), gt);
            }
            acc.add_phase(q, gt, v);
        }
    }

    template <int TIER>
    __device__ __forceinline__ void walk(const unsigned char* s, int i0, int ie, const Grid& g, Acc& acc) const
    {
#pragma unroll B::kUnroll
        for (int i = i0; i < ie; ++i) point<TIER>(s, i, g, acc);
    }
    // one block of at most kSumBlock staged points, [i0, ie)
    __device__ __forceinline__ void block(const unsigned char* s, int i0, int ie, const Grid& g, Acc& acc) const
    {
        const int tier = block_tier(s, i0, g);
        switch (tier) {
            case 0: walk<0>(s, i0, ie, g, acc); break;
            case 1: walk<1>(s, i0, ie, g, acc); break;
            case 2: walk<2>(s, i0, ie, g, acc); break;
            case 3: walk<3>(s, i0, ie, g, acc); break;
            case 4: walk<4>(s, i0, ie, g, acc); break;
            default: walk<5>(s, i0, ie, g, acc); break;
        }
    }
};

// ------------------------------------------------------------------------------------------------------------
// flux tube, eq. (68): f_lambda = rho^2/(lambda^2+rho^2),
//     g = script-F/(lambda^2 + rho^2),   b = 2 script-F lambda^2/(lambda^2 + |x|^2)^2      (eq. (14), (15), (17))
// With all squared radii carried as a = 1 + w/lambda^2 (the "+1" sits in the grid-point constant):
//     g = (script-F/lambda^2)/a_q,   b = (2 script-F/lambda^2)/a_p^2,   x_i x x_{i+1} carried divided by lambda^2
// so a point-eval is a handful of packed FMA-pipe instructions and ONE special-function op (the reciprocal of
// a_p prod_q a_q, shared by the point and the nodes): FMA-pipe bound, not XU bound.  No square root:
// the profile is a function of rho^2, as PAPER.md:149 advises.
// ------------------------------------------------------------------------------------------------------------
template <int P_, int THREADS_, bool HAS_PHI, int Q_, int MINB_ = 4>
struct FluxTubePackedF32 : PackedF32Base<P_, THREADS_, HAS_PHI, Q_, MINB_> {
    typedef PackedF32Base<P_, THREADS_, HAS_PHI, Q_, MINB_> B;
    using typename B::Acc;
    using B::NP; using B::NFP; using B::C; using B::iPT; using B::iNODE;
    double F, lambda, k2;              // script-F = eF/2pi (eq. (17)), lambda, 1/lambda^2

    __device__ explicit FluxTubePackedF32(const EvalArgs& a) : F(a.p0), lambda(a.p1), k2(1.0 / (a.p1 * a.p1)) {}
    struct Grid : B::Grid {
        __device__ __forceinline__ void load(const FluxTubePackedF32& t, const double (&T)[P_], const double (&rho)[P_],
                                             const double (&cx)[P_], const double (&cy)[P_])
        {
            B::load_grid(*this, t.k2, 1.0, T, rho, cx, cy);              // a = 1 + w/lambda^2
        }
    };
    __device__ double g_scale() const { return F * (Q_ == 2 ? 0.5 : (Q_ == 3 ? 5.0 / 18.0 : 1.0)); }   // (F/lambda^2) x lambda^2 from the scaled cross term
    __device__ double b_scale() const { return 2.0 * F * k2; }

    __device__ __forceinline__ void point(const unsigned char* s, int i, const Grid& g, Acc& acc) const
    {
        float v[NFP];
        B::load_record(s, i, v);
#pragma unroll
        for (int q = 0; q < NP; ++q) {
            // a_p = 1 + |x_i|^2/lambda^2, a_q = 1 + rho_i^2(t_q)/lambda^2: eq. (8), (25)-(28)
            const u64 ap = B::radius2(g, q, v, iPT);
            u64 am[Q_];
#pragma unroll
            for (int n = 0; n < Q_; ++n) am[n] = B::radius2(g, q, v, iNODE + C * n);
            u64 ip, gt;
            if constexpr (Q_ == 1) {
                const u64 r = xu_rcp2(mul2(ap, am[0]));                       // 1/(a_p a_m): one reciprocal for both
                ip = mul2(r, am[0]);                                          // 1/a_p
                gt = mul2(r, ap);                                             // 1/a_m          -> g
            } else if constexpr (Q_ == 2) {
                const u64 PD = mul2(am[0], am[1]);
                const u64 r = xu_rcp2(mul2(ap, PD));
                ip = mul2(r, PD);
                gt = mul2(mul2(r, ap), add2(am[0], am[1]));                   // 1/a_0 + 1/a_1 = (a_0 + a_1)/(a_0 a_1)
            } else {
                const u64 D01 = mul2(am[0], am[1]);
                const u64 PD = mul2(D01, am[2]);
                const u64 r = xu_rcp2(mul2(ap, PD));
                ip = mul2(r, PD);
                const u64 rDp = mul2(r, ap);                                  // 1/(a_0 a_1 a_2)
                // 1/a_0 + 1/a_2 + (8/5)/a_1 = [ a_1 (a_0 + a_2) + (8/5) a_0 a_2 ] / (a_0 a_1 a_2)
                gt = mul2(rDp, fma2(mul2(am[0], am[2]), pk1(1.6f), mul2(am[1], add2(am[0], am[2]))));
            }
            acc.sp[q] = fma2(ip, ip, acc.sp[q]);                              // 1/a_p^2        -> b
            acc.add_phase(q, gt, v);
        }
    }
};

}  // namespace wl
