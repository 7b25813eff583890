// wl_wilson_body.cuh -- the ONE scaffold of every Wilson-loop kernel (k_wilson<Term, DISC, BULK>).  CUDA path, sm_100a.
//
// Mapping.  One CTA = (one unit of `loops_per_unit` consecutive loops) x (one tile of
// kThreads*P grid points).  LANES RUN OVER GRID POINTS, each thread owns P grid points in registers; the loop
// is staged chunk by chunk in shared memory as derived per-point / per-segment quantities of the UNIT loop,
// and every thread walks the staged points serially: all lanes of a warp read the same shared-memory address
// (a broadcast), and every sum round the loop is taken by one thread in index order.  No shuffles, no
// atomics: the result does not depend on how CTAs are scheduled.
//
// What the scaffold owns: the unit / tile decomposition, where the raw loop coordinates come from (HBM, a
// cp.async.bulk pipeline, or regenerated in shared memory from the Philox seed), the chunk loop with its
// two barriers, the two virtual passes of the discretisation estimate, the FP64 epilogue
// W = cos(phase) cosh(spin) and the partial-sum layout.  What a Term owns (wl_terms_*.cuh): the per-thread
// grid-point constants, which derived quantities are staged, and the arithmetic of one staged point.
//
// Term concept:
//   static constexpr int kP, kThreads, kMinBlocks, kChunk, kSumBlock (0: accumulate straight into FP64), kUnroll
//   static size_t stage_bytes(int quad)                       bytes of staged data per chunk (multiple of 16)
//   Term(const EvalArgs&)                                     field constants
//   struct Grid { void load(term, T[P], rho[P], cx[P], cy[P]) }   per-thread grid-point constants
//   struct Acc  { void zero(); void flush(grid, dph[P], dsp[P]) } running sums of one block of terms
//   void stage(smem, i, yx, yy, zx, zy)                       derive and store point i (y) and its neighbour (z)
//   void point(smem, i, grid, acc)                            add staged point i to the sums of all P grid points
//   double g_scale(), b_scale()                               constant factors of phase and spin
// Optional (a Term that declares kBlockBounds = true; blocks of kSumBlock staged points, or of kBoundsBlock if kSumBlock = 0):
//   void note_bounds(smem, ib, valid, yx, yy, zx, zy)         called by EVERY thread next to stage(): the Term keeps a
//                                                             bounding box of every block of kSumBlock staged segments
//   void block(smem, i0, ie, grid, acc)                       walks the block [i0, ie) itself instead of point() calls
//                                                             (it may pick a cheaper code path for the whole warp)
//
// Algebra (eq. (8), (21)-(28)), with c = x_cm, s = sqrt(T), unit-loop point y_i,
// node y_i(t) = y_i + t (y_{i+1} - y_i) (t = 1/2: the midpoint), step dy_i = y_{i+1} - y_i:
//     |x_i|^2      = |c|^2 + 2 s (c . y_i)    + T |y_i|^2
//     rho_i^2(t)   = |c|^2 + 2 s (c . y_i(t)) + T |y_i(t)|^2          (= A_i + 2 B_i t + C_i t^2, eq. (25))
//     x_i x x_{i+1} = s (c x dy_i) + T (y_i x y_{i+1})                 (the prefactor of eq. (24))
// so per term the grid point contributes (|c|^2, 2 s c, T) and the loop contributes per-point values computed
// once per staged point in FP64.  With phi_cm = 0 (c on the x axis) the y components drop out.
#pragma once

#include "wl_dloop_device.cuh"
#include "wl_internal.cuh"

namespace wl {

// Gauss-Legendre nodes on [0, 1] for the t-integral of eq. (24): Q = 1 midpoint,
// Q = 2: 1/2 -+ 1/(2 sqrt 3), Q = 3: 1/2 -+ sqrt(3/5)/2 and 1/2.  Weights are applied by the Terms.
__device__ __forceinline__ double gl_node(int Q, int q)
{
    if (Q == 2) return q == 0 ? 0.5 - 0.28867513459481288225 : 0.5 + 0.28867513459481288225;
    if (Q == 3) return q == 0 ? 0.5 - 0.38729833462074168852 : (q == 1 ? 0.5 : 0.5 + 0.38729833462074168852);
    return 0.5;
}
__device__ __forceinline__ double gl_weight(int Q, int q)
{
    if (Q == 2) return 0.5;
    if (Q == 3) return q == 1 ? 4.0 / 9.0 : 5.0 / 18.0;
    return 1.0;
}

// y_i(t) and |y_i(t)|^2 of a segment, FP64.  t = 1/2 gives exactly (y + z)/2.
__device__ __forceinline__ void segment_node(double yx, double yy, double zx, double zy, double t,
                                             double& nx, double& ny, double& n2)
{
    if (t == 0.5) { nx = 0.5 * (yx + zx); ny = 0.5 * (yy + zy); }
    else { nx = fma(t, zx - yx, yx); ny = fma(t, zy - yy, yy); }
    n2 = nx * nx + ny * ny;
}

// ---- cp.async.bulk + mbarrier (the staging variant north_star names; measured in profiles/r03_wilson_f32_ncu.md, "Tried") ----
__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(uint64_t* bar, int count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count));
}
__device__ __forceinline__ void mbar_expect_tx(uint64_t* bar, uint32_t bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t* bar, uint32_t parity)
{
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "WAIT_%=:\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
        "@p bra DONE_%=;\n"
        "bra WAIT_%=;\n"
        "DONE_%=:\n"
        "}\n" ::"r"(smem_u32(bar)), "r"(parity) : "memory");
}
__device__ __forceinline__ void bulk_g2s(void* dst, const void* src, uint32_t bytes, uint64_t* bar)
{
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                 ::"r"(smem_u32(dst)), "l"(src), "r"(bytes), "r"(smem_u32(bar)) : "memory");
}

template <class T, class = void> struct term_block_bounds { static constexpr bool value = false; };
template <class T> struct term_block_bounds<T, decltype((void)T::kBlockBounds)> { static constexpr bool value = T::kBlockBounds; };

// Shared memory a launch needs beyond the staged chunk.
template <class Term>
__host__ __device__ inline size_t wilson_extra_smem(int n_ppl, bool seeded, bool bulk, bool loops_are_f64)
{
    // every seeded loop the ABI accepts must fit the skeleton array: a shorter chunk than this would overrun it silently
    static_assert(kMaxPplSeeded / Term::kChunk <= kSkeletonMax, "DLoopScratch::skel is too small for this Term's chunk length");
    size_t b = 0;
    if (seeded) {
        const DLoopShape sh = dloop_shape(n_ppl, Term::kChunk);
        b += sizeof(double2) * (size_t)(sh.Cg + 1) + sizeof(DLoopScratch);
    }
    if (bulk) b += 2 * (size_t)(Term::kChunk + 2) * (loops_are_f64 ? 16 : 8) + 2 * sizeof(uint64_t);
    return b;
}

// SEEDED is a template parameter (like DISC and BULK) so that the stored-loop kernels -- the ones the benchmarks
// time -- do not carry the FP64 Philox / Box-Muller generator in their code and register allocation.
template <class Term, bool DISC, bool BULK, bool SEEDED>
__device__ __forceinline__ void wilson_body(const EvalArgs& a, const int n_grid, const int n_tiles,
                                            const int loops_per_unit, const int64_t n_units)
{
    constexpr int P = Term::kP, THREADS = Term::kThreads, CHUNK = Term::kChunk, SB = Term::kSumBlock;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    unsigned char* const sStaged = smem_raw;
    unsigned char* const sExtra = smem_raw + Term::stage_bytes(a.quad);

    const int tid = threadIdx.x;
    const int tile = blockIdx.x % n_tiles;
    const int64_t unit = blockIdx.x / n_tiles;
    const int N = a.n_ppl;
    const Term term(a);

    // ---- per-thread grid-point constants (FP64 on the way in, then the Term's compute type) ----
    // Which grid points a thread owns.  The grid is walked in strips of kRhoStrip = 8 neighbouring rho_cm: within a strip
    // rho runs fastest, then the proper time, so that 128 consecutive positions v are a compact patch of 16 proper
    // times x 8 rho_cm (the last strip may be narrower).  With v = ((tile * warps + warp) * P + j) * 32 + lane a warp
    // owns one such patch and the P points of a thread share rho_cm: the whole warp sees the flux tube's axis from
    // about one distance at about one loop size, which is what lets a Term choose one code path for all of its lanes
    // (wl_terms_packed_f32.cuh, "far blocks").  gp[j] = t * n_rho + r is the point's index in every output array.
    typename Term::Grid grid;
    int gp[P], vp[P];                                     // output index and walk position
    unsigned gp_ok = 0;
    {
        double Tj[P], rj[P], cxj[P], cyj[P];
#pragma unroll
        for (int j = 0; j < P; ++j) {
            const int v = ((tile * (THREADS / 32) + (tid >> 5)) * P + j) * 32 + (tid & 31);
            if (v < n_grid) gp_ok |= 1u << j;
            const int vc = min(v, n_grid - 1);
            int it, ir;
            walk_position(vc, a.n_T, a.n_rho, &it, &ir);
            vp[j] = vc;
            gp[j] = it * a.n_rho + ir;
            Tj[j] = a.T[it];
            rj[j] = a.rho[ir];
            cxj[j] = rj[j];
            cyj[j] = 0.0;
            if (Term::kHasPhi) { const double ph = a.phi[ir]; cxj[j] = rj[j] * cos(ph); cyj[j] = rj[j] * sin(ph); }
        }
        grid.load(term, Tj, rj, cxj, cyj);
    }

    constexpr int kLevels = DISC ? 3 : 1;
    double Wsum[kLevels][P];
#pragma unroll
    for (int v = 0; v < kLevels; ++v)
#pragma unroll
        for (int j = 0; j < P; ++j) Wsum[v][j] = 0.0;

    // ---- seeded mode: the loop is regenerated chunk by chunk in shared memory (wl_dloop_device.cuh) ----
    static_assert(!SEEDED || (!DISC && !BULK), "seeded evaluation: ordinary pass, ordinary staging only");
    constexpr bool seeded = SEEDED;
    DLoopShape shp = dloop_shape(N, CHUNK);
    double2* const yraw = reinterpret_cast<double2*>(sExtra);
    DLoopScratch* const sc = reinterpret_cast<DLoopScratch*>(sExtra + sizeof(double2) * (size_t)(shp.Cg + 1));

    // ---- bulk-copy mode: raw chunks land in a two-slot ring, one chunk ahead of the evaluation ----
    const int raw_elem = a.loops_are_f64 ? 16 : 8;
    unsigned char* const sRing = sExtra;
    uint64_t* const sBar = reinterpret_cast<uint64_t*>(sExtra + 2 * (size_t)(CHUNK + 2) * raw_elem);
    const int chunks_per_loop = (N + CHUNK - 1) / CHUNK;
    int ring_idx = 0;                                   // chunks consumed so far by this CTA
    auto bulk_issue = [&](int idx) {                    // thread 0: start the copy of the idx-th chunk of this unit
        const int ll = idx / chunks_per_loop, c0 = (idx % chunks_per_loop) * CHUNK;
        const int cn = min(CHUNK, N - c0);
        const unsigned char* src = reinterpret_cast<const unsigned char*>(a.loops)
                                   + ((unit * loops_per_unit + ll) * (int64_t)N + c0) * raw_elem;
        unsigned char* dst = sRing + (size_t)(idx & 1) * (CHUNK + 2) * raw_elem;
        uint64_t* bar = sBar + (idx & 1);
        const bool last = (c0 + cn == N);
        // whole 16-byte units; the point after the chunk comes along (or, for the last chunk, y_0 by a second copy)
        const uint32_t main_bytes = last ? (uint32_t)(cn * raw_elem) : (uint32_t)(((cn + 1) * raw_elem + 15) & ~15);
        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
        mbar_expect_tx(bar, main_bytes + (last ? 16u : 0u));
        bulk_g2s(dst, src, main_bytes, bar);
        if (last) bulk_g2s(dst + (size_t)cn * raw_elem, src - (size_t)c0 * raw_elem, 16u, bar);
    };
    if (BULK) {
        if (tid == 0) { mbar_init(sBar, 1); mbar_init(sBar + 1, 1); }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
        __syncthreads();
        if (tid == 0) bulk_issue(0);
    }

    for (int ll = 0; ll < loops_per_unit; ++ll) {
        const int64_t loop = unit * loops_per_unit + ll;
        const double2* L64 = reinterpret_cast<const double2*>(a.loops) + loop * N;
        const float2* L32 = reinterpret_cast<const float2*>(a.loops) + loop * N;
        if constexpr (seeded) {
            __syncthreads();                                  // the previous loop's last chunk has been consumed
            dloop_begin(a.seed, (uint64_t)(a.loop_begin + loop), shp, sc, yraw);
        }
        double dph[P], dsp[P];
#pragma unroll
        for (int j = 0; j < P; ++j) { dph[j] = 0.0; dsp[j] = 0.0; }
        // DISC = true: the discretisation estimate of Sec. IV.A (eq. (48)-(50)).  Each loop is
        // walked as two VIRTUAL loops of N/2 terms: pass 0 = the even points with neighbour +2 (the "circle"
        // sub-worldline, N/2 points), pass 1 = the odd points with neighbour +4 (the "box" and "triangle"
        // sub-worldlines, N/4 points each, summed together).  With S2, S4 the phase sums and B2, B4 the spin
        // sums of the two passes, the three levels are
        //   N/4: phase = S4/2,          spin = 2 (T/N) B4      (mean of the two N/4 sub-worldlines)
        //   N/2: phase = S2,            spin = 2 (T/N) B2
        //   N  : phase = S2/2 + S4/4,   spin = (T/N)(B2 + B4)
        // and the partial sums are written level-major: partial[level][unit][grid].
        double S2[DISC ? P : 1], B2[DISC ? P : 1];            // pass-0 sums (DISC only)

        const int Nv = DISC ? N / 2 : N;                      // terms per pass
        for (int pass = 0; pass < (DISC ? 2 : 1); ++pass) {
            if (DISC && pass == 1) {
#pragma unroll
                for (int j = 0; j < P; ++j) { S2[j] = dph[j]; B2[j] = dsp[j]; dph[j] = 0.0; dsp[j] = 0.0; }
            }
            typename Term::Acc acc;
            if (SB == 0) acc.zero();
            for (int c0 = 0; c0 < Nv; c0 += CHUNK) {
                const int cn = min(CHUNK, Nv - c0);
                __syncthreads();                              // the previous chunk has been consumed
                if constexpr (seeded) dloop_chunk(a.seed, (uint64_t)(a.loop_begin + loop), shp, c0 / CHUNK, sc->skel, yraw);
                const unsigned char* ring = sRing + (size_t)(ring_idx & 1) * (CHUNK + 2) * raw_elem;
                if (BULK) mbar_wait(sBar + (ring_idx & 1), (uint32_t)((ring_idx >> 1) & 1));
                for (int ib = 0; ib < cn; ib += THREADS) {    // stage: derived unit-loop quantities, FP64
                    const int i = ib + tid;
                    const bool valid = i < cn;
                    double yx = 0.0, yy = 0.0, zx = 0.0, zy = 0.0;
                    if (valid) {
                        if (BULK) {
                            if (a.loops_are_f64) {
                                const double2 u = reinterpret_cast<const double2*>(ring)[i], v = reinterpret_cast<const double2*>(ring)[i + 1];
                                yx = u.x; yy = u.y; zx = v.x; zy = v.y;
                            } else {
                                const float2 u = reinterpret_cast<const float2*>(ring)[i], v = reinterpret_cast<const float2*>(ring)[i + 1];
                                yx = u.x; yy = u.y; zx = v.x; zy = v.y;
                            }
                        } else if constexpr (seeded) {
                            // what wl_loops_generate stores: y - centre of mass, rounded once to the storage type
                            const double2 u = yraw[i], v = yraw[i + 1], m = sc->mean;
                            yx = u.x - m.x; yy = u.y - m.y; zx = v.x - m.x; zy = v.y - m.y;
                            if (!a.loops_are_f64) { yx = (double)(float)yx; yy = (double)(float)yy; zx = (double)(float)zx; zy = (double)(float)zy; }
                        } else {
                            int n = c0 + i;
                            int n1 = (n + 1 == N) ? 0 : n + 1;    // closed loop, i+1 mod N
                            if (DISC) {                           // sub-worldline: every 2nd / 4th point, closed on itself
                                n = pass + 2 * (c0 + i);
                                n1 = n + (pass ? 4 : 2);
                                if (n1 >= N) n1 -= N;
                            }
                            if (a.loops_are_f64) {
                                const double2 u = L64[n], v = L64[n1];
                                yx = u.x; yy = u.y; zx = v.x; zy = v.y;
                            } else {
                                const float2 u = L32[n], v = L32[n1];
                                yx = u.x; yy = u.y; zx = v.x; zy = v.y;
                            }
                        }
                        term.stage(sStaged, i, yx, yy, zx, zy);
                    }
                    if constexpr (term_block_bounds<Term>::value) term.note_bounds(sStaged, ib, valid, yx, yy, zx, zy);
                }
                __syncthreads();
                if (BULK) {                                   // slot (ring_idx + 1) & 1 was last read one chunk ago
                    ++ring_idx;
                    if (tid == 0 && ring_idx < loops_per_unit * chunks_per_loop) bulk_issue(ring_idx);
                }

                if (SB > 0) {
                    for (int i0 = 0; i0 < cn; i0 += (SB > 0 ? SB : 1)) {
                        acc.zero();
                        const int ie = min(i0 + SB, cn);
                        if constexpr (term_block_bounds<Term>::value) {
                            term.block(sStaged, i0, ie, grid, acc);
                        } else {
#pragma unroll Term::kUnroll
                            for (int i = i0; i < ie; ++i) term.point(sStaged, i, grid, acc);
                        }
                        acc.flush(grid, dph, dsp);
                    }
                } else if constexpr (term_block_bounds<Term>::value) {
                    for (int i0 = 0; i0 < cn; i0 += Term::kBoundsBlock) term.block(sStaged, i0, min(i0 + Term::kBoundsBlock, cn), grid, acc);
                } else {
#pragma unroll Term::kUnroll
                    for (int i = 0; i < cn; ++i) term.point(sStaged, i, grid, acc);
                }
            }
            if (SB == 0) acc.flush(grid, dph, dsp);
        }   // pass

        // ---- W = cos(phase) cosh(spin), FP64, once per (loop, grid point): eq. (18), PAPER.md:121 ----
        const double g_scale = term.g_scale(), b_scale = term.b_scale();
#pragma unroll
        for (int j = 0; j < P; ++j) {
            const double T = a.T[gp[j] / a.n_rho];
            if (!DISC) {
                const double phase = g_scale * dph[j];
                const double spin = b_scale * (T / double(N)) * dsp[j];
                const double W = a.scalar ? cos(phase) : cos(phase) * cosh(spin);
                Wsum[0][j] += W;
                if (gp_ok >> j & 1) {
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
            if (gp_ok >> j & 1) a.partial[((int64_t)v * n_units + unit) * n_grid + (a.partial_in_walk_order ? vp[j] : gp[j])] = Wsum[v][j];
}

template <class Term, bool DISC, bool BULK, bool SEEDED = false>
__global__ void __launch_bounds__(Term::kThreads, Term::kMinBlocks)
k_wilson(const EvalArgs a, const int n_grid, const int n_tiles, const int loops_per_unit, const int64_t n_units)
{
    wilson_body<Term, DISC, BULK, SEEDED>(a, n_grid, n_tiles, loops_per_unit, n_units);
}

// One launch of k_wilson<Term, DISC, BULK, SEEDED> over plan.n_units x n_tiles CTAs.
template <class Term, bool DISC, bool BULK, bool SEEDED>
cudaError_t launch_term_seeded(const EvalPlan& plan, const EvalArgs& a, cudaStream_t s)
{
    const int n_tiles = (plan.n_grid + Term::kThreads * Term::kP - 1) / (Term::kThreads * Term::kP);
    const size_t smem = Term::stage_bytes(a.quad) + wilson_extra_smem<Term>(a.n_ppl, SEEDED, BULK, a.loops_are_f64 != 0);
    const int64_t n_ctas = plan.n_units * n_tiles;
    if (n_ctas > 0x7fffffffLL) return cudaErrorInvalidConfiguration;
    if (smem > 48 * 1024) {
        cudaError_t e = cudaFuncSetAttribute(k_wilson<Term, DISC, BULK, SEEDED>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (e != cudaSuccess) return e;
    }
    k_wilson<Term, DISC, BULK, SEEDED><<<(unsigned)n_ctas, Term::kThreads, smem, s>>>(a, plan.n_grid, n_tiles,
                                                                                    plan.loops_per_unit, plan.n_units);
    return cudaGetLastError();
}

// The seeded instantiation exists for the ordinary pass with ordinary staging only (as before, a.seeded is ignored
// by the discretisation and bulk-staging kernels).
template <class Term, bool DISC, bool BULK>
cudaError_t launch_term(const EvalPlan& plan, const EvalArgs& a, cudaStream_t s)
{
    if constexpr (!DISC && !BULK) {
        if (a.seeded) return launch_term_seeded<Term, false, false, true>(plan, a, s);
    }
    return launch_term_seeded<Term, DISC, BULK, false>(plan, a, s);
}

// BULK staging needs whole 16-byte units: FP32 loops with an even number of points (FP64 points are 16 bytes).
inline bool bulk_ok(const EvalArgs& a) { return a.bulk && !a.seeded && !a.disc && a.n_ppl >= 2 && (a.loops_are_f64 || a.n_ppl % 2 == 0); }

}  // namespace wl
