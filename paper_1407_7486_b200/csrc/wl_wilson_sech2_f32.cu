// wl_wilson_sech2_f32.cu -- instantiations of k_wilson<Sech2PackedF32<...>> (wl_terms_packed_f32.cuh on the
// scaffold of wl_wilson_body.cuh): the FP32 hot loop for the sech^2 profile, i.e. the kernel configs 3, 4
// and 5 of BASELINE.json are timed on.  CUDA path, sm_100a only.
#include "wl_terms_packed_f32.cuh"

namespace wl {

namespace {

// Which (quadrature order, phi_cm, discretisation estimate, staging) combinations are compiled:
//   Q = 1: with and without phi_cm, with and without the discretisation estimate
//   Q = 2, 3: without phi_cm, ordinary evaluation only
//   the cp.async.bulk staging variant: Q = 1, no phi_cm, ordinary evaluation, P = 4
//   the scalar-only variant (no spin sum): Q = 1, no phi_cm, ordinary evaluation
template <int P, int TH>
cudaError_t launch_shape(const EvalPlan& plan, const EvalArgs& a, cudaStream_t s)
{
    const bool phi = a.phi != nullptr;
    if (a.disc) {
        if (a.quad != 1) return cudaErrorInvalidValue;
        return phi ? launch_term<Sech2PackedF32<P, TH, true, 1>, true, false>(plan, a, s)
                   : launch_term<Sech2PackedF32<P, TH, false, 1>, true, false>(plan, a, s);
    }
    if (a.quad == 1) {
        if (phi) return launch_term<Sech2PackedF32<P, TH, true, 1>, false, false>(plan, a, s);
        if (P == 4 && bulk_ok(a)) return launch_term<Sech2PackedF32<4, 256, false, 1>, false, true>(plan, a, s);
        // scalar loops (W = cos(phase)) in the reducing path: the spin sum is not computed (2 + 1/P MUFU per point-eval);
        // the per-loop triage path keeps the full kernel so that its spin output stays meaningful
        if (a.scalar && !a.phase_out && !a.spin_out) return launch_term<Sech2PackedF32<P, TH, false, 1, 4, true>, false, false>(plan, a, s);
        return launch_term<Sech2PackedF32<P, TH, false, 1>, false, false>(plan, a, s);
    }
    if (phi) return cudaErrorInvalidValue;
    if (P == 4) return cudaErrorInvalidValue;            // Q > 1 runs two grid points per thread (launch_wilson_sech2_f32)
    if (a.quad == 2) return launch_term<Sech2PackedF32<(P == 4 ? 2 : P), TH, false, 2>, false, false>(plan, a, s);
    if (a.quad == 3) return launch_term<Sech2PackedF32<(P == 4 ? 2 : P), TH, false, 3>, false, false>(plan, a, s);
    return cudaErrorInvalidValue;
}

}  // namespace

// plan.P grid points per thread (2 or 4); grids of at most 256 points run 128 threads x 2 grid points, so that
// no thread of the tile idles.  256 threads x P = 4 at 4 CTAs/SM (64 registers), inner loop unrolled by 2, is
// the fastest of the combinations measured (profiles/r03_wilson_f32_ncu.md, "Tried").
cudaError_t launch_wilson_sech2_f32(const EvalPlan& plan, const EvalArgs& a, cudaStream_t s)
{
    if (plan.n_grid <= 256) return launch_shape<2, 128>(plan, a, s);
    // Q > 1 carries Q times the node state: two grid points per thread (no spills; Q = 2: 253.6 against 261.8 ms on
    // config 3 with four; Q = 3 is FMA-pipe bound either way)
    if (plan.P == 2 || a.quad > 1) return launch_shape<2, 256>(plan, a, s);
    if (plan.P == 4) return launch_shape<4, 256>(plan, a, s);
    return cudaErrorInvalidValue;
}

}  // namespace wl
