// wl_wilson_sech2_f64.cu -- instantiations of k_wilson<Sech2LeanF64<...>> (wl_terms_sech2_f64.cuh on the
// scaffold of wl_wilson_body.cuh): the FP64 hot loop for the sech^2 profile, configs 1 and 4 (FP64 variant)
// of BASELINE.json.  CUDA path, sm_100a.
#include "wl_terms_sech2_f64.cuh"

namespace wl {

namespace {

template <int P>
cudaError_t launch_shape(const EvalPlan& plan, const EvalArgs& a, cudaStream_t s)
{
    const bool phi = a.phi != nullptr;
    if (a.disc) {
        if (a.quad != 1) return cudaErrorInvalidValue;
        return phi ? launch_term<Sech2LeanF64<P, true, 1>, true, false>(plan, a, s)
                   : launch_term<Sech2LeanF64<P, false, 1>, true, false>(plan, a, s);
    }
    if (a.quad == 1) {
        if (phi) return launch_term<Sech2LeanF64<P, true, 1>, false, false>(plan, a, s);
        if (P == 2 && bulk_ok(a)) return launch_term<Sech2LeanF64<2, false, 1>, false, true>(plan, a, s);
        return launch_term<Sech2LeanF64<P, false, 1>, false, false>(plan, a, s);
    }
    if (phi) return cudaErrorInvalidValue;
    if (a.quad == 2) return launch_term<Sech2LeanF64<P, false, 2>, false, false>(plan, a, s);
    if (a.quad == 3) return launch_term<Sech2LeanF64<P, false, 3>, false, false>(plan, a, s);
    return cudaErrorInvalidValue;
}

}  // namespace

cudaError_t launch_wilson_sech2_f64(const EvalPlan& plan, const EvalArgs& a, cudaStream_t s)
{
    if (plan.P == 1) return launch_shape<1>(plan, a, s);
    if (plan.P == 2) return launch_shape<2>(plan, a, s);
    return cudaErrorInvalidValue;
}

}  // namespace wl
