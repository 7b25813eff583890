// wl_wilson_fluxtube_f32.cu -- instantiations of k_wilson<FluxTubePackedF32<...>> (wl_terms_packed_f32.cuh on
// the scaffold of wl_wilson_body.cuh): the FP32 hot loop for the paper's own validation profile
// f_lambda = rho^2/(lambda^2+rho^2) (eq. (68); Fig. 11, 12).  CUDA path, sm_100a only.
#include "wl_terms_packed_f32.cuh"

namespace wl {

namespace {

// Same combinations as the sech^2 kernels (wl_wilson_sech2_f32.cu), without the bulk-staging variant.
template <int P, int TH>
cudaError_t launch_shape(const EvalPlan& plan, const EvalArgs& a, cudaStream_t s)
{
    const bool phi = a.phi != nullptr;
    if (a.disc) {
        if (a.quad != 1) return cudaErrorInvalidValue;
        return phi ? launch_term<FluxTubePackedF32<P, TH, true, 1>, true, false>(plan, a, s)
                   : launch_term<FluxTubePackedF32<P, TH, false, 1>, true, false>(plan, a, s);
    }
    if (a.quad == 1)
        return phi ? launch_term<FluxTubePackedF32<P, TH, true, 1>, false, false>(plan, a, s)
                   : launch_term<FluxTubePackedF32<P, TH, false, 1>, false, false>(plan, a, s);
    if (phi) return cudaErrorInvalidValue;
    if (a.quad == 2) return launch_term<FluxTubePackedF32<P, TH, false, 2>, false, false>(plan, a, s);
    if (a.quad == 3) return launch_term<FluxTubePackedF32<P, TH, false, 3>, false, false>(plan, a, s);
    return cudaErrorInvalidValue;
}

}  // namespace

cudaError_t launch_wilson_fluxtube_f32(const EvalPlan& plan, const EvalArgs& a, cudaStream_t s)
{
    if (plan.n_grid <= 256) return launch_shape<2, 128>(plan, a, s);
    if (plan.P == 2) return launch_shape<2, 256>(plan, a, s);
    if (plan.P == 4) return launch_shape<4, 256>(plan, a, s);
    return cudaErrorInvalidValue;
}

}  // namespace wl
