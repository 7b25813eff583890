// wl_host.cu -- wl_eval_host: the end-to-end call on HOST buffers (include/wl.h).
// The only entry point that allocates device memory, copies and synchronises.
#include "wl_internal.cuh"

namespace {

struct DeviceBuffers {
    void* p[8] = {nullptr, nullptr, nullptr, nullptr, nullptr, nullptr, nullptr, nullptr};
    cudaStream_t s = nullptr;
    ~DeviceBuffers()
    {
        for (void* q : p) if (q) cudaFree(q);
        if (s) cudaStreamDestroy(s);
    }
};

}  // namespace

extern "C" wl_status wl_eval_host(const wl_field* field, const void* h_loops, wl_dtype loop_dtype,
                                  int64_t n_loops, int n_ppl, const double* h_T, int n_T,
                                  const double* h_rho_cm, const double* h_phi_cm, int n_rho, int n_groups,
                                  wl_dtype compute, double* h_W_mean, double* h_err, double* h_group_sums)
{
    if (!field || !h_loops || !h_T || !h_rho_cm || !h_W_mean) return WL_ERR_INVALID_ARG;
    if (loop_dtype != WL_F32 && loop_dtype != WL_F64) return WL_ERR_INVALID_ARG;
    const size_t ws = wl_eval_workspace_bytes(n_loops, n_ppl, n_T, n_rho, n_groups, compute);
    if (ws == 0) return WL_ERR_INVALID_ARG;
    if (h_err && n_groups < 2) return WL_ERR_INVALID_ARG;

    const size_t n_grid = (size_t)n_T * n_rho;
    const size_t loop_bytes = (size_t)n_loops * n_ppl * 2 * (loop_dtype == WL_F64 ? 8 : 4);
    DeviceBuffers d;
    enum { LOOPS, T, RHO, PHI, MEAN, GS, ERR, WS };
#define WL_TRY(call) do { if ((call) != cudaSuccess) { cudaGetLastError(); return WL_ERR_CUDA; } } while (0)
    WL_TRY(cudaStreamCreateWithFlags(&d.s, cudaStreamNonBlocking));
    WL_TRY(cudaMalloc(&d.p[LOOPS], loop_bytes));
    WL_TRY(cudaMalloc(&d.p[T], n_T * sizeof(double)));
    WL_TRY(cudaMalloc(&d.p[RHO], n_rho * sizeof(double)));
    if (h_phi_cm) WL_TRY(cudaMalloc(&d.p[PHI], n_rho * sizeof(double)));
    WL_TRY(cudaMalloc(&d.p[MEAN], 2 * n_grid * sizeof(double)));          // W_mean, then finalised mean
    WL_TRY(cudaMalloc(&d.p[GS], (size_t)n_groups * n_grid * sizeof(double)));
    WL_TRY(cudaMalloc(&d.p[ERR], n_grid * sizeof(double)));
    WL_TRY(cudaMalloc(&d.p[WS], ws));

    WL_TRY(cudaMemcpyAsync(d.p[LOOPS], h_loops, loop_bytes, cudaMemcpyHostToDevice, d.s));
    WL_TRY(cudaMemcpyAsync(d.p[T], h_T, n_T * sizeof(double), cudaMemcpyHostToDevice, d.s));
    WL_TRY(cudaMemcpyAsync(d.p[RHO], h_rho_cm, n_rho * sizeof(double), cudaMemcpyHostToDevice, d.s));
    if (h_phi_cm) WL_TRY(cudaMemcpyAsync(d.p[PHI], h_phi_cm, n_rho * sizeof(double), cudaMemcpyHostToDevice, d.s));

    double* mean = reinterpret_cast<double*>(d.p[MEAN]);
    wl_status st = wl_eval(field, d.p[LOOPS], loop_dtype, n_loops, n_ppl,
                           reinterpret_cast<const double*>(d.p[T]), n_T,
                           reinterpret_cast<const double*>(d.p[RHO]), reinterpret_cast<const double*>(d.p[PHI]),
                           n_rho, n_groups, compute, mean, reinterpret_cast<double*>(d.p[GS]), d.p[WS], ws, d.s);
    if (st != WL_OK) return st;
    if (h_err) {
        st = wl_jackknife_finalize(reinterpret_cast<const double*>(d.p[GS]), n_groups, n_loops, n_T, n_rho,
                                   mean + n_grid, reinterpret_cast<double*>(d.p[ERR]), nullptr, d.s);
        if (st != WL_OK) return st;
        WL_TRY(cudaMemcpyAsync(h_err, d.p[ERR], n_grid * sizeof(double), cudaMemcpyDeviceToHost, d.s));
    }
    WL_TRY(cudaMemcpyAsync(h_W_mean, mean, n_grid * sizeof(double), cudaMemcpyDeviceToHost, d.s));
    if (h_group_sums)
        WL_TRY(cudaMemcpyAsync(h_group_sums, d.p[GS], (size_t)n_groups * n_grid * sizeof(double),
                               cudaMemcpyDeviceToHost, d.s));
    WL_TRY(cudaStreamSynchronize(d.s));
#undef WL_TRY
    return WL_OK;
}
