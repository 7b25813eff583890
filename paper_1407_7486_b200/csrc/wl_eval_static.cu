// wl_eval_static.cu -- wl_eval for callers that can neither allocate device memory nor lend a workspace.
//
// Who that is: a host program that claimed the whole of HBM for its own pool at start-up (a later cudaMalloc
// fails, or fragments what the pool thinks it owns); a plug-in or callback that runs in a phase of its host
// application where cudaMalloc / cudaFree are forbidden because they synchronise the whole device and stall every
// other stream (a latency-bound service loop, a solver's inner iteration); code whose memory budget was fixed and
// audited before launch.  Such a caller has device buffers for its inputs and its results and nothing else, so
// the per-unit partial sums that k_wilson writes and k_group_reduce reads (wl_eval's `d_workspace`, eq. (60),
// PAPER.md:386, 399) have to live somewhere the library already owns.  Here that is a fixed array in the
// library's own device image: it exists on every GPU that loads this translation unit, from that moment until
// the process exits, and costs kStaticScratchBytes of that GPU's memory whether or not anybody calls this.
//
// The kernels, the plan and the summation order are wl_eval's (this file calls it), so the results have
// wl_eval's bits.  CUDA path, sm_100a.  Shares nothing with oracle/.
#include <mutex>

#include "wl_internal.cuh"

namespace {

// The limit (include/wl.h quotes it): 16 MiB = 2^21 FP64 partial sums.  Enough for BASELINE.json's config 1
// (1024 units x 256 grid points = 2 MiB) and for, e.g., 2048 loops on a 32 x 32 grid; the paper-scale
// configurations (134 MB and up) need wl_eval with a workspace of the caller's.
constexpr size_t kStaticScratchBytes = (size_t)16 << 20;

// In HOST code this name is only a handle for cudaGetSymbolAddress: it is not a device address, and a kernel
// handed `g_static_scratch` from the host side would fault (or, where the GPU can reach host memory, quietly
// scribble on the wrong memory).  Only scratch_address() below may touch it.
static __device__ __align__(256) double g_static_scratch[kStaticScratchBytes / sizeof(double)];

constexpr int kMaxDevices = 64;
std::mutex g_setup_mutex;
void* g_scratch_address[kMaxDevices];     // the array's device address on device ordinal d; null until set up

// Device address of g_static_scratch on the CURRENT device, looked up once per device and cached.  The array is
// one symbol but one copy per GPU, each at its own address, so the lookup must run with that device current.
cudaError_t scratch_address(void** out)
{
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    if (dev < 0 || dev >= kMaxDevices) return cudaErrorInvalidDevice;
    std::lock_guard<std::mutex> lock(g_setup_mutex);
    if (!g_scratch_address[dev]) {
        void* p = nullptr;
        e = cudaGetSymbolAddress(&p, g_static_scratch);
        if (e != cudaSuccess) return e;
        if (!p) return cudaErrorInvalidSymbol;
        g_scratch_address[dev] = p;
    }
    *out = g_scratch_address[dev];
    return cudaSuccess;
}

}  // namespace

extern "C" {

size_t wl_eval_static_max_bytes(void) { return kStaticScratchBytes; }

wl_status wl_eval_static(const wl_field* field, const void* d_loops, wl_dtype loop_dtype, int64_t n_loops, int n_ppl,
                         const double* d_T, int n_T, const double* d_rho_cm, const double* d_phi_cm, int n_rho,
                         int n_groups, wl_dtype compute, double* d_W_mean, double* d_group_sums, void* stream)
{
    if (!field || !d_loops || !d_T || !d_rho_cm || !d_W_mean || !d_group_sums) return WL_ERR_INVALID_ARG;
    // wl_eval's own size rules first (0 = sizes it would refuse), then this entry point's ceiling
    const size_t need = wl_eval_workspace_bytes(n_loops, n_ppl, n_T, n_rho, n_groups, compute);
    if (need == 0) return WL_ERR_INVALID_ARG;
    if (need > kStaticScratchBytes) return WL_ERR_STATIC_LIMIT;
    void* scratch = nullptr;
    if (scratch_address(&scratch) != cudaSuccess) {
        cudaGetLastError();
        return WL_ERR_CUDA;
    }
    // Nothing in the array has to start at zero: k_wilson stores every partial sum k_group_reduce will read
    // before that kernel runs, on the same stream, so whatever the previous call left behind is never read.
    return wl_eval(field, d_loops, loop_dtype, n_loops, n_ppl, d_T, n_T, d_rho_cm, d_phi_cm, n_rho, n_groups,
                   compute, d_W_mean, d_group_sums, scratch, kStaticScratchBytes, stream);
}

}  // extern "C"
