// wl_host.cu -- wl_eval_host: the end-to-end call on HOST buffers (include/wl.h).
// The only entry point that allocates device memory, copies and synchronises.
#include <mutex>

#include "wl_internal.cuh"

namespace {

// Device memory of wl_eval_host comes from a private stream-ordered pool (one per device) that keeps
// what it has been given between calls (release threshold = max), so that a second call of the
// same size pays no cudaMalloc/cudaFree; wl_eval_host_trim() gives the memory back.
cudaMemPool_t g_pool[64] = {};
std::mutex g_pool_mutex;

// The two streams (compute, copy) and two events of a call are created once per device and kept, like the
// pool; g_call_mutex[device] serialises the wl_eval_host calls on one device (they share these handles), while
// threads that drive different devices run side by side.
struct HostHandles {
    cudaStream_t s = nullptr, copy = nullptr;
    cudaEvent_t ev[2] = {nullptr, nullptr};
};
HostHandles g_handles[64];
std::mutex g_call_mutex[64];

cudaError_t host_handles(HostHandles** out)
{
    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    if (dev < 0 || dev >= 64) return cudaErrorInvalidDevice;
    HostHandles& h = g_handles[dev];
    if (!h.s && (e = cudaStreamCreateWithFlags(&h.s, cudaStreamNonBlocking)) != cudaSuccess) return e;
    if (!h.copy && (e = cudaStreamCreateWithFlags(&h.copy, cudaStreamNonBlocking)) != cudaSuccess) return e;
    for (cudaEvent_t& ev : h.ev)
        if (!ev && (e = cudaEventCreateWithFlags(&ev, cudaEventDisableTiming)) != cudaSuccess) return e;
    *out = &h;
    return cudaSuccess;
}

cudaError_t host_pool(cudaMemPool_t* out)
{
    std::lock_guard<std::mutex> lock(g_pool_mutex);
    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    if (dev < 0 || dev >= 64) return cudaErrorInvalidDevice;
    if (!g_pool[dev]) {
        cudaMemPoolProps props = {};
        props.allocType = cudaMemAllocationTypePinned;
        props.handleTypes = cudaMemHandleTypeNone;
        props.location.type = cudaMemLocationTypeDevice;
        props.location.id = dev;
        cudaMemPool_t pool;
        e = cudaMemPoolCreate(&pool, &props);
        if (e != cudaSuccess) return e;
        unsigned long long keep = ~0ull;
        e = cudaMemPoolSetAttribute(pool, cudaMemPoolAttrReleaseThreshold, &keep);
        if (e != cudaSuccess) { cudaMemPoolDestroy(pool); return e; }
        g_pool[dev] = pool;
    }
    *out = g_pool[dev];
    return cudaSuccess;
}

struct DeviceBuffers {
    void* p[8] = {nullptr, nullptr, nullptr, nullptr, nullptr, nullptr, nullptr, nullptr};
    cudaStream_t s = nullptr, copy = nullptr;
    cudaEvent_t ev[2] = {nullptr, nullptr};
    ~DeviceBuffers()
    {
        if (s) {
            if (copy) cudaStreamSynchronize(copy);   // a copy may still be writing into a buffer (early error return)
            for (void* q : p) if (q) cudaFreeAsync(q, s);
            cudaStreamSynchronize(s);
        }
    }
};

}  // namespace

extern "C" wl_status wl_eval_host_trim(void)
{
    std::lock_guard<std::mutex> lock(g_pool_mutex);
    int dev = 0;
    if (cudaGetDevice(&dev) != cudaSuccess) { cudaGetLastError(); return WL_ERR_CUDA; }
    if (dev >= 0 && dev < 64 && g_pool[dev]) {
        if (cudaMemPoolTrimTo(g_pool[dev], 0) != cudaSuccess) { cudaGetLastError(); return WL_ERR_CUDA; }
    }
    return WL_OK;
}

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
    enum { LOOPS, T, RHO, PHI, MEAN, GS, ERR, WS };
#define WL_TRY(call) do { if ((call) != cudaSuccess) { cudaGetLastError(); return WL_ERR_CUDA; } } while (0)
    int dev = -1;
    WL_TRY(cudaGetDevice(&dev));
    if (dev < 0 || dev >= 64) return WL_ERR_CUDA;
    // The lock is taken BEFORE the buffers exist, so that it is released AFTER ~DeviceBuffers has freed them and
    // synchronised the two shared streams: the next caller on this device never sees this call's work in flight.
    std::lock_guard<std::mutex> call_lock(g_call_mutex[dev]);
    DeviceBuffers d;
    HostHandles* hh = nullptr;
    WL_TRY(host_handles(&hh));
    d.s = hh->s; d.copy = hh->copy; d.ev[0] = hh->ev[0]; d.ev[1] = hh->ev[1];
    cudaMemPool_t pool;
    WL_TRY(host_pool(&pool));
#define WL_ALLOC(slot, bytes) do { const cudaError_t ea = cudaMallocFromPoolAsync(&d.p[slot], (bytes), pool, d.s); \
        if (ea != cudaSuccess) { cudaGetLastError(); return ea == cudaErrorMemoryAllocation ? WL_ERR_NOMEM : WL_ERR_CUDA; } } while (0)
    WL_ALLOC(LOOPS, loop_bytes);
    WL_ALLOC(T, n_T * sizeof(double));
    WL_ALLOC(RHO, n_rho * sizeof(double));
    if (h_phi_cm) WL_ALLOC(PHI, n_rho * sizeof(double));
    WL_ALLOC(MEAN, 2 * n_grid * sizeof(double));          // W_mean, then finalised mean
    WL_ALLOC(GS, (size_t)n_groups * n_grid * sizeof(double));
    WL_ALLOC(ERR, n_grid * sizeof(double));
    WL_ALLOC(WS, ws);
#undef WL_ALLOC

    WL_TRY(cudaMemcpyAsync(d.p[T], h_T, n_T * sizeof(double), cudaMemcpyHostToDevice, d.s));
    WL_TRY(cudaMemcpyAsync(d.p[RHO], h_rho_cm, n_rho * sizeof(double), cudaMemcpyHostToDevice, d.s));
    if (h_phi_cm) WL_TRY(cudaMemcpyAsync(d.p[PHI], h_phi_cm, n_rho * sizeof(double), cudaMemcpyHostToDevice, d.s));

    // Pipeline over chunks of whole jackknife groups: the copy of chunk 1 (copy stream) overlaps
    // k_wilson on chunk 0 (compute stream).  The units, their order and the partial-sum layout are
    // exactly those of one wl_eval over the whole ensemble, so the result has the same bits.
    const wl::EvalPlan plan = wl::make_eval_plan(n_loops, n_ppl, n_T, n_rho, n_groups, compute, false);
    const int64_t per_group = n_loops / n_groups;
    // Two chunks: a small first one (1/32 of the groups) whose evaluation hides the copy of the rest
    // (H2D moves a group ~30x faster than k_wilson evaluates it); more chunks would only add launch tails.
    const int n_chunks = n_groups >= 2 ? 2 : 1;
    const int g_first = n_groups >= 2 ? (n_groups / 32 > 0 ? n_groups / 32 : 1) : n_groups;
    const size_t loop_stride = (size_t)n_ppl * 2 * (loop_dtype == WL_F64 ? 8 : 4);
    double* mean = reinterpret_cast<double*>(d.p[MEAN]);
    double* partial = reinterpret_cast<double*>(d.p[WS]);
    WL_TRY(cudaEventRecord(d.ev[1], d.s));                    // the loop buffer exists (stream-ordered allocation)
    WL_TRY(cudaStreamWaitEvent(d.copy, d.ev[1], 0));
    for (int c = 0; c < n_chunks; ++c) {
        const int g0 = (c == 0) ? 0 : g_first, g1 = (c == n_chunks - 1) ? n_groups : g_first;
        const int64_t l0 = g0 * per_group, nl = (g1 - g0) * per_group;
        if (nl == 0) continue;
        char* dst = reinterpret_cast<char*>(d.p[LOOPS]) + (size_t)l0 * loop_stride;
        WL_TRY(cudaMemcpyAsync(dst, reinterpret_cast<const char*>(h_loops) + (size_t)l0 * loop_stride,
                               (size_t)nl * loop_stride, cudaMemcpyHostToDevice, d.copy));
        WL_TRY(cudaEventRecord(d.ev[0], d.copy));
        WL_TRY(cudaStreamWaitEvent(d.s, d.ev[0], 0));
        wl::EvalPlan sub = plan;
        sub.n_units = nl / plan.loops_per_unit;
        wl::EvalArgs a;
        a.loops = dst; a.loops_are_f64 = (loop_dtype == WL_F64); a.n_loops = nl; a.n_ppl = n_ppl;
        a.T = reinterpret_cast<const double*>(d.p[T]); a.rho = reinterpret_cast<const double*>(d.p[RHO]);
        a.phi = reinterpret_cast<const double*>(d.p[PHI]); a.n_T = n_T; a.n_rho = n_rho;
        a.p0 = field->p0; a.p1 = field->p1; a.scalar = field->scalar; a.disc = 0;
        a.quad = 1; a.seeded = 0; a.bulk = 0; a.seed = 0; a.loop_begin = 0;
        a.partial = partial + (size_t)(l0 / plan.loops_per_unit) * plan.n_grid;
        a.partial_in_walk_order = 1;
        a.phase_out = nullptr; a.spin_out = nullptr;
        cudaError_t e = wl::launch_wilson(sub, a, field->profile, compute, d.s);
        if (e != cudaSuccess) { cudaGetLastError(); return e == cudaErrorInvalidValue ? WL_ERR_UNSUPPORTED : WL_ERR_CUDA; }
    }
    if (wl::launch_group_reduce(partial, plan.units_per_group, n_groups, n_T, n_rho, n_loops,
                                reinterpret_cast<double*>(d.p[GS]), mean, d.s) != cudaSuccess) {
        cudaGetLastError();
        return WL_ERR_CUDA;
    }
    wl_status st = WL_OK;
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
