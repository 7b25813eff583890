// wl_api.cu -- the extern "C" entry points of include/wl.h: argument checks and launches only.
#include <cmath>
#include <new>

#include "wl_internal.cuh"

using namespace wl;

namespace {

bool sizes_ok(int64_t n_loops, int n_ppl, int n_T, int n_rho, int n_groups)
{
    if (n_loops < 1 || n_ppl < 1 || n_T < 1 || n_rho < 1 || n_groups < 1) return false;
    if (n_loops % n_groups != 0) return false;                       // equal groups
    if ((int64_t)n_T * n_rho > (1 << 24)) return false;
    if (n_loops > (1LL << 40)) return false;
    // launch limits, checked before anything is enqueued.  k_wilson: the exact CTA count (units x tiles) depends on
    // the kernel that is dispatched and is checked by launch_term before its launch (cudaErrorInvalidConfiguration ->
    // WL_ERR_INVALID_ARG, launch_status); here only what no kernel can launch: the largest unit is 8 loops, the
    // largest tile 1024 grid points (256 threads x 4).  The group reductions: n_groups x tiles(256 points), exact.
    const int64_t n_grid = (int64_t)n_T * n_rho;
    if (((n_loops + 7) / 8) * ((n_grid + 1023) / 1024) > 0x7fffffffLL) return false;
    if ((int64_t)n_groups * ((n_grid + 255) / 256) > 0x7fffffffLL) return false;
    return true;
}

bool dtype_ok(wl_dtype d) { return d == WL_F32 || d == WL_F64; }

bool seeded_ppl_ok(int n_ppl) { return n_ppl >= 2 && n_ppl <= kMaxPplSeeded && (n_ppl & (n_ppl - 1)) == 0; }

// Options as the launches see them; false on an invalid option block.
struct Opt {
    int quad = 1, seeded = 0, shuffle = 0, bulk = 0;
    uint64_t seed = 0, shuffle_seed = 0;
    int64_t loop_begin = 0;
    int64_t ensemble_loops = 0;      // 0: this call is the whole ensemble
    void* ev0 = nullptr;
    void* ev1 = nullptr;
};

bool read_options(const wl_eval_options* o, int n_ppl, int64_t n_loops, Opt* out)
{
    if (!o) return true;
    if (o->struct_size != sizeof(wl_eval_options)) return false;
    if (o->quadrature_order < 0 || o->quadrature_order > 3) return false;
    out->quad = o->quadrature_order == 0 ? 1 : o->quadrature_order;
    out->seeded = o->seeded != 0;
    out->seed = o->seed;
    out->loop_begin = o->loop_begin;
    if (out->seeded && (!seeded_ppl_ok(n_ppl) || o->loop_begin < 0)) return false;
    out->shuffle = o->shuffle_groups != 0;
    out->shuffle_seed = o->shuffle_seed;
    if (out->shuffle && n_loops > 0x7fffffffLL) return false;
    if (o->staging != 0 && o->staging != 1) return false;
    out->bulk = o->staging;
    if (o->ensemble_loops < 0 || (o->ensemble_loops > 0 && o->ensemble_loops < n_loops)) return false;
    out->ensemble_loops = o->ensemble_loops;
    out->ev0 = o->event_wilson_begin;
    out->ev1 = o->event_wilson_end;
    return true;
}

EvalArgs make_args(const wl_field* field, const void* d_loops, wl_dtype loop_dtype, int64_t n_loops, int n_ppl,
                   const double* d_T, int n_T, const double* d_rho_cm, const double* d_phi_cm, int n_rho,
                   const Opt& o)
{
    EvalArgs a;
    a.loops = d_loops; a.loops_are_f64 = (loop_dtype == WL_F64); a.n_loops = n_loops; a.n_ppl = n_ppl;
    a.T = d_T; a.rho = d_rho_cm; a.phi = d_phi_cm; a.n_T = n_T; a.n_rho = n_rho;
    a.p0 = field->p0; a.p1 = field->p1; a.scalar = field->scalar; a.disc = 0;
    a.quad = o.quad; a.seeded = o.seeded; a.bulk = o.bulk; a.seed = o.seed; a.loop_begin = o.loop_begin;
    a.partial = nullptr; a.partial_in_walk_order = 0; a.phase_out = nullptr; a.spin_out = nullptr;
    return a;
}

size_t align256(size_t b) { return (b + 255) & ~(size_t)255; }

wl_status launch_status(cudaError_t e)
{
    if (e == cudaSuccess) return WL_OK;
    cudaGetLastError();
    if (e == cudaErrorInvalidConfiguration) return WL_ERR_INVALID_ARG;     // more CTAs than a grid holds: nothing was launched
    return e == cudaErrorInvalidValue ? WL_ERR_UNSUPPORTED : WL_ERR_CUDA;
}

}  // namespace

extern "C" {

wl_status wl_field_create(wl_profile profile, const double* h_params, int n_params, wl_field** out)
{
    return wl_field_create_particle(profile, h_params, n_params, WL_FERMION, out);
}

wl_status wl_field_create_particle(wl_profile profile, const double* h_params, int n_params,
                                   wl_particle particle, wl_field** out)
{
    if (!out) return WL_ERR_INVALID_ARG;
    *out = nullptr;
    if (!h_params) return WL_ERR_INVALID_ARG;
    if (profile == WL_PROFILE_UNIFORM) {
        if (n_params != 1 || !std::isfinite(h_params[0])) return WL_ERR_INVALID_ARG;
    } else if (profile == WL_PROFILE_SECH2 || profile == WL_PROFILE_FLUXTUBE) {
        if (n_params != 2 || !std::isfinite(h_params[0]) || !std::isfinite(h_params[1]) || !(h_params[1] > 0.0))
            return WL_ERR_INVALID_ARG;
    } else {
        return WL_ERR_INVALID_ARG;
    }
    if (particle != WL_FERMION && particle != WL_SCALAR) return WL_ERR_INVALID_ARG;
    wl_field* f = new (std::nothrow) wl_field;
    if (!f) return WL_ERR_NOMEM;
    f->profile = (int)profile;
    f->p0 = h_params[0];
    f->p1 = (n_params > 1) ? h_params[1] : 0.0;
    f->scalar = (particle == WL_SCALAR);
    *out = f;
    return WL_OK;
}

void wl_field_destroy(wl_field* field) { delete field; }

wl_status wl_grid_validate(const double* h_T, int n_T, const double* h_rho_cm, int n_rho)
{
    if (!h_T || !h_rho_cm || n_T < 1 || n_rho < 1) return WL_ERR_INVALID_ARG;
    for (int k = 0; k < n_T; ++k)
        if (!std::isfinite(h_T[k]) || !(h_T[k] > 0.0)) return WL_ERR_INVALID_ARG;
    for (int k = 0; k < n_rho; ++k)
        if (!std::isfinite(h_rho_cm[k]) || !(h_rho_cm[k] >= 0.0)) return WL_ERR_INVALID_ARG;
    return WL_OK;
}

wl_status wl_loops_generate(void* d_loops, wl_dtype storage, int64_t loop_begin, int64_t n_loops, int n_ppl,
                            uint64_t seed, void* stream)
{
    if (!dtype_ok(storage) || n_loops < 0 || loop_begin < 0) return WL_ERR_INVALID_ARG;
    if (!seeded_ppl_ok(n_ppl)) return WL_ERR_INVALID_ARG;
    if (n_loops == 0) return WL_OK;
    if (!d_loops) return WL_ERR_INVALID_ARG;
    return launch_status(launch_generate(d_loops, storage == WL_F64, loop_begin, n_loops, n_ppl, seed,
                                         (cudaStream_t)stream));
}

void wl_eval_options_default(wl_eval_options* opt)
{
    if (!opt) return;
    *opt = wl_eval_options();
    opt->struct_size = sizeof(wl_eval_options);
    opt->quadrature_order = 1;
}

size_t wl_eval_workspace_bytes(int64_t n_loops, int n_ppl, int n_T, int n_rho, int n_groups, wl_dtype compute)
{
    return wl_eval_opt_workspace_bytes(n_loops, n_ppl, n_T, n_rho, n_groups, compute, nullptr);
}

size_t wl_eval_opt_workspace_bytes(int64_t n_loops, int n_ppl, int n_T, int n_rho, int n_groups, wl_dtype compute,
                                   const wl_eval_options* opt)
{
    if (!sizes_ok(n_loops, n_ppl, n_T, n_rho, n_groups) || !dtype_ok(compute)) return 0;
    Opt o;
    if (!read_options(opt, n_ppl, n_loops, &o)) return 0;
    if (o.ensemble_loops % (n_loops / n_groups) != 0) return 0;
    const EvalPlan p = make_eval_plan(n_loops, n_ppl, n_T, n_rho, n_groups, compute, o.shuffle != 0, o.ensemble_loops);
    const size_t partial = (size_t)p.n_units * (size_t)p.n_grid * sizeof(double);
    if (!o.shuffle) return partial;
    return align256(partial) + align256((size_t)n_T * (size_t)n_loops * sizeof(int32_t));   // W per loop, membership table
}

int wl_eval_launch_count(int64_t n_loops, int n_ppl, int n_T, int n_rho, int n_groups, wl_dtype compute)
{
    if (!sizes_ok(n_loops, n_ppl, n_T, n_rho, n_groups) || !dtype_ok(compute)) return 0;
    return 3;   // k_wilson, k_group_reduce, k_mean
}

wl_status wl_eval(const wl_field* field, const void* d_loops, wl_dtype loop_dtype, int64_t n_loops, int n_ppl,
                  const double* d_T, int n_T, const double* d_rho_cm, const double* d_phi_cm, int n_rho,
                  int n_groups, wl_dtype compute, double* d_W_mean, double* d_group_sums,
                  void* d_workspace, size_t workspace_bytes, void* stream)
{
    return wl_eval_opt(field, d_loops, loop_dtype, n_loops, n_ppl, d_T, n_T, d_rho_cm, d_phi_cm, n_rho, n_groups,
                       compute, d_W_mean, d_group_sums, d_workspace, workspace_bytes, stream, nullptr);
}

wl_status wl_eval_instrumented(const wl_field* field, const void* d_loops, wl_dtype loop_dtype, int64_t n_loops,
                               int n_ppl, const double* d_T, int n_T, const double* d_rho_cm,
                               const double* d_phi_cm, int n_rho, int n_groups, wl_dtype compute,
                               double* d_W_mean, double* d_group_sums, void* d_workspace,
                               size_t workspace_bytes, void* stream, void* event_wilson_begin,
                               void* event_wilson_end)
{
    wl_eval_options opt;
    wl_eval_options_default(&opt);
    opt.event_wilson_begin = event_wilson_begin;
    opt.event_wilson_end = event_wilson_end;
    return wl_eval_opt(field, d_loops, loop_dtype, n_loops, n_ppl, d_T, n_T, d_rho_cm, d_phi_cm, n_rho, n_groups,
                       compute, d_W_mean, d_group_sums, d_workspace, workspace_bytes, stream, &opt);
}

wl_status wl_eval_seeded(const wl_field* field, uint64_t seed, int64_t loop_begin, wl_dtype storage,
                         int64_t n_loops, int n_ppl, const double* d_T, int n_T, const double* d_rho_cm,
                         const double* d_phi_cm, int n_rho, int n_groups, wl_dtype compute, double* d_W_mean,
                         double* d_group_sums, void* d_workspace, size_t workspace_bytes, void* stream)
{
    wl_eval_options opt;
    wl_eval_options_default(&opt);
    opt.seeded = 1;
    opt.seed = seed;
    opt.loop_begin = loop_begin;
    return wl_eval_opt(field, nullptr, storage, n_loops, n_ppl, d_T, n_T, d_rho_cm, d_phi_cm, n_rho, n_groups,
                       compute, d_W_mean, d_group_sums, d_workspace, workspace_bytes, stream, &opt);
}

wl_status wl_eval_opt(const wl_field* field, const void* d_loops, wl_dtype loop_dtype, int64_t n_loops, int n_ppl,
                      const double* d_T, int n_T, const double* d_rho_cm, const double* d_phi_cm, int n_rho,
                      int n_groups, wl_dtype compute, double* d_W_mean, double* d_group_sums,
                      void* d_workspace, size_t workspace_bytes, void* stream, const wl_eval_options* opt)
{
    if (!field || !d_T || !d_rho_cm || !d_W_mean || !d_group_sums) return WL_ERR_INVALID_ARG;
    if (!dtype_ok(loop_dtype) || !dtype_ok(compute)) return WL_ERR_INVALID_ARG;
    if (!sizes_ok(n_loops, n_ppl, n_T, n_rho, n_groups)) return WL_ERR_INVALID_ARG;
    Opt o;
    if (!read_options(opt, n_ppl, n_loops, &o)) return WL_ERR_INVALID_ARG;
    if (!o.seeded && !d_loops) return WL_ERR_INVALID_ARG;
    if (o.shuffle && o.ensemble_loops > 0) return WL_ERR_UNSUPPORTED;     // a shard cannot shuffle across shards
    const size_t need = wl_eval_opt_workspace_bytes(n_loops, n_ppl, n_T, n_rho, n_groups, compute, opt);
    if (need == 0) return WL_ERR_INVALID_ARG;
    if (!d_workspace || workspace_bytes < need) return WL_ERR_WORKSPACE;
    const EvalPlan plan = make_eval_plan(n_loops, n_ppl, n_T, n_rho, n_groups, compute, o.shuffle != 0, o.ensemble_loops);

    EvalArgs a = make_args(field, d_loops, loop_dtype, n_loops, n_ppl, d_T, n_T, d_rho_cm, d_phi_cm, n_rho, o);
    a.partial = reinterpret_cast<double*>(d_workspace);
    a.partial_in_walk_order = o.shuffle ? 0 : 1;          // shuffled groups: the array is W per loop, read as [t][r]
    cudaStream_t s = (cudaStream_t)stream;
    if (o.ev0 && cudaEventRecord((cudaEvent_t)o.ev0, s) != cudaSuccess) return launch_status(cudaErrorUnknown);
    cudaError_t e = launch_wilson(plan, a, field->profile, compute, s);
    if (e != cudaSuccess) return launch_status(e);
    if (o.ev1 && cudaEventRecord((cudaEvent_t)o.ev1, s) != cudaSuccess) return launch_status(cudaErrorUnknown);
    if (!o.shuffle)
        return launch_status(launch_group_reduce(a.partial, plan.units_per_group, n_groups, n_T, n_rho, n_loops,
                                                 d_group_sums, d_W_mean, s));
    // shuffled groups: the workspace holds W per loop, then the membership table
    int32_t* perm = reinterpret_cast<int32_t*>(reinterpret_cast<unsigned char*>(d_workspace)
                                               + align256((size_t)n_loops * plan.n_grid * sizeof(double)));
    e = launch_group_permutation(o.shuffle_seed, n_loops, n_T, perm, s);
    if (e != cudaSuccess) return launch_status(e);
    return launch_status(launch_group_reduce_shuffled(a.partial, perm, n_loops, n_T, n_rho, n_groups, d_group_sums,
                                                      d_W_mean, s));
}

wl_status wl_group_permutation(uint64_t shuffle_seed, int64_t n_loops, int n_T, int32_t* d_perm, void* stream)
{
    if (!d_perm || n_loops < 1 || n_loops > 0x7fffffffLL || n_T < 1) return WL_ERR_INVALID_ARG;
    if ((n_loops * n_T + 255) / 256 > 0x7fffffffLL) return WL_ERR_INVALID_ARG;
    return launch_status(launch_group_permutation(shuffle_seed, n_loops, n_T, d_perm, (cudaStream_t)stream));
}

namespace {

// Plan of the discretisation run: the plan of an ordinary run over N/2 terms per pass, with at most
// two grid points per thread (each carries three running W sums).
EvalPlan make_disc_plan(int64_t n_loops, int n_ppl, int n_T, int n_rho, int n_groups, wl_dtype compute)
{
    EvalPlan p = make_eval_plan(n_loops, n_ppl / 2, n_T, n_rho, n_groups, compute, false);
    if (p.P > 2) { p.P = 2; p.n_tiles = (p.n_grid + p.threads * 2 - 1) / (p.threads * 2); }
    return p;
}

}  // namespace

size_t wl_eval_discretization_workspace_bytes(int64_t n_loops, int n_ppl, int n_T, int n_rho, int n_groups,
                                              wl_dtype compute)
{
    if (!sizes_ok(n_loops, n_ppl, n_T, n_rho, n_groups) || !dtype_ok(compute)) return 0;
    if (n_ppl < 4 || n_ppl % 4 != 0) return 0;
    const EvalPlan p = make_disc_plan(n_loops, n_ppl, n_T, n_rho, n_groups, compute);
    return 3 * (size_t)p.n_units * (size_t)p.n_grid * sizeof(double);
}

wl_status wl_eval_discretization(const wl_field* field, const void* d_loops, wl_dtype loop_dtype,
                                 int64_t n_loops, int n_ppl, const double* d_T, int n_T,
                                 const double* d_rho_cm, const double* d_phi_cm, int n_rho, int n_groups,
                                 wl_dtype compute, double* d_group_sums3, void* d_workspace,
                                 size_t workspace_bytes, void* stream)
{
    if (!field || !d_loops || !d_T || !d_rho_cm || !d_group_sums3) return WL_ERR_INVALID_ARG;
    if (!dtype_ok(loop_dtype) || !dtype_ok(compute)) return WL_ERR_INVALID_ARG;
    if (!sizes_ok(n_loops, n_ppl, n_T, n_rho, n_groups)) return WL_ERR_INVALID_ARG;
    if (n_ppl < 4 || n_ppl % 4 != 0) return WL_ERR_INVALID_ARG;            // three interleaved sub-worldlines
    const EvalPlan plan = make_disc_plan(n_loops, n_ppl, n_T, n_rho, n_groups, compute);
    const size_t level = (size_t)plan.n_units * (size_t)plan.n_grid;
    if (!d_workspace || workspace_bytes < 3 * level * sizeof(double)) return WL_ERR_WORKSPACE;

    EvalArgs a = make_args(field, d_loops, loop_dtype, n_loops, n_ppl, d_T, n_T, d_rho_cm, d_phi_cm, n_rho, Opt());
    a.disc = 1;
    a.partial = reinterpret_cast<double*>(d_workspace);
    a.partial_in_walk_order = 1;
    cudaStream_t s = (cudaStream_t)stream;
    cudaError_t e = launch_wilson(plan, a, field->profile, compute, s);
    if (e != cudaSuccess) return launch_status(e);
    for (int lev = 0; lev < 3; ++lev) {
        e = launch_group_reduce(a.partial + lev * level, plan.units_per_group, n_groups, n_T, n_rho,
                                n_loops, d_group_sums3 + (size_t)lev * n_groups * plan.n_grid, nullptr, s);
        if (e != cudaSuccess) return launch_status(e);
    }
    return WL_OK;
}

wl_status wl_extrapolate(const double* d_levels3, int64_t n, double* d_W_inf, double* d_delta, void* stream)
{
    if (!d_levels3 || !d_W_inf || n < 1) return WL_ERR_INVALID_ARG;
    return launch_status(launch_extrapolate(d_levels3, n, d_W_inf, d_delta, (cudaStream_t)stream));
}

wl_status wl_eval_per_loop(const wl_field* field, const void* d_loops, wl_dtype loop_dtype, int64_t n_loops,
                           int n_ppl, const double* d_T, int n_T, const double* d_rho_cm,
                           const double* d_phi_cm, int n_rho, wl_dtype compute,
                           double* d_W, double* d_phase, double* d_spin, void* stream)
{
    return wl_eval_per_loop_opt(field, d_loops, loop_dtype, n_loops, n_ppl, d_T, n_T, d_rho_cm, d_phi_cm, n_rho,
                                compute, d_W, d_phase, d_spin, stream, nullptr);
}

wl_status wl_eval_per_loop_opt(const wl_field* field, const void* d_loops, wl_dtype loop_dtype, int64_t n_loops,
                               int n_ppl, const double* d_T, int n_T, const double* d_rho_cm,
                               const double* d_phi_cm, int n_rho, wl_dtype compute,
                               double* d_W, double* d_phase, double* d_spin, void* stream,
                               const wl_eval_options* opt)
{
    if (!field || !d_T || !d_rho_cm || !d_W) return WL_ERR_INVALID_ARG;
    if (!dtype_ok(loop_dtype) || !dtype_ok(compute)) return WL_ERR_INVALID_ARG;
    if (!sizes_ok(n_loops, n_ppl, n_T, n_rho, 1)) return WL_ERR_INVALID_ARG;
    Opt o;
    if (!read_options(opt, n_ppl, 1, &o)) return WL_ERR_INVALID_ARG;
    if (!o.seeded && !d_loops) return WL_ERR_INVALID_ARG;
    const EvalPlan plan = make_eval_plan(n_loops, n_ppl, n_T, n_rho, 1, compute, true);
    EvalArgs a = make_args(field, d_loops, loop_dtype, n_loops, n_ppl, d_T, n_T, d_rho_cm, d_phi_cm, n_rho, o);
    a.partial = d_W; a.phase_out = d_phase; a.spin_out = d_spin;
    return launch_status(launch_wilson(plan, a, field->profile, compute, (cudaStream_t)stream));
}

wl_status wl_jackknife_finalize(const double* d_group_sums, int n_groups, int64_t n_loops, int n_T, int n_rho,
                                double* d_mean, double* d_err, double* d_delete_one, void* stream)
{
    if (!d_group_sums || !d_mean || !d_err) return WL_ERR_INVALID_ARG;
    if (n_groups < 2 || n_loops < 1 || n_loops % n_groups != 0 || n_T < 1 || n_rho < 1) return WL_ERR_INVALID_ARG;
    if ((int64_t)n_T * n_rho > (1 << 24)) return WL_ERR_INVALID_ARG;
    return launch_status(launch_finalize(d_group_sums, n_groups, n_loops, n_T * n_rho, d_mean, d_err, d_delete_one,
                                         (cudaStream_t)stream));
}

const char* wl_status_string(wl_status status)
{
    switch (status) {
        case WL_OK: return "ok";
        case WL_ERR_INVALID_ARG: return "invalid argument";
        case WL_ERR_UNSUPPORTED: return "unsupported configuration";
        case WL_ERR_WORKSPACE: return "workspace missing or too small";
        case WL_ERR_CUDA: return "CUDA runtime error";
        case WL_ERR_NOMEM: return "out of host or device memory";
        case WL_ERR_STATIC_LIMIT: return "sizes need more scratch than wl_eval_static's built-in array (wl_eval_static_max_bytes): use wl_eval with a workspace";
    }
    return "unknown status";
}

const char* wl_version(void) { return "2.1"; }

}  // extern "C"
