/*
 * wl.h -- C ABI of the B200-native worldline-numerics hot path (libwl.so).
 *
 * Method: Mazur & Heyl, "Parallel Worldline Numerics: Implementation and Error
 * Analysis", arXiv:1407.7486.  Citations are "PAPER.md:<line>" of the text of
 * that paper plus its section / equation number.
 *
 * What the library computes (DESIGN.md section 1 has the full statement):
 *   for every unit loop y_l (N points, 2-D), proper time T_t and centre of
 *   mass x_cm,r = rho_r (cos phi_r, sin phi_r):
 *     x_i   = x_cm + sqrt(T) y_i                                eq. (8),
 *     phase = sum_i g(|m_i|) (m_i x d_i),  m_i = (x_i+x_{i+1})/2,
 *             d_i = x_{i+1}-x_i, i+1 mod N, g = e A_phi/rho     eq. (21)-(24)
 *     spin  = (T/N) sum_i e B(|x_i|)                            eq. (31)-(33)
 *     W     = cos(phase) cosh(spin)                             eq. (18)
 *   S_g = sum of W over the loops of jackknife group g          eq. (60)
 *   <W> = (sum_g S_g)/N_l                                       eq. (61)-(62)
 *   err = sqrt(sum_g (<W>_g - <W>)^2 / (G (G-1)))               eq. (63)
 *
 * Conventions
 *   - "d_" pointers are DEVICE pointers, "h_" pointers are HOST pointers.
 *   - The caller owns every buffer.  Except for wl_eval_host (which says so),
 *     no call allocates device memory, synchronises the stream or the device,
 *     or copies between host and device: all work is enqueued on `stream`.
 *   - `stream` is a cudaStream_t passed as void* (NULL = the legacy default
 *     stream), so that this header needs no CUDA header.
 *   - All grids and results are FP64.  Loop coordinates are FP32 or FP64,
 *     array-of-points: loops[l][i][c], c = 0 (x), 1 (y), contiguous.
 *   - Every call returns a wl_status; nothing is printed, nothing aborts.
 *     Argument errors (WL_ERR_INVALID_ARG, WL_ERR_UNSUPPORTED, WL_ERR_WORKSPACE) are found before
 *     anything is enqueued; on any status other than WL_OK no result buffer is valid.
 *     (The paper's convention is "check the code, print the string",
 *     PAPER.md:603-628; wl_status_string gives the string.)
 *   - There is no CPU fallback: without a CUDA device the compute calls
 *     return WL_ERR_CUDA.
 */
#ifndef WL_H
#define WL_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef enum {
    WL_OK = 0,
    WL_ERR_INVALID_ARG = 1,   /* null pointer, bad size, bad parameter value     */
    WL_ERR_UNSUPPORTED = 2,   /* valid request this build has no kernel for      */
    WL_ERR_WORKSPACE = 3,     /* workspace null or smaller than *_workspace_bytes */
    WL_ERR_CUDA = 4,          /* a CUDA runtime call failed (no device, launch)  */
    WL_ERR_STATIC_LIMIT = 5,  /* wl_eval_static only: the sizes need more scratch than the library's
                                 built-in array holds (wl_eval_static_max_bytes); use wl_eval */
    WL_ERR_NOMEM = 6          /* an allocation failed: the field object (host), wl_eval_host's buffers (device) */
} wl_status;

/* Field profiles B_z(rho), gauge A = A_phi(rho) e_phi, A_phi = Phi(rho)/(2 pi rho)
 * (eq. (13)-(17)).  The charge e is folded into the strength. */
typedef enum {
    WL_PROFILE_UNIFORM = 0,   /* params {eB}:           B_z = B, A = (B/2)(-y, x)            */
    WL_PROFILE_SECH2 = 1,     /* params {eB0, lambda}:  B_z = B0 sech^2(rho/lambda),
                                 Phi = 2 pi B0 [lambda rho tanh(rho/lambda)
                                               - lambda^2 ln cosh(rho/lambda)]               */
    WL_PROFILE_FLUXTUBE = 2   /* params {script-F, lambda}: the paper's validation profile
                                 f_lambda = rho^2/(lambda^2+rho^2), eq. (68), in
                                 A_phi = F f_lambda/(2 pi rho), eq. (14); script-F = eF/2pi, eq. (17):
                                 e A_phi/rho = script-F/(lambda^2+rho^2),
                                 e B_z = 2 script-F lambda^2/(lambda^2+rho^2)^2              */
} wl_profile;

/* What the loop belongs to (eq. (18)): a fermion loop carries the spin factor,
 * W = cos(phase) cosh(spin); a scalar loop (scalar QED, the paper's Wsscal)
 * has W = cos(phase) only (exact uniform-field average eq. (43)). */
typedef enum { WL_FERMION = 0, WL_SCALAR = 1 } wl_particle;

typedef enum { WL_F32 = 0, WL_F64 = 1 } wl_dtype;

typedef struct wl_field wl_field;   /* opaque, host memory, immutable after creation */

/* Creates a field description: the profile B_z(rho) and its gauge potential, eq. (13)-(17).
 * h_params: UNIFORM n_params == 1 {eB};
 * SECH2 n_params == 2 {eB0, lambda}, lambda > 0.  Non-finite values, lambda <= 0,
 * a wrong n_params or an unknown profile give WL_ERR_INVALID_ARG and *out = NULL.
 * The caller releases it with wl_field_destroy.  Host-only; no CUDA call. */
wl_status wl_field_create(wl_profile profile, const double* h_params, int n_params, wl_field** out);
/* Same with the particle type stated (wl_field_create = WL_FERMION; eq. (18)); FLUXTUBE: n_params == 2,
 * {script-F, lambda}, lambda > 0.  An unknown particle gives WL_ERR_INVALID_ARG. */
wl_status wl_field_create_particle(wl_profile profile, const double* h_params, int n_params,
                                   wl_particle particle, wl_field** out);
void wl_field_destroy(wl_field* field);   /* NULL is allowed */

/* Seeded unit-loop ensemble: d-loops, steps (1)-(5), eq. (10)-(11), PAPER.md:65-81,
 * centre of mass shifted to the origin, driven by Philox4x32-10 with counter
 * (point, loop_lo, loop_hi, 0) and key (seed_lo, seed_hi) (reading A11).
 * Writes loops [loop_begin, loop_begin + n_loops) of the ensemble `seed` to
 * d_loops[n_loops][n_ppl][2] in `storage` precision (arithmetic is FP64; FP32
 * storage rounds once at the store).  Loop l of an ensemble is the same whatever
 * loop_begin / n_loops window it is generated in.
 * n_ppl: power of two, 2 <= n_ppl <= 65536.  n_loops == 0 is a no-op.  */
wl_status wl_loops_generate(void* d_loops, wl_dtype storage, int64_t loop_begin, int64_t n_loops,
                            int n_ppl, uint64_t seed, void* stream);

/* Bytes of device workspace wl_eval needs for these sizes (0 on invalid sizes).
 * The workspace holds the partial sums of eq. (60), one per unit of consecutive loops and grid
 * point, which the group reduction adds in unit order; its contents are scratch. */
size_t wl_eval_workspace_bytes(int64_t n_loops, int n_ppl, int n_T, int n_rho, int n_groups,
                               wl_dtype compute);

/* The hot path.  For every (T_t, rho_r[, phi_r]) evaluates W for all loops and
 * reduces them, in a fixed order that depends only on the argument sizes:
 *   d_W_mean[t][r]        = <W>                    (n_T x n_rho, FP64)
 *   d_group_sums[g][t][r] = S_g, group g = loops [g n_loops/G, (g+1) n_loops/G)
 * d_loops [n_loops][n_ppl][2] of loop_dtype; n_ppl >= 1 (any value, not only
 * powers of two).  d_T[n_T] > 0; d_rho_cm[n_rho] >= 0; d_phi_cm[n_rho] or NULL
 * (= all zero).  Grid VALUES live on the device and are not read by this call: T <= 0 or a
 * non-finite value gives NaN rows, not an error.  wl_grid_validate checks a host copy.
 * FP32 range: for the sech^2 and flux-tube profiles with 1e-4 <= lambda <= 1e4 the FP32 kernels carry
 * squared radii divided by lambda^2; they stay finite while (rho_cm + sqrt(T) |y|)/lambda < 1e18.
 * compute = WL_F64: all arithmetic FP64.  compute = WL_F32: per-term arithmetic
 * FP32 with fast intrinsics, the sums round a loop accumulated in FP64 from
 * FP32 partials of at most 128 terms, cos/cosh and all sums over loops FP64.
 * Errors: null pointers, sizes < 1, n_groups < 1, n_loops % n_groups != 0
 * (equal groups are required), n_T * n_rho > 2^24, more than 2^31 - 1 CTAs
 * -> WL_ERR_INVALID_ARG; workspace too small -> WL_ERR_WORKSPACE. */
wl_status wl_eval(const wl_field* field,
                  const void* d_loops, wl_dtype loop_dtype, int64_t n_loops, int n_ppl,
                  const double* d_T, int n_T,
                  const double* d_rho_cm, const double* d_phi_cm, int n_rho,
                  int n_groups, wl_dtype compute,
                  double* d_W_mean, double* d_group_sums,
                  void* d_workspace, size_t workspace_bytes, void* stream);

/* wl_eval for a caller that cannot allocate device memory and has no buffer to lend as workspace.
 *
 * wl_eval keeps its per-unit partial sums (k_wilson writes them, the group reduction of eq. (60),
 * PAPER.md:386, 399, reads them) in a workspace the caller allocates.  Some callers cannot: a program
 * that gave all of HBM to its own pool when it started, so that a cudaMalloc now fails; a plug-in or
 * callback running where its host application forbids cudaMalloc / cudaFree because both stall every
 * stream of the device; a job whose device-memory budget was fixed before launch.  For them the same
 * evaluation runs with the partial sums in an array that is part of the library's device image:
 *   - the array is wl_eval_static_max_bytes() = 16 MiB, present on every GPU that has used this entry
 *     point (or whose CUDA module holding it was loaded) until the process exits, used or not;
 *   - sizes with wl_eval_workspace_bytes(...) above that limit are refused with WL_ERR_STATIC_LIMIT
 *     before anything is enqueued (BASELINE.json's config 1 needs 2 MiB; the paper-scale ones do not fit);
 *   - the call makes no cudaMalloc, cudaFree or other allocating call, on the host or on the device; the
 *     caller passes inputs and outputs exactly as to wl_eval, and the results have wl_eval's bits;
 *   - the first call on each device looks the array's address up (cudaGetSymbolAddress, with that device
 *     current, which may load the module) and caches it: make that first call during set-up, on the
 *     device the later calls will use, and before any stream capture is begun;
 *   - there is ONE array per device and every call uses it, keeping whatever the last call left there.
 *     No clearing is needed (each call writes every partial sum before reading it), but two calls whose
 *     kernels can overlap on the GPU -- different streams, or different host threads on different
 *     streams -- race on it and both results are garbage.  Calls on one stream are ordered and safe.
 * Plain midpoint rule, stored loops, contiguous groups only (no options block).
 * Errors: as wl_eval; WL_ERR_STATIC_LIMIT as above; WL_ERR_CUDA if the address look-up fails. */
size_t wl_eval_static_max_bytes(void);
wl_status wl_eval_static(const wl_field* field,
                         const void* d_loops, wl_dtype loop_dtype, int64_t n_loops, int n_ppl,
                         const double* d_T, int n_T,
                         const double* d_rho_cm, const double* d_phi_cm, int n_rho,
                         int n_groups, wl_dtype compute,
                         double* d_W_mean, double* d_group_sums, void* stream);

/* Host helper: WL_OK if every h_T[k] is finite and > 0 and every h_rho_cm[k] is finite and >= 0
 * ("T <= 0, negative rho_cm -> invalid"), else WL_ERR_INVALID_ARG.
 * The evaluation calls take DEVICE grids and cannot check them without a synchronisation. */
wl_status wl_grid_validate(const double* h_T, int n_T, const double* h_rho_cm, int n_rho);

/* ---- Options of the extended evaluation calls ------------------
 *
 * quadrature_order (eq. (24)-(28)): number Q of Gauss-Legendre points in t for
 *   int_0^1 dt f(rho_i^2(t))/rho_i^2(t) with rho_i^2(t) = A_i + 2 B_i t + C_i t^2 (eq. (25)):
 *   0 or 1 = the one-point midpoint rule of wl_eval; 2: t = 1/2 -+ 1/(2 sqrt 3), weights 1/2;
 *   3: t = 1/2 -+ sqrt(3/5)/2, 1/2, weights 5/18, 4/9, 5/18.  The spin sum is unchanged.
 *   Q > 1 together with the discretisation estimate -> WL_ERR_UNSUPPORTED.
 *
 * seeded ("generating the loops on-the-fly directly on the GPU device itself without
 *   storing the entire loop in memory", the device-memory ceiling): non-zero = d_loops
 *   is ignored (may be NULL); loop l is regenerated inside the kernel as loop (loop_begin + l) of
 *   the ensemble `seed`, exactly as wl_loops_generate would have stored it in `loop_dtype`
 *   precision: the results have the same bits as wl_loops_generate followed by wl_eval.
 *   n_ppl must be a power of two, 2 <= n_ppl <= 65536.
 *
 * shuffle_groups (Sec. IV.B.3; Fig. 6: "randomize how worldlines are
 *   assigned to groups between each evaluation of the integrand"): non-zero = every proper-time
 *   index t has its own permutation pi_t of the loops (see wl_group_permutation) and group g at
 *   that T holds the loops pi_t(i), g n_loops/G <= i < (g+1) n_loops/G, summed in the order of i.
 *   <W> is unchanged up to rounding (eq. (61)-(62)).  Needs n_loops < 2^31 and the larger
 *   workspace of wl_eval_opt_workspace_bytes (all per-loop W values are kept: 8 n_loops n_T n_rho bytes).
 *
 * staging: 0 = loop chunks are read by ordinary coalesced loads; 1 = by cp.async.bulk into a
 *   two-slot shared-memory ring with mbarrier completion, one chunk ahead of the evaluation
 *   (compiled for the main kernels only, silently 0 elsewhere; same bits either way).
 *
 * ensemble_loops: 0, or the number of loops of the whole ensemble when this call evaluates one shard of it
 *   (whole jackknife groups).  The work is then cut into the same units of loops as
 *   in one call over the whole ensemble, so every group sum has the same bits however many shards there are.
 *   Must be a multiple of n_loops' group size and >= n_loops, else WL_ERR_INVALID_ARG.
 *
 * event_wilson_begin / event_wilson_end: optional cudaEvent_t (as void*) recorded on the stream
 *   immediately before and after the k_wilson launch. */
typedef struct wl_eval_options {
    size_t struct_size;          /* sizeof(wl_eval_options): set by wl_eval_options_default */
    int quadrature_order;
    int seeded;
    uint64_t seed;
    int64_t loop_begin;
    int shuffle_groups;
    int staging;
    uint64_t shuffle_seed;
    int64_t ensemble_loops;
    void* event_wilson_begin;
    void* event_wilson_end;
} wl_eval_options;

/* Fills *opt with the defaults (= plain wl_eval).  NULL is ignored. */
void wl_eval_options_default(wl_eval_options* opt);

/* wl_eval with options (opt == NULL: exactly wl_eval; the options are those above: eq. (24), PAPER.md:152-168;
 * PAPER.md:576).  Workspace: wl_eval_opt_workspace_bytes
 * (0 on invalid sizes or options).  Errors as wl_eval; an unknown quadrature order, a struct_size
 * that is not sizeof(wl_eval_options), seeded with a bad n_ppl -> WL_ERR_INVALID_ARG. */
size_t wl_eval_opt_workspace_bytes(int64_t n_loops, int n_ppl, int n_T, int n_rho, int n_groups,
                                   wl_dtype compute, const wl_eval_options* opt);
wl_status wl_eval_opt(const wl_field* field,
                      const void* d_loops, wl_dtype loop_dtype, int64_t n_loops, int n_ppl,
                      const double* d_T, int n_T,
                      const double* d_rho_cm, const double* d_phi_cm, int n_rho,
                      int n_groups, wl_dtype compute,
                      double* d_W_mean, double* d_group_sums,
                      void* d_workspace, size_t workspace_bytes, void* stream,
                      const wl_eval_options* opt);

/* wl_eval without an ensemble buffer: loops [loop_begin, loop_begin + n_loops) of the ensemble `seed`
 * are regenerated inside the kernel (= wl_eval_opt with seeded set).  `storage` is the
 * precision wl_loops_generate would have stored them in.  Workspace: wl_eval_workspace_bytes. */
wl_status wl_eval_seeded(const wl_field* field, uint64_t seed, int64_t loop_begin, wl_dtype storage,
                         int64_t n_loops, int n_ppl,
                         const double* d_T, int n_T,
                         const double* d_rho_cm, const double* d_phi_cm, int n_rho,
                         int n_groups, wl_dtype compute,
                         double* d_W_mean, double* d_group_sums,
                         void* d_workspace, size_t workspace_bytes, void* stream);

/* wl_eval_per_loop with options (quadrature_order, seeded; shuffle_groups is ignored): W, phase and spin of
 * eq. (18), (21)-(24), (31)-(33), for every loop separately. */
wl_status wl_eval_per_loop_opt(const wl_field* field,
                               const void* d_loops, wl_dtype loop_dtype, int64_t n_loops, int n_ppl,
                               const double* d_T, int n_T,
                               const double* d_rho_cm, const double* d_phi_cm, int n_rho,
                               wl_dtype compute,
                               double* d_W, double* d_phase, double* d_spin, void* stream,
                               const wl_eval_options* opt);

/* The group-membership table of shuffle_groups (Sec. IV.B.3; reading A17): d_perm[t][i] = pi_t(i) (int32, [n_T][n_loops]).
 * pi_t is a keyed bijection of [0, n_loops): a balanced Feistel network of 6 rounds on 2b bits (b the
 * smallest integer with 4^b >= n_loops) whose round function is word 0 of Philox4x32-10 with counter
 * (R, round, t, 0x5348464C) and key (seed_lo, seed_hi), applied again while the image is >= n_loops
 * (cycle walking).  1 <= n_loops < 2^31, n_T >= 1. */
wl_status wl_group_permutation(uint64_t shuffle_seed, int64_t n_loops, int n_T, int32_t* d_perm, void* stream);

/* wl_eval with two optional CUDA events (cudaEvent_t passed as void*, NULL = none)
 * recorded on `stream` immediately before and after the k_wilson launch, so that a
 * benchmark can time the dominant kernel alone inside the step (SURVEY.md section 8(d):
 * a2+a3 are > 99.9 % of the work).  Everything else is exactly wl_eval. */
wl_status wl_eval_instrumented(const wl_field* field,
                  const void* d_loops, wl_dtype loop_dtype, int64_t n_loops, int n_ppl,
                  const double* d_T, int n_T,
                  const double* d_rho_cm, const double* d_phi_cm, int n_rho,
                  int n_groups, wl_dtype compute,
                  double* d_W_mean, double* d_group_sums,
                  void* d_workspace, size_t workspace_bytes, void* stream,
                  void* event_wilson_begin, void* event_wilson_end);

/* Same kernels, but the per-loop values W, phase, spin of eq. (18), (21)-(24), (31)-(33), PAPER.md:121-185,
 * are written instead of reduced (for parity triage; not part of the timed path):  d_W, d_phase, d_spin are each
 * [n_loops][n_T][n_rho] FP64; d_phase / d_spin may be NULL.  No workspace. */
wl_status wl_eval_per_loop(const wl_field* field,
                           const void* d_loops, wl_dtype loop_dtype, int64_t n_loops, int n_ppl,
                           const double* d_T, int n_T,
                           const double* d_rho_cm, const double* d_phi_cm, int n_rho,
                           wl_dtype compute,
                           double* d_W, double* d_phase, double* d_spin, void* stream);

/* Discretisation estimate, Sec. IV.A, eq. (48)-(52), PAPER.md:269-304 (reading A15).
 * Every N-point loop is divided into three interleaved sub-worldlines, each closed on itself:
 * "circle" = points 0, 2, 4, ... (N/2 points), "box" = 1, 5, 9, ..., "triangle" = 3, 7, 11, ...
 * (N/4 points each).  With I the worldline integral (phase) of a sub-worldline,
 *   level 0 (N/4): W = cos(I_tri/2 + I_box/2)                 eq. (48)
 *   level 1 (N/2): W = cos(I_circ)                            eq. (49)
 *   level 2 (N)  : W = cos(I_circ/2 + I_box/4 + I_tri/4)      eq. (50)
 * times, for a fermion field, cosh of the sub-worldlines' spin integrals combined with the same weights.
 * Writes d_group_sums3[3][n_groups][n_T][n_rho] (levels N/4, N/2, N), in the fixed order of wl_eval.
 * n_ppl must be a multiple of 4 (else WL_ERR_INVALID_ARG).  Other arguments and errors as wl_eval;
 * the workspace size is wl_eval_discretization_workspace_bytes (0 on invalid sizes). */
size_t wl_eval_discretization_workspace_bytes(int64_t n_loops, int n_ppl, int n_T, int n_rho, int n_groups,
                                              wl_dtype compute);
wl_status wl_eval_discretization(const wl_field* field,
                                 const void* d_loops, wl_dtype loop_dtype, int64_t n_loops, int n_ppl,
                                 const double* d_T, int n_T,
                                 const double* d_rho_cm, const double* d_phi_cm, int n_rho,
                                 int n_groups, wl_dtype compute, double* d_group_sums3,
                                 void* d_workspace, size_t workspace_bytes, void* stream);

/* eq. (51)-(52), element-wise on d_levels3[3][n] (levels N/4, N/2, N: means or group sums):
 *   d_W_inf[k] = 8/3 W_N - 2 W_{N/2} + 1/3 W_{N/4},   d_delta[k] = |W_N - W_inf|  (d_delta may be NULL). */
wl_status wl_extrapolate(const double* d_levels3, int64_t n, double* d_W_inf, double* d_delta, void* stream);

/* Effective-action integrals (eq. (12), (44)-(47), (70); DESIGN.md
 * reading A16), done separately for every group of worldlines so that the error of the result is the
 * standard error of the group values.
 *
 * wl_proper_time_nodes (host only): the n_T (even) proper times at which <W> must be evaluated, the
 * Simpson nodes of x = 1/(1 + T/Tmax) on [0, x_a], x_a = 1/(1 + a/Tmax):
 *   h_T[j] = Tmax (1/x_j - 1),  x_j = x_a (n_T - j)/n_T,  j = 0..n_T-1   (h_T[0] = a, increasing).
 *
 * wl_action_density: from d_group_sums[G][n_T][n_rho] (wl_eval at those nodes),
 *   d_density[g][r] = int_0^a (small-T expansion eq. (44), or (45) for a scalar field)   [eq. (47)]
 *                   + Simpson int_a^inf dT e^{-m2 T}/T^3 [ <W>_g - 1 - (eB(rho_r) T)^2/3 ]  [eq. (12), (70)]
 *   (scalar field: [ <W>_g - 1 + (eB T)^2/6 ]), <W>_g = S_g G/n_loops, eB(rho) from the field profile.
 *   m2 = m^2 >= 0, a > 0, Tmax > 0, n_T even >= 2, n_loops % G == 0; else WL_ERR_INVALID_ARG.
 *   wl_jackknife_finalize(d_density, G, G, 1, n_rho, ...) then gives its mean and error over the groups.
 *
 * wl_action_radial: d_action[g] = (1/4 pi) int rho d_density[g](rho) d rho by Simpson's rule on the uniform
 *   grid d_rho_cm (n_rho odd >= 3, else WL_ERR_INVALID_ARG): Gamma/(T L_z) of eq. (12) per group. */
wl_status wl_proper_time_nodes(double a, double Tmax, int n_T, double* h_T);
wl_status wl_action_density(const wl_field* field, const double* d_group_sums, int n_groups, int64_t n_loops,
                            const double* d_T, int n_T, const double* d_rho_cm, int n_rho,
                            double m2, double a, double Tmax, double* d_density, void* stream);
wl_status wl_action_radial(const double* d_density, int n_groups, const double* d_rho_cm, int n_rho,
                           double* d_action, void* stream);

/* Jackknife finalise, eq. (60)-(63).  From d_group_sums[G][n_T][n_rho]:
 *   d_mean[t][r] = (sum_g S_g)/n_loops,
 *   d_err[t][r]  = sqrt(sum_g (S_g G/n_loops - mean)^2 / (G (G-1))),
 *   d_delete_one[g][t][r] = (sum_g' S_g' - S_g)/(n_loops - n_loops/G)   (NULL = skip).
 * n_groups >= 2 and n_loops % n_groups == 0, else WL_ERR_INVALID_ARG. */
wl_status wl_jackknife_finalize(const double* d_group_sums, int n_groups, int64_t n_loops,
                                int n_T, int n_rho,
                                double* d_mean, double* d_err, double* d_delete_one, void* stream);

/* End-to-end convenience call on HOST buffers (the whole path of eq. (8)-(63), in one
 * call): allocates device memory, copies
 * h_loops / grids to the device, runs wl_eval + wl_jackknife_finalize on an
 * internal stream (the copy of all but the first few jackknife groups overlaps the
 * evaluation of those; same bits as one wl_eval), copies h_W_mean[n_T][n_rho], h_err[n_T][n_rho]
 * and h_group_sums[G][n_T][n_rho] back, returns the device memory to the library's pool (see
 * wl_eval_host_trim) and returns after everything has completed.  h_phi_cm, h_err and h_group_sums may be NULL.
 * This is the only call that allocates, copies and synchronises.  Calls on the same device are serialised
 * (they share two internal streams); threads driving different devices run concurrently.
 * A failed device allocation gives WL_ERR_NOMEM. */
wl_status wl_eval_host(const wl_field* field,
                       const void* h_loops, wl_dtype loop_dtype, int64_t n_loops, int n_ppl,
                       const double* h_T, int n_T,
                       const double* h_rho_cm, const double* h_phi_cm, int n_rho,
                       int n_groups, wl_dtype compute,
                       double* h_W_mean, double* h_err, double* h_group_sums);

/* wl_eval_host takes its device memory from a private stream-ordered pool that keeps it between
 * calls; this returns the pool's unused memory to the device.  WL_OK if there is nothing to release. */
wl_status wl_eval_host_trim(void);

/* Measurement helper ("rooflines"; not part of the method): enqueues on `stream` one kernel
 * (4 CTAs of 256 threads per SM) that issues nothing but `iters` x 128 independent instructions per thread on ONE
 * pipe: pipe 0 = scalar FP32 FMA (the FP32 non-tensor issue roofline), 1 = MUFU.EX2 (the special-function pipe that
 * binds the FP32 sech^2 kernel), 2 = FP64 FMA.  *lane_ops (nullable) receives the number of thread-level instructions
 * the launch executes and *n_sms (nullable) the SM count, so that the caller, timing the launch with its own events,
 * gets lanes per clock and SM = lane_ops / (seconds x SM clock x n_sms).  d_sink: >= 4 bytes of device memory, not
 * written in practice.  1 <= iters <= 2^32; else, or for an unknown pipe or a NULL d_sink, WL_ERR_INVALID_ARG. */
wl_status wl_pipe_probe(int pipe, int64_t iters, float* d_sink, void* stream, int64_t* lane_ops, int* n_sms);

/* Number of kernels wl_eval enqueues for these sizes (for launch accounting). */
int wl_eval_launch_count(int64_t n_loops, int n_ppl, int n_T, int n_rho, int n_groups,
                         wl_dtype compute);

/* Static string for a status code (never NULL); the paper's "check the code, print the string". */
const char* wl_status_string(wl_status status);

/* "major.minor" of this ABI. */
const char* wl_version(void);

#ifdef __cplusplus
}
#endif
#endif /* WL_H */
