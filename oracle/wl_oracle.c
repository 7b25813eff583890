/*
 * wl_oracle.c -- FP64 CPU oracle for the worldline-numerics hot path.
 *
 * TEST INFRASTRUCTURE, NOT PRODUCT.  Only tests/, __graft_entry__.smoke() and
 * bench.py's cpu_baseline / --impl reference legs may build, load or call this
 * file.  It shares no code with paper_1407_7486_b200/csrc (the CUDA path) and
 * never receives a value computed by it.
 *
 * What it is: the definition of the estimator, written out in the order and
 * notation of the paper (arXiv:1407.7486, /root/reference/PAPER.md), in double
 * precision, with no blocking, fusion or reordering:
 *
 *   x_i   = x_cm + sqrt(T) y_i                          eq. (8),
 *   phase = sum_i  g(|m_i|) (m_i x d_i)                  eq. (21)-(24)
 *           m_i = (x_i + x_{i+1})/2,  d_i = x_{i+1} - x_i, i+1 taken mod N,
 *           g(rho) = e A_phi(rho)/rho = e Phi(rho)/(2 pi rho^2)   (one-point
 *           midpoint rule for the t-integral of eq. (24); reading A2)
 *   spin  = (T/N) sum_i e B(|x_i|)                       eq. (31)-(33)
 *   W     = cos(phase) cosh(spin)                        eq. (18)
 *   S_g   = sum of W over loops [g N_l/G, (g+1) N_l/G)   eq. (60)
 *   <W>   = (sum_g S_g)/N_l                              eq. (61)-(62)
 *   err   = sqrt(sum_g (<W>_g - <W>)^2 / (G (G-1)))      eq. (63)
 *
 * plus the unit-loop generator (d-loops, steps (1)-(5), eq. (10)-(11),
 * PAPER.md:65-81) driven by Philox4x32-10 (reading A11).
 *
 * Also: the paper's own flux-tube profile f_lambda = rho^2/(lambda^2+rho^2)
 * (eq. (68)) and the scalar-QED output W = cos(phase), pinned
 * in tests/test_oracle_fluxtube_scalar.py.
 *
 * Also (NEXT-4): the Q-point Gauss-Legendre rule for the t-integral of eq. (24) (wlo_loop_phase_spin_q,
 * pinned in tests/test_oracle_quadrature.py) and shuffled group assignment per proper time (wlo_shuffle_index,
 * wlo_regroup_shuffled; pinned in tests/test_oracle_shuffle.py).
 *
 * Pins (tests/test_oracle_*.py, all -m "not gpu"): zero field, uniform-field
 * shoelace area, finite-N uniform closed form, Stokes flux of the sech^2
 * profile by independent quadrature, mpmath evaluation of the profile,
 * lambda->infinity limit, rotation/relabelling invariances, 4-point brute
 * force, sampler moments and a Fourier-mode twin, Philox known answers.
 * No function here is "parity unpinned".
 *
 * OpenMP is used only to run independent loops on several cores; every sum is
 * taken serially in index order.
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define WLO_PROFILE_UNIFORM 0
#define WLO_PROFILE_SECH2 1
#define WLO_PROFILE_FLUXTUBE 2   /* f_lambda(rho^2) = rho^2/(lambda^2+rho^2), eq. (68) */

/* ------------------------------------------------------------------------- */
/* Field profiles.  e is folded into the field strength: only eB, eB0 enter.  */
/* ------------------------------------------------------------------------- */

/* h(u) = [u tanh u - ln cosh u]/u^2, so that for B = B0 sech^2(rho/lambda),
 * Phi(rho) = 2 pi B0 [lambda rho tanh(rho/lambda) - lambda^2 ln cosh(rho/lambda)]
 * (BASELINE.json config 1) gives g = e Phi/(2 pi rho^2) = eB0 h(rho/lambda).
 * u < 0.1: Maclaurin series (next term 3.3e-3 u^12 < 4e-15);
 * else the cancellation-free form with E = exp(-2u) (never calls cosh).      */
static double sech2_h(double u)
{
    if (u < 0.1) {
        double w = u * u;
        return 0.5 + w * (-1.0 / 4.0 + w * (1.0 / 9.0 + w * (-17.0 / 360.0
                 + w * (31.0 / 1575.0 + w * (-691.0 / 85050.0)))));
    }
    double E = exp(-2.0 * u);
    double P = M_LN2 - log1p(E) - 2.0 * u * E / (1.0 + E);
    return P / (u * u);
}

/* sech^2(u) = 4E/(1+E)^2, E = exp(-2u). */
static double sech2_b(double u)
{
    double E = exp(-2.0 * u);
    return 4.0 * E / ((1.0 + E) * (1.0 + E));
}

/* g(rho) = e A_phi(rho)/rho   (eq. (14), (23)) */
double wlo_field_g(int profile, const double *params, double rho)
{
    if (profile == WLO_PROFILE_UNIFORM)
        return 0.5 * params[0];                 /* A = (B/2)(-y, x) */
    if (profile == WLO_PROFILE_FLUXTUBE)
        /* eq. (14) with eq. (68): e A_phi/rho = (eF/2pi) f_lambda/rho^2 = script-F/(lambda^2+rho^2),
         * params = {script-F (eq. (17)), lambda} */
        return params[0] / (params[1] * params[1] + rho * rho);
    return params[0] * sech2_h(rho / params[1]);
}

/* b(rho) = e B_z(rho)         (eq. (13), (15)) */
double wlo_field_b(int profile, const double *params, double rho)
{
    if (profile == WLO_PROFILE_UNIFORM)
        return params[0];
    if (profile == WLO_PROFILE_FLUXTUBE) {
        /* eq. (15) with eq. (68): e B_z = (eF/2pi rho) d f_lambda/d rho = 2 script-F lambda^2/(lambda^2+rho^2)^2 */
        double l2 = params[1] * params[1];
        double D = l2 + rho * rho;
        return 2.0 * params[0] * l2 / (D * D);
    }
    return params[0] * sech2_b(rho / params[1]);
}

/* ------------------------------------------------------------------------- */
/* One Wilson loop at one (T, x_cm).  y: [N][2] unit loop.                    */
/* ------------------------------------------------------------------------- */
void wlo_loop_phase_spin(int profile, const double *params,
                         const double *y, int N, double T, double cx, double cy,
                         double *phase_out, double *spin_out)
{
    double s = sqrt(T);
    double phase = 0.0, spin = 0.0;
    for (int i = 0; i < N; ++i) {
        int j = (i + 1) % N;
        double xi_x = cx + s * y[2 * i], xi_y = cy + s * y[2 * i + 1];
        double xj_x = cx + s * y[2 * j], xj_y = cy + s * y[2 * j + 1];
        double m_x = 0.5 * (xi_x + xj_x), m_y = 0.5 * (xi_y + xj_y);
        double d_x = xj_x - xi_x, d_y = xj_y - xi_y;
        phase += wlo_field_g(profile, params, sqrt(m_x * m_x + m_y * m_y)) * (m_x * d_y - m_y * d_x);
        spin += wlo_field_b(profile, params, sqrt(xi_x * xi_x + xi_y * xi_y));
    }
    *phase_out = phase;
    *spin_out = T / (double)N * spin;
}

/* ------------------------------------------------------------------------- */
/* Whole ensemble on a (T, rho_cm[, phi_cm]) grid.                            */
/*   loops      [n_loops][N][2]                                               */
/*   W_mean     [n_T][n_rho]                                                  */
/*   group_sums [G][n_T][n_rho]                                               */
/*   W_loop, phase_loop, spin_loop: nullable, [n_loops][n_T][n_rho]           */
/* Returns 0, or -1 on a bad argument.                                        */
/* ------------------------------------------------------------------------- */
/* scalar != 0: scalar QED, W = cos(phase) only (the paper's Wsscal;         */
/* exact uniform-field average eq. (43)); scalar == 0: fermion, eq. (18).               */
int wlo_eval_particle(int profile, const double *params, int scalar,
             const double *loops, int64_t n_loops, int N,
             const double *T, int n_T,
             const double *rho_cm, const double *phi_cm, int n_rho,
             int n_groups,
             double *W_mean, double *group_sums,
             double *W_loop, double *phase_loop, double *spin_loop);

int wlo_eval(int profile, const double *params,
             const double *loops, int64_t n_loops, int N,
             const double *T, int n_T,
             const double *rho_cm, const double *phi_cm, int n_rho,
             int n_groups,
             double *W_mean, double *group_sums,
             double *W_loop, double *phase_loop, double *spin_loop)
{
    return wlo_eval_particle(profile, params, 0, loops, n_loops, N, T, n_T, rho_cm, phi_cm, n_rho, n_groups,
                             W_mean, group_sums, W_loop, phase_loop, spin_loop);
}

int wlo_eval_particle(int profile, const double *params, int scalar,
             const double *loops, int64_t n_loops, int N,
             const double *T, int n_T,
             const double *rho_cm, const double *phi_cm, int n_rho,
             int n_groups,
             double *W_mean, double *group_sums,
             double *W_loop, double *phase_loop, double *spin_loop)
{
    if (n_loops <= 0 || N < 1 || n_T < 1 || n_rho < 1 || n_groups < 1) return -1;
    if (n_loops % n_groups != 0) return -1;         /* equal groups */
    const int64_t n_grid = (int64_t)n_T * n_rho;
    const int64_t per_group = n_loops / n_groups;

    double *W = W_loop ? W_loop : (double *)malloc(sizeof(double) * n_loops * n_grid);
    if (!W) return -1;

#pragma omp parallel for schedule(dynamic, 1)
    for (int64_t l = 0; l < n_loops; ++l) {
        const double *y = loops + l * (int64_t)N * 2;
        for (int t = 0; t < n_T; ++t)
            for (int r = 0; r < n_rho; ++r) {
                double ph = phi_cm ? phi_cm[r] : 0.0;
                double cx = rho_cm[r] * cos(ph), cy = rho_cm[r] * sin(ph);
                double phase, spin;
                wlo_loop_phase_spin(profile, params, y, N, T[t], cx, cy, &phase, &spin);
                int64_t o = l * n_grid + (int64_t)t * n_rho + r;
                W[o] = scalar ? cos(phase) : cos(phase) * cosh(spin);
                if (phase_loop) phase_loop[o] = phase;
                if (spin_loop) spin_loop[o] = spin;
            }
    }

    for (int64_t k = 0; k < n_grid; ++k) {
        double total = 0.0;
        for (int g = 0; g < n_groups; ++g) {
            double S = 0.0;
            for (int64_t l = g * per_group; l < (g + 1) * per_group; ++l) S += W[l * n_grid + k];
            group_sums[(int64_t)g * n_grid + k] = S;
            total += S;
        }
        W_mean[k] = total / (double)n_loops;
    }
    if (!W_loop) free(W);
    return 0;
}

/* ------------------------------------------------------------------------- */
/* Higher-order quadrature of the t-integral of eq. (24) (SURVEY.md 8(f)      */
/* NEXT-4; "in general, we wish to compute these integrals  */
/* numerically ... gauge invariance ... can be preserved to any numerical     */
/* precision that's desired").  Segment i contributes, eq. (24),              */
/*   (x^i y^{i+1} - y^i x^{i+1}) int_0^1 dt g(rho_i(t)),                      */
/*   rho_i^2(t) = A_i + 2 B_i t + C_i t^2,                    eq. (25)         */
/*   A_i = |x^i|^2, B_i = x^i . (x^{i+1} - x^i), C_i = |x^{i+1} - x^i|^2       */
/*                                                            eq. (26)-(28)    */
/* with g(rho) = F f_lambda(rho^2)/rho^2 = e A_phi/rho (eq. (23)), and the     */
/* t-integral is taken by the Q-point Gauss-Legendre rule on [0, 1]:           */
/*   Q = 1: t = 1/2 (the midpoint rule of wlo_loop_phase_spin),                */
/*   Q = 2: t = 1/2 -+ 1/(2 sqrt 3),            weights 1/2, 1/2,              */
/*   Q = 3: t = 1/2 -+ sqrt(3/5)/2, 1/2,        weights 5/18, 4/9, 5/18.       */
/* The spin factor is the point-sampled sum of wlo_loop_phase_spin (north_star).*/
/* Returns 0, or -1 if Q is not 1, 2 or 3.                                     */
/* ------------------------------------------------------------------------- */
int wlo_gauss_legendre_01(int Q, double *t, double *w)
{
    if (Q == 1) { t[0] = 0.5; w[0] = 1.0; return 0; }
    if (Q == 2) {
        double d = 0.5 / sqrt(3.0);
        t[0] = 0.5 - d; t[1] = 0.5 + d; w[0] = 0.5; w[1] = 0.5;
        return 0;
    }
    if (Q == 3) {
        double d = 0.5 * sqrt(3.0 / 5.0);
        t[0] = 0.5 - d; t[1] = 0.5; t[2] = 0.5 + d;
        w[0] = 5.0 / 18.0; w[1] = 4.0 / 9.0; w[2] = 5.0 / 18.0;
        return 0;
    }
    return -1;
}

int wlo_loop_phase_spin_q(int profile, const double *params,
                          const double *y, int N, double T, double cx, double cy, int Q,
                          double *phase_out, double *spin_out)
{
    double tq[3], wq[3];
    if (wlo_gauss_legendre_01(Q, tq, wq) != 0) return -1;
    double s = sqrt(T);
    double phase = 0.0, spin = 0.0;
    for (int i = 0; i < N; ++i) {
        int j = (i + 1) % N;
        double xi = cx + s * y[2 * i], yi = cy + s * y[2 * i + 1];
        double xj = cx + s * y[2 * j], yj = cy + s * y[2 * j + 1];
        double A = xi * xi + yi * yi;                                   /* eq. (26) */
        double B = xi * (xj - xi) + yi * (yj - yi);                     /* eq. (27) */
        double Cc = (xj - xi) * (xj - xi) + (yj - yi) * (yj - yi);      /* eq. (28) */
        double integral = 0.0;
        for (int q = 0; q < Q; ++q) {
            double rho2 = A + 2.0 * B * tq[q] + Cc * tq[q] * tq[q];     /* eq. (25) */
            if (rho2 < 0.0) rho2 = 0.0;                                 /* rounding, segment through the axis */
            integral += wq[q] * wlo_field_g(profile, params, sqrt(rho2));
        }
        phase += (xi * yj - yi * xj) * integral;                        /* eq. (24) */
        spin += wlo_field_b(profile, params, sqrt(xi * xi + yi * yi));
    }
    *phase_out = phase;
    *spin_out = T / (double)N * spin;
    return 0;
}

/* wlo_eval_particle with the Q-point rule for eq. (24); same outputs, same group order. */
int wlo_eval_quadrature(int profile, const double *params, int scalar, int Q,
             const double *loops, int64_t n_loops, int N,
             const double *T, int n_T,
             const double *rho_cm, const double *phi_cm, int n_rho,
             int n_groups,
             double *W_mean, double *group_sums,
             double *W_loop, double *phase_loop, double *spin_loop)
{
    if (n_loops <= 0 || N < 1 || n_T < 1 || n_rho < 1 || n_groups < 1) return -1;
    if (n_loops % n_groups != 0 || Q < 1 || Q > 3) return -1;
    const int64_t n_grid = (int64_t)n_T * n_rho;
    const int64_t per_group = n_loops / n_groups;
    double *W = W_loop ? W_loop : (double *)malloc(sizeof(double) * n_loops * n_grid);
    if (!W) return -1;

#pragma omp parallel for schedule(dynamic, 1)
    for (int64_t l = 0; l < n_loops; ++l) {
        const double *y = loops + l * (int64_t)N * 2;
        for (int t = 0; t < n_T; ++t)
            for (int r = 0; r < n_rho; ++r) {
                double ph = phi_cm ? phi_cm[r] : 0.0;
                double cx = rho_cm[r] * cos(ph), cy = rho_cm[r] * sin(ph);
                double phase, spin;
                wlo_loop_phase_spin_q(profile, params, y, N, T[t], cx, cy, Q, &phase, &spin);
                int64_t o = l * n_grid + (int64_t)t * n_rho + r;
                W[o] = scalar ? cos(phase) : cos(phase) * cosh(spin);
                if (phase_loop) phase_loop[o] = phase;
                if (spin_loop) spin_loop[o] = spin;
            }
    }
    for (int64_t k = 0; k < n_grid; ++k) {
        double total = 0.0;
        for (int g = 0; g < n_groups; ++g) {
            double S = 0.0;
            for (int64_t l = g * per_group; l < (g + 1) * per_group; ++l) S += W[l * n_grid + k];
            group_sums[(int64_t)g * n_grid + k] = S;
            total += S;
        }
        W_mean[k] = total / (double)n_loops;
    }
    if (!W_loop) free(W);
    return 0;
}

/* ------------------------------------------------------------------------- */
/* Discretisation estimate, Sec. IV.A, eq. (48)-(52).       */
/* Each N-point worldline is divided into three interleaved sub-worldlines    */
/* (Fig. 2): "circle" = every other point (N/2 points: 0, 2, 4, ...), and the */
/* remaining points split alternately into "box" (1, 5, 9, ...) and           */
/* "triangle" (3, 7, 11, ...), N/4 points each; every sub-worldline is closed */
/* on itself and evaluated as a loop of its own (same T, same x_cm;           */
/* a sub-loop of a d-loop has the prescribed distribution).     */
/* With I = the worldline integral of a sub-worldline:                        */
/*   level 0:  <W>_{N/4} = < e^{i I_tri/2} e^{i I_box/2} >              (48)  */
/*   level 1:  <W>_{N/2} = < e^{i I_circ} >                             (49)  */
/*   level 2:  <W>_{N}   = < e^{i I_circ/2} e^{i I_box/4} e^{i I_tri/4} > (50) */
/* Real part only (reading A5); for a fermion loop the spin integrals of the  */
/* sub-worldlines are combined with the same weights (reading A15). */
/*   group_sums3 [3][G][n_T][n_rho]; W3_loop nullable [3][n_loops][n_T][n_rho] */
/* N must be a multiple of 4.  Returns 0 or -1.                               */
/* ------------------------------------------------------------------------- */
int wlo_eval_discretization(int profile, const double *params, int scalar,
                            const double *loops, int64_t n_loops, int N,
                            const double *T, int n_T,
                            const double *rho_cm, const double *phi_cm, int n_rho,
                            int n_groups, double *group_sums3, double *W3_loop)
{
    if (n_loops <= 0 || N < 4 || N % 4 != 0 || n_T < 1 || n_rho < 1 || n_groups < 1) return -1;
    if (n_loops % n_groups != 0) return -1;
    const int64_t n_grid = (int64_t)n_T * n_rho;
    const int64_t per_group = n_loops / n_groups;
    double *W = W3_loop ? W3_loop : (double *)malloc(sizeof(double) * 3 * n_loops * n_grid);
    if (!W) return -1;
    int fail = 0;

#pragma omp parallel for schedule(dynamic, 1)
    for (int64_t l = 0; l < n_loops; ++l) {
        const double *y = loops + l * (int64_t)N * 2;
        double *circ = (double *)malloc(sizeof(double) * N * 2);   /* N/2 + N/4 + N/4 points */
        if (!circ) { fail = 1; continue; }
        double *box = circ + N, *tri = box + N / 2;
        for (int q = 0; q < N / 2; ++q) { circ[2 * q] = y[2 * (2 * q)]; circ[2 * q + 1] = y[2 * (2 * q) + 1]; }
        for (int q = 0; q < N / 4; ++q) {
            box[2 * q] = y[2 * (4 * q + 1)]; box[2 * q + 1] = y[2 * (4 * q + 1) + 1];
            tri[2 * q] = y[2 * (4 * q + 3)]; tri[2 * q + 1] = y[2 * (4 * q + 3) + 1];
        }
        for (int t = 0; t < n_T; ++t)
            for (int r = 0; r < n_rho; ++r) {
                double ph = phi_cm ? phi_cm[r] : 0.0;
                double cx = rho_cm[r] * cos(ph), cy = rho_cm[r] * sin(ph);
                double Ic, Sc, Ib, Sb, It, St;
                wlo_loop_phase_spin(profile, params, circ, N / 2, T[t], cx, cy, &Ic, &Sc);
                wlo_loop_phase_spin(profile, params, box, N / 4, T[t], cx, cy, &Ib, &Sb);
                wlo_loop_phase_spin(profile, params, tri, N / 4, T[t], cx, cy, &It, &St);
                double phase[3] = { 0.5 * It + 0.5 * Ib, Ic, 0.5 * Ic + 0.25 * Ib + 0.25 * It };
                double spin[3] = { 0.5 * St + 0.5 * Sb, Sc, 0.5 * Sc + 0.25 * Sb + 0.25 * St };
                for (int lev = 0; lev < 3; ++lev)
                    W[((int64_t)lev * n_loops + l) * n_grid + (int64_t)t * n_rho + r] =
                        scalar ? cos(phase[lev]) : cos(phase[lev]) * cosh(spin[lev]);
            }
        free(circ);
    }
    if (!fail)
        for (int lev = 0; lev < 3; ++lev)
            for (int64_t k = 0; k < n_grid; ++k)
                for (int g = 0; g < n_groups; ++g) {
                    double S = 0.0;
                    for (int64_t l = g * per_group; l < (g + 1) * per_group; ++l)
                        S += W[((int64_t)lev * n_loops + l) * n_grid + k];
                    group_sums3[((int64_t)lev * n_groups + g) * n_grid + k] = S;
                }
    if (!W3_loop) free(W);
    return fail ? -1 : 0;
}

/* eq. (51)-(52): parabola through the three levels in 1/N.  */
void wlo_extrapolate(const double *lev3, int64_t n, double *W_inf, double *delta)
{
    for (int64_t k = 0; k < n; ++k) {
        double w4 = lev3[k], w2 = lev3[n + k], w1 = lev3[2 * n + k];
        W_inf[k] = 8.0 / 3.0 * w1 - 2.0 * w2 + 1.0 / 3.0 * w4;
        if (delta) delta[k] = fabs(w1 - W_inf[k]);
    }
}

/* ------------------------------------------------------------------------- */
/* Effective-action integrals, eq. (12), (44)-(47), (70),     */
/* 234-255, 417, 472, 495 (reading A16).                            */
/*   density(rho) = int_0^inf dT e^{-m^2 T}/T^3 [ <W> - 1 - (eB_cm T)^2/3 ]    */
/*   (scalar QED: [ <W> - 1 + (eB_cm T)^2/6 ], eq. (45))                       */
/* = int_0^a of the small-T expansion (44)/(45), integrated term by term       */
/* (eq. (47)), + int_a^inf by Simpson's rule in x = 1/(1 + T/Tmax)             */
/* on n equal intervals of [0, x_a], x_a = 1/(1 + a/Tmax); the  */
/* node x = 0 (T = inf) contributes nothing.  Done separately for every group  */
/* of worldlines, so the error is the SEM of the group values.  */
/* ------------------------------------------------------------------------- */

/* Proper-time nodes T_j, j = 0..n-1, x_j = x_a (n - j)/n, T_j = Tmax (1/x_j - 1): T_0 = a, increasing. */
int wlo_proper_time_nodes(double a, double Tmax, int n, double *T)
{
    if (!(a > 0.0) || !(Tmax > 0.0) || n < 2 || n % 2 != 0) return -1;
    double xa = 1.0 / (1.0 + a / Tmax);
    for (int j = 0; j < n; ++j) {
        double x = xa * (double)(n - j) / (double)n;
        T[j] = Tmax * (1.0 / x - 1.0);
    }
    T[0] = a;
    return 0;
}

/* int_0^a of eq. (44) (fermion) or eq. (45) (scalar), b = eB(r_cm). */
double wlo_small_T_integral(double b, double m2, double a, int scalar)
{
    double b4 = b * b * b * b, b6 = b4 * b * b;
    double c1, c2, c3, c4;
    if (!scalar) {                                  /* eq. (44) */
        c1 = -b4 / 45.0;
        c2 = b4 * m2 / 45.0;
        c3 = 2.0 * b6 / 945.0 - b4 * m2 * m2 / 90.0;
        c4 = (7.0 * b4 * m2 * m2 * m2 - 4.0 * b6 * m2) / 1890.0;
    } else {                                        /* eq. (45) */
        c1 = 7.0 * b4 / 360.0;
        c2 = -7.0 * b4 * m2 / 360.0;
        c3 = (147.0 * b4 * m2 * m2 - 31.0 * b6) / 15120.0;
        c4 = (31.0 * b6 * m2 - 49.0 * b4 * m2 * m2 * m2) / 15120.0;
    }
    return c1 * a * a / 2.0 + c2 * a * a * a / 3.0 + c3 * a * a * a * a / 4.0 + c4 * a * a * a * a * a / 5.0;
}

/* group_sums [G][n_T][n_rho] at the nodes of wlo_proper_time_nodes(a, Tmax, n_T); density [G][n_rho]. */
int wlo_action_density(int profile, const double *params, int scalar,
                       const double *group_sums, int n_groups, int64_t n_loops,
                       const double *T, int n_T, const double *rho_cm, int n_rho,
                       double m2, double a, double Tmax, double *density)
{
    if (n_groups < 1 || n_loops < 1 || n_loops % n_groups != 0 || n_T < 2 || n_T % 2 != 0 || n_rho < 1) return -1;
    if (!(a > 0.0) || !(Tmax > 0.0)) return -1;
    const double per_group = (double)(n_loops / n_groups);
    const double xa = 1.0 / (1.0 + a / Tmax);
    const double h = xa / (double)n_T;
    for (int g = 0; g < n_groups; ++g)
        for (int r = 0; r < n_rho; ++r) {
            double b = wlo_field_b(profile, params, rho_cm[r]);
            double simpson = 0.0;
            for (int j = 0; j < n_T; ++j) {
                int k = n_T - j;                                     /* Simpson node index, x_k = k h */
                double x = h * (double)k;
                double Tj = T[j];
                double W = group_sums[((int64_t)g * n_T + j) * n_rho + r] / per_group;     /* <W>_g, eq. (60) */
                double bT = b * Tj;
                double bracket = scalar ? W - 1.0 + bT * bT / 6.0 : W - 1.0 - bT * bT / 3.0;
                double I = exp(-m2 * Tj) / (Tj * Tj * Tj) * bracket;                       /* eq. (70) */
                double weight = (k == n_T) ? 1.0 : ((k % 2) ? 4.0 : 2.0);
                simpson += weight * I * Tmax / (x * x);                                    /* dT = Tmax dx/x^2 */
            }
            density[(int64_t)g * n_rho + r] = wlo_small_T_integral(b, m2, a, scalar) + simpson * h / 3.0;
        }
    return 0;
}

/* eq. (12): action[g] = (1/4 pi) int rho density_g(rho) d rho by Simpson on a uniform rho grid (n_rho odd). */
int wlo_action_radial(const double *density, int n_groups, const double *rho_cm, int n_rho, double *action)
{
    if (n_groups < 1 || n_rho < 3 || n_rho % 2 != 1) return -1;
    const double h = (rho_cm[n_rho - 1] - rho_cm[0]) / (double)(n_rho - 1);
    for (int g = 0; g < n_groups; ++g) {
        double s = 0.0;
        for (int r = 0; r < n_rho; ++r) {
            double weight = (r == 0 || r == n_rho - 1) ? 1.0 : ((r % 2) ? 4.0 : 2.0);
            s += weight * rho_cm[r] * density[(int64_t)g * n_rho + r];
        }
        action[g] = s * h / 3.0 / (4.0 * M_PI);
    }
    return 0;
}

/* ------------------------------------------------------------------------- */
/* Jackknife finalise, eq. (60)-(63); delete-one-group means (reading A7).    */
/*   mean, err [n_grid]; delete_one nullable [G][n_grid]                      */
/* ------------------------------------------------------------------------- */
int wlo_finalize(const double *group_sums, int n_groups, int64_t n_loops, int64_t n_grid,
                 double *mean, double *err, double *delete_one)
{
    if (n_groups < 2 || n_loops % n_groups != 0) return -1;
    const double G = (double)n_groups;
    const double per_group = (double)(n_loops / n_groups);
    for (int64_t k = 0; k < n_grid; ++k) {
        double total = 0.0;
        for (int g = 0; g < n_groups; ++g) total += group_sums[(int64_t)g * n_grid + k];
        double m = total / (double)n_loops;
        double ss = 0.0;
        for (int g = 0; g < n_groups; ++g) {
            double mg = group_sums[(int64_t)g * n_grid + k] / per_group;   /* eq. (60) */
            ss += (mg - m) * (mg - m);
            if (delete_one)
                delete_one[(int64_t)g * n_grid + k] =
                    (total - group_sums[(int64_t)g * n_grid + k]) / ((double)n_loops - per_group);
        }
        mean[k] = m;
        err[k] = sqrt(ss / (G * (G - 1.0)));                               /* eq. (63) */
    }
    return 0;
}

/* ------------------------------------------------------------------------- */
/* Philox4x32-10 (Salmon et al., SC'11), restated from the published          */
/* algorithm: 10 rounds of two 32x32->64 multiplies, key bumped by the Weyl   */
/* constants between rounds.                                                  */
/* ------------------------------------------------------------------------- */
void wlo_philox4x32_10(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4])
{
    uint32_t c0 = ctr[0], c1 = ctr[1], c2 = ctr[2], c3 = ctr[3];
    uint32_t k0 = key[0], k1 = key[1];
    for (int round = 0; round < 10; ++round) {
        uint64_t p0 = (uint64_t)0xD2511F53u * c0;
        uint64_t p1 = (uint64_t)0xCD9E8D57u * c2;
        uint32_t n0 = (uint32_t)(p1 >> 32) ^ c1 ^ k0;
        uint32_t n1 = (uint32_t)p1;
        uint32_t n2 = (uint32_t)(p0 >> 32) ^ c3 ^ k1;
        uint32_t n3 = (uint32_t)p0;
        c0 = n0; c1 = n1; c2 = n2; c3 = n3;
        k0 += 0x9E3779B9u; k1 += 0xBB67AE85u;
    }
    out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

/* Two standard normals for (seed, loop, point): counter = (point, loop_lo,
 * loop_hi, 0), key = (seed_lo, seed_hi); words (0,1) and (2,3) give two
 * 53-bit uniforms in (0,1]; Box-Muller in FP64.  (reading A11.)   */
void wlo_normal_pair(uint64_t seed, uint64_t loop, uint32_t point, double *nx, double *ny)
{
    uint32_t ctr[4] = { point, (uint32_t)loop, (uint32_t)(loop >> 32), 0u };
    uint32_t key[2] = { (uint32_t)seed, (uint32_t)(seed >> 32) };
    uint32_t w[4];
    wlo_philox4x32_10(ctr, key, w);
    uint64_t a = ((uint64_t)w[1] << 32) | w[0];
    uint64_t b = ((uint64_t)w[3] << 32) | w[2];
    double u1 = (double)((a >> 11) + 1) * 0x1.0p-53;
    double u2 = (double)((b >> 11) + 1) * 0x1.0p-53;
    double r = sqrt(-2.0 * log(u1));
    double th = 6.283185307179586476925286766559 * u2;
    *nx = r * cos(th);
    *ny = r * sin(th);
}

/* ------------------------------------------------------------------------- */
/* Shuffled group assignment (Sec. IV.B.3,             */
/* PAPER.md:411-417, Fig. 6 at PAPER.md:380): "randomize how worldlines are    */
/* assigned to groups between each evaluation of the integrand".  One          */
/* evaluation of the integrand = one proper time T_t, so every T index t gets  */
/* its own seeded permutation pi_t of the loops, and group g at that T is      */
/*   { pi_t(i) : g N_l/G <= i < (g+1) N_l/G },  summed in the order of i       */
/* (reading A17).  pi_t is a keyed bijection of [0, n_loops): a      */
/* balanced Feistel network of 6 rounds on 2b bits (b the smallest integer     */
/* with 4^b >= n_loops) whose round function is word 0 of Philox4x32-10 with   */
/* counter (R, round, t, 0x5348464C) and key (seed_lo, seed_hi), followed by   */
/* cycle walking (apply again while the image is >= n_loops).  A Feistel       */
/* network is a bijection of [0, 4^b) whatever its round function, and cycle   */
/* walking restricts a bijection to a bijection of the subset.                 */
/* ------------------------------------------------------------------------- */
int64_t wlo_shuffle_index(uint64_t seed, int t, int64_t n_loops, int64_t i)
{
    int b = 1;
    while (((int64_t)1 << (2 * b)) < n_loops) ++b;
    const uint32_t mask = (uint32_t)(((uint64_t)1 << b) - 1u);
    const uint32_t key[2] = { (uint32_t)seed, (uint32_t)(seed >> 32) };
    uint64_t x = (uint64_t)i;
    do {
        uint32_t L = (uint32_t)(x >> b), R = (uint32_t)(x & mask);
        for (uint32_t round = 0; round < 6; ++round) {
            uint32_t ctr[4] = { R, round, (uint32_t)t, 0x5348464Cu };
            uint32_t w[4];
            wlo_philox4x32_10(ctr, key, w);
            uint32_t nR = L ^ (w[0] & mask);
            L = R;
            R = nR;
        }
        x = ((uint64_t)L << b) | R;
    } while (x >= (uint64_t)n_loops);
    return (int64_t)x;
}

/* perm[t][i] = pi_t(i), [n_T][n_loops]. */
int wlo_group_permutation(uint64_t seed, int64_t n_loops, int n_T, int64_t *perm)
{
    if (n_loops < 1 || n_T < 1) return -1;
    for (int t = 0; t < n_T; ++t)
        for (int64_t i = 0; i < n_loops; ++i)
            perm[(int64_t)t * n_loops + i] = wlo_shuffle_index(seed, t, n_loops, i);
    return 0;
}

/* Group sums and mean from per-loop W [n_loops][n_T][n_rho] with the groups of table perm[n_T][n_loops]:
 * S_g[t][r] = sum_{i = g N_l/G}^{(g+1) N_l/G - 1} W[perm[t][i]][t][r]  (eq. (60) with shuffled membership),
 * <W>[t][r] = (sum_g S_g[t][r])/N_l  (eq. (61)-(62): unchanged by the grouping, up to rounding). */
int wlo_regroup_shuffled(const double *W_loop, int64_t n_loops, int n_T, int n_rho, int n_groups,
                         const int64_t *perm, double *group_sums, double *W_mean)
{
    if (n_loops < 1 || n_T < 1 || n_rho < 1 || n_groups < 1 || n_loops % n_groups != 0) return -1;
    const int64_t n_grid = (int64_t)n_T * n_rho;
    const int64_t per_group = n_loops / n_groups;
    for (int t = 0; t < n_T; ++t)
        for (int r = 0; r < n_rho; ++r) {
            int64_t k = (int64_t)t * n_rho + r;
            double total = 0.0;
            for (int g = 0; g < n_groups; ++g) {
                double S = 0.0;
                for (int64_t i = g * per_group; i < (g + 1) * per_group; ++i)
                    S += W_loop[perm[(int64_t)t * n_loops + i] * n_grid + k];
                group_sums[(int64_t)g * n_grid + k] = S;
                total += S;
            }
            W_mean[k] = total / (double)n_loops;
        }
    return 0;
}

/* d-loop generator.  Step (1): y_N = 0 (stored at index 0).
 * Step (2)-(3): level k = 1..log2 N adds the odd multiples of h = N/2^k,
 *   y_p = (y_{p-h} + y_{p+h})/2 + sigma_k n_p,  sigma_k^2 = 1/N_k = 2^-k per
 *   component (eq. (10): exp(-(y-y_N)^2) at k = 1; eq. (11) at k > 1).
 * Step (5): subtract the centre of mass.
 * Writes loops [loop_begin, loop_begin + n_loops) into out[n_loops][N][2].
 * N must be a power of two >= 2.  Returns 0 or -1.                           */
int wlo_generate_loops(uint64_t seed, int64_t loop_begin, int64_t n_loops, int N, double *out)
{
    if (N < 2 || (N & (N - 1)) != 0 || n_loops < 0) return -1;
    int log2N = 0;
    while ((1 << log2N) < N) ++log2N;
#pragma omp parallel for schedule(static)
    for (int64_t q = 0; q < n_loops; ++q) {
        double *y = out + q * (int64_t)N * 2;
        uint64_t loop = (uint64_t)(loop_begin + q);
        y[0] = 0.0; y[1] = 0.0;
        for (int k = 1; k <= log2N; ++k) {
            int h = N >> k;
            double sigma = ldexp((k & 1) ? M_SQRT1_2 : 1.0, -(k / 2));
            for (int p = h; p < N; p += 2 * h) {
                int lo = p - h, hi = (p + h) % N;
                double nx, ny;
                wlo_normal_pair(seed, loop, (uint32_t)p, &nx, &ny);
                y[2 * p] = 0.5 * (y[2 * lo] + y[2 * hi]) + sigma * nx;
                y[2 * p + 1] = 0.5 * (y[2 * lo + 1] + y[2 * hi + 1]) + sigma * ny;
            }
        }
        double mx = 0.0, my = 0.0;
        for (int i = 0; i < N; ++i) { mx += y[2 * i]; my += y[2 * i + 1]; }
        mx /= (double)N; my /= (double)N;
        for (int i = 0; i < N; ++i) { y[2 * i] -= mx; y[2 * i + 1] -= my; }
    }
    return 0;
}

int wlo_num_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}
