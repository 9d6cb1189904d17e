/*
 * bloch_ref.c -- CPU fp64 ORACLE for the spin-parallel Bloch solve of KomaMRI (arxiv 2301.02702).
 *
 * THIS IS TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only tests/, __graft_entry__.smoke() and bench.py's
 * cpu_baseline / --impl reference legs may call it.  It shares no code, header, table or constant
 * generator with the CUDA path under paper_2301_02702_b200/csrc/.
 *
 * It follows the paper step by step, in the paper's order and notation, with no blocking, fusion or
 * reordering:
 *   - effective field                      Eq (2)
 *   - first-order splitting, rotation then relaxation, every interval   Eq (3)-(4)
 *   - excitation regime: spinor (alpha, beta) Eq (6)-(8), applied by Eq (9)
 *   - precession regime: Mxy <- Mxy e^{i phi}, phi of Eq (8) with B1 = 0  Eq (10)
 *   - relaxation                            Eq (11)
 *   - trapezoidal rule on gradient vertices Eq (12)-(13) PAPER.md:173-180
 *   - piecewise-constant B1, refined to dt_rf_max
 *   - per-thread signal buffers added at the end
 * Readings of silent / garbled passages (G1..G18) are those of SURVEY.md 8(c), restated in DESIGN.md.
 *
 * Motion: bloch_ref_simulate_motion moves every spin as x(t) = x + v t
 * and takes the trapezoid of Eq (12)-(13) on Bz(t_n) = G(t_n) . x(t_n); dt_max adds the intermediate points.  Pins M1-M5:
 * tests/test_oracle_motion_pins.py (closed-form phase under constant G, bipolar velocity encoding, O(dt^2)
 * convergence on a ramp, regime consistency).
 * General motion ("motion field u(x, t)"; reading M2): bloch_ref_simulate_waveform moves every spin
 * as x(t) = x + a u(t), a per-spin amplitude vector, u(t) a shared piecewise-linear waveform given by vertices (held at
 * its end values outside them; the vertices join the time grid).  u(t) = t is the constant-velocity case.  Pins W1-W5
 * in the same test file (closed forms under constant G for sinusoidal and stop-and-go u, reduction to x + v t,
 * displacement-only phase, O(dt^2) convergence under a ramp).
 *
 * Pins (tests/test_oracle_pins.py): closed forms and invariants P1-P12 (the adiabatic
 * hyperbolic-secant profile P11, the frequency-offset slice shift P12), the count pin of reading G18 (an RF train late
 * in a long sequence keeps its nominal step count) and the grouped FISP pin; motion M1-M5 and W1-W5, coils C1 in their
 * own test files.  No value printed by the paper exists for this path, so "against the paper's own numbers" the parity
 * is unpinned (stated in DESIGN.md).
 *
 * Build: gcc -O2 -std=c11 -fopenmp -fPIC -shared bloch_ref.c -o libbloch_ref.so -lm   (no fast-math)
 */
#include <complex.h>
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define REF_TOL_T 1e-12 /* reading G13: times closer than this are one point */

typedef struct {
    int64_t n;        /* number of intervals; points are 0..n */
    double *t;        /* n+1 time points */
    double *G;        /* (n+1) x 3 gradient at the points, linear interpolation of the vertices */
    double *b1re;     /* n : B1 on [t_n, t_{n+1}), 0 if RF-free */
    double *b1im;     /* n */
    uint8_t *rf;      /* n : 1 if the interval is covered by an RF sample (reading G18) */
    int64_t *adc;     /* n+1 : ADC sample index recorded at point n, or -1 */
    double *u;        /* n+1 : motion waveform u(t_n) (x(t) = x + a u(t)); u(t) = t without a waveform */
} ref_grid;

static int cmp_double(const void *a, const void *b) {
    double x = *(const double *)a, y = *(const double *)b;
    return (x > y) - (x < y);
}

/* linear interpolation of one axis at time t; 0 outside the vertex range */
static double interp_axis(const double *gt, const double *gv, int64_t n, double t) {
    if (n <= 0) return 0.0;
    if (t < gt[0] - REF_TOL_T || t > gt[n - 1] + REF_TOL_T) return 0.0;
    if (n == 1) return gv[0];
    /* binary search for the segment [gt[lo], gt[lo+1]] containing t */
    int64_t lo = 0, hi = n - 1;
    while (hi - lo > 1) {
        int64_t mid = (lo + hi) / 2;
        if (gt[mid] <= t) lo = mid; else hi = mid;
    }
    double t0 = gt[lo], t1 = gt[hi];
    if (t1 - t0 <= 0.0) return gv[hi];
    double w = (t - t0) / (t1 - t0);
    if (w < 0.0) w = 0.0;
    if (w > 1.0) w = 1.0;
    return gv[lo] + w * (gv[hi] - gv[lo]);
}

/* index of the RF sample covering time tm, or -1 */
static int64_t rf_cover(const double *rf_t, const double *rf_dt, int64_t rf_n, double tm) {
    int64_t lo = 0, hi = rf_n - 1, j = -1;
    while (lo <= hi) {
        int64_t mid = (lo + hi) / 2;
        if (rf_t[mid] <= tm) { j = mid; lo = mid + 1; } else hi = mid - 1;
    }
    if (j >= 0 && tm < rf_t[j] + rf_dt[j]) return j;
    return -1;
}

/* motion waveform u at time t: linear interpolation of the vertices, held at the end values outside them */
static double interp_waveform(const double *mt, const double *mu, int64_t n, double t) {
    if (n <= 0) return t;
    if (t <= mt[0]) return mu[0];
    if (t >= mt[n - 1]) return mu[n - 1];
    int64_t lo = 0, hi = n - 1;
    while (hi - lo > 1) {
        int64_t mid = (lo + hi) / 2;
        if (mt[mid] <= t) lo = mid; else hi = mid;
    }
    double w = (t - mt[lo]) / (mt[hi] - mt[lo]);
    return mu[lo] + w * (mu[hi] - mu[lo]);
}

static void grid_free(ref_grid *g) {
    free(g->t); free(g->G); free(g->b1re); free(g->b1im); free(g->rf); free(g->adc); free(g->u);
    memset(g, 0, sizeof(*g));
}

/* Number of equal sub-steps of the interval [a, b]: RF-covered intervals are limited to dt_rf_max (:182),
 * and, with motion, every interval to dt_max (the paper's "intermediate points in the case of motion", :180). */
static int64_t ref_parts(double a, double b, int covered, double dt_rf_max, double dt_max) {
    double lim = 0.0;
    if (covered && dt_rf_max > 0.0) lim = dt_rf_max;
    if (dt_max > 0.0 && isfinite(dt_max) && (lim == 0.0 || dt_max < lim)) lim = dt_max;
    if (lim <= 0.0) return 1;
    int64_t parts = (int64_t)ceil(((b - a) - REF_TOL_T) / lim);
    return parts < 1 ? 1 : parts;
}

/*
 * Time grid: sorted unique union of 0, t_end, gradient vertices, RF sample edges and ADC times, refined so
 * that no RF-covered interval exceeds dt_rf_max (an RF piece of length L is cut into ceil(L/dt_rf_max)
 * equal sub-steps, reading G18; L is taken with the time tolerance of reading G13, i.e. a piece is longer
 * than dt_rf_max only if it exceeds it by more than 1e-12 s, so that the rounding of t_{n+1} - t_n late in a
 * long sequence -- ulp(10 s) = 1.8e-15 s -- never splits a nominal dt_rf_max step).  Returns 0 or a negative error.
 */
static int grid_build(ref_grid *g,
                      const double *const gt[3], const double *const gv[3], const int64_t gn[3],
                      const double *rf_t, const double *rf_dt, const double *rf_re, const double *rf_im,
                      int64_t rf_n, const double *adc_t, int64_t adc_n, double t_end, double dt_rf_max,
                      double dt_max, const double *mo_t, const double *mo_u, int64_t mo_n) {
    memset(g, 0, sizeof(*g));
    if (!(t_end > 0.0)) return -1;
    for (int64_t i = 1; i < mo_n; ++i) if (!(mo_t[i] > mo_t[i - 1])) return -6;
    int64_t cap = 2 + gn[0] + gn[1] + gn[2] + 2 * rf_n + adc_n + (mo_n > 0 ? mo_n : 0);
    double *raw = (double *)malloc(sizeof(double) * (size_t)cap);
    if (!raw) return -2;
    int64_t m = 0;
    raw[m++] = 0.0;
    raw[m++] = t_end;
    for (int a = 0; a < 3; ++a)
        for (int64_t i = 0; i < gn[a]; ++i) raw[m++] = gt[a][i];
    for (int64_t i = 0; i < rf_n; ++i) { raw[m++] = rf_t[i]; raw[m++] = rf_t[i] + rf_dt[i]; }
    for (int64_t i = 0; i < adc_n; ++i) raw[m++] = adc_t[i];
    /* the vertices of the motion waveform are points of the grid (those inside the sequence) */
    for (int64_t i = 0; i < mo_n; ++i) if (mo_t[i] >= 0.0 && mo_t[i] <= t_end) raw[m++] = mo_t[i];
    qsort(raw, (size_t)m, sizeof(double), cmp_double);
    /* unique with tolerance, clipped to [0, t_end] */
    int64_t u = 0;
    for (int64_t i = 0; i < m; ++i) {
        double t = raw[i];
        if (t < -REF_TOL_T || t > t_end + REF_TOL_T) { free(raw); return -3; }
        if (u == 0 || t - raw[u - 1] > REF_TOL_T) raw[u++] = t;
    }
    /* count refined points */
    int64_t total = 1;
    for (int64_t i = 0; i + 1 < u; ++i) {
        double a = raw[i], b = raw[i + 1];
        int64_t parts = ref_parts(a, b, rf_n > 0 && rf_cover(rf_t, rf_dt, rf_n, 0.5 * (a + b)) >= 0, dt_rf_max, dt_max);
        total += parts;
    }
    g->n = total - 1;
    g->t = (double *)malloc(sizeof(double) * (size_t)total);
    g->G = (double *)malloc(sizeof(double) * 3 * (size_t)total);
    g->b1re = (double *)calloc((size_t)total, sizeof(double));
    g->b1im = (double *)calloc((size_t)total, sizeof(double));
    g->rf = (uint8_t *)calloc((size_t)total, 1);
    g->adc = (int64_t *)malloc(sizeof(int64_t) * (size_t)total);
    g->u = (double *)malloc(sizeof(double) * (size_t)total);
    if (!g->t || !g->G || !g->b1re || !g->b1im || !g->rf || !g->adc || !g->u) { free(raw); grid_free(g); return -2; }
    int64_t k = 0;
    g->t[k++] = raw[0];
    for (int64_t i = 0; i + 1 < u; ++i) {
        double a = raw[i], b = raw[i + 1];
        int64_t parts = ref_parts(a, b, rf_n > 0 && rf_cover(rf_t, rf_dt, rf_n, 0.5 * (a + b)) >= 0, dt_rf_max, dt_max);
        for (int64_t p = 1; p < parts; ++p) g->t[k++] = a + (b - a) * ((double)p / (double)parts);
        g->t[k++] = b;
    }
    free(raw);
    for (int64_t n = 0; n <= g->n; ++n) {
        for (int a = 0; a < 3; ++a) g->G[3 * n + a] = interp_axis(gt[a], gv[a], gn[a], g->t[n]);
        g->u[n] = interp_waveform(mo_t, mo_u, mo_n, g->t[n]);
        g->adc[n] = -1;
    }
    for (int64_t n = 0; n < g->n; ++n) {
        int64_t j = (rf_n > 0) ? rf_cover(rf_t, rf_dt, rf_n, 0.5 * (g->t[n] + g->t[n + 1])) : -1;
        if (j >= 0) { g->rf[n] = 1; g->b1re[n] = rf_re[j]; g->b1im[n] = rf_im[j]; }
    }
    /* ADC sample i is recorded at the grid point equal to adc_t[i] (ADC order = sample order) */
    for (int64_t i = 0; i < adc_n; ++i) {
        int64_t lo = 0, hi = g->n;
        while (hi - lo > 1) {
            int64_t mid = (lo + hi) / 2;
            if (g->t[mid] <= adc_t[i] + REF_TOL_T) lo = mid; else hi = mid;
        }
        int64_t best = (fabs(g->t[hi] - adc_t[i]) < fabs(g->t[lo] - adc_t[i])) ? hi : lo;
        if (fabs(g->t[best] - adc_t[i]) > 2 * REF_TOL_T) { grid_free(g); return -4; }
        if (g->adc[best] != -1) { grid_free(g); return -5; } /* two ADC samples on one point */
        g->adc[best] = i;
    }
    return 0;
}

/* One spin, all intervals, exactly as the listing of SURVEY.md 8(c). */
static void integrate_spin(const ref_grid *g, double gamma, double x, double y, double z, double M0,
                           double T1, double T2, double dw, const double *vel, double complex *pMxy, double *pMz,
                           double complex *S, int accumulate, int force_excitation) {
    double complex Mxy = *pMxy;
    double Mz = *pMz;
    if (g->adc[0] >= 0) { if (accumulate) S[g->adc[0]] += Mxy; else S[g->adc[0]] = Mxy; }
    for (int64_t n = 0; n < g->n; ++n) {
        double dt = g->t[n + 1] - g->t[n];
        /* trapezoidal rule, Eq (12)-(13): mean of the two vertex values */
        double Gx = 0.5 * (g->G[3 * n + 0] + g->G[3 * n + 3]);
        double Gy = 0.5 * (g->G[3 * n + 1] + g->G[3 * n + 4]);
        double Gz = 0.5 * (g->G[3 * n + 2] + g->G[3 * n + 5]);
        double Bz = Gx * x + Gy * y + Gz * z + dw / gamma;                 /* Eq (2) */
        if (vel) {
            /* motion x(t) = x + v u(t), u(t) = t for a constant velocity: the trapezoid of
             * Eq (12)-(13) is taken on the effective field itself, Bz(t_n) = G(t_n) . x(t_n), at the two ends of the
             * interval (:180, :336) */
            double t0 = g->u[n], t1 = g->u[n + 1];
            double b0 = g->G[3 * n + 0] * (x + vel[0] * t0) + g->G[3 * n + 1] * (y + vel[1] * t0)
                        + g->G[3 * n + 2] * (z + vel[2] * t0);
            double b1 = g->G[3 * n + 3] * (x + vel[0] * t1) + g->G[3 * n + 4] * (y + vel[1] * t1)
                        + g->G[3 * n + 5] * (z + vel[2] * t1);
            Bz = 0.5 * (b0 + b1) + dw / gamma;
        }
        if (g->rf[n] || force_excitation) {
            /* excitation regime, Eq (5)-(9) */
            double complex B1 = g->b1re[n] + I * g->b1im[n];
            double B = sqrt(creal(B1) * creal(B1) + cimag(B1) * cimag(B1) + Bz * Bz);
            double complex alpha = 1.0, beta = 0.0;                         /* reading G10 */
            if (B > 0.0) {
                double phi = -gamma * B * dt;                               /* Eq (8) */
                double s = sin(0.5 * phi), c = cos(0.5 * phi);
                alpha = c - I * (Bz / B) * s;                               /* Eq (6) */
                beta = -I * (B1 / B) * s;                                   /* Eq (7) */
            }
            double complex Mxy_new = 2.0 * conj(alpha) * beta * Mz + conj(alpha) * conj(alpha) * Mxy
                                     - beta * beta * conj(Mxy);             /* Eq (9), row 1 */
            double Mz_new = (creal(alpha) * creal(alpha) + cimag(alpha) * cimag(alpha)
                             - creal(beta) * creal(beta) - cimag(beta) * cimag(beta)) * Mz
                            - 2.0 * creal(alpha * beta * conj(Mxy));        /* Eq (9), row 2 */
            Mxy = Mxy_new;
            Mz = Mz_new;
        } else {
            /* precession regime, Eq (10) with phi = -gamma Bz dt */
            double phi = -gamma * Bz * dt;
            Mxy = Mxy * (cos(phi) + I * sin(phi));
        }
        /* relaxation, Eq (11) */
        double E2 = exp(-dt / T2), E1 = exp(-dt / T1);
        Mxy = Mxy * E2;
        Mz = Mz * E1 + M0 * (1.0 - E1);
        int64_t a = g->adc[n + 1];
        if (a >= 0) { if (accumulate) S[a] += Mxy; else S[a] = Mxy; }
    }
    *pMxy = Mxy;
    *pMz = Mz;
}

/*
 * bloch_ref_simulate
 *   gamma        rad/s/T
 *   g_t/g_v/g_n  per-axis gradient vertices (ascending times), G = 0 outside
 *   rf_*         piecewise-constant B1 samples on [rf_t, rf_t + rf_dt)
 *   adc_t        ADC sample times; t_end: sequence end; dt_rf_max: RF refinement step
 *   spins        x, y, z, M0, T1, T2, dw (fp64 arrays of n_spins)
 *   Mxy (interleaved re,im; 2*n_spins) and Mz: in-out state, used only if use_state != 0; if NULL or
 *                use_state == 0 the state starts at equilibrium (reading G8) and is discarded
 *   signal       output_mode 0: 2*adc_n doubles (sum over spins); 1: n_spins x adc_n x 2 doubles
 *   flags        bit 0: force every interval through the excitation branch (invariant I5 only)
 *   returns 0, or <0 on invalid input.
 */
int bloch_ref_simulate_waveform(double gamma,
                       const double *gx_t, const double *gx_v, int64_t gx_n,
                       const double *gy_t, const double *gy_v, int64_t gy_n,
                       const double *gz_t, const double *gz_v, int64_t gz_n,
                       const double *rf_t, const double *rf_dt, const double *rf_re, const double *rf_im,
                       int64_t rf_n, const double *adc_t, int64_t adc_n, double t_end, double dt_rf_max,
                       int64_t n_spins, const double *x, const double *y, const double *z,
                       const double *M0, const double *T1, const double *T2, const double *dw,
                       double *Mxy, double *Mz, int use_state,
                       double *signal, int output_mode, int n_threads, int flags,
                       double dt_max, const double *vx, const double *vy, const double *vz,
                       const double *mo_t, const double *mo_u, int64_t mo_n) {
    const double *const gt[3] = {gx_t, gy_t, gz_t};
    const double *const gv[3] = {gx_v, gy_v, gz_v};
    const int64_t gn[3] = {gx_n, gy_n, gz_n};
    ref_grid g;
    int rc = grid_build(&g, gt, gv, gn, rf_t, rf_dt, rf_re, rf_im, rf_n, adc_t, adc_n, t_end, dt_rf_max, dt_max,
                        mo_t, mo_u, mo_n);
    if (rc) return rc;
    const int moving = vx && vy && vz;
    int nth = n_threads > 0 ? n_threads : 1;
#ifndef _OPENMP
    nth = 1;
#endif
    int force = flags & 1;
    if (output_mode == 1) {
#pragma omp parallel for num_threads(nth) schedule(static)
        for (int64_t i = 0; i < n_spins; ++i) {
            double complex mxy = 0.0;
            double mz = M0[i];
            if (use_state && Mxy && Mz) { mxy = Mxy[2 * i] + I * Mxy[2 * i + 1]; mz = Mz[i]; }
            double complex *S = (double complex *)(signal + 2 * i * adc_n);
            double vel[3] = {0.0, 0.0, 0.0};
            if (moving) { vel[0] = vx[i]; vel[1] = vy[i]; vel[2] = vz[i]; }
            integrate_spin(&g, gamma, x[i], y[i], z[i], M0[i], T1[i], T2[i], dw[i], moving ? vel : NULL, &mxy, &mz,
                           S, 0, force);
            if (Mxy && Mz) { Mxy[2 * i] = creal(mxy); Mxy[2 * i + 1] = cimag(mxy); Mz[i] = mz; }
        }
    } else {
        /* per-thread signal matrices, added afterwards */
        double complex *bufs = (double complex *)calloc((size_t)nth * (size_t)(adc_n > 0 ? adc_n : 1),
                                                        sizeof(double complex));
        if (!bufs) { grid_free(&g); return -2; }
#pragma omp parallel num_threads(nth)
        {
            int tid = 0;
#ifdef _OPENMP
            tid = omp_get_thread_num();
#endif
            double complex *S = bufs + (size_t)tid * (size_t)adc_n;
#pragma omp for schedule(static)
            for (int64_t i = 0; i < n_spins; ++i) {
                double complex mxy = 0.0;
                double mz = M0[i];
                if (use_state && Mxy && Mz) { mxy = Mxy[2 * i] + I * Mxy[2 * i + 1]; mz = Mz[i]; }
                double vel[3] = {0.0, 0.0, 0.0};
                if (moving) { vel[0] = vx[i]; vel[1] = vy[i]; vel[2] = vz[i]; }
                integrate_spin(&g, gamma, x[i], y[i], z[i], M0[i], T1[i], T2[i], dw[i], moving ? vel : NULL, &mxy,
                               &mz, S, 1, force);
                if (Mxy && Mz) { Mxy[2 * i] = creal(mxy); Mxy[2 * i + 1] = cimag(mxy); Mz[i] = mz; }
            }
        }
        for (int64_t a = 0; a < adc_n; ++a) {
            double complex s = 0.0;
            for (int t = 0; t < nth; ++t) s += bufs[(size_t)t * (size_t)adc_n + a];
            signal[2 * a] = creal(s);
            signal[2 * a + 1] = cimag(s);
        }
        free(bufs);
    }
    grid_free(&g);
    return 0;
}

/* Constant velocities: x(t) = x + v t, i.e. the waveform entry with u(t) = t. */
int bloch_ref_simulate_motion(double gamma,
                       const double *gx_t, const double *gx_v, int64_t gx_n,
                       const double *gy_t, const double *gy_v, int64_t gy_n,
                       const double *gz_t, const double *gz_v, int64_t gz_n,
                       const double *rf_t, const double *rf_dt, const double *rf_re, const double *rf_im,
                       int64_t rf_n, const double *adc_t, int64_t adc_n, double t_end, double dt_rf_max,
                       int64_t n_spins, const double *x, const double *y, const double *z,
                       const double *M0, const double *T1, const double *T2, const double *dw,
                       double *Mxy, double *Mz, int use_state,
                       double *signal, int output_mode, int n_threads, int flags,
                       double dt_max, const double *vx, const double *vy, const double *vz) {
    return bloch_ref_simulate_waveform(gamma, gx_t, gx_v, gx_n, gy_t, gy_v, gy_n, gz_t, gz_v, gz_n, rf_t, rf_dt, rf_re,
                                       rf_im, rf_n, adc_t, adc_n, t_end, dt_rf_max, n_spins, x, y, z, M0, T1, T2, dw,
                                       Mxy, Mz, use_state, signal, output_mode, n_threads, flags, dt_max, vx, vy, vz,
                                       NULL, NULL, 0);
}

/* The static-phantom entry: no motion, no dt_max refinement. */
int bloch_ref_simulate(double gamma,
                       const double *gx_t, const double *gx_v, int64_t gx_n,
                       const double *gy_t, const double *gy_v, int64_t gy_n,
                       const double *gz_t, const double *gz_v, int64_t gz_n,
                       const double *rf_t, const double *rf_dt, const double *rf_re, const double *rf_im,
                       int64_t rf_n, const double *adc_t, int64_t adc_n, double t_end, double dt_rf_max,
                       int64_t n_spins, const double *x, const double *y, const double *z,
                       const double *M0, const double *T1, const double *T2, const double *dw,
                       double *Mxy, double *Mz, int use_state,
                       double *signal, int output_mode, int n_threads, int flags) {
    return bloch_ref_simulate_motion(gamma, gx_t, gx_v, gx_n, gy_t, gy_v, gy_n, gz_t, gz_v, gz_n, rf_t, rf_dt, rf_re,
                                     rf_im, rf_n, adc_t, adc_n, t_end, dt_rf_max, n_spins, x, y, z, M0, T1, T2, dw,
                                     Mxy, Mz, use_state, signal, output_mode, n_threads, flags, 0.0, NULL, NULL, NULL);
}

/*
 * bloch_ref_grid: expose the oracle's own discretisation for tests (refinement invariance, trapezoid areas).
 * Call with t_out == NULL to get the number of intervals; otherwise fills t_out[n+1], G_out[3(n+1)],
 * rf_out[n], adc_out[n+1] (caller-allocated).  Returns n (>= 0) or <0 on error.
 */
int64_t bloch_ref_grid_waveform(const double *gx_t, const double *gx_v, int64_t gx_n,
                       const double *gy_t, const double *gy_v, int64_t gy_n,
                       const double *gz_t, const double *gz_v, int64_t gz_n,
                       const double *rf_t, const double *rf_dt, const double *rf_re, const double *rf_im,
                       int64_t rf_n, const double *adc_t, int64_t adc_n, double t_end, double dt_rf_max,
                       double *t_out, double *G_out, uint8_t *rf_out, int64_t *adc_out, double dt_max,
                       const double *mo_t, const double *mo_u, int64_t mo_n, double *u_out) {
    const double *const gt[3] = {gx_t, gy_t, gz_t};
    const double *const gv[3] = {gx_v, gy_v, gz_v};
    const int64_t gn[3] = {gx_n, gy_n, gz_n};
    ref_grid g;
    int rc = grid_build(&g, gt, gv, gn, rf_t, rf_dt, rf_re, rf_im, rf_n, adc_t, adc_n, t_end, dt_rf_max, dt_max,
                        mo_t, mo_u, mo_n);
    if (rc) return rc;
    int64_t n = g.n;
    if (t_out) {
        memcpy(t_out, g.t, sizeof(double) * (size_t)(n + 1));
        if (G_out) memcpy(G_out, g.G, sizeof(double) * 3 * (size_t)(n + 1));
        if (rf_out) memcpy(rf_out, g.rf, (size_t)n);
        if (adc_out) memcpy(adc_out, g.adc, sizeof(int64_t) * (size_t)(n + 1));
        if (u_out) memcpy(u_out, g.u, sizeof(double) * (size_t)(n + 1));
    }
    grid_free(&g);
    return n;
}

int64_t bloch_ref_grid_motion(const double *gx_t, const double *gx_v, int64_t gx_n,
                       const double *gy_t, const double *gy_v, int64_t gy_n,
                       const double *gz_t, const double *gz_v, int64_t gz_n,
                       const double *rf_t, const double *rf_dt, const double *rf_re, const double *rf_im,
                       int64_t rf_n, const double *adc_t, int64_t adc_n, double t_end, double dt_rf_max,
                       double *t_out, double *G_out, uint8_t *rf_out, int64_t *adc_out, double dt_max) {
    return bloch_ref_grid_waveform(gx_t, gx_v, gx_n, gy_t, gy_v, gy_n, gz_t, gz_v, gz_n, rf_t, rf_dt, rf_re, rf_im, rf_n,
                                   adc_t, adc_n, t_end, dt_rf_max, t_out, G_out, rf_out, adc_out, dt_max, NULL, NULL, 0, NULL);
}

int64_t bloch_ref_grid(const double *gx_t, const double *gx_v, int64_t gx_n,
                       const double *gy_t, const double *gy_v, int64_t gy_n,
                       const double *gz_t, const double *gz_v, int64_t gz_n,
                       const double *rf_t, const double *rf_dt, const double *rf_re, const double *rf_im,
                       int64_t rf_n, const double *adc_t, int64_t adc_n, double t_end, double dt_rf_max,
                       double *t_out, double *G_out, uint8_t *rf_out, int64_t *adc_out) {
    return bloch_ref_grid_motion(gx_t, gx_v, gx_n, gy_t, gy_v, gy_n, gz_t, gz_v, gz_n, rf_t, rf_dt, rf_re, rf_im, rf_n,
                                 adc_t, adc_n, t_end, dt_rf_max, t_out, G_out, rf_out, adc_out, 0.0);
}
