/*
 * next_oracle.c -- plain, slow, scalar CPU oracle for SURVEY.md sec. 8(f) rows f2-f4.
 * TEST INFRASTRUCTURE ONLY; read next_oracle.h first (scope, citations, readings).
 *
 * Built into liblongtrack_oracle.so together with longtrack_oracle.c (oracle/__init__.py):
 *   gcc -O2 -ffp-contract=off -fopenmp -fPIC -shared ... longtrack_oracle.c next_oracle.c -lm
 */
#include "next_oracle.h"

#include <math.h>
#include <string.h>

/* ---- the base map's constants + the programme map, in double and in long double -------- */
#define REAL double
#define SIN  sin
#define SQRT sqrt
#define CBRT cbrt
#define PI   3.14159265358979323846
#define NAME(x) n64_##x
#include "map.inc"
#include "programme.inc"
#include "ramp.inc"
#undef REAL
#undef SIN
#undef SQRT
#undef CBRT
#undef PI
#undef NAME

#define REAL long double
#define SIN  sinl
#define SQRT sqrtl
#define CBRT cbrtl
#define PI   3.14159265358979323846264338327950288L
#define NAME(x) n80_##x
#include "map.inc"
#include "programme.inc"
#include "ramp.inc"
#undef REAL
#undef SIN
#undef SQRT
#undef CBRT
#undef PI
#undef NAME

/* map.inc defines helpers this file does not call (it is compiled twice here for its
 * constants only); keep -Wall quiet without touching the pinned file */
static void touch_unused(void) __attribute__((unused));
static void touch_unused(void)
{
    (void)n64_track_particles; (void)n80_track_particles;
    (void)n64_one_turn;        (void)n80_one_turn;
}

/* ---- f2 ---------------------------------------------------------------------------------- */
void lto_track_programme(const lto_params *p, double *z, double *delta, size_t n,
                         unsigned long long turns, const double *volt_scale,
                         const double *phase_off)
{
    n64_prog_track_particles(p, z, delta, n, turns, volt_scale, phase_off);
}

void lto_track_programme_ld(const lto_params *p, long double *z, long double *delta, size_t n,
                            unsigned long long turns, const double *volt_scale,
                            const double *phase_off)
{
    n80_prog_track_particles(p, z, delta, n, turns, volt_scale, phase_off);
}

void lto_track_programme_moments(const lto_params *p, double *z, double *delta, size_t n,
                                 unsigned long long turns, const double *volt_scale,
                                 const double *phase_off, lto_moments *out)
{
    unsigned long long t;
    for (t = 0; t < turns; ++t) {
        n64_prog_track_particles(p, z, delta, n, 1ULL, volt_scale + t, phase_off + t);
        lto_moments_of(p, z, delta, n, &out[t]);
    }
}

/* ---- f2, energy ramp (reading G32) ------------------------------------------------------- */
void lto_track_ramp(const lto_params *p, double *z, double *delta, size_t n,
                    unsigned long long turns, const double *p0c, const double *volt_scale,
                    const double *phase_off)
{
    n64_ramp_track_particles(p, z, delta, n, turns, p0c, volt_scale, phase_off);
}

void lto_track_ramp_ld(const lto_params *p, long double *z, long double *delta, size_t n,
                       unsigned long long turns, const double *p0c, const double *volt_scale,
                       const double *phase_off)
{
    n80_ramp_track_particles(p, z, delta, n, turns, p0c, volt_scale, phase_off);
}

void lto_track_ramp_moments(const lto_params *p, double *z, double *delta, size_t n,
                            unsigned long long turns, const double *p0c, const double *volt_scale,
                            const double *phase_off, lto_moments *out)
{
    unsigned long long t;
    for (t = 0; t < turns; ++t) {
        n64_ramp_track_particles(p, z, delta, n, 1ULL, p0c + t, volt_scale ? volt_scale + t : NULL,
                                 phase_off ? phase_off + t : NULL);
        lto_moments_of(p, z, delta, n, &out[t]);
    }
}

void lto_ramp_numbers(const lto_params *p, double p0c, double *mc2, double *beta, double *eta,
                      double *A, double *d)
{
    const double m = n64_ramp_rest_energy(p);
    const n64_ramp_point q = n64_ramp_at(p, m, p0c);
    if (mc2) *mc2 = m;
    if (beta) *beta = (double)p->charge_e * p->voltage_V / (q.A * p0c);
    if (eta) *eta = 2.0 * q.d / p->circumference_m;
    if (A) *A = q.A;
    if (d) *d = q.d;
}

/* ---- f4 ---------------------------------------------------------------------------------- */
void lto_slice_histogram(const double *z, size_t n, double z_lo, double z_hi, int n_slices,
                         unsigned long long *hist)
{
    const double inv = (double)n_slices / (z_hi - z_lo);
    size_t i;
    memset(hist, 0, ((size_t)n_slices + 2) * sizeof(hist[0]));
    for (i = 0; i < n; ++i) {
        const double zi = z[i];
        if (zi < z_lo) {
            hist[0] += 1;
        } else if (!(zi < z_hi)) {
            hist[(size_t)n_slices + 1] += 1;
        } else {
            double u = (zi - z_lo) * inv;
            long long s = (long long)floor(u);
            if (s > (long long)n_slices - 1) s = (long long)n_slices - 1;
            hist[1 + (size_t)s] += 1;
        }
    }
}

void lto_track_slices(const lto_params *p, double *z, double *delta, size_t n,
                      unsigned long long turns, double z_lo, double z_hi, int n_slices,
                      unsigned long long *hist)
{
    unsigned long long t;
    for (t = 0; t < turns; ++t) {
        lto_track(p, z, delta, n, 1ULL);
        lto_slice_histogram(z, n, z_lo, z_hi, n_slices, hist + t * ((size_t)n_slices + 2));
    }
}

/* ---- f3 ---------------------------------------------------------------------------------- */
void lto_track_transverse(const lto_params *p, const double *matrices, int n_seg,
                          double *x, double *xp, double *y, double *yp,
                          double *z, double *delta, size_t n, unsigned long long turns)
{
    long long i;
#pragma omp parallel for schedule(static) if (n > 2048)
    for (i = 0; i < (long long)n; ++i) {
        double u0 = x[i], u1 = xp[i], u2 = y[i], u3 = yp[i];
        unsigned long long t;
        int s;
        for (t = 0; t < turns; ++t) {
            for (s = 0; s < n_seg; ++s) {
                const double *M = matrices + 16 * (size_t)s;
                double w0 = ((M[0]  * u0 + M[1]  * u1) + M[2]  * u2) + M[3]  * u3;
                double w1 = ((M[4]  * u0 + M[5]  * u1) + M[6]  * u2) + M[7]  * u3;
                double w2 = ((M[8]  * u0 + M[9]  * u1) + M[10] * u2) + M[11] * u3;
                double w3 = ((M[12] * u0 + M[13] * u1) + M[14] * u2) + M[15] * u3;
                u0 = w0; u1 = w1; u2 = w2; u3 = w3;
            }
        }
        x[i] = u0; xp[i] = u1; y[i] = u2; yp[i] = u3;
    }
    /* the longitudinal plane is not coupled to the transverse one here, so its turn loop can
     * run after the transverse one without changing a bit */
    if (z && delta) lto_track(p, z, delta, n, turns);
}
