/*
 * next_oracle.h -- CPU ORACLE for the rows SURVEY.md sec. 8(f) marks "next":
 *   f2  turn-dependent RF programme      (sec. 2.2)
 *   f3  transverse linear transfer maps  (sec. 1.1.1; Fig. 2)
 *   f4  longitudinal slicing histogram   (sec. 1.1; sec. 3)
 *
 * THIS IS TEST INFRASTRUCTURE, NOT THE PRODUCT (same rules as longtrack_oracle.h): only
 * tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
 * build, load or call it; it shares no code, header, constant or helper with the CUDA path.
 * Plain C, scalar, fp64, libm, compiled with -ffp-contract=off: every '*', '+', '-' and '/'
 * rounds once, exactly as written; OpenMP only over particles, which are independent
 * (PAPER.md:163).
 *
 * The paper prints no formula for any of the three; the readings are DESIGN.md G28-G30 and
 * are restated at each function.  Pins: tests/test_next_oracle_pins.py (-m "not gpu").
 */
#ifndef NEXT_ORACLE_H
#define NEXT_ORACLE_H

#include <stddef.h>

#include "longtrack_oracle.h"

#ifdef __cplusplus
extern "C" {
#endif

/* ---- f2: RF programme (reading G28) ---------------------------------------------------
 * Entry t (0-based) of volt_scale[] / phase_off[] applies to every kick of turn t+1:
 *   F_t(z) = a_t A [ sin(phi_s + kappa z + psi_t) - sin(phi_s) + r sin(2 (kappa z + psi_t)) ]
 * a_t = volt_scale[t] (dimensionless, V_t / V), psi_t = phase_off[t] (rad). */
void lto_track_programme(const lto_params *p, double *z, double *delta, size_t n,
                         unsigned long long turns, const double *volt_scale,
                         const double *phase_off);
void lto_track_programme_ld(const lto_params *p, long double *z, long double *delta, size_t n,
                            unsigned long long turns, const double *volt_scale,
                            const double *phase_off);
/* out[t] = moments of the state after turn t+1 (as lto_track_moments) */
void lto_track_programme_moments(const lto_params *p, double *z, double *delta, size_t n,
                                 unsigned long long turns, const double *volt_scale,
                                 const double *phase_off, lto_moments *out);

/* ---- f2, energy ramp (reading G32; the formulas are restated in ramp.inc) ----------------
 * p0c[0 .. turns]: reference momentum x c (eV) before turn 1 and after every turn.
 * volt_scale / phase_off: as above, or NULL for a_t = 1 / psi_t = 0.  p->phi_s must be 0.
 *   sub-step(tau, pb -> pa):  z -= tau d(pb) delta
 *                             delta = (delta + tau a_t A(pb) [sin(kappa z + psi_t) + r sin(2(kappa z + psi_t))]
 *                                      - (pa - pb)/pb) * (pb/pa)
 *                             z -= tau d(pa) delta
 * with A(p) = qV/(beta(p) p), d(p) = eta(p) C/2, beta, eta from p and mc2 = p0c_create/(beta gamma). */
void lto_track_ramp(const lto_params *p, double *z, double *delta, size_t n,
                    unsigned long long turns, const double *p0c, const double *volt_scale,
                    const double *phase_off);
void lto_track_ramp_ld(const lto_params *p, long double *z, long double *delta, size_t n,
                       unsigned long long turns, const double *p0c, const double *volt_scale,
                       const double *phase_off);
/* out[t] = moments of the state after turn t+1 (membership: the stationary bucket of p) */
void lto_track_ramp_moments(const lto_params *p, double *z, double *delta, size_t n,
                            unsigned long long turns, const double *p0c, const double *volt_scale,
                            const double *phase_off, lto_moments *out);
/* the momentum-dependent ring numbers at reference momentum p0c (for the tests and recipes) */
void lto_ramp_numbers(const lto_params *p, double p0c, double *mc2, double *beta, double *eta,
                      double *A, double *d);

/* ---- f4: longitudinal slicing (reading G29) --------------------------------------------
 * Uniform slices of z over [z_lo, z_hi): inv = S / (z_hi - z_lo);
 *   z < z_lo            -> hist[0]     ("below")
 *   not (z < z_hi)      -> hist[S+1]   ("above"; NaN lands here)
 *   otherwise             u = (z - z_lo) * inv;  s = floor(u), clamped to S-1;  hist[1+s]
 * hist has S+2 entries and is OVERWRITTEN. */
void lto_slice_histogram(const double *z, size_t n, double z_lo, double z_hi, int n_slices,
                         unsigned long long *hist);
/* per-turn mode: track one turn, then slice; hist[t] (S+2 entries each) <-> state after turn t+1 */
void lto_track_slices(const lto_params *p, double *z, double *delta, size_t n,
                      unsigned long long turns, double z_lo, double z_hi, int n_slices,
                      unsigned long long *hist);

/* ---- f3: transverse plane (reading G30) -------------------------------------------------
 * State (x, x', y, y') per particle, structure of arrays.  One turn = for every segment
 * s = 0 .. n_seg-1 in order: u <- M_s u with M_s a 4x4 matrix, ROW-MAJOR in
 * matrices[16 s + 4 i + j] = (M_s)_ij, each row evaluated left to right
 *   u'_i = ((M_i0 x + M_i1 x') + M_i2 y) + M_i3 y'
 * followed by the longitudinal turn of (z, delta) (lto_track's map; the two planes are not
 * coupled in the linear-matrix description of PAPER.md:39). z/delta may be NULL (transverse
 * only). */
void lto_track_transverse(const lto_params *p, const double *matrices, int n_seg,
                          double *x, double *xp, double *y, double *yp,
                          double *z, double *delta, size_t n, unsigned long long turns);

#ifdef __cplusplus
}
#endif
#endif
