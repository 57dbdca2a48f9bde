/*
 * longtrack_oracle.h -- CPU ORACLE for the longitudinal tracking hot path.
 *
 * THIS IS TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only tests/, __graft_entry__.smoke()
 * and bench.py's cpu_baseline / --impl reference legs may build, load or call it.
 * It shares no code, header, constant or helper with the CUDA path
 * (paper_1610_05801_b200/csrc/, include/longtrack.h) and neither includes the other.
 *
 * What it computes (citations: PAPER.md = /root/reference/PAPER.md at build time,
 * BASELINE.json = repo root):
 *   - the turn-by-turn longitudinal map of every macro-particle's (z, delta)
 *     [PAPER.md:43 (sec. 1.1.2) names the integrators Euler-Cromer (1st order),
 *      Leap-Frog (2nd order Verlet) and Ruth (4th order); PAPER.md:163-165 (sec. 2.3)
 *      fixes the loop structure: turns sequential, particles independent;
 *      the paper prints no map equation, so the formula is BASELINE.json:configs[0]:
 *        "One turn: z-=eta*C/2*delta; delta+=A*sin(h*z/R); z-=eta*C/2*delta"
 *      and BASELINE.json:configs[4] for the double-harmonic kick
 *        "delta+=A*[sin(h*z/R)+r*sin(2h*z/R)]"],
 *   - per-turn bunch moments (mean and rms of z and delta) [BASELINE.json:configs[3]],
 *   - the Hamiltonian and the bucket-membership count [BASELINE.json:north_star,
 *     "bucket-membership counts (exact)"; readings G11/G15 in DESIGN.md].
 *
 * It is an ITERATION, so the oracle follows the algorithm step by step in fp64,
 * scalar, with libm sin/cos, compiled with -ffp-contract=off (no FMA contraction):
 * every '*' and '+' below rounds once, exactly as written.  No blocking, no fusion,
 * no reordering.  The only parallelism is an OpenMP 'parallel for' over particles,
 * which are independent.
 *
 * Pins (tests/test_oracle_pins.py, -m "not gpu"): exact discrete tune, determinant,
 * time reversal, bounded Hamiltonian, pendulum period vs the complete elliptic
 * integral, 40-digit hand-iterated values (tests/golden/; incl. phi_s = 0.3 and -0.7 for the
 * generic kick of reading G3), pure-shear / pure-kick
 * special cases, matrix-power small-amplitude limit, 80-bit self-check, moments vs
 * numpy, membership vs brute force.  The ARITHMETIC of every function here is pinned;
 * the CHOICE of map is pinned by BASELINE.json only (the paper prints none) -- see
 * DESIGN.md "Readings".
 */
#ifndef LONGTRACK_ORACLE_H
#define LONGTRACK_ORACLE_H

#include <stddef.h>

#ifdef __cplusplus
extern "C" {
#endif

enum { LTO_EULER_CROMER = 0, LTO_LEAPFROG = 1, LTO_RUTH4 = 2 };

/* Ring / RF parameters, BASELINE.json:north_star (1) "(C, gamma, alpha_c, h, V, phi_s,
 * integrator)" plus p0 and the charge that A needs (configs[0]: "A=qV/(beta*c*p0)")
 * and the second-harmonic ratio r (configs[4]). */
typedef struct {
    double circumference_m; /* C */
    double gamma;           /* Lorentz gamma; beta = sqrt(1-1/gamma^2) */
    double alpha_c;         /* momentum compaction; eta = alpha_c - 1/gamma^2 */
    double p0c_eV;          /* reference momentum times c, in eV */
    double charge_e;        /* q in units of e */
    int    harmonic;        /* h */
    double voltage_V;       /* V */
    double phi_s;           /* synchronous phase, rad (0 in every config) */
    double ratio2;          /* r: amplitude ratio of the harmonic at 2h (0 = off) */
    int    integrator;      /* LTO_* */
} lto_params;

/* Derived constants, notation of DESIGN.md / SURVEY.md sec. 8. */
typedef struct {
    double R;      /* C/(2 pi)                               */
    double beta;   /* sqrt(1 - 1/gamma^2)                    */
    double eta;    /* alpha_c - 1/gamma^2                    */
    double A;      /* q V / (beta p0c)                       */
    double d;      /* eta C / 2  (half-turn drift coeff)     */
    double kappa;  /* h / R                                  */
    double K;      /* eta C A h / R                          */
    double z_max;  /* pi R / h  (bucket half length)         */
    double H_sep;  /* 2 A R / h (Hamiltonian on separatrix)  */
} lto_derived;

/* mean_z, rms_z, mean_d, rms_d over all n particles (population rms about the mean),
 * cov_zd = <(z-<z>)(d-<d>)>, n_in_bucket = membership count of the same state. */
typedef struct {
    double mean_z, rms_z, mean_d, rms_d, cov_zd;
    unsigned long long n_in_bucket;
} lto_moments;

int  lto_derive(const lto_params *p, lto_derived *out);

/* Kick function F(z) = A [ sin(phi_s + kappa z) - sin(phi_s) + r sin(2 kappa z) ]. */
double lto_kick(const lto_params *p, double z);

/* One turn / N turns, in place, on n particles. */
void lto_one_turn(const lto_params *p, double *z, double *delta, size_t n);
void lto_track(const lto_params *p, double *z, double *delta, size_t n,
               unsigned long long turns);

/* Adjoint (time-reversed ordering) of Euler-Cromer, used only by the reversibility pin. */
void lto_one_turn_ec_adjoint(const lto_params *p, double *z, double *delta, size_t n);

/* Same map in 80-bit long double (constants derived in long double too). */
void lto_track_ld(const lto_params *p, long double *z, long double *delta, size_t n,
                  unsigned long long turns);

/* N turns, emitting the moments of the state AFTER each turn: out[t] <-> turn t+1. */
void lto_track_moments(const lto_params *p, double *z, double *delta, size_t n,
                       unsigned long long turns, lto_moments *out);

void lto_moments_of(const lto_params *p, const double *z, const double *delta, size_t n,
                    lto_moments *out);

/* H(z, delta) = eta C delta^2 / 2 + (A R / h) [ (1 - cos kappa z) + (r/2)(1 - cos 2 kappa z) ]. */
double lto_hamiltonian(const lto_params *p, double z, double delta);
void   lto_hamiltonian_n(const lto_params *p, const double *z, const double *delta,
                         size_t n, double *H);

/* Membership: |z| < z_max  and  H(z, delta) < H_sep. */
int  lto_in_bucket(const lto_params *p, double z, double delta);
unsigned long long lto_bucket_count(const lto_params *p, const double *z,
                                    const double *delta, size_t n);
void lto_bucket_mask(const lto_params *p, const double *z, const double *delta,
                     size_t n, unsigned char *mask);

int  lto_num_threads(void);
void lto_set_num_threads(int n);

#ifdef __cplusplus
}
#endif
#endif
