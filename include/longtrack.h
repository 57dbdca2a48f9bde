/*
 * longtrack.h -- C ABI of liblongtrack.so: the B200 (sm_100a) hot path of PyHEADTAIL's
 * longitudinal tracking engine (arxiv/paper_1610_05801, A. Oeftiger, "Parallelisation of
 * PyHEADTAIL").
 *
 * Citations: PAPER.md = the paper's text (/root/reference/PAPER.md when this was written),
 * BASELINE.json = the task statement at the repo root, DESIGN.md = this repo.
 *
 * The operation (sec. 1.1.2): "the particles' motion in longitudinal phase
 * space -- which comprises two coordinates, the spatial location z and the corresponding
 * (dimensionless) conjugate momentum delta -- is integrated turn by turn [...] via either
 * the Euler-Cromer (first order), Leap-Frog (second order Verlet) or Runge-Kutta resp.
 * Ruth (fourth order) numerical integration algorithms [...] independently done for each
 * particle's entry in the z and delta arrays".  The paper prints no map equation; the map
 * is BASELINE.json:configs[0]:
 *
 *     one turn (leap-frog):  z -= eta*C/2*delta;  delta += F(z);  z -= eta*C/2*delta
 *     F(z) = A*[ sin(phi_s + h*z/R) - sin(phi_s) + r*sin(2*h*z/R) ]     (configs[0], [4])
 *     R = C/2pi, beta = sqrt(1-1/gamma^2), eta = alpha_c - 1/gamma^2, A = q*V/(beta*p0c)
 *     Euler-Cromer:  delta += F(z);  z -= eta*C*delta                    (G8)
 *     Ruth4:         three leap-frog steps with factors x1, x0, x1,
 *                    x1 = 1/(2-2^(1/3)), x0 = -2^(1/3)/(2-2^(1/3))        (G9)
 *
 * Loop structure (sec. 2.3): turns are sequential, particles independent;
 * a thread keeps its particle in registers over many turns ("fused" mode below), or the
 * turn loop is driven from the host with the state going through device memory every turn
 * ("per-turn" mode; BASELINE.json:configs[3] adds the per-turn bunch moments).
 *
 * Conventions for every call
 *   - Pointers named *_dev are DEVICE pointers (cudaMalloc / torch CUDA tensors), those
 *     named *_host are HOST pointers.  The caller owns every array; the library owns the
 *     tracker handle and a small device scratch (grown lazily, freed by lt_destroy).
 *   - z and delta are two separate, contiguous arrays of n values (structure of arrays,
 *     PAPER.md:163-165), updated IN PLACE.  8-byte (fp64) / 4-byte (fp32) alignment is
 *     required; 16-byte alignment enables the vector path (otherwise a scalar path runs).
 *   - `stream` is a cudaStream_t passed as void* (NULL = the legacy default stream).  Device
 *     calls only ENQUEUE work on that stream and return; nothing synchronises the device.
 *     Results are valid once the caller has synchronised the stream.  The *_host calls are the
 *     exception: they run to completion before they return.
 *     The tracker's scratch is grown STREAM-ORDERED on the caller's stream (cudaMallocAsync /
 *     cudaFreeAsync): a call that needs more scratch than any before it (a larger n, a longer
 *     table) allocates without a device synchronisation, but it must not be issued while the
 *     stream is being CAPTURED into a CUDA graph by the caller -- run the call once uncaptured
 *     at the largest size first.
 *   - If a device call returns LT_E_CUDA part-way through a fused call that needed several
 *     launches (LT_OPT_CHUNK_TURNS smaller than `turns`), the arrays hold an intermediate state:
 *     in the default merged-drift mode z is then the RF phase in half periods, mid-drift, NOT
 *     metres.  Treat z/delta as lost after LT_E_CUDA.
 *   - Return value: 0 = LT_OK, negative = error (below).  The library never throws, aborts
 *     or prints.  n == 0 or turns == 0 is LT_OK and a no-op.
 *   - One tracker may have ONE call in flight at a time (the scratch is per tracker); use
 *     one tracker per stream for concurrency.  Trackers are cheap.
 *   - There is no CPU fallback: without a CUDA device every device call returns LT_E_CUDA.
 */
#ifndef LONGTRACK_H
#define LONGTRACK_H

#include <stddef.h>

#ifdef __cplusplus
extern "C" {
#endif

#define LT_VERSION 100 /* 0.1.0 */

typedef struct lt_tracker lt_tracker; /* opaque, library-owned */

typedef enum { LT_EULER_CROMER = 0, LT_LEAPFROG = 1, LT_RUTH4 = 2 } lt_integrator;

enum {
    LT_OK         = 0,
    LT_E_NULL     = -1, /* a required pointer is NULL                                     */
    LT_E_PARAM    = -2, /* gamma <= 1, C <= 0, h <= 0, p0c <= 0, unknown integrator/option,
                           non-finite parameter, n too large                              */
    LT_E_UNSTABLE = -3, /* linearised map unstable: K_eff = K*(cos(phi_s)+2r) < 0 or >= 4
                           (K_eff == 0 is allowed, G10)                         */
    LT_E_ALIGN    = -4, /* array pointer not aligned to its element size                  */
    LT_E_CUDA     = -5, /* a CUDA runtime call failed; see lt_last_cuda_error()           */
    LT_E_NOMEM    = -6, /* host allocation failed                                         */
    LT_E_CAPACITY = -7  /* n exceeds the fixed capacity of an entry point that works in the
                           library's built-in scratch (lt_moments_now_static)             */
};

/* Ring / RF parameters: BASELINE.json:north_star (1) "(C, gamma, alpha_c, h, V, phi_s,
 * integrator)" plus p0 and the charge that A needs (configs[0]) and the second-harmonic
 * amplitude ratio (configs[4]). */
typedef struct {
    double circumference_m; /* C [m]                                             */
    double gamma;           /* Lorentz gamma (> 1); beta is derived from it       */
    double alpha_c;         /* momentum compaction factor                         */
    double p0c_eV;          /* reference momentum times c [eV]                    */
    double charge_e;        /* q in units of e (1 for protons)                    */
    int    harmonic;        /* h (> 0)                                            */
    double voltage_V;       /* V [volt]                                           */
    double phi_s;           /* synchronous phase [rad]; 0 in every BASELINE config */
    double ratio2;          /* r: amplitude ratio of the harmonic at 2h; 0 = off   */
    int    integrator;      /* lt_integrator                                      */
} lt_params;

/* Derived constants (notation of DESIGN.md): filled by lt_derived(). */
typedef struct {
    double R;      /* C/(2 pi)                                                   */
    double beta;   /* sqrt(1 - 1/gamma^2)                                        */
    double eta;    /* alpha_c - 1/gamma^2                                        */
    double A;      /* q V / (beta p0c)                                           */
    double d;      /* eta C / 2                                                  */
    double kappa;  /* h / R                                                      */
    double K;      /* eta C A h / R  (single-harmonic, phi_s = 0)                */
    double mu;     /* arccos(1 - K/2): exact leap-frog / Euler-Cromer tune [rad] */
    double z_max;  /* pi R / h                                                   */
    double H_sep;  /* 2 A R / h                                                  */
} lt_derived_t;

/* Bunch moments of one state (BASELINE.json:configs[3]: "per-turn mean and rms of z and
 * delta"): population rms about the mean over all n particles (G14), the z-delta
 * covariance, and the bucket-membership count of the same state (north_star). */
typedef struct {
    double mean_z, rms_z, mean_d, rms_d, cov_zd;
    unsigned long long n_in_bucket;
} lt_moments;

/* Raw sums behind lt_moments; additive over disjoint particle ranges, which is what a
 * multi-GPU run all-reduces. */
typedef struct {
    double n;                       /* particle count (as double so one SUM all-reduce does it) */
    double sum_z, sum_zz, sum_d, sum_dd, sum_zd;
    double n_in_bucket;             /* exact for counts < 2^53 */
    double pad_;                    /* keeps sizeof == 64 */
} lt_sums;

/* Options for lt_set_option / lt_get_option. */
enum {
    LT_OPT_SPLIT_DRIFTS   = 1, /* 0 (default): fused mode merges the trailing half drift of a
                                  turn with the leading one of the next (one FMA with 2d);
                                  1: every half drift is its own FMA, bit-identical to the
                                  per-turn kernel and to any chunking by the caller.       */
    LT_OPT_CHUNK_TURNS    = 2, /* turns per fused kernel launch (default 2^22); the result
                                  of one call does not depend on it     */
    LT_OPT_FUSED_ILP      = 3, /* particles per lane in fused mode: 0 = planner decides; 1, 2 for
                                  the persistent kernels (fp32: PAIRS of particles per lane, the
                                  arithmetic is packed two to a value), 1, 2, 4 for the plain one,
                                  1, 2, 4, 8 for the fused transverse kernel (other kernels read 8
                                  as 0)                                                            */
    LT_OPT_FUSED_BLOCK    = 4, /* threads per block in fused mode: 0 = planner decides     */
    LT_OPT_PER_TURN_GRAPH = 5, /* 1 (default): per-turn launches are replayed from a CUDA
                                  graph in batches; 0: plain stream launches               */
    LT_OPT_PER_TURN_CTAS_PER_SM = 6, /* CTAs per SM of the per-turn kernels' grid; 0 (default):
                                  planner -- 6 up to 1.5e7 particles, 12 beyond; 1..32 forces it */
    LT_OPT_PER_TURN_REVERSE = 7, /* 1 (default): odd turns walk the arrays backwards so the
                                  tail the previous turn left in L2 is read first          */
    LT_OPT_FUSED_MODE     = 8, /* 0 (default): planner picks the persistent kernel's schedule;
                                  1: plain one-thread-per-particle kernel (LT_OPT_FUSED_ILP /
                                  _BLOCK apply); 2: static slots (group g on slot g mod slots for
                                  all turns); 3: on-device ticket queue of work items; 4: static
                                  wrap-around schedule (needs at least as many groups as slots,
                                  else static slots).  Same bits in every mode.               */
    LT_OPT_ITEM_TURNS     = 9, /* turns per work item of the dynamic persistent kernel
                                  (0 = planner: 128..2048; the last items of a launch are halved
                                  again and again); results do not depend on it                    */
    LT_OPT_WARPS_PER_SMSP = 10,/* resident warps per SM sub-partition of the persistent kernel
                                  (0 = planner; 1..8, or even values up to 16; with two particles
                                  per lane at most 4).  Forced options that admit no launch shape
                                  together are given up in a fixed order -- FUSED_MODE 4 -> 2, then
                                  FUSED_ILP 2 -> planner (the warp count is kept), then all of them
                                  -- and LT_STAT_LAST_* report what was launched                    */
    LT_OPT_FLIP_ON_Q      = 11,/* where the sign of the reduced sine is applied: -1 planner,
                                  0 on the argument, 1 on the polynomial; same bits either way */
    LT_OPT_RAMP_SCALED    = 12,/* lt_track_ramp, merged drifts: 1 (default) carries delta divided by
                                  the running kick amplitude (15 FP64 instructions per sub-step,
                                  four table values) unless a voltage scale of the call is zero, not
                                  finite or beyond 1e+-100 (scanned on the device, per call);
                                  0 always the plain form (16 instructions, five values).  The two
                                  round differently (both far inside the 1e-9 gate).              */
    LT_OPT_LATTICE_SOURCE = 13 /* where the fused transverse kernel keeps the lattice: 0 (default)
                                  planner -- the kernel-parameter space (constant bank, uniform
                                  registers) for lattices of at most 24 segments, else shared
                                  memory; 1 shared memory; 2 parameter space (longer lattices
                                  still use shared memory).  Same bits either way.              */
};

/* Counters for lt_get_stat. */
enum {
    LT_STAT_KERNEL_LAUNCHES = 1, /* kernels launched by this tracker since creation        */
    LT_STAT_LAST_GRID       = 2, /* grid / block / ilp of the last fused launch            */
    LT_STAT_LAST_BLOCK      = 3,
    LT_STAT_LAST_ILP        = 4, /* particles per lane of the last fused launch             */
    LT_STAT_SM_COUNT        = 5,
    LT_STAT_LAST_MODE       = 6, /* 1 plain, 2 static slots, 3 ticket queue, 4 wrap-around         */
    LT_STAT_LAST_ITEM_TURNS = 7
};

/* -- lifetime ------------------------------------------------------------------------ */

/* Validates p, derives the constants, allocates the handle.  Touches no GPU. */
int lt_create(const lt_params *p, lt_tracker **out);
int lt_destroy(lt_tracker *tr); /* frees the handle and its device scratch; NULL is LT_OK */
int lt_derived(const lt_tracker *tr, lt_derived_t *out);
int lt_set_option(lt_tracker *tr, int option, long long value);
int lt_get_option(const lt_tracker *tr, int option, long long *value);
int lt_get_stat(const lt_tracker *tr, int stat, long long *value);
const char *lt_strerror(int code);
int lt_last_cuda_error(const lt_tracker *tr); /* cudaError_t of the last LT_E_CUDA, else 0 */
int lt_version(void);

/* -- fused multi-turn mode ("a single thread contains a long enough loop to
 *    make use of the registers [...] and circumvent memory access") ------------------------
 * Advances every particle by `turns` turns.  z/delta are read once at entry and written once
 * at exit of each chunk (LT_OPT_CHUNK_TURNS); FP64-pipe bound. */
int lt_track_fused(lt_tracker *tr, double *z_dev, double *delta_dev, size_t n,
                   unsigned long long turns, void *stream);
int lt_track_fused_f32(lt_tracker *tr, float *z_dev, float *delta_dev, size_t n,
                       unsigned long long turns, void *stream);

/* -- per-turn mode ("each GPU thread advances the corresponding particle by one
 *    turn"; BASELINE.json:configs[3]) -----------------------------------------------------
 * One kernel launch per turn; each reads and writes z/delta (32 B per particle-turn in fp64)
 * and reduces the turn's moments in the same pass.  moments_dev / sums_dev: [turns] entries
 * or NULL; entry t describes the state AFTER turn t+1.  In the fp32 variant the state is
 * fp32 and the sums are accumulated in fp64.  HBM-bandwidth bound. */
int lt_track_per_turn(lt_tracker *tr, double *z_dev, double *delta_dev, size_t n,
                      unsigned long long turns, lt_moments *moments_dev, lt_sums *sums_dev,
                      void *stream);
int lt_track_per_turn_f32(lt_tracker *tr, float *z_dev, float *delta_dev, size_t n,
                          unsigned long long turns, lt_moments *moments_dev,
                          lt_sums *sums_dev, void *stream);

/* -- observables of the current state ---------------------------------------------------- */

/* Bucket membership (BASELINE.json:north_star "bucket-membership counts (exact)";
 * DESIGN.md G15): count_dev[0] = #{ i : |z_i| < z_max  and  H(z_i, delta_i) < H_sep } with
 *     H(z, delta) = eta C delta^2 / 2 + (A R / h) [(1 - cos kappa z) + (r/2)(1 - cos 2 kappa z)],
 *     z_max = pi R / h,  H_sep = 2 A R / h
 * -- the STATIONARY bucket of phi_s = 0 with -1/2 <= r <= 1/2, which is every BASELINE config.
 * The same predicate fills n_in_bucket of lt_moments / lt_sums everywhere.  Outside that range
 * it is still evaluated as written but is no longer "the bucket": for phi_s != 0 the bucket is
 * asymmetric and smaller, for |r| > 1/2 the potential has extra extrema inside +-z_max; with
 * A = 0 (no RF) H_sep = 0 and the count is 0. */
int lt_bucket_count(lt_tracker *tr, const double *z_dev, const double *delta_dev, size_t n,
                    unsigned long long *count_dev, void *stream);
int lt_bucket_count_f32(lt_tracker *tr, const float *z_dev, const float *delta_dev, size_t n,
                        unsigned long long *count_dev, void *stream);
/* Moments of the current state (no tracking); either output may be NULL. */
int lt_moments_now(lt_tracker *tr, const double *z_dev, const double *delta_dev, size_t n,
                   lt_moments *moments_dev, lt_sums *sums_dev, void *stream);

/* lt_moments_now for callers that must not allocate device memory.
 *
 * Why it exists: lt_moments_now keeps its per-CTA partial sums in a tracker-owned buffer that
 * its first call on a tracker (and any later call with a larger grid) takes from
 * cudaMallocAsync.  Not every user of this library may do that -- a long-running tracking
 * service that gives the whole GPU to its own memory pool at start-up leaves nothing for the
 * driver's allocator; a turn-by-turn monitor at an interaction point must not
 * stall on, or fail in, an allocation in the middle of a run; a plug-in inside somebody else's
 * application may simply be forbidden to touch the CUDA heap.  This call computes the same
 * observables (same predicate, same sums, fp64 accumulation; either output may be NULL, not
 * both) and calls no cudaMalloc*, no cudaFree* and no library routine that allocates.
 *
 * How: the partial sums live in a fixed 128 KB array (`static __device__`, 256-byte aligned)
 * that is part of the library image, one 64-byte record per 8192 particles.  Every GPU on which
 * this library is loaded holds that array from load until the process exits, used or not.
 *
 * Limit: n <= LT_STATIC_MAX_PARTICLES (2^24 = 16 777 216, enough for BASELINE.json:configs[3]).
 * A larger n returns LT_E_CAPACITY and enqueues nothing; use lt_moments_now there.
 *
 * Set-up: the FIRST call on each device asks the runtime once for the array's device address
 * (cudaGetSymbolAddress, with that device current; a failure is LT_E_CUDA) and keeps it for
 * the life of the process.  Make that first call during initialisation, before any stream
 * capture is begun.  The current device must be the one z_dev / delta_dev live on, as for every
 * other call; at most 64 devices per process (beyond that LT_E_PARAM).
 *
 * Sharing: there is ONE array per GPU for the whole process -- all trackers, all streams, all
 * host threads.  It keeps what the previous call left in it; that is harmless, because each call
 * writes every record it later reads and nothing has to start at zero.  But two calls whose
 * kernels overlap on the same GPU (different streams, or different host threads on unordered
 * streams) RACE on it and both results are garbage: order such calls on one stream or with
 * events.  Calls on different GPUs do not interact.
 *
 * Results agree with lt_moments_now to rounding (the partition of the sum differs: ~1e-15
 * relative on the sums); n_in_bucket is the same integer.  n == 0 writes all-zero outputs.
 * Two launches on `stream`; asynchronous like every device call. */
#define LT_STATIC_MAX_PARTICLES (1 << 24)
int lt_moments_now_static(lt_tracker *tr, const double *z_dev, const double *delta_dev, size_t n,
                          lt_moments *moments_dev, lt_sums *sums_dev, void *stream);

/* Host helper: turns `count` raw sums (e.g. after an all-reduce over ranks) into moments. */
int lt_moments_from_sums(const lt_sums *sums_host, size_t count, lt_moments *out_host);

/* -- host-buffer entry point (the paper's long_tracking_cu flow, PAPER.md:242-260:
 *    cudaMalloc, cudaMemcpyHostToDevice, kernel, cudaMemcpyDeviceToHost) ------------------
 * z_host/delta_host: n doubles each (pinned memory makes the copies asynchronous but is not
 * required).  Uses an internal stream and staging buffers kept by the tracker; returns after
 * the results are in the host arrays.  count_host may be NULL; if not, it receives the
 * bucket-membership count of the final state. */
int lt_track_fused_host(lt_tracker *tr, double *z_host, double *delta_host, size_t n,
                        unsigned long long turns, unsigned long long *count_host);

/* ========================================================================================
 * Rows SURVEY.md sec. 8(f) marks "next" (fp64 only).  The paper prints no formula for any of
 * them; the readings are DESIGN.md G28-G30.
 * ======================================================================================== */

/* -- f2: turn-dependent RF programme (sec. 2.2: the "parameter changes of the
 *    accelerator setting (as in the above hollow bunch setting)" that the paper's C/CUDA
 *    extraction left out; G28) ----------------------------------------------------
 * volt_scale_dev[t], phase_off_dev[t] (device, `turns` doubles each; t = 0-based) apply to
 * EVERY kick of turn t+1 (Ruth4: all three sub-kicks):
 *     F_t(z) = a_t A [ sin(phi_s + kappa z + psi_t) - sin(phi_s) + r sin(2 (kappa z + psi_t)) ]
 * a_t = volt_scale[t] = V_t / V (dimensionless), psi_t = phase_off[t] [rad].  a_t = 1, psi_t = 0
 * is the plain map.  The tables are read while the call's work runs: keep them unchanged until
 * the stream has been synchronised.  lt_track_programme is the fused multi-turn mode (state in
 * registers, FP64-pipe bound, 15 instead of 13 FP64 instructions per particle-turn);
 * lt_track_programme_per_turn is the per-turn mode with the same outputs as lt_track_per_turn. */
int lt_track_programme(lt_tracker *tr, double *z_dev, double *delta_dev, size_t n,
                       unsigned long long turns, const double *volt_scale_dev,
                       const double *phase_off_dev, void *stream);
int lt_track_programme_per_turn(lt_tracker *tr, double *z_dev, double *delta_dev, size_t n,
                                unsigned long long turns, const double *volt_scale_dev,
                                const double *phase_off_dev, lt_moments *moments_dev,
                                lt_sums *sums_dev, void *stream);

/* -- f2 with acceleration: energy ramp ("V, phi_s, gamma ramps per
 *    turn from small device tables [...] gives acceleration"; G32) --------
 * p0c_dev[0 .. turns] (device, turns + 1 doubles, eV, all > 0): the reference momentum x c BEFORE
 * turn 1 and AFTER every turn.  volt_scale_dev / phase_off_dev as above, or NULL for a_t = 1 /
 * psi_t = 0.  With the rest energy mc2 = p0c_eV / (beta gamma) of lt_params and, for a reference
 * momentum p,  bg = p/mc2, beta = bg/sqrt(1 + bg^2), eta = alpha_c - 1/(1 + bg^2),
 * A(p) = q V/(beta p), d(p) = eta C/2,  one leap-frog sub-step with factor tau that takes the
 * reference from pb to pa is
 *     z     -= tau d(pb) delta
 *     delta  = (delta + tau a_t A(pb) [sin(kappa z + psi_t) + r sin(2 (kappa z + psi_t))]
 *               - (pa - pb)/pb) * (pb/pa)
 *     z     -= tau d(pa) delta
 * Turn t+1 (pb = p0c[t], pa = p0c[t+1], D = pa - pb): leap-frog = sub-step(1, pb, pa);
 * Euler-Cromer = the kick line (old z), then z -= 2 d(pa) delta; Ruth4 = sub-steps x1, x0, x1 over
 * pb -> pb + x1 D -> (that) + x0 D -> pa.  A particle at z = 0, delta = 0 stays on the reference iff
 * a_t A(pb) sin(psi_t) = D/pb: the caller programmes the synchronous phase through psi_t, so
 * lt_params.phi_s must be 0 here (else LT_E_PARAM).  The tracker's own parameters are not changed
 * by the call.  lt_track_ramp: fused multi-turn mode (16 FP64 instructions per sub-step);
 * lt_track_ramp_per_turn: per-turn mode with the outputs of lt_track_per_turn (n_in_bucket is the
 * stationary-bucket predicate of lt_params, whatever the ramp does; at most 2^26 turns per call,
 * else LT_E_PARAM: the whole call's table is packed at once).  The tables are read while the
 * call's work runs: keep them unchanged until the stream has been synchronised. */
int lt_track_ramp(lt_tracker *tr, double *z_dev, double *delta_dev, size_t n,
                  unsigned long long turns, const double *p0c_dev, const double *volt_scale_dev,
                  const double *phase_off_dev, void *stream);
int lt_track_ramp_per_turn(lt_tracker *tr, double *z_dev, double *delta_dev, size_t n,
                           unsigned long long turns, const double *p0c_dev,
                           const double *volt_scale_dev, const double *phase_off_dev,
                           lt_moments *moments_dev, lt_sums *sums_dev, void *stream);

/* -- f4: longitudinal slicing at the interaction point (sec. 1.1: "the fields of
 *    the particle distribution are constructed"; the memory-bound regime;
 *    DESIGN.md G29) ---------------------------------------------------------------------------
 * Uniform slices of z over [z_lo, z_hi), inv = n_slices / (z_hi - z_lo) in fp64:
 *     z < z_lo        -> hist[0]             ("below")
 *     not (z < z_hi)  -> hist[n_slices + 1]  ("above"; NaN lands here)
 *     otherwise          u = (z - z_lo) * inv (two roundings, no FMA); s = floor(u) clamped to
 *                        n_slices - 1;  hist[1 + s]
 * hist_dev has n_slices + 2 counters (unsigned 64-bit) per histogram and is OVERWRITTEN.
 * Requires z_lo < z_hi (finite) and 1 <= n_slices <= 2^20, else LT_E_PARAM.
 * lt_slice_histogram: histogram of a given state.  lt_track_slices: per-turn mode -- one launch
 * per turn tracks the turn and, in the same pass over HBM, fills hist_dev[t * (n_slices + 2) ..]
 * with the histogram of z AFTER turn t+1 (t = 0 .. turns-1); moments_dev / sums_dev as in
 * lt_track_per_turn, or NULL. */
int lt_slice_histogram(lt_tracker *tr, const double *z_dev, size_t n, double z_lo, double z_hi,
                       int n_slices, unsigned long long *hist_dev, void *stream);
int lt_track_slices(lt_tracker *tr, double *z_dev, double *delta_dev, size_t n,
                    unsigned long long turns, double z_lo, double z_hi, int n_slices,
                    unsigned long long *hist_dev, lt_moments *moments_dev, lt_sums *sums_dev,
                    void *stream);

/* -- f3: transverse plane (sec. 1.1.1: "linear transfer matrices, i.e. the same
 *    matrix is repeatedly acting on the typically 10^5 to 10^7 macro-particles' state vectors";
 *    Fig. 2: pushed "from one interaction point to another"; G30) --------
 * lt_set_transverse: the lattice, n_seg (1..256) 4x4 matrices in HOST memory, ROW-MAJOR,
 * matrices_host[16 s + 4 i + j] = (M_s)_ij; copied by the call (n_seg = 0 clears it).
 * One turn = for s = 0 .. n_seg-1 in order: u <- M_s u with u = (x, x', y, y'), row i evaluated
 * left to right, ((M_i0 x + M_i1 x') + M_i2 y) + M_i3 y' (the library uses FMAs in that order);
 * then the longitudinal turn of (z, delta) by the tracker's map.  The planes are not coupled.
 * x/xp/y/yp (and z/delta) are separate device arrays of n doubles, updated in place; z_dev and
 * delta_dev may both be NULL (transverse plane only).  Without a lattice: LT_E_PARAM.
 * _fused: `turns` turns with the state in registers (FP64-pipe bound, 16 FP64 instructions per
 * segment and particle); _per_turn: one launch per turn, every coordinate through HBM (64 B per
 * particle-turn, 96 B with the longitudinal plane; HBM bound). */
int lt_set_transverse(lt_tracker *tr, const double *matrices_host, int n_seg);
int lt_track_transverse_fused(lt_tracker *tr, double *x_dev, double *xp_dev, double *y_dev,
                              double *yp_dev, double *z_dev, double *delta_dev, size_t n,
                              unsigned long long turns, void *stream);
int lt_track_transverse_per_turn(lt_tracker *tr, double *x_dev, double *xp_dev, double *y_dev,
                                 double *yp_dev, double *z_dev, double *delta_dev, size_t n,
                                 unsigned long long turns, void *stream);

/* -- introspection of the host logic (no GPU needed; what the CPU tests call) ---------------
 * lt_plan_fused: the launch shape lt_track_fused would pick for n particles and `turns` turns on
 * a device with sm_count SMs (options of the tracker apply): plan[0] = 1 dynamic work queue / 0
 * static slots, plan[1] = warps per sub-partition, plan[2] = CTAs per SM, plan[3] = threads per
 * CTA, plan[4] = turns per work item (0 = all), plan[5] = sign flip on q, plan[6] = particles per
 * lane (fp32: pairs count double).
 * lt_item_schedule: the tapered work-item schedule of a launch: number of
 * chunks, and first turn / length of chunk c (c >= *nchunks: LT_E_PARAM). */
int lt_plan_fused(const lt_tracker *tr, size_t n, unsigned long long turns, int sm_count, int fp32,
                  long long plan[7]);
int lt_item_schedule(unsigned int turns, unsigned int item_turns, int taper, unsigned int c,
                     unsigned int *nchunks, unsigned int *start, unsigned int *len);

#ifdef __cplusplus
}
#endif
#endif /* LONGTRACK_H */
