// kernels_ramp.cuh -- sm_100a device code for the ENERGY RAMP of SURVEY.md sec. 8(f) row f2
// ("V, phi_s, gamma ramps per turn from small device tables"; G32).
// CUDA path only: shares nothing with oracle/.
//
// The reference momentum goes p0c[t] -> p0c[t+1] over turn t+1, which makes beta, eta, the kick
// amplitude A and the drift coefficient d functions of the turn, and re-expresses delta relative
// to the new reference after every kick.  A turn is a sequence of SUB-STEPS (1 for leap-frog and
// Euler-Cromer, 3 for Ruth4), each
//     z -= db delta;   delta = g (delta + amp [sin(kappa z + psi) + r sin(2(kappa z + psi))]) + c;
//     z -= da delta
// with amp = tau a_t A(p_b), g = p_b/p_a, c = -(p_a - p_b)/p_a, db = tau d(p_b), da = tau d(p_a)
// (Euler-Cromer: db = 0, da = 2 d(p_a)).  ramp_pack_kernel turns the caller's tables into one
// 48-byte entry per sub-step; the tracking kernels are then generic in the integrator.
// The kick line is evaluated as  delta = (g amp) [..] + (g delta + c):  the product g*amp comes
// from the pack kernel, f*(g amp) and g*delta + c run BESIDE the Horner chain, and the last FMA
// of the sine is the whole update -- the dependent chain of a sub-step is 14 FP64 instructions
// of its 17 (it was 16 with q*amp, the kick FMA and the damping FMA in a row).
#pragma once

#include "kernels.cuh"

namespace lt {

// One sub-step, 48 bytes = three double2.
//   exact layout (split drifts, per-turn kernel):  p = psi/pi;  d0 = db, d1 = da      (metres)
//   fast layout (merged drifts, state = phase u = v + p INCLUDING the sub-step's RF phase offset):
//       p  = (psi of the NEXT sub-step - psi of this one)/pi, minus the last psi/pi at the end of
//            the API call, so that the offset is one DADD beside the sine chain and the state
//            leaves the call as the plain phase;
//       d0 = (da + db of the NEXT sub-step) kappa/pi,  d1 = db kappa/pi (the call's first sub-step)
//   The fast table starts with a header entry whose p is the absolute psi/pi of its first sub-step.
struct RampEntry {
    double ga, p;       // g * kick amplitude; RF phase offset in half periods (see the layouts)
    double g, c;        // delta <- g * (delta + kick) + c
    double d0, d1;
};

// SCALED fast layout (round 2): the fused kernel carries  y = delta / lambda_K  instead of delta,
// with lambda_0 = 1 and lambda_(K+1) = g_K amp_K, the scale in effect after sub-step K.  Then
//     y' = (lambda_K / amp_K) y + c_K / lambda_(K+1) + [sin(pi u) + r sin(2 pi u)]
// -- the kick amplitude has left the kick: no f * ga multiply, FOUR table values per sub-step
// instead of five (two 16-byte shared-memory loads instead of three), 15 FP64 instructions
// instead of 16.  The drift coefficient carries the scale: u' = (u + dp) - (d0 lambda_(K+1)) y'.
// Needs amp_K != 0 for every sub-step of the call: a scan of the voltage table decides per CALL
// between this layout and the plain fast layout above (ramp_scan_kernel, *flag != 0: plain).
// Header entry: dp = absolute psi/pi of the launch's first sub-step, C = lambda after the
// launch's LAST sub-step (delta = y * C at the end of a call), D = leading drift of the call.
struct RampScaled {
    double G, dp;       // lambda_K / amp_K;  RF phase offset difference to the next sub-step (half periods)
    double C, D;        // c_K / lambda_(K+1);  merged drift coefficient times lambda_(K+1)
};

struct RampRing {
    double mc2, alpha_c, qV, C;   // rest energy (eV), momentum compaction, q V (eV), circumference
    double x1, x0;                // Ruth4 step factors
    double to_phase, inv_pi;      // kappa/pi, 1/pi
};

__device__ __forceinline__ void ramp_ring_at(const RampRing& R, double p, double* A, double* d) {
    const double bg = p / R.mc2;
    const double g2 = __fma_rn(bg, bg, 1.0);
    const double beta = bg / sqrt(g2);
    const double eta = R.alpha_c - 1.0 / g2;
    *A = R.qV / (beta * p);
    *d = eta * R.C * 0.5;
}

// Momenta, kick amplitudes and drift coefficients of the sub-steps of ONE turn (reference
// pb -> pa, voltage scale av): ps[0..nsub], A[..], d[..] at those momenta, tau[0..nsub-1].
struct RampTurn { double ps[4], A[4], d[4], tau[3]; int nsub; };
__device__ __forceinline__ void ramp_turn_at(const RampRing& R, double pb, double pa, int integ, RampTurn* t) {
    t->nsub = integ == kRuth4 ? 3 : 1;
    t->ps[0] = pb;
    if (t->nsub == 3) {
        const double D = pa - pb;
        t->ps[1] = __fma_rn(R.x1, D, pb);
        t->ps[2] = __fma_rn(R.x0, D, t->ps[1]);
        t->ps[3] = pa;
        t->tau[0] = R.x1; t->tau[1] = R.x0; t->tau[2] = R.x1;
    } else {
        t->ps[1] = pa;
        t->tau[0] = 1.0; t->tau[1] = 0.0; t->tau[2] = 0.0;
    }
    for (int k = 0; k <= t->nsub; ++k) ramp_ring_at(R, t->ps[k], &t->A[k], &t->d[k]);
}
// g = p_b/p_a and g * amp of sub-step k (the scale lambda in effect after it)
__device__ __forceinline__ double ramp_g(const RampTurn& t, int k) { return t.ps[k] / t.ps[k + 1]; }
__device__ __forceinline__ double ramp_ga(const RampTurn& t, int k, double av) {
    return ramp_g(t, k) * (t.tau[k] * t.A[k] * av);
}

// *flag |= 1 when any voltage scale of the call is zero, not finite or beyond 1e+-100 (the scaled
// layout divides by the kick amplitude)
static __global__ void ramp_scan_kernel(const double* __restrict__ volt, unsigned long long turns,
                                        unsigned int* __restrict__ flag) {
    bool zero = false;
    for (unsigned long long i = (unsigned long long)blockIdx.x * blockDim.x + threadIdx.x; i < turns;
         i += (unsigned long long)gridDim.x * blockDim.x)
        zero |= !(fabs(volt[i]) > 1e-100 && fabs(volt[i]) < 1e100);   // zero, NaN, or so extreme that delta / amp could leave the fp64 range
    if (__syncthreads_or(zero) && threadIdx.x == 0) atomicOr(flag, 1u);
}

// One thread per turn of the launch.  p0c / volt / phase are the CALL's tables (volt, phase may be
// nullptr), t_first the absolute index of the launch's first turn, call_turns the call's length
// (the trailing drift of the call's last sub-step is not merged with anything).
// fast = 1: the plain fast layout into `out`; and, when out2 != nullptr, the scaled layout into out2.
static __global__ void ramp_pack_kernel(const double* __restrict__ p0c, const double* __restrict__ volt,
                                 const double* __restrict__ phase, unsigned long long t_first,
                                 unsigned int count, unsigned long long call_turns, int integ,
                                 int fast, const __grid_constant__ RampRing R,
                                 RampEntry* __restrict__ out, RampScaled* __restrict__ out2) {
    const unsigned int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= count) return;
    const unsigned long long T = t_first + i;
    const double pb = p0c[T], pa = p0c[T + 1];
    const double av = volt ? volt[T] : 1.0;
    const double psi = phase ? phase[T] : 0.0;
    const double psi_next = (phase && T + 1 < call_turns) ? phase[T + 1] : 0.0;
    RampTurn t;
    ramp_turn_at(R, pb, pa, integ, &t);
    const int nsub = t.nsub;
    const double* ps = t.ps; const double* A = t.A; const double* d = t.d; const double* tau = t.tau;
    const double tau_first = integ == kEulerCromer ? 0.0 : tau[0];
    const double p_here = __dmul_rn(psi, R.inv_pi);
    RampEntry* dst = out + (fast ? 1 : 0);                 // fast layout: behind the header entry
    if (fast && i == 0) {
        RampEntry h;
        h.ga = 0.0; h.p = p_here; h.g = 1.0; h.c = 0.0; h.d0 = 0.0; h.d1 = 0.0;
        out[0] = h;
    }
    // scaled layout: the scale in effect before this turn's first sub-step is the one the previous
    // turn's last sub-step left (recomputed here with the same function: the same bits)
    double lam = 1.0;
    if (fast && out2 && T > 0) {
        RampTurn prev;
        ramp_turn_at(R, p0c[T - 1], pb, integ, &prev);
        lam = ramp_ga(prev, prev.nsub - 1, volt ? volt[T - 1] : 1.0);
    }
    for (int k = 0; k < nsub; ++k) {
        RampEntry e;
        e.g = ramp_g(t, k);
        e.ga = ramp_ga(t, k, av);
        e.p = p_here;
        e.c = -(ps[k + 1] - ps[k]) / ps[k + 1];
        double db = tau[k] * d[k], da = tau[k] * d[k + 1];
        if (integ == kEulerCromer) { db = 0.0; da = 2.0 * d[1]; }
        if (fast) {
            double db_next;
            if (k + 1 < nsub) db_next = tau[k + 1] * d[k + 1];
            else db_next = (T + 1 == call_turns) ? 0.0 : tau_first * d[nsub];
            e.d0 = (da + db_next) * R.to_phase;
            e.d1 = db * R.to_phase;
            // every sub-step of a turn sees the same psi: the offset changes behind the last one
            e.p = (k + 1 < nsub) ? 0.0 : __dsub_rn(__dmul_rn(psi_next, R.inv_pi), p_here);
            if (out2) {
                RampScaled q;
                const double amp = tau[k] * A[k] * av;
                const double lam_next = e.ga;              // g_K amp_K
                q.G = lam / amp;
                q.dp = e.p;
                q.C = e.c / lam_next;
                q.D = e.d0 * lam_next;
                out2[1 + (size_t)i * nsub + k] = q;
                if (i == 0 && k == 0) { out2[0].G = 0.0; out2[0].dp = p_here; out2[0].D = e.d1; }
                lam = lam_next;
            }
        } else {
            e.d0 = db;
            e.d1 = da;
        }
        dst[(size_t)i * nsub + k] = e;
    }
    if (fast && out2 && i == count - 1) out2[0].C = lam;   // the scale the launch leaves: delta = y * lam
}

static __global__ void ramp_advance_cursor_kernel(unsigned long long* cursor, unsigned long long by) {
    *cursor += by;
}

// delta <- g (delta + amp F) + c  for the phase v (half periods, psi already added):
//     fma(+-f ga, sin(pi f)/f [(1 + 2 r cos(pi f))], fma(g, delta, c)),   ga = g amp
template <int HARM>
__device__ __forceinline__ double ramp_kick(double v, double dl, const MapConsts<double>& P,
                                            double ga, double g, double c) {
    typedef Real<double> R;
    double t;
    const double f = reduce_half_periods(v, &t);
    const double s = __dmul_rn(f, f);
    const double fa = __dmul_rn(f, ga);
    const double base = __fma_rn(g, dl, c);
    double q = horner<double, R::NS>(P.sin1, s);
    if (HARM == 2) {
        const double cc = horner<double, R::NC>(P.cos1, s);
        q = __dmul_rn(q, __fma_rn(P.two_r, cc, R::sign_of(t)));      // one sign for sine and cosine (kick<> in kernels.cuh)
        return __fma_rn(fa, q, base);
    }
    return __fma_rn(R::flip(fa, t), q, base);
}

// exact sub-step: state z, every drift its own FMA (bit-identical between the fused split-drift
// kernel, the per-turn kernel and any chunking)
template <int HARM>
__device__ __forceinline__ void ramp_substep_exact(double& z, double& dl, const MapConsts<double>& P,
                                                   double ga, double p, double g, double c,
                                                   double db, double da) {
    z = __fma_rn(-db, dl, z);
    dl = ramp_kick<HARM>(__fma_rn(z, P.to_phase, p), dl, P, ga, g, c);
    z = __fma_rn(-da, dl, z);
}

// fast sub-step: state u = v + p (phase in half periods including the RF phase offset), trailing
// drift merged with the next leading one.  16 FP64 instructions (single harmonic): 3 reduction,
// f^2, f * ga, g * delta + c, u + dp, 7 Horner, the kick FMA, the drift FMA; 13 of them on the
// dependent chain (reduction, f^2, Horner, kick, drift).
template <int HARM>
__device__ __forceinline__ void ramp_substep_fast(double& u, double& dl, const MapConsts<double>& P,
                                                  double ga, double dp, double g, double c, double dm) {
    const double w = __dadd_rn(u, dp);
    dl = ramp_kick<HARM>(u, dl, P, ga, g, c);
    u = __fma_rn(-dm, dl, w);
}

// scaled fast sub-step (RampScaled): state (u, y = delta / lambda_K); 15 FP64 instructions (single
// harmonic): u + dp, 3 reduction, f^2, G y + C, 7 Horner, the kick FMA, the drift FMA
template <int HARM>
__device__ __forceinline__ void ramp_substep_scaled(double& u, double& y, const MapConsts<double>& P,
                                                    double G, double dp, double C, double D) {
    typedef Real<double> R;
    const double w = __dadd_rn(u, dp);
    double t;
    const double f = reduce_half_periods(u, &t);
    const double s = __dmul_rn(f, f);
    const double base = __fma_rn(G, y, C);
    double q = horner<double, R::NS>(P.sin1, s);
    if (HARM == 2) {
        const double cc = horner<double, R::NC>(P.cos1, s);
        q = __dmul_rn(q, __fma_rn(P.two_r, cc, R::sign_of(t)));
        y = __fma_rn(f, q, base);
    } else {
        y = __fma_rn(R::flip(f, t), q, base);
    }
    u = __fma_rn(-D, y, w);
}

__device__ __forceinline__ void cp_async_16(void* smem_dst, const void* gmem_src) {
    const unsigned int dst = (unsigned int)__cvta_generic_to_shared(smem_dst);
    asm volatile("cp.async.ca.shared.global [%0], [%1], 16;" ::"r"(dst), "l"(gmem_src) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
__device__ __forceinline__ void cp_async_wait_1() { asm volatile("cp.async.wait_group 1;" ::: "memory"); }

// `nsteps` sub-steps of the ILP particles of a lane; tab = the item's first entry as
// double2[E * nsteps] (E = 3 double2 per entry: RampEntry; E = 2, SCALED: RampScaled); stage = the
// warp's private double buffer in shared memory (2 x 32 entries = 3072 B / 2048 B).  While the warp
// works through one block of 32 entries, the next block arrives by
// cp.async (no registers held, no L2 latency on the dependent FP64 chain; a per-sub-step global
// load stalled the RF-programme kernel once per 128-byte line, profiles/r1_next_rows_ncu.md).
// hdr = the launch's header entry (SCALED: leading drift, absolute offset, final scale).
template <int HARM, bool SPLIT, int ILP, bool SCALED>
__device__ __forceinline__ void ramp_advance(double (&x)[ILP], double (&dl)[ILP], unsigned int nsteps,
                                             int first, int last, const MapConsts<double>& P,
                                             const double2* __restrict__ tab,
                                             const double2* __restrict__ hdr,
                                             double2* __restrict__ stage) {
    constexpr unsigned int E = SCALED ? 2u : 3u;
    const unsigned int lane = threadIdx.x & 31u;
    const unsigned int total2 = E * nsteps;
    auto fetch = [&](unsigned int t0, unsigned int buf) {
#pragma unroll
        for (int j = 0; j < (int)E; ++j) {
            const unsigned int idx = E * t0 + lane + 32u * j;
            if (idx < total2) cp_async_16(stage + 32u * E * buf + lane + 32u * j, tab + idx);
        }
        cp_async_commit();
    };
    fetch(0, 0);
    if (!SPLIT && first) {
        // header entry: absolute offset; leading drift of the call's first sub-step
        const double lead = SCALED ? __ldg(hdr + 1).y : __ldg(tab + 2).y;
        const double p0 = __ldg(hdr).y;
#pragma unroll
        for (int j = 0; j < ILP; ++j) {
            x[j] = __dmul_rn(x[j], P.to_phase);
            x[j] = __fma_rn(-lead, dl[j], x[j]);
            x[j] = __dadd_rn(x[j], p0);                 // SCALED: lambda_0 = 1, y = delta
        }
    }
    unsigned int buf = 0;
    for (unsigned int t0 = 0; t0 < nsteps; t0 += 32, buf ^= 1u) {
        fetch(t0 + 32u, buf ^ 1u);           // the block after this one (an empty group at the end)
        cp_async_wait_1();                   // this block has landed
        __syncwarp();
        const double2* __restrict__ cur = stage + 32u * E * buf;
        const unsigned int m = min(32u, nsteps - t0);
        // the whole staged block unrolled: LDS addresses become immediates and the loop's counter and
        // uniform-register reloads disappear (unroll 4 -> 32: 77.8 % -> 83.3 % of the FP64 peak)
        constexpr int kUnrollR = 32;
#pragma unroll kUnrollR
        for (unsigned int k = 0; k < m; ++k) {
            if (SCALED) {
                const double2 e0 = cur[2 * k], e1 = cur[2 * k + 1];
#pragma unroll
                for (int j = 0; j < ILP; ++j) ramp_substep_scaled<HARM>(x[j], dl[j], P, e0.x, e0.y, e1.x, e1.y);
            } else {
                const double2 e0 = cur[3 * k], e1 = cur[3 * k + 1], e2 = cur[3 * k + 2];
#pragma unroll
                for (int j = 0; j < ILP; ++j) {
                    if (SPLIT) ramp_substep_exact<HARM>(x[j], dl[j], P, e0.x, e0.y, e1.x, e1.y, e2.x, e2.y);
                    else ramp_substep_fast<HARM>(x[j], dl[j], P, e0.x, e0.y, e1.x, e1.y, e2.x);
                }
            }
        }
        __syncwarp();                        // all lanes are done with `buf` before it is refilled
    }
    if (!SPLIT && last) {
        const double lam = SCALED ? __ldg(hdr + 1).x : 1.0;
#pragma unroll
        for (int j = 0; j < ILP; ++j) {
            x[j] = __dmul_rn(x[j], P.from_phase);
            if (SCALED) dl[j] = __dmul_rn(dl[j], lam);
        }
    }
}

// Fused multi-turn kernel with the ramp: the persistent ticketed work queue of
// fused_persistent_kernel (kernels.cuh), work item = (chunk of item_steps sub-steps) x (32 particles).
// table = the launch's table INCLUDING its header entry (SPLIT: no header).  SCALED: RampScaled
// entries.  flag (may be nullptr) = the per-call choice between the two fast layouts, written by
// ramp_scan_kernel: the SCALED instantiation runs when *flag == 0, the plain one when *flag != 0;
// the other launch of the pair returns at once.
template <int HARM, bool SPLIT, int ILP, bool SCALED = false>
__global__ void __launch_bounds__(ILP == 1 ? 1024 : 512, 1)
ramp_persistent_kernel(double* __restrict__ z_arr, double* __restrict__ d_arr, size_t n,
                       unsigned int nsteps, unsigned int item_steps, int first_launch, int last_launch,
                       int dynamic, unsigned long long* __restrict__ ticket,
                       unsigned int* __restrict__ done, const __grid_constant__ MapConsts<double> P,
                       const double2* __restrict__ table_hdr, const unsigned int* __restrict__ flag) {
    extern __shared__ __align__(16) unsigned char ramp_smem[];   // 3072 B per warp + residency cap
    static_assert(!(SCALED && SPLIT), "the scaled layout is a fast-path layout");
    if (flag && ((*flag != 0u) == SCALED)) return;
    constexpr unsigned int E = SCALED ? 2u : 3u;
    const double2* __restrict__ table = table_hdr + (SPLIT ? 0u : E);
    constexpr unsigned int G = 32u * ILP;
    const unsigned int lane = threadIdx.x & 31u;
    const unsigned long long groups = (n + G - 1) / G;
    const unsigned long long slots = (unsigned long long)gridDim.x * (blockDim.x >> 5);
    const unsigned long long slot = (unsigned long long)(threadIdx.x >> 5) * gridDim.x + blockIdx.x;
    double2* stage = reinterpret_cast<double2*>(ramp_smem) + 192u * (threadIdx.x >> 5);

    // sub-steps [s_begin, s_begin + ns) of group g (see run_piece in kernels.cuh)
    auto run_piece = [&](unsigned long long g, unsigned int s_begin, unsigned int ns, unsigned int need,
                         unsigned int publish) {
        if (need) {
            while (ld_acquire_u32(done + g) < need) __nanosleep(64);
        }
        const size_t i0 = (size_t)g * G + lane;
        double x[ILP], dl[ILP];
#pragma unroll
        for (int j = 0; j < ILP; ++j) {
            const size_t i = i0 + 32u * j;
            x[j] = (i < n) ? __ldcg(z_arr + i) : 0.0;
            dl[j] = (i < n) ? __ldcg(d_arr + i) : 0.0;
        }
        const int first = first_launch && s_begin == 0;
        const int last = last_launch && s_begin + ns == nsteps;
        ramp_advance<HARM, SPLIT, ILP, SCALED>(x, dl, ns, first, last, P, table + E * (size_t)s_begin, table_hdr, stage);
#pragma unroll
        for (int j = 0; j < ILP; ++j) {
            const size_t i = i0 + 32u * j;
            if (i < n) { __stcg(z_arr + i, x[j]); __stcg(d_arr + i, dl[j]); }
        }
        if (publish) {
            __threadfence();
            __syncwarp();
            if (lane == 0) st_release_u32(done + g, publish);
        }
        __syncwarp();            // the warp is converged again before the next piece (see run_piece's callers)
    };

    if (dynamic == 2) {                       // wrap-around schedule, see fused_persistent_kernel
        const unsigned __int128 X = (unsigned __int128)groups * nsteps;
        const unsigned long long x_lo = (unsigned long long)(X * slot / slots);
        unsigned long long x = (unsigned long long)(X * (slot + 1) / slots);
        while (x > x_lo) {
            const unsigned long long g = (x - 1) / nsteps;
            const unsigned long long gx = g * (unsigned long long)nsteps;
            const unsigned int s_end = (unsigned int)(x - gx);
            const unsigned int s_begin = x_lo > gx ? (unsigned int)(x_lo - gx) : 0u;
            run_piece(__shfl_sync(0xffffffffu, g, 0), __shfl_sync(0xffffffffu, s_begin, 0),
                      __shfl_sync(0xffffffffu, s_end - s_begin, 0), s_begin ? 1u : 0u, s_end < nsteps ? 1u : 0u);
            x = gx + s_begin;
        }
        return;
    }

    ItemSchedule sched;
    sched.init(nsteps, item_steps, dynamic);
    const unsigned int nchunks = sched.nchunks;
    const unsigned long long total = groups * nchunks;
    unsigned long long next = slot;
    for (;;) {
        unsigned long long t = next;
        if (dynamic) {
            if (lane == 0) t = atomicAdd(ticket, 1ULL);
        } else {
            next += slots;
        }
        // in static mode too: the broadcast tells ptxas that the work item, and every loop below
        // it, is warp-uniform (counters and table addresses then live in uniform registers)
        t = __shfl_sync(0xffffffffu, t, 0);
        if (t >= total) break;
        const unsigned int c = (unsigned int)(t / groups);
        const unsigned long long g = t - (unsigned long long)c * groups;
        unsigned int s_start, ns;
        sched.span(c, dynamic, &s_start, &ns);
        run_piece(g, s_start, ns, c, nchunks > 1 ? c + 1 : 0u);
    }
}

// Per-turn mode with the ramp: the structure of per_turn_kernel (persistent CTAs, double2 tiles,
// all loads of a tile before its arithmetic, moments fused, sweep direction alternating), the
// turn's NSUB entries read once per thread from the packed table at turn *cursor + k.
template <int HARM, int NSUB, bool MOMENTS, bool VEC, int UNR>
__global__ void ramp_per_turn_kernel(double* __restrict__ z_arr, double* __restrict__ d_arr, size_t n,
                                     int reverse, double* __restrict__ partials,
                                     const __grid_constant__ MapConsts<double> P,
                                     const RampEntry* __restrict__ table,
                                     const unsigned long long* __restrict__ cursor, int k) {
    RampEntry e[NSUB];
    {
        const double2* src = reinterpret_cast<const double2*>(table + (*cursor + (unsigned long long)k) * NSUB);
#pragma unroll
        for (int s = 0; s < NSUB; ++s) {
            const double2 a = __ldg(src + 3 * s), b = __ldg(src + 3 * s + 1), c = __ldg(src + 3 * s + 2);
            e[s].ga = a.x; e[s].p = a.y; e[s].g = b.x; e[s].c = b.y; e[s].d0 = c.x; e[s].d1 = c.y;
        }
    }
    auto turn = [&](double& z, double& dl) {
#pragma unroll
        for (int s = 0; s < NSUB; ++s)
            ramp_substep_exact<HARM>(z, dl, P, e[s].ga, e[s].p, e[s].g, e[s].c, e[s].d0, e[s].d1);
    };
    Sums acc;
    acc.zero();
    if (VEC) {
        const size_t npair = n >> 1;
        const size_t tile_pairs = (size_t)blockDim.x * UNR;
        const size_t ntiles = (npair + tile_pairs - 1) / tile_pairs;
        for (size_t tl = blockIdx.x; tl < ntiles; tl += gridDim.x) {
            const size_t tix = reverse ? (ntiles - 1 - tl) : tl;
            const size_t base = tix * tile_pairs;
            double2 a[UNR], b[UNR];
#pragma unroll
            for (int u = 0; u < UNR; ++u) {
                const size_t p = base + (size_t)u * blockDim.x + threadIdx.x;
                if (p < npair) {
                    a[u] = reinterpret_cast<const double2*>(z_arr)[p];
                    b[u] = reinterpret_cast<const double2*>(d_arr)[p];
                }
            }
#pragma unroll
            for (int u = 0; u < UNR; ++u) {
                const size_t p = base + (size_t)u * blockDim.x + threadIdx.x;
                if (p < npair) {
                    turn(a[u].x, b[u].x);
                    turn(a[u].y, b[u].y);
                    reinterpret_cast<double2*>(z_arr)[p] = a[u];
                    reinterpret_cast<double2*>(d_arr)[p] = b[u];
                    if (MOMENTS) {
                        acc.add(a[u].x, b[u].x, in_bucket<double>(a[u].x, b[u].x, P));
                        acc.add(a[u].y, b[u].y, in_bucket<double>(a[u].y, b[u].y, P));
                    }
                }
            }
        }
        if ((n & 1) && blockIdx.x == 0 && threadIdx.x == 0) {
            double zz = z_arr[n - 1], dd = d_arr[n - 1];
            turn(zz, dd);
            z_arr[n - 1] = zz; d_arr[n - 1] = dd;
            if (MOMENTS) acc.add(zz, dd, in_bucket<double>(zz, dd, P));
        }
    } else {
        for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n;
             i += (size_t)gridDim.x * blockDim.x) {
            double zz = z_arr[i], dd = d_arr[i];
            turn(zz, dd);
            z_arr[i] = zz; d_arr[i] = dd;
            if (MOMENTS) acc.add(zz, dd, in_bucket<double>(zz, dd, P));
        }
    }
    if (MOMENTS) block_reduce_store(acc, partials + (size_t)blockIdx.x * kPartialStride);
}

}  // namespace lt
