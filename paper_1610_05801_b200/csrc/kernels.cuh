// kernels.cuh -- sm_100a device code of liblongtrack (CUDA path only; shares nothing with oracle/).
//
// Notation: the state of a particle is (z, delta).  Inside the kernels the position
// is carried as the RF phase in HALF PERIODS,  v = kappa*z/pi  (kappa = h/R), so that
//     sin(kappa z) = sin(pi v) = (-1)^n sin(pi f),   n = rint(v),  f = v - n  in [-1/2, 1/2]
// and the range reduction is EXACT for any |v| < 2^51 (unbound particles stream to |v| ~ 1e4):
//     t = v + 1.5*2^52  (DADD; the low mantissa bit of t is the parity of n)
//     n = t - 1.5*2^52  (DADD, exact)        f = v - n  (DADD, exact)
// The sign (-1)^n is XORed into the sign bit of f on the integer pipe; sin(pi f) = f*S(f^2) is
// a degree-7 polynomial in s = f^2 with the kick amplitude folded into its coefficients, so
//     delta += A sin(kappa z)   ==   delta = fma(f_signed, S_A(s), delta).
// FP64-pipe instructions per particle-turn, leap-frog / Euler-Cromer, single harmonic, merged
// drifts:  1 (drift) + 3 (reduction) + 1 (s) + 7 (Horner) + 1 (kick FMA) = 13.
// (BASELINE.json:configs[0] gives the map; PAPER.md:175 the register-resident turn loop.)
#pragma once

#include <cstdint>
#include <cuda_runtime.h>

namespace lt {

#ifndef LT_TURN_UNROLL
#define LT_TURN_UNROLL 96     // particle-turns per iteration of the fused single-harmonic turn loop (see advance())
#endif

constexpr int kEulerCromer = 0, kLeapfrog = 1, kRuth4 = 2;
constexpr int kMaxSin = 8, kMaxCos = 9;

// ------------------------------------------------------------------------------------------
// Per-tracker constants, passed by value as a __grid_constant__ kernel parameter: they sit in
// the constant bank and feed DFMA/FFMA as direct operands (no registers, no loads).
// ------------------------------------------------------------------------------------------
template <typename T>
struct MapConsts {
    T to_phase;             // kappa/pi:        v = z * to_phase
    T from_phase;           // pi/kappa:        z = v * from_phase
    T d;                    // eta*C/2          (half-turn drift of z, exact path)
    T c_half;               // d*kappa/pi       (half-turn drift of v)
    // drift coefficients of v per stage, fast path.  Leap-frog: lead = c_half, mid unused,
    // trail = c_half, merged = 2 c_half.  Ruth4: lead = x1 c_half, mid = (x1+x0) c_half, ...
    T drift_lead, drift_mid, drift_trail, drift_merged;
    // the same for z on the exact (split-drift) path
    T zdrift_lead, zdrift_mid, zdrift_trail;
    T sinA[3][kMaxSin];     // tau_k * A * S coefficients, k = stage (Ruth4: x1, x0, x1)
    T sin1[kMaxSin];        // S coefficients, unscaled (membership test, generic kick)
    T cos1[kMaxCos];        // C coefficients: cos(pi f) = C(f^2)
    T two_r;                // 2 r
    T kickA[3];             // tau_k * A           (generic phi_s path)
    T phi_off;              // phi_s/pi
    T sin_phi_s;            // sin(phi_s)
    T r;                    // r
    T z_max;                // pi R / h
    T hn_delta;             // eta C / (2 H_sep): H/H_sep = hn_delta delta^2 + S^2 (1 + 2r(1-S^2))
};

// ------------------------------------------------------------------------------------------
// fp64 / fp32 traits
// ------------------------------------------------------------------------------------------
template <typename T> struct Real;

template <> struct Real<double> {
    static constexpr int NS = 8, NC = 9;
    typedef double2 vec2;
    static __device__ __forceinline__ double magic() { return 6755399441055744.0; }  // 1.5*2^52
    static __device__ __forceinline__ double fma(double a, double b, double c) { return __fma_rn(a, b, c); }
    static __device__ __forceinline__ double add(double a, double b) { return __dadd_rn(a, b); }
    static __device__ __forceinline__ double sub(double a, double b) { return __dsub_rn(a, b); }
    static __device__ __forceinline__ double mul(double a, double b) { return __dmul_rn(a, b); }
    static __device__ __forceinline__ double mul_rounded(double a, double b) { return __dmul_rn(a, b); }   // see Real<f32x2>
    // f with the sign bit flipped when the integer held in the low mantissa bits of t is odd.
    // hi + (lo << 31) mod 2^32 == hi ^ ((lo & 1) << 31): ONE IMAD instead of shift + xor, in
    // unsigned arithmetic (defined on overflow).  Next to a saturated FP64 pipe the IMAD costs
    // 2.6 points of the pipe, a shift + LOP3 pair 12 (profiles/r2_fp64_pipe_probe.md).
    static __device__ __forceinline__ double flip(double f, double t) {
        const unsigned int hi = (unsigned int)__double2hiint(f) + ((unsigned int)__double2loint(t) << 31);
        return __hiloint2double((int)hi, __double2loint(f));
    }
    static __device__ __forceinline__ double flip_by(double x, double t) { return flip(x, t); }
    // (-1)^n as a value, n the integer in the low mantissa bits of t: +-1.0 (one IMAD; the low word is zero)
    static __device__ __forceinline__ double sign_of(double t) {
        return __hiloint2double((int)(0x3FF00000u + ((unsigned int)__double2loint(t) << 31)), 0);
    }
    // the same, written into the register pair of a previous sign value (whose low word is zero):
    // one instruction, where sign_of() also has to clear a low word
    static __device__ __forceinline__ double resign(double prev, double t) {
        return __hiloint2double((int)(0x3FF00000u + ((unsigned int)__double2loint(t) << 31)), __double2loint(prev));
    }
};

template <> struct Real<float> {
    static constexpr int NS = 5, NC = 6;
    typedef float2 vec2;
    static __device__ __forceinline__ float magic() { return 12582912.0f; }          // 1.5*2^23
    static __device__ __forceinline__ float fma(float a, float b, float c) { return __fmaf_rn(a, b, c); }
    static __device__ __forceinline__ float add(float a, float b) { return __fadd_rn(a, b); }
    static __device__ __forceinline__ float sub(float a, float b) { return __fsub_rn(a, b); }
    static __device__ __forceinline__ float mul(float a, float b) { return __fmul_rn(a, b); }
    static __device__ __forceinline__ float mul_rounded(float a, float b) { return __fmul_rn(a, b); }     // see Real<f32x2>
    static __device__ __forceinline__ float flip(float f, float t) {
        return __uint_as_float(__float_as_uint(f) + (__float_as_uint(t) << 31));
    }
    static __device__ __forceinline__ float flip_by(float x, float t) { return flip(x, t); }
    static __device__ __forceinline__ float sign_of(float t) {
        return __uint_as_float(0x3F800000u + (__float_as_uint(t) << 31));
    }
    static __device__ __forceinline__ float resign(float, float t) { return sign_of(t); }
};

// Two fp32 particles in one 64-bit register pair.  sm_100a has packed FP32 instructions (FFMA2,
// FADD2, FMUL2: one issue slot, two lanes' worth of arithmetic per thread), and the fp32 turn is
// issue-bound -- the FP32 pipe takes one warp instruction per cycle, which is also all the
// scheduler can issue, so every IMAD and loop instruction displaced an FFMA (67 % of the FP32
// peak with scalar instructions).  Each half rounds exactly like the scalar instruction: the
// results are the bits of Real<float>.
struct f32x2 {
    float2 v;
    __host__ __device__ f32x2() {}
    __host__ __device__ f32x2(float a) { v.x = a; v.y = a; }
    __host__ __device__ f32x2(float a, float b) { v.x = a; v.y = b; }
    __host__ __device__ f32x2 operator-() const { return f32x2(-v.x, -v.y); }
};

template <> struct Real<f32x2> {
    static constexpr int NS = 5, NC = 6;
    static __device__ __forceinline__ f32x2 magic() { return f32x2(12582912.0f); }
    static __device__ __forceinline__ f32x2 wrap(float2 a) { f32x2 r; r.v = a; return r; }
    static __device__ __forceinline__ f32x2 fma(f32x2 a, f32x2 b, f32x2 c) { return wrap(__ffma2_rn(a.v, b.v, c.v)); }
    static __device__ __forceinline__ f32x2 add(f32x2 a, f32x2 b) { return wrap(__fadd2_rn(a.v, b.v)); }
    static __device__ __forceinline__ f32x2 sub(f32x2 a, f32x2 b) { return wrap(__fadd2_rn(a.v, (-b).v)); }
    static __device__ __forceinline__ f32x2 mul(f32x2 a, f32x2 b) { return wrap(__fmul2_rn(a.v, b.v)); }
    // A product that feeds an ADDITION and has to keep its own rounding (the phase v = z * kappa/pi
    // of the exact path, which the reduction adds to and subtracts from).  ptxas 12.9 contracts
    // mul.rn.f32x2 + add.rn.f32x2 into one FFMA2 in spite of the explicit roundings -- also with
    // --fmad=false, also when the product is written fma(a, b, -0) -- which it never does to the
    // scalar mul.rn.f32 / mul.rn.f64; the packed kernels then returned other bits than the scalar
    // fp32 kernels (plain fused, per-turn) on the split-drift path.  Two scalar FMULs are left
    // alone (checked in the SASS); they cost one issue slot more, on the exact path only.
    static __device__ __forceinline__ f32x2 mul_rounded(f32x2 a, f32x2 b) {
        return f32x2(__fmul_rn(a.v.x, b.v.x), __fmul_rn(a.v.y, b.v.y));
    }
    // With packed arithmetic the FMA pipe is the bound (two cycles per FFMA2) and issue slots are
    // free, so the sign flip leaves that pipe: funnel shift + XOR on the ALU pipe instead of the
    // IMAD of the scalar kernels (an IMAD occupies the FMA pipe; profiles/r2_ncu_summary.md).
    static __device__ __forceinline__ float flip1(float f, float t) {
        return __uint_as_float(__float_as_uint(f) ^ __funnelshift_l(0u, __float_as_uint(t), 31));
    }
    static __device__ __forceinline__ f32x2 flip(f32x2 f, f32x2 t) {
        return f32x2(flip1(f.v.x, t.v.x), flip1(f.v.y, t.v.y));
    }
    static __device__ __forceinline__ f32x2 flip_by(f32x2 x, f32x2 t) { return flip(x, t); }
    static __device__ __forceinline__ f32x2 sign_of(f32x2 t) { return flip(f32x2(1.0f), t); }
    static __device__ __forceinline__ f32x2 resign(f32x2, f32x2 t) { return sign_of(t); }
};

// how many array elements of type T a register value V carries, and access to them
template <typename T, typename V> struct Lanes {
    static constexpr int PV = 1;
    static __device__ __forceinline__ void set(V& v, int, T x) { v = x; }
    static __device__ __forceinline__ T get(const V& v, int) { return v; }
};
template <> struct Lanes<float, f32x2> {
    static constexpr int PV = 2;
    static __device__ __forceinline__ void set(f32x2& v, int h, float x) { if (h) v.v.y = x; else v.v.x = x; }
    static __device__ __forceinline__ float get(const f32x2& v, int h) { return h ? v.v.y : v.v.x; }
};

// exact reduction: returns f = v - rint(v); *t_out keeps the parity of rint(v) in its low bit
template <typename T>
__device__ __forceinline__ T reduce_half_periods(T v, T* t_out) {
    typedef Real<T> R;
    T t = R::add(v, R::magic());
    T n = R::sub(t, R::magic());
    *t_out = t;
    return R::sub(v, n);
}

// Horner evaluation of c[0] + c[1] s + ... + c[NUSED-1] s^(NUSED-1)
template <typename T, int NUSED, int N>
__device__ __forceinline__ T horner(const T (&c)[N], T s) {
    static_assert(NUSED <= N, "polynomial longer than its table");
    T q = c[NUSED - 1];
#pragma unroll
    for (int k = NUSED - 2; k >= 0; --k) q = Real<T>::fma(q, s, c[k]);
    return q;
}

// ------------------------------------------------------------------------------------------
// The kick  delta += tau_k * F(z)  for the phase v (half periods).
//   HARM = 1: F = A sin(pi v)                              (configs[0])
//   HARM = 2: F = A [sin(pi v) + r sin(2 pi v)] = A sin(pi v) (1 + 2 r cos(pi v))   (configs[4])
//   HARM = 0: generic, phi_s != 0:  A [sin(phi_s + pi v) - sin(phi_s) + r sin(2 pi v)]   (G3)
// ------------------------------------------------------------------------------------------
// FQ selects WHERE the sign (-1)^n is applied: to f (beside the Horner chain: wins with two
// particles per lane at every warp count) or to the polynomial value q (one dependent integer
// op later, but faster with ONE particle per lane from 5 warps per sub-partition on;
// profiles/r2_fp64_pipe_probe.md).  Same bits either way.
// PROG (RF programme; G28): the kick of this turn is
//     a * A [ sin(phi_s + pi (v + p)) - sin(phi_s) + r sin(2 pi (v + p)) ],
// a = voltage scale, p = phase offset in half periods.  PROG = 1: add p here (fast path, the
// state is v); PROG = 2: the caller already folded p into v (exact path: v = fma(z, kappa/pi, p)).
// The scale multiplies f, not q: f*a is ready three instructions after the reduction and runs
// beside the Horner chain, so the dependent chain of a turn is one FP64 instruction shorter than
// with q*a behind the polynomial (same 15 instructions; a = 1 still returns the plain map's bits).
template <typename T, int HARM, bool FQ = false, int PROG = 0>
__device__ __forceinline__ T kick(T v, T delta, const MapConsts<T>& P, int stage, T a = T(1),
                                  T p = T(0), T* sg = nullptr) {
    typedef Real<T> R;
    constexpr int NS = R::NS, NC = R::NC;
    static_assert(PROG >= 0 && PROG <= 2, "the energy ramp has its own kick (kernels_ramp.cuh)");
    const T (&sin_coef)[kMaxSin] = P.sinA[stage];
    if (PROG == 1) v = R::add(v, p);
    if (HARM == 1) {
        T t;
        T f = reduce_half_periods(v, &t);
        T s = R::mul(f, f);
        T fa = PROG ? R::mul(f, a) : f;
        T q = horner<T, NS>(sin_coef, s);
        if (FQ) return R::fma(fa, R::flip(q, t), delta);
        return R::fma(R::flip(fa, t), q, delta);
    } else if (HARM == 2) {
        T t;
        T f = reduce_half_periods(v, &t);
        T s = R::mul(f, f);
        T fa = PROG ? R::mul(f, a) : f;
        T q = horner<T, NS>(sin_coef, s);         // tau A sin(pi f)/f
        T c = horner<T, NC>(P.cos1, s);           // cos(pi f)
        // sin and cos both change sign with the parity of n:  sigma s (1 + 2 r sigma c) = s (sigma + 2 r c),
        // so ONE sign value sigma = +-1 does for both (it was a flip of f and a flip of 2r; the bits are
        // the same: a sign moved through a product or an FMA commutes with the rounding)
        // sg (fused turn loop): the particle's previous sign value, overwritten in place
        const T sigma = sg ? R::resign(*sg, t) : R::sign_of(t);
        if (sg) *sg = sigma;
        T m = R::fma(P.two_r, c, sigma);
        return R::fma(fa, R::mul(q, m), delta);
    } else {
        T t1, t2;
        T f1 = reduce_half_periods(R::add(v, P.phi_off), &t1);
        T s1 = R::mul(f1, f1);
        T sn = R::mul_rounded(R::flip(f1, t1), horner<T, NS>(P.sin1, s1));   // feeds a subtraction
        T acc = R::sub(sn, P.sin_phi_s);
        T f2 = reduce_half_periods(R::add(v, v), &t2);
        T s2 = R::mul(f2, f2);
        T sn2 = R::mul(R::flip(f2, t2), horner<T, NS>(P.sin1, s2));
        acc = R::fma(P.r, sn2, acc);
        return R::fma(PROG ? R::mul(P.kickA[stage], a) : P.kickA[stage], acc, delta);
    }
}

// ------------------------------------------------------------------------------------------
// One full turn on the EXACT path: the state is z itself, every half drift is its own FMA
// (bit-identical between the per-turn kernel, the split-drift fused kernel and any chunking).
// ------------------------------------------------------------------------------------------
template <typename T, int INTEG, int HARM, bool PROG = false>
__device__ __forceinline__ void turn_exact(T& z, T& delta, const MapConsts<T>& P, T a = T(1),
                                           T p = T(0)) {
    typedef Real<T> R;
    constexpr int PK = PROG ? 2 : 0;
#define LT_PHASE(zz) (PROG ? R::fma(zz, P.to_phase, p) : R::mul_rounded(zz, P.to_phase))
    if (INTEG == kLeapfrog) {
        z = R::fma(-P.zdrift_lead, delta, z);
        delta = kick<T, HARM, false, PK>(LT_PHASE(z), delta, P, 0, a);
        z = R::fma(-P.zdrift_trail, delta, z);
    } else if (INTEG == kEulerCromer) {
        delta = kick<T, HARM, false, PK>(LT_PHASE(z), delta, P, 0, a);
        z = R::fma(-P.zdrift_trail, delta, z);
    } else {
        z = R::fma(-P.zdrift_lead, delta, z);
        delta = kick<T, HARM, false, PK>(LT_PHASE(z), delta, P, 0, a);
        z = R::fma(-P.zdrift_mid, delta, z);
        delta = kick<T, HARM, false, PK>(LT_PHASE(z), delta, P, 1, a);
        z = R::fma(-P.zdrift_mid, delta, z);
        delta = kick<T, HARM, false, PK>(LT_PHASE(z), delta, P, 2, a);
        z = R::fma(-P.zdrift_trail, delta, z);
    }
#undef LT_PHASE
}

// One turn on the FAST path, state = phase v, WITHOUT its leading drift and with the trailing
// drift given by the caller (merged with the next turn's leading drift, or the plain trailing
// one at the end of a call).
// PROG: the state is u = v + p_t, the phase INCLUDING this turn's RF phase offset; dp = p_(t+1) - p_t
// is added to u beside the sine chain and the trailing drift is an FMA onto that sum, so the
// offset costs one FP64 instruction and none on the dependent chain.
template <typename T, int INTEG, int HARM, bool FQ = false, bool PROG = false>
__device__ __forceinline__ void turn_fast(T& v, T& delta, const MapConsts<T>& P, T trailing,
                                          T a = T(1), T dp = T(0), T* sg = nullptr) {
    typedef Real<T> R;
    constexpr int PK = PROG ? 2 : 0;
    if (INTEG == kRuth4) {
        delta = kick<T, HARM, FQ, PK>(v, delta, P, 0, a, T(0), sg);
        v = R::fma(-P.drift_mid, delta, v);
        delta = kick<T, HARM, FQ, PK>(v, delta, P, 1, a, T(0), sg);
        v = R::fma(-P.drift_mid, delta, v);
        const T w = PROG ? R::add(v, dp) : v;
        delta = kick<T, HARM, FQ, PK>(v, delta, P, 2, a, T(0), sg);
        v = R::fma(-trailing, delta, w);
    } else {
        const T w = PROG ? R::add(v, dp) : v;
        delta = kick<T, HARM, FQ, PK>(v, delta, P, 0, a, T(0), sg);
        v = R::fma(-trailing, delta, w);
    }
}

// `turns` turns of ILP particles held in registers (steps a2-a6).  Fast path: the state is the
// phase v; `first` converts z -> v and applies the leading drift, `last` applies the plain
// trailing drift and converts back, in between consecutive half drifts are merged.  Between
// chunks of one call the z array therefore holds v mid-drift, which makes the result of a
// call independent of how its turns are chunked.  SPLIT: exact path, state is z.
// PROG: prog[k] = (a, p) of the k-th turn of this call to advance on the exact path (voltage
// scale, phase offset in half periods); on the fast path prog[k] = (a, p_(k+1) - p_k) -- the
// difference to the NEXT turn's offset, minus the last offset at the end of the API call -- and
// prog[-1].y = the absolute offset of turn 0 of the launch (used by `first` only).
template <typename T, int INTEG, int HARM, bool SPLIT, int ILP, bool FQ, bool PROG = false>
__device__ __forceinline__ void advance(T (&x)[ILP], T (&dl)[ILP], unsigned int turns, int first,
                                        int last, const MapConsts<T>& P,
                                        const double2* __restrict__ prog = nullptr,
                                        double2* __restrict__ stage = nullptr) {
    typedef Real<T> R;
    if (PROG) {
        // RF programme.  The table is read 32 turns ahead: lane l fetches entry t0 + 32 + l
        // while the warp works through entries t0 .. t0 + 31 out of its private 512-byte
        // buffer in shared memory (one broadcast LDS.128 per turn).  A per-turn uniform LDG
        // left the warps waiting on L2 once per 128-byte line (long-scoreboard stalls, 76 %
        // of the FP64 peak; profiles/r1_next_rows_ncu.md).
        const unsigned int lane = threadIdx.x & 31u;
        if (!SPLIT && first) {
            const T p0 = (T)__ldg(prog - 1).y;
#pragma unroll
            for (int j = 0; j < ILP; ++j) {
                x[j] = R::mul(x[j], P.to_phase);
                if (INTEG != kEulerCromer) x[j] = R::fma(-P.drift_lead, dl[j], x[j]);
                x[j] = R::add(x[j], p0);
            }
        }
        // the fast path peels the last turn (its trailing drift differs at the end of a call)
        const unsigned int nmain = SPLIT ? turns : turns - 1;
        double2 tail = make_double2(1.0, 0.0);
        if (!SPLIT) tail = __ldg(prog + (turns - 1));
        double2 nxt = make_double2(1.0, 0.0);
        if (lane < nmain) nxt = __ldg(prog + lane);
        for (unsigned int t0 = 0; t0 < nmain; t0 += 32) {
            __syncwarp();
            stage[lane] = nxt;
            __syncwarp();
            if (t0 + 32 + lane < nmain) nxt = __ldg(prog + t0 + 32 + lane);
            const unsigned int m = min(32u, nmain - t0);
            // the whole staged block of 32 turns unrolled: the loop's counter, address arithmetic and
            // uniform-register reloads cost issue slots next to the saturated FP64 pipe (+0.8 points)
            constexpr int kUnrollP = (INTEG == kRuth4 || HARM != 1) ? 8 : 32;
#pragma unroll kUnrollP
            for (unsigned int k = 0; k < m; ++k) {
                const double2 e = stage[k];
                const T a = (T)e.x, p = (T)e.y;
#pragma unroll
                for (int j = 0; j < ILP; ++j) {
                    if (SPLIT) turn_exact<T, INTEG, HARM, true>(x[j], dl[j], P, a, p);
                    else turn_fast<T, INTEG, HARM, FQ, true>(x[j], dl[j], P, P.drift_merged, a, p);
                }
            }
        }
        if (!SPLIT) {
            const T trailing = last ? P.drift_trail : P.drift_merged;
#pragma unroll
            for (int j = 0; j < ILP; ++j) {
                turn_fast<T, INTEG, HARM, FQ, true>(x[j], dl[j], P, trailing, (T)tail.x, (T)tail.y);
                if (last) x[j] = R::mul(x[j], P.from_phase);
            }
        }
        return;
    }
    if (SPLIT) {
        for (unsigned int t = 0; t < turns; ++t) {
#pragma unroll
            for (int j = 0; j < ILP; ++j) turn_exact<T, INTEG, HARM, false>(x[j], dl[j], P);
        }
    } else {
        if (first) {
#pragma unroll
            for (int j = 0; j < ILP; ++j) {
                x[j] = R::mul_rounded(x[j], P.to_phase);     // Euler-Cromer: goes straight into the reduction
                if (INTEG != kEulerCromer) x[j] = R::fma(-P.drift_lead, dl[j], x[j]);
            }
        }
        // every non-FP64 instruction costs issue capacity next to the saturated FP64 pipe
        // (profiles/r2_fp64_pipe_probe.md): the loop's 8 instructions of overhead (5 uniform-register
        // reloads, counter, compare, branch) are spread over LT_TURN_UNROLL particle-turns.  Configs[1]:
        // 16 particle-turns per iteration 0.905 of the FP64 peak, 64: 0.912, 128: 0.915, 160: 0.911 --
        // and 192 (43 KB of code): 0.858, 256 (57 KB): 0.59, the loop no longer fits the instruction
        // cache; the default keeps a good third of headroom below the largest body that measured well.  The double harmonic and
        // Ruth4 measured BEST at 4 turns per iteration in fp64 (2: -2 points, 8: -1.5) and at 2 in the
        // packed fp32 kernels (0.864 of the FP32 peak against 0.845 at 4, 0.83 at 1 and 3).
#ifndef LT_UNROLL_OTHER
#define LT_UNROLL_OTHER 4
#endif
#ifndef LT_UNROLL_OTHER_F32
#define LT_UNROLL_OTHER_F32 2
#endif
        constexpr int kOther = sizeof(T) == 8 && R::NS == 8 ? LT_UNROLL_OTHER : LT_UNROLL_OTHER_F32;   // fp64 : fp32 (scalar or packed)
        constexpr int kUnroll = (INTEG == kRuth4 || HARM != 1 || ILP > 2) ? kOther : LT_TURN_UNROLL / ILP;
        T sg[ILP];                           // double harmonic: the particles' sign values (see kick)
#pragma unroll
        for (int j = 0; j < ILP; ++j) sg[j] = T(1);
#pragma unroll kUnroll
        for (unsigned int t = 1; t < turns; ++t) {
#pragma unroll
            for (int j = 0; j < ILP; ++j)
                turn_fast<T, INTEG, HARM, FQ, false>(x[j], dl[j], P, P.drift_merged, T(1), T(0), &sg[j]);
        }
        const T trailing = last ? P.drift_trail : P.drift_merged;
#pragma unroll
        for (int j = 0; j < ILP; ++j) {
            turn_fast<T, INTEG, HARM, FQ, false>(x[j], dl[j], P, trailing, T(1), T(0), &sg[j]);
            if (last) x[j] = R::mul(x[j], P.from_phase);
        }
    }
}

// ------------------------------------------------------------------------------------------
// Fused multi-turn kernel (registers hold the state over the inner turn
// loop; the host loops over chunks).  One thread owns ILP particles; a block owns a tile of
// blockDim.x * ILP consecutive particles, element j of thread t = tile + j*blockDim.x + t
// (coalesced; double2 when VEC).  `first` / `last` mark the first / last chunk of a call:
// between chunks the z array holds the phase v mid-drift, so that the result of a call does
// not depend on the chunk length.
// ------------------------------------------------------------------------------------------
template <typename T, int INTEG, int HARM, bool SPLIT, int ILP, bool VEC>
__global__ void fused_kernel(T* __restrict__ z_arr, T* __restrict__ d_arr, size_t n,
                             unsigned int turns, int first, int last,
                             const __grid_constant__ MapConsts<T> P) {
    typedef Real<T> R;
    typedef typename R::vec2 V2;
    T x[ILP], dl[ILP];
    const size_t tile = (size_t)blockIdx.x * blockDim.x * ILP;

    // ---- entry load (a1)
    if (VEC) {
#pragma unroll
        for (int j = 0; j < ILP / 2; ++j) {
            size_t i = tile + 2 * ((size_t)j * blockDim.x + threadIdx.x);
            if (i + 1 < n) {
                V2 a = *reinterpret_cast<const V2*>(z_arr + i);
                V2 b = *reinterpret_cast<const V2*>(d_arr + i);
                x[2 * j] = a.x; x[2 * j + 1] = a.y; dl[2 * j] = b.x; dl[2 * j + 1] = b.y;
            } else {
                x[2 * j] = (i < n) ? z_arr[i] : T(0); dl[2 * j] = (i < n) ? d_arr[i] : T(0);
                x[2 * j + 1] = T(0); dl[2 * j + 1] = T(0);
            }
        }
    } else {
#pragma unroll
        for (int j = 0; j < ILP; ++j) {
            size_t i = tile + (size_t)j * blockDim.x + threadIdx.x;
            x[j] = (i < n) ? z_arr[i] : T(0);
            dl[j] = (i < n) ? d_arr[i] : T(0);
        }
    }

    advance<T, INTEG, HARM, SPLIT, ILP, false>(x, dl, turns, first, last, P);

    // ---- exit store (a7)
    if (VEC) {
#pragma unroll
        for (int j = 0; j < ILP / 2; ++j) {
            size_t i = tile + 2 * ((size_t)j * blockDim.x + threadIdx.x);
            if (i + 1 < n) {
                V2 a, b;
                a.x = x[2 * j]; a.y = x[2 * j + 1]; b.x = dl[2 * j]; b.y = dl[2 * j + 1];
                *reinterpret_cast<V2*>(z_arr + i) = a;
                *reinterpret_cast<V2*>(d_arr + i) = b;
            } else if (i < n) {
                z_arr[i] = x[2 * j]; d_arr[i] = dl[2 * j];
            }
        }
    } else {
#pragma unroll
        for (int j = 0; j < ILP; ++j) {
            size_t i = tile + (size_t)j * blockDim.x + threadIdx.x;
            if (i < n) { z_arr[i] = x[j]; d_arr[i] = dl[j]; }
        }
    }
}

// ------------------------------------------------------------------------------------------
// Fused multi-turn kernel with ON-DEVICE DYNAMIC CHUNKING -- the paper's hybrid loop (CPU outer
// loop x in-kernel inner loop) with the outer loop moved onto the GPU.
//
// Why: a warp-wide FP64 instruction occupies a sub-partition's FP64 pipe for two cycles whatever
// the ensemble size, so 10^5 particles = 3125 warps over 592 sub-partitions leave some with 6
// and some with 5 warps for the WHOLE run: 12 % of the pipe idles, and nothing static fixes it.
// Here a persistent grid (one CTA of 4W warps per SM) keeps W warps on every sub-partition; work items are
// (chunk c of `item_turns` turns) x (group g of 32 particles), handed out by one atomic ticket
// in c-major order; the state goes through L2 between items (512 B per item, noise).  Every
// sub-partition stays saturated until the last few items.  An item's predecessor (c-1, g) has a
// smaller ticket, so it is finished or running: the acquire-poll on done[g] cannot deadlock and
// is in practice never taken when there are more groups than resident warps.
// The arithmetic per particle is identical to fused_kernel, so results are bit-identical to it
// and independent of item_turns and of the scheduling order.
// ------------------------------------------------------------------------------------------
// Work-item schedule of the persistent kernels: a launch of `turns` turns is cut into chunks, the
// same for every group of particles.  Plain: ceil(turns / item) chunks of `item` turns.  Tapered
// (dynamic scheduling): full items first, then the last item..2*item turns are halved again and
// again down to kMinTaper turns, so that the warps which find the ticket queue empty wait for a
// short item, not a long one (an untapered tail cost 1.7 % at 10^5 particles,
// profiles/r2_fused_shapes.md).  Chunk boundaries never change the arithmetic (G16).
constexpr unsigned int kMinTaper = 64;
struct ItemSchedule {
    unsigned int turns, item, nfull, nchunks;
    __host__ __device__ void init(unsigned int turns_, unsigned int item_, int taper) {
        turns = turns_; item = item_ < 1u ? 1u : item_;
        if (!taper) {
            nfull = turns / item;
            nchunks = (turns + item - 1) / item;
            return;
        }
        const unsigned int q = turns / item;
        nfull = q > 0 ? q - 1 : 0;
        unsigned int r = turns - nfull * item, k = 0;
        while (r > 0) { const unsigned int len = r <= kMinTaper ? r : (r + 1) / 2; r -= len; ++k; }
        nchunks = nfull + k;
    }
    // first turn and length of chunk c
    __host__ __device__ void span(unsigned int c, int taper, unsigned int* start, unsigned int* len) const {
        if (!taper || c < nfull) {
            *start = c * item;
            *len = (turns - *start < item) ? turns - *start : item;
            return;
        }
        unsigned int s0 = nfull * item, r = turns - s0, l = 0;
        for (unsigned int k = nfull;; ++k) {
            l = r <= kMinTaper ? r : (r + 1) / 2;
            if (k == c) break;
            s0 += l; r -= l;
        }
        *start = s0; *len = l;
    }
};

__device__ __forceinline__ unsigned int ld_acquire_u32(const unsigned int* p) {
    unsigned int v;
    asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
    return v;
}
__device__ __forceinline__ void st_release_u32(unsigned int* p, unsigned int v) {
    asm volatile("st.release.gpu.global.u32 [%0], %1;" ::"l"(p), "r"(v) : "memory");
}

// PROG: prog[k] = (a, p) of the k-th turn of THIS launch (RF programme, f2).
// ILP: particles per lane.  A work item is (chunk) x (group of 32*ILP particles); particle j of a
// lane is element g*32*ILP + 32*j + lane (coalesced).  Two independent chains per warp issue
// back to back without a warp switch: the turn loop measures 91.5 % of the FP64 peak at 4 chains
// per sub-partition as 2 warps x 2 chains against 87.5 % as 4 warps x 1 chain
// (profiles/r2_fp64_pipe_probe.md).  The arithmetic per particle does not depend on ILP.
// V: the register value a chain is computed in -- T itself, or f32x2 = two fp32 particles in one
// packed value (then a lane carries 2*ILP particles and MapConsts<V> holds every constant twice).
template <typename T, int INTEG, int HARM, bool SPLIT, bool FQ, bool PROG = false, int ILP = 1, typename V = T>
__global__ void __launch_bounds__(ILP == 1 ? 1024 : 512, 1)
fused_persistent_kernel(T* __restrict__ z_arr, T* __restrict__ d_arr, size_t n, unsigned int turns,
                        unsigned int item_turns, int first_launch, int last_launch, int dynamic,
                        unsigned long long* __restrict__ ticket, unsigned int* __restrict__ done,
                        const __grid_constant__ MapConsts<V> P,
                        const double2* __restrict__ prog = nullptr) {
    extern __shared__ __align__(16) unsigned char residency_cap[];   // sized to cap CTAs per SM; PROG: 512 B per warp of staged programme entries
    typedef Lanes<T, V> L;
    constexpr unsigned int G = 32u * ILP * L::PV;
    const unsigned int lane = threadIdx.x & 31u;
    const unsigned long long groups = (n + G - 1) / G;
    const unsigned long long slots = (unsigned long long)gridDim.x * (blockDim.x >> 5);
    // slots are numbered SM-first so that consecutive slots sit on different SMs
    const unsigned long long slot = (unsigned long long)(threadIdx.x >> 5) * gridDim.x + blockIdx.x;

    // turns [t_begin, t_begin + nt) of group g: wait until progress word `done[g]` has reached
    // `need` (0 = nothing to wait for), advance, publish `publish` (0 = nothing follows)
    auto run_piece = [&](unsigned long long g, unsigned int t_begin, unsigned int nt, unsigned int need,
                         unsigned int publish) {
        if (need) {
            while (ld_acquire_u32(done + g) < need) __nanosleep(64);
        }
        const size_t i0 = (size_t)g * G + lane;
        V x[ILP], dl[ILP];
#pragma unroll
        for (int j = 0; j < ILP; ++j) {
#pragma unroll
            for (int h = 0; h < L::PV; ++h) {
                const size_t i = i0 + 32u * (j * L::PV + h);
                L::set(x[j], h, (i < n) ? __ldcg(z_arr + i) : T(0));   // L2 only: another SM may have written it
                L::set(dl[j], h, (i < n) ? __ldcg(d_arr + i) : T(0));
            }
        }
        const int first = first_launch && t_begin == 0;
        const int last = last_launch && t_begin + nt == turns;
        advance<V, INTEG, HARM, SPLIT, ILP, FQ, PROG>(
            x, dl, nt, first, last, P, PROG ? prog + t_begin : nullptr,
            PROG ? reinterpret_cast<double2*>(residency_cap) + (threadIdx.x & ~31u) : nullptr);
#pragma unroll
        for (int j = 0; j < ILP; ++j) {
#pragma unroll
            for (int h = 0; h < L::PV; ++h) {
                const size_t i = i0 + 32u * (j * L::PV + h);
                if (i < n) { __stcg(z_arr + i, L::get(x[j], h)); __stcg(d_arr + i, L::get(dl[j], h)); }
            }
        }
        if (publish) {
            __threadfence();
            __syncwarp();
            if (lane == 0) st_release_u32(done + g, publish);
        }
        __syncwarp();            // the warp is converged again before the next piece (see run_piece's callers)
    };

    if (dynamic == 2) {
        // WRAP-AROUND schedule (McNaughton's rule for preemptive scheduling on identical machines):
        // the work of the launch is the line x in [0, groups * turns), group-major; slot s owns
        // [s X / S, (s+1) X / S) and walks it from the top down, piece by piece.  Its first piece
        // is the EARLY part of a group (turns 0 .. t), its last piece the LATE part of another
        // (turns t' .. end) whose early part was the first piece of slot s - 1: with groups >=
        // slots a group is cut at most once, the late part starts groups/slots - 1 group-runs
        // after the early one ended, and every slot finishes at the same moment -- no ticket, no
        // tail, two or three item switches per warp instead of dozens.  All FP64 timing is
        // data-independent and every sub-partition holds the same number of warps, which is
        // what makes a static preemptive schedule exact here.
        const unsigned __int128 X = (unsigned __int128)groups * turns;
        const unsigned long long x_lo = (unsigned long long)(X * slot / slots);
        unsigned long long x = (unsigned long long)(X * (slot + 1) / slots);
        while (x > x_lo) {
            const unsigned long long g = (x - 1) / turns;
            const unsigned long long gx = g * (unsigned long long)turns;
            const unsigned int t_end = (unsigned int)(x - gx);
            const unsigned int t_begin = x_lo > gx ? (unsigned int)(x_lo - gx) : 0u;
            run_piece(__shfl_sync(0xffffffffu, g, 0), __shfl_sync(0xffffffffu, t_begin, 0),
                      __shfl_sync(0xffffffffu, t_end - t_begin, 0), t_begin ? 1u : 0u, t_end < turns ? 1u : 0u);
            x = gx + t_begin;
        }
        return;
    }

    ItemSchedule sched;
    sched.init(turns, item_turns, dynamic);
    const unsigned int nchunks = sched.nchunks;
    const unsigned long long total = groups * nchunks;
    // static mode (few groups): slot s of the grid owns groups s, s + S, ... for all turns
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
        unsigned int t_start, nt;
        sched.span(c, dynamic, &t_start, &nt);
        run_piece(g, t_start, nt, c, nchunks > 1 ? c + 1 : 0u);
    }
}

// ------------------------------------------------------------------------------------------
// Bucket membership of one state (G15):  |z| < z_max  and  H/H_sep < 1 with
//     H/H_sep = hn_delta delta^2 + S^2 (1 + 2 r (1 - S^2)),   S = sin(kappa z / 2).
// ------------------------------------------------------------------------------------------
template <typename T>
__device__ __forceinline__ bool in_bucket(T z, T delta, const MapConsts<T>& P) {
    typedef Real<T> R;
    // |z| < z_max means |g| < 1/2 for g = kappa z / (2 pi): already inside the polynomial's range,
    // so no range reduction is needed (outside it the value is garbage, and the |z| test is false).
    // Same bits as with the reduction, 3 FP64 instructions fewer; the r-term only when r != 0
    // (a warp-uniform branch on a constant): 15 instead of 22 FP64 instructions per particle for
    // the single harmonic -- the per-turn kernel spends 3.5 us of its 45 on the moments.
    T g = R::mul(z, R::mul(P.to_phase, T(0.5)));
    T S = R::mul(g, horner<T, R::NS>(P.sin1, R::mul(g, g)));
    T pot = R::mul(S, S);
    if (P.two_r != T(0)) pot = R::mul(pot, R::fma(P.two_r, R::sub(T(1), pot), T(1)));
    T hn = R::fma(P.hn_delta, R::mul(delta, delta), pot);
    return (fabs(z) < P.z_max) && (hn < T(1));
}

// Raw sums of a state, always accumulated in fp64.
struct Sums {
    double sz, szz, sd, sdd, szd;
    unsigned int nin;          // per THREAD: a thread sees at most n / (6 * 256) of the n <= 2^40 particles, < 2^32
    __device__ __forceinline__ void zero() { sz = szz = sd = sdd = szd = 0.0; nin = 0u; }
    __device__ __forceinline__ void add(double z, double d, bool inb) {
        sz += z; szz = __fma_rn(z, z, szz); sd += d; sdd = __fma_rn(d, d, sdd);
        szd = __fma_rn(z, d, szd); nin += inb ? 1u : 0u;
    }
};

constexpr int kPartialStride = 8;   // doubles per (turn, CTA) partial: sz szz sd sdd szd nin pad pad

__device__ __forceinline__ double warp_sum(double x) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) x += __shfl_xor_sync(0xffffffffu, x, o);
    return x;
}

// block combine: warp shuffles, then shared memory across warps, fixed order -> deterministic
__device__ __forceinline__ void block_reduce_store(Sums s, double* __restrict__ out) {
    __shared__ double sh[32][6];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, nw = (blockDim.x + 31) >> 5;
    double v[6] = {s.sz, s.szz, s.sd, s.sdd, s.szd, (double)s.nin};
#pragma unroll
    for (int k = 0; k < 6; ++k) v[k] = warp_sum(v[k]);
    if (lane == 0) {
#pragma unroll
        for (int k = 0; k < 6; ++k) sh[warp][k] = v[k];
    }
    __syncthreads();
    if (threadIdx.x < 6) {
        double a = 0.0;
        for (int w = 0; w < nw; ++w) a += sh[w][threadIdx.x];
        out[threadIdx.x] = a;
    }
}

// ------------------------------------------------------------------------------------------
// Per-turn kernel (BASELINE.json:configs[3]): ONE turn per launch, z/delta read
// and written through HBM (32 B per particle-turn in fp64), the turn's raw sums reduced in the
// same pass (a8 + a9).  Persistent CTAs, each walking tiles of blockDim.x*2*UNR particles with
// stride gridDim.x; `reverse` walks the array backwards (odd turns) so that the tail the
// previous launch left in the 126 MB L2 is consumed first.
// partials: [gridDim.x][kPartialStride] doubles for this turn.
// ------------------------------------------------------------------------------------------
template <typename T, int INTEG, int HARM, bool MOMENTS, int UNR>
__global__ void per_turn_kernel(T* __restrict__ z_arr, T* __restrict__ d_arr, size_t n,
                                int reverse, double* __restrict__ partials,
                                const __grid_constant__ MapConsts<T> P) {
    typedef typename Real<T>::vec2 V2;
    Sums acc;
    acc.zero();
    const size_t npair = n >> 1;                                   // full pairs
    const size_t tile_pairs = (size_t)blockDim.x * UNR;
    const size_t ntiles = (npair + tile_pairs - 1) / tile_pairs;
    for (size_t tl = blockIdx.x; tl < ntiles; tl += gridDim.x) {
        const size_t tix = reverse ? (ntiles - 1 - tl) : tl;
        const size_t base = tix * tile_pairs;
        V2 a[UNR], b[UNR];
#pragma unroll
        for (int u = 0; u < UNR; ++u) {
            size_t p = base + (size_t)u * blockDim.x + threadIdx.x;
            if (p < npair) {
                a[u] = reinterpret_cast<const V2*>(z_arr)[p];
                b[u] = reinterpret_cast<const V2*>(d_arr)[p];
            }
        }
#pragma unroll
        for (int u = 0; u < UNR; ++u) {
            size_t p = base + (size_t)u * blockDim.x + threadIdx.x;
            if (p < npair) {
                turn_exact<T, INTEG, HARM>(a[u].x, b[u].x, P);
                turn_exact<T, INTEG, HARM>(a[u].y, b[u].y, P);
                reinterpret_cast<V2*>(z_arr)[p] = a[u];
                reinterpret_cast<V2*>(d_arr)[p] = b[u];
                if (MOMENTS) {
                    acc.add((double)a[u].x, (double)b[u].x, in_bucket<T>(a[u].x, b[u].x, P));
                    acc.add((double)a[u].y, (double)b[u].y, in_bucket<T>(a[u].y, b[u].y, P));
                }
            }
        }
    }
    // odd tail particle
    if ((n & 1) && blockIdx.x == 0 && threadIdx.x == 0) {
        T zz = z_arr[n - 1], dd = d_arr[n - 1];
        turn_exact<T, INTEG, HARM>(zz, dd, P);
        z_arr[n - 1] = zz; d_arr[n - 1] = dd;
        if (MOMENTS) acc.add((double)zz, (double)dd, in_bucket<T>(zz, dd, P));
    }
    if (MOMENTS) block_reduce_store(acc, partials + (size_t)blockIdx.x * kPartialStride);
}

// scalar variant for arrays that are not 16-byte (fp64) / 8-byte (fp32) aligned
template <typename T, int INTEG, int HARM, bool MOMENTS>
__global__ void per_turn_kernel_scalar(T* __restrict__ z_arr, T* __restrict__ d_arr, size_t n,
                                       double* __restrict__ partials,
                                       const __grid_constant__ MapConsts<T> P) {
    Sums acc;
    acc.zero();
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n;
         i += (size_t)gridDim.x * blockDim.x) {
        T zz = z_arr[i], dd = d_arr[i];
        turn_exact<T, INTEG, HARM>(zz, dd, P);
        z_arr[i] = zz; d_arr[i] = dd;
        if (MOMENTS) acc.add((double)zz, (double)dd, in_bucket<T>(zz, dd, P));
    }
    if (MOMENTS) block_reduce_store(acc, partials + (size_t)blockIdx.x * kPartialStride);
}

// Sums of the current state without tracking (lt_moments_now, lt_bucket_count).
template <typename T, bool ONLY_COUNT>
__global__ void state_sums_kernel(const T* __restrict__ z_arr, const T* __restrict__ d_arr,
                                  size_t n, double* __restrict__ partials,
                                  const __grid_constant__ MapConsts<T> P) {
    Sums acc;
    acc.zero();
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n;
         i += (size_t)gridDim.x * blockDim.x) {
        T zz = z_arr[i], dd = d_arr[i];
        bool inb = in_bucket<T>(zz, dd, P);
        if (ONLY_COUNT) acc.nin += inb ? 1u : 0u;
        else acc.add((double)zz, (double)dd, inb);
    }
    block_reduce_store(acc, partials + (size_t)blockIdx.x * kPartialStride);
}

// ------------------------------------------------------------------------------------------
// Finalise: one CTA per turn of a batch sums that turn's per-CTA partials in a fixed order
// (deterministic) and writes lt_sums / lt_moments / the count.  `cursor` (device) holds the
// index of the batch's first turn in the output arrays; the last CTA to finish advances it, so
// that the same launch can be replayed from a CUDA graph.
// ------------------------------------------------------------------------------------------
struct SumsOut { double n, sum_z, sum_zz, sum_d, sum_dd, sum_zd, n_in_bucket, pad_; };
struct MomentsOut { double mean_z, rms_z, mean_d, rms_d, cov_zd; unsigned long long n_in_bucket; };

__device__ __forceinline__ MomentsOut moments_from(const SumsOut& s) {
    MomentsOut m;
    const double inv = s.n > 0.0 ? 1.0 / s.n : 0.0;
    m.mean_z = s.sum_z * inv;
    m.mean_d = s.sum_d * inv;
    double vz = __fma_rn(-m.mean_z, m.mean_z, s.sum_zz * inv);
    double vd = __fma_rn(-m.mean_d, m.mean_d, s.sum_dd * inv);
    m.rms_z = sqrt(vz > 0.0 ? vz : 0.0);
    m.rms_d = sqrt(vd > 0.0 ? vd : 0.0);
    m.cov_zd = __fma_rn(-m.mean_z, m.mean_d, s.sum_zd * inv);
    m.n_in_bucket = (unsigned long long)(s.n_in_bucket + 0.5);
    return m;
}

static __global__ void finalize_kernel(const double* __restrict__ partials, int nparts, size_t n,
                                unsigned long long* __restrict__ cursor, unsigned int* done,
                                MomentsOut* __restrict__ moments, SumsOut* __restrict__ sums,
                                unsigned long long* __restrict__ count_out) {
    __shared__ double sh[6][8];
    const double* mine = partials + (size_t)blockIdx.x * nparts * kPartialStride;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;   // blockDim.x == 256
    double v[6] = {0, 0, 0, 0, 0, 0};
    for (int p = threadIdx.x; p < nparts; p += blockDim.x) {
#pragma unroll
        for (int k = 0; k < 6; ++k) v[k] += mine[(size_t)p * kPartialStride + k];
    }
#pragma unroll
    for (int k = 0; k < 6; ++k) {
        v[k] = warp_sum(v[k]);
        if (lane == 0) sh[k][warp] = v[k];
    }
    __syncthreads();
    if (threadIdx.x == 0) {
        SumsOut s;
        double r[6];
        for (int k = 0; k < 6; ++k) {
            double a = 0.0;
            for (int w = 0; w < 8; ++w) a += sh[k][w];
            r[k] = a;
        }
        s.n = (double)n; s.sum_z = r[0]; s.sum_zz = r[1]; s.sum_d = r[2]; s.sum_dd = r[3];
        s.sum_zd = r[4]; s.n_in_bucket = r[5]; s.pad_ = 0.0;
        const unsigned long long t = (cursor ? *cursor : 0ULL) + blockIdx.x;
        if (sums) sums[t] = s;
        if (moments) moments[t] = moments_from(s);
        if (count_out) count_out[t] = (unsigned long long)(r[5] + 0.5);
        if (cursor) {
            __threadfence();
            if (atomicAdd(done, 1u) == gridDim.x - 1) {
                *done = 0u;
                *cursor += gridDim.x;
            }
        }
    }
}

static __global__ void set_cursor_kernel(unsigned long long* cursor, unsigned int* done,
                                  unsigned long long value) {
    *cursor = value;
    *done = 0u;
}

// ------------------------------------------------------------------------------------------
// FP64 roofline probe: CHAINS independent dependent-FMA chains per thread.
// ------------------------------------------------------------------------------------------
template <int CHAINS>
__global__ void probe_dfma_kernel(double* out, long long iters, double a, double b) {
    double x[CHAINS];
#pragma unroll
    for (int c = 0; c < CHAINS; ++c) x[c] = 1.0 + 1e-9 * (threadIdx.x + c);
    const int n16 = (int)(iters / 16);
    for (int i = 0; i < n16; ++i) {
#pragma unroll
        for (int u = 0; u < 16; ++u) {
#pragma unroll
            for (int c = 0; c < CHAINS; ++c) x[c] = __fma_rn(x[c], a, b);
        }
    }
    double s = 0.0;
#pragma unroll
    for (int c = 0; c < CHAINS; ++c) s += x[c];
    if (s == 12345.678) out[0] = s;   // never true; keeps the chains alive
}

}  // namespace lt
