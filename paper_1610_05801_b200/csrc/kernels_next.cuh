// kernels_next.cuh -- sm_100a device code for the rows SURVEY.md sec. 8(f) marks "next":
//   f2  turn-dependent RF programme in per-turn mode      (PAPER.md:76;  DESIGN.md G28)
//       (its fused-mode form is the PROG option of kernels.cuh's persistent kernel)
//   f4  longitudinal slicing fused into the per-turn pass  (G29)
//   f3  transverse linear transfer maps                    (Fig. 2; G30)
// CUDA path only: shares nothing with oracle/.
#pragma once

#include "kernels.cuh"

namespace lt {

// ------------------------------------------------------------------------------------------
// f4: slice index of one particle (reading G29).  The decision is taken exactly as stated --
// one subtraction, one multiplication by inv = S/(z_hi - z_lo), each rounded once, no FMA --
// so that for the same z every implementation lands in the same slice.
//   0: z < z_lo ("below")    S+1: not (z < z_hi) ("above", NaN included)    1+s otherwise
// ------------------------------------------------------------------------------------------
__device__ __forceinline__ int slice_bin(double z, double z_lo, double z_hi, double inv, int S) {
    // Branch-free (the histogram pass is bound by instruction issue, not by its loads: with an early
    // return per case it was 18 instructions and two branches per particle).
    const double d = __dsub_rn(z, z_lo);
    const double u = __dmul_rn(d, inv);                    // in range: 0 <= u < 2^21
    // floor(u) without a conversion: 2^52 + u rounded toward -inf carries floor(u) in its low
    // mantissa word, exactly (F2I.F64 runs at a quarter of the FP64 rate; this is one DADD)
    const int s = __double2loint(__dadd_rd(u, 4503599627370496.0));
    const int in = 1 + min(s, S - 1);                      // meaningful only for z_lo <= z < z_hi
    const int lo_or_in = (z < z_lo) ? 0 : in;              // "below" (a sign test of d would misplace z = -0.0 at z_lo = 0)
    return (z < z_hi) ? lo_or_in : S + 1;                  // not (z < z_hi): "above", NaN included
}

// What the per-turn kernel needs beyond the plain map; every field is uniform over the grid.
struct TurnExtras {
    const double* volt_scale;            // [turns] a_t or nullptr (device)
    const double* phase_off;             // [turns] psi_t in rad or nullptr (device)
    const unsigned long long* cursor;    // absolute index of the batch's first turn (device)
    int k;                               // this launch's turn within the batch
    double inv_pi;
    unsigned long long* hist;            // [turns][S+2] or nullptr (device), zeroed by the caller
    double z_lo, z_hi, inv;
    int n_slices;
    int replicas;                        // shared-memory copies of the histogram; 0 = global atomics
};

// CTA-private histogram in shared memory, `replicas` copies indexed by lane so that the
// particles of one warp that fall into the same slice do not serialise on one address (a
// Gaussian bunch puts 40 % of the particles into the 10 central slices of 64).  Copy-major with
// an odd stride; a counter-major layout (bank = lane, no bank conflicts at all) measured no
// faster: the kernel is bound by its loads, not by the shared atomics
// (profiles/r2_histogram.md).
struct SliceAcc {
    unsigned int* sh;
    unsigned int* mine;                  // this lane's copy
    unsigned long long* out;
    double z_lo, z_hi, inv;
    int S, stride, rep_mask;
    __device__ __forceinline__ void init(const TurnExtras& X, unsigned long long turn,
                                         unsigned int* smem) {
        sh = smem; S = X.n_slices; stride = (S + 2) | 1; rep_mask = X.replicas - 1;   // odd stride: the copies of one slice sit in different banks
        z_lo = X.z_lo; z_hi = X.z_hi; inv = X.inv;
        out = X.hist + turn * (unsigned long long)(S + 2);
        mine = sh + ((int)(threadIdx.x & 31u) & rep_mask) * stride;
        if (X.replicas > 0) {
            for (int i = threadIdx.x; i < X.replicas * stride; i += blockDim.x) sh[i] = 0u;
            __syncthreads();
        }
    }
    __device__ __forceinline__ void add(double z) {
        const int b = slice_bin(z, z_lo, z_hi, inv, S);
        if (rep_mask >= 0) atomicAdd(mine + b, 1u);
        else atomicAdd(out + b, 1ULL);
    }
    __device__ __forceinline__ void flush() {
        if (rep_mask < 0) return;
        __syncthreads();
        for (int b = threadIdx.x; b < S + 2; b += blockDim.x) {
            unsigned int c = 0u;
            for (int r = 0; r <= rep_mask; ++r) c += sh[r * stride + b];
            if (c) atomicAdd(out + b, (unsigned long long)c);
        }
    }
};

// ------------------------------------------------------------------------------------------
// Per-turn kernel with the f2 / f4 extras: the structure of per_turn_kernel (persistent CTAs,
// double2 tiles, all loads of a tile before its arithmetic, moments fused), plus
//   - the turn's programme entry (a_t, psi_t/pi), read once per CTA from the device tables at
//     index *cursor + k (the cursor lives on the device so one CUDA graph serves every batch);
//   - the slice histogram of z after the turn, in shared memory, flushed with one 64-bit
//     atomic per non-empty slice and CTA (integer adds: the result is order-independent).
// Still 32 B of HBM traffic per particle-turn.
// ------------------------------------------------------------------------------------------
template <int INTEG, int HARM, bool MOMENTS, int UNR>
__global__ void per_turn_extra_kernel(double* __restrict__ z_arr, double* __restrict__ d_arr,
                                      size_t n, int reverse, double* __restrict__ partials,
                                      const __grid_constant__ MapConsts<double> P,
                                      const __grid_constant__ TurnExtras X) {
    extern __shared__ unsigned int slice_smem[];
    const unsigned long long turn = *X.cursor + (unsigned long long)X.k;
    const bool prog = X.volt_scale != nullptr;
    const bool slices = X.hist != nullptr;
    double a = 1.0, p = 0.0;
    if (prog) {
        a = __ldg(X.volt_scale + turn);
        p = __dmul_rn(__ldg(X.phase_off + turn), X.inv_pi);
    }
    SliceAcc sl;
    if (slices) sl.init(X, turn, slice_smem);
    Sums acc;
    acc.zero();
    const size_t npair = n >> 1;
    const size_t tile_pairs = (size_t)blockDim.x * UNR;
    const size_t ntiles = (npair + tile_pairs - 1) / tile_pairs;
    for (size_t tl = blockIdx.x; tl < ntiles; tl += gridDim.x) {
        const size_t tix = reverse ? (ntiles - 1 - tl) : tl;
        const size_t base = tix * tile_pairs;
        double2 zz[UNR], dd[UNR];
#pragma unroll
        for (int u = 0; u < UNR; ++u) {
            size_t q = base + (size_t)u * blockDim.x + threadIdx.x;
            if (q < npair) {
                zz[u] = reinterpret_cast<const double2*>(z_arr)[q];
                dd[u] = reinterpret_cast<const double2*>(d_arr)[q];
            }
        }
#pragma unroll
        for (int u = 0; u < UNR; ++u) {
            size_t q = base + (size_t)u * blockDim.x + threadIdx.x;
            if (q < npair) {
                if (prog) {
                    turn_exact<double, INTEG, HARM, true>(zz[u].x, dd[u].x, P, a, p);
                    turn_exact<double, INTEG, HARM, true>(zz[u].y, dd[u].y, P, a, p);
                } else {
                    turn_exact<double, INTEG, HARM>(zz[u].x, dd[u].x, P);
                    turn_exact<double, INTEG, HARM>(zz[u].y, dd[u].y, P);
                }
                reinterpret_cast<double2*>(z_arr)[q] = zz[u];
                reinterpret_cast<double2*>(d_arr)[q] = dd[u];
                if (MOMENTS) {
                    acc.add(zz[u].x, dd[u].x, in_bucket<double>(zz[u].x, dd[u].x, P));
                    acc.add(zz[u].y, dd[u].y, in_bucket<double>(zz[u].y, dd[u].y, P));
                }
                if (slices) { sl.add(zz[u].x); sl.add(zz[u].y); }
            }
        }
    }
    if ((n & 1) && blockIdx.x == 0 && threadIdx.x == 0) {
        double z1 = z_arr[n - 1], d1 = d_arr[n - 1];
        if (prog) turn_exact<double, INTEG, HARM, true>(z1, d1, P, a, p);
        else turn_exact<double, INTEG, HARM>(z1, d1, P);
        z_arr[n - 1] = z1; d_arr[n - 1] = d1;
        if (MOMENTS) acc.add(z1, d1, in_bucket<double>(z1, d1, P));
        if (slices) sl.add(z1);
    }
    if (slices) sl.flush();
    if (MOMENTS) block_reduce_store(acc, partials + (size_t)blockIdx.x * kPartialStride);
}

// scalar variant for arrays that are not 16-byte aligned (moments decided at run time)
template <int INTEG, int HARM>
__global__ void per_turn_extra_kernel_scalar(double* __restrict__ z_arr, double* __restrict__ d_arr,
                                             size_t n, int moments, double* __restrict__ partials,
                                             const __grid_constant__ MapConsts<double> P,
                                             const __grid_constant__ TurnExtras X) {
    extern __shared__ unsigned int slice_smem[];
    const unsigned long long turn = *X.cursor + (unsigned long long)X.k;
    const bool prog = X.volt_scale != nullptr;
    const bool slices = X.hist != nullptr;
    double a = 1.0, p = 0.0;
    if (prog) {
        a = __ldg(X.volt_scale + turn);
        p = __dmul_rn(__ldg(X.phase_off + turn), X.inv_pi);
    }
    SliceAcc sl;
    if (slices) sl.init(X, turn, slice_smem);
    Sums acc;
    acc.zero();
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n;
         i += (size_t)gridDim.x * blockDim.x) {
        double z1 = z_arr[i], d1 = d_arr[i];
        if (prog) turn_exact<double, INTEG, HARM, true>(z1, d1, P, a, p);
        else turn_exact<double, INTEG, HARM>(z1, d1, P);
        z_arr[i] = z1; d_arr[i] = d1;
        if (moments) acc.add(z1, d1, in_bucket<double>(z1, d1, P));
        if (slices) sl.add(z1);
    }
    if (slices) sl.flush();
    if (moments) block_reduce_store(acc, partials + (size_t)blockIdx.x * kPartialStride);
}

// Advances the device turn cursor when a batch has no finalize launch to do it.
static __global__ void advance_cursor_kernel(unsigned long long* cursor, unsigned long long by) {
    *cursor += by;
}

// Histogram of a given state (lt_slice_histogram): 8 B read per particle, HBM bound.
// One wave of persistent CTAs (grid = a multiple of the SM count, 512 threads); every thread
// keeps TWO tiles of UNR 16-byte loads in flight: the loads of tile k+1 are issued before the
// shared-memory atomics of tile k (128 B per thread; the first version issued a tile's loads only
// after the previous tile's atomics and ran 1184 short-lived CTAs whose zero / load / flush
// phases coincided: 3.7 TB/s in the kernel, profiles/r1_next_rows_ncu.md).
// No memset launch and no serial tail: CTA 0 zeroes the caller's histogram while its first tile is
// in flight and then sets flag[0] = 1 (release); every CTA streams its share into its
// shared-memory copies and, ~15 us later, adds them to the caller's histogram after an
// acquire-read of flag[0] (CTA 0 is normally the first CTA dispatched, so the flag is hardly ever
// waited on; correctness does not rest on that -- the grid is one wave, CTA 0 is resident).
// The protocol's state lives on the DEVICE only: each CTA signs off in flag[1] once it is past the
// wait, and the last one to do so puts both words back to 0, which is what the next launch --
// stream-ordered behind this one -- starts from.  No per-call value comes from the host, so a
// launch replayed from a CUDA graph behaves like a fresh call (round 2 passed a host-side call
// number as a kernel argument, which a replay would have repeated).
// Round 2's first version summed into a tracker-owned accumulator
// that the LAST CTA copied out: a serial fence + ticket + copy behind the slowest CTA.
// flag == nullptr: the caller zeroed `out` (more slices than the shared-memory path holds).
// A z array that is only 8-byte aligned is shifted by one element (`head`).
template <int UNR>
static __global__ void __launch_bounds__(512)
slice_histogram_kernel(const double* __restrict__ z_arr, size_t n, const __grid_constant__ TurnExtras X,
                       unsigned int* __restrict__ flag) {
    extern __shared__ unsigned int slice_smem[];
    const size_t head = ((reinterpret_cast<uintptr_t>(z_arr) & 15u) != 0 && n > 0) ? 1 : 0;
    const double* __restrict__ zb = z_arr + head;
    const size_t m = n - head;
    const size_t tile = (size_t)blockDim.x * 2 * UNR;
    const size_t stride = (size_t)gridDim.x * tile;
    size_t base = (size_t)blockIdx.x * tile;
    double2 cur[UNR];
    bool have = base + tile <= m;
    if (have) {                               // the first tile is on its way while the counters are zeroed
#pragma unroll
        for (int u = 0; u < UNR; ++u)
            cur[u] = __ldcs(reinterpret_cast<const double2*>(zb + base) + u * blockDim.x + threadIdx.x);
    }
    if (flag && blockIdx.x == 0) {
        for (int b = threadIdx.x; b < X.n_slices + 2; b += blockDim.x) X.hist[b] = 0ULL;
        __threadfence();
        __syncthreads();
        if (threadIdx.x == 0) st_release_u32(flag, 1u);
    }
    SliceAcc sl;
    sl.init(X, 0ULL, slice_smem);
    if (head && blockIdx.x == 0 && threadIdx.x == 0) sl.add(z_arr[0]);
    while (have) {
        const size_t nb = base + stride;
        const bool more = nb + tile <= m;
        double2 nxt[UNR];
        if (more) {
#pragma unroll
            for (int u = 0; u < UNR; ++u)
                nxt[u] = __ldcs(reinterpret_cast<const double2*>(zb + nb) + u * blockDim.x + threadIdx.x);
        }
#pragma unroll
        for (int u = 0; u < UNR; ++u) { sl.add(cur[u].x); sl.add(cur[u].y); }
#pragma unroll
        for (int u = 0; u < UNR; ++u) cur[u] = nxt[u];
        base = nb;
        have = more;
    }
    // `base` is this CTA's first tile that is not full: at most one ragged tile in the whole grid
    for (size_t i = base + threadIdx.x; i < m && base < m; i += blockDim.x) {
        if (i < base + tile) sl.add(zb[i]);
    }
    if (flag && threadIdx.x == 0) {
        if (blockIdx.x != 0) {                // the histogram has been zeroed by THIS launch
            while (ld_acquire_u32(flag) != 1u) __nanosleep(32);
        }
        // past the wait: sign off; the last CTA to do so re-arms both words for the next launch
        if (atomicAdd(flag + 1, 1u) == gridDim.x - 1) {
            flag[1] = 0u;
            st_release_u32(flag, 0u);
        }
        // SliceAcc::flush starts with a __syncthreads(), which orders every thread behind the acquire
    }
    sl.flush();
}

// Programme table of one fused launch, double2 per turn behind a one-entry header:
//   exact path:  out[1 + i] = (a_T, p_T),          p_T = psi_T / pi,  T = t_first + i
//   fast path:   out[1 + i] = (a_T, p_(T+1) - p_T), with p_(call_turns) := 0 (the state leaves the
//                call as the plain phase);  out[0].y = p_(t_first) for the launch's first turn.
static __global__ void programme_pack_kernel(const double* __restrict__ volt_scale,
                                      const double* __restrict__ phase_off,
                                      unsigned long long t_first, unsigned int count,
                                      unsigned long long call_turns, double inv_pi, int fast,
                                      double2* __restrict__ out) {
    const unsigned int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= count) return;
    const unsigned long long T = t_first + i;
    const double p = __dmul_rn(phase_off[T], inv_pi);
    if (i == 0) out[0] = make_double2(0.0, p);
    if (fast) {
        const double pn = (T + 1 < call_turns) ? __dmul_rn(phase_off[T + 1], inv_pi) : 0.0;
        out[1 + i] = make_double2(volt_scale[T], __dsub_rn(pn, p));
    } else {
        out[1 + i] = make_double2(volt_scale[T], p);
    }
}

// ------------------------------------------------------------------------------------------
// f3: transverse plane.  One turn = for every segment s in order  u <- M_s u,  u = (x, x', y, y'),
// M_s row-major; row i is  fma(M_i3, y', fma(M_i2, y, fma(M_i1, x', M_i0 * x)))  -- the
// association order of the definition, 16 FP64 instructions per segment and particle.
// sm_100a has no constant-bank operands for DFMA: every matrix element has to sit in a register.
// Two homes for the lattice: shared memory (any length; a thread carries ILP particles, so each
// 16-byte fetch of a matrix row feeds 2*ILP FP64 instructions, all in the three-register form), or
// the kernel-parameter space for short lattices (LatticeParam below: uniform registers, the
// two-register form, no fetches from shared memory at all).
// ------------------------------------------------------------------------------------------
constexpr int kSegUnrolled = 4;      // lattices up to this length are unrolled at compile time

__device__ __forceinline__ void apply_matrix(double (&u)[4], const double* __restrict__ M) {
    double w[4];
#pragma unroll
    for (int i = 0; i < 4; ++i) {
        double acc = __dmul_rn(M[4 * i], u[0]);
        acc = __fma_rn(M[4 * i + 1], u[1], acc);
        acc = __fma_rn(M[4 * i + 2], u[2], acc);
        w[i] = __fma_rn(M[4 * i + 3], u[3], acc);
    }
#pragma unroll
    for (int i = 0; i < 4; ++i) u[i] = w[i];
}

// 16-byte shared-memory load that ptxas may not hoist: left alone it lifts the loads of a short
// lattice out of the turn loop into (uniform) registers and then spills the particles' state
__device__ __forceinline__ double2 lds_pair(unsigned int addr) {
    double2 r;
    asm volatile("ld.shared.v2.f64 {%0, %1}, [%2];" : "=d"(r.x), "=d"(r.y) : "r"(addr));
    return r;
}

// the same for ILP particles of one thread: a matrix row is read once (two 16-byte loads from
// shared memory at byte address M) and feeds 4*ILP FP64 instructions
template <int ILP>
__device__ __forceinline__ void apply_matrix_ilp(double (&u)[ILP][4], unsigned int M) {
    double w[ILP][4];
#pragma unroll
    for (int i = 0; i < 4; ++i) {
        const double2 a = lds_pair(M + 32u * i), b = lds_pair(M + 32u * i + 16u);
#pragma unroll
        for (int j = 0; j < ILP; ++j) {
            double acc = __dmul_rn(a.x, u[j][0]);
            acc = __fma_rn(a.y, u[j][1], acc);
            acc = __fma_rn(b.x, u[j][2], acc);
            w[j][i] = __fma_rn(b.y, u[j][3], acc);
        }
    }
#pragma unroll
    for (int j = 0; j < ILP; ++j)
#pragma unroll
        for (int i = 0; i < 4; ++i) u[j][i] = w[j][i];
}

template <int NSEG, int ILP>
__device__ __forceinline__ void transverse_turn(double (&u)[ILP][4], unsigned int lat, int n_seg) {
    if (NSEG > 0) {
#pragma unroll
        for (int s = 0; s < NSEG; ++s) apply_matrix_ilp<ILP>(u, lat + 128u * s);
    } else {
#pragma unroll 1
        for (int s = 0; s < n_seg; ++s) apply_matrix_ilp<ILP>(u, lat + 128u * s);
    }
}

// The lattice as a KERNEL PARAMETER (constant bank), for lattices of up to kParamSegments segments:
// inside a segment loop that is NOT unrolled, ptxas fetches the 16 elements of the segment with
// uniform loads (LDCU c[0x0][UR + off]) into uniform registers and every FP64 instruction of the
// matrix product takes the form  DFMA R, R, UR, R  -- two vector-register operands, which the FP64
// pipe issues every 2.00 cycles, against 2.17 for the three-register form a matrix element fetched
// from shared memory forces (profiles/r2_fp64_pipe_probe.md) -- and no shared-memory loads at all.
// Two conditions, both found by bisecting the SASS: (1) the segment count is read from the
// parameter struct itself and the loop is not unrolled (unrolled, ptxas hoists the loads out of
// the turn loop into vector registers and moves them back with R2UR, spilling); (2) ptxas must
// see the work item as warp-uniform and the warp CONVERGED around the turn loop: the item index is
// broadcast with __shfl_sync in every scheduling mode, and the work-item loop ends in a
// __syncwarp() -- a trailing `if (lane == 0) store` without one is enough to make ptxas keep the
// segment counter in a vector register and fetch the elements with LDC into vector registers
// (0.74 of the peak instead of 0.88).
constexpr int kParamSegments = 24;                      // 3 KB of the 4 KB parameter space
struct LatticeParam { double m[kParamSegments][16]; int n_seg; };

template <int ILP>
__device__ __forceinline__ void apply_matrix_param(double (&u)[ILP][4], const double (&M)[16]) {
    double w[ILP][4];
#pragma unroll
    for (int i = 0; i < 4; ++i) {
#pragma unroll
        for (int j = 0; j < ILP; ++j) {
            double acc = __dmul_rn(M[4 * i], u[j][0]);
            acc = __fma_rn(M[4 * i + 1], u[j][1], acc);
            acc = __fma_rn(M[4 * i + 2], u[j][2], acc);
            w[j][i] = __fma_rn(M[4 * i + 3], u[j][3], acc);
        }
    }
#pragma unroll
    for (int j = 0; j < ILP; ++j)
#pragma unroll
        for (int i = 0; i < 4; ++i) u[j][i] = w[j][i];
}

// where a kernel's lattice lives: shared memory (any length) or the parameter space
struct LatticeInShared {
    unsigned int base; int n_seg;
    template <int NSEG, int ILP> __device__ __forceinline__ void turn(double (&u)[ILP][4]) const {
        transverse_turn<NSEG, ILP>(u, base, n_seg);
    }
};
struct LatticeInParam {
    const LatticeParam& L;
    template <int NSEG, int ILP> __device__ __forceinline__ void turn(double (&u)[ILP][4]) const {
#pragma unroll 1
        for (int s = 0; s < L.n_seg; ++s) apply_matrix_param<ILP>(u, L.m[s]);
    }
};

// Fused multi-turn transverse kernel: the persistent, ticketed work queue of
// fused_persistent_kernel (items = chunk of item_turns turns x group of 32*ILP particles) with the
// four transverse coordinates -- and, when LONGI, the leap-frog single-harmonic longitudinal
// turn of the same particle (fast path: phase state, merged drifts) -- held in registers.
// Particle j of a lane is element  g*32*ILP + j*32 + lane  (coalesced).  The arithmetic per
// particle does not depend on ILP, so every launch shape returns the same bits.
template <int NSEG, bool LONGI, int ILP, typename LAT>
__device__ __forceinline__ void
transverse_persistent_body(double* __restrict__ x_arr, double* __restrict__ xp_arr,
                             double* __restrict__ y_arr, double* __restrict__ yp_arr,
                             double* __restrict__ z_arr, double* __restrict__ d_arr, size_t n,
                             unsigned int turns, unsigned int item_turns, int first_launch,
                             int last_launch, int dynamic, unsigned long long* __restrict__ ticket,
                             unsigned int* __restrict__ done, const LAT lat,
                             const MapConsts<double>& P) {
    constexpr unsigned int G = 32u * ILP;
    const unsigned int lane = threadIdx.x & 31u;
    const unsigned long long groups = (n + G - 1) / G;
    ItemSchedule sched;
    sched.init(turns, item_turns, dynamic);
    const unsigned int nchunks = sched.nchunks;
    const unsigned long long total = groups * nchunks;
    const unsigned long long slots = (unsigned long long)gridDim.x * (blockDim.x >> 5);
    unsigned long long next = (unsigned long long)(threadIdx.x >> 5) * gridDim.x + blockIdx.x;
    for (;;) {
        unsigned long long t = next;
        if (dynamic) {
            if (lane == 0) t = atomicAdd(ticket, 1ULL);
        } else {
            next += slots;
        }
        // also in static mode, where every lane already holds the same t: the broadcast is what
        // tells ptxas that the work item -- and with it every loop below -- is warp-uniform
        t = __shfl_sync(0xffffffffu, t, 0);
        if (t >= total) break;
        const unsigned int c = (unsigned int)(t / groups);
        const unsigned long long g = t - (unsigned long long)c * groups;
        if (c > 0) {
            while (ld_acquire_u32(done + g) < c) __nanosleep(64);
        }
        const size_t i0 = (size_t)g * G + lane;
        const int first = first_launch && c == 0;
        const int last = last_launch && c == nchunks - 1;
        unsigned int t_start, nt;
        sched.span(c, dynamic, &t_start, &nt);
        double u[ILP][4], v[ILP], dl[ILP];
#pragma unroll
        for (int j = 0; j < ILP; ++j) {
            const size_t i = i0 + 32u * j;
            const bool live = i < n;
            u[j][0] = live ? __ldcg(x_arr + i) : 0.0;
            u[j][1] = live ? __ldcg(xp_arr + i) : 0.0;
            u[j][2] = live ? __ldcg(y_arr + i) : 0.0;
            u[j][3] = live ? __ldcg(yp_arr + i) : 0.0;
            v[j] = 0.0; dl[j] = 0.0;
            if (LONGI) {
                v[j] = live ? __ldcg(z_arr + i) : 0.0;
                dl[j] = live ? __ldcg(d_arr + i) : 0.0;
                if (first) v[j] = __fma_rn(-P.drift_lead, dl[j], __dmul_rn(v[j], P.to_phase));
            }
        }
#pragma unroll 1
        for (unsigned int k = 1; k < nt; ++k) {
            lat.template turn<NSEG, ILP>(u);
            if (LONGI) {
#pragma unroll
                for (int j = 0; j < ILP; ++j)
                    turn_fast<double, kLeapfrog, 1, true>(v[j], dl[j], P, P.drift_merged);
            }
        }
        lat.template turn<NSEG, ILP>(u);
#pragma unroll
        for (int j = 0; j < ILP; ++j) {
            const size_t i = i0 + 32u * j;
            if (LONGI) {
                turn_fast<double, kLeapfrog, 1, true>(v[j], dl[j], P, last ? P.drift_trail : P.drift_merged);
                if (last) v[j] = __dmul_rn(v[j], P.from_phase);
            }
            if (i < n) {
                __stcg(x_arr + i, u[j][0]); __stcg(xp_arr + i, u[j][1]);
                __stcg(y_arr + i, u[j][2]); __stcg(yp_arr + i, u[j][3]);
                if (LONGI) { __stcg(z_arr + i, v[j]); __stcg(d_arr + i, dl[j]); }
            }
        }
        if (nchunks > 1) {
            __threadfence();
            __syncwarp();
            if (lane == 0) st_release_u32(done + g, c + 1);
        }
        __syncwarp();            // ptxas must see the warp converged at the next work item (LatticeInParam)
    }
}

template <int NSEG, bool LONGI, int ILP>
__global__ void __launch_bounds__(ILP == 1 ? 1024 : (ILP == 8 ? 256 : 512), 1)
transverse_persistent_kernel(double* __restrict__ x_arr, double* __restrict__ xp_arr,
                             double* __restrict__ y_arr, double* __restrict__ yp_arr,
                             double* __restrict__ z_arr, double* __restrict__ d_arr, size_t n,
                             unsigned int turns, unsigned int item_turns, int first_launch,
                             int last_launch, int dynamic, unsigned long long* __restrict__ ticket,
                             unsigned int* __restrict__ done, const double* __restrict__ Mg,
                             int n_seg, const __grid_constant__ MapConsts<double> P) {
    // dynamic shared memory: the lattice; the request is padded to cap the CTAs per SM
    extern __shared__ double2 lattice2[];
    for (int k = threadIdx.x; k < 8 * n_seg; k += blockDim.x)
        lattice2[k] = __ldg(reinterpret_cast<const double2*>(Mg) + k);
    __syncthreads();
    const LatticeInShared lat = {(unsigned int)__cvta_generic_to_shared(lattice2), n_seg};
    transverse_persistent_body<NSEG, LONGI, ILP>(x_arr, xp_arr, y_arr, yp_arr, z_arr, d_arr, n, turns, item_turns,
                                                 first_launch, last_launch, dynamic, ticket, done, lat, P);
}

// the same kernel with the lattice in the parameter space (n_seg <= kParamSegments)
template <bool LONGI, int ILP>
__global__ void __launch_bounds__(ILP == 1 ? 1024 : (ILP == 8 ? 256 : 512), 1)
transverse_persistent_param_kernel(double* __restrict__ x_arr, double* __restrict__ xp_arr,
                                   double* __restrict__ y_arr, double* __restrict__ yp_arr,
                                   double* __restrict__ z_arr, double* __restrict__ d_arr, size_t n,
                                   unsigned int turns, unsigned int item_turns, int first_launch,
                                   int last_launch, int dynamic, unsigned long long* __restrict__ ticket,
                                   unsigned int* __restrict__ done,
                                   const __grid_constant__ LatticeParam Lp,
                                   const __grid_constant__ MapConsts<double> P) {
    extern __shared__ double2 lattice2[];               // residency cap only
    const LatticeInParam lat = {Lp};
    transverse_persistent_body<0, LONGI, ILP>(x_arr, xp_arr, y_arr, yp_arr, z_arr, d_arr, n, turns, item_turns,
                                              first_launch, last_launch, dynamic, ticket, done, lat, P);
}

// Per-turn transverse kernel: ONE turn per launch, all coordinates through HBM -- 64 B per
// particle-turn for the transverse plane, 96 B with the longitudinal plane (LONGI: leap-frog,
// single harmonic, exact path = bit-identical to per_turn_kernel).  The lattice (n_seg x 16
// doubles) is staged in shared memory once per CTA.  VEC: every array is 16-byte aligned.
template <bool LONGI, bool VEC>
__global__ void transverse_per_turn_kernel(double* __restrict__ x_arr, double* __restrict__ xp_arr,
                                           double* __restrict__ y_arr, double* __restrict__ yp_arr,
                                           double* __restrict__ z_arr, double* __restrict__ d_arr,
                                           size_t n, int reverse, const double* __restrict__ Mg,
                                           int n_seg, const __grid_constant__ MapConsts<double> P) {
    extern __shared__ double lattice[];
    for (int k = threadIdx.x; k < 16 * n_seg; k += blockDim.x) lattice[k] = Mg[k];
    __syncthreads();
    if (VEC) {
        const size_t npair = n >> 1;
        const size_t ntiles = (npair + blockDim.x - 1) / blockDim.x;
        for (size_t tl = blockIdx.x; tl < ntiles; tl += gridDim.x) {
            const size_t tix = reverse ? (ntiles - 1 - tl) : tl;
            const size_t q = tix * blockDim.x + threadIdx.x;
            if (q >= npair) continue;
            const double2 a0 = reinterpret_cast<const double2*>(x_arr)[q];
            const double2 a1 = reinterpret_cast<const double2*>(xp_arr)[q];
            const double2 a2 = reinterpret_cast<const double2*>(y_arr)[q];
            const double2 a3 = reinterpret_cast<const double2*>(yp_arr)[q];
            double2 zz, dd;
            if (LONGI) {
                zz = reinterpret_cast<const double2*>(z_arr)[q];
                dd = reinterpret_cast<const double2*>(d_arr)[q];
            }
            double u[4] = {a0.x, a1.x, a2.x, a3.x}, w[4] = {a0.y, a1.y, a2.y, a3.y};
            for (int s = 0; s < n_seg; ++s) {
                apply_matrix(u, lattice + 16 * s);
                apply_matrix(w, lattice + 16 * s);
            }
            reinterpret_cast<double2*>(x_arr)[q] = make_double2(u[0], w[0]);
            reinterpret_cast<double2*>(xp_arr)[q] = make_double2(u[1], w[1]);
            reinterpret_cast<double2*>(y_arr)[q] = make_double2(u[2], w[2]);
            reinterpret_cast<double2*>(yp_arr)[q] = make_double2(u[3], w[3]);
            if (LONGI) {
                turn_exact<double, kLeapfrog, 1>(zz.x, dd.x, P);
                turn_exact<double, kLeapfrog, 1>(zz.y, dd.y, P);
                reinterpret_cast<double2*>(z_arr)[q] = zz;
                reinterpret_cast<double2*>(d_arr)[q] = dd;
            }
        }
    }
    // scalar path: everything when !VEC, the odd last particle when VEC
    const size_t i0 = VEC ? ((n & ~(size_t)1) + (size_t)blockIdx.x * blockDim.x + threadIdx.x)
                          : ((size_t)blockIdx.x * blockDim.x + threadIdx.x);
    for (size_t i = i0; i < n; i += (size_t)gridDim.x * blockDim.x) {
        double u[4] = {x_arr[i], xp_arr[i], y_arr[i], yp_arr[i]};
        for (int s = 0; s < n_seg; ++s) apply_matrix(u, lattice + 16 * s);
        x_arr[i] = u[0]; xp_arr[i] = u[1]; y_arr[i] = u[2]; yp_arr[i] = u[3];
        if (LONGI) {
            double z1 = z_arr[i], d1 = d_arr[i];
            turn_exact<double, kLeapfrog, 1>(z1, d1, P);
            z_arr[i] = z1; d_arr[i] = d1;
        }
    }
}

}  // namespace lt
