// kernels_probe.cuh -- FP64-pipe probes behind lt_probe_pipe (measurement only, not on the hot
// path).  They answer, on the device at hand, what the roofline of the fused mode is made of:
//   kind 0  DFMA, three register operands          kind 1  DFMA, two registers + one uniform operand
//   kind 2  DADD                                   kind 3  DMUL
//   kind 10 the 13-instruction leap-frog turn of kernels.cuh, sign flip on q (1 IMAD)
//   kind 11 the same, sign flip on f               kind 12 the same without any sign flip
// Each thread runs CHAINS independent dependent chains; the rate is counted with clock64, so it
// is in FP64 warp-instructions per cycle and sub-partition whatever the clock does.
// CUDA path only: shares nothing with oracle/.
#pragma once

#include "kernels.cuh"

namespace lt {

struct ProbeConsts { double c[8]; double drift, a, b; };

template <int CHAINS, int KIND>
__global__ void __launch_bounds__(1024, 1)
probe_pipe_kernel(double* out, int iters, const __grid_constant__ ProbeConsts P,
                  unsigned long long* __restrict__ cycles, unsigned long long* __restrict__ nanos) {
    typedef Real<double> R;
    double v[CHAINS], d[CHAINS];
#pragma unroll
    for (int c = 0; c < CHAINS; ++c) { v[c] = 0.1 + 1e-3 * (threadIdx.x + c); d[c] = 1e-3; }
    // kind 0 wants its multiplier and addend in REGISTERS: make them thread-dependent
    const double ra = P.a + 1e-30 * threadIdx.x, rb = P.b + 1e-30 * threadIdx.x;
    const double s = 0.25 + 1e-9 * threadIdx.x;
    __syncthreads();
    unsigned long long t0;
    asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t0));
    const unsigned long long c0 = clock64();
    // the turn kinds are unrolled as deep as the kernel's own turn loop (LT_TURN_UNROLL particle-turns)
    constexpr int kOuter = KIND >= 10 && LT_TURN_UNROLL / (8 * CHAINS) > 1 ? LT_TURN_UNROLL / (8 * CHAINS) : 1;
#pragma unroll kOuter
    for (int i = 0; i < iters; ++i) {
#pragma unroll
        for (int u = 0; u < 8; ++u) {
#pragma unroll
            for (int c = 0; c < CHAINS; ++c) {
                if (KIND == 0) v[c] = __fma_rn(v[c], ra, rb);
                else if (KIND == 1) v[c] = __fma_rn(v[c], s, P.c[u]);
                else if (KIND == 2) v[c] = __dadd_rn(v[c], s);
                else if (KIND == 3) v[c] = __dmul_rn(v[c], ra);
                else {
                    double t;
                    const double f = reduce_half_periods(v[c], &t);
                    const double ss = __dmul_rn(f, f);
                    const double q = horner<double, 8>(P.c, ss);
                    if (KIND == 10) d[c] = __fma_rn(f, R::flip(q, t), d[c]);
                    else if (KIND == 11) d[c] = __fma_rn(R::flip(f, t), q, d[c]);
                    else d[c] = __fma_rn(f, q, d[c]);
                    v[c] = __fma_rn(-P.drift, d[c], v[c]);
                }
            }
        }
    }
    const unsigned long long c1 = clock64();
    unsigned long long t1;
    asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t1));
    double acc = 0.0;
#pragma unroll
    for (int c = 0; c < CHAINS; ++c) acc += v[c] + d[c];
    if (acc == 12345.678) out[0] = acc;   // never true; keeps the chains alive
    if (threadIdx.x == 0) { cycles[blockIdx.x] = c1 - c0; nanos[blockIdx.x] = t1 - t0; }
}

}  // namespace lt
