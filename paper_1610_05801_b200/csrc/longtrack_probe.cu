// longtrack_probe.cu -- liblongtrack_probe.so: the FP64-pipe probes behind bench.py's roofline
// denominators (include/longtrack_probe.h).  Measurement tooling, NOT part of the product ABI:
// liblongtrack.so exports the calls of SURVEY.md sec. 8(b) and 8(f) only; nothing in it depends on
// this file.  Built from the same headers so that the probed turn loop is the kernel's own code.
// CUDA path only: nothing here includes, links or calls anything under oracle/.
#include "../../include/longtrack_probe.h"

#include <cuda_runtime.h>

#include "kernels.cuh"
#include "kernels_probe.cuh"
#include "sinpi_coeffs.h"

using namespace lt;

extern "C" {

int lt_probe_fp64(int blocks, int threads, int chains, long long iters, double* rate_host,
                  double* ms_host) {
    if (!rate_host) return LT_E_NULL;
    if (blocks < 1 || threads < 1 || threads > 1024 || iters < 16 || iters > (1LL << 34)) return LT_E_PARAM;
    double* out = nullptr;
    cudaEvent_t e0, e1;
    if (cudaMalloc(&out, sizeof(double)) != cudaSuccess) { (void)cudaGetLastError(); return LT_E_CUDA; }
    cudaEventCreate(&e0);
    cudaEventCreate(&e1);
    float ms = 0.f;
    for (int rep = 0; rep < 2; ++rep) {      // first repetition warms up
        cudaEventRecord(e0, 0);
        switch (chains) {
            case 1: probe_dfma_kernel<1><<<blocks, threads>>>(out, iters, 0.999999, 1e-6); break;
            case 2: probe_dfma_kernel<2><<<blocks, threads>>>(out, iters, 0.999999, 1e-6); break;
            case 4: probe_dfma_kernel<4><<<blocks, threads>>>(out, iters, 0.999999, 1e-6); break;
            case 8: probe_dfma_kernel<8><<<blocks, threads>>>(out, iters, 0.999999, 1e-6); break;
            default:
                cudaFree(out); cudaEventDestroy(e0); cudaEventDestroy(e1);
                return LT_E_PARAM;
        }
        cudaEventRecord(e1, 0);
        cudaError_t e = cudaEventSynchronize(e1);
        if (e != cudaSuccess || cudaGetLastError() != cudaSuccess) {
            cudaFree(out); cudaEventDestroy(e0); cudaEventDestroy(e1);
            return LT_E_CUDA;
        }
        cudaEventElapsedTime(&ms, e0, e1);
    }
    cudaFree(out);
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    *rate_host = (double)blocks * threads * chains * (double)(iters / 16 * 16) / (ms * 1e-3);
    if (ms_host) *ms_host = ms;
    return LT_OK;
}

}  // extern "C"

namespace {

template <int CHAINS>
cudaError_t launch_probe_pipe(int kind, int blocks, int threads, int iters, const ProbeConsts& P, double* out,
                              unsigned long long* cyc, unsigned long long* ns) {
#define LT_PP(K)                                                                                        \
    case K: {                                                                                           \
        auto kern = probe_pipe_kernel<CHAINS, K>;                                                       \
        cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, 120 * 1024); \
        if (e != cudaSuccess) return e;                                                                 \
        kern<<<blocks, threads, 120 * 1024>>>(out, iters, P, cyc, ns);                                  \
        return cudaGetLastError();                                                                      \
    }
    switch (kind) {
        LT_PP(0) LT_PP(1) LT_PP(2) LT_PP(3) LT_PP(10) LT_PP(11) LT_PP(12)
        default: return cudaErrorInvalidValue;
    }
#undef LT_PP
}

}  // namespace

extern "C" {

int lt_probe_pipe(int kind, int blocks, int threads, int chains, long long iters,
                  double* instr_per_cycle_host, double* sm_clock_mhz_host) {
    if (!instr_per_cycle_host) return LT_E_NULL;
    if (blocks < 1 || blocks > 1024 || threads < 32 || threads > 1024 || (threads & 31) || iters < 1 ||
        iters > (1LL << 28))
        return LT_E_PARAM;
    if (chains != 1 && chains != 2 && chains != 4) return LT_E_PARAM;
    if (kind != 0 && kind != 1 && kind != 2 && kind != 3 && kind != 10 && kind != 11 && kind != 12) return LT_E_PARAM;
    ProbeConsts P;
    for (int k = 0; k < 8; ++k) P.c[k] = (double)(7.6973252442360035e-5L * LT_SINPI_F64[k]);
    P.drift = 5.7; P.a = 0.999999; P.b = 1e-6;
    double* out = nullptr;
    unsigned long long* cyc = nullptr;
    if (cudaMalloc(&out, sizeof(double)) != cudaSuccess ||
        cudaMalloc(&cyc, 2 * sizeof(unsigned long long) * (size_t)blocks) != cudaSuccess) {
        (void)cudaGetLastError();
        if (out) cudaFree(out);
        return LT_E_CUDA;
    }
    unsigned long long* ns = cyc + blocks;
    cudaError_t e = cudaSuccess;
    for (int rep = 0; rep < 2 && e == cudaSuccess; ++rep) {     // first repetition warms up
        e = chains == 1 ? launch_probe_pipe<1>(kind, blocks, threads, (int)iters, P, out, cyc, ns)
          : chains == 2 ? launch_probe_pipe<2>(kind, blocks, threads, (int)iters, P, out, cyc, ns)
                        : launch_probe_pipe<4>(kind, blocks, threads, (int)iters, P, out, cyc, ns);
        if (e == cudaSuccess) e = cudaDeviceSynchronize();
    }
    int rc = LT_OK;
    if (e != cudaSuccess) {
        (void)cudaGetLastError();
        rc = LT_E_CUDA;
    } else {
        unsigned long long* h = (unsigned long long*)std::malloc(2 * sizeof(unsigned long long) * (size_t)blocks);
        if (!h) rc = LT_E_NOMEM;
        else if (cudaMemcpy(h, cyc, 2 * sizeof(unsigned long long) * (size_t)blocks, cudaMemcpyDeviceToHost) != cudaSuccess) {
            (void)cudaGetLastError();
            rc = LT_E_CUDA;
        } else {
            double mc = 0.0, mn = 0.0;
            for (int i = 0; i < blocks; ++i) { mc += (double)h[i]; mn += (double)h[blocks + i]; }
            mc /= blocks; mn /= blocks;
            const double per = kind >= 10 ? 13.0 : 1.0;        // FP64 instructions per step and chain
            const double warp_instr_per_smsp = (threads / 32) / 4.0 * chains * 8.0 * (double)iters * per;
            *instr_per_cycle_host = warp_instr_per_smsp / mc;
            if (sm_clock_mhz_host) *sm_clock_mhz_host = mn > 0.0 ? mc / mn * 1e3 : 0.0;
        }
        std::free(h);
    }
    cudaFree(out);
    cudaFree(cyc);
    return rc;
}

}  // extern "C"
