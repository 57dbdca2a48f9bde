// longtrack_static.cu -- lt_moments_now_static: the moments / bucket-membership observables of
// lt_moments_now for callers that must not allocate device memory (include/longtrack.h).
//
// lt_moments_now keeps its per-CTA partial sums in a tracker-owned buffer that the first call
// (and any call with a larger grid) obtains from cudaMallocAsync.  Some users of this library
// cannot afford that: a tracking service that hands the whole device to its own pool at start-up
// and has nothing left for the driver's allocator, a turn-by-turn monitoring loop next to the
// machine that may not stall on (or fail in) an allocation half-way through a fill, a plug-in
// running inside a host application whose rules forbid touching the CUDA heap.  For them the
// same reduction is offered here with the partial sums in a fixed array that is part of the
// library image: it exists on every GPU from the moment the library is loaded there until the
// process exits, costs kStaticBytes (128 KB) of device memory per GPU, and needs no allocation,
// no free and no allocating library routine -- the price is a maximum particle count
// (LT_STATIC_MAX_PARTICLES) and one array shared by every caller in the process.
//
// CUDA path only: nothing here includes, links or calls anything under oracle/.
#include "tracker.hpp"

#include <mutex>

using namespace lt;
using namespace lt_host;

namespace {

constexpr int kStaticThreads = 256;
constexpr int kStaticPerThread = 32;
constexpr size_t kStaticChunk = (size_t)kStaticThreads * kStaticPerThread;   // particles per CTA
constexpr size_t kStaticMaxCtas = LT_STATIC_MAX_PARTICLES / kStaticChunk;    // 2048
constexpr size_t kStaticBytes = kStaticMaxCtas * kPartialStride * sizeof(double);
static_assert(kStaticMaxCtas * kStaticChunk == LT_STATIC_MAX_PARTICLES, "whole chunks");
static_assert(kStaticBytes == 128 * 1024, "the size documented in include/longtrack.h");

// The scratch: one record of kPartialStride doubles (sz szz sd sdd szd nin pad pad) per CTA, as
// in the tracker-owned buffer of the allocating path.  File scope, so every GPU that loads this
// library holds its own copy until exit.  In HOST code this name is only a handle for
// cudaGetSymbolAddress -- it is not a device address and must never be given to a kernel.
static __device__ __align__(256) double g_static_partials[kStaticMaxCtas * kPartialStride];

// Device address of g_static_partials, per device: looked up once, with that device current.
constexpr int kMaxDevices = 64;
std::mutex g_static_mu;
double* g_static_ptr[kMaxDevices];

int static_scratch(lt_tracker* tr, double** out) {
    int dev = -1;
    LT_CUDA(tr, cudaGetDevice(&dev));
    if (dev < 0 || dev >= kMaxDevices) return LT_E_PARAM;
    std::lock_guard<std::mutex> lock(g_static_mu);
    if (!g_static_ptr[dev]) {
        void* p = nullptr;
        LT_CUDA(tr, cudaGetSymbolAddress(&p, g_static_partials));
        if (!p) { tr->last_cuda_error = (int)cudaErrorInvalidSymbol; return LT_E_CUDA; }
        g_static_ptr[dev] = static_cast<double*>(p);
    }
    *out = g_static_ptr[dev];
    return LT_OK;
}

// Raw sums of the state, CTA b owning particles [b * kStaticChunk, (b + 1) * kStaticChunk): the
// grid, and with it the number of records written, follows from n alone.  Every record that the
// finalising launch reads is written here first, so nothing in the array has to start at zero
// and whatever an earlier call left behind is never looked at.
__global__ void __launch_bounds__(kStaticThreads)
static_sums_kernel(const double* __restrict__ z_arr, const double* __restrict__ d_arr, size_t n,
                   double* __restrict__ partials, const __grid_constant__ MapConsts<double> P) {
    Sums acc;
    acc.zero();
    const size_t base = (size_t)blockIdx.x * kStaticChunk + threadIdx.x;
#pragma unroll 4
    for (int k = 0; k < kStaticPerThread; ++k) {
        const size_t i = base + (size_t)k * kStaticThreads;
        if (i < n) {
            const double zz = z_arr[i], dd = d_arr[i];
            acc.add(zz, dd, in_bucket<double>(zz, dd, P));
        }
    }
    block_reduce_store(acc, partials + (size_t)blockIdx.x * kPartialStride);
}

}  // namespace

extern "C" int lt_moments_now_static(lt_tracker* tr, const double* z_dev, const double* delta_dev,
                                     size_t n, lt_moments* moments_dev, lt_sums* sums_dev,
                                     void* stream) {
    if (!tr) return LT_E_NULL;
    if (!moments_dev && !sums_dev) return LT_E_NULL;
    if (n > 0 && (!z_dev || !delta_dev)) return LT_E_NULL;
    if (n > (size_t)LT_STATIC_MAX_PARTICLES) return LT_E_CAPACITY;
    if (n > 0 && (!aligned(z_dev, sizeof(double)) || !aligned(delta_dev, sizeof(double))))
        return LT_E_ALIGN;
    double* scratch = nullptr;
    int rc = static_scratch(tr, &scratch);
    if (rc) return rc;
    cudaStream_t st = (cudaStream_t)stream;
    size_t g = (n + kStaticChunk - 1) / kStaticChunk;
    if (g < 1) g = 1;               // n == 0: one CTA writes an all-zero record (moments of nothing are 0)
    static_sums_kernel<<<(unsigned)g, kStaticThreads, 0, st>>>(z_dev, delta_dev, n, scratch, tr->c64);
    LT_CUDA(tr, cudaGetLastError());
    finalize_kernel<<<1, 256, 0, st>>>(scratch, (int)g, n, nullptr, nullptr,
                                       reinterpret_cast<MomentsOut*>(moments_dev),
                                       reinterpret_cast<SumsOut*>(sums_dev), nullptr);
    LT_CUDA(tr, cudaGetLastError());
    tr->launches += 2;
    return LT_OK;
}
