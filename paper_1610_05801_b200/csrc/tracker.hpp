// tracker.hpp -- host-side internals shared by the translation units of liblongtrack.so
// (longtrack.cu: the BASELINE path; longtrack_next.cu: SURVEY.md sec. 8(f) rows f2-f4).
// Not part of the ABI.  CUDA path only: nothing here touches oracle/.
#pragma once

#include "../../include/longtrack.h"

#include <atomic>
#include <cstdint>
#include <tuple>
#include <utility>
#include <cuda_runtime.h>

#include "kernels.cuh"

namespace lt_host {

constexpr int kBatchTurns = 64;          // per-turn launches per finalize launch / per graph
constexpr int kPerTurnThreads = 256;
constexpr int kPerTurnUnroll = 2;        // double2 pairs per thread per tile
constexpr int kMaxSlices = 1 << 20;
constexpr int kMaxSharedSlices = 8190;   // histograms up to here are counted in shared memory (32 KB per CTA)
constexpr int kMaxSegments = 256;        // lattice staged in shared memory by the per-turn kernel

struct GraphKey {
    void *z, *d, *moments, *sums;
    size_t n;
    int f32, reverse, grid;
    // extras (f2 / f4): tables, histogram and slicing grid baked into the captured launches
    const void *volt, *phase;
    void* hist;
    double z_lo, z_hi;
    int n_slices;
    const void* ramp;         // energy ramp: the packed table baked into the captured launches
    int nsub;
    bool operator==(const GraphKey& o) const {
        return z == o.z && d == o.d && moments == o.moments && sums == o.sums && n == o.n &&
               f32 == o.f32 && reverse == o.reverse && grid == o.grid && volt == o.volt &&
               phase == o.phase && hist == o.hist && z_lo == o.z_lo && z_hi == o.z_hi &&
               n_slices == o.n_slices && ramp == o.ramp && nsub == o.nsub;
    }
};

struct PersistentPlan {
    int dynamic, warps_per_smsp, ctas_per_sm, threads;
    unsigned int item_turns;
    bool flip_on_q;
    int ilp;                  // particles per lane of the persistent kernel (1 or 2)
    unsigned int queue_item_turns;   // item length the ticket queue would use (always set): what a
                                     // refused wrap-around launch falls back to
};

}  // namespace lt_host

struct lt_tracker {
    lt_params p;
    lt_derived_t g;
    lt::MapConsts<double> c64;
    lt::MapConsts<float> c32;
    lt::MapConsts<lt::f32x2> c32x2;   // c32 with every constant twice (packed fp32 pairs)
    int harm;                 // 0 generic (phi_s != 0), 1 single, 2 double harmonic
    // options
    long long split_drifts, chunk_turns, fused_ilp, fused_block, per_turn_graph,
        per_turn_ctas_per_sm, per_turn_reverse, fused_mode, item_turns, warps_per_smsp, flip_on_q, ramp_scaled, lattice_source;
    // stats
    long long launches, last_grid, last_block, last_ilp, last_mode, last_item_turns;
    int sm_count;             // 0 until the first device call
    int last_cuda_error;
    // device scratch
    double* partials;         // [kBatchTurns][grid][kPartialStride]
    size_t partials_doubles;
    unsigned long long* cursor;   // + done flag right behind it
    unsigned long long* sched;    // persistent fused kernel: ticket, then done[groups] (u32)
    size_t sched_bytes;
    // host-buffer entry point
    cudaStream_t own_stream;
    double *stage_z, *stage_d;
    unsigned long long* stage_count;
    size_t stage_n;
    // per-turn graph cache
    cudaGraphExec_t graph_exec;
    lt_host::GraphKey graph_key;
    cudaStream_t capture_stream;
    // f2: packed programme table of the current fused chunk
    double2* prog_table;
    size_t prog_entries;
    // f4: the two protocol words of lt_slice_histogram ("zeroed" flag, sign-off count), 0 between launches
    unsigned long long* hist_acc;
    // f2 with acceleration: packed sub-step entries (lt::RampEntry, 48 B each)
    void* ramp_table;
    size_t ramp_entries;
    // f3: lattice
    double* lattice_host;     // [n_seg][16], row-major
    double* lattice_dev;
    int n_seg, lattice_dirty;
};

#define LT_CUDA(tr, call)                                   \
    do {                                                    \
        cudaError_t e_ = (call);                            \
        if (e_ != cudaSuccess) {                            \
            (tr)->last_cuda_error = (int)e_;                \
            (void)cudaGetLastError();                       \
            return LT_E_CUDA;                               \
        }                                                   \
    } while (0)

namespace lt_host {

inline bool aligned(const void* p, size_t a) { return ((uintptr_t)p % a) == 0; }

// Grows a tracker-owned device buffer to `need` bytes, STREAM-ORDERED on the caller's stream
// (cudaMallocAsync + cudaFreeAsync): no device synchronisation, unlike cudaFree/cudaMalloc.  The
// old block is released after the work already enqueued on `st`, the new one is usable by what
// is enqueued after this call (one call in flight per tracker: include/longtrack.h).
// The new block is obtained FIRST: when that fails, *ptr and *have -- and with them whatever
// capacity the tracker derives from *have -- still describe the old block, which stays usable.
inline cudaError_t grow_async(void** ptr, size_t* have, size_t need, cudaStream_t st) {
    if (*have >= need && *ptr) return cudaSuccess;
    void* fresh = nullptr;
    cudaError_t e = cudaMallocAsync(&fresh, need, st);
    if (e != cudaSuccess) return e;
    if (*ptr) {
        e = cudaFreeAsync(*ptr, st);
        if (e != cudaSuccess) {
            (void)cudaFreeAsync(fresh, st);
            return e;
        }
    }
    *ptr = fresh;
    *have = need;
    return cudaSuccess;
}

// cudaFuncAttributeMaxDynamicSharedMemorySize is a property of (kernel, DEVICE): set it once per
// kernel instantiation and device (`devices` = bit d set when done on device d), not once per
// process -- a second GPU would otherwise refuse the 80-120 KB launches.  Beyond 64 devices, or
// when two host threads get here together, the attribute is simply set again (idempotent).
template <typename Kernel>
inline cudaError_t allow_dynamic_smem(std::atomic<unsigned long long>& devices, Kernel kern, int bytes) {
    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    const bool tracked = dev >= 0 && dev < 64;
    const unsigned long long bit = tracked ? 1ULL << dev : 0ULL;
    if (tracked && (devices.load(std::memory_order_acquire) & bit)) return cudaSuccess;
    e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, bytes);
    if (e == cudaSuccess && tracked) devices.fetch_or(bit, std::memory_order_release);
    return e;
}

// The wrap-around schedule lets a CTA wait for a piece that ANOTHER CTA of the same grid runs
// (kernels.cuh, `dynamic == 2`): that terminates only if every CTA of the grid is resident at
// once.  One CTA (or two) per SM always fits a whole, idle GPU, but not an MPS / green-context
// partition with fewer SMs than cudaDevAttrMultiProcessorCount reports.  So such a grid goes out
// as a COOPERATIVE launch: the runtime then either guarantees co-residency or refuses the launch
// (cudaErrorCooperativeLaunchTooLarge) instead of letting it hang.  `args` are converted to the
// kernel's exact parameter types before their addresses are taken.
template <typename... KArgs, typename... Args>
inline cudaError_t launch_coresident(void (*kern)(KArgs...), int grid, int threads, size_t smem,
                                     cudaStream_t st, Args&&... args) {
    static_assert(sizeof...(KArgs) == sizeof...(Args), "one argument per kernel parameter");
    std::tuple<std::remove_cv_t<KArgs>...> vals(std::forward<Args>(args)...);
    return std::apply(
        [&](auto&... v) {
            void* argv[] = {static_cast<void*>(&v)...};
            return cudaLaunchCooperativeKernel(reinterpret_cast<const void*>(kern), dim3((unsigned)grid),
                                               dim3((unsigned)threads), argv, smem, st);
        },
        vals);
}
inline bool coresidency_refused(cudaError_t e) {
    return e == cudaErrorCooperativeLaunchTooLarge || e == cudaErrorNotSupported;
}
// Set by a launch site whose wrap-around launch was refused and which ran the ticket queue instead
// (safe with any number of resident CTAs: a work item only ever waits for one with a smaller
// ticket, i.e. for a CTA that is running or done); read and cleared by the entry point, which
// reports it in LT_STAT_LAST_MODE.  Per host thread, like the call itself.
inline thread_local int g_wrap_refused = 0;

int ensure_device(lt_tracker* tr);
int ensure_scratch(lt_tracker* tr, int grid, cudaStream_t st);
int ensure_sched(lt_tracker* tr, size_t n, cudaStream_t st);
// max_ilp: 2 where the kernel has a two-particles-per-lane instantiation, else 1
// pv: particles per chain value (2 for packed fp32 pairs)
PersistentPlan plan_persistent(const lt_tracker* tr, size_t n, unsigned long long turns, int max_ilp = 1, int pv = 1);
int per_turn_grid(const lt_tracker* tr, size_t n);
// the BASELINE path's fused / per-turn entry points, for calls that compose with them
int track_fused_f64(lt_tracker* tr, double* z, double* d, size_t n, unsigned long long turns,
                    void* stream);
cudaError_t launch_per_turn_f64(const lt_tracker* tr, double* z, double* d, size_t n, int reverse,
                                double* partials, bool moments, bool vec_ok, int grid,
                                cudaStream_t st);
void destroy_next(lt_tracker* tr);       // frees what longtrack_next.cu allocated
void destroy_ramp(lt_tracker* tr);       // frees what longtrack_ramp.cu allocated

}  // namespace lt_host
