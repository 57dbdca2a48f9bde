// longtrack_next.cu -- host side of the entry points for SURVEY.md sec. 8(f) rows f2-f4:
// RF programme (fused and per-turn), slicing histogram, transverse linear maps.
// CUDA path only: nothing here includes, links or calls anything under oracle/.
#include "tracker.hpp"

#include <algorithm>
#include <cmath>
#include <cstdlib>
#include <cstring>

#include "kernels_next.cuh"

using namespace lt;
using namespace lt_host;

namespace {

const double kInvPi = 0.31830988618379067154;   // 1/pi rounded to fp64
constexpr unsigned long long kProgChunkMax = 1ULL << 20;   // programme entries packed per launch

int residency_smem(const PersistentPlan& pl) {
    // 1 CTA/SM: > half of the 227 KB; 2 CTAs/SM: > a third
    return pl.ctas_per_sm == 1 ? 120 * 1024 : 80 * 1024;
}

// ------------------------------------------------------------------------------------------
// f2, fused mode: the persistent kernel with PROG, one packed table per launch
// ------------------------------------------------------------------------------------------
template <int INTEG, int HARM, bool SPLIT, bool FQ, int ILP>
cudaError_t launch_prog_ilp(double* z, double* d, size_t n, unsigned int turns, unsigned int item_turns,
                            int first, int last, const PersistentPlan& pl, int sms,
                            unsigned long long* sched, const MapConsts<double>& c,
                            const double2* prog, cudaStream_t st) {
    auto kern = fused_persistent_kernel<double, INTEG, HARM, SPLIT, FQ, true, ILP>;
    const int smem = residency_smem(pl);                     // >= 512 B of staged entries per warp
    static std::atomic<unsigned long long> attr_devices{0};   // per instantiation: the devices it is set on
    {
        cudaError_t e = allow_dynamic_smem(attr_devices, kern, 120 * 1024);
        if (e != cudaSuccess) return e;
    }
    unsigned int* const done = reinterpret_cast<unsigned int*>(sched + 1);
    int dynamic = pl.dynamic;
    if (dynamic == 2) {                                      // CTAs wait on one another: co-resident or not at all
        const cudaError_t e = launch_coresident(kern, sms * pl.ctas_per_sm, pl.threads, (size_t)smem, st, z, d, n,
                                                turns, item_turns, first, last, 2, sched, done, c, prog);
        if (!coresidency_refused(e)) return e;
        (void)cudaGetLastError();
        g_wrap_refused = 1;                                  // same bits from the ticket queue
        dynamic = 1;
        item_turns = std::min(pl.queue_item_turns, turns);
    }
    kern<<<sms * pl.ctas_per_sm, pl.threads, smem, st>>>(z, d, n, turns, item_turns, first, last,
                                                         dynamic, sched, done, c, prog);
    return cudaGetLastError();
}

template <int INTEG, int HARM, bool SPLIT>
cudaError_t launch_prog_one(double* z, double* d, size_t n, unsigned int turns, unsigned int item_turns,
                            int first, int last, const PersistentPlan& pl, int sms,
                            unsigned long long* sched, const MapConsts<double>& c,
                            const double2* prog, cudaStream_t st) {
#define LT_PI(Q, I) launch_prog_ilp<INTEG, HARM, SPLIT, Q, I>(z, d, n, turns, item_turns, first, last, pl, sms, sched, c, prog, st)
    if (SPLIT || HARM == 0) return pl.ilp == 2 ? LT_PI(false, 2) : LT_PI(false, 1);
    if (pl.ilp == 2) return pl.flip_on_q ? LT_PI(true, 2) : LT_PI(false, 2);
    return pl.flip_on_q ? LT_PI(true, 1) : LT_PI(false, 1);
#undef LT_PI
}

template <int INTEG>
cudaError_t launch_prog_integ(int harm, bool split, double* z, double* d, size_t n, unsigned int turns,
                              unsigned int item_turns, int first, int last, const PersistentPlan& pl,
                              int sms, unsigned long long* sched, const MapConsts<double>& c,
                              const double2* prog, cudaStream_t st) {
#define LT_PG(H, S) launch_prog_one<INTEG, H, S>(z, d, n, turns, item_turns, first, last, pl, sms, sched, c, prog, st)
    if (harm == 0) return LT_PG(0, true);
    if (harm == 1) return split ? LT_PG(1, true) : LT_PG(1, false);
    return split ? LT_PG(2, true) : LT_PG(2, false);
#undef LT_PG
}

int track_programme_fused(lt_tracker* tr, double* z, double* d, size_t n, unsigned long long turns,
                          const double* volt, const double* phase, void* stream) {
    if (!tr) return LT_E_NULL;
    if (n == 0 || turns == 0) return LT_OK;
    if (!z || !d || !volt || !phase) return LT_E_NULL;
    if (!aligned(z, 8) || !aligned(d, 8) || !aligned(volt, 8) || !aligned(phase, 8)) return LT_E_ALIGN;
    if (n > ((size_t)1 << 40)) return LT_E_PARAM;
    int rc = ensure_device(tr);
    if (rc) return rc;
    cudaStream_t st = (cudaStream_t)stream;
    rc = ensure_sched(tr, n, st);
    if (rc) return rc;
    const bool split = tr->split_drifts != 0 || tr->harm == 0;
    const unsigned long long chunk_max =
        std::min<unsigned long long>((unsigned long long)tr->chunk_turns, kProgChunkMax);
    const size_t want = (size_t)std::min<unsigned long long>(turns, chunk_max);
    {
        size_t have = tr->prog_entries ? (tr->prog_entries + 1) * sizeof(double2) : 0;
        LT_CUDA(tr, grow_async((void**)&tr->prog_table, &have, (want + 1) * sizeof(double2), st));   // + the header entry
        if (tr->prog_entries < want) tr->prog_entries = want;
    }
    const PersistentPlan pl = plan_persistent(tr, n, turns, 2);
    g_wrap_refused = 0;
    unsigned long long done = 0;
    while (done < turns) {
        const unsigned long long chunk = std::min<unsigned long long>(turns - done, chunk_max);
        const int first = done == 0, last = done + chunk == turns;
        const unsigned int item = pl.dynamic == 1 ? std::min<unsigned int>(pl.item_turns, (unsigned int)chunk)
                                                  : (unsigned int)chunk;
        // the table of the previous chunk is free again: its kernel precedes this one on the stream
        programme_pack_kernel<<<(unsigned)((chunk + 255) / 256), 256, 0, st>>>(
            volt, phase, done, (unsigned int)chunk, turns, kInvPi, split ? 0 : 1, tr->prog_table);
        LT_CUDA(tr, cudaGetLastError());
        if (pl.dynamic) LT_CUDA(tr, cudaMemsetAsync(tr->sched, 0, 8 + 4 * ((n + 31) / 32), st));
        cudaError_t e;
        switch (tr->p.integrator) {
            case LT_EULER_CROMER:
                e = launch_prog_integ<kEulerCromer>(tr->harm, split, z, d, n, (unsigned)chunk, item, first, last, pl, tr->sm_count, tr->sched, tr->c64, tr->prog_table + 1, st);
                break;
            case LT_LEAPFROG:
                e = launch_prog_integ<kLeapfrog>(tr->harm, split, z, d, n, (unsigned)chunk, item, first, last, pl, tr->sm_count, tr->sched, tr->c64, tr->prog_table + 1, st);
                break;
            default:
                e = launch_prog_integ<kRuth4>(tr->harm, split, z, d, n, (unsigned)chunk, item, first, last, pl, tr->sm_count, tr->sched, tr->c64, tr->prog_table + 1, st);
        }
        LT_CUDA(tr, e);
        tr->launches += 2;
        done += chunk;
    }
    tr->last_grid = (long long)tr->sm_count * pl.ctas_per_sm;
    tr->last_block = pl.threads;
    tr->last_ilp = pl.ilp;
    tr->last_mode = pl.dynamic == 2 ? (g_wrap_refused ? 3 : 4) : (pl.dynamic ? 3 : 2);
    tr->last_item_turns = pl.dynamic == 1 ? pl.item_turns : (pl.dynamic == 2 && g_wrap_refused ? pl.queue_item_turns : 0);
    return LT_OK;
}

// ------------------------------------------------------------------------------------------
// f2 / f4, per-turn mode
// ------------------------------------------------------------------------------------------
struct ExtraArgs {
    const double *volt, *phase;
    unsigned long long* hist;
    double z_lo, z_hi;
    int n_slices;
};

size_t slice_stride(int n_slices) { return ((size_t)n_slices + 2) | 1; }

// shared-memory copies of the histogram: one per lane when they fit (no two lanes of a warp ever
// share a counter), halved until the copies fit 32 KB per CTA; 0 = global atomics
int slice_replicas(int n_slices) {
    const size_t one = slice_stride(n_slices) * sizeof(unsigned int);
    int r = 32;
    while (r > 0 && (size_t)r * one > 32 * 1024) r >>= 1;
    return r;
}

size_t slice_smem_bytes(const TurnExtras& X) {
    return (size_t)X.replicas * slice_stride(X.n_slices) * sizeof(unsigned int);
}

TurnExtras make_extras(const lt_tracker* tr, const ExtraArgs& a, int k) {
    TurnExtras X;
    std::memset(&X, 0, sizeof(X));
    X.volt_scale = a.volt;
    X.phase_off = a.phase;
    X.cursor = tr->cursor;
    X.k = k;
    X.inv_pi = kInvPi;
    X.hist = a.hist;
    if (a.hist) {
        X.z_lo = a.z_lo; X.z_hi = a.z_hi;
        X.inv = (double)a.n_slices / (a.z_hi - a.z_lo);      // as the definition states it (G29)
        X.n_slices = a.n_slices;
        X.replicas = slice_replicas(a.n_slices);
    }
    return X;
}

template <int INTEG, int HARM>
cudaError_t launch_extra_one(double* z, double* d, size_t n, int reverse, double* partials,
                             bool moments, bool vec_ok, int grid, const MapConsts<double>& c,
                             const TurnExtras& X, cudaStream_t st) {
    const size_t smem = slice_smem_bytes(X);
    if (vec_ok) {
        if (moments)
            per_turn_extra_kernel<INTEG, HARM, true, kPerTurnUnroll><<<grid, kPerTurnThreads, smem, st>>>(z, d, n, reverse, partials, c, X);
        else
            per_turn_extra_kernel<INTEG, HARM, false, kPerTurnUnroll><<<grid, kPerTurnThreads, smem, st>>>(z, d, n, reverse, partials, c, X);
    } else {
        per_turn_extra_kernel_scalar<INTEG, HARM><<<grid, kPerTurnThreads, smem, st>>>(z, d, n, moments ? 1 : 0, partials, c, X);
    }
    return cudaGetLastError();
}

cudaError_t launch_extra(const lt_tracker* tr, double* z, double* d, size_t n, int reverse,
                         double* partials, bool moments, bool vec_ok, int grid, const TurnExtras& X,
                         cudaStream_t st) {
#define LT_PX(INTEG)                                                                                            \
    (tr->harm == 0   ? launch_extra_one<INTEG, 0>(z, d, n, reverse, partials, moments, vec_ok, grid, tr->c64, X, st) \
     : tr->harm == 1 ? launch_extra_one<INTEG, 1>(z, d, n, reverse, partials, moments, vec_ok, grid, tr->c64, X, st) \
                     : launch_extra_one<INTEG, 2>(z, d, n, reverse, partials, moments, vec_ok, grid, tr->c64, X, st))
    switch (tr->p.integrator) {
        case LT_EULER_CROMER: return LT_PX(kEulerCromer);
        case LT_LEAPFROG: return LT_PX(kLeapfrog);
        default: return LT_PX(kRuth4);
    }
#undef LT_PX
}

// `nb` turns starting at absolute turn t0 (only its parity matters here: the kernels take the
// absolute index from the device cursor), then the finalize / cursor advance
cudaError_t enqueue_extra_batch(lt_tracker* tr, double* z, double* d, size_t n, unsigned long long t0,
                                int nb, bool moments, lt_moments* mo, lt_sums* so, bool vec_ok, int grid,
                                const ExtraArgs& a, cudaStream_t st) {
    for (int k = 0; k < nb; ++k) {
        const int reverse = tr->per_turn_reverse ? (int)((t0 + k) & 1ULL) : 0;
        double* part = tr->partials + (size_t)k * grid * kPartialStride;
        const TurnExtras X = make_extras(tr, a, k);
        cudaError_t e = launch_extra(tr, z, d, n, reverse, part, moments, vec_ok, grid, X, st);
        if (e != cudaSuccess) return e;
        tr->launches++;
    }
    if (moments)
        finalize_kernel<<<nb, 256, 0, st>>>(tr->partials, grid, n, tr->cursor,
                                            reinterpret_cast<unsigned int*>(tr->cursor + 1),
                                            reinterpret_cast<MomentsOut*>(mo),
                                            reinterpret_cast<SumsOut*>(so), nullptr);
    else
        advance_cursor_kernel<<<1, 1, 0, st>>>(tr->cursor, (unsigned long long)nb);
    tr->launches++;
    return cudaGetLastError();
}

int track_per_turn_extra(lt_tracker* tr, double* z, double* d, size_t n, unsigned long long turns,
                         const ExtraArgs& a, lt_moments* mo, lt_sums* so, void* stream) {
    if (!tr) return LT_E_NULL;
    if (a.hist) {
        if (a.n_slices < 1 || a.n_slices > kMaxSlices) return LT_E_PARAM;
        if (!std::isfinite(a.z_lo) || !std::isfinite(a.z_hi) || !(a.z_hi > a.z_lo)) return LT_E_PARAM;
        if (!aligned(a.hist, 8)) return LT_E_ALIGN;
    }
    if (turns == 0) return LT_OK;
    if (n > 0 && (!z || !d)) return LT_E_NULL;
    if (n > 0 && (!aligned(z, 8) || !aligned(d, 8))) return LT_E_ALIGN;
    if ((a.volt && !aligned(a.volt, 8)) || (a.phase && !aligned(a.phase, 8))) return LT_E_ALIGN;
    if ((mo && !aligned(mo, 8)) || (so && !aligned(so, 8))) return LT_E_ALIGN;
    if (n > ((size_t)1 << 40)) return LT_E_PARAM;
    int rc = ensure_device(tr);
    if (rc) return rc;
    cudaStream_t st = (cudaStream_t)stream;
    if (a.hist)
        LT_CUDA(tr, cudaMemsetAsync(a.hist, 0, (size_t)turns * ((size_t)a.n_slices + 2) * sizeof(unsigned long long), st));
    if (n == 0) return LT_OK;                    // empty bunch: every histogram is zero
    const bool moments = mo || so;
    const bool vec_ok = aligned(z, 16) && aligned(d, 16);
    const int grid = per_turn_grid(tr, n);
    rc = ensure_scratch(tr, grid, st);
    if (rc) return rc;
    set_cursor_kernel<<<1, 1, 0, st>>>(tr->cursor, reinterpret_cast<unsigned int*>(tr->cursor + 1), 0ULL);
    LT_CUDA(tr, cudaGetLastError());
    tr->launches++;
    unsigned long long t0 = 0;
    if (tr->per_turn_graph && turns >= 2ULL * kBatchTurns) {
        GraphKey key = {(void*)z, (void*)d, (void*)mo, (void*)so, n, 0, (int)tr->per_turn_reverse, grid,
                        (const void*)a.volt, (const void*)a.phase, (void*)a.hist,
                        a.hist ? a.z_lo : 0.0, a.hist ? a.z_hi : 0.0, a.hist ? a.n_slices : 0};
        if (!tr->graph_exec || !(tr->graph_key == key)) {
            if (tr->graph_exec) { cudaGraphExecDestroy(tr->graph_exec); tr->graph_exec = nullptr; }
            if (!tr->capture_stream)
                LT_CUDA(tr, cudaStreamCreateWithFlags(&tr->capture_stream, cudaStreamNonBlocking));
            cudaGraph_t graph = nullptr;
            LT_CUDA(tr, cudaStreamBeginCapture(tr->capture_stream, cudaStreamCaptureModeThreadLocal));
            const long long before = tr->launches;
            cudaError_t e = enqueue_extra_batch(tr, z, d, n, 0, kBatchTurns, moments, mo, so, vec_ok, grid, a, tr->capture_stream);
            tr->launches = before;      // capture enqueues nothing
            cudaError_t e2 = cudaStreamEndCapture(tr->capture_stream, &graph);
            if (e != cudaSuccess || e2 != cudaSuccess) {        // no graph is left behind on failure
                if (graph) cudaGraphDestroy(graph);
                LT_CUDA(tr, e != cudaSuccess ? e : e2);
            }
            cudaError_t e3 = cudaGraphInstantiate(&tr->graph_exec, graph, 0);
            cudaGraphDestroy(graph);
            LT_CUDA(tr, e3);
            tr->graph_key = key;
        }
        while (turns - t0 >= (unsigned long long)kBatchTurns) {
            LT_CUDA(tr, cudaGraphLaunch(tr->graph_exec, st));
            tr->launches += kBatchTurns + 1;
            t0 += kBatchTurns;
        }
    }
    while (t0 < turns) {
        const int nb = (int)std::min<unsigned long long>(kBatchTurns, turns - t0);
        LT_CUDA(tr, enqueue_extra_batch(tr, z, d, n, t0, nb, moments, mo, so, vec_ok, grid, a, st));
        t0 += nb;
    }
    return LT_OK;
}

// ------------------------------------------------------------------------------------------
// f3: transverse plane
// ------------------------------------------------------------------------------------------
int ensure_lattice(lt_tracker* tr, cudaStream_t st) {
    if (tr->n_seg <= 0 || !tr->lattice_host) return LT_E_PARAM;   // lt_set_transverse not called
    if (!tr->lattice_dev) LT_CUDA(tr, cudaMallocAsync((void**)&tr->lattice_dev, (size_t)kMaxSegments * 16 * sizeof(double), st));
    if (tr->lattice_dirty) {
        // pageable source: the copy is staged before the call returns and ordered on the stream
        LT_CUDA(tr, cudaMemcpyAsync(tr->lattice_dev, tr->lattice_host, (size_t)tr->n_seg * 16 * sizeof(double),
                                    cudaMemcpyHostToDevice, st));
        tr->lattice_dirty = 0;
    }
    return LT_OK;
}

// launch shape of the fused transverse kernel: ILP particles per thread (8 at 2 warps per
// sub-partition and 220 registers per thread -- a matrix row fetched from shared memory then feeds
// 32 FP64 instructions: 0.893 of the FP64 peak against 0.882 with 4 --, 4 or 2 at 4 warps per
// sub-partition and 128 registers; 1 at the plan of the longitudinal kernel), the largest ILP
// that still fills one wave of warps; dynamic chunk scheduling beyond one wave
struct TransPlan { int ilp; PersistentPlan pl; };

TransPlan plan_transverse(const lt_tracker* tr, size_t n, unsigned long long turns) {
    TransPlan tp;
    tp.ilp = 1;
    const unsigned long long slots = (unsigned long long)tr->sm_count * 16;
    int ilp = 0;
    if (tr->fused_ilp == 1 || tr->fused_ilp == 2 || tr->fused_ilp == 4 || tr->fused_ilp == 8) ilp = (int)tr->fused_ilp;
    else if ((n + 255) / 256 >= slots / 2) ilp = 8;
    else if ((n + 127) / 128 >= slots) ilp = 4;
    else if ((n + 63) / 64 >= slots) ilp = 2;
    else ilp = 1;
    if (ilp == 1) {
        tp.pl = plan_persistent(tr, n, turns);
        if (tp.pl.dynamic == 2) {                            // this kernel has no wrap-around schedule
            tp.pl.dynamic = 1;
            const unsigned long long it = tr->item_turns > 0
                                              ? (unsigned long long)tr->item_turns
                                              : std::min<unsigned long long>(2048, std::max<unsigned long long>(128, turns / 8));
            tp.pl.item_turns = (unsigned int)std::min<unsigned long long>(it, turns);
        }
        return tp;
    }
    tp.ilp = ilp;
    const unsigned long long groups = (n + 32 * ilp - 1) / (32 * ilp);
    PersistentPlan pl = {0, 4, 1, 512, 0, true, 1};
    if (ilp == 8) { pl.warps_per_smsp = 2; pl.threads = 256; }   // 220 registers per thread
    // more groups than slots: the ticket queue (4 warps per sub-partition hide its item switches; the
    // wrap-around static schedule measured 1.2 points lower and its code cost the kernel a register
    // spill, so this kernel does not carry it: LT_OPT_FUSED_MODE = 4 means the queue here)
    const unsigned long long my_slots = ilp == 8 ? slots / 2 : slots;
    pl.dynamic = tr->fused_mode == 2 ? 0 : ((groups > my_slots || tr->fused_mode >= 3) ? 1 : 0);
    if (pl.dynamic == 1) {
        unsigned long long it = tr->item_turns > 0
                                    ? (unsigned long long)tr->item_turns
                                    : std::min<unsigned long long>(2048, std::max<unsigned long long>(128, turns / 8));
        pl.item_turns = (unsigned int)std::min<unsigned long long>(it, turns);
    }
    tp.pl = pl;
    return tp;
}

template <int NSEG, bool LONGI, int ILP>
cudaError_t launch_transverse_one(double* x, double* xp, double* y, double* yp, double* z, double* d,
                                  size_t n, unsigned int turns, unsigned int item_turns, int first, int last,
                                  const PersistentPlan& pl, const lt_tracker* tr, cudaStream_t st) {
    auto kern = transverse_persistent_kernel<NSEG, LONGI, ILP>;
    const int smem = residency_smem(pl);                 // >= the lattice (256 x 128 B)
    static std::atomic<unsigned long long> attr_devices{0};   // per instantiation: the devices it is set on
    {
        cudaError_t e = allow_dynamic_smem(attr_devices, kern, 120 * 1024);
        if (e != cudaSuccess) return e;
    }
    kern<<<tr->sm_count * pl.ctas_per_sm, pl.threads, smem, st>>>(
        x, xp, y, yp, z, d, n, turns, item_turns, first, last, pl.dynamic, tr->sched,
        reinterpret_cast<unsigned int*>(tr->sched + 1), tr->lattice_dev, tr->n_seg, tr->c64);
    return cudaGetLastError();
}

// lattice in the parameter space (constant bank -> uniform registers; kernels_next.cuh)
template <bool LONGI, int ILP>
cudaError_t launch_transverse_param(double* x, double* xp, double* y, double* yp, double* z, double* d,
                                    size_t n, unsigned int turns, unsigned int item_turns, int first, int last,
                                    const PersistentPlan& pl, const lt_tracker* tr, cudaStream_t st) {
    auto kern = transverse_persistent_param_kernel<LONGI, ILP>;
    const int smem = residency_smem(pl);
    static std::atomic<unsigned long long> attr_devices{0};   // per instantiation: the devices it is set on
    {
        cudaError_t e = allow_dynamic_smem(attr_devices, kern, 120 * 1024);
        if (e != cudaSuccess) return e;
    }
    LatticeParam lp;
    std::memcpy(lp.m, tr->lattice_host, (size_t)tr->n_seg * 16 * sizeof(double));
    lp.n_seg = tr->n_seg;
    kern<<<tr->sm_count * pl.ctas_per_sm, pl.threads, smem, st>>>(
        x, xp, y, yp, z, d, n, turns, item_turns, first, last, pl.dynamic, tr->sched,
        reinterpret_cast<unsigned int*>(tr->sched + 1), lp, tr->c64);
    return cudaGetLastError();
}

template <bool LONGI, int ILP>
cudaError_t launch_transverse_ilp(double* x, double* xp, double* y, double* yp, double* z, double* d,
                                  size_t n, unsigned int turns, unsigned int item_turns, int first, int last,
                                  const PersistentPlan& pl, const lt_tracker* tr, cudaStream_t st) {
    if (tr->lattice_source != 1 && tr->n_seg <= kParamSegments)
        return launch_transverse_param<LONGI, ILP>(x, xp, y, yp, z, d, n, turns, item_turns, first, last, pl, tr, st);
#define LT_TV(NS) launch_transverse_one<NS, LONGI, ILP>(x, xp, y, yp, z, d, n, turns, item_turns, first, last, pl, tr, st)
    switch (tr->n_seg <= kSegUnrolled ? tr->n_seg : 0) {
        case 1: return LT_TV(1);
        case 2: return LT_TV(2);
        case 3: return LT_TV(3);
        case 4: return LT_TV(4);
        default: return LT_TV(0);
    }
#undef LT_TV
}

template <bool LONGI>
cudaError_t launch_transverse(double* x, double* xp, double* y, double* yp, double* z, double* d,
                              size_t n, unsigned int turns, unsigned int item_turns, int first, int last,
                              const TransPlan& tp, const lt_tracker* tr, cudaStream_t st) {
    if (tp.ilp == 8) return launch_transverse_ilp<LONGI, 8>(x, xp, y, yp, z, d, n, turns, item_turns, first, last, tp.pl, tr, st);
    if (tp.ilp == 4) return launch_transverse_ilp<LONGI, 4>(x, xp, y, yp, z, d, n, turns, item_turns, first, last, tp.pl, tr, st);
    if (tp.ilp == 2) return launch_transverse_ilp<LONGI, 2>(x, xp, y, yp, z, d, n, turns, item_turns, first, last, tp.pl, tr, st);
    return launch_transverse_ilp<LONGI, 1>(x, xp, y, yp, z, d, n, turns, item_turns, first, last, tp.pl, tr, st);
}

int check_transverse_args(lt_tracker* tr, double* x, double* xp, double* y, double* yp, double* z,
                          double* d, size_t n) {
    if (!tr) return LT_E_NULL;
    if ((z == nullptr) != (d == nullptr)) return LT_E_NULL;
    if (n > 0 && (!x || !xp || !y || !yp)) return LT_E_NULL;
    if (!aligned(x, 8) || !aligned(xp, 8) || !aligned(y, 8) || !aligned(yp, 8) || !aligned(z, 8) || !aligned(d, 8))
        return LT_E_ALIGN;
    if (n > ((size_t)1 << 40)) return LT_E_PARAM;
    if (tr->n_seg <= 0) return LT_E_PARAM;
    return LT_OK;
}

// the longitudinal turn rides in the transverse kernels for the BASELINE map (leap-frog, single
// harmonic); any other map runs as its own launch after it -- the planes are not coupled
// (PAPER.md:39), so the composition is the same map
bool longitudinal_rides_along(const lt_tracker* tr, bool fused) {
    return tr->p.integrator == LT_LEAPFROG && tr->harm == 1 && (!fused || tr->split_drifts == 0);
}

int track_transverse_fused(lt_tracker* tr, double* x, double* xp, double* y, double* yp, double* z,
                           double* d, size_t n, unsigned long long turns, void* stream) {
    int rc = check_transverse_args(tr, x, xp, y, yp, z, d, n);
    if (rc) return rc;
    if (n == 0 || turns == 0) return LT_OK;
    rc = ensure_device(tr);
    if (rc) return rc;
    cudaStream_t st = (cudaStream_t)stream;
    rc = ensure_lattice(tr, st);
    if (rc) return rc;
    rc = ensure_sched(tr, n, st);
    if (rc) return rc;
    const bool longi = z && longitudinal_rides_along(tr, true);
    const TransPlan tp = plan_transverse(tr, n, turns);
    const PersistentPlan& pl = tp.pl;
    unsigned long long done = 0;
    while (done < turns) {
        const unsigned long long chunk = std::min<unsigned long long>(turns - done, (unsigned long long)tr->chunk_turns);
        const int first = done == 0, last = done + chunk == turns;
        const unsigned int item = pl.dynamic == 1 ? std::min<unsigned int>(pl.item_turns, (unsigned int)chunk) : (unsigned int)chunk;
        if (pl.dynamic) LT_CUDA(tr, cudaMemsetAsync(tr->sched, 0, 8 + 4 * ((n + 31) / 32), st));
        cudaError_t e = longi ? launch_transverse<true>(x, xp, y, yp, z, d, n, (unsigned)chunk, item, first, last, tp, tr, st)
                              : launch_transverse<false>(x, xp, y, yp, z, d, n, (unsigned)chunk, item, first, last, tp, tr, st);
        LT_CUDA(tr, e);
        tr->launches++;
        done += chunk;
    }
    if (z && !longi) {
        rc = track_fused_f64(tr, z, d, n, turns, stream);
        if (rc) return rc;
    }
    tr->last_grid = (long long)tr->sm_count * pl.ctas_per_sm;
    tr->last_block = pl.threads;
    tr->last_ilp = tp.ilp;
    tr->last_mode = pl.dynamic == 2 ? 4 : (pl.dynamic ? 3 : 2);
    tr->last_item_turns = pl.dynamic == 1 ? pl.item_turns : 0;
    return LT_OK;
}

int track_transverse_per_turn(lt_tracker* tr, double* x, double* xp, double* y, double* yp, double* z,
                              double* d, size_t n, unsigned long long turns, void* stream) {
    int rc = check_transverse_args(tr, x, xp, y, yp, z, d, n);
    if (rc) return rc;
    if (n == 0 || turns == 0) return LT_OK;
    rc = ensure_device(tr);
    if (rc) return rc;
    cudaStream_t st = (cudaStream_t)stream;
    rc = ensure_lattice(tr, st);
    if (rc) return rc;
    const bool longi = z && longitudinal_rides_along(tr, false);
    const bool vec = aligned(x, 16) && aligned(xp, 16) && aligned(y, 16) && aligned(yp, 16) &&
                     (!longi || (aligned(z, 16) && aligned(d, 16)));
    const size_t per_cta = (size_t)kPerTurnThreads * (vec ? 2 : 1);
    size_t g = (n + per_cta - 1) / per_cta;
    g = std::max<size_t>(1, std::min<size_t>(g, (size_t)tr->sm_count * (size_t)(tr->per_turn_ctas_per_sm > 0 ? tr->per_turn_ctas_per_sm : 6)));
    const size_t smem = (size_t)tr->n_seg * 16 * sizeof(double);
    const bool zvec = z && aligned(z, 16) && aligned(d, 16);
    const int zgrid = z ? per_turn_grid(tr, n) : 0;
    for (unsigned long long t = 0; t < turns; ++t) {
        const int reverse = tr->per_turn_reverse ? (int)(t & 1ULL) : 0;
        if (longi) {
            if (vec) transverse_per_turn_kernel<true, true><<<(unsigned)g, kPerTurnThreads, smem, st>>>(x, xp, y, yp, z, d, n, reverse, tr->lattice_dev, tr->n_seg, tr->c64);
            else transverse_per_turn_kernel<true, false><<<(unsigned)g, kPerTurnThreads, smem, st>>>(x, xp, y, yp, z, d, n, reverse, tr->lattice_dev, tr->n_seg, tr->c64);
        } else {
            if (vec) transverse_per_turn_kernel<false, true><<<(unsigned)g, kPerTurnThreads, smem, st>>>(x, xp, y, yp, z, d, n, reverse, tr->lattice_dev, tr->n_seg, tr->c64);
            else transverse_per_turn_kernel<false, false><<<(unsigned)g, kPerTurnThreads, smem, st>>>(x, xp, y, yp, z, d, n, reverse, tr->lattice_dev, tr->n_seg, tr->c64);
        }
        LT_CUDA(tr, cudaGetLastError());
        tr->launches++;
        if (z && !longi) {
            LT_CUDA(tr, launch_per_turn_f64(tr, z, d, n, reverse, nullptr, false, zvec, zgrid, st));
            tr->launches++;
        }
    }
    return LT_OK;
}

}  // namespace

namespace lt_host {
void destroy_next(lt_tracker* tr) {
    if (tr->prog_table) cudaFree(tr->prog_table);
    if (tr->hist_acc) cudaFree(tr->hist_acc);
    if (tr->lattice_dev) cudaFree(tr->lattice_dev);
    std::free(tr->lattice_host);
}
}  // namespace lt_host

// ------------------------------------------------------------------------------------------
// C ABI
// ------------------------------------------------------------------------------------------
extern "C" {

int lt_track_programme(lt_tracker* tr, double* z_dev, double* delta_dev, size_t n,
                       unsigned long long turns, const double* volt_scale_dev,
                       const double* phase_off_dev, void* stream) {
    return track_programme_fused(tr, z_dev, delta_dev, n, turns, volt_scale_dev, phase_off_dev, stream);
}

int lt_track_programme_per_turn(lt_tracker* tr, double* z_dev, double* delta_dev, size_t n,
                                unsigned long long turns, const double* volt_scale_dev,
                                const double* phase_off_dev, lt_moments* moments_dev,
                                lt_sums* sums_dev, void* stream) {
    if (turns > 0 && n > 0 && (!volt_scale_dev || !phase_off_dev)) return LT_E_NULL;
    const ExtraArgs a = {volt_scale_dev, phase_off_dev, nullptr, 0.0, 0.0, 0};
    return track_per_turn_extra(tr, z_dev, delta_dev, n, turns, a, moments_dev, sums_dev, stream);
}

int lt_track_slices(lt_tracker* tr, double* z_dev, double* delta_dev, size_t n,
                    unsigned long long turns, double z_lo, double z_hi, int n_slices,
                    unsigned long long* hist_dev, lt_moments* moments_dev, lt_sums* sums_dev,
                    void* stream) {
    if (!tr) return LT_E_NULL;
    if (turns > 0 && !hist_dev) return LT_E_NULL;
    const ExtraArgs a = {nullptr, nullptr, hist_dev, z_lo, z_hi, n_slices};
    if (turns == 0) {           // still validate the slicing grid
        if (n_slices < 1 || n_slices > kMaxSlices || !std::isfinite(z_lo) || !std::isfinite(z_hi) || !(z_hi > z_lo))
            return LT_E_PARAM;
        return LT_OK;
    }
    return track_per_turn_extra(tr, z_dev, delta_dev, n, turns, a, moments_dev, sums_dev, stream);
}

int lt_slice_histogram(lt_tracker* tr, const double* z_dev, size_t n, double z_lo, double z_hi,
                       int n_slices, unsigned long long* hist_dev, void* stream) {
    if (!tr || !hist_dev) return LT_E_NULL;
    if (n_slices < 1 || n_slices > kMaxSlices) return LT_E_PARAM;
    if (!std::isfinite(z_lo) || !std::isfinite(z_hi) || !(z_hi > z_lo)) return LT_E_PARAM;
    if (n > 0 && !z_dev) return LT_E_NULL;
    if (!aligned(z_dev, 8) || !aligned(hist_dev, 8)) return LT_E_ALIGN;
    int rc = ensure_device(tr);
    if (rc) return rc;
    cudaStream_t st = (cudaStream_t)stream;
    const ExtraArgs a = {nullptr, nullptr, hist_dev, z_lo, z_hi, n_slices};
    const TurnExtras X = make_extras(tr, a, 0);
    const bool direct = X.replicas == 0 || n == 0;           // counts straight into hist_dev
    if (direct) {
        LT_CUDA(tr, cudaMemsetAsync(hist_dev, 0, ((size_t)n_slices + 2) * sizeof(unsigned long long), st));
        if (n == 0) return LT_OK;
    } else if (!tr->hist_acc) {
        // the two words of the shared-memory path's protocol ("zeroed" flag, sign-off count): both 0
        // between launches, the kernel itself puts them back
        LT_CUDA(tr, cudaMallocAsync((void**)&tr->hist_acc, sizeof(unsigned long long), st));
        LT_CUDA(tr, cudaMemsetAsync(tr->hist_acc, 0, sizeof(unsigned long long), st));
    }
    constexpr int kUnr = 4, kThreads = 512;                   // 2 x 64 B in flight per thread
    size_t g = (n + kThreads * 2 * kUnr - 1) / (kThreads * 2 * kUnr);
    const size_t smem = slice_smem_bytes(X);
    // one wave: as many CTAs as are resident together (the flag protocol of the kernel needs CTA 0
    // running while the others wait for it; it is the first one dispatched)
    g = std::max<size_t>(1, std::min<size_t>(g, (size_t)tr->sm_count * 2));   // 3 per SM measured the same
    slice_histogram_kernel<kUnr><<<(unsigned)g, kThreads, smem, st>>>(
        z_dev, n, X, direct ? nullptr : reinterpret_cast<unsigned int*>(tr->hist_acc));
    LT_CUDA(tr, cudaGetLastError());
    tr->launches++;
    return LT_OK;
}

int lt_set_transverse(lt_tracker* tr, const double* matrices_host, int n_seg) {
    if (!tr) return LT_E_NULL;
    if (n_seg == 0) { tr->n_seg = 0; return LT_OK; }
    if (!matrices_host) return LT_E_NULL;
    if (n_seg < 0 || n_seg > kMaxSegments) return LT_E_PARAM;
    for (int k = 0; k < 16 * n_seg; ++k)
        if (!std::isfinite(matrices_host[k])) return LT_E_PARAM;
    if (!tr->lattice_host) {
        tr->lattice_host = (double*)std::malloc((size_t)kMaxSegments * 16 * sizeof(double));
        if (!tr->lattice_host) return LT_E_NOMEM;
    }
    std::memcpy(tr->lattice_host, matrices_host, (size_t)n_seg * 16 * sizeof(double));
    tr->n_seg = n_seg;
    tr->lattice_dirty = 1;
    return LT_OK;
}

int lt_track_transverse_fused(lt_tracker* tr, double* x_dev, double* xp_dev, double* y_dev,
                              double* yp_dev, double* z_dev, double* delta_dev, size_t n,
                              unsigned long long turns, void* stream) {
    return track_transverse_fused(tr, x_dev, xp_dev, y_dev, yp_dev, z_dev, delta_dev, n, turns, stream);
}

int lt_track_transverse_per_turn(lt_tracker* tr, double* x_dev, double* xp_dev, double* y_dev,
                                 double* yp_dev, double* z_dev, double* delta_dev, size_t n,
                                 unsigned long long turns, void* stream) {
    return track_transverse_per_turn(tr, x_dev, xp_dev, y_dev, yp_dev, z_dev, delta_dev, n, turns, stream);
}

}  // extern "C"
