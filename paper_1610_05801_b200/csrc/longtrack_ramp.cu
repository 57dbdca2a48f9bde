// longtrack_ramp.cu -- host side of lt_track_ramp / lt_track_ramp_per_turn: the energy ramp of
// SURVEY.md sec. 8(f) row f2 (G32).
// CUDA path only: nothing here includes, links or calls anything under oracle/.
#include "tracker.hpp"

#include <algorithm>
#include <cmath>
#include <cstring>

#include "kernels_ramp.cuh"

using namespace lt;
using namespace lt_host;

namespace {

constexpr unsigned long long kRampChunkMax = 1ULL << 18;   // turns packed per fused launch

int nsub_of(const lt_tracker* tr) { return tr->p.integrator == LT_RUTH4 ? 3 : 1; }

RampRing make_ring(const lt_tracker* tr) {
    RampRing R;
    const long double gamma = tr->p.gamma;
    const long double beta = sqrtl(1.0L - 1.0L / (gamma * gamma));
    R.mc2 = (double)((long double)tr->p.p0c_eV / (beta * gamma));
    R.alpha_c = tr->p.alpha_c;
    R.qV = tr->p.charge_e * tr->p.voltage_V;
    R.C = tr->p.circumference_m;
    const long double w = cbrtl(2.0L);
    R.x1 = (double)(1.0L / (2.0L - w));
    R.x0 = (double)(-w / (2.0L - w));
    R.to_phase = tr->c64.to_phase;
    R.inv_pi = 0.31830988618379067154;
    return R;
}

// One buffer: `cap` RampEntry (48 B), then `cap` RampScaled (32 B), then the layout flag of the call.
constexpr size_t kRampBytesPerEntry = sizeof(RampEntry) + sizeof(RampScaled);
int ensure_ramp_table(lt_tracker* tr, size_t entries, cudaStream_t st) {
    size_t have = tr->ramp_entries ? tr->ramp_entries * kRampBytesPerEntry + 8 : 0;
    LT_CUDA(tr, grow_async(&tr->ramp_table, &have, entries * kRampBytesPerEntry + 8, st));
    if (tr->ramp_entries < entries) tr->ramp_entries = entries;
    return LT_OK;
}
RampScaled* scaled_table(const lt_tracker* tr) {
    return reinterpret_cast<RampScaled*>(reinterpret_cast<char*>(tr->ramp_table) + tr->ramp_entries * sizeof(RampEntry));
}
unsigned int* layout_flag(const lt_tracker* tr) {
    return reinterpret_cast<unsigned int*>(reinterpret_cast<char*>(tr->ramp_table) + tr->ramp_entries * kRampBytesPerEntry);
}

int check_args(const lt_tracker* tr, const double* z, const double* d, size_t n,
               unsigned long long turns, const double* p0c, const double* volt, const double* phase) {
    if (!tr) return LT_E_NULL;
    if (tr->harm == 0) return LT_E_PARAM;               // phi_s != 0: programme psi_t instead (G32)
    if (n == 0 || turns == 0) return LT_OK;
    if (!z || !d || !p0c) return LT_E_NULL;
    if (!aligned(z, 8) || !aligned(d, 8) || !aligned(p0c, 8)) return LT_E_ALIGN;
    if ((volt && !aligned(volt, 8)) || (phase && !aligned(phase, 8))) return LT_E_ALIGN;
    if (n > ((size_t)1 << 40)) return LT_E_PARAM;
    return LT_OK;
}

// SCALED: the scaled fast layout; flag: the call's layout choice on the device, or nullptr = run
template <int HARM, bool SPLIT, int ILP, bool SCALED>
cudaError_t launch_ramp_fused_ilp(double* z, double* d, size_t n, unsigned int nsteps, unsigned int item_steps,
                                  int first, int last, const PersistentPlan& pl, const lt_tracker* tr,
                                  const unsigned int* flag, cudaStream_t st) {
    auto kern = ramp_persistent_kernel<HARM, SPLIT, ILP, SCALED>;
    // the request caps the CTAs per SM (1 CTA/SM: > half of the 227 KB; 2 CTAs/SM: > a third) and
    // holds 3072 B of staging per warp: 32 warps of a 2-CTA launch need 96 KB, which still fits twice
    const int warps = pl.threads / 32;
    const int smem = std::max(pl.ctas_per_sm == 1 ? 120 * 1024 : 80 * 1024, warps * 3072);
    static std::atomic<unsigned long long> attr_devices{0};   // per instantiation: the devices it is set on
    {
        cudaError_t e = allow_dynamic_smem(attr_devices, kern, 120 * 1024);
        if (e != cudaSuccess) return e;
    }
    unsigned int* const done = reinterpret_cast<unsigned int*>(tr->sched + 1);
    const double2* const table = SCALED ? reinterpret_cast<const double2*>(scaled_table(tr))
                                        : reinterpret_cast<const double2*>(tr->ramp_table);
    int dynamic = pl.dynamic;
    if (dynamic == 2) {                                      // CTAs wait on one another: co-resident or not at all
        const cudaError_t e = launch_coresident(kern, tr->sm_count * pl.ctas_per_sm, pl.threads, (size_t)smem, st,
                                                z, d, n, nsteps, item_steps, first, last, 2, tr->sched, done,
                                                tr->c64, table, flag);
        if (!coresidency_refused(e)) return e;
        (void)cudaGetLastError();
        g_wrap_refused = 1;                                  // same bits from the ticket queue
        dynamic = 1;
        item_steps = std::min(pl.queue_item_turns * (unsigned int)nsub_of(tr), nsteps);
    }
    kern<<<tr->sm_count * pl.ctas_per_sm, pl.threads, smem, st>>>(
        z, d, n, nsteps, item_steps, first, last, dynamic, tr->sched, done, tr->c64, table, flag);
    return cudaGetLastError();
}

// layout: 0 the plain layout only (split drifts, or no RF at all); 1 the scaled layout only (no
// voltage table: the kick amplitude cannot vanish); 2 both launches, the device flag picks one
template <int HARM, bool SPLIT>
cudaError_t launch_ramp_fused(double* z, double* d, size_t n, unsigned int nsteps, unsigned int item_steps,
                              int first, int last, const PersistentPlan& pl, const lt_tracker* tr,
                              int layout, cudaStream_t st) {
    const unsigned int* flag = layout == 2 ? layout_flag(tr) : nullptr;
    cudaError_t e = cudaSuccess;
    if (SPLIT || layout != 1) {
        e = pl.ilp == 2 ? launch_ramp_fused_ilp<HARM, SPLIT, 2, false>(z, d, n, nsteps, item_steps, first, last, pl, tr, flag, st)
                        : launch_ramp_fused_ilp<HARM, SPLIT, 1, false>(z, d, n, nsteps, item_steps, first, last, pl, tr, flag, st);
        if (e != cudaSuccess) return e;
    }
    if (!SPLIT && layout != 0) {
        e = pl.ilp == 2 ? launch_ramp_fused_ilp<HARM, false, 2, true>(z, d, n, nsteps, item_steps, first, last, pl, tr, flag, st)
                        : launch_ramp_fused_ilp<HARM, false, 1, true>(z, d, n, nsteps, item_steps, first, last, pl, tr, flag, st);
    }
    return e;
}

template <int HARM, int NSUB>
cudaError_t launch_ramp_turn(double* z, double* d, size_t n, int reverse, double* partials, bool moments,
                             bool vec, int grid, const lt_tracker* tr, int k, cudaStream_t st) {
    const RampEntry* tab = reinterpret_cast<const RampEntry*>(tr->ramp_table);
#define LT_RT(M, V) ramp_per_turn_kernel<HARM, NSUB, M, V, kPerTurnUnroll><<<grid, kPerTurnThreads, 0, st>>>( \
        z, d, n, reverse, partials, tr->c64, tab, tr->cursor, k)
    if (moments) { if (vec) LT_RT(true, true); else LT_RT(true, false); }
    else         { if (vec) LT_RT(false, true); else LT_RT(false, false); }
#undef LT_RT
    return cudaGetLastError();
}

cudaError_t enqueue_ramp_batch(lt_tracker* tr, double* z, double* d, size_t n, unsigned long long t0,
                               int nb, bool moments, lt_moments* mo, lt_sums* so, bool vec, int grid,
                               cudaStream_t st) {
    const int nsub = nsub_of(tr);
    for (int k = 0; k < nb; ++k) {
        const int reverse = tr->per_turn_reverse ? (int)((t0 + k) & 1ULL) : 0;
        double* part = tr->partials + (size_t)k * grid * kPartialStride;
        cudaError_t e;
        if (tr->harm == 1)
            e = nsub == 3 ? launch_ramp_turn<1, 3>(z, d, n, reverse, part, moments, vec, grid, tr, k, st)
                          : launch_ramp_turn<1, 1>(z, d, n, reverse, part, moments, vec, grid, tr, k, st);
        else
            e = nsub == 3 ? launch_ramp_turn<2, 3>(z, d, n, reverse, part, moments, vec, grid, tr, k, st)
                          : launch_ramp_turn<2, 1>(z, d, n, reverse, part, moments, vec, grid, tr, k, st);
        if (e != cudaSuccess) return e;
        tr->launches++;
    }
    if (moments)
        finalize_kernel<<<nb, 256, 0, st>>>(tr->partials, grid, n, tr->cursor,
                                            reinterpret_cast<unsigned int*>(tr->cursor + 1),
                                            reinterpret_cast<MomentsOut*>(mo),
                                            reinterpret_cast<SumsOut*>(so), nullptr);
    else
        ramp_advance_cursor_kernel<<<1, 1, 0, st>>>(tr->cursor, (unsigned long long)nb);
    tr->launches++;
    return cudaGetLastError();
}

}  // namespace

namespace lt_host {
void destroy_ramp(lt_tracker* tr) {
    if (tr->ramp_table) cudaFree(tr->ramp_table);
    tr->ramp_table = nullptr;
    tr->ramp_entries = 0;
}
}  // namespace lt_host

extern "C" {

int lt_track_ramp(lt_tracker* tr, double* z, double* d, size_t n, unsigned long long turns,
                  const double* p0c, const double* volt, const double* phase, void* stream) {
    int rc = check_args(tr, z, d, n, turns, p0c, volt, phase);
    if (rc || n == 0 || turns == 0) return rc;
    rc = ensure_device(tr);
    if (rc) return rc;
    cudaStream_t st = (cudaStream_t)stream;
    rc = ensure_sched(tr, n, st);
    if (rc) return rc;
    const int nsub = nsub_of(tr);
    const bool split = tr->split_drifts != 0;
    const unsigned long long chunk_max =
        std::min<unsigned long long>((unsigned long long)tr->chunk_turns, kRampChunkMax);
    rc = ensure_ramp_table(tr, (size_t)std::min<unsigned long long>(turns, chunk_max) * nsub + 1, st);   // + header
    if (rc) return rc;
    const PersistentPlan pl = plan_persistent(tr, n, turns, 2);
    g_wrap_refused = 0;
    const RampRing R = make_ring(tr);
    // which fast layout: the scaled one divides by the kick amplitude tau a_t A(p) of every sub-step
    int layout = 0;
    if (!split && R.qV != 0.0 && tr->ramp_scaled != 0) {
        layout = volt ? 2 : 1;
        if (layout == 2) {
            LT_CUDA(tr, cudaMemsetAsync(layout_flag(tr), 0, sizeof(unsigned int), st));
            const unsigned int blocks = (unsigned int)std::min<unsigned long long>((turns + 255) / 256, 1024);
            ramp_scan_kernel<<<blocks, 256, 0, st>>>(volt, turns, layout_flag(tr));
            LT_CUDA(tr, cudaGetLastError());
            tr->launches++;
        }
    }
    unsigned long long done = 0;
    while (done < turns) {
        const unsigned long long chunk = std::min<unsigned long long>(turns - done, chunk_max);
        const int first = done == 0, last = done + chunk == turns;
        const unsigned int item_turns =
            pl.dynamic == 1 ? std::min<unsigned int>(pl.item_turns, (unsigned int)chunk) : (unsigned int)chunk;
        // the table of the previous chunk is free again: its kernel precedes this one on the stream
        ramp_pack_kernel<<<(unsigned)((chunk + 255) / 256), 256, 0, st>>>(
            p0c, volt, phase, done, (unsigned int)chunk, turns, tr->p.integrator, split ? 0 : 1, R,
            reinterpret_cast<RampEntry*>(tr->ramp_table), layout ? scaled_table(tr) : nullptr);
        LT_CUDA(tr, cudaGetLastError());
        if (pl.dynamic) LT_CUDA(tr, cudaMemsetAsync(tr->sched, 0, 8 + 4 * ((n + 31) / 32), st));
        const unsigned int nsteps = (unsigned int)chunk * nsub, item_steps = item_turns * nsub;
        cudaError_t e;
        if (tr->harm == 1)
            e = split ? launch_ramp_fused<1, true>(z, d, n, nsteps, item_steps, first, last, pl, tr, layout, st)
                      : launch_ramp_fused<1, false>(z, d, n, nsteps, item_steps, first, last, pl, tr, layout, st);
        else
            e = split ? launch_ramp_fused<2, true>(z, d, n, nsteps, item_steps, first, last, pl, tr, layout, st)
                      : launch_ramp_fused<2, false>(z, d, n, nsteps, item_steps, first, last, pl, tr, layout, st);
        LT_CUDA(tr, e);
        tr->launches += layout == 2 ? 3 : 2;
        done += chunk;
    }
    tr->last_grid = (long long)tr->sm_count * pl.ctas_per_sm;
    tr->last_block = pl.threads;
    tr->last_ilp = pl.ilp;
    tr->last_mode = pl.dynamic == 2 ? (g_wrap_refused ? 3 : 4) : (pl.dynamic ? 3 : 2);
    tr->last_item_turns = pl.dynamic == 1 ? pl.item_turns : (pl.dynamic == 2 && g_wrap_refused ? pl.queue_item_turns : 0);
    return LT_OK;
}

int lt_track_ramp_per_turn(lt_tracker* tr, double* z, double* d, size_t n, unsigned long long turns,
                           const double* p0c, const double* volt, const double* phase,
                           lt_moments* mo, lt_sums* so, void* stream) {
    int rc = check_args(tr, z, d, n, turns, p0c, volt, phase);
    if (rc || n == 0 || turns == 0) return rc;
    if ((mo && !aligned(mo, 8)) || (so && !aligned(so, 8))) return LT_E_ALIGN;
    if (turns > (1ULL << 26)) return LT_E_PARAM;         // the whole call's table is packed at once
    rc = ensure_device(tr);
    if (rc) return rc;
    cudaStream_t st = (cudaStream_t)stream;
    const int nsub = nsub_of(tr);
    rc = ensure_ramp_table(tr, (size_t)turns * nsub, st);
    if (rc) return rc;
    const bool moments = mo || so;
    const bool vec = aligned(z, 16) && aligned(d, 16);
    const int grid = per_turn_grid(tr, n);
    rc = ensure_scratch(tr, grid, st);
    if (rc) return rc;
    const RampRing R = make_ring(tr);
    for (unsigned long long off = 0; off < turns; off += 1ULL << 20) {
        const unsigned int cnt = (unsigned int)std::min<unsigned long long>(1ULL << 20, turns - off);
        ramp_pack_kernel<<<(cnt + 255) / 256, 256, 0, st>>>(
            p0c, volt, phase, off, cnt, turns, tr->p.integrator, 0, R,
            reinterpret_cast<RampEntry*>(tr->ramp_table) + (size_t)off * nsub, nullptr);
        LT_CUDA(tr, cudaGetLastError());
        tr->launches++;
    }
    set_cursor_kernel<<<1, 1, 0, st>>>(tr->cursor, reinterpret_cast<unsigned int*>(tr->cursor + 1), 0ULL);
    LT_CUDA(tr, cudaGetLastError());
    tr->launches++;
    unsigned long long t0 = 0;
    if (tr->per_turn_graph && turns >= 2ULL * kBatchTurns) {
        GraphKey key;
        std::memset(&key, 0, sizeof(key));
        key.z = z; key.d = d; key.moments = mo; key.sums = so; key.n = n;
        key.reverse = (int)tr->per_turn_reverse; key.grid = grid;
        key.ramp = tr->ramp_table; key.nsub = nsub;
        if (!tr->graph_exec || !(tr->graph_key == key)) {
            if (tr->graph_exec) { cudaGraphExecDestroy(tr->graph_exec); tr->graph_exec = nullptr; }
            if (!tr->capture_stream)
                LT_CUDA(tr, cudaStreamCreateWithFlags(&tr->capture_stream, cudaStreamNonBlocking));
            cudaGraph_t graph = nullptr;
            LT_CUDA(tr, cudaStreamBeginCapture(tr->capture_stream, cudaStreamCaptureModeThreadLocal));
            const long long before = tr->launches;
            cudaError_t e = enqueue_ramp_batch(tr, z, d, n, 0, kBatchTurns, moments, mo, so, vec, grid,
                                               tr->capture_stream);
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
        LT_CUDA(tr, enqueue_ramp_batch(tr, z, d, n, t0, nb, moments, mo, so, vec, grid, st));
        t0 += nb;
    }
    return LT_OK;
}

}  // extern "C"
