// longtrack.cu -- host side of liblongtrack.so: the C ABI of include/longtrack.h, parameter
// validation, derived constants, the launch planner and the kernel dispatch.
// CUDA path only: nothing here includes, links or calls anything under oracle/.
#include "tracker.hpp"

#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <new>

#include "sinpi_coeffs.h"

using namespace lt;
using namespace lt_host;

static_assert(sizeof(lt_sums) == sizeof(SumsOut) && sizeof(lt_sums) == 64, "lt_sums layout");
static_assert(sizeof(lt_moments) == sizeof(MomentsOut) && sizeof(lt_moments) == 48, "lt_moments layout");

namespace {

bool finite_all(const lt_params* p) {
    return std::isfinite(p->circumference_m) && std::isfinite(p->gamma) && std::isfinite(p->alpha_c) &&
           std::isfinite(p->p0c_eV) && std::isfinite(p->charge_e) && std::isfinite(p->voltage_V) &&
           std::isfinite(p->phi_s) && std::isfinite(p->ratio2);
}

// Derived constants in fp64, written in the order include/longtrack.h documents.
void derive(const lt_params* p, lt_derived_t* g) {
    const double pi = 3.14159265358979323846;
    g->R = p->circumference_m / (2.0 * pi);
    g->beta = std::sqrt(1.0 - 1.0 / (p->gamma * p->gamma));
    g->eta = p->alpha_c - 1.0 / (p->gamma * p->gamma);
    g->A = p->charge_e * p->voltage_V / (g->beta * p->p0c_eV);
    g->d = g->eta * p->circumference_m / 2.0;
    g->kappa = (double)p->harmonic / g->R;
    g->K = g->eta * p->circumference_m * g->A * (double)p->harmonic / g->R;
    double c = 1.0 - 0.5 * g->K;
    g->mu = (c <= 1.0 && c >= -1.0) ? std::acos(c) : 0.0;
    g->z_max = pi * g->R / (double)p->harmonic;
    g->H_sep = 2.0 * g->A * g->R / (double)p->harmonic;
}

// Kernel constants.  Everything is first formed in 80-bit long double from the raw parameters
// and rounded ONCE to T, so that the folded polynomial coefficients (tau*A*S_k) carry no more
// than half an ulp of error each.
template <typename T>
void fill_consts(const lt_params* p, MapConsts<T>* c) {
    typedef long double L;
    const L pi = 3.14159265358979323846264338327950288L;
    const L C = p->circumference_m, gamma = p->gamma;
    const L R = C / (2.0L * pi);
    const L beta = sqrtl(1.0L - 1.0L / (gamma * gamma));
    const L eta = (L)p->alpha_c - 1.0L / (gamma * gamma);
    const L A = (L)p->charge_e * (L)p->voltage_V / (beta * (L)p->p0c_eV);
    const L d = eta * C / 2.0L;
    const L kappa = (L)p->harmonic / R;
    const L w = cbrtl(2.0L);
    const L x1 = 1.0L / (2.0L - w), x0 = -w / (2.0L - w);
    const L c_half = d * kappa / pi;
    L tau[3] = {1.0L, 1.0L, 1.0L};
    L lead, mid, trail, merged;
    if (p->integrator == LT_RUTH4) {
        tau[0] = x1; tau[1] = x0; tau[2] = x1;
        lead = x1; mid = x1 + x0; trail = x1; merged = 2.0L * x1;
    } else if (p->integrator == LT_EULER_CROMER) {
        lead = 0.0L; mid = 0.0L; trail = 2.0L; merged = 2.0L;
    } else {
        lead = 1.0L; mid = 0.0L; trail = 1.0L; merged = 2.0L;
    }
    std::memset(c, 0, sizeof(*c));
    c->to_phase = (T)(kappa / pi);
    c->from_phase = (T)(pi / kappa);
    c->d = (T)d;
    c->c_half = (T)c_half;
    c->drift_lead = (T)(lead * c_half);
    c->drift_mid = (T)(mid * c_half);
    c->drift_trail = (T)(trail * c_half);
    c->drift_merged = (T)(merged * c_half);
    c->zdrift_lead = (T)(lead * d);
    c->zdrift_mid = (T)(mid * d);
    c->zdrift_trail = (T)(trail * d);
    const long double* S = sizeof(T) == 8 ? LT_SINPI_F64 : LT_SINPI_F32;
    const long double* Cc = sizeof(T) == 8 ? LT_COSPI_F64 : LT_COSPI_F32;
    const int ns = sizeof(T) == 8 ? LT_SINPI_F64_N : LT_SINPI_F32_N;
    const int nc = sizeof(T) == 8 ? LT_COSPI_F64_N : LT_COSPI_F32_N;
    for (int k = 0; k < 3; ++k) {
        for (int j = 0; j < ns; ++j) c->sinA[k][j] = (T)(tau[k] * A * S[j]);
        c->kickA[k] = (T)(tau[k] * A);
    }
    for (int j = 0; j < ns; ++j) c->sin1[j] = (T)S[j];
    for (int j = 0; j < nc; ++j) c->cos1[j] = (T)Cc[j];
    c->two_r = (T)(2.0L * (L)p->ratio2);
    c->phi_off = (T)((L)p->phi_s / pi);
    c->sin_phi_s = (T)sinl((L)p->phi_s);
    c->r = (T)p->ratio2;
    // the two membership thresholds are formed exactly like lt_derived() reports them
    lt_derived_t g;
    derive(p, &g);
    c->z_max = (T)g.z_max;
    c->hn_delta = (T)(eta * C / (2.0L * (L)g.H_sep));
}

}  // namespace
namespace lt_host {
int ensure_device(lt_tracker* tr) {
    if (tr->sm_count > 0) return LT_OK;
    int dev = 0, sms = 0;
    LT_CUDA(tr, cudaGetDevice(&dev));
    LT_CUDA(tr, cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
    if (sms <= 0) { tr->last_cuda_error = (int)cudaErrorNoDevice; return LT_E_CUDA; }
    tr->sm_count = sms;
    return LT_OK;
}
}  // namespace lt_host
namespace {

}  // namespace
namespace lt_host {
int ensure_scratch(lt_tracker* tr, int grid, cudaStream_t st) {
    const size_t need = (size_t)kBatchTurns * (size_t)grid * kPartialStride;
    if (tr->partials_doubles < need) {
        // the cached per-turn graph has the old scratch address baked in
        if (tr->graph_exec) { cudaGraphExecDestroy(tr->graph_exec); tr->graph_exec = nullptr; }
        size_t have = tr->partials_doubles * sizeof(double);
        LT_CUDA(tr, grow_async((void**)&tr->partials, &have, need * sizeof(double), st));
        tr->partials_doubles = need;
    }
    if (!tr->cursor) {
        LT_CUDA(tr, cudaMallocAsync((void**)&tr->cursor, 2 * sizeof(unsigned long long), st));
        LT_CUDA(tr, cudaMemsetAsync(tr->cursor, 0, 2 * sizeof(unsigned long long), st));
    }
    return LT_OK;
}
}  // namespace lt_host
namespace {

// ------------------------------------------------------------------------------------------
// Launch planner for the fused kernel.  The whole ensemble should sit on the chip as ONE
// balanced wave (a particle cannot migrate while its turns run), with enough independent FP64
// chains per SM sub-partition to cover the DFMA latency: score = balance * latency cover.
// ------------------------------------------------------------------------------------------
struct FusedPlan { int block, ilp; long long grid; double score; };

FusedPlan plan_fused(const lt_tracker* tr, size_t n) {
    static const int blocks[] = {64, 128, 32};
    static const int ilps[] = {1, 2, 4};
    const double kChainsWanted = 8.0;     // dependent FP64 chains per sub-partition (measured knee)
    const int sms = tr->sm_count;
    FusedPlan best = {64, 1, 1, -1.0};
    for (int b : blocks) {
        if (tr->fused_block > 0 && b != tr->fused_block) continue;
        for (int ilp : ilps) {
            if (tr->fused_ilp > 0 && tr->fused_ilp <= 4 && ilp != tr->fused_ilp) continue;   // 8: transverse kernel only
            const long long tile = (long long)b * ilp;
            const long long grid = (long long)((n + tile - 1) / tile);
            const int max_res = std::min(32, 2048 / b);           // resident CTAs per SM
            double balance, chains;
            if (grid <= (long long)sms * max_res) {
                const long long per_sm = (grid + sms - 1) / sms;
                balance = ((double)grid / sms) / (double)per_sm;
                chains = (double)per_sm * (b / 32.0) * ilp / 4.0;
            } else {
                const double waves = (double)grid / ((double)sms * max_res);
                balance = waves / std::ceil(waves);
                chains = (double)max_res * (b / 32.0) * ilp / 4.0;
            }
            // effective work per chain also shrinks when n is not a multiple of the tile
            balance *= (double)n / ((double)grid * tile);
            double score = balance * std::min(1.0, chains / kChainsWanted);
            score -= 1e-3 * ilp;                                   // ties: fewer registers
            if (score > best.score) best = {b, ilp, grid, score};
        }
    }
    return best;
}

template <typename T, int INTEG, int HARM, bool SPLIT>
cudaError_t launch_fused_layout(T* z, T* d, size_t n, unsigned int turns, int first, int last,
                                const MapConsts<T>& c, const FusedPlan& pl, bool vec_ok,
                                cudaStream_t st) {
    dim3 grid((unsigned)pl.grid), block((unsigned)pl.block);
    if (pl.ilp == 1)
        fused_kernel<T, INTEG, HARM, SPLIT, 1, false><<<grid, block, 0, st>>>(z, d, n, turns, first, last, c);
    else if (pl.ilp == 2 && vec_ok)
        fused_kernel<T, INTEG, HARM, SPLIT, 2, true><<<grid, block, 0, st>>>(z, d, n, turns, first, last, c);
    else if (pl.ilp == 2)
        fused_kernel<T, INTEG, HARM, SPLIT, 2, false><<<grid, block, 0, st>>>(z, d, n, turns, first, last, c);
    else if (vec_ok)
        fused_kernel<T, INTEG, HARM, SPLIT, 4, true><<<grid, block, 0, st>>>(z, d, n, turns, first, last, c);
    else
        fused_kernel<T, INTEG, HARM, SPLIT, 4, false><<<grid, block, 0, st>>>(z, d, n, turns, first, last, c);
    return cudaGetLastError();
}

template <typename T, int INTEG>
cudaError_t launch_fused_integ(int harm, bool split, T* z, T* d, size_t n, unsigned int turns,
                               int first, int last, const MapConsts<T>& c, const FusedPlan& pl,
                               bool vec_ok, cudaStream_t st) {
    if (harm == 0) return launch_fused_layout<T, INTEG, 0, true>(z, d, n, turns, first, last, c, pl, vec_ok, st);
    if (harm == 1)
        return split ? launch_fused_layout<T, INTEG, 1, true>(z, d, n, turns, first, last, c, pl, vec_ok, st)
                     : launch_fused_layout<T, INTEG, 1, false>(z, d, n, turns, first, last, c, pl, vec_ok, st);
    return split ? launch_fused_layout<T, INTEG, 2, true>(z, d, n, turns, first, last, c, pl, vec_ok, st)
                 : launch_fused_layout<T, INTEG, 2, false>(z, d, n, turns, first, last, c, pl, vec_ok, st);
}

// ------------------------------------------------------------------------------------------
// Persistent fused kernel: one CTA of 4W warps per SM (W warps per sub-partition), residency
// pinned by a dummy dynamic shared-memory request so that the CTA scheduler cannot stack two on
// one SM and leave another empty.
// ------------------------------------------------------------------------------------------
// FP64 warp-instructions per cycle per sub-partition of the turn loop (peak 0.5) at W resident
// warps carrying ILP independent particles per lane, sign flip on f / on q: measured with clock64
// on B200 (profiles/r2_fp64_pipe_probe.md).  Two chains per warp saturate the pipe with half the
// warps, and with them the flip on f wins; with one chain per warp the flip on q wins from W = 5.
double loop_rate(int ilp, int w, bool fq) {
    static const double f1[] = {0, .1234, .2440, .3559, .4380, .4379, .4409, .4420, .4430};
    static const double q1[] = {0, .1157, .2300, .3373, .4266, .4433, .4576, .4600, .4623};
    static const double f2[] = {0, .2455, .4575, .4650, .4665, .4672, .4675, .4678, .4680};
    static const double q2[] = {0, .2283, .4310, .4580, .4626, .4626, .4630, .4632, .4634};
    if (w > 8) w = 8;
    if (w < 0) w = 0;
    return ilp == 2 ? (fq ? q2[w] : f2[w]) : (fq ? q1[w] : f1[w]);
}

}  // namespace
namespace lt_host {
// The best launch shape that the tracker's forced options allow; false when they allow none.
static bool search_persistent(const lt_tracker* tr, size_t n, int max_ilp, int pv, PersistentPlan* out) {
    const int sms = tr->sm_count;
    PersistentPlan best = {0, 4, 1, 512, 0, false, 1, 1};
    double best_score = -1.0;
    for (int ilp = 1; ilp <= max_ilp; ++ilp) {
        if (max_ilp > 1 && (tr->fused_ilp == 1 || tr->fused_ilp == 2) && ilp != tr->fused_ilp) continue;
        const unsigned long long groups = (n + 32 * ilp * pv - 1) / (32 * ilp * pv);
        const double avg = (double)groups / ((double)sms * 4);      // groups per sub-partition
        for (int w = 1; w <= 16; ++w) {
            if (w > 8 && (w & 1)) continue;                  // two CTAs per SM above 8
            if (ilp == 2 && w > 4) continue;                 // 512 threads: 128 registers each
            if (tr->warps_per_smsp > 0 && w != tr->warps_per_smsp) continue;
            const unsigned long long slots = (unsigned long long)sms * 4 * w;
            for (int fq = 0; fq < 2; ++fq) {
                if (tr->flip_on_q >= 0 && fq != tr->flip_on_q) continue;
                for (int dyn = 0; dyn < 3; ++dyn) {          // 0 static, 1 ticket queue, 2 wrap-around
                    double score;
                    // measured (profiles/r2_fused_shapes.md): with 2 warps per sub-partition the ticket
                    // queue costs 1.5 % (an item switch halves the sub-partition's rate, dozens of
                    // switches per warp, tapered tail) and the wrap-around schedule nothing; from 3
                    // warps on the queue's switches hide behind the other warps and its dynamic
                    // balancing is worth 0.3 % over the static schedule
                    if (dyn == 2) {                          // static pre-emptive schedule: no queue, no tail
                        if (groups < slots) continue;
                        if (groups > (1ULL << 31)) continue;   // groups x turns must stay below 2^63
                        score = (w <= 2 ? 1.0 : 0.994) * loop_rate(ilp, w, fq);
                    } else if (dyn == 1) {                   // ticket queue: every slot busy until the tail
                        if (groups <= slots && tr->fused_mode != 3) continue;
                        score = (w <= 2 ? 0.985 : 0.997) * loop_rate(ilp, w, fq);
                        if (groups < slots) score *= (double)groups / (double)slots;   // forced: idle warps
                    } else if (groups <= slots) {            // one wave: busiest sub-partition rules
                        const double per_smsp = std::ceil(avg);
                        if (tr->warps_per_smsp == 0 && (double)w != std::min(per_smsp, ilp == 2 ? 4.0 : 16.0)) continue;
                        score = loop_rate(ilp, (int)per_smsp, fq) * avg / per_smsp;
                    } else {                                 // static, several groups per slot in turn
                        const double rounds = std::ceil((double)groups / (double)slots);
                        score = loop_rate(ilp, w, fq) * avg / (rounds * w);
                    }
                    if (tr->fused_mode == 4 && dyn != 2) continue;
                    if (tr->fused_mode == 3 && dyn != 1) continue;
                    if (tr->fused_mode == 2 && dyn != 0) continue;
                    if (score > best_score) {
                        best_score = score;
                        best.dynamic = dyn;
                        best.warps_per_smsp = w;
                        best.ctas_per_sm = w > 8 ? 2 : 1;
                        best.threads = 128 * w / best.ctas_per_sm;
                        best.flip_on_q = fq != 0;
                        best.ilp = ilp;
                    }
                }
            }
        }
    }
    *out = best;
    return best_score >= 0.0;
}

PersistentPlan plan_persistent(const lt_tracker* tr, size_t n, unsigned long long turns, int max_ilp, int pv) {
    PersistentPlan best = {0, 4, 1, 512, 0, false, 1, 1};
    if (!search_persistent(tr, n, max_ilp, pv, &best)) {
        // The forced options (each valid on its own, include/longtrack.h) admit no launch shape
        // together.  Give them up one at a time, the least binding first -- a fixed, finite list,
        // so the planner always returns; what was actually launched is in LT_STAT_LAST_*.
        lt_tracker relaxed = *tr;
        bool found = false;
        if (relaxed.fused_mode == 4) {                       // wrap-around with fewer groups than slots
            relaxed.fused_mode = 2;
            found = search_persistent(&relaxed, n, max_ilp, pv, &best);
        }
        if (!found && relaxed.fused_ilp == 2) {              // two particles per lane exist up to 4 warps
            relaxed.fused_ilp = 0;                           // per sub-partition only: keep the warp count
            found = search_persistent(&relaxed, n, max_ilp, pv, &best);
        }
        if (!found) {
            relaxed.fused_mode = 0;
            relaxed.warps_per_smsp = 0;
            relaxed.flip_on_q = -1;
            relaxed.fused_ilp = 0;
            found = search_persistent(&relaxed, n, max_ilp, pv, &best);
        }
        if (!found) best = PersistentPlan{0, 4, 1, 512, 0, false, 1, 1};   // n == 0: nothing to place
    }
    // an item switch costs a warp about 3 us (ticket, progress word, state load; store, fence,
    // release), during which its sub-partition runs at half rate when it holds two warps: long
    // items (2048 turns = 120 us) amortise that, and the tapered tail of the schedule
    // (ItemSchedule) keeps the last round short all the same (profiles/r2_fused_shapes.md)
    unsigned long long it = tr->item_turns > 0
                                ? (unsigned long long)tr->item_turns
                                : std::min<unsigned long long>(2048, std::max<unsigned long long>(128, turns / 8));
    best.queue_item_turns = (unsigned int)std::max<unsigned long long>(1, std::min<unsigned long long>(it, turns));
    best.item_turns = best.dynamic == 1 ? best.queue_item_turns : 0;   // 0 = all turns of the launch
    return best;
}
}  // namespace lt_host
namespace {

// V = the register value of a chain: double, or f32x2 (two fp32 particles per packed value)
template <typename T> struct ChainValue { typedef T type; };
template <> struct ChainValue<float> { typedef f32x2 type; };

template <typename T, int INTEG, int HARM, bool SPLIT, bool FQ, int ILP>
cudaError_t launch_persistent_ilp(T* z, T* d, size_t n, unsigned int turns, unsigned int item_turns,
                                  int first, int last, const PersistentPlan& pl, int sms,
                                  unsigned long long* sched, const MapConsts<typename ChainValue<T>::type>& c,
                                  cudaStream_t st) {
    auto kern = fused_persistent_kernel<T, INTEG, HARM, SPLIT, FQ, false, ILP, typename ChainValue<T>::type>;
    // 1 CTA/SM: > half of the 227 KB; 2 CTAs/SM: > a third
    const int smem = pl.ctas_per_sm == 1 ? 120 * 1024 : 80 * 1024;
    static std::atomic<unsigned long long> attr_devices{0};   // per instantiation: the devices it is set on
    {
        cudaError_t e = allow_dynamic_smem(attr_devices, kern, 120 * 1024);
        if (e != cudaSuccess) return e;
    }
    unsigned int* const done = reinterpret_cast<unsigned int*>(sched + 1);
    int dynamic = pl.dynamic;
    if (dynamic == 2) {                                      // CTAs wait on one another: co-resident or not at all
        const cudaError_t e = launch_coresident(kern, sms * pl.ctas_per_sm, pl.threads, (size_t)smem, st, z, d, n,
                                                turns, item_turns, first, last, 2, sched, done, c, nullptr);
        if (!coresidency_refused(e)) return e;
        (void)cudaGetLastError();
        g_wrap_refused = 1;                                  // same bits from the ticket queue
        dynamic = 1;
        item_turns = std::min(pl.queue_item_turns, turns);
    }
    kern<<<sms * pl.ctas_per_sm, pl.threads, smem, st>>>(z, d, n, turns, item_turns, first, last, dynamic, sched,
                                                         done, c, nullptr);
    return cudaGetLastError();
}

template <typename T, int INTEG, int HARM, bool SPLIT, bool FQ>
cudaError_t launch_persistent_one(T* z, T* d, size_t n, unsigned int turns, unsigned int item_turns,
                                  int first, int last, const PersistentPlan& pl, int sms,
                                  unsigned long long* sched, const MapConsts<typename ChainValue<T>::type>& c,
                                  cudaStream_t st) {
    if (pl.ilp == 2)
        return launch_persistent_ilp<T, INTEG, HARM, SPLIT, FQ, 2>(z, d, n, turns, item_turns, first, last, pl, sms, sched, c, st);
    return launch_persistent_ilp<T, INTEG, HARM, SPLIT, FQ, 1>(z, d, n, turns, item_turns, first, last, pl, sms, sched, c, st);
}

template <typename T, int INTEG>
cudaError_t launch_persistent_integ(int harm, bool split, T* z, T* d, size_t n, unsigned int turns,
                                    unsigned int item_turns, int first, int last,
                                    const PersistentPlan& pl, int sms, unsigned long long* sched,
                                    const MapConsts<typename ChainValue<T>::type>& c, cudaStream_t st) {
#define LT_PK(H, S, Q) launch_persistent_one<T, INTEG, H, S, Q>(z, d, n, turns, item_turns, first, last, pl, sms, sched, c, st)
    if (harm == 0) return LT_PK(0, true, false);
    if (harm == 1) {
        if (split) return LT_PK(1, true, false);
        return pl.flip_on_q ? LT_PK(1, false, true) : LT_PK(1, false, false);
    }
    if (split) return LT_PK(2, true, false);
    return pl.flip_on_q ? LT_PK(2, false, true) : LT_PK(2, false, false);
#undef LT_PK
}

}  // namespace
namespace lt_host {
int ensure_sched(lt_tracker* tr, size_t n, cudaStream_t st) {
    const size_t groups = (n + 31) / 32;
    const size_t need = 8 + 4 * groups + 8;
    LT_CUDA(tr, grow_async((void**)&tr->sched, &tr->sched_bytes, need, st));
    return LT_OK;
}
}  // namespace lt_host
namespace {

inline const MapConsts<double>& chain_consts(const lt_tracker* tr, double) { return tr->c64; }
inline const MapConsts<f32x2>& chain_consts(const lt_tracker* tr, float) { return tr->c32x2; }

template <typename T>
int track_fused_persistent(lt_tracker* tr, T* z, T* d, size_t n, unsigned long long turns,
                           cudaStream_t st) {
    const MapConsts<typename ChainValue<T>::type>& c = chain_consts(tr, T());
    constexpr int kPV = sizeof(typename ChainValue<T>::type) / sizeof(T);   // particles per chain value
    const bool split = tr->split_drifts != 0 || tr->harm == 0;
    int rc = ensure_sched(tr, n, st);
    if (rc) return rc;
    unsigned long long done = 0;
    PersistentPlan pl = plan_persistent(tr, n, turns, 2, kPV);
    g_wrap_refused = 0;
    while (done < turns) {
        unsigned long long chunk = std::min<unsigned long long>(turns - done, (unsigned long long)tr->chunk_turns);
        const int first = done == 0, last = done + chunk == turns;
        // a launch of a few turns is launch-bound (bench.py's f1 sweep): static slots then,
        // which need neither the memset of the progress words nor any flag traffic
        if (pl.dynamic && chunk <= 64 && tr->fused_mode == 0) pl.dynamic = 0;
        const unsigned int item = pl.dynamic == 1 ? std::min<unsigned int>(pl.item_turns, (unsigned int)chunk) : (unsigned int)chunk;
        if (pl.dynamic) {                                    // ticket + progress words of this launch
            LT_CUDA(tr, cudaMemsetAsync(tr->sched, 0, 8 + 4 * ((n + 31) / 32), st));
        }
        cudaError_t e;
        switch (tr->p.integrator) {
            case LT_EULER_CROMER:
                e = launch_persistent_integ<T, kEulerCromer>(tr->harm, split, z, d, n, (unsigned)chunk, item, first, last, pl, tr->sm_count, tr->sched, c, st);
                break;
            case LT_LEAPFROG:
                e = launch_persistent_integ<T, kLeapfrog>(tr->harm, split, z, d, n, (unsigned)chunk, item, first, last, pl, tr->sm_count, tr->sched, c, st);
                break;
            default:
                e = launch_persistent_integ<T, kRuth4>(tr->harm, split, z, d, n, (unsigned)chunk, item, first, last, pl, tr->sm_count, tr->sched, c, st);
        }
        LT_CUDA(tr, e);
        tr->launches++;
        done += chunk;
    }
    tr->last_grid = (long long)tr->sm_count * pl.ctas_per_sm;
    tr->last_block = pl.threads;
    tr->last_ilp = pl.ilp * kPV;
    tr->last_mode = pl.dynamic == 2 ? (g_wrap_refused ? 3 : 4) : (pl.dynamic ? 3 : 2);
    tr->last_item_turns = pl.dynamic == 1 ? pl.item_turns : (pl.dynamic == 2 && g_wrap_refused ? pl.queue_item_turns : 0);
    return LT_OK;
}

template <typename T>
int track_fused(lt_tracker* tr, T* z, T* d, size_t n, unsigned long long turns, void* stream) {
    if (!tr) return LT_E_NULL;
    if (n == 0 || turns == 0) return LT_OK;
    if (!z || !d) return LT_E_NULL;
    if (!aligned(z, sizeof(T)) || !aligned(d, sizeof(T))) return LT_E_ALIGN;
    if (n > ((size_t)1 << 40)) return LT_E_PARAM;
    int rc = ensure_device(tr);
    if (rc) return rc;
    const MapConsts<T>& c = *reinterpret_cast<const MapConsts<T>*>(
        sizeof(T) == 8 ? (const void*)&tr->c64 : (const void*)&tr->c32);
    if (tr->fused_mode != 1) return track_fused_persistent<T>(tr, z, d, n, turns, (cudaStream_t)stream);
    const FusedPlan pl = plan_fused(tr, n);
    const bool vec_ok = aligned(z, 2 * sizeof(T)) && aligned(d, 2 * sizeof(T));
    const bool split = tr->split_drifts != 0 || tr->harm == 0;
    cudaStream_t st = (cudaStream_t)stream;
    unsigned long long done = 0;
    while (done < turns) {
        unsigned long long chunk = turns - done;
        if (chunk > (unsigned long long)tr->chunk_turns) chunk = (unsigned long long)tr->chunk_turns;
        const int first = done == 0, last = done + chunk == turns;
        cudaError_t e;
        switch (tr->p.integrator) {
            case LT_EULER_CROMER:
                e = launch_fused_integ<T, kEulerCromer>(tr->harm, split, z, d, n, (unsigned)chunk, first, last, c, pl, vec_ok, st);
                break;
            case LT_LEAPFROG:
                e = launch_fused_integ<T, kLeapfrog>(tr->harm, split, z, d, n, (unsigned)chunk, first, last, c, pl, vec_ok, st);
                break;
            default:
                e = launch_fused_integ<T, kRuth4>(tr->harm, split, z, d, n, (unsigned)chunk, first, last, c, pl, vec_ok, st);
        }
        LT_CUDA(tr, e);
        tr->launches++;
        done += chunk;
    }
    tr->last_grid = pl.grid; tr->last_block = pl.block; tr->last_ilp = pl.ilp;
    tr->last_mode = 1; tr->last_item_turns = 0;
    return LT_OK;
}

// ------------------------------------------------------------------------------------------
// per-turn mode
// ------------------------------------------------------------------------------------------
template <typename T, int INTEG, int HARM>
cudaError_t launch_per_turn_one(T* z, T* d, size_t n, int reverse, double* partials, bool moments,
                                bool vec_ok, int grid, const MapConsts<T>& c, cudaStream_t st) {
    if (vec_ok) {
        if (moments)
            per_turn_kernel<T, INTEG, HARM, true, kPerTurnUnroll><<<grid, kPerTurnThreads, 0, st>>>(z, d, n, reverse, partials, c);
        else
            per_turn_kernel<T, INTEG, HARM, false, kPerTurnUnroll><<<grid, kPerTurnThreads, 0, st>>>(z, d, n, reverse, partials, c);
    } else {
        if (moments)
            per_turn_kernel_scalar<T, INTEG, HARM, true><<<grid, kPerTurnThreads, 0, st>>>(z, d, n, partials, c);
        else
            per_turn_kernel_scalar<T, INTEG, HARM, false><<<grid, kPerTurnThreads, 0, st>>>(z, d, n, partials, c);
    }
    return cudaGetLastError();
}

template <typename T>
cudaError_t launch_per_turn(const lt_tracker* tr, T* z, T* d, size_t n, int reverse,
                            double* partials, bool moments, bool vec_ok, int grid,
                            const MapConsts<T>& c, cudaStream_t st) {
#define LT_PT(INTEG)                                                                                   \
    (tr->harm == 0   ? launch_per_turn_one<T, INTEG, 0>(z, d, n, reverse, partials, moments, vec_ok, grid, c, st) \
     : tr->harm == 1 ? launch_per_turn_one<T, INTEG, 1>(z, d, n, reverse, partials, moments, vec_ok, grid, c, st) \
                     : launch_per_turn_one<T, INTEG, 2>(z, d, n, reverse, partials, moments, vec_ok, grid, c, st))
    switch (tr->p.integrator) {
        case LT_EULER_CROMER: return LT_PT(kEulerCromer);
        case LT_LEAPFROG: return LT_PT(kLeapfrog);
        default: return LT_PT(kRuth4);
    }
#undef LT_PT
}

}  // namespace
namespace lt_host {
int per_turn_grid(const lt_tracker* tr, size_t n) {
    const size_t tile = (size_t)kPerTurnThreads * kPerTurnUnroll * 2;
    size_t tiles = (n + tile - 1) / tile;
    // 0 = planner: 6 CTAs of 256 threads per SM (4 are resident at 56 registers, the rest refill
    // the SMs as the first ones retire) while the state is at most ~2x the L2; 12 beyond that,
    // where nothing of a turn survives in L2 and the finer grain wins (+5-7 % at 2e7 .. 8e7 particles)
    const size_t per_sm = tr->per_turn_ctas_per_sm > 0 ? (size_t)tr->per_turn_ctas_per_sm
                                                       : (n <= (size_t)15000000 ? 6 : 12);
    size_t g = (size_t)tr->sm_count * per_sm;
    if (g > tiles) g = tiles;
    if (g < 1) g = 1;
    return (int)g;
}
}  // namespace lt_host
namespace {

// enqueue `nb` (<= kBatchTurns) turns starting at absolute turn index t0, then their finalize
template <typename T>
cudaError_t enqueue_batch(lt_tracker* tr, T* z, T* d, size_t n, unsigned long long t0, int nb,
                          bool moments, lt_moments* mo, lt_sums* so, bool vec_ok, int grid,
                          const MapConsts<T>& c, cudaStream_t st) {
    for (int k = 0; k < nb; ++k) {
        const int reverse = tr->per_turn_reverse ? (int)((t0 + k) & 1ULL) : 0;
        double* part = tr->partials ? tr->partials + (size_t)k * grid * kPartialStride : nullptr;
        cudaError_t e = launch_per_turn<T>(tr, z, d, n, reverse, part, moments, vec_ok, grid, c, st);
        if (e != cudaSuccess) return e;
        tr->launches++;
    }
    if (moments) {
        finalize_kernel<<<nb, 256, 0, st>>>(tr->partials, grid, n, tr->cursor,
                                            reinterpret_cast<unsigned int*>(tr->cursor + 1),
                                            reinterpret_cast<MomentsOut*>(mo),
                                            reinterpret_cast<SumsOut*>(so), nullptr);
        tr->launches++;
        return cudaGetLastError();
    }
    return cudaSuccess;
}

template <typename T>
int track_per_turn(lt_tracker* tr, T* z, T* d, size_t n, unsigned long long turns,
                   lt_moments* mo, lt_sums* so, void* stream) {
    if (!tr) return LT_E_NULL;
    if (n == 0 || turns == 0) return LT_OK;
    if (!z || !d) return LT_E_NULL;
    if (!aligned(z, sizeof(T)) || !aligned(d, sizeof(T))) return LT_E_ALIGN;
    if ((mo && !aligned(mo, 8)) || (so && !aligned(so, 8))) return LT_E_ALIGN;
    if (n > ((size_t)1 << 40)) return LT_E_PARAM;
    int rc = ensure_device(tr);
    if (rc) return rc;
    const MapConsts<T>& c = *reinterpret_cast<const MapConsts<T>*>(
        sizeof(T) == 8 ? (const void*)&tr->c64 : (const void*)&tr->c32);
    const bool moments = mo || so;
    const bool vec_ok = aligned(z, 2 * sizeof(T)) && aligned(d, 2 * sizeof(T));
    const int grid = per_turn_grid(tr, n);
    cudaStream_t st = (cudaStream_t)stream;
    if (moments) {
        rc = ensure_scratch(tr, grid, st);
        if (rc) return rc;
        set_cursor_kernel<<<1, 1, 0, st>>>(tr->cursor, reinterpret_cast<unsigned int*>(tr->cursor + 1), 0ULL);
        LT_CUDA(tr, cudaGetLastError());
        tr->launches++;
    }
    unsigned long long t0 = 0;
    // full batches, replayed from a cached CUDA graph when enabled
    if (tr->per_turn_graph && turns >= 2ULL * kBatchTurns) {
        GraphKey key = {(void*)z, (void*)d, (void*)mo, (void*)so, n, sizeof(T) == 4,
                        (int)tr->per_turn_reverse, grid, nullptr, nullptr, nullptr, 0.0, 0.0, 0};
        if (!tr->graph_exec || !(tr->graph_key == key)) {
            if (tr->graph_exec) { cudaGraphExecDestroy(tr->graph_exec); tr->graph_exec = nullptr; }
            if (!tr->capture_stream)
                LT_CUDA(tr, cudaStreamCreateWithFlags(&tr->capture_stream, cudaStreamNonBlocking));
            cudaGraph_t graph = nullptr;
            LT_CUDA(tr, cudaStreamBeginCapture(tr->capture_stream, cudaStreamCaptureModeThreadLocal));
            const long long before = tr->launches;
            cudaError_t e = enqueue_batch<T>(tr, z, d, n, 0, kBatchTurns, moments, mo, so, vec_ok, grid, c, tr->capture_stream);
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
            tr->launches += kBatchTurns + (moments ? 1 : 0);
            t0 += kBatchTurns;
        }
    }
    while (t0 < turns) {
        const int nb = (int)std::min<unsigned long long>(kBatchTurns, turns - t0);
        LT_CUDA(tr, enqueue_batch<T>(tr, z, d, n, t0, nb, moments, mo, so, vec_ok, grid, c, st));
        t0 += nb;
    }
    return LT_OK;
}

template <typename T, bool ONLY_COUNT>
int state_sums(lt_tracker* tr, const T* z, const T* d, size_t n, lt_moments* mo, lt_sums* so,
               unsigned long long* count, void* stream) {
    if (!tr) return LT_E_NULL;
    if (ONLY_COUNT ? !count : (!mo && !so)) return LT_E_NULL;
    if (n > 0 && (!z || !d)) return LT_E_NULL;
    if (n > 0 && (!aligned(z, sizeof(T)) || !aligned(d, sizeof(T)))) return LT_E_ALIGN;
    int rc = ensure_device(tr);
    if (rc) return rc;
    const MapConsts<T>& c = *reinterpret_cast<const MapConsts<T>*>(
        sizeof(T) == 8 ? (const void*)&tr->c64 : (const void*)&tr->c32);
    cudaStream_t st = (cudaStream_t)stream;
    size_t g = (n + 255) / 256;
    if (g > (size_t)tr->sm_count * 8) g = (size_t)tr->sm_count * 8;
    if (g < 1) g = 1;
    rc = ensure_scratch(tr, (int)g, st);
    if (rc) return rc;
    state_sums_kernel<T, ONLY_COUNT><<<(unsigned)g, 256, 0, st>>>(z, d, n, tr->partials, c);
    LT_CUDA(tr, cudaGetLastError());
    finalize_kernel<<<1, 256, 0, st>>>(tr->partials, (int)g, n, nullptr, nullptr,
                                       reinterpret_cast<MomentsOut*>(mo),
                                       reinterpret_cast<SumsOut*>(so), count);
    LT_CUDA(tr, cudaGetLastError());
    tr->launches += 2;
    return LT_OK;
}

}  // namespace

namespace lt_host {
int track_fused_f64(lt_tracker* tr, double* z, double* d, size_t n, unsigned long long turns,
                    void* stream) {
    return track_fused<double>(tr, z, d, n, turns, stream);
}
cudaError_t launch_per_turn_f64(const lt_tracker* tr, double* z, double* d, size_t n, int reverse,
                                double* partials, bool moments, bool vec_ok, int grid,
                                cudaStream_t st) {
    return launch_per_turn<double>(tr, z, d, n, reverse, partials, moments, vec_ok, grid, tr->c64, st);
}
}  // namespace lt_host

// ------------------------------------------------------------------------------------------
// C ABI
// ------------------------------------------------------------------------------------------
extern "C" {

int lt_version(void) { return LT_VERSION; }

const char* lt_strerror(int code) {
    switch (code) {
        case LT_OK: return "ok";
        case LT_E_NULL: return "required pointer is NULL";
        case LT_E_PARAM: return "invalid parameter";
        case LT_E_UNSTABLE: return "linearised map is unstable (K_eff outside [0, 4))";
        case LT_E_ALIGN: return "array pointer is not aligned to its element size";
        case LT_E_CUDA: return "CUDA runtime error (see lt_last_cuda_error)";
        case LT_E_NOMEM: return "out of host memory";
        case LT_E_CAPACITY: return "n exceeds the fixed capacity of this no-allocation entry point (LT_STATIC_MAX_PARTICLES)";
        default: return "unknown error code";
    }
}

int lt_create(const lt_params* p, lt_tracker** out) {
    if (!p || !out) return LT_E_NULL;
    *out = nullptr;
    if (!finite_all(p)) return LT_E_PARAM;
    if (!(p->gamma > 1.0) || !(p->circumference_m > 0.0) || p->harmonic <= 0 || !(p->p0c_eV > 0.0))
        return LT_E_PARAM;
    if (p->integrator != LT_EULER_CROMER && p->integrator != LT_LEAPFROG && p->integrator != LT_RUTH4)
        return LT_E_PARAM;
    lt_derived_t g;
    derive(p, &g);
    const double k_eff = g.K * (std::cos(p->phi_s) + 2.0 * p->ratio2);
    if (!(k_eff >= 0.0) || !(k_eff < 4.0)) return LT_E_UNSTABLE;
    lt_tracker* tr = new (std::nothrow) lt_tracker;
    if (!tr) return LT_E_NOMEM;
    std::memset(tr, 0, sizeof(*tr));
    tr->p = *p;
    tr->g = g;
    fill_consts<double>(p, &tr->c64);
    fill_consts<float>(p, &tr->c32);
    {   // every fp32 constant twice: the packed (two particles per value) form of the same numbers
        static_assert(sizeof(MapConsts<f32x2>) == 2 * sizeof(MapConsts<float>), "packed constants");
        const float* src = reinterpret_cast<const float*>(&tr->c32);
        float* dst = reinterpret_cast<float*>(&tr->c32x2);
        for (size_t k = 0; k < sizeof(MapConsts<float>) / sizeof(float); ++k) { dst[2 * k] = src[k]; dst[2 * k + 1] = src[k]; }
    }
    tr->harm = (p->phi_s != 0.0) ? 0 : (p->ratio2 != 0.0 ? 2 : 1);
    tr->split_drifts = 0;
    tr->chunk_turns = 1LL << 22;
    tr->per_turn_graph = 1;
    tr->per_turn_ctas_per_sm = 0;
    tr->per_turn_reverse = 1;
    tr->fused_mode = 0;
    tr->item_turns = 0;
    tr->warps_per_smsp = 0;
    tr->flip_on_q = -1;
    tr->ramp_scaled = 1;
    *out = tr;
    return LT_OK;
}

int lt_destroy(lt_tracker* tr) {
    if (!tr) return LT_OK;
    if (tr->graph_exec) cudaGraphExecDestroy(tr->graph_exec);
    if (tr->capture_stream) cudaStreamDestroy(tr->capture_stream);
    if (tr->partials) cudaFree(tr->partials);
    if (tr->cursor) cudaFree(tr->cursor);
    if (tr->sched) cudaFree(tr->sched);
    if (tr->stage_z) cudaFree(tr->stage_z);
    if (tr->stage_d) cudaFree(tr->stage_d);
    if (tr->stage_count) cudaFree(tr->stage_count);
    if (tr->own_stream) cudaStreamDestroy(tr->own_stream);
    destroy_next(tr);
    destroy_ramp(tr);
    (void)cudaGetLastError();
    delete tr;
    return LT_OK;
}

int lt_derived(const lt_tracker* tr, lt_derived_t* out) {
    if (!tr || !out) return LT_E_NULL;
    *out = tr->g;
    return LT_OK;
}

int lt_set_option(lt_tracker* tr, int option, long long value) {
    if (!tr) return LT_E_NULL;
    switch (option) {
        case LT_OPT_SPLIT_DRIFTS: tr->split_drifts = value != 0; return LT_OK;
        case LT_OPT_CHUNK_TURNS:
            if (value < 1 || value > (1LL << 31) - 1) return LT_E_PARAM;
            tr->chunk_turns = value; return LT_OK;
        case LT_OPT_FUSED_ILP:
            if (value != 0 && value != 1 && value != 2 && value != 4 && value != 8) return LT_E_PARAM;
            tr->fused_ilp = value; return LT_OK;
        case LT_OPT_FUSED_BLOCK:
            if (value != 0 && value != 32 && value != 64 && value != 128) return LT_E_PARAM;
            tr->fused_block = value; return LT_OK;
        case LT_OPT_PER_TURN_GRAPH: tr->per_turn_graph = value != 0; return LT_OK;
        case LT_OPT_PER_TURN_CTAS_PER_SM:
            if (value < 0 || value > 32) return LT_E_PARAM;
            tr->per_turn_ctas_per_sm = value; return LT_OK;
        case LT_OPT_PER_TURN_REVERSE: tr->per_turn_reverse = value != 0; return LT_OK;
        case LT_OPT_FUSED_MODE:
            if (value < 0 || value > 4) return LT_E_PARAM;
            tr->fused_mode = value; return LT_OK;
        case LT_OPT_ITEM_TURNS:
            if (value < 0 || value > (1LL << 31) - 1) return LT_E_PARAM;
            tr->item_turns = value; return LT_OK;
        case LT_OPT_WARPS_PER_SMSP:
            if (value < 0 || value > 16 || (value > 8 && (value & 1))) return LT_E_PARAM;
            tr->warps_per_smsp = value; return LT_OK;
        case LT_OPT_FLIP_ON_Q:
            if (value < -1 || value > 1) return LT_E_PARAM;
            tr->flip_on_q = value; return LT_OK;
        case LT_OPT_RAMP_SCALED: tr->ramp_scaled = value != 0; return LT_OK;
        case LT_OPT_LATTICE_SOURCE:
            if (value < 0 || value > 2) return LT_E_PARAM;
            tr->lattice_source = value; return LT_OK;
        default: return LT_E_PARAM;
    }
}

int lt_get_option(const lt_tracker* tr, int option, long long* value) {
    if (!tr || !value) return LT_E_NULL;
    switch (option) {
        case LT_OPT_SPLIT_DRIFTS: *value = tr->split_drifts; return LT_OK;
        case LT_OPT_CHUNK_TURNS: *value = tr->chunk_turns; return LT_OK;
        case LT_OPT_FUSED_ILP: *value = tr->fused_ilp; return LT_OK;
        case LT_OPT_FUSED_BLOCK: *value = tr->fused_block; return LT_OK;
        case LT_OPT_PER_TURN_GRAPH: *value = tr->per_turn_graph; return LT_OK;
        case LT_OPT_PER_TURN_CTAS_PER_SM: *value = tr->per_turn_ctas_per_sm; return LT_OK;
        case LT_OPT_PER_TURN_REVERSE: *value = tr->per_turn_reverse; return LT_OK;
        case LT_OPT_FUSED_MODE: *value = tr->fused_mode; return LT_OK;
        case LT_OPT_ITEM_TURNS: *value = tr->item_turns; return LT_OK;
        case LT_OPT_WARPS_PER_SMSP: *value = tr->warps_per_smsp; return LT_OK;
        case LT_OPT_FLIP_ON_Q: *value = tr->flip_on_q; return LT_OK;
        case LT_OPT_RAMP_SCALED: *value = tr->ramp_scaled; return LT_OK;
        case LT_OPT_LATTICE_SOURCE: *value = tr->lattice_source; return LT_OK;
        default: return LT_E_PARAM;
    }
}

int lt_get_stat(const lt_tracker* tr, int stat, long long* value) {
    if (!tr || !value) return LT_E_NULL;
    switch (stat) {
        case LT_STAT_KERNEL_LAUNCHES: *value = tr->launches; return LT_OK;
        case LT_STAT_LAST_GRID: *value = tr->last_grid; return LT_OK;
        case LT_STAT_LAST_BLOCK: *value = tr->last_block; return LT_OK;
        case LT_STAT_LAST_ILP: *value = tr->last_ilp; return LT_OK;
        case LT_STAT_SM_COUNT: *value = tr->sm_count; return LT_OK;
        case LT_STAT_LAST_MODE: *value = tr->last_mode; return LT_OK;
        case LT_STAT_LAST_ITEM_TURNS: *value = tr->last_item_turns; return LT_OK;
        default: return LT_E_PARAM;
    }
}

int lt_last_cuda_error(const lt_tracker* tr) { return tr ? tr->last_cuda_error : 0; }

int lt_track_fused(lt_tracker* tr, double* z_dev, double* delta_dev, size_t n,
                   unsigned long long turns, void* stream) {
    return track_fused<double>(tr, z_dev, delta_dev, n, turns, stream);
}

int lt_track_fused_f32(lt_tracker* tr, float* z_dev, float* delta_dev, size_t n,
                       unsigned long long turns, void* stream) {
    return track_fused<float>(tr, z_dev, delta_dev, n, turns, stream);
}

int lt_track_per_turn(lt_tracker* tr, double* z_dev, double* delta_dev, size_t n,
                      unsigned long long turns, lt_moments* moments_dev, lt_sums* sums_dev,
                      void* stream) {
    return track_per_turn<double>(tr, z_dev, delta_dev, n, turns, moments_dev, sums_dev, stream);
}

int lt_track_per_turn_f32(lt_tracker* tr, float* z_dev, float* delta_dev, size_t n,
                          unsigned long long turns, lt_moments* moments_dev, lt_sums* sums_dev,
                          void* stream) {
    return track_per_turn<float>(tr, z_dev, delta_dev, n, turns, moments_dev, sums_dev, stream);
}

int lt_bucket_count(lt_tracker* tr, const double* z_dev, const double* delta_dev, size_t n,
                    unsigned long long* count_dev, void* stream) {
    return state_sums<double, true>(tr, z_dev, delta_dev, n, nullptr, nullptr, count_dev, stream);
}

int lt_bucket_count_f32(lt_tracker* tr, const float* z_dev, const float* delta_dev, size_t n,
                        unsigned long long* count_dev, void* stream) {
    return state_sums<float, true>(tr, z_dev, delta_dev, n, nullptr, nullptr, count_dev, stream);
}

int lt_moments_now(lt_tracker* tr, const double* z_dev, const double* delta_dev, size_t n,
                   lt_moments* moments_dev, lt_sums* sums_dev, void* stream) {
    return state_sums<double, false>(tr, z_dev, delta_dev, n, moments_dev, sums_dev, nullptr, stream);
}

int lt_moments_from_sums(const lt_sums* s, size_t count, lt_moments* out) {
    if (count == 0) return LT_OK;
    if (!s || !out) return LT_E_NULL;
    for (size_t i = 0; i < count; ++i) {
        const double inv = s[i].n > 0.0 ? 1.0 / s[i].n : 0.0;
        const double mz = s[i].sum_z * inv, md = s[i].sum_d * inv;
        const double vz = std::fma(-mz, mz, s[i].sum_zz * inv);
        const double vd = std::fma(-md, md, s[i].sum_dd * inv);
        out[i].mean_z = mz;
        out[i].mean_d = md;
        out[i].rms_z = std::sqrt(vz > 0.0 ? vz : 0.0);
        out[i].rms_d = std::sqrt(vd > 0.0 ? vd : 0.0);
        out[i].cov_zd = std::fma(-mz, md, s[i].sum_zd * inv);
        out[i].n_in_bucket = (unsigned long long)(s[i].n_in_bucket + 0.5);
    }
    return LT_OK;
}

int lt_track_fused_host(lt_tracker* tr, double* z_host, double* delta_host, size_t n,
                        unsigned long long turns, unsigned long long* count_host) {
    if (!tr) return LT_E_NULL;
    if (n == 0) { if (count_host) *count_host = 0; return LT_OK; }
    if (!z_host || !delta_host) return LT_E_NULL;
    int rc = ensure_device(tr);
    if (rc) return rc;
    if (!tr->own_stream) LT_CUDA(tr, cudaStreamCreateWithFlags(&tr->own_stream, cudaStreamNonBlocking));
    if (tr->stage_n < n) {
        if (tr->stage_z) { cudaFree(tr->stage_z); tr->stage_z = nullptr; }
        if (tr->stage_d) { cudaFree(tr->stage_d); tr->stage_d = nullptr; }
        tr->stage_n = 0;
        LT_CUDA(tr, cudaMalloc(&tr->stage_z, n * sizeof(double)));
        LT_CUDA(tr, cudaMalloc(&tr->stage_d, n * sizeof(double)));
        tr->stage_n = n;
    }
    if (!tr->stage_count) LT_CUDA(tr, cudaMalloc(&tr->stage_count, sizeof(unsigned long long)));
    cudaStream_t st = tr->own_stream;
    LT_CUDA(tr, cudaMemcpyAsync(tr->stage_z, z_host, n * sizeof(double), cudaMemcpyHostToDevice, st));
    LT_CUDA(tr, cudaMemcpyAsync(tr->stage_d, delta_host, n * sizeof(double), cudaMemcpyHostToDevice, st));
    rc = track_fused<double>(tr, tr->stage_z, tr->stage_d, n, turns, (void*)st);
    if (rc) return rc;
    if (count_host) {
        rc = state_sums<double, true>(tr, tr->stage_z, tr->stage_d, n, nullptr, nullptr, tr->stage_count, (void*)st);
        if (rc) return rc;
        LT_CUDA(tr, cudaMemcpyAsync(count_host, tr->stage_count, sizeof(unsigned long long), cudaMemcpyDeviceToHost, st));
    }
    LT_CUDA(tr, cudaMemcpyAsync(z_host, tr->stage_z, n * sizeof(double), cudaMemcpyDeviceToHost, st));
    LT_CUDA(tr, cudaMemcpyAsync(delta_host, tr->stage_d, n * sizeof(double), cudaMemcpyDeviceToHost, st));
    LT_CUDA(tr, cudaStreamSynchronize(st));
    return LT_OK;
}

int lt_plan_fused(const lt_tracker* tr, size_t n, unsigned long long turns, int sm_count, int fp32,
                  long long plan[7]) {
    if (!tr || !plan) return LT_E_NULL;
    if (sm_count < 1 || n == 0 || turns == 0) return LT_E_PARAM;
    lt_tracker tmp = *tr;                                 // plain data: the planner only reads it
    tmp.sm_count = sm_count;
    const int pv = fp32 ? 2 : 1;
    const PersistentPlan pl = plan_persistent(&tmp, n, turns, 2, pv);
    plan[0] = pl.dynamic; plan[1] = pl.warps_per_smsp; plan[2] = pl.ctas_per_sm; plan[3] = pl.threads;
    plan[4] = pl.item_turns; plan[5] = pl.flip_on_q ? 1 : 0; plan[6] = (long long)pl.ilp * pv;
    return LT_OK;
}

int lt_item_schedule(unsigned int turns, unsigned int item_turns, int taper, unsigned int c,
                     unsigned int* nchunks, unsigned int* start, unsigned int* len) {
    if (!nchunks) return LT_E_NULL;
    if (turns == 0 || item_turns == 0) return LT_E_PARAM;
    ItemSchedule s;
    s.init(turns, item_turns, taper);
    *nchunks = s.nchunks;
    if (start || len) {
        if (c >= s.nchunks) return LT_E_PARAM;
        unsigned int a = 0, b = 0;
        s.span(c, taper, &a, &b);
        if (start) *start = a;
        if (len) *len = b;
    }
    return LT_OK;
}

}  // extern "C"
