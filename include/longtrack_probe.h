/*
 * longtrack_probe.h -- C ABI of liblongtrack_probe.so: FP64-pipe probes of the device at hand.
 *
 * Measurement tooling for bench.py (the roofline denominators of DESIGN.md sec. 8: SURVEY.md
 * sec. 7 step 5, "FP64 peak probe"), kept OUT of liblongtrack.so so that the product library
 * exports the tracking calls only.  Built from the same kernel headers, so the probed turn loop
 * is the fused kernel's own code.  Error codes are those of longtrack.h.  Both calls allocate a
 * few bytes of device memory, run to completion and synchronise before they return.
 */
#ifndef LONGTRACK_PROBE_H
#define LONGTRACK_PROBE_H

#include "longtrack.h"

#ifdef __cplusplus
extern "C" {
#endif

/* -- roofline probes (measurement only, not on the hot path) ------------------------------
 * Runs a dependent-chain DFMA kernel (`chains` independent chains per thread, `iters` FMAs
 * per chain) and returns achieved FP64 lane-instructions per second in *rate. Synchronises. */
int lt_probe_fp64(int blocks, int threads, int chains, long long iters, double *rate_host,
                  double *ms_host);
/* What the FP64 pipe of the device at hand issues, counted with clock64 (so independent of the
 * clock): `threads` (multiple of 32, <= 1024) threads in each of `blocks` CTAs (one CTA per SM:
 * pass the SM count) run `chains` (1, 2, 4) independent dependent chains of 8 * iters steps of
 *   kind 0  DFMA with three register operands      kind 1  DFMA, two registers + a uniform operand
 *   kind 2  DADD                                   kind 3  DMUL
 *   kind 10 / 11 / 12  the 13-instruction leap-frog turn of the fused kernel
 *                      with the sign flip on the polynomial / on the argument / left out.
 * *instr_per_cycle_host = FP64 warp-instructions per cycle and SM sub-partition (the pipe's
 * nominal peak is 0.5: 16 lanes per sub-partition); *sm_clock_mhz_host (may be NULL) = SM clock
 * during the probe, from clock64 against the nanosecond global timer.  Synchronises. */
int lt_probe_pipe(int kind, int blocks, int threads, int chains, long long iters,
                  double *instr_per_cycle_host, double *sm_clock_mhz_host);

#ifdef __cplusplus
}
#endif

#endif /* LONGTRACK_PROBE_H */
