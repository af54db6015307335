/* rex_trex_diag.h -- diagnostics of librex_trex.so: probes, counters, kernel-selection knobs and per-flow dumps.
 *
 * NOT part of the product boundary (include/rex_trex.h is: SURVEY.md 8(b)). These entry points exist for tests/,
 * bench.py's roofline denominator and profiles/; a user of the reweighting path never needs them.
 */
#ifndef REX_TREX_DIAG_H
#define REX_TREX_DIAG_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

/* Per-helicity colour-flow amplitudes J_c of ONE event from the first-path walker (one thread per helicity walking
 * every ordering with private currents; momenta_one: HOST [npar][4]), for parity at the level of SURVEY.md I-4.
 * out HOST [nhel][ncolor][2 orders in kappa][re,im], couplings included, order 1 per unit kappa.
 * Only for TREX_SP_GG_TT .. TREX_SP_GG_TTGGG. Synchronous. */
int trex_debug_flow_amps(int subproc_id, const double* momenta_one, const double* theta, double* out);

/* The same for the PRODUCTION kernels (the ones trex_reweight launches and bench.py times: k_gg_tt, k_table<3>,
 * k_table4w, k_table<5>): one event is run through the regular launch with a side buffer that receives the operand of
 * the colour sum. out HOST [nhel][ncolor][2: theta_old, theta_new][re, im] = J_c(theta) = g_s^N (A0 + (kappa/g_s) A1),
 * flows in lexicographic order of the gluon ordering, h as above. fp64 mode; when top mass or width differ between the
 * two parameter points the two-pass kernels are the ones exercised. Synchronous. */
int trex_debug_xtile(int subproc_id, const double* momenta_one, const double* theta_old, const double* theta_new, double* out);

/* Per-helicity |M_h|^2 of the PRODUCTION quark-channel kernels (k_qq: one light line + one gluon; k_qq2: + two gluons):
 * one event is run through the regular launch path, with the kernel template instantiated with its per-helicity dump
 * compiled in (otherwise the same code), and a side buffer receives every helicity configuration's colour-summed value
 * before the helicity sum. out HOST [nhel][2: theta_old, theta_new], h = sum_leg bit(leg) * (helicity
 * of leg is +), couplings and 1 / N_avg included, so that sum_h out[h][.] is what trex_reweight returns as me2; the
 * helicity configurations the massless line forbids are exact zeros. fp64 mode. Synchronous. */
int trex_debug_helicity_me2(int subproc_id, const double* momenta_one, const double* theta_old, const double* theta_new, double* out);

/* Roofline denominator: enqueues ONE launch of a register-resident FMA chain kernel (blocks x 256 threads, 64 FMAs per
 * thread and iteration) on the library stream and returns the floating-point operations it executes (2 per FMA), or a
 * negative error code. mode 0 / 1: FP64 / FP32 chains with two constant-bank operands (pipe peak); 2 / 3: three
 * register operands; 4: FP64 tensor cores (mma.sync.m8n8k4.f64). The caller times it with events on that stream
 * (no FP64 peak is provided, it has to be measured in the same run). */
double trex_probe_fma(int mode, int blocks, int iters);

/* Evaluation strategy of g g -> t t~ + (N-2) g: processes with N >= algo gluons (algo = 3, 4, 5; default 3) use the
 * fused current-table kernel (per-event shared-memory table of off-shell gluon currents shared by all helicities,
 * "helicity recycling"); the others, and all of them for algo = 0, use one thread per helicity unit walking every
 * ordering with private currents. Both evaluate the same colour-ordered recursion; the second one is
 * kept as an in-library cross-check of the first. */
int trex_set_algorithm(int algo);

/* kernels launched by this library since load (bench.py's gpu_launches) */
int64_t trex_launch_count(void);
/* trex_run calls served by replaying the captured CUDA graph since load (tests assert the replay branch was taken) */
int64_t trex_graph_replays(void);

/* Kernel timing for bench.py's roofline: while on, every |M|^2 launch (inside trex_reweight, trex_run, ...) is bracketed by
 * CUDA events on the library stream and trex_run does not replay its CUDA graph. trex_kernel_time synchronises the
 * stream, returns the summed duration [ms] and the number of launches recorded since its last call, and resets both. */
int trex_kernel_timing(int on);
int trex_kernel_time(double* total_ms, int64_t* launches);

#ifdef __cplusplus
}
#endif
#endif /* REX_TREX_DIAG_H */
