/*
 * tfstat_probe.h -- ALU-roofline probe: libtfstat_probe.so, a bench-only library built beside
 * libtfstat.so (not part of the product library, not part of the paper's calls).
 *
 * The exponential-window direct sum is bound by the FP32 and XU (MUFU) pipes, not by HBM or
 * tensor cores.  MEASURED_PEAKS.json holds only HBM and bf16 numbers, so
 * bench.py measures the denominators of that roofline live, on the same GPU and clocks as the
 * timed run, with these register-only micro-kernels.
 */
#ifndef TFSTAT_PROBE_H_
#define TFSTAT_PROBE_H_
#include <stdint.h>
#ifdef __cplusplus
extern "C" {
#endif

#define TFSTAT_PROBE_FFMA 0     /* acc_j = a*b + acc_j, 16 independent chains per thread     */
#define TFSTAT_PROBE_FADD 1     /* acc_j = acc_j + a                                           */
#define TFSTAT_PROBE_MUFU_EX2 2 /* x_j = ex2.approx(x_j)                                       */
#define TFSTAT_PROBE_FFMA2 3    /* packed fma.rn.f32x2 (2 lane-ops per thread-instruction)     */
#define TFSTAT_PROBE_FADD2 4    /* packed add.rn.f32x2                                         */
#define TFSTAT_PROBE_FFMA_MUFU 5 /* 8 FFMA : 1 MUFU.EX2 mix (do the pipes overlap?)           */
#define TFSTAT_PROBE_LDS128 6   /* broadcast LDS.128 (one address per warp)                    */
#define TFSTAT_PROBE_DFMA 7     /* fp64 fma                                                    */
#define TFSTAT_PROBE_FFMA2_PAIRS 8       /* fma.rn.f32x2 acc, X, Y: two distinct register pairs */
#define TFSTAT_PROBE_FFMA2_SCALAR_PAIR 9 /* ... acc, (w, w), X: a broadcast scalar and a pair   */
#define TFSTAT_PROBE_FFMA2_SCALARS 10    /* ... acc, (w, w), (x, x): two broadcast scalars      */
#define TFSTAT_PROBE_KINDS 11

/* Runs probe `kind` on the current device (synchronous; default stream; CUDA-event timed,
 * 1 warm-up + `reps` timed launches, best taken).  All outputs are HOST pointers:
 *   *lane_ops_per_s   thread-level operations per second over the whole GPU (a packed x2
 *                     instruction counts 2, an LDS.128 counts 1)
 *   *ops_per_clk_sm   the same per SM clock per SM, from clock64() inside the kernel
 *   *sm_mhz           SM clock implied by clock64() and the event time
 * Returns 0, or a negative tfstat_status. */
int tfstat_probe_alu(int kind, int reps, double *lane_ops_per_s, double *ops_per_clk_sm,
                     double *sm_mhz);

/* The core loop of the direct exponential sum (exp_direct.cu) with NOTHING around it: 192 atoms
 * resident in shared memory, summed `reps` times by 128-thread CTAs (4 per SM for 8 cells per
 * thread, 3 for 16), in one of two accumulator layouts:
 *   form 0  pairs of CHANNELS of one cell: FFMA2 acc, w (broadcast scalar), atom register pair
 *   form 1  pairs of CELLS of one channel: FFMA2 acc, w, x (two broadcast scalars)
 *   form 2, 3  form 1 with two / four more broadcast LDS.128 per atom whose results are not used:
 *           8 / 16 more register write-backs per atom and nothing else
 * cells = 8 or 16 per thread.  Outputs (HOST pointers): window-atom terms per SM clock per SM
 * (clock64 span on SM 0) and terms per second over the whole GPU. */
int tfstat_probe_direct_loop(int form, int cells, int reps, double *terms_per_clk_sm,
                             double *terms_per_s);

#ifdef __cplusplus
}
#endif
#endif
