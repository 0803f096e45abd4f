/* include/lbm_test.h — test and measurement hooks of liblbm_b200.so.  Not part of the product boundary
 * (include/lbm.h): tests/ and bench.py use them to check single nodes against the oracle and to split a
 * step into its kernels.  Same conventions, ownership and error rules as lbm.h.
 */
#ifndef LBM_B200_TEST_H
#define LBM_B200_TEST_H
#include "lbm.h"

#ifdef __cplusplus
extern "C" {
#endif

/* Test hook: the local update of `count` independent nodes on the device, in the context-free
 * precision `precision` (32/64).  N: HOST 9*count doubles (node-major: N[9*k + q]), phi_nb: HOST
 * 9*count doubles, phi_nb[9*k + q] = phi(x + c_q); outputs Nstar, Bstar (9*count) and fields
 * (8*count: rho, tau, ux, uy, p, Fx, Fy, |grad phi|), any may be NULL. */
int lbm_node_update_batch(const lbm_params* prm, int64_t count, const double* N,
                          const double* phi_nb, double* Nstar, double* Bstar, double* fields);

/* Measurement helper: advances n steps like lbm_step but brackets every kernel launch with CUDA
 * events on the context's stream and returns, after synchronising, the summed device time in
 * milliseconds per kernel kind: ms[0] = collide(+stream), ms[1] = phi-sum (BASELINE only),
 * ms[2] = ghost update.  The event records add a little launch overhead; use lbm_step for
 * throughput and this call for the per-kernel split. */
int lbm_step_timed(lbm_ctx* ctx, int64_t n, double ms[3]);

/* Measurement helper: the ceiling of the state layout.  Runs `iters` passes of a plain copy kernel
 * over the context's own arrays (every 32-byte sector of the 9 population planes and of phi that holds
 * a fluid node is read and written once; no halos, no arithmetic; destination is scratch memory, the
 * state is not disturbed) and returns the mean device time of one pass in milliseconds.  bench.py
 * reports it beside the roofline fraction: it is what a pure streaming pass over this layout costs.
 * LBM_EINVAL if nx*ny is not a whole number of sectors, and for contexts of the compacted layouts (PACK, SPARSE,
 * AUTO), which keep no dense planes: create the context with LBM_SCHEDULE_PAIR to measure. */
int lbm_layout_copy_timed(lbm_ctx* ctx, int32_t iters, double* ms_per_pass);

/* Device-timing helper: per-kernel-kind accumulated launch counts since the last reset;
 * counts[0] = collide(+stream), [1] = phi-sum, [2] = ghost, [3] = other. */
int lbm_launch_counts(lbm_ctx* ctx, int64_t counts[4], int32_t reset);

#ifdef __cplusplus
}
#endif
#endif
