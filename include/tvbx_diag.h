/* tvbx_diag.h -- DIAGNOSTICS of libtvbx.so: reports for bench.py and the tests, not part of the method's boundary.
 *
 * include/tvbx.h is the boundary SURVEY.md section 8(b) lists (connectome, sweep, run, readout and the bit-exact
 * bookkeeping accessors).  The calls below only describe HOW the library ran a sweep -- which kernel, which launch
 * geometry, how long each kernel class took, how many bytes crossed PCIe -- so that the measurement of DESIGN.md
 * section 7 can be taken from outside the library.  None of them changes a result.
 * Same conventions as tvbx.h: int32 status, thread-local error text, host pointers.
 */
#ifndef TVBX_DIAG_H
#define TVBX_DIAG_H

#include "tvbx.h"

#ifdef __cplusplus
extern "C" {
#endif

/* Kernel timing (bench.py's roofline line): while enabled, every kernel launch of this sweep is bracketed by CUDA
 * events on the launching stream.  tvbx_profile_read synchronises those events, returns the summed durations [ms]
 * and launch counts per kernel class since the last read (0 = integrator, 1 = FC epilogue kernels, 2 = readout,
 * 3 = reset fills) and clears the list. */
int32_t tvbx_profile_enable(tvbx_sweep* sw, int32_t on);
int32_t tvbx_profile_read(tvbx_sweep* sw, double ms[4], int64_t launches[4]);
/* bytes this sweep object copied host->device and device->host so far (tables, parameters, results) */
int32_t tvbx_bytes_copied(const tvbx_sweep* sw, int64_t* h2d, int64_t* d2h);
/* launch geometry chosen for the integrator: CTAs, threads per CTA, sims per CTA, registers per thread, dynamic
 * shared memory bytes, region passes per time block, samples per FC chunk, local-memory bytes per thread,
 * CTAs per group (thread-block cluster size), 2 if the low-latency warp-pair form runs (else 1) */
int32_t tvbx_launch_info(const tvbx_sweep* sw, int32_t info[10]);
/* name of the integrator kernel this sweep runs: "tvbx::integrate2_kernel" = the packed FP32 product kernel
 * (tau_e == tau_i, regions-per-CTA * sims_per_cta <= 480, sims_per_cta <= 8), "tvbx::integrate_kernel" = the general
 * one (FP64 build mode, tau_e != tau_i, larger CTAs).  Copies at most n bytes including the NUL. */
int32_t tvbx_kernel_name(const tvbx_sweep* sw, char* buf, int32_t n);
/* which kernel forms the co-moment X^T X of the FC epilogue: "tvbx::fc_xtx_tc_kernel" (tcgen05 kind::tf32, S7') or
 * "tvbx::fc_comoment_kernel" (FP32/FP64 register tiles, S7); see tvbx_sweep_opts.fc_mode. */
int32_t tvbx_fc_kernel_name(const tvbx_sweep* sw, char* buf, int32_t n);
/* number of kernel launches enqueued by this sweep object so far */
int32_t tvbx_launch_count(const tvbx_sweep* sw, int64_t* n);
/* Test hook for the transfer function of the product kernel (tests/test_gpu_tf2.py): evaluates the packed closed form
 * tf_closed2 (csrc/tvbx_tf2.cuh; Eq. (5), Table 1) ON THE DEVICE in FP32
 * for n input points and returns, per point and population, F and its five partial derivatives with respect to
 * (f_e, f_i) -- unscaled by kappa -- and mu_V.  params: the model parameters (NULL = defaults); fe, fi [n] input rates
 * in kHz (> 0); w_e, w_i [n] adaptation currents in pA; out [n][2][7] doubles (population e then i; F, F_e, F_i, F_ee,
 * F_ei, F_ii, mu_V).  All pointers HOST.  TVBX_EINVAL if tau_e != tau_i (the closed form does not apply). */
int32_t tvbx_diag_tf_closed2(const tvbx_model_params* params, int32_t n, const double* fe, const double* fi,
                             const double* w_e, const double* w_i, double* out);

#ifdef __cplusplus
}
#endif
#endif /* TVBX_DIAG_H */
