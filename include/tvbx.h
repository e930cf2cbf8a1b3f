/* tvbx.h -- C ABI of the B200-native batched TVB-AdEx parameter-sweep integrator.
 *
 * What is computed is defined in DESIGN.md section 2 ("the frozen definition"), which restates
 * PAPER.md (arxiv 2311.13337) Eqs. (1)-(5), Table 1 and sections 2.2-2.4; "P:NN" below is a line of
 * /root/reference/PAPER.md and "A<n>" a reading listed in DESIGN.md section 3.
 *
 * Conventions
 *  - plain C, every call returns an int32 status (0 = TVBX_OK, < 0 = error); nothing throws across
 *    the boundary; tvbx_last_error() returns a thread-local message for the last failing call.
 *  - input arrays are HOST pointers unless stated, are copied, and stay owned by the caller.
 *  - output buffers are caller-allocated; a flag says whether the pointer is host or device memory
 *    (device = on the CUDA device that was current when the sweep was created).
 *  - objects behind handles are owned by the library until the matching *_destroy.
 *  - units: ms, kHz, mV, pA, nS, pF (0.001 kHz = 1 Hz).
 *  - all work of tvbx_run / tvbx_fc_readout is enqueued on the CUDA stream passed in (NULL = the
 *    legacy default stream).  Calls that fill HOST buffers synchronise that stream before returning;
 *    calls that fill DEVICE buffers return without synchronising.
 *  - there is no CPU fallback: without a CUDA device every compute entry point fails with TVBX_ECUDA.
 */
#ifndef TVBX_H
#define TVBX_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define TVBX_VERSION 200 /* 0.2.0: diagnostics moved to tvbx_diag.h; latency_form, tvbx_top_k */

enum tvbx_status {
  TVBX_OK = 0,
  TVBX_EINVAL = -1, /* bad argument (message says which) */
  TVBX_ENOMEM = -2, /* host or device allocation failed (e.g. the history ring does not fit) */
  TVBX_ECUDA = -3,  /* CUDA runtime error, or no device */
  TVBX_ESTATE = -4  /* call not valid in the object's current state */
};

/* Model parameters (DESIGN.md section 3 table).  Index into tvbx_model_params.p. */
enum tvbx_param_id {
  TVBX_P_G = 0,      /* global coupling g of nu_e^{k,tot} */
  TVBX_P_B_E,        /* spike-frequency adaptation b_e [pA] (Eq. 3) */
  TVBX_P_A_E,        /* sub-threshold adaptation a_e [nS] */
  TVBX_P_TAU_W_E,    /* adaptation time constant tau_w,e [ms] */
  TVBX_P_V,          /* conduction speed [m/s] = [mm/ms]; delays = length / speed */
  TVBX_P_WNOISE,     /* wNoise of Eq. (5) */
  TVBX_P_EL_E,       /* leak reversal E_L,e [mV] */
  TVBX_P_EL_I,       /* E_L,i [mV] */
  TVBX_P_T,          /* time constant T of Eqs. (1)-(2) [ms] */
  TVBX_P_CFEE,       /* c_{F e,e}: constant excitatory input to the excitatory population [kHz] */
  TVBX_P_CFEI,       /* c_{F e,i}: constant inhibitory input to the excitatory population */
  TVBX_P_CFIE,       /* c_{F i,e} */
  TVBX_P_CFII,       /* c_{F i,i} */
  /* ---- the ids above may be swept with tvbx_axis; the ids below are uniform over a sweep ---- */
  TVBX_P_B_I, TVBX_P_A_I, TVBX_P_TAU_W_I,
  TVBX_P_GL, TVBX_P_CM,
  TVBX_P_QE, TVBX_P_TAUE, TVBX_P_EE,
  TVBX_P_QI, TVBX_P_TAUI, TVBX_P_EI,
  TVBX_P_NTOT, TVBX_P_PCONN, TVBX_P_GINH,
  TVBX_P_TAU_OU, TVBX_P_MU_OU, TVBX_P_SIGMA_OU, /* Eq. (4) */
  TVBX_P_MUV0, TVBX_P_DMUV0, TVBX_P_SV0, TVBX_P_DSV0, TVBX_P_TVN0, TVBX_P_DTVN0, /* A2 */
  TVBX_P_EPS_NU,     /* input floor (A10) [kHz] */
  TVBX_P_MUV_LOCAL,  /* != 0: mu_V of Eq. (3) from the local rates only (A9b alternative) */
  TVBX_P_KAPPA,      /* unit of the differentiated rate in dF/dnu relative to kHz (A22) */
  TVBX_P_POLY_E,     /* 10 coefficients: Table 1 RS row, order P0,mu,sigma,tau,mu2,sigma2,tau2,mu.sigma,mu.tau,sigma.tau */
  TVBX_P_POLY_I = TVBX_P_POLY_E + 10, /* 10 coefficients: Table 1 FS row */
  TVBX_N_PARAMS = TVBX_P_POLY_I + 10
};
#define TVBX_N_SWEEPABLE 13 /* ids 0 .. TVBX_P_CFII */

typedef struct tvbx_model_params { double p[TVBX_N_PARAMS]; } tvbx_model_params;

/* One axis of the parameter grid ("-s0 6 generates six values equally spaced within the
 * defined range").  values == NULL: value_i = lo + i*((hi-lo)/(n-1)) in FP64, last value forced to
 * hi, n == 1 -> lo (bit-identical to numpy.linspace).  values != NULL: n explicit values. */
typedef struct tvbx_axis {
  int32_t param_id; /* < TVBX_N_SWEEPABLE */
  int32_t n;        /* >= 1 */
  double lo, hi;
  const double* values; /* host, n doubles, or NULL */
} tvbx_axis;

enum tvbx_precision { TVBX_F32 = 0, TVBX_F64 = 1 };

typedef struct tvbx_sweep_opts {
  int32_t precision;      /* TVBX_F32 (default) or TVBX_F64 (the 1e-9 parity build mode) */
  int32_t sims_per_cta;   /* 0 = choose; else 1..32: simulations integrated by one CTA (they share a delay table);
                             more than 8, or N * sims_per_cta > 480, selects the general kernel */
  int64_t n_sims;         /* 0 = the whole grid; else number of entries of sim_ids */
  const int64_t* sim_ids; /* host: external (grid) indices of the simulations this sweep object holds,
                             e.g. one rank's shard; results are returned in this order */
  int64_t chunk_samples;  /* 0 = choose; downsampled samples buffered between FC reductions */
  int32_t threads_per_cta;/* 0 = choose; a value below the lanes one pass over the regions needs selects the general
                             kernel with several region passes per time block */
  int32_t ctas_per_group; /* 0 = choose; else 1..8: CTAs (one thread-block cluster) that share the regions of a group of
                             sims_per_cta simulations -- lets N = 360 run 8 simulations per group (6 CTAs x 60 regions);
                             packed FP32 kernel only */
  int32_t fc_mode;        /* co-moment X^T X of the FC epilogue (S7 / S7'): TVBX_FC_AUTO = tensor cores
                             (tcgen05 kind::tf32, samples centred in FP32 before rounding to TF32, FP32 accumulate,
                             FP64 merge) for FP32 sweeps with N <= 512, else FP32/FP64 register tiles;
                             TVBX_FC_FP32 = register tiles always; TVBX_FC_TF32 = tensor cores or TVBX_EINVAL */
  int32_t rate_stats_inhibitory; /* 1: also keep the inhibitory 1-ms samples of the chunk (as much memory again as the
                                    sample chunk) so that tvbx_rate_stats can return var_i, max_i, n_above_i.  Selects
                                    the general integrator ("tvbx::integrate_kernel", about 0.65 x the throughput of
                                    the packed one, which is kept free of the extra store) */
  double rate_threshold_khz; /* tvbx_rate_stats counts the 1-ms excitatory samples above this rate; 0 = 0.1 kHz
                                ("high firing rate activity exceeding 100 Hz") */
  int32_t latency_form;   /* 0 = choose; 1 = off; 2 = on (TVBX_EINVAL where it does not apply).  The LOW-LATENCY form of the packed
                             kernel for small sweeps / long runs ("a lesser thread count per GPU to
                             hide latency"): when the sweep offers about one warp of nodes per warp scheduler, throughput is the
                             latency of one warp's step; a producer warp per consumer warp then takes the delayed gather, the
                             Philox draws and their bookkeeping off that chain and runs on the schedulers' idle issue slots
                             (csrc/tvbx_integrate2_ws.cuh).  Same arithmetic and Philox stream: results are bit-identical.
                             Applies to one-CTA groups of <= 160 nodes with 8-step chunks (minimum delay >= 15 steps).
                             3 = on, GROUPED: the regions of a group of simulations are split over ctas_per_group CTAs on
                             different SMs (cooperative launch, chunk hand-over through counters in global memory), so that
                             every warp scheduler hosts at most ONE consumer warp -- chosen by 0 when the one-CTA mapping would
                             put two on one scheduler and the whole grid fits the GPU at once (cfg 4: 7 simulations per 4
                             CTAs).  With 3, sims_per_cta / ctas_per_group = 0 are chosen by the library */
  int32_t reserved0;
  double updown_threshold_khz; /* > 0: also keep the up / down-state episode statistics of the kept 1-ms excitatory samples
                                  (tvbx_state_durations; Tab. 2 P:131 `mean_UD_duration`): a sample is UP iff it exceeds
                                  this rate.  0 = off (the paper prints no threshold: DESIGN.md A25) */
} tvbx_sweep_opts;

enum tvbx_fc_mode { TVBX_FC_AUTO = 0, TVBX_FC_FP32 = 1, TVBX_FC_TF32 = 2 };

typedef struct tvbx_run_opts {
  int32_t noise_on;       /* 0: deterministic, OU neither used nor advanced; 1: Philox OU noise (A11, A12) */
  int32_t ds;             /* temporal-average window in steps; 0 = no downsampling / FC */
  int64_t discard_steps;  /* windows ending at a step <= discard_steps are dropped (A17) */
  void* traj;             /* optional: post-update state of the first traj_steps steps of THIS call,
                             layout [n_sims][traj_steps][7][N], float (F32 sweeps) or double (F64) */
  int64_t traj_steps;
  int32_t traj_on_device; /* 1: traj is a device pointer */
  int32_t reserved;
  void* cuda_stream;      /* cudaStream_t or NULL */
} tvbx_run_opts;

typedef struct tvbx_connectome tvbx_connectome;
typedef struct tvbx_sweep tvbx_sweep;

/* Library defaults of every model parameter (DESIGN.md section 3 table). */
int32_t tvbx_default_params(tvbx_model_params* out);

/* Connectome: W, L_mm row-major n x n, W[k*n+j] = weight u_kj of SOURCE j into TARGET k,
 * L_mm[k*n+j] = tract length in mm.  Rejects n < 1, non-finite or negative entries.  Zero weights
 * are dropped; the kept edges of a row are stored in ascending j (the FP64 summation order, A16). */
int32_t tvbx_create_connectome(int32_t n, const double* W, const double* L_mm, tvbx_connectome** out);
int32_t tvbx_destroy_connectome(tvbx_connectome* c);

/* Parameter sweep: S = prod n_i simulations, sim index in C order over the axes, FIRST
 * AXIS SLOWEST (A19).  Every simulation starts from E = I = 0.001 kHz, all else 0 (override with
 * tvbx_sweep_set_initial), OU = 0, constant initial history (A14), step counter 0.  seed keys the
 * Philox4x32-10 noise streams (A12).  opts may be NULL.  Device memory is allocated at the first
 * tvbx_run (the ring depth needs dt). */
int32_t tvbx_sweep_create(const tvbx_connectome* c, const tvbx_model_params* defaults, int32_t n_axes,
                          const tvbx_axis* axes, uint64_t seed, const tvbx_sweep_opts* opts,
                          tvbx_sweep** out);
int32_t tvbx_sweep_destroy(tvbx_sweep* sw);

/* Initial state E, I, C_ee, C_ei, C_ii, W_e, W_i (the seven variables of Eqs. (1)-(3)) of every region of
 * every simulation; the history is filled with init[0] (PAPER.md gives no initial condition: readings A11, A14;
 * BASELINE.json cfg 1 states E = I = 0.001 kHz, the rest 0).  TVBX_ESTATE after the first tvbx_run. */
int32_t tvbx_sweep_set_initial(tvbx_sweep* sw, const double init[7]);

/* Advance every simulation `steps` forward-Euler steps of dt ms: per step the delayed
 * coupling sum, both transfer functions with first and second derivatives (Eq. 5, Table 1),
 * Eqs. (1)-(3), the OU update (Eq. 4), the history write, the temporal-average downsample
 * and the mean / co-moment accumulation for the FC.  Resumable:
 * run(a); run(b) is bit-identical to run(a+b).  dt must equal the dt of the first call
 * (TVBX_EINVAL otherwise); noise_on, ds and discard_steps are expected to stay the same. */
int32_t tvbx_run(tvbx_sweep* sw, int64_t steps, double dt, const tvbx_run_opts* opts);

/* Pearson FC of the kept excitatory samples (Eq. 6) and the per-region means, without
 * consuming the accumulators.  fc [n_sims][N][N], mean_e / mean_i [n_sims][N], FP32, in the order of
 * sim_ids (grid order by default); any pointer may be NULL.  Degenerate variance -> 0 off the
 * diagonal, 1 on it (A18).  TVBX_ESTATE if fewer than 2 samples were kept. */
int32_t tvbx_fc_readout(tvbx_sweep* sw, float* fc, float* mean_e, float* mean_i, int32_t on_device,
                        void* cuda_stream);

/* FC scores per simulation (Eq. (6), Tab. 2; A23), over the
 * N(N-1)/2 region pairs k < l of the Pearson matrix tvbx_fc_readout would return (formed in FP64 from the
 * accumulators, open chunk included, accumulators untouched):
 *   fcsc[s]    = Pearson(FC_kl, W_kl)      structure-function correlation with the connectome weights (SC)
 *   fitness[s] = Pearson(FC_kl, ref_kl)    against an externally obtained reference FC; ref_fc = HOST, row-major
 *                                          N x N doubles (only k < l is read), copied before the call returns
 *   mean_fc[s] = mean(FC_kl)
 * Any output may be NULL; outputs are n_sims floats in this sweep's simulation order, host or device
 * (on_device).  Zero variance gives 0.  TVBX_ESTATE with fewer than 2 kept samples, TVBX_EINVAL if fitness is
 * asked for without ref_fc or ref_fc holds a non-finite value. */
int32_t tvbx_fc_scores(tvbx_sweep* sw, const double* ref_fc, float* fcsc, float* fitness, float* mean_fc,
                       int32_t on_device, void* stream);

/* Rate statistics per (simulation, region) over the kept 1-ms samples (the series the FC is computed from; PAPER.md
 * P:288 "the maximum and variance in firing rates for both excitatory and inhibitory populations", P:235 / P:282
 * activity "exceeding 100 Hz" as the mark of the paroxysmal fixed point; A24), for the excitatory (_e) and,
 * if the sweep was created with rate_stats_inhibitory, the inhibitory (_i) population:
 *   var[s][k]     = population variance (1/n) sum (x - mean)^2   [kHz^2]
 *   max[s][k]     = maximum                                      [kHz]
 *   n_above[s][k] = number of samples > rate_threshold_khz (a region "visits" the paroxysmal state iff > 0)
 * Outputs n_sims x N, host or device (on_device), any may be NULL; the open chunk is included and the
 * accumulators stay untouched.  TVBX_ESTATE before the first kept sample; TVBX_EINVAL if an _i output is asked for
 * without rate_stats_inhibitory. */
int32_t tvbx_rate_stats(tvbx_sweep* sw, float* var_e, float* max_e, int32_t* n_above_e, float* var_i, float* max_i,
                        int32_t* n_above_i, int32_t on_device, void* stream);

/* Up / down-state durations per (simulation, region) (Tab. 2 P:131 `mean_UD_duration` "Mean duration of UP and
 * DOWN states"; A25), over the kept 1-ms excitatory samples: a sample is UP iff it exceeds
 * tvbx_sweep_opts.updown_threshold_khz; an episode is a maximal run of equal states; episodes cut by the start of the
 * record or still open now are not counted.  n_up / n_down = number of episodes, mean_*_ms = their mean duration in ms
 * (0 where there is none).  Outputs n_sims x N, host or device (on_device), any may be NULL; the open chunk is included,
 * the accumulators stay untouched.  TVBX_ESTATE if the sweep was created without a threshold or before the first run. */
int32_t tvbx_state_durations(tvbx_sweep* sw, int32_t* n_up, float* mean_up_ms, int32_t* n_down, float* mean_down_ms,
                             int32_t on_device, void* stream);

/* The k best simulations by an FC score (the grid search "output[s] the best ten fittest simulations";
 * scores as in tvbx_fc_scores, Eq. (6)): which = 0 fcsc, 1 fitness (needs ref_fc), 2 mean_fc.  sim_ids[i] = external
 * (grid) index of the i-th best simulation of this sweep object, scores[i] its score, best first, equal scores in ascending
 * local order (A23); both HOST arrays of k entries; *n_out = min(k, n_sims).  1 <= k <= 1024. */
int32_t tvbx_top_k(tvbx_sweep* sw, int32_t which, const double* ref_fc, int32_t k, int64_t* sim_ids, float* scores,
                   int32_t* n_out, void* stream);

/* Back to step 0 without re-allocating: state, OU, history ring, window sums and FC accumulators are
 * re-initialised on the device (enqueued on cuda_stream), the step and sample counters are zeroed.
 * A no-op before the first tvbx_run.  reset; run(n) is bit-identical to a fresh sweep's run(n). */
int32_t tvbx_sweep_reset(tvbx_sweep* sw, void* cuda_stream);

/* ---- bookkeeping accessors (the bit-exact part of the definition: parameter grid P:100 / A19, delays P:82 / A13,
 * ring depth P:113 "-cs ... determines the depth of the temporal buffer") -------------------------------------- */
/* number of simulations this object holds, size of the whole Cartesian grid, regions of the connectome */
int32_t tvbx_sweep_size(const tvbx_sweep* sw, int64_t* n_sims, int64_t* grid_size, int32_t* n_regions);
/* parameter value of local simulation `sim` (index into sim_ids): the value its grid digit selects on the axis that
 * sweeps param_id (A19: closed interval, equally spaced, first axis slowest), else the sweep's default */
int32_t tvbx_sweep_param(const tvbx_sweep* sw, int64_t sim, int32_t param_id, double* out);
/* external (grid) index of local simulation `sim`: the work-item number of P:100, also the Philox stream id (A12) */
int32_t tvbx_sweep_ext_id(const tvbx_sweep* sw, int64_t sim, int64_t* out);
/* d_kj = nearbyint((L_kj / v) / dt) in FP64, round-half-to-even (A13); -1 if W_kj == 0.
 * Valid after the first tvbx_run (needs dt), or pass dt > 0 explicitly. */
int32_t tvbx_delay_index(const tvbx_sweep* sw, int64_t sim, int32_t k, int32_t j, double dt, int32_t* out);
/* logical ring length H = D + 1 and the physical one the kernel uses: H plus the steps the fastest warp of a
 * CTA may be ahead of the slowest (at most the minimum delay + 1). */
int32_t tvbx_ring_len(const tvbx_sweep* sw, int64_t sim, double dt, int32_t* H, int32_t* H_phys);
/* Euler steps taken so far and temporal-average samples kept so far (A17: windows ending at a
 * step <= discard_steps are dropped) */
int32_t tvbx_steps_done(const tvbx_sweep* sw, int64_t* n);
int32_t tvbx_samples_kept(const tvbx_sweep* sw, int64_t* n);
/* current state, [n_sims][7][N] + OU [n_sims][N], as double, to HOST buffers (synchronises) */
int32_t tvbx_sweep_state(tvbx_sweep* sw, double* y, double* ou);
const char* tvbx_last_error(void);
int32_t tvbx_version(void);
/* Device buffers of destroyed sweeps are cached inside the library (per device, exact size; capacity
 * TVBX_POOL_BYTES, default a quarter of the device memory, 0 disables) and reused by the next sweep of the same
 * shape, so create / run / destroy cycles do not pay cudaMalloc / cudaFree each time.  This call returns every
 * cached buffer to the driver; *bytes_freed (may be NULL) receives the amount. */
int32_t tvbx_trim_memory(int64_t* bytes_freed);

#ifdef __cplusplus
}
#endif
#endif /* TVBX_H */
