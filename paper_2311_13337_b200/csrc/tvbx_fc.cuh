// tvbx_fc.cuh -- the epilogue kernels: per-chunk mean, centred co-moment (X^T X) merged into the
// running accumulators in Welford/Chan form (S7), and the Pearson finalisation (S8).
// DESIGN.md section 6.4; PAPER.md P:113 ("covariance of the resulting time-series for all
// concurrent simulations"), Eq. (6) P:161.
//
// The integrator leaves the kept 1-ms excitatory samples of the current chunk in
//   xbar[group][sample][region][SPC]            (R = float or double)
// For every simulation the running statistics are (cnt, mean[N], M[N][N]) in FP64:
//   M_kl = sum_q (x_qk - mean_k)(x_ql - mean_l).
// A chunk (n_c samples, chunk mean m_c, centred co-moment M_c computed in R after centring on m_c)
// is merged with Chan's pairwise update
//   delta = m_c - mean;  M += M_c + delta_k delta_l * cnt*n_c/(cnt+n_c);  mean += delta*n_c/(cnt+n_c).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace tvbx {

template <typename R>
struct FcParams {
  const R* xbar;        // [G][CS][N][SPC]
  double* cmean;        // [G][N][SPC]   chunk means (scratch)
  double* mean;         // [G][N][SPC]   running mean
  double* M;            // [G][SPC][N][N] running co-moment
  int64_t cnt;          // samples merged so far (same for all sims)
  int32_t n_c;          // samples in this chunk
  int32_t CS, N, SPC, G;
  // rate statistics of the excitatory 1-ms samples (f4; "high firing rate activity exceeding 100 Hz",
  // P:288 "maximum and variance in firing rates"): chunk maximum / count above thr (scratch) and the running ones
  float* cmax;          // [G][N][SPC]
  int32_t* ccnt;        // [G][N][SPC]
  float* rmax;          // [G][N][SPC] running maximum
  int32_t* rcnt;        // [G][N][SPC] running count of samples above thr
  float thr;            // kHz
};

// chunk mean per (group, region, sim lane): a block of 32 columns x 32 sample slices (coalesced 128-byte rows),
// the slices folded in shared memory in a fixed order (deterministic)
template <typename R>
__global__ void __launch_bounds__(1024) fc_chunk_mean_kernel(FcParams<R> P) {
  __shared__ double part[32][33];
  __shared__ float pmax[32][33];
  __shared__ int pcnt[32][33];
  const int g = blockIdx.x;                                  // (the group count may exceed the 65,535 of gridDim.y)
  const int cx = threadIdx.x & 31, sy = threadIdx.x >> 5;
  const int idx = blockIdx.y * 32 + cx;                      // region*SPC + lane
  const int row = P.N * P.SPC;
  double acc = 0.0;
  float mx = -INFINITY;
  int ct = 0;
  if (idx < row) {
    const R* x = P.xbar + (size_t)g * P.CS * row + idx;
    for (int q = sy; q < P.n_c; q += 32) {
      const R v = x[(size_t)q * row];
      acc += (double)v;
      mx = fmaxf(mx, (float)v);
      ct += (float)v > P.thr ? 1 : 0;
    }
  }
  part[sy][cx] = acc; pmax[sy][cx] = mx; pcnt[sy][cx] = ct;
  __syncthreads();
  if (sy == 0 && idx < row) {
    double tot = 0.0;
    float m = -INFINITY;
    int c = 0;
#pragma unroll
    for (int j = 0; j < 32; ++j) { tot += part[j][cx]; m = fmaxf(m, pmax[j][cx]); c += pcnt[j][cx]; }
    P.cmean[(size_t)g * row + idx] = tot / (double)P.n_c;
    P.cmax[(size_t)g * row + idx] = m;
    P.ccnt[(size_t)g * row + idx] = c;
  }
}

// centred co-moment of one (group, sim lane, 32x32 output tile), merged into M.
// 64 threads, each a 4x4 register tile; samples are staged through shared memory 32 at a time.
template <typename R>
__global__ void __launch_bounds__(64) fc_comoment_kernel(FcParams<R> P) {
  constexpr int TS = 32, QT = 32;
  __shared__ R sa[QT][TS + 1];
  __shared__ R sb[QT][TS + 1];
  const int g = blockIdx.x / P.SPC, sl = blockIdx.x % P.SPC;
  const int tk = blockIdx.z, tl = blockIdx.y;
  if (tl < tk) return;                                        // upper-triangular tiles only
  const int row = P.N * P.SPC;
  const R* x = P.xbar + (size_t)g * P.CS * row + sl;
  const double* cm = P.cmean + (size_t)g * row + sl;
  const int k0 = tk * TS, l0 = tl * TS;
  const int ty = threadIdx.x / 8, tx = threadIdx.x % 8;       // 8x8 threads, 4x4 outputs each
  R acc[4][4];
#pragma unroll
  for (int a = 0; a < 4; ++a)
#pragma unroll
    for (int b = 0; b < 4; ++b) acc[a][b] = R(0);
  for (int q0 = 0; q0 < P.n_c; q0 += QT) {
    for (int i = threadIdx.x; i < QT * TS; i += 64) {
      const int q = i / TS, c = i % TS;
      R va = R(0), vb = R(0);
      if (q0 + q < P.n_c) {
        if (k0 + c < P.N) va = (R)((double)x[((size_t)(q0 + q) * P.N + k0 + c) * P.SPC] - cm[(size_t)(k0 + c) * P.SPC]);
        if (l0 + c < P.N) vb = (R)((double)x[((size_t)(q0 + q) * P.N + l0 + c) * P.SPC] - cm[(size_t)(l0 + c) * P.SPC]);
      }
      sa[q][c] = va; sb[q][c] = vb;
    }
    __syncthreads();
#pragma unroll 4
    for (int q = 0; q < QT; ++q) {
      R a[4], b[4];
#pragma unroll
      for (int u = 0; u < 4; ++u) { a[u] = sa[q][ty * 4 + u]; b[u] = sb[q][tx * 4 + u]; }
#pragma unroll
      for (int u = 0; u < 4; ++u)
#pragma unroll
        for (int w = 0; w < 4; ++w) acc[u][w] += a[u] * b[w];
    }
    __syncthreads();
  }
  // Chan merge into the FP64 accumulators (both triangles)
  const double* mean = P.mean + (size_t)g * row + sl;
  double* M = P.M + ((size_t)g * P.SPC + sl) * P.N * P.N;
  const double f = P.cnt > 0 ? (double)P.cnt * (double)P.n_c / (double)(P.cnt + P.n_c) : 0.0;
#pragma unroll
  for (int u = 0; u < 4; ++u)
#pragma unroll
    for (int w = 0; w < 4; ++w) {
      const int k = k0 + ty * 4 + u, l = l0 + tx * 4 + w;
      if (k >= P.N || l >= P.N) continue;
      if (tk == tl && l < k) continue;
      double v = (double)acc[u][w];
      if (P.cnt > 0) {
        const double dk = cm[(size_t)k * P.SPC] - mean[(size_t)k * P.SPC];
        const double dl = cm[(size_t)l * P.SPC] - mean[(size_t)l * P.SPC];
        v += dk * dl * f;
      }
      M[(size_t)k * P.N + l] += v;
      if (k != l) M[(size_t)l * P.N + k] += v;
    }
}

// running mean update (after every tile of fc_comoment_kernel has read the old mean)
template <typename R>
__global__ void fc_mean_update_kernel(FcParams<R> P) {
  const int g = blockIdx.x;
  const int idx = blockIdx.y * blockDim.x + threadIdx.x;
  const int row = P.N * P.SPC;
  if (idx >= row) return;
  const size_t o = (size_t)g * row + idx;
  if (P.cnt == 0) { P.mean[o] = P.cmean[o]; P.rmax[o] = P.cmax[o]; P.rcnt[o] = P.ccnt[o]; }
  else {
    P.mean[o] += (P.cmean[o] - P.mean[o]) * ((double)P.n_c / (double)(P.cnt + P.n_c));
    P.rmax[o] = fmaxf(P.rmax[o], P.cmax[o]);
    P.rcnt[o] += P.ccnt[o];
  }
}

// f4, inhibitory population (optional, tvbx_sweep_opts.rate_stats_inhibitory): one pass over the chunk's inhibitory
// samples per (group, region, lane) column -- Welford per sample slice, the 32 slices merged with Chan's update in a
// fixed order -- then merged into the running (mean, M2, max, count).  st[4]: {count is P.cnt, [0] mean, [1] M2}.
template <typename R>
struct RateIParams {
  const R* xbar_i;      // [G][CS][N][SPC]
  double* mean;         // [G][N][SPC] running mean
  double* m2;           // [G][N][SPC] running sum of squared deviations
  float* rmax;          // [G][N][SPC]
  int32_t* rcnt;        // [G][N][SPC]
  int64_t cnt;          // samples merged before this chunk
  int32_t n_c, CS, N, SPC, G;
  float thr;
};
template <typename R>
__global__ void __launch_bounds__(1024) rate_i_chunk_kernel(RateIParams<R> P) {
  __shared__ double pm[32][33], p2[32][33];
  __shared__ float pmax[32][33];
  __shared__ int pcnt[32][33], pn[32][33];
  const int g = blockIdx.x;
  const int cx = threadIdx.x & 31, sy = threadIdx.x >> 5;
  const int idx = blockIdx.y * 32 + cx;
  const int row = P.N * P.SPC;
  double mean = 0.0, m2 = 0.0;
  float mx = -INFINITY;
  int ct = 0, n = 0;
  if (idx < row) {
    const R* x = P.xbar_i + (size_t)g * P.CS * row + idx;
    for (int q = sy; q < P.n_c; q += 32) {
      const double v = (double)x[(size_t)q * row];
      ++n;
      const double d = v - mean;
      mean += d / (double)n;
      m2 += d * (v - mean);
      mx = fmaxf(mx, (float)v);
      ct += (float)v > P.thr ? 1 : 0;
    }
  }
  pm[sy][cx] = mean; p2[sy][cx] = m2; pmax[sy][cx] = mx; pcnt[sy][cx] = ct; pn[sy][cx] = n;
  __syncthreads();
  if (sy == 0 && idx < row) {
    double cm = 0.0, c2 = 0.0;
    double cn = 0.0;
    float m = -INFINITY;
    int c = 0;
    for (int j = 0; j < 32; ++j) {
      const double nj = (double)pn[j][cx];
      if (nj > 0.0) {
        const double d = pm[j][cx] - cm, tot = cn + nj;
        c2 += p2[j][cx] + d * d * (cn * nj / tot);
        cm += d * (nj / tot);
        cn = tot;
      }
      m = fmaxf(m, pmax[j][cx]); c += pcnt[j][cx];
    }
    const size_t o = (size_t)g * row + idx;
    if (P.cnt == 0) { P.mean[o] = cm; P.m2[o] = c2; P.rmax[o] = m; P.rcnt[o] = c; }
    else {
      const double a = (double)P.cnt, tot = a + cn, d = cm - P.mean[o];
      P.m2[o] += c2 + d * d * (a * cn / tot);
      P.mean[o] += d * (cn / tot);
      P.rmax[o] = fmaxf(P.rmax[o], m);
      P.rcnt[o] += c;
    }
  }
}

// f4 readout: per (simulation, region) variance (M_kk / n, the population variance of the kept 1-ms samples), maximum
// and number of samples above the threshold, in local-simulation order
struct RateStatsParams {
  const double* M;       // [G][SPC][N][N]
  const float* rmax;     // [G][N][SPC]
  const int32_t* rcnt;   // [G][N][SPC]
  const int32_t* loc_id; // [G][SPC]
  float* var_e;          // [n_sims][N] or null
  float* max_e;          // [n_sims][N] or null
  int32_t* above;        // [n_sims][N] or null
  const double* m2_i;    // inhibitory running statistics [G][N][SPC], or null
  const float* rmax_i;
  const int32_t* rcnt_i;
  float* var_i;          // [n_sims][N] or null
  float* max_i;
  int32_t* above_i;
  int64_t cnt;
  int32_t N, SPC, G;
};
__global__ void rate_stats_kernel(RateStatsParams P) {
  const int g = blockIdx.x / P.SPC, sl = blockIdx.x % P.SPC;
  const int loc = P.loc_id[(size_t)g * P.SPC + sl];
  if (loc < 0) return;
  const int k = blockIdx.y * blockDim.x + threadIdx.x;
  if (k >= P.N) return;
  const size_t o = ((size_t)g * P.N + k) * P.SPC + sl;
  if (P.var_e) P.var_e[(size_t)loc * P.N + k] = (float)(P.M[((size_t)g * P.SPC + sl) * P.N * P.N + (size_t)k * P.N + k] / (double)P.cnt);
  if (P.max_e) P.max_e[(size_t)loc * P.N + k] = P.rmax[o];
  if (P.above) P.above[(size_t)loc * P.N + k] = P.rcnt[o];
  if (P.m2_i) {
    if (P.var_i) P.var_i[(size_t)loc * P.N + k] = (float)(P.m2_i[o] / (double)P.cnt);
    if (P.max_i) P.max_i[(size_t)loc * P.N + k] = P.rmax_i[o];
    if (P.above_i) P.above_i[(size_t)loc * P.N + k] = P.rcnt_i[o];
  }
}

struct ReadoutParams {
  const double* M;       // [G][SPC][N][N]
  const double* sums;    // [G][2][N][SPC]
  const int32_t* loc_id; // [G][SPC]
  float* fc;             // [n_sims][N][N] or null
  float* mean_e;         // [n_sims][N] or null
  float* mean_i;
  int64_t cnt;
  int32_t N, SPC, G;
  int32_t diag_in_smem;  // the launch carries N doubles of dynamic shared memory
};

// Pearson finalise (Eq. 6; A18) in local-simulation order.  grid (G * SPC, ceil(N / RO_ROWS)), 256 threads: a
// block stages the simulation's N variances in shared memory (the strided M_ll lookups stay on chip) and writes RO_ROWS
// rows of the matrix; block row 0 also writes the mean rates.
constexpr int RO_ROWS = 8;
__global__ void __launch_bounds__(256) fc_readout_kernel(ReadoutParams P) {
  extern __shared__ double rdiag[];
  const int g = blockIdx.x / P.SPC, sl = blockIdx.x % P.SPC;
  const int loc = P.loc_id[(size_t)g * P.SPC + sl];
  if (loc < 0) return;
  const int N = P.N;
  const double* M = P.M + ((size_t)g * P.SPC + sl) * N * N;
  const bool staged = P.diag_in_smem != 0;
  if (P.fc && staged) {
    for (int k = threadIdx.x; k < N; k += 256) rdiag[k] = M[(size_t)k * N + k];
    __syncthreads();
  }
  const int k0 = blockIdx.y * RO_ROWS;
  const int nrow = min(RO_ROWS, N - k0);
  if (P.fc) {
    for (int i = threadIdx.x; i < nrow * N; i += 256) {
      const int k = k0 + i / N, l = i % N;
      float r;
      if (k == l) r = 1.0f;
      else {
        const double den = staged ? rdiag[k] * rdiag[l] : M[(size_t)k * N + k] * M[(size_t)l * N + l];
        double v = (den > 0.0 && isfinite(den)) ? M[(size_t)k * N + l] / sqrt(den) : 0.0;
        r = isfinite(v) ? (float)fmin(1.0, fmax(-1.0, v)) : 0.0f;   // |rho| <= 1 (Cauchy-Schwarz); FP32 chunk co-moments can round past it
      }
      P.fc[(size_t)loc * N * N + (size_t)k * N + l] = r;
    }
  }
  if (blockIdx.y == 0) {
    const size_t row = (size_t)N * P.SPC;
    for (int k = threadIdx.x; k < N; k += 256) {
      const double* s = P.sums + (size_t)g * 2 * row + (size_t)k * P.SPC + sl;
      if (P.mean_e) P.mean_e[(size_t)loc * N + k] = (float)(s[0] / (double)P.cnt);
      if (P.mean_i) P.mean_i[(size_t)loc * N + k] = (float)(s[row] / (double)P.cnt);
    }
  }
}

// ---- FC scores ("FCSC, the correlation with the structure connectivity
// (SC) ... determined with the Pearson correlation", "comparison to an externally obtained reference FC matrix by
// correlating it to the computed FC", fitness P:159 with Eq. (6), mean_FC Tab. 2) ----
// Per simulation, over the N(N-1)/2 region pairs k < l (reading A23: both matrices are symmetric, the diagonal is
// trivial: FC_kk = 1, W_kk = 0):  fcsc = Pearson(FC_kl, SC_kl), fitness = Pearson(FC_kl, REF_kl),
// mean_fc = mean(FC_kl).  FC_kl is formed in FP64 from the co-moments exactly as fc_readout_kernel does (before the
// rounding to float); sums in FP64, folded in a fixed order (deterministic).  Zero variance -> 0 (A18).
struct ScoreParams {
  const double* M;       // [G][SPC][N][N]
  const double* sc;      // [N][N] structural connectivity (the connectome weights), device
  const double* ref;     // [N][N] reference FC, device, or null
  const int32_t* loc_id; // [G][SPC]
  float* fcsc;           // [n_sims] or null
  float* fitness;        // [n_sims] or null
  float* mean_fc;        // [n_sims] or null
  int32_t N, SPC, G;
  int32_t diag_in_smem;  // the launch carries N doubles of dynamic shared memory
};

// one CTA of 256 threads per (group, lane); sums: x, xx, a, aa, xa, b, bb, xb  (x = FC, a = SC, b = REF)
__global__ void __launch_bounds__(256) fc_scores_kernel(ScoreParams P) {
  __shared__ double part[8][256];
  const int g = blockIdx.x / P.SPC, sl = blockIdx.x % P.SPC;
  const int loc = P.loc_id[(size_t)g * P.SPC + sl];
  if (loc < 0) return;
  const int N = P.N;
  const double* M = P.M + ((size_t)g * P.SPC + sl) * N * N;
  // the diagonal (variances) staged in shared memory when it fits: the strided M_ll lookups stay on chip
  extern __shared__ double diag[];
  const bool staged = P.diag_in_smem != 0;
  if (staged) {
    for (int k = threadIdx.x; k < N; k += 256) diag[k] = M[(size_t)k * N + k];
    __syncthreads();
  }
  double acc[8] = {0, 0, 0, 0, 0, 0, 0, 0};
  for (int i = threadIdx.x; i < N * N; i += 256) {
    const int k = i / N, l = i % N;
    if (l <= k) continue;
    const double den = staged ? diag[k] * diag[l] : M[(size_t)k * N + k] * M[(size_t)l * N + l];
    double x = (den > 0.0 && isfinite(den)) ? M[i] / sqrt(den) : 0.0;
    x = isfinite(x) ? fmin(1.0, fmax(-1.0, x)) : 0.0;
    const double a = P.sc[i], b = P.ref ? P.ref[i] : 0.0;
    acc[0] += x; acc[1] += x * x; acc[2] += a; acc[3] += a * a; acc[4] += x * a; acc[5] += b; acc[6] += b * b; acc[7] += x * b;
  }
#pragma unroll
  for (int q = 0; q < 8; ++q) part[q][threadIdx.x] = acc[q];
  __syncthreads();
  for (int w = 128; w > 0; w >>= 1) {
    if (threadIdx.x < w)
#pragma unroll
      for (int q = 0; q < 8; ++q) part[q][threadIdx.x] += part[q][threadIdx.x + w];
    __syncthreads();
  }
  if (threadIdx.x == 0) {
    const double n = 0.5 * (double)N * (double)(N - 1);
    const double sx = part[0][0], vx = part[1][0] - sx * sx / n;
    auto pearson = [&](double sy, double syy, double sxy) {
      const double vy = syy - sy * sy / n, c = sxy - sx * sy / n, den = vx * vy;
      const double r = (n > 1.0 && den > 0.0 && isfinite(den)) ? c / sqrt(den) : 0.0;
      return (float)fmin(1.0, fmax(-1.0, r));
    };
    if (P.fcsc) P.fcsc[loc] = pearson(part[2][0], part[3][0], part[4][0]);
    if (P.fitness) P.fitness[loc] = P.ref ? pearson(part[5][0], part[6][0], part[7][0]) : 0.0f;
    if (P.mean_fc) P.mean_fc[loc] = n > 0.0 ? (float)(sx / n) : 0.0f;
  }
}


// ---- up / down-state durations (f4; Tab. 2 P:131 `mean_UD_duration`; A25) ----
// Per (group, region, lane) column the kept excitatory 1-ms samples are binarised (UP iff x > thr) and scanned in
// time order; an episode = a maximal run of equal states, counted when it ENDS and only if it did not start at the
// first kept sample (episodes cut by either end of the record have no known duration; the run still open at
// readout is simply never counted).  State per column, 6 ints: [0] prev state (-1 none yet, 0 down, 1 up),
// [1] length of the current run, [2] 1 while the current run is the record's first, [3] UP episodes,
// [4] samples in UP episodes, [5] DOWN episodes, [6] samples in DOWN episodes.
enum { UD_NSTATE = 7 };
template <typename R>
struct UpDownParams {
  const R* xbar;        // [G][CS][N][SPC]
  int32_t* st;          // [UD_NSTATE][G][N][SPC]
  int32_t n_c, CS, N, SPC, G;
  float thr;            // kHz
};
// one thread per column, the chunk's samples in order (coalesced across columns)
template <typename R>
__global__ void __launch_bounds__(128) updown_chunk_kernel(UpDownParams<R> P) {
  const int g = blockIdx.x;
  const int idx = blockIdx.y * blockDim.x + threadIdx.x;
  const int row = P.N * P.SPC;
  if (idx >= row) return;
  const size_t plane = (size_t)P.G * row, o = (size_t)g * row + idx;
  int prev = P.st[o], run = P.st[plane + o], first = P.st[2 * plane + o];
  int cnt[2] = {P.st[5 * plane + o], P.st[3 * plane + o]}, tot[2] = {P.st[6 * plane + o], P.st[4 * plane + o]};
  const R* x = P.xbar + (size_t)g * P.CS * row + idx;
  for (int q = 0; q < P.n_c; ++q) {
    const int s = (float)x[(size_t)q * row] > P.thr ? 1 : 0;
    if (prev < 0) { prev = s; run = 1; first = 1; }
    else if (s == prev) ++run;
    else {
      if (!first) { cnt[prev] += 1; tot[prev] += run; }
      prev = s; run = 1; first = 0;
    }
  }
  P.st[o] = prev; P.st[plane + o] = run; P.st[2 * plane + o] = first;
  P.st[3 * plane + o] = cnt[1]; P.st[4 * plane + o] = tot[1]; P.st[5 * plane + o] = cnt[0]; P.st[6 * plane + o] = tot[0];
}
struct UpDownReadParams {
  const int32_t* st;     // [UD_NSTATE][G][N][SPC]
  const int32_t* loc_id; // [G][SPC]
  int32_t* n_up;         // [n_sims][N] or null
  float* mean_up_ms;
  int32_t* n_down;
  float* mean_down_ms;
  float sample_ms;       // ds * dt
  int32_t N, SPC, G;
};
__global__ void updown_read_kernel(UpDownReadParams P) {
  const int g = blockIdx.x / P.SPC, sl = blockIdx.x % P.SPC;
  const int loc = P.loc_id[(size_t)g * P.SPC + sl];
  if (loc < 0) return;
  const int k = blockIdx.y * blockDim.x + threadIdx.x;
  if (k >= P.N) return;
  const size_t plane = (size_t)P.G * P.N * P.SPC, o = ((size_t)g * P.N + k) * P.SPC + sl;
  const int cu = P.st[3 * plane + o], tu = P.st[4 * plane + o], cd = P.st[5 * plane + o], td = P.st[6 * plane + o];
  const size_t w = (size_t)loc * P.N + k;
  if (P.n_up) P.n_up[w] = cu;
  if (P.n_down) P.n_down[w] = cd;
  if (P.mean_up_ms) P.mean_up_ms[w] = cu > 0 ? (float)((double)tu * (double)P.sample_ms / (double)cu) : 0.0f;
  if (P.mean_down_ms) P.mean_down_ms[w] = cd > 0 ? (float)((double)td * (double)P.sample_ms / (double)cd) : 0.0f;
}

// ---- top-k of a per-simulation score (f3; "output the best ten fittest simulations"; A23b) ----
// One CTA of 1024 threads: k rounds of a block-wide arg-max over the S scores (local simulation order), equal scores
// to the lower index; a taken entry is marked in `taken` (S bytes, zeroed by the caller).  k and S are small.
__global__ void __launch_bounds__(1024) topk_kernel(const float* __restrict__ score, unsigned char* __restrict__ taken, int S, int k,
                                                    int32_t* __restrict__ out_idx, float* __restrict__ out_val) {
  __shared__ float sv[1024];
  __shared__ int si[1024];
  for (int r = 0; r < k && r < S; ++r) {
    float bv = -INFINITY; int bi = -1;
    for (int i = threadIdx.x; i < S; i += 1024)
      if (!taken[i] && (bi < 0 || score[i] > bv)) { bv = score[i]; bi = i; }      // ascending i: the first maximum wins
    sv[threadIdx.x] = bv; si[threadIdx.x] = bi;
    __syncthreads();
    for (int w = 512; w > 0; w >>= 1) {
      if (threadIdx.x < w) {
        const float ov = sv[threadIdx.x + w]; const int oi = si[threadIdx.x + w];
        const int mi = si[threadIdx.x];
        if (oi >= 0 && (mi < 0 || ov > sv[threadIdx.x] || (ov == sv[threadIdx.x] && oi < mi))) { sv[threadIdx.x] = ov; si[threadIdx.x] = oi; }
      }
      __syncthreads();
    }
    if (threadIdx.x == 0) { out_idx[r] = si[0]; out_val[r] = sv[0]; taken[si[0]] = 1; }
    __syncthreads();
  }
}

}  // namespace tvbx
