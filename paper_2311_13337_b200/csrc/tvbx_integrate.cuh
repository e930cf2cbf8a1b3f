// tvbx_integrate.cuh -- the GENERAL integrator kernel (FP64 build mode, tau_e != tau_i, CTAs that need
// several region passes); the FP32 product path is tvbx_integrate2.cuh.  Delayed gather + coupling sum (S1), both transfer
// functions with derivatives (S2), Euler update of the 7 state variables (S3), OU noise from
// in-kernel Philox4x32-10 (S4), history-ring write (S5), temporal-average downsample (S6) and the
// per-thread running sums for the mean rates.  DESIGN.md section 6 describes the mapping.
//
// Mapping (B200-first, not the paper's thread-per-simulation kernel):
//   CTA      = one "group" of SPC simulations that share a delay table (same speed v), all N regions
//   lane pair= one (simulation, region); the EVEN lane integrates the excitatory population
//              (E, C_ee, W_e), the ODD lane the inhibitory one (I, C_ii, W_i).  Both run the same
//              transfer-function code on different constants (no divergence) and exchange E/I, C,
//              (F - nu) and the C_ei half-sums with five warp shuffles per step.
//   ring     = ring[group][region][slot][sim]  (E only, "temporal buffer"): the SPC simulations
//              of a group are the fastest index, so the lanes that share a region read one contiguous
//              run per (edge, step).  Rows carry GC-1 mirror slots so that a chunk of GC reads never wraps.
//   time     = the kernel is persistent over time: it runs B <= min delay steps between CTA
//              barriers (step n only reads E at times <= n - d_min), and inside a block it
//              alternates a GATHER phase (coupling sums of the next <= GC steps, pure loads + FMAs,
//              the edge list split between the two lanes of a pair) with a COMPUTE phase (<= GC
//              steps of pure register arithmetic).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include "tvbx_tf.cuh"

namespace tvbx {

enum { GC = 8 };        // steps per gather chunk (and mirror slots + 1)

// ---- Philox4x32-10 (A12) -------------------------------------------------------------------------
__device__ __forceinline__ void philox4x32_10(uint32_t c0, uint32_t c1, uint32_t c2, uint32_t c3,
                                              uint32_t k0, uint32_t k1, uint32_t out[4]) {
#pragma unroll
  for (int r = 0; r < 10; ++r) {
    const uint32_t hi0 = __umulhi(0xD2511F53u, c0), lo0 = 0xD2511F53u * c0;
    const uint32_t hi1 = __umulhi(0xCD9E8D57u, c2), lo1 = 0xCD9E8D57u * c2;
    c0 = hi1 ^ c1 ^ k0; c1 = lo1; c2 = hi0 ^ c3 ^ k1; c3 = lo0;
    k0 += 0x9E3779B9u; k1 += 0xBB67AE85u;
  }
  out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

// two N(0,1) variates from two 32-bit words: Box-Muller on 23-bit uniforms u = (k + 1/2) 2^-23 (exact
// in FP32 and FP64, A12).  FP32: r = sqrt(-2 ln u1) and sin/cos(2 pi u2) on the SFU (lg2, sqrt, sin, cos
// approximations, absolute error ~1e-6 on a unit-variance variate); FP64: libm.
template <typename R> __device__ __forceinline__ void box_muller(uint32_t xa, uint32_t xb, R& zc, R& zs);
template <> __device__ __forceinline__ void box_muller<float>(uint32_t xa, uint32_t xb, float& zc, float& zs) {
  const float u1 = ((float)(xa >> 9) + 0.5f) * (1.0f / 8388608.0f);
  const float u2 = ((float)(xb >> 9) + 0.5f) * (1.0f / 8388608.0f);
  float l2, r;
  asm("lg2.approx.ftz.f32 %0, %1;" : "=f"(l2) : "f"(u1));
  asm("sqrt.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(-1.3862943611198906f * l2));     // -2 ln2 log2(u1)
  const float th = 6.2831853071795865f * u2;
  zc = r * __cosf(th); zs = r * __sinf(th);
}
template <> __device__ __forceinline__ void box_muller<double>(uint32_t xa, uint32_t xb, double& zc, double& zs) {
  const double u1 = ((double)(xa >> 9) + 0.5) * (1.0 / 8388608.0);
  const double u2 = ((double)(xb >> 9) + 0.5) * (1.0 / 8388608.0);
  const double r = sqrt(-2.0 * log(u1));
  double s, c;
  sincospi(2.0 * u2, &s, &c);
  zc = r * c; zs = r * s;
}
// the four normals of steps 4q .. 4q+3 of (sim, region)
template <typename R>
__device__ __forceinline__ void normals4(uint64_t seed, uint32_t sim, uint32_t region, uint64_t q, R xi[4]) {
  uint32_t x[4];
  philox4x32_10((uint32_t)q, (uint32_t)(q >> 32), region, sim, (uint32_t)seed, (uint32_t)(seed >> 32), x);
  box_muller<R>(x[0], x[1], xi[0], xi[1]);
  box_muller<R>(x[2], x[3], xi[2], xi[3]);
}

template <typename R> __device__ __forceinline__ R shfl_x1(unsigned mask, R v) { return __shfl_xor_sync(mask, v, 1); }

// ---- device-side descriptors ------------------------------------------------------------------------
// one non-zero weight: w = W_kj, jbase = j * Hs * SPC (element offset of the source region's ring row),
// back = Hp - d_kj
template <typename R> struct Edge;
template <> struct __align__(16) Edge<float> { float w; uint32_t jbase; uint32_t back; uint32_t pad; };   // pad = jbase + back * (ring columns)
template <> struct __align__(16) Edge<double> { double w; uint32_t jbase; uint32_t back; };

struct TableDesc {      // one per distinct speed v
  int32_t Hp;           // ring period (D + B + 1, or D + CH (LAG + 1) + 1 for the rolling pipeline)
  int32_t Hs;           // row stride Hp + GC - 1 (mirror slots)
  int32_t B;            // steps between CTA barriers (integrate_kernel)
  int32_t n_edges;
  int32_t CH;           // steps per chunk (integrate2_kernel): min(GC, d_min + 1)
  int32_t LAG;          // chunks a warp may run ahead of the slowest one (integrate2_kernel)
  int64_t edge_off;     // first edge in the edge array
  int64_t rowptr_off;   // first entry of this table's row pointer (N+1 ints)
  int64_t seg_off;      // VEC tables (integrate2_kernel, quad ring layout): first entry of the [N][4] class ends
  int32_t vec;          // 1: quad ring layout, rows sorted by window alignment class
  int32_t pad0;         // 1: every ring slot is mirrored (row length Hs = 2 Hp): one-step chunks of integrate2_kernel (GCE == 1)
};
struct GroupDesc {      // one per CTA
  int32_t table;
  int32_t pad;
  int64_t ring_off;     // in elements of R
};

enum { NPS = 12 };      // per-simulation scalars: G, wNoise, b_e, a_e/tau_w_e, 1/tau_w_e, E_L_e, E_L_i, 1/T, cFee, cFei, cFie, cFii
enum { NSV = 12 };      // persisted per (sim, region): E,I,Cee,Cei,Cii,We,Wi,OU, winE, winI, sumE, sumI

template <typename R>
struct IntegrateParams {
  TFConst<R> tf;
  // uniform model scalars
  R b_i, a_i_over_tau, inv_tau_w_i, inv_Ne, inv_Ni, kappa;
  R ou_rho, ou_s, ou_m;         // OU_{n+1} = ou_m + rho*OU_n + ou_s*xi,  ou_m = mu (1 - rho)
  R dt;
  int32_t muV_local;
  int32_t N;
  int32_t SPC;                  // simulations per CTA
  int32_t noise_on;
  int32_t ds;                   // 0 = no downsampling
  int64_t n_begin, n_end;       // global step range of this launch
  int64_t discard_steps;
  int32_t sample_base;          // chunk-local index of the first sample this launch may emit
  int32_t chunk_samples;        // CS: capacity of the sample buffer per group
  uint64_t seed;
  // arrays
  const TableDesc* tables;
  const GroupDesc* groups;
  const Edge<R>* edges;
  const int32_t* rowptr;
  const R* psim;                // [group][NPS][SPC]
  const int32_t* ext_id;        // [group][SPC]  external sim index (Philox counter)
  const int32_t* loc_id;        // [group][SPC]  local sim index (row of traj), -1 = padding lane
  R* ring;                      // [group][SPC][N][Hs]
  R* state;                     // [group][NSV-2][N][SPC]
  double* sums;                 // [group][2][N][SPC]  running sums of kept E / I samples
  R* xbar;                      // [group][CS][N][SPC] kept excitatory samples of the current chunk
  R* xbar_i;                    // same for the inhibitory population, or null (only tvbx_rate_stats uses them)
  R* traj;                      // optional [n_sims][traj_steps][7][N]
  int64_t traj_steps;
  int64_t traj_n0;              // global step index of traj row 0
  int32_t smem_table;           // edges + rowptr staged in shared memory
};

// per-lane registers: one population of one (sim, region)
template <typename R> struct Local {
  R nu;      // E (even lane) or I (odd lane)
  R Cs;      // C_ee or C_ii
  R Cei;     // both lanes keep the same copy
  R W;       // W_e or W_i
  R ou;      // both lanes keep the same copy
  R win;     // running window sum of nu
  double sum;
};

template <typename R>
__device__ __forceinline__ void load_local(const IntegrateParams<R>& P, int g, int k, int sl, int pop, Local<R>& s) {
  const size_t stride = (size_t)P.N * P.SPC;
  const R* p = P.state + (size_t)g * (NSV - 2) * stride + (size_t)k * P.SPC + sl;
  s.nu = p[(0 + pop) * stride]; s.Cs = p[(pop ? 4 : 2) * stride]; s.Cei = p[3 * stride];
  s.W = p[(5 + pop) * stride]; s.ou = p[7 * stride]; s.win = p[(8 + pop) * stride];
  s.sum = P.sums[(size_t)g * 2 * stride + pop * stride + (size_t)k * P.SPC + sl];
}
template <typename R>
__device__ __forceinline__ void store_local(const IntegrateParams<R>& P, int g, int k, int sl, int pop, const Local<R>& s) {
  const size_t stride = (size_t)P.N * P.SPC;
  R* p = P.state + (size_t)g * (NSV - 2) * stride + (size_t)k * P.SPC + sl;
  p[(0 + pop) * stride] = s.nu; p[(pop ? 4 : 2) * stride] = s.Cs; p[(5 + pop) * stride] = s.W;
  p[(8 + pop) * stride] = s.win;
  if (pop == 0) { p[3 * stride] = s.Cei; p[7 * stride] = s.ou; }
  P.sums[(size_t)g * 2 * stride + pop * stride + (size_t)k * P.SPC + sl] = s.sum;
}

// per-lane constants kept in shared memory (one column per thread; 64 registers per thread do not
// hold them next to the transfer function's temporaries)
enum { L_G = 0, L_WN, L_IT, L_B, L_AT, L_ITW, L_ATEL, L_GLEL, L_CFE, L_CFI, L_INVN, L_NPAR };

// SINGLE: every (sim, region) of the group has its own lane pair (blockDim >= 2*N*SPC): state stays
// in registers for the whole launch.  Otherwise the CTA makes several passes over the regions inside
// each time block and the state round-trips through global memory (L1/L2 resident).
// CLOSED: tau_e == tau_i -> tf_closed, else tf_jet.
// SPC_T: simulations per CTA as a compile-time constant (0 = take P.SPC): the ring loads of a gather
// chunk then use immediate offsets.
template <typename R, bool SINGLE, bool CLOSED, int SPC_T, int MAXT>
__global__ void __launch_bounds__(MAXT, 1) integrate_kernel(const __grid_constant__ IntegrateParams<R> P) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  const int g = blockIdx.x;
  const int N = P.N, SPC = SPC_T > 0 ? SPC_T : P.SPC;
  const int T = blockDim.x;
  const int pop = threadIdx.x & 1;
  const int pair = threadIdx.x >> 1;
  const int PT = T >> 1;                          // lane pairs per CTA (a multiple of SPC)
  const int RT = PT / SPC;                        // regions per pass
  const int rl = pair / SPC, sl = pair - rl * SPC;
  const GroupDesc gd = P.groups[g];
  const TableDesc td = P.tables[gd.table];
  const int Hp = td.Hp, Hs = td.Hs;
  const Edge<R>* edges = P.edges + td.edge_off;
  const int32_t* rowptr = P.rowptr + td.rowptr_off;
  // shared memory: [PT][GC+1] coupling sums | [PT][9] normals | [T][L_NPAR] lane constants (odd row
  // lengths: conflict-free) | 2 x 10 polynomial coefficients | optional edge table + row pointers
  R* s_cpl = reinterpret_cast<R*>(smem_raw) + (size_t)pair * (GC + 1);
  R* s_xi = reinterpret_cast<R*>(smem_raw) + (size_t)PT * (GC + 1) + (size_t)pair * 9;
  R* s_par = reinterpret_cast<R*>(smem_raw) + (size_t)PT * (GC + 10) + (size_t)threadIdx.x * L_NPAR;
  R* s_poly = reinterpret_cast<R*>(smem_raw) + (size_t)PT * (GC + 10) + (size_t)L_NPAR * T;
  {
    unsigned char* tab = reinterpret_cast<unsigned char*>(s_poly + 20);
    tab += (16 - (reinterpret_cast<uintptr_t>(tab) & 15)) & 15;
    if (threadIdx.x < 20)
      s_poly[threadIdx.x] = CLOSED ? P.tf.C[threadIdx.x / 10][threadIdx.x % 10] : P.tf.P[threadIdx.x / 10][threadIdx.x % 10];
    if (P.smem_table) {
      Edge<R>* se = reinterpret_cast<Edge<R>*>(tab);
      int32_t* sr = reinterpret_cast<int32_t*>(se + td.n_edges);
      for (int i = threadIdx.x; i < td.n_edges; i += T) se[i] = edges[i];
      for (int i = threadIdx.x; i <= N; i += T) sr[i] = rowptr[i];
      edges = se; rowptr = sr;
    }
    // per-simulation scalars of this lane's population
    const R* ps = P.psim + (size_t)g * NPS * SPC + sl;
    const R pEL = ps[(5 + pop) * SPC];
    const R pAT = pop ? P.a_i_over_tau : ps[3 * SPC];
    s_par[L_G] = ps[0 * SPC]; s_par[L_WN] = ps[1 * SPC]; s_par[L_IT] = ps[7 * SPC];
    s_par[L_B] = pop ? P.b_i : ps[2 * SPC];                 // b
    s_par[L_AT] = pAT;                                      // a / tau_w
    s_par[L_ITW] = pop ? P.inv_tau_w_i : ps[4 * SPC];       // 1 / tau_w
    s_par[L_ATEL] = pAT * pEL;
    s_par[L_GLEL] = P.tf.gL * pEL;
    s_par[L_CFE] = ps[(pop ? 10 : 8) * SPC]; s_par[L_CFI] = ps[(pop ? 11 : 9) * SPC];
    s_par[L_INVN] = pop ? P.inv_Ni : P.inv_Ne;
    __syncthreads();
  }
  const R* poly = s_poly + 10 * pop;
  // ring[group][region][slot][sim]: this lane's simulation column, as 32-bit element offsets
  R* const ringg = P.ring + gd.ring_off + sl;
  const uint32_t uSPC = (uint32_t)SPC;
  const int ext = P.ext_id[(size_t)g * SPC + sl];
  const int loc = P.loc_id[(size_t)g * SPC + sl];
  const R dt = P.dt;
  const R inv_ds = P.ds > 0 ? R(1) / R(P.ds) : R(0);
  const bool noise = P.noise_on != 0;

  Local<R> st;
  st.nu = st.Cs = st.Cei = st.W = st.ou = st.win = R(0); st.sum = 0.0;
  if (SINGLE && rl < N) load_local<R>(P, g, rl, sl, pop, st);

  int64_t n = P.n_begin;
  int cur = (int)(n % Hp);                       // ring slot of time index n
  // steps left in the current downsample window (uniform), and the next sample index
  int win_left0 = P.ds > 0 ? P.ds - (int)(n % P.ds) : 0x7fffffff;
  int sidx0 = P.sample_base;

  while (n < P.n_end) {
    const int nb = (int)min((int64_t)td.B, P.n_end - n);
    int win_left = win_left0, sidx = sidx0;
    for (int k0 = 0; k0 < N; k0 += RT) {
      const int k = k0 + rl;
      const unsigned mask = __ballot_sync(0xffffffffu, k < N);   // lanes of this warp that work in this pass
      if (k >= N) continue;
      if (!SINGLE) load_local<R>(P, g, k, sl, pop, st);
      win_left = win_left0; sidx = sidx0;
      const int e0 = rowptr[k], e1 = rowptr[k + 1];
      const uint32_t myrow = (uint32_t)(k * Hs) * uSPC;
      // Philox: at every step that is a multiple of 8 the even lane draws the quad of steps 8m..8m+3, the
      // odd lane that of 8m+4..8m+7 (no divergence); re-enter a partly used octet here
      if (noise && (n & 7) && (!SINGLE || n == P.n_begin)) {
        R xi[4];
        normals4<R>(P.seed, (uint32_t)ext, (uint32_t)k, (((uint64_t)n >> 3) << 1) + pop, xi);
#pragma unroll
        for (int q = 0; q < 4; ++q) s_xi[pop * 4 + q] = xi[q];
        __syncwarp(mask);
      }
      int c = cur;
      for (int c0 = 0; c0 < nb; c0 += GC) {
        const int ch = min(GC, nb - c0);
        // ================= GATHER: coupling sums of steps n+c0 .. n+c0+ch-1 (S1) =================
        {
          R acc[GC];
#pragma unroll
          for (int i = 0; i < GC; ++i) acc[i] = R(0);
          if (ch == GC) {
            for (int e = e0 + pop; e < e1; e += 2) {
              const Edge<R> ed = edges[e];
              int start = c + (int)ed.back;
              start = start >= Hp ? start - Hp : start;
              const R* src = ringg + (ed.jbase + (uint32_t)start * uSPC);
#pragma unroll
              for (int i = 0; i < GC; ++i) acc[i] = tfma(ed.w, src[i * SPC], acc[i]);
            }
          } else {
            for (int e = e0 + pop; e < e1; e += 2) {
              const Edge<R> ed = edges[e];
              int start = c + (int)ed.back;
              start = start >= Hp ? start - Hp : start;
              const R* src = ringg + (ed.jbase + (uint32_t)start * uSPC);
#pragma unroll
              for (int i = 0; i < GC; ++i)
                if (i < ch) acc[i] = tfma(ed.w, src[i * SPC], acc[i]);
            }
          }
#pragma unroll
          for (int i = 0; i < GC; ++i) {
            const R tot = acc[i] + shfl_x1(mask, acc[i]);    // a + b == b + a: both lanes get the same bits
            if (pop == 0) s_cpl[i] = tot;
          }
          __syncwarp(mask);
        }
        // ================= COMPUTE: ch steps in registers (S2-S6) =================
        const int64_t nn0 = n + c0;
        const bool traj_on = P.traj != nullptr && loc >= 0 && nn0 - P.traj_n0 < P.traj_steps;
        for (int i = 0; i < ch; ++i) {
          const uint32_t nlo = (uint32_t)nn0 + (uint32_t)i;      // low bits of the step index
          // ---- noise: new octet of normals ----
          if (noise && (nlo & 7u) == 0) {
            R xi[4];
            __syncwarp(mask);
            normals4<R>(P.seed, (uint32_t)ext, (uint32_t)k, ((uint64_t)(nn0 + i) >> 2) + pop, xi);
#pragma unroll
            for (int q = 0; q < 4; ++q) s_xi[pop * 4 + q] = xi[q];
            __syncwarp(mask);
          }
          const R cpl = s_cpl[i];
          // ---- exchange with the partner lane ----
          const R nu_o = shfl_x1(mask, st.nu), Cs_o = shfl_x1(mask, st.Cs);
          const R E = pop ? nu_o : st.nu, I = pop ? st.nu : nu_o;
          const R Cei = st.Cei;
          const R Ca = pop ? Cei : st.Cs, Cb = pop ? st.Cs : Cei;     // row `pop` of C   (own covariance)
          const R Co = pop ? Cs_o : Cei, Cp = pop ? Cei : Cs_o;       // the other row    (half of the C_ei equation)
          // ---- S2 inputs and transfer function of this lane's population (Eq. 5; A5, A6, A10) ----
          R drive = tfma(s_par[L_G], cpl, E);
          if (noise) drive = tfma(s_par[L_WN], st.ou, drive);
          const R xe = drive + s_par[L_CFE], xi_ = I + s_par[L_CFI];
          const R se = xe > R(0) ? P.kappa : R(0), si = xi_ > R(0) ? P.kappa : R(0);   // A22 and the clamp of A10
          const R c0w = s_par[L_GLEL] - st.W;
          R muV;
          Jet<R> F;
          if (CLOSED) F = tf_closed<R>(P.tf, poly, fmax(xe, R(0)) + P.tf.eps, fmax(xi_, R(0)) + P.tf.eps, c0w, &muV);
          else        F = tf_jet<R>(P.tf, poly, fmax(xe, R(0)) + P.tf.eps, fmax(xi_, R(0)) + P.tf.eps, c0w, &muV);
          if (P.muV_local)                    // A9b alternative: mu_V of the local rates only
            muV = mu_V_only<R>(P.tf, fmax(E, R(0)) + P.tf.eps, fmax(I, R(0)) + P.tf.eps, c0w);
          const R Fe = F.e * se, Fi = F.i * si;
          // ---- S3 Eqs. (1)-(3), forward Euler (A7, A9) ----
          const R pIT = s_par[L_IT];
          const R dF = F.v - st.nu;
          const R Cee_h = R(0.5) * (pop ? Co : Ca) * se * se, Cei_s = Cei * se * si, Cii_h = R(0.5) * (pop ? Cb : Cp) * si * si;
          const R dnu = tfma(Cee_h, F.ee, tfma(Cei_s, F.ei, tfma(Cii_h, F.ii, dF))) * pIT;
          const R dCs = tfma(F.v * (pIT - F.v), s_par[L_INVN], tfma(dF, dF, R(2) * (tfma(Ca, Fe, Cb * Fi) - st.Cs))) * pIT;
          const R h = tfma(Co, Fe, Cp * Fi);
          const R dF_o = shfl_x1(mask, dF), h_o = shfl_x1(mask, h);
          const R dCei = tfma(dF, dF_o, (h + h_o) - R(2) * Cei) * pIT;
          const R dW = tfma(s_par[L_AT], muV, tfma(s_par[L_B], st.nu, -tfma(st.W, s_par[L_ITW], s_par[L_ATEL])));
          st.nu = tfma(dt, dnu, st.nu);
          st.Cs = tfma(dt, dCs, st.Cs);
          st.Cei = tfma(dt, dCei, st.Cei);
          st.W = tfma(dt, dW, st.W);
          // ---- S4 OU (Eq. 4, A11) ----
          if (noise) st.ou = tfma(P.ou_rho, st.ou, tfma(P.ou_s, s_xi[nlo & 7u], P.ou_m));
          // ---- S5 ring write: E at time nn+1 (mirror the first GC-1 slots behind the period) ----
          c = c + 1 == Hp ? 0 : c + 1;
          if (pop == 0) {
            const uint32_t o = myrow + (uint32_t)c * uSPC;
            ringg[o] = st.nu;
            if (c < GC - 1) ringg[o + (uint32_t)Hp * uSPC] = st.nu;
          }
          // ---- trajectory (tests / cfg 1) ----
          if (traj_on && nn0 + i - P.traj_n0 < P.traj_steps) {
            R* t = P.traj + (((size_t)loc * P.traj_steps + (size_t)(nn0 + i - P.traj_n0)) * 7) * N + k;
            if (pop == 0) { t[0] = st.nu; t[2 * N] = st.Cs; t[3 * N] = st.Cei; t[5 * N] = st.W; }
            else { t[N] = st.nu; t[4 * N] = st.Cs; t[6 * N] = st.W; }
          }
          // ---- S6 temporal average (A17) ----
          st.win += st.nu;
          if (--win_left == 0) {
            win_left = P.ds;
            if (nn0 + i + 1 > P.discard_steps) {
              const R m = st.win * inv_ds;
              if (pop == 0) P.xbar[(((size_t)g * P.chunk_samples + sidx) * N + k) * SPC + sl] = m;
              else if (P.xbar_i) P.xbar_i[(((size_t)g * P.chunk_samples + sidx) * N + k) * SPC + sl] = m;
              st.sum += (double)m;
              ++sidx;
            }
            st.win = R(0);
          }
        }
        __syncwarp(mask);
      }
      if (!SINGLE) store_local<R>(P, g, k, sl, pop, st);
    }
    win_left0 = win_left; sidx0 = sidx;      // (lanes that never work never use them)
    n += nb;
    cur += nb; if (cur >= Hp) cur -= Hp;
    __syncthreads();
  }
  if (SINGLE && rl < N) store_local<R>(P, g, rl, sl, pop, st);
}

}  // namespace tvbx
