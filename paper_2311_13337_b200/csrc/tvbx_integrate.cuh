// tvbx_integrate.cuh -- the integrator kernel: delayed gather + coupling sum (S1), both transfer
// functions with derivatives (S2), Euler update of the 7 state variables (S3), OU noise from
// in-kernel Philox4x32-10 (S4), history-ring write (S5), temporal-average downsample (S6) and the
// per-thread running sums for the mean rates.  DESIGN.md section 6 describes the mapping.
//
// Mapping (B200-first, not the paper's thread-per-simulation kernel):
//   CTA      = one "group" of SPC simulations that share a delay table (same speed v), all N regions
//   thread   = (region lane rl, simulation lane sl); sl is the fastest thread index, so a warp holds
//              32/SPC regions x SPC sims and every ring access of SPC sims is one contiguous line
//   ring     = ring[group][region][slot][SPC]  (E only, "temporal buffer")
//   time     = the kernel is persistent over time: it runs B = max(1, min delay) steps between CTA
//              barriers, because step n only reads E at times <= n - d_min
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include "tvbx_tf.cuh"

namespace tvbx {

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

// four N(0,1) variates for steps 4q .. 4q+3 of (sim, region): Box-Muller on 23-bit uniforms
template <typename R> __device__ __forceinline__ void box_muller(uint32_t xa, uint32_t xb, R& zc, R& zs);
template <> __device__ __forceinline__ void box_muller<float>(uint32_t xa, uint32_t xb, float& zc, float& zs) {
  const float u1 = ((float)(xa >> 9) + 0.5f) * (1.0f / 8388608.0f);
  const float u2 = ((float)(xb >> 9) + 0.5f) * (1.0f / 8388608.0f);
  const float r = sqrtf(-2.0f * logf(u1));
  float s, c;
  sincospif(2.0f * u2, &s, &c);
  zc = r * c; zs = r * s;
}
template <> __device__ __forceinline__ void box_muller<double>(uint32_t xa, uint32_t xb, double& zc, double& zs) {
  const double u1 = ((double)(xa >> 9) + 0.5) * (1.0 / 8388608.0);
  const double u2 = ((double)(xb >> 9) + 0.5) * (1.0 / 8388608.0);
  const double r = sqrt(-2.0 * log(u1));
  double s, c;
  sincospi(2.0 * u2, &s, &c);
  zc = r * c; zs = r * s;
}
template <typename R>
__device__ __forceinline__ void normals4(uint64_t seed, uint32_t sim, uint32_t region, uint64_t q, R xi[4]) {
  uint32_t x[4];
  philox4x32_10((uint32_t)q, (uint32_t)(q >> 32), region, sim, (uint32_t)seed, (uint32_t)(seed >> 32), x);
  box_muller<R>(x[0], x[1], xi[0], xi[1]);
  box_muller<R>(x[2], x[3], xi[2], xi[3]);
}

// ---- device-side descriptors ------------------------------------------------------------------------
template <typename R> struct Edge { R w; int32_t jbase; int32_t back; };   // jbase = j*Hp, back = Hp - d
template <> struct __align__(16) Edge<float> { float w; int32_t jbase; int32_t back; int32_t pad; };
template <> struct __align__(16) Edge<double> { double w; int32_t jbase; int32_t back; };

struct TableDesc {      // one per distinct speed v
  int32_t Hp;           // physical ring length D + B + 1
  int32_t B;            // steps between CTA barriers
  int32_t n_edges;
  int32_t pad;
  int64_t edge_off;     // first edge in the edge array
  int64_t rowptr_off;   // first entry of this table's row pointer (N+1 ints)
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
  const int32_t* ext_id;        // [group][SPC]  external sim index (Philox counter), -1 = padding lane
  const int32_t* loc_id;        // [group][SPC]  local sim index (row of traj), -1 = padding lane
  R* ring;                      // [group][N][Hp][SPC]
  R* state;                     // [group][NSV-2][N][SPC]
  double* sums;                 // [group][2][N][SPC]  running sums of kept E / I samples
  R* xbar;                      // [group][CS][N][SPC] kept excitatory samples of the current chunk
  R* traj;                      // optional [n_sims][traj_steps][7][N]
  int64_t traj_steps;
  int64_t traj_n0;              // global step index of traj row 0
  int32_t smem_table;           // edges + rowptr staged in shared memory
};

template <typename R> struct Local {   // per (sim, region) registers
  R E, I, Cee, Cei, Cii, We, Wi, ou, winE, winI;
  double sumE, sumI;
};

template <typename R, int SPC>
__device__ __forceinline__ void load_local(const IntegrateParams<R>& P, int g, int k, int sl, Local<R>& s) {
  const size_t stride = (size_t)P.N * SPC;
  const R* p = P.state + (size_t)g * (NSV - 2) * stride + (size_t)k * SPC + sl;
  s.E = p[0 * stride]; s.I = p[1 * stride]; s.Cee = p[2 * stride]; s.Cei = p[3 * stride];
  s.Cii = p[4 * stride]; s.We = p[5 * stride]; s.Wi = p[6 * stride]; s.ou = p[7 * stride];
  s.winE = p[8 * stride]; s.winI = p[9 * stride];
  const double* q = P.sums + (size_t)g * 2 * stride + (size_t)k * SPC + sl;
  s.sumE = q[0]; s.sumI = q[stride];
}
template <typename R, int SPC>
__device__ __forceinline__ void store_local(const IntegrateParams<R>& P, int g, int k, int sl, const Local<R>& s) {
  const size_t stride = (size_t)P.N * SPC;
  R* p = P.state + (size_t)g * (NSV - 2) * stride + (size_t)k * SPC + sl;
  p[0 * stride] = s.E; p[1 * stride] = s.I; p[2 * stride] = s.Cee; p[3 * stride] = s.Cei;
  p[4 * stride] = s.Cii; p[5 * stride] = s.We; p[6 * stride] = s.Wi; p[7 * stride] = s.ou;
  p[8 * stride] = s.winE; p[9 * stride] = s.winI;
  double* q = P.sums + (size_t)g * 2 * stride + (size_t)k * SPC + sl;
  q[0] = s.sumE; q[stride] = s.sumI;
}

// SINGLE: every (sim, region) of the group has its own thread (blockDim >= N*SPC): state stays in
// registers for the whole launch.  Otherwise the CTA makes several passes over the regions inside
// each time block and the state round-trips through global memory (L1/L2 resident).
template <typename R, int SPC, bool SINGLE, int MAXT>
__global__ void __launch_bounds__(MAXT, 1) integrate_kernel(const __grid_constant__ IntegrateParams<R> P) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  const int g = blockIdx.x;
  const int sl = threadIdx.x % SPC;
  const int rl = threadIdx.x / SPC;
  const int RT = blockDim.x / SPC;
  const int N = P.N;
  const GroupDesc gd = P.groups[g];
  const TableDesc td = P.tables[gd.table];
  const int Hp = td.Hp;
  const Edge<R>* edges = P.edges + td.edge_off;
  const int32_t* rowptr = P.rowptr + td.rowptr_off;
  if (P.smem_table) {
    Edge<R>* se = reinterpret_cast<Edge<R>*>(smem_raw);
    int32_t* sr = reinterpret_cast<int32_t*>(se + td.n_edges);
    for (int i = threadIdx.x; i < td.n_edges; i += blockDim.x) se[i] = edges[i];
    for (int i = threadIdx.x; i <= N; i += blockDim.x) sr[i] = rowptr[i];
    __syncthreads();
    edges = se; rowptr = sr;
  }
  R* ring = P.ring + gd.ring_off + sl;

  // per-simulation scalars
  const R* ps = P.psim + (size_t)g * NPS * SPC + sl;
  const R pG = ps[0 * SPC], pWn = ps[1 * SPC], pBe = ps[2 * SPC], pAeT = ps[3 * SPC], pITw = ps[4 * SPC];
  const R pELe = ps[5 * SPC], pELi = ps[6 * SPC], pIT = ps[7 * SPC];
  const R cFee = ps[8 * SPC], cFei = ps[9 * SPC], cFie = ps[10 * SPC], cFii = ps[11 * SPC];
  const R gLELe = P.tf.gL * pELe, gLELi = P.tf.gL * pELi;
  const int ext = P.ext_id[(size_t)g * SPC + sl];
  const int loc = P.loc_id[(size_t)g * SPC + sl];
  const R dt = P.dt, kap = P.kappa, kap2 = P.kappa * P.kappa;
  const R inv_ds = P.ds > 0 ? R(1) / R(P.ds) : R(0);

  Local<R> st;
  if (SINGLE && rl < N) load_local<R, SPC>(P, g, rl, sl, st);
  R xi[4] = {R(0), R(0), R(0), R(0)};   // the four normals of the current Philox call

  int64_t n = P.n_begin;
  int cur = (int)(n % Hp);                       // ring slot of time index n
  // steps left in the current downsample window (uniform), and the next sample index
  int win_left0 = P.ds > 0 ? P.ds - (int)(n % P.ds) : 0x7fffffff;
  int sidx0 = P.sample_base;

  while (n < P.n_end) {
    const int nb = (int)min((int64_t)td.B, P.n_end - n);
    int win_left = win_left0, sidx = sidx0;
    for (int k = rl; k < N; k += RT) {
      if (!SINGLE) load_local<R, SPC>(P, g, k, sl, st);
      win_left = win_left0; sidx = sidx0;
      const int e0 = rowptr[k], e1 = rowptr[k + 1];
      R* myring = ring + (size_t)k * Hp * SPC;
      if (P.noise_on && (n & 3) && (!SINGLE || n == P.n_begin))   // re-enter a partly used quad
        normals4<R>(P.seed, (uint32_t)ext, (uint32_t)k, (uint64_t)n >> 2, xi);
      int c = cur;
      for (int i = 0; i < nb; ++i) {
        const int64_t nn = n + i;
        // ---- S1 delayed gather + coupling sum (ascending j, A16) ----
        R cpl = R(0);
        for (int e = e0; e < e1; ++e) {
          const Edge<R> ed = edges[e];
          int slot = c + ed.back;
          slot = slot >= Hp ? slot - Hp : slot;
          cpl = tfma(ed.w, ring[(size_t)(ed.jbase + slot) * SPC], cpl);
        }
        // ---- S2 inputs and transfer functions (Eq. 5; A5, A6, A10) ----
        if (P.noise_on && (nn & 3) == 0) normals4<R>(P.seed, (uint32_t)ext, (uint32_t)k, (uint64_t)nn >> 2, xi);
        const R eta = P.noise_on ? pWn * st.ou : R(0);
        const R drive = tfma(pG, cpl, st.E) + eta;
        R muVe, muVi;
        Jet<R> Fe, Fi;
        {
          const R xe = drive + cFee, xi_ = st.I + cFei;
          const R se = xe > R(0) ? R(1) : R(0), si = xi_ > R(0) ? R(1) : R(0);
          Fe = transfer_function<R>(P.tf, 0, fmax(xe, R(0)) + P.tf.eps, fmax(xi_, R(0)) + P.tf.eps,
                                    gLELe - st.We, &muVe);
          Fe.e *= kap * se; Fe.i *= kap * si;
          Fe.ee *= kap2 * se; Fe.ei *= kap2 * se * si; Fe.ii *= kap2 * si;
        }
        {
          const R xe = drive + cFie, xi_ = st.I + cFii;
          const R se = xe > R(0) ? R(1) : R(0), si = xi_ > R(0) ? R(1) : R(0);
          Fi = transfer_function<R>(P.tf, 1, fmax(xe, R(0)) + P.tf.eps, fmax(xi_, R(0)) + P.tf.eps,
                                    gLELi - st.Wi, &muVi);
          Fi.e *= kap * se; Fi.i *= kap * si;
          Fi.ee *= kap2 * se; Fi.ei *= kap2 * se * si; Fi.ii *= kap2 * si;
        }
        if (P.muV_local) {   // A9b alternative: mu_V of the local rates only
          const R le = fmax(st.E, R(0)) + P.tf.eps, li = fmax(st.I, R(0)) + P.tf.eps;
          muVe = mu_V_only<R>(P.tf, le, li, gLELe - st.We);
          muVi = mu_V_only<R>(P.tf, le, li, gLELi - st.Wi);
        }
        // ---- S3 Eqs. (1)-(3), forward Euler (A7, A9) ----
        const R h = R(0.5);
        const R dFe = Fe.v - st.E, dFi = Fi.v - st.I;
        const R dE = (dFe + h * st.Cee * Fe.ee + st.Cei * Fe.ei + h * st.Cii * Fe.ii) * pIT;
        const R dI = (dFi + h * st.Cee * Fi.ee + st.Cei * Fi.ei + h * st.Cii * Fi.ii) * pIT;
        const R dCee = (Fe.v * (pIT - Fe.v) * P.inv_Ne + dFe * dFe +
                        R(2) * (st.Cee * Fe.e + st.Cei * Fe.i) - R(2) * st.Cee) * pIT;
        const R dCii = (Fi.v * (pIT - Fi.v) * P.inv_Ni + dFi * dFi +
                        R(2) * (st.Cei * Fi.e + st.Cii * Fi.i) - R(2) * st.Cii) * pIT;
        const R dCei = (dFe * dFi + (st.Cei * Fe.e + st.Cii * Fe.i) + (st.Cee * Fi.e + st.Cei * Fi.i) -
                        R(2) * st.Cei) * pIT;
        const R dWe = -st.We * pITw + pBe * st.E + pAeT * (muVe - pELe);
        const R dWi = -st.Wi * P.inv_tau_w_i + P.b_i * st.I + P.a_i_over_tau * (muVi - pELi);
        st.E = tfma(dt, dE, st.E);       st.I = tfma(dt, dI, st.I);
        st.Cee = tfma(dt, dCee, st.Cee); st.Cei = tfma(dt, dCei, st.Cei); st.Cii = tfma(dt, dCii, st.Cii);
        st.We = tfma(dt, dWe, st.We);    st.Wi = tfma(dt, dWi, st.Wi);
        // ---- S4 OU (Eq. 4, A11) ----
        if (P.noise_on) {
          const int w = (int)(nn & 3);      // select chain keeps xi[] in registers
          const R x = w == 0 ? xi[0] : (w == 1 ? xi[1] : (w == 2 ? xi[2] : xi[3]));
          st.ou = tfma(P.ou_rho, st.ou, tfma(P.ou_s, x, P.ou_m));
        }
        // ---- S5 ring write: E at time nn+1 ----
        c = c + 1 == Hp ? 0 : c + 1;
        myring[(size_t)c * SPC] = st.E;
        // ---- trajectory (tests / cfg 1) ----
        if (P.traj && nn - P.traj_n0 < P.traj_steps && loc >= 0) {
          R* t = P.traj + (((size_t)loc * P.traj_steps + (size_t)(nn - P.traj_n0)) * 7) * N + k;
          t[0] = st.E; t[N] = st.I; t[2 * N] = st.Cee; t[3 * N] = st.Cei; t[4 * N] = st.Cii;
          t[5 * N] = st.We; t[6 * N] = st.Wi;
        }
        // ---- S6 temporal average (A17) ----
        st.winE += st.E; st.winI += st.I;
        if (--win_left == 0) {
          win_left = P.ds;
          if (nn + 1 > P.discard_steps) {
            const R me = st.winE * inv_ds, mi = st.winI * inv_ds;
            P.xbar[(((size_t)g * P.chunk_samples + sidx) * N + k) * SPC + sl] = me;
            st.sumE += (double)me; st.sumI += (double)mi;
            ++sidx;
          }
          st.winE = R(0); st.winI = R(0);
        }
      }
      if (!SINGLE) store_local<R, SPC>(P, g, k, sl, st);
    }
    if (rl >= N || N <= 0) {   // idle lanes still have to advance the uniform counters
      win_left = win_left0; sidx = sidx0;
      for (int i = 0; i < nb; ++i) {
        if (--win_left == 0) { win_left = P.ds; if (n + i + 1 > P.discard_steps) ++sidx; }
      }
    }
    win_left0 = win_left; sidx0 = sidx;
    n += nb;
    cur += nb; if (cur >= Hp) cur -= Hp;
    __syncthreads();
  }
  if (SINGLE && rl < N) store_local<R, SPC>(P, g, rl, sl, st);
}

}  // namespace tvbx
