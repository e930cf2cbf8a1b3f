// tvbx_integrate2.cuh -- the FP32 product integrator (closed-form transfer function, tau_e == tau_i):
// delayed gather + coupling sum (S1), both transfer functions with derivatives (S2), Euler update of
// the 7 state variables (S3), OU noise from in-kernel Philox4x32-10 (S4), history-ring write (S5),
// temporal-average downsample (S6) and the running sums for the mean rates.  DESIGN.md section 6.2.
//
// Mapping (B200-first; the paper's kernel is one thread per whole simulation):
//   CTA     = one "group" of SPC simulations that share a delay table (same speed v), all N regions,
//             persistent over the time steps of a launch
//   thread  = one (simulation, region).  The excitatory and the inhibitory population of that node
//             live in the two halves of packed FP32 pairs (float2: .x = e, .y = i) and are advanced
//             by Blackwell's two-wide FP32 instructions (FFMA2 / FMUL2 / FADD2): the two transfer
//             functions are the same formulas on different constants, so one instruction stream
//             serves both (tvbx_tf2.cuh).
//   ring    = ring[group][region][slot][sim] (E only, "temporal buffer"): the SPC simulations
//             of a group are the fastest index, so the lanes that share a region read one contiguous
//             run per (edge, step).  Rows carry GC-1 mirror slots so that a chunk of GC reads never wraps.
//   time    = chunks of CH <= min(GC, d_min + 1) steps: a GATHER of the chunk's coupling sums (per edge
//             one 16-byte table entry, CH loads with immediate offsets, CH/2 FFMA2) followed by CH
//             COMPUTE steps in registers.  Step n reads E only at times <= n - d_min, so chunk m needs
//             the ring writes of chunks <= m - LAG of all warps, LAG = ceil((d_min + 2)/CH) - 1 >= 1.
//             Instead of a CTA-wide barrier per time block the warps run a ROLLING pipeline on a ring
//             of 8 shared-memory mbarriers: every warp arrives (release) on barrier m mod 8 when it has
//             written chunk m and waits (acquire) for phase m - LAG before gathering chunk m, so a warp
//             may run up to LAG chunks ahead of the slowest one and nobody idles at a block boundary.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include "tvbx_integrate.cuh"
#include "tvbx_tf2.cuh"

namespace tvbx {

enum { NP2 = 9 };       // packed per-simulation parameters, see P2_*
enum { P2_GW = 0, P2_IT, P2_B, P2_AT, P2_ITW, P2_ATEL, P2_GLEL, P2_CFE, P2_CFI };
enum { NBAR = 8, LAGMAX = NBAR - 1 };

struct Integrate2Params {
  TF2Const tf;
  float kappa, inv_Ne, inv_Ni;
  float ou_rho, ou_s, ou_m;       // OU_{n+1} = ou_m + rho*OU_n + ou_s*xi,  ou_m = mu (1 - rho)
  float dt;
  int32_t muV_local;
  int32_t N;
  int32_t SPC;                    // simulations per CTA
  int32_t noise_on;
  int32_t ds;                     // 0 = no downsampling
  int64_t n_begin, n_end;         // global step range of this launch
  int64_t discard_steps;
  int32_t sample_base;            // chunk-local index of the first sample this launch may emit
  int32_t chunk_samples;          // CS: capacity of the sample buffer per group
  uint64_t seed;
  const TableDesc* tables;
  const GroupDesc* groups;
  const Edge<float>* edges;
  const int32_t* rowptr;
  const float2* psim2;            // [group][NP2][SPC]
  const int32_t* ext_id;          // [group][SPC]  external sim index (Philox counter)
  const int32_t* loc_id;          // [group][SPC]  local sim index (row of traj), -1 = padding lane
  float* ring;                    // [group][N][Hs][SPC]
  float* state;                   // [group][NSV-2][N][SPC]
  double* sums;                   // [group][2][N][SPC]
  float* xbar;                    // [group][CS][N][SPC]
  float* traj;                    // optional [n_sims][traj_steps][7][N]
  int64_t traj_steps;
  int64_t traj_n0;
  int32_t smem_table;
};

__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(uint64_t* bar, uint32_t count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
}
// default semantics: arrive = release.cta, try_wait = acquire.cta (orders the ring stores of the
// arriving warps before the ring loads of the waiting ones)
__device__ __forceinline__ void mbar_arrive(uint64_t* bar) {
  asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t* bar, uint32_t parity) {
  asm volatile(
      "{\n"
      ".reg .pred p;\n"
      "WAIT_%=:\n"
      "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
      "@p bra DONE_%=;\n"
      "bra WAIT_%=;\n"
      "DONE_%=:\n"
      "}\n" ::"r"(smem_u32(bar)), "r"(parity)
      : "memory");
}

// SPC_T: simulations per CTA as a compile-time constant (0 = take P.SPC): the ring loads of a gather
// chunk then use immediate offsets.
template <int SPC_T>
__global__ void __launch_bounds__(512, 1) integrate2_kernel(const __grid_constant__ Integrate2Params P) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  const int g = blockIdx.x;
  const int N = P.N, SPC = SPC_T > 0 ? SPC_T : P.SPC;
  const int T = blockDim.x, tid = threadIdx.x;
  const int rl = tid / SPC, sl = tid - rl * SPC;
  const bool active = rl < N;                     // threads past the last region replay it, stores suppressed
  const int k = active ? rl : N - 1;
  const GroupDesc gd = P.groups[g];
  const TableDesc td = P.tables[gd.table];
  const int Hp = td.Hp, Hs = td.Hs, CH = td.CH, LAG = td.LAG;
  const Edge<float>* edges = P.edges + td.edge_off;
  const int32_t* rowptr = P.rowptr + td.rowptr_off;
  // shared memory: NBAR mbarriers | [GC][T] coupling sums | [4][T] normals | [NP2][SPC] packed per-sim
  // parameters | optional edge table + row pointers
  uint64_t* bars = reinterpret_cast<uint64_t*>(smem_raw);
  float* s_cpl = reinterpret_cast<float*>(smem_raw + NBAR * 8) + tid;
  float* s_xi = reinterpret_cast<float*>(smem_raw + NBAR * 8) + (size_t)GC * T + tid;
  float2* s_ps = reinterpret_cast<float2*>(reinterpret_cast<float*>(smem_raw + NBAR * 8) + (size_t)(GC + 4) * T);
  {
    if (tid < NBAR) mbar_init(bars + tid, (uint32_t)(T >> 5));
    for (int i = tid; i < NP2 * SPC; i += T) s_ps[i] = P.psim2[(size_t)g * NP2 * SPC + i];
    if (P.smem_table) {
      unsigned char* tab = reinterpret_cast<unsigned char*>(s_ps + NP2 * SPC);
      tab += (16 - (reinterpret_cast<uintptr_t>(tab) & 15)) & 15;
      Edge<float>* se = reinterpret_cast<Edge<float>*>(tab);
      int32_t* sr = reinterpret_cast<int32_t*>(se + td.n_edges);
      for (int i = tid; i < td.n_edges; i += T) se[i] = edges[i];
      for (int i = tid; i <= N; i += T) sr[i] = rowptr[i];
      edges = se; rowptr = sr;
    }
    __syncthreads();
  }
  s_ps += sl;
  float* const ringg = P.ring + gd.ring_off + sl;
  const uint32_t uSPC = (uint32_t)SPC;
  const uint32_t myrow = (uint32_t)(k * Hs) * uSPC;
  const int e0 = rowptr[k], e1 = rowptr[k + 1];
  const int ext = P.ext_id[(size_t)g * SPC + sl];
  const int loc = P.loc_id[(size_t)g * SPC + sl];
  const float dt = P.dt;
  const float inv_ds = P.ds > 0 ? 1.0f / (float)P.ds : 0.0f;
  const bool noise = P.noise_on != 0;
  const f2 invN = mk2(P.inv_Ne, P.inv_Ni);

  // ---- state of this (sim, region) in registers: nu = (E, I), Cs = (C_ee, C_ii), W = (W_e, W_i) ----
  f2 nu, Cs, W, win;
  float Cei, ou;
  double sumE, sumI;
  const size_t stride = (size_t)N * SPC;
  float* const sp = P.state + (size_t)g * (NSV - 2) * stride + (size_t)k * SPC + sl;
  double* const sump = P.sums + (size_t)g * 2 * stride + (size_t)k * SPC + sl;
  nu = mk2(sp[0], sp[stride]); Cs = mk2(sp[2 * stride], sp[4 * stride]); Cei = sp[3 * stride];
  W = mk2(sp[5 * stride], sp[6 * stride]); ou = sp[7 * stride]; win = mk2(sp[8 * stride], sp[9 * stride]);
  sumE = sump[0]; sumI = sump[stride];

  int64_t n = P.n_begin;
  int cur = (int)(n % Hp);                        // ring slot of time index n
  int win_left = P.ds > 0 ? P.ds - (int)(n % P.ds) : 0x7fffffff;   // steps left in the current window
  int sidx = P.sample_base;
  // Philox (A12): one call per (sim, region) per 4 steps gives the quad of normals of steps 4q..4q+3;
  // re-enter a partly used quad at the start of a launch
  if (noise && (n & 3)) {
    float xi[4];
    normals4<float>(P.seed, (uint32_t)ext, (uint32_t)k, (uint64_t)n >> 2, xi);
#pragma unroll
    for (int q = 0; q < 4; ++q) s_xi[q * T] = xi[q];
  }

  for (uint32_t m = 0; n < P.n_end; ++m) {
    const int ch = (int)min((int64_t)CH, P.n_end - n);
    // the ring writes of chunk m - LAG (all warps) must be visible before this chunk's gather
    if (m >= (uint32_t)LAG) { const uint32_t w = m - (uint32_t)LAG; mbar_wait(bars + (w & (NBAR - 1)), (w / NBAR) & 1u); }
    // ================= GATHER: coupling sums of steps n .. n+ch-1 (S1) =================
    {
      f2 acc[GC / 2];
#pragma unroll
      for (int i = 0; i < GC / 2; ++i) acc[i] = mk2(0.0f, 0.0f);
      if (ch == GC) {
        for (int e = e0; e < e1; ++e) {
          const Edge<float> ed = edges[e];
          int start = cur + (int)ed.back;
          start = start >= Hp ? start - Hp : start;
          const float* src = ringg + (ed.jbase + (uint32_t)start * uSPC);
#pragma unroll
          for (int i = 0; i < GC / 2; ++i) acc[i] = fma2(bc2(ed.w), mk2(src[(2 * i) * SPC], src[(2 * i + 1) * SPC]), acc[i]);
        }
      } else {
        for (int e = e0; e < e1; ++e) {
          const Edge<float> ed = edges[e];
          int start = cur + (int)ed.back;
          start = start >= Hp ? start - Hp : start;
          const float* src = ringg + (ed.jbase + (uint32_t)start * uSPC);
#pragma unroll
          for (int i = 0; i < GC / 2; ++i) {
            const float v0 = 2 * i < ch ? src[(2 * i) * SPC] : 0.0f;
            const float v1 = 2 * i + 1 < ch ? src[(2 * i + 1) * SPC] : 0.0f;
            acc[i] = fma2(bc2(ed.w), mk2(v0, v1), acc[i]);
          }
        }
      }
#pragma unroll
      for (int i = 0; i < GC / 2; ++i) { s_cpl[(2 * i) * T] = acc[i].x; s_cpl[(2 * i + 1) * T] = acc[i].y; }
    }
    // ================= COMPUTE: ch steps in registers (S2-S6) =================
    const bool traj_on = P.traj != nullptr && loc >= 0 && active && n - P.traj_n0 < P.traj_steps;
    int c = cur;
    for (int i = 0; i < ch; ++i) {
      const int64_t nn = n + i;
      const uint32_t nlo = (uint32_t)nn;
      if (noise && (nlo & 3u) == 0) {             // new quad of normals
        float xi[4];
        normals4<float>(P.seed, (uint32_t)ext, (uint32_t)k, (uint64_t)nn >> 2, xi);
#pragma unroll
        for (int q = 0; q < 4; ++q) s_xi[q * T] = xi[q];
      }
      const float cpl = s_cpl[i * T];
      // ---- S2 inputs (Eq. 5; A5, A6, A10) ----
      const f2 gw = s_ps[P2_GW * SPC];
      float drive = __fmaf_rn(gw.x, cpl, nu.x);
      if (noise) drive = __fmaf_rn(gw.y, ou, drive);
      const f2 xe = add2(bc2(drive), s_ps[P2_CFE * SPC]);
      const f2 xi_ = add2(bc2(nu.y), s_ps[P2_CFI * SPC]);
      const f2 se = mk2(xe.x > 0.0f ? P.kappa : 0.0f, xe.y > 0.0f ? P.kappa : 0.0f);      // A22 and the clamp of A10
      const f2 si = mk2(xi_.x > 0.0f ? P.kappa : 0.0f, xi_.y > 0.0f ? P.kappa : 0.0f);
      const f2 fe = add2(mk2(fmaxf(xe.x, 0.0f), fmaxf(xe.y, 0.0f)), bc2(P.tf.eps));
      const f2 fi = add2(mk2(fmaxf(xi_.x, 0.0f), fmaxf(xi_.y, 0.0f)), bc2(P.tf.eps));
      const f2 c0 = sub2(s_ps[P2_GLEL * SPC], W);
      f2 muV;
      const Jet2 F = tf_closed2(P.tf, fe, fi, c0, &muV);
      if (P.muV_local) {                          // A9b alternative: mu_V of the local rates only
        const float le = fmaxf(nu.x, 0.0f) + P.tf.eps, li = fmaxf(nu.y, 0.0f) + P.tf.eps;
        const float den = __fmaf_rn(P.tf.ae, le, __fmaf_rn(P.tf.ai, li, P.tf.gL));
        const float base = __fmaf_rn(P.tf.aeEe, le, P.tf.aiEi * li);
        muV = mk2((base + c0.x) / den, (base + c0.y) / den);
      }
      // ---- S3 Eqs. (1)-(3), forward Euler (A7, A9) ----
      const f2 IT = bc2(s_ps[P2_IT * SPC].x);
      const f2 Fe = mul2(F.e, se), Fi = mul2(F.i, si);
      const f2 dF = sub2(F.v, nu);
      f2 a2nd = fma2(bc2(0.5f * Cs.x), mul2(F.ee, mul2(se, se)), dF);
      a2nd = fma2(bc2(Cei), mul2(F.ei, mul2(se, si)), a2nd);
      a2nd = fma2(bc2(0.5f * Cs.y), mul2(F.ii, mul2(si, si)), a2nd);
      const f2 dnu = mul2(a2nd, IT);
      const f2 Ca = mk2(Cs.x, Cei), Cb = mk2(Cei, Cs.y);            // row mu of the covariance matrix
      const f2 gC = fma2(Ca, Fe, fms2(Cb, Fi, Cs));                 // (C dF/dnu)_mu,mu - C_mu,mu
      const f2 dCs = mul2(fma2(mul2(F.v, sub2(IT, F.v)), invN, fma2(dF, dF, add2(gC, gC))), IT);
      const f2 Co = mk2(Cei, Cs.x), Cp = mk2(Cs.y, Cei);            // the other row
      const f2 h2 = fma2(Co, Fe, mul2(Cp, Fi));
      const float dCei = __fmaf_rn(dF.x, dF.y, (h2.x + h2.y) - 2.0f * Cei) * IT.x;
      const f2 dW = fma2(s_ps[P2_AT * SPC], muV, fms2(s_ps[P2_B * SPC], nu, fma2(W, s_ps[P2_ITW * SPC], s_ps[P2_ATEL * SPC])));
      nu = fma2(bc2(dt), dnu, nu);
      Cs = fma2(bc2(dt), dCs, Cs);
      Cei = __fmaf_rn(dt, dCei, Cei);
      W = fma2(bc2(dt), dW, W);
      // ---- S4 OU (Eq. 4, A11) ----
      if (noise) ou = __fmaf_rn(P.ou_rho, ou, __fmaf_rn(P.ou_s, s_xi[(nlo & 3u) * T], P.ou_m));
      // ---- S5 ring write: E at time nn+1 (mirror the first GC-1 slots behind the period) ----
      c = c + 1 == Hp ? 0 : c + 1;
      if (active) {
        const uint32_t o = myrow + (uint32_t)c * uSPC;
        ringg[o] = nu.x;
        if (c < GC - 1) ringg[o + (uint32_t)Hp * uSPC] = nu.x;
      }
      // ---- trajectory (tests / cfg 1) ----
      if (traj_on && nn - P.traj_n0 < P.traj_steps) {
        float* t = P.traj + (((size_t)loc * P.traj_steps + (size_t)(nn - P.traj_n0)) * 7) * N + k;
        t[0] = nu.x; t[N] = nu.y; t[2 * N] = Cs.x; t[3 * N] = Cei; t[4 * N] = Cs.y; t[5 * N] = W.x; t[6 * N] = W.y;
      }
      // ---- S6 temporal average (A17) ----
      win = add2(win, nu);
      if (--win_left == 0) {
        win_left = P.ds;
        if (nn + 1 > P.discard_steps) {
          const f2 mm = scl2(inv_ds, win);
          if (active) P.xbar[(((size_t)g * P.chunk_samples + sidx) * N + k) * SPC + sl] = mm.x;
          sumE += (double)mm.x; sumI += (double)mm.y;
          ++sidx;
        }
        win = mk2(0.0f, 0.0f);
      }
    }
    // chunk m is written: publish it
    __syncwarp();
    if ((tid & 31) == 0) mbar_arrive(bars + (m & (NBAR - 1)));
    n += ch;
    cur += ch; if (cur >= Hp) cur -= Hp;
  }
  if (active) {
    sp[0] = nu.x; sp[stride] = nu.y; sp[2 * stride] = Cs.x; sp[3 * stride] = Cei; sp[4 * stride] = Cs.y;
    sp[5 * stride] = W.x; sp[6 * stride] = W.y; sp[7 * stride] = ou; sp[8 * stride] = win.x; sp[9 * stride] = win.y;
    sump[0] = sumE; sump[stride] = sumI;
  }
}

}  // namespace tvbx
