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
enum { NBAR = 8, NST = 4, LAGMAX = NST };   // mbarrier ring of the consumers, stages of coupling sums
enum { K2_MAXT_SELF = 480, K2_MAXT_DED = 608 };   // threads per CTA: every warp produces (128 registers) / + 4 dedicated producer warps (96)
enum { EB = 16 };       // load rounds a producer warp keeps in flight per region (8-byte loads, 2 registers each)

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

// Gather of one (simulation, region) node for the chunk whose first step sits in ring slot `cur`:
// acc[i] = (c_{2i}, c_{2i+1}), c_i = sum over the row's edges of W_kj E_j(n + i - d_kj).
// EBT edges per iteration: all EBT*GC loads are issued before the first FFMA2 needs one.  Every thread adds its
// row's edges in ascending order, so the sum does not depend on the other simulations of the CTA.
template <int RS, int EBT, typename EdgePtr>
__device__ __forceinline__ void gather_node(EdgePtr edges, int e0, int e1, const float* ringg, int cur, int Hp, int ch,
                                            f2 acc[GC / 2]) {
  constexpr int SPC = RS;                         // simulation columns of a ring slot
  constexpr uint32_t uSPC = (uint32_t)RS;
#pragma unroll
  for (int i = 0; i < GC / 2; ++i) acc[i] = mk2(0.0f, 0.0f);
  if (ch == GC) {
    int e = e0;
    for (; e + EBT <= e1; e += EBT) {
      float w[EBT], v[EBT][GC];
#pragma unroll
      for (int b = 0; b < EBT; ++b) {
        const Edge<float> ed = edges[e + b];
        int start = cur + (int)ed.back;
        start = start >= Hp ? start - Hp : start;
        const float* src = ringg + (ed.jbase + (uint32_t)start * uSPC);
        w[b] = ed.w;
#pragma unroll
        for (int i = 0; i < GC; ++i) v[b][i] = src[i * SPC];
      }
#pragma unroll
      for (int b = 0; b < EBT; ++b)
#pragma unroll
        for (int i = 0; i < GC / 2; ++i) acc[i] = fma2(bc2(w[b]), mk2(v[b][2 * i], v[b][2 * i + 1]), acc[i]);
    }
    for (; e < e1; ++e) {
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
}

// Warp-cooperative gather of one region k for a chunk whose first step sits in ring slot `cur`.
// ring[region][slot][SPCP] keeps the SPCP (power of two >= SPC) simulation columns of a slot together, so the
// GC slots x SPCP simulations one edge needs are 8*SPCP contiguous floats: LPE = 4*SPCP lanes read them with
// ONE 8-byte load each (a fully coalesced 32*SPCP-byte run), and a warp covers EPL = 32/LPE edges per load
// instruction.  Lane l of an edge group holds floats (2l, 2l+1) of the run = (slot, sim pair) for SPCP >= 2,
// (slot pair) for SPCP = 1, so the weighted sum over the row's edges is one FFMA2 per load (P:82:
// c_k = sum_j W_kj E_j(t - d_kj)).  EBT loads are in flight per lane.
// Summation order (the same for every SPCP, so a simulation's result does not depend on how many
// simulations share its CTA): edge e of the row goes to partial sum (e - e0) mod 8; the 8 partial sums are
// added as the binary tree ((P0+P1)+(P2+P3))+((P4+P5)+(P6+P7)) -- across the edge groups by xor shuffles
// (low bits of the class), then inside the lane (high bits).
template <int SPCP, int EBT, typename EdgePtr>
__device__ __forceinline__ f2 gather_region(EdgePtr edges, int e0, int e1, const float* ringb, int cur, int Hp, int lane) {
  constexpr int LPE = 4 * SPCP;                   // lanes per edge
  constexpr int EPL = 32 / LPE;                   // edges per load instruction
  constexpr int NA = 8 / EPL;                     // partial sums per lane (= SPCP)
  static_assert(EBT % NA == 0, "EBT must be a multiple of the partial sums per lane");
  const int grp = lane / LPE, off = 2 * (lane % LPE);
  f2 acc[NA];
#pragma unroll
  for (int a = 0; a < NA; ++a) acc[a] = mk2(0.0f, 0.0f);
  for (int e = e0 + grp; e < e1; e += EPL * EBT) {
    f2 v[EBT];
    float w[EBT];
#pragma unroll
    for (int b = 0; b < EBT; ++b) {
      const int eb = e + b * EPL;
      v[b] = mk2(0.0f, 0.0f); w[b] = 0.0f;
      if (eb < e1) {
        const Edge<float> ed = edges[eb];
        int start = cur + (int)ed.back;
        start = start >= Hp ? start - Hp : start;
        const float* src = ringb + (ed.jbase + (uint32_t)(start * SPCP + off));
        if (SPCP >= 2) v[b] = *reinterpret_cast<const f2*>(src);      // 8-byte aligned: every term is even
        else v[b] = mk2(src[0], src[1]);
        w[b] = ed.w;
      }
    }
#pragma unroll
    for (int b = 0; b < EBT; ++b) acc[b % NA] = fma2(bc2(w[b]), v[b], acc[b % NA]);
  }
#pragma unroll
  for (int o = LPE; o < 32; o <<= 1) {
#pragma unroll
    for (int a = 0; a < NA; ++a) {
      acc[a].x += __shfl_xor_sync(0xffffffffu, acc[a].x, o);
      acc[a].y += __shfl_xor_sync(0xffffffffu, acc[a].y, o);
    }
  }
#pragma unroll
  for (int st = 1; st < NA; st <<= 1)
#pragma unroll
    for (int a = 0; a < NA; a += 2 * st) acc[a] = add2(acc[a], acc[a + st]);
  return acc[0];
}

// SPC: simulations per CTA (1..8, compile time); SPCP = the next power of two = simulation columns of a ring slot.
// blockDim = TC consumer threads (N*SPC rounded up to whole warps) + NPW*32 dedicated producer threads (NPW >= 0).
__host__ __device__ constexpr int spc_pad(int spc) { return spc <= 1 ? 1 : (spc <= 2 ? 2 : (spc <= 4 ? 4 : 8)); }

// MODE: how the coupling sums are gathered
//   K2_THREAD     every thread gathers its own node right before it computes the chunk (ring[region][slot][SPC])
//   K2_WARP       every warp gathers whole regions for the NEXT chunk with coalesced 8-byte loads
//                 (ring[region][slot][SPCP]), then computes the current one
//   K2_DEDICATED  the same warp-cooperative gather by dedicated producer warps
//   K2_PIPE       K2_THREAD software-pipelined: compute step i of chunk m issues the ring loads of edges
//                 [EPS i, EPS (i+1)) of chunk m + 1 before the transfer function and adds them after it, so the
//                 L2/HBM latency of the gather hides behind the thread's own arithmetic
enum { K2_THREAD = 0, K2_WARP = 1, K2_DEDICATED = 2, K2_PIPE = 3 };
enum { EPS = 3 };        // K2_PIPE: edges of the next chunk gathered per compute step
__host__ __device__ constexpr int ring_cols(int spc, int mode) { return (mode == K2_THREAD || mode == K2_PIPE) ? spc : spc_pad(spc); }

template <int SPC, int MODE>
__global__ void __launch_bounds__(MODE == K2_DEDICATED ? K2_MAXT_DED : K2_MAXT_SELF, 1) integrate2_kernel(const __grid_constant__ Integrate2Params P) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  constexpr int SPCP = spc_pad(SPC);
  constexpr int RS = ring_cols(SPC, MODE);        // simulation columns of a ring slot
  const int g = blockIdx.x;
  const int N = P.N;
  const int tid = threadIdx.x;
  const int NODES = N * SPC;
  const int TC = (NODES + 31) & ~31;              // consumer threads
  constexpr bool PRIV = MODE == K2_THREAD || MODE == K2_PIPE;   // every thread gathers its own node
  const int CPLS = PRIV ? TC : N * SPCP + 8;   // row stride of the coupling sums (padded against bank conflicts)
  const int NPT = MODE == K2_DEDICATED ? (int)blockDim.x - TC : 0;   // dedicated producer threads
  constexpr int NSTG = PRIV ? 1 : NST;   // stages of coupling sums / normals (private columns need one)
  const GroupDesc gd = P.groups[g];
  const TableDesc td = P.tables[gd.table];
  const int Hp = td.Hp, Hs = td.Hs, CH = td.CH, LAG = td.LAG;
  const Edge<float>* edges = P.edges + td.edge_off;
  const int32_t* rowptr = P.rowptr + td.rowptr_off;
  // shared memory: NBAR "done" + NST "full" mbarriers | [NST][GC][CPLS] coupling sums | [NST][GC][TC] normals |
  // [NP2][SPC] packed per-sim parameters | optional edge table + row pointers
  uint64_t* bar_done = reinterpret_cast<uint64_t*>(smem_raw);
  uint64_t* bar_full = bar_done + NBAR;
  float* const s_cpl0 = reinterpret_cast<float*>(smem_raw + (NBAR + NST) * 8);
  float* const s_xi0 = s_cpl0 + (size_t)NSTG * GC * CPLS;
  float2* s_ps = reinterpret_cast<float2*>(s_xi0 + (size_t)NSTG * GC * TC);
  Edge<float>* s_edges;
  int32_t* s_rowptr;
  // producing warps: the dedicated ones if the launch has any, else every warp (gather for chunk m + 1, then
  // compute chunk m)
  const int NW_P = NPT > 0 ? NPT >> 5 : TC >> 5;
  const int ptid = NPT > 0 ? tid - TC : tid;      // index among the producing threads (< 0: pure consumer)
  {
    if (tid < NBAR) mbar_init(bar_done + tid, (uint32_t)(TC >> 5));
    else if (tid < NBAR + NST) mbar_init(bar_full + (tid - NBAR), (uint32_t)NW_P);
    for (int i = tid; i < NP2 * SPC; i += blockDim.x) s_ps[i] = P.psim2[(size_t)g * NP2 * SPC + i];
    unsigned char* tab = reinterpret_cast<unsigned char*>(s_ps + NP2 * SPC);
    tab += (16 - (reinterpret_cast<uintptr_t>(tab) & 15)) & 15;
    s_edges = reinterpret_cast<Edge<float>*>(tab);
    s_rowptr = reinterpret_cast<int32_t*>(s_edges + td.n_edges);
    if (P.smem_table) {
      for (int i = tid; i < td.n_edges; i += blockDim.x) s_edges[i] = edges[i];
      for (int i = tid; i <= N; i += blockDim.x) s_rowptr[i] = rowptr[i];
    }
    __syncthreads();
  }
  const bool noise = P.noise_on != 0;

  // ---- produce chunk m (first step n0, ring slot cur0): S1 coupling sums + S4 normals into stage m mod NST ----
  auto produce = [&](uint32_t m, int64_t n0, int cur0) {
    const int ch = (int)min((int64_t)CH, P.n_end - n0);
    // the ring writes of chunk m - LAG (all warps) must be visible before this chunk's gather; LAG <= NST, so
    // the stage written below has also been read by everybody
    if (m >= (uint32_t)LAG) { const uint32_t w = m - (uint32_t)LAG; mbar_wait(bar_done + (w & (NBAR - 1)), (w / NBAR) & 1u); }
    float* const cpl = s_cpl0 + (size_t)(m & (NSTG - 1)) * GC * CPLS;
    float* const sxi = s_xi0 + (size_t)(m & (NSTG - 1)) * GC * TC;
    const int lane = tid & 31;
    if (PRIV) {                                   // S1 + S4 for this thread's own node, private columns of the stage
      const int nd = tid < NODES ? tid : NODES - 1;
      const int rl = nd / SPC, sl = nd - rl * SPC;
      f2 acc[GC / 2];
      if (P.smem_table) gather_node<RS, 4>(s_edges, s_rowptr[rl], s_rowptr[rl + 1], P.ring + gd.ring_off + sl, cur0, Hp, ch, acc);
      else gather_node<RS, 4>(edges, rowptr[rl], rowptr[rl + 1], P.ring + gd.ring_off + sl, cur0, Hp, ch, acc);
#pragma unroll
      for (int i = 0; i < GC / 2; ++i) { cpl[(2 * i) * CPLS + tid] = acc[i].x; cpl[(2 * i + 1) * CPLS + tid] = acc[i].y; }
      if (noise) {
        const uint32_t ext = (uint32_t)P.ext_id[(size_t)g * SPC + sl];
        float xi[4] = {0.f, 0.f, 0.f, 0.f};
        for (int i = 0; i < ch; ++i) {
          const uint64_t nn = (uint64_t)(n0 + i);
          if (i == 0 || (nn & 3) == 0) normals4<float>(P.seed, ext, (uint32_t)rl, nn >> 2, xi);
          const uint32_t q = (uint32_t)nn & 3u;
          sxi[i * TC + tid] = q == 0 ? xi[0] : (q == 1 ? xi[1] : (q == 2 ? xi[2] : xi[3]));
        }
      }
      return;
    }
    for (int k = ptid >> 5; k < N; k += NW_P) {   // S1: one region per warp at a time
      f2 acc;
      if (P.smem_table) acc = gather_region<SPCP, EB>(s_edges, s_rowptr[k], s_rowptr[k + 1], P.ring + gd.ring_off, cur0, Hp, lane);
      else acc = gather_region<SPCP, EB>(edges, rowptr[k], rowptr[k + 1], P.ring + gd.ring_off, cur0, Hp, lane);
      const int f = 2 * lane;                     // float index in the [GC][SPCP] run of this region
      if (f < GC * SPCP) {
        if (SPCP >= 2) *reinterpret_cast<f2*>(cpl + (f / SPCP) * CPLS + k * SPCP + (f % SPCP)) = acc;
        else { cpl[f * CPLS + k] = acc.x; cpl[(f + 1) * CPLS + k] = acc.y; }
      }
    }
    if (noise) {                                  // S4: Philox (A12): one call per (sim, region) per 4 steps
      for (int node = ptid; node < NODES; node += NW_P * 32) {
        const int rl = node / SPC, sl = node - rl * SPC;
        const uint32_t ext = (uint32_t)P.ext_id[(size_t)g * SPC + sl];
        float xi[4] = {0.f, 0.f, 0.f, 0.f};
        for (int i = 0; i < ch; ++i) {
          const uint64_t nn = (uint64_t)(n0 + i);
          if (i == 0 || (nn & 3) == 0) normals4<float>(P.seed, ext, (uint32_t)rl, nn >> 2, xi);
          const uint32_t q = (uint32_t)nn & 3u;
          sxi[i * TC + node] = q == 0 ? xi[0] : (q == 1 ? xi[1] : (q == 2 ? xi[2] : xi[3]));
        }
      }
    }
    __syncwarp();
    if (lane == 0) mbar_arrive(bar_full + (m & (NST - 1)));
  };

  if (tid >= TC) {
    // ============================ dedicated PRODUCER warps ============================
    int64_t n = P.n_begin;
    int cur = (int)(n % Hp);
    for (uint32_t m = 0; n < P.n_end; ++m) {
      produce(m, n, cur);
      const int ch = (int)min((int64_t)CH, P.n_end - n);
      n += ch;
      cur += ch; if (cur >= Hp) cur -= Hp;
    }
    return;
  }
  // without dedicated producers every warp produces: one chunk ahead of its compute when the delays allow
  // it (LAG >= 2), else just before it
  const bool self = MODE != K2_DEDICATED;
  const int LA = ((MODE == K2_WARP || MODE == K2_PIPE) && LAG >= 2) ? 1 : 0;
  if (self && LA && P.n_begin < P.n_end) produce(0, P.n_begin, (int)(P.n_begin % Hp));   // chunk 0 has no predecessor to hide behind

  // ============================ CONSUMER warps: S2, S3, S5, S6 ============================
  const bool active = tid < NODES;                // lanes past the last node replay it, stores suppressed
  const int node = active ? tid : NODES - 1;
  const int k = node / SPC, sl = node - k * SPC;
  s_ps += sl;
  float* const ringg = P.ring + gd.ring_off + sl;
  const uint32_t uSPC = (uint32_t)RS;
  const uint32_t myrow = (uint32_t)(k * Hs) * uSPC;
  const int loc = P.loc_id[(size_t)g * SPC + sl];
  const float dt = P.dt;
  const float inv_ds = P.ds > 0 ? 1.0f / (float)P.ds : 0.0f;
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
  int c = (int)(n % Hp);                          // ring slot of time index n
  int win_left = P.ds > 0 ? P.ds - (int)(n % P.ds) : 0x7fffffff;   // steps left in the current window
  int sidx = P.sample_base;
  const int pe0 = MODE == K2_PIPE ? s_rowptr[k] : 0, pe1 = MODE == K2_PIPE ? s_rowptr[k + 1] : 0;   // this node's row (K2_PIPE)

  for (uint32_t m = 0; n < P.n_end; ++m) {
    const int ch = (int)min((int64_t)CH, P.n_end - n);
    const bool has_next = n + ch < P.n_end;
    const int cur1 = c + ch >= Hp ? c + ch - Hp : c + ch;          // ring slot of the next chunk's first step
    if (self) {
      if (!LA) produce(m, n, c);
      else if (MODE == K2_WARP && has_next) produce(m + 1, n + ch, cur1);
    }
    const bool pipe = MODE == K2_PIPE && LA && has_next;
    if (pipe && m + 1 >= (uint32_t)LAG) { const uint32_t w = m + 1 - (uint32_t)LAG; mbar_wait(bar_done + (w & (NBAR - 1)), (w / NBAR) & 1u); }
    f2 pacc[GC / 2];
#pragma unroll
    for (int j = 0; j < GC / 2; ++j) pacc[j] = mk2(0.0f, 0.0f);
    if (!PRIV) mbar_wait(bar_full + (m & (NST - 1)), (m / NST) & 1u);   // coupling sums and normals of chunk m are in
    const float* const cplp = s_cpl0 + (size_t)(m & (NSTG - 1)) * GC * CPLS + (PRIV ? tid : k * SPCP + sl);
    const float* const xip = s_xi0 + (size_t)(m & (NSTG - 1)) * GC * TC + (PRIV ? tid : node);
    const bool traj_on = P.traj != nullptr && loc >= 0 && active && n - P.traj_n0 < P.traj_steps;
    for (int i = 0; i < ch; ++i) {
      const int64_t nn = n + i;
      const float cpl = cplp[i * CPLS];
      // K2_PIPE: ring loads of edges [EPS i, EPS (i + 1)) of this row for the NEXT chunk, consumed below
      float pv[EPS][GC];
      if (MODE == K2_PIPE) {
#pragma unroll
        for (int b = 0; b < EPS; ++b) {
          const int e = pe0 + EPS * i + b;
          const bool on = pipe && e < pe1;
          const Edge<float> ed = s_edges[on ? e : pe0];
          int start = cur1 + (int)ed.back;
          start = start >= Hp ? start - Hp : start;
          const float* src = ringg + (ed.jbase + (uint32_t)start * uSPC);
#pragma unroll
          for (int j = 0; j < GC; ++j) pv[b][j] = on ? src[j * RS] : 0.0f;
        }
      }
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
      if (noise) ou = __fmaf_rn(P.ou_rho, ou, __fmaf_rn(P.ou_s, xip[i * TC], P.ou_m));
      if (MODE == K2_PIPE) {
#pragma unroll
        for (int b = 0; b < EPS; ++b) {
          const int e = pe0 + EPS * i + b;
          const float w = (pipe && e < pe1) ? s_edges[e].w : 0.0f;
#pragma unroll
          for (int j = 0; j < GC / 2; ++j) pacc[j] = fma2(bc2(w), mk2(pv[b][2 * j], pv[b][2 * j + 1]), pacc[j]);
        }
      }
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
    if (pipe) {       // the row's remaining edges, then the next chunk's sums and normals replace this chunk's
      for (int e = pe0 + EPS * ch; e < pe1; ++e) {
        const Edge<float> ed = s_edges[e];
        int start = cur1 + (int)ed.back;
        start = start >= Hp ? start - Hp : start;
        const float* src = ringg + (ed.jbase + (uint32_t)start * uSPC);
#pragma unroll
        for (int j = 0; j < GC / 2; ++j) pacc[j] = fma2(bc2(ed.w), mk2(src[(2 * j) * RS], src[(2 * j + 1) * RS]), pacc[j]);
      }
      float* const cw = s_cpl0 + tid;
#pragma unroll
      for (int j = 0; j < GC / 2; ++j) { cw[(2 * j) * CPLS] = pacc[j].x; cw[(2 * j + 1) * CPLS] = pacc[j].y; }
      if (noise) {
        const uint32_t ext = (uint32_t)P.ext_id[(size_t)g * SPC + sl];
        const int ch1 = (int)min((int64_t)CH, P.n_end - (n + ch));
        float xi[4] = {0.f, 0.f, 0.f, 0.f};
        for (int i = 0; i < ch1; ++i) {
          const uint64_t nn = (uint64_t)(n + ch + i);
          if (i == 0 || (nn & 3) == 0) normals4<float>(P.seed, ext, (uint32_t)k, nn >> 2, xi);
          const uint32_t q = (uint32_t)nn & 3u;
          s_xi0[i * TC + tid] = q == 0 ? xi[0] : (q == 1 ? xi[1] : (q == 2 ? xi[2] : xi[3]));
        }
      }
    }
    // chunk m is written (and its stage of coupling sums read): publish it
    __syncwarp();
    if ((tid & 31) == 0) mbar_arrive(bar_done + (m & (NBAR - 1)));
    n += ch;
  }
  if (active) {
    sp[0] = nu.x; sp[stride] = nu.y; sp[2 * stride] = Cs.x; sp[3 * stride] = Cei; sp[4 * stride] = Cs.y;
    sp[5 * stride] = W.x; sp[6 * stride] = W.y; sp[7 * stride] = ou; sp[8 * stride] = win.x; sp[9 * stride] = win.y;
    sump[0] = sumE; sump[stride] = sumI;
  }
}

}  // namespace tvbx
