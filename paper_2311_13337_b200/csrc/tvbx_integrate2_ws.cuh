// tvbx_integrate2_ws.cuh -- the LOW-LATENCY form of the packed FP32 integrator for small sweeps and long runs
// (BASELINE.json cfg 4: 256 simulations x 3,000,000 steps, cfg 1: 8 simulations; PAPER.md
// with few work-items per GPU there are too few threads to hide latency).
//
// A sweep of a few hundred simulations offers about ONE warp per warp scheduler (cfg 4: 544 warps of nodes on the 592
// schedulers of a B200), so its throughput is the latency of one warp's Euler step: ~520 dependent-ish instructions, of
// which only ~300 are the model (both transfer functions with their jets, Eqs. (1)-(3)); the rest is the delayed gather for
// the next chunk (table reads, address arithmetic, 24 ring loads and their FMAs per step), the Philox / Box-Muller draws
// and bookkeeping -- and the schedulers sit at a third of their issue slots.  This form splits the two roles over a warp
// PAIR on the idle slots (warp specialisation):
//   consumer warp  = the nodes' state in registers; per step: inputs, transfer functions, Euler, OU, ring write, sample
//   producer warp  = the same 32 nodes (lane for lane); per chunk of <= 8 steps: waits until the ring holds what the chunk
//                    needs, gathers the whole row for its steps, draws the chunk's normals, and leaves both in the pair's
//                    double-buffered shared-memory columns
// Hand-over per pair through two full / empty mbarriers per buffer; the ring dependency across warps through the same
// rolling chunk barriers as integrate2_kernel (a consumer arrives when it has written a chunk, a producer waits for chunk
// m - LAG of all consumers before it gathers chunk m).  Arithmetic, association of the coupling sum (the row's edges in
// ascending order into each slot) and the Philox stream are those of integrate2_kernel: results are bit-identical.
// One CTA per group, delay table in shared memory, chunks of 8 steps (minimum delay >= 15 steps); SRING: the group's ring
// in shared memory for the launch (cfg 1).
//
// GRP (the grouped form, cfg 4): the unit of this form's speed is ONE consumer warp per warp
// scheduler, and no one-CTA mapping of a few hundred simulations gives that (cfg 4: 2 x 68 nodes = 5 warps per SM).  So the
// REGIONS of a group are split over P.grp_ctas CTAs (cfg 4: 7 simulations x 17 regions per CTA, 4 CTAs per group, 148 CTAs
// of 4 pairs).  The CTAs of a group sit on different SMs and wait on one another: cooperative launch (all resident), ring in
// global memory read through L2, chunk hand-over through counters in global memory.  Two helper warps per CTA keep that
// hand-over off the pairs: the publisher (release-add when all local consumers have written a chunk) and the relay (polls
// until every CTA of the group has, then completes the local barrier the producers wait on).  Still bit-identical.
#pragma once
#include "tvbx_integrate2.cuh"

namespace tvbx {

enum { RELAY_POLL_NS = 2400, LAZY_WAIT_NS = 400 };      // GRP relay warp: poll period; producer / publisher warps: sleep between barrier tries
enum { K2_WST = 320 };           // threads per CTA of this form (consumers + producers): 65536 / 320 -> 204 registers per thread

// release-add on / acquire-load of a chunk counter in global memory (GRP: the CTAs of a group sit on different SMs)
__device__ __forceinline__ void grp_arrive(uint32_t* p) {
  asm volatile("red.release.gpu.global.add.u32 [%0], 1;" ::"l"(p) : "memory");
}
__device__ __forceinline__ uint32_t grp_poll_relaxed(const uint32_t* p) {
  uint32_t v;
  asm volatile("ld.relaxed.gpu.global.u32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
  return v;
}
__device__ __forceinline__ uint32_t grp_poll(const uint32_t* p) {
  uint32_t v;
  asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
  return v;
}

// wait of a HELPER-side warp (producer, publisher): between two failed tries the warp sleeps, so that it does not take
// issue slots from the consumer warp on its scheduler (the consumer's own waits stay plain spins)
__device__ __forceinline__ void mbar_wait_lazy(uint64_t* bar, uint32_t parity) {
  uint32_t done;
  for (;;) {
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n"
        "selp.u32 %0, 1, 0, p;\n"
        "}\n" : "=r"(done) : "r"(smem_u32(bar)), "r"(parity) : "memory");
    if (done) break;
    __nanosleep(LAZY_WAIT_NS);
  }
}

template <int SPC, bool SRING, bool GRP = false>
__global__ void __launch_bounds__(K2_WST, 1) integrate2_ws_kernel(const __grid_constant__ Integrate2Params P) {
  static_assert(!(GRP && SRING), "a group's ring is shared by its CTAs: global memory");
  extern __shared__ __align__(16) unsigned char smem_raw[];
  constexpr int RS = SPC;
  // GRP: the regions of a group are split over P.grp_ctas CTAs (any SMs; cooperative launch: all resident); CTA r owns the
  // regions [r NL, (r + 1) NL), NL = ceil(N / grp_ctas)
  const int GR = GRP ? P.grp_ctas : 1;
  const int crank = GRP ? (int)blockIdx.x % GR : 0;
  const int g = (GRP ? (int)blockIdx.x / GR : (int)blockIdx.x) + P.group0;
  const int N = P.N;
  const int NLr = GRP ? (N + GR - 1) / GR : N;
  const int k0 = crank * NLr;
  // GRP: two helper warps behind the pairs (publisher, relay -- see below); blockDim = 2 TC + 64
  const int T = blockDim.x, TC = (GRP ? T - 64 : T) >> 1;  // consumer threads = producer threads (whole warps)
  const int NW = TC >> 5;                                  // warp pairs
  // Which warp plays which role.  Warp w issues on scheduler w mod 4; a consumer carries ~3x the instructions of a producer.
  // Consumers take warps 0 .. 3, one per scheduler; with a fifth pair (cfg 4: 136 nodes) its consumer is warp 6, so that the
  // scheduler hosting two consumers hosts no producer (loads 530 / 530 / 660 / 430 issue slots per step instead of 760 / ...).
  const int w = (int)threadIdx.x >> 5;
  bool prod; int wp;
  if (NW == 5) { prod = !(w < 4 || w == 6); wp = prod ? (w < 6 ? w - 4 : w - 5) : (w < 4 ? w : 4); }
  else { prod = w >= NW; wp = prod ? w - NW : w; }
  const int helper = GRP && w >= 2 * NW ? w - 2 * NW + 1 : 0;      // 1 = publisher, 2 = relay
  if (helper) wp = 0;
  const int tid = wp * 32 + ((int)threadIdx.x & 31);       // node slot: the same for the two warps of a pair
  const int NODES = min(NLr, N - k0) * SPC;
  const GroupDesc gd = P.groups[g];
  const TableDesc td = P.tables[gd.table];
  const int Hp = td.Hp, Hs = td.Hs, CH = td.CH, LAG = td.LAG;
  // shared memory: NBAR chunk barriers | [NW][2] full, [NW][2] empty | 2 x [GC][TC] coupling sums | 2 x [GC][TC] normals |
  // [NP2][SPC] parameters | edge table, row pointers | (SRING) ring
  uint64_t* const bar_done = reinterpret_cast<uint64_t*>(smem_raw);
  uint64_t* const bar_full = bar_done + NBAR + (size_t)wp * 2;
  uint64_t* const bar_empty = bar_done + NBAR + (size_t)NW * 2 + (size_t)wp * 2;
  uint64_t* const bar_grp = bar_done + NBAR + (size_t)NW * 4;      // GRP: NBAR barriers "chunk w is in the ring, group-wide"
  uint64_t* const bar_end = bar_grp + (GRP ? NBAR : 0);
  float* const s_cpl = reinterpret_cast<float*>(bar_end) + tid;       // + b * GC * TC + i * TC
  float* const s_xi = s_cpl + (size_t)2 * GC * TC;
  float2* s_ps = reinterpret_cast<float2*>(reinterpret_cast<float*>(bar_end) + (size_t)4 * GC * TC);
  unsigned char* tab = reinterpret_cast<unsigned char*>(s_ps + NP2 * SPC);
  tab += (16 - (reinterpret_cast<uintptr_t>(tab) & 15)) & 15;
  Edge<float>* const s_edges = reinterpret_cast<Edge<float>*>(tab);
  int32_t* const s_rowptr = reinterpret_cast<int32_t*>(s_edges + td.n_edges);
  const Edge<float>* const g_edges = P.edges + td.edge_off;
  const int32_t* const g_rowptr = P.rowptr + td.rowptr_off;
  float* s_ring = nullptr;
  if (SRING) {
    const size_t off = (size_t)(reinterpret_cast<unsigned char*>(s_rowptr + N + 1) - smem_raw);
    s_ring = reinterpret_cast<float*>(smem_raw + ((off + 15) & ~(size_t)15));
  }
  {
    const int t = (int)threadIdx.x;
    if (t < NBAR) mbar_init(bar_done + t, (uint32_t)NW);
    if (t < NW * 4) mbar_init(bar_done + NBAR + t, 1u);
    if (GRP && t < NBAR) mbar_init(bar_grp + t, 1u);
    for (int i = t; i < NP2 * SPC; i += T) s_ps[i] = P.psim2[(size_t)g * NP2 * SPC + i];
    for (int i = t; i < td.n_edges; i += T) s_edges[i] = g_edges[i];
    for (int i = t; i <= N; i += T) s_rowptr[i] = g_rowptr[i];
    if (SRING) {
      const float* gr = P.ring + gd.ring_off;
      const int nr = N * Hs * RS;
      for (int i = t; i < nr; i += T) s_ring[i] = gr[i];
    }
    __syncthreads();
  }
  const bool noise = P.noise_on != 0;
  const bool active = tid < NODES;
  const int node = active ? tid : NODES - 1;      // lanes past the last node replay it (same values to the same addresses)
  const int kl = node / SPC, sl = node - kl * SPC, k = k0 + kl;
  s_ps += sl;
  float* ringg = (SRING ? s_ring : P.ring + gd.ring_off) + sl;
  if (!SRING) {      // (one register pair, an access is base + 4 * offset: see integrate2_kernel)
    asm volatile("" : "+l"(ringg));
    __builtin_assume(__isGlobal(ringg));
  }
  const int e_last = td.n_edges - 1;
  const int pe0 = s_rowptr[k];
  int pe1 = s_rowptr[k + 1];
  while (pe1 > pe0 && s_edges[pe1 - 1].w == 0.0f) --pe1;      // (the row's zero-weight padding, tvbx_host.h kRowMin, is for the pipelined form)
  const uint32_t ext = (uint32_t)P.ext_id[(size_t)g * SPC + sl];
  uint32_t* const grp_cnt = GRP ? P.grp_cnt + (size_t)g * NBAR : nullptr;
  const int64_t n0 = P.n_begin;
  const int c0 = (int)(n0 % Hp);

  if (helper) {
    // ================= GRP helpers: the chunk hand-over between the CTAs of the group, off the consumers' chain =================
    // publisher: when every local consumer has written chunk m (bar_done), one gpu-scope release-add on the group's counter of
    //            slot m mod NBAR.  (Done by the consumers themselves, the release waits for their stores to reach L2 -- about
    //            a microsecond per chunk on the chain that bounds the form.)
    // relay:     polls that counter (relaxed loads, no L1 invalidation per poll) until all grp_arrivals CTAs have published
    //            chunk w of this launch, takes one acquire, and completes the local barrier bar_grp the producers wait on.
    // Causality: consumer stores -> arrive (release.cta) -> publisher wait (acquire.cta) -> red.release.gpu -> relay
    // ld.acquire.gpu -> arrive (release.cta) -> producer wait (acquire.cta) -> ring loads through L2.
    int64_t n = n0;
    for (uint32_t m = 0; n < P.n_end; ++m, n += CH) {
      const uint32_t slot = m & (NBAR - 1);
      if (helper == 1) {
        mbar_wait_lazy(bar_done + slot, (m / NBAR) & 1u);
        if ((threadIdx.x & 31) == 0) grp_arrive(grp_cnt + slot);
      } else {
        const uint32_t want = (uint32_t)P.grp_arrivals * (m / NBAR + 1u);
        if ((threadIdx.x & 31) == 0) {
          // A slow poll, on purpose.  Measured on cfg 4 (chunk time of a consumer 4.9 us): spinning 2.84e10; a poll every
          // 0.2 / 0.8 / 1.6 / 2.4 / 3.2 / 6.4 us -> 2.86 / 2.96 / 3.03 / 3.05 / 3.05 / 2.51e10.  Polling fast and then holding
          // the hand-over back by 1.5 or 3 us gives 3.00e10 as well, sleeping first and then polling fast 2.86e10: what pays is
          // that the producers start their gather LATER inside the LAG - 1 >= 1 chunks of slack they have (their loads and
          // Philox draws then overlap the second half of the consumers' chunk instead of its start), not the saved issue
          // slots.  The period must stay below the chunk time (8 steps of one consumer warp, ~0.5 us each in this form).
          while (grp_poll_relaxed(grp_cnt + slot) < want) __nanosleep(RELAY_POLL_NS);
          (void)grp_poll(grp_cnt + slot);
          mbar_arrive(bar_grp + slot);
        }
        __syncwarp();
      }
    }
  } else if (prod) {
    // ================= producer: coupling sums and normals of chunk m into buffer m & 1 =================
    int64_t n = n0;
    int c = c0;
    for (uint32_t m = 0; n < P.n_end; ++m) {
      const int ch = (int)min((int64_t)CH, P.n_end - n);
      const uint32_t b = m & 1u;
      // Gather and draw FIRST, into registers, as soon as the ring holds what chunk m needs -- up to LAG chunks ahead of the
      // consumer; only the hand-over waits for the buffer.  (Waiting for the buffer first left the producer one chunk-time
      // for all of it, too little once the ring loads cross to another SM's writes through L2: GRP.)
      if (m >= (uint32_t)LAG) {                   // every consumer of the group has written chunk m - LAG
        const uint32_t w = m - (uint32_t)LAG;
        mbar_wait_lazy((GRP ? bar_grp : bar_done) + (w & (NBAR - 1)), (w / NBAR) & 1u);      // (GRP: signalled by the relay warp)
      }
      f2 acc[GC / 2];
#pragma unroll
      for (int j = 0; j < GC / 2; ++j) acc[j] = mk2(0.0f, 0.0f);
      gather_rounds<RS, GC, GRP>(s_edges, pe0, pe1, e_last, ringg, c, Hp, acc);     // the row's edges in ascending order (GRP: through L2)
      float xv[GC];
#pragma unroll
      for (int i = 0; i < GC; ++i) xv[i] = 0.0f;
      if (noise) {                                // A12: one Philox call per (sim, region) per 4 steps
        float xi[4] = {0.f, 0.f, 0.f, 0.f};
        if (ch == GC && (n & 3) == 0) {           // a whole chunk on a quad boundary: two calls
#pragma unroll
          for (int h = 0; h < GC / 4; ++h) {
            normals4<float>(P.seed, ext, (uint32_t)k, ((uint64_t)n >> 2) + (uint64_t)h, xi);
#pragma unroll
            for (int q = 0; q < 4; ++q) xv[4 * h + q] = xi[q];
          }
        } else {
#pragma unroll
          for (int i = 0; i < GC; ++i) {
            if (i < ch) {
              const uint64_t nn = (uint64_t)(n + i);
              if (i == 0 || (nn & 3) == 0) normals4<float>(P.seed, ext, (uint32_t)k, nn >> 2, xi);
              const uint32_t q = (uint32_t)nn & 3u;
              xv[i] = q == 0 ? xi[0] : (q == 1 ? xi[1] : (q == 2 ? xi[2] : xi[3]));
            }
          }
        }
      }
      if (m >= 2) mbar_wait_lazy(bar_empty + b, ((m >> 1) - 1u) & 1u);                  // the consumer has finished chunk m - 2
      float* const cpl = s_cpl + (size_t)b * GC * TC;
#pragma unroll
      for (int j = 0; j < GC / 2; ++j) { cpl[(2 * j) * TC] = acc[j].x; cpl[(2 * j + 1) * TC] = acc[j].y; }
      if (noise) {
        float* const xo = s_xi + (size_t)b * GC * TC;
#pragma unroll
        for (int i = 0; i < GC; ++i) xo[i * TC] = xv[i];
      }
      __syncwarp();
      if ((tid & 31) == 0) mbar_arrive(bar_full + b);
      n += ch;
      c += ch; if (c >= Hp) c -= Hp;
    }
  } else {
    // ================= consumer: the nodes' state in registers, one Euler step after the other =================
    f2 ps_reg[NP2];
#pragma unroll
    for (int q = 0; q < NP2; ++q) ps_reg[q] = s_ps[q * SPC];
    auto par = [&](int q) -> f2 { return ps_reg[q]; };
    const uint32_t myrow = (uint32_t)(k * Hs) * (uint32_t)RS;
    const int loc = P.loc_id[(size_t)g * SPC + sl];
    const float dt = P.dt;
    const float inv_ds = P.ds > 0 ? 1.0f / (float)P.ds : 0.0f;
    const f2 invN = mk2(P.inv_Ne, P.inv_Ni);
    const size_t stride = (size_t)N * SPC;
    float* const sp = P.state + (size_t)g * (NSV - 2) * stride + (size_t)k * SPC + sl;
    double* const sump = P.sums + (size_t)g * 2 * stride + (size_t)k * SPC + sl;
    f2 nu = mk2(sp[0], sp[stride]), Cs = mk2(sp[2 * stride], sp[4 * stride]), W = mk2(sp[5 * stride], sp[6 * stride]);
    f2 win = mk2(sp[8 * stride], sp[9 * stride]);
    float Cei = sp[3 * stride], ou = sp[7 * stride];
    double sumE = sump[0], sumI = sump[stride];
    int64_t n = n0;
    int c = c0;
    int win_left = P.ds > 0 ? P.ds - (int)(n % P.ds) : 0x7fffffff;
    int sidx = P.sample_base;
    for (uint32_t m = 0; n < P.n_end; ++m) {
      const int ch = (int)min((int64_t)CH, P.n_end - n);
      const uint32_t b = m & 1u;
      const int64_t t_rel = n - P.traj_n0;
      const bool traj_any = P.traj != nullptr && t_rel < P.traj_steps;             // (uniform: one branch around the per-lane test)
      const bool traj_on = traj_any && loc >= 0 && active;
      const int traj_left = traj_on ? (int)min(P.traj_steps - t_rel, (int64_t)GC) : 0;
      float* const traj0 = traj_on ? P.traj + (((size_t)loc * P.traj_steps + (size_t)t_rel) * 7) * N + k : nullptr;
      const int keep_from = (int)max((int64_t)-1, min(P.discard_steps - n, (int64_t)GC));
      mbar_wait(bar_full + b, (m >> 1) & 1u);                                      // the pair's producer has filled buffer b
      const float* cpl_p = s_cpl + (size_t)b * GC * TC;      // running pointers into the thread's private columns
      const float* xi_p = s_xi + (size_t)b * GC * TC;
#pragma unroll 2
      for (int i = 0; i < ch; ++i) {
        const float cpl = *cpl_p;
        cpl_p += TC;
        node_step2(P, par, cpl, noise, dt, invN, nu, Cs, W, Cei, ou);
        if (noise) ou = __fmaf_rn(P.ou_rho, ou, __fmaf_rn(P.ou_s, *xi_p, P.ou_m));      // S4 (Eq. 4, A11)
        xi_p += TC;
        // S5 ring write: E at the next time index (the first GC - 1 slots are mirrored behind the period)
        c = c + 1 == Hp ? 0 : c + 1;
        {
          const uint32_t o = myrow + (uint32_t)c * (uint32_t)RS;
          ringg[o] = nu.x;
          if (c < GC - 1) ringg[o + (uint32_t)Hp * (uint32_t)RS] = nu.x;
        }
        if (traj_any && i < traj_left) {
          float* t = traj0 + (size_t)i * 7 * N;
          t[0] = nu.x; t[N] = nu.y; t[2 * N] = Cs.x; t[3 * N] = Cei; t[4 * N] = Cs.y; t[5 * N] = W.x; t[6 * N] = W.y;
        }
        // S6 temporal average (A17)
        win = add2(win, nu);
        if (--win_left == 0) {
          win_left = P.ds;
          if (i >= keep_from) {
            const f2 mm = scl2(inv_ds, win);
            P.xbar[(((size_t)g * P.chunk_samples + sidx) * N + k) * SPC + sl] = mm.x;
            sumE += (double)mm.x; sumI += (double)mm.y;
            ++sidx;
          }
          win = mk2(0.0f, 0.0f);
        }
      }
      __syncwarp();
      if ((tid & 31) == 0) {
        mbar_arrive(bar_done + (m & (NBAR - 1)));      // chunk m is in the ring (GRP: the publisher warp tells the other SMs)
        mbar_arrive(bar_empty + b);                    // buffer b may be refilled
      }
      n += ch;
    }
    if (active) {
      sp[0] = nu.x; sp[stride] = nu.y; sp[2 * stride] = Cs.x; sp[3 * stride] = Cei; sp[4 * stride] = Cs.y;
      sp[5 * stride] = W.x; sp[6 * stride] = W.y; sp[7 * stride] = ou; sp[8 * stride] = win.x; sp[9 * stride] = win.y;
      sump[0] = sumE; sump[stride] = sumI;
    }
  }
  if (SRING) {                                    // the ring goes back to global memory for the next launch
    __syncthreads();
    float* gr = P.ring + gd.ring_off;
    const int nr = N * Hs * RS;
    for (int i = (int)threadIdx.x; i < nr; i += T) gr[i] = s_ring[i];
  }
}

}  // namespace tvbx
