// tvbx_integrate2.cuh -- the FP32 product integrator (closed-form transfer function, tau_e == tau_i):
// delayed gather + coupling sum (S1), both transfer functions with derivatives (S2), Euler update of
// the 7 state variables (S3), OU noise from in-kernel Philox4x32-10 (S4), history-ring write (S5),
// temporal-average downsample (S6) and the running sums for the mean rates.  DESIGN.md section 6.2.
//
// Mapping (B200-first; the paper's kernel is one thread per whole simulation):
//   CTA     = one "group" of SPC <= 8 simulations that share a delay table (same speed v), all N regions,
//             persistent over the time steps of a launch
//   thread  = one (simulation, region) node.  Its excitatory and inhibitory population live in the two
//             halves of packed FP32 pairs (float2: .x = e, .y = i) and are advanced by Blackwell's two-wide
//             FP32 instructions (FFMA2 / FMUL2 / FADD2): the two transfer functions are the same
//             formulas on different constants, so one instruction stream serves both (tvbx_tf2.cuh).
//   ring    = ring[group][region][slot][sim] (E only, "temporal buffer"): the simulations of a group
//             are the fastest index, so the lanes that share a region read one contiguous run per
//             (edge, step).  Rows carry GC-1 mirror slots so that a chunk of GC reads never wraps.
//   time    = chunks of CH = clamp((d_min + 1)/2, 1, GC) steps.  Step n reads E only at times <= n - d_min,
//             so the gather of chunk m needs the ring writes of chunks <= m - LAG of ALL warps,
//             LAG = ceil((d_min + 2)/CH) - 1 (>= 2 unless d_min = 0).  There is no CTA-wide barrier: the
//             warps run a ROLLING pipeline on a ring of 8 shared-memory mbarriers -- a warp arrives
//             (release) on barrier m mod 8 when it has written chunk m and waits (acquire) for phase
//             m + 1 - LAG before it touches the ring for chunk m + 1, so it may run ahead of the slowest
//             warp and nobody idles at a block boundary.
//   gather  = software-pipelined into the compute loop: step i of chunk m issues the ring loads of the next
//             PVN / GCE edges of the thread's row for chunk m + 1 (GCE slots each) BEFORE the transfer function and
//             adds them (FFMA2 on slot pairs) AFTER it, so the L2/HBM latency of the gather hides behind
//             the thread's own ~500 instructions of arithmetic; a CTA has only ~4 warps per scheduler
//             (the sweep's parallelism is sims x regions), too few to hide it by switching warps.
//             The sums of chunk m + 1 replace those of chunk m in the thread's private shared-memory column
//             when chunk m is done.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include "tvbx_integrate.cuh"
#include "tvbx_tf2.cuh"

namespace tvbx {

enum { NP2 = 9 };       // packed per-simulation parameters, see P2_*
enum { P2_GW = 0, P2_IT, P2_B, P2_AT, P2_ITW, P2_ATEL, P2_GLEL, P2_CFE, P2_CFI };   // P2_IT = (1/T, dt/T)
enum { NBAR = 8, LAGMAX = 4 };   // mbarrier ring; chunks a warp may run ahead
enum { K2_MAXT = 480 };          // threads per CTA: 65536 / 480 -> 128 registers per thread (rounded down from 136)
enum { K2_SMALLT = 224 };        // small CTAs: launch bound 224 -> 255 registers per thread
enum { PVN = 24 };               // ring values of the next chunk a thread keeps in flight across one compute step:
                                 // PVN / GCE edges x the first GCE = 8, 4 or 2 slots (GCE >= the chunk length).  Rows up to
                                 // (PVN / GCE) * CH edges are fully pipelined; longer rows finish in rounds of 8 edges.
                                 // The host pads every row of a packed-kernel table to >= PVN entries (tvbx_host.h kRowMin).

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
  const int32_t* seg;             // VEC tables: [N][8] ends of the 7 segments of a row (class 0, classes 1-3 shifted, classes 1-3 near; TableDesc::seg_off)
  const float2* psim2;            // [group][NP2][SPC]
  const int32_t* ext_id;          // [group][SPC]  external sim index (Philox counter)
  const int32_t* loc_id;          // [group][SPC]  local sim index (row of traj), -1 = padding lane
  float* ring;                    // [group][N][Hs][SPC]
  float* state;                   // [group][NSV-2][N][SPC]
  double* sums;                   // [group][2][N][SPC]
  float* xbar;                    // [group][CS][N][SPC]
  float* xbar_i;                  // the same for the inhibitory population (ISAMP instances), else null
  float* traj;                    // optional [n_sims][traj_steps][7][N]
  int64_t traj_steps;
  int64_t traj_n0;
  int32_t smem_table;             // edge table + row pointers staged in shared memory (else read through L1/L2)
  int32_t group0;                 // first group of this launch (groups of one launch share GCE)
  // grouped low-latency form (tvbx_integrate2_ws.cuh, GRP): CTAs per group, consumer warps per group (= arrivals per
  // chunk), and the chunk counters [group][NBAR] in global memory (zeroed before every launch)
  int32_t grp_ctas, grp_arrivals;
  uint32_t* grp_cnt;
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

// ---- thread-block cluster forms (CLU): the regions of a group are split over the CTAs of a cluster; the ring
// lives in global memory, only the chunk hand-over crosses CTAs: a warp arrives (release.cluster) on the barrier
// of EVERY CTA of its cluster through distributed shared memory and waits (acquire.cluster) on its own CTA's.
__device__ __forceinline__ uint32_t cluster_ctarank() { uint32_t r; asm volatile("mov.u32 %0, %%cluster_ctarank;" : "=r"(r)); return r; }
__device__ __forceinline__ uint32_t cluster_nctarank() { uint32_t r; asm volatile("mov.u32 %0, %%cluster_nctarank;" : "=r"(r)); return r; }
__device__ __forceinline__ void cluster_sync_all() {
  asm volatile("barrier.cluster.arrive.release.aligned;\n\tbarrier.cluster.wait.acquire.aligned;" ::: "memory");
}
// one release fence, then a relaxed arrive per CTA of the cluster (fence + relaxed write = release pattern)
__device__ __forceinline__ void mbar_arrive_cluster(uint64_t* bar, uint32_t nrank) {
  const uint32_t local = smem_u32(bar);
  asm volatile("fence.acq_rel.cluster;" ::: "memory");
  for (uint32_t r = 0; r < nrank; ++r) {
    uint32_t remote;
    asm volatile("mapa.shared::cluster.u32 %0, %1, %2;" : "=r"(remote) : "r"(local), "r"(r));
    asm volatile("mbarrier.arrive.relaxed.cluster.shared::cluster.b64 _, [%0];" ::"r"(remote) : "memory");
  }
}
// spin relaxed, then observe the completed phase once with acquire semantics (the acquire form invalidates the
// L1 -- CCTL.IVALL -- on every poll)
__device__ __forceinline__ void mbar_wait_cluster(uint64_t* bar, uint32_t parity) {
  asm volatile(
      "{\n"
      ".reg .pred p;\n"
      "WAITC_%=:\n"
      "mbarrier.try_wait.parity.relaxed.cluster.shared::cta.b64 p, [%0], %1;\n"
      "@p bra ACQC_%=;\n"
      "bra WAITC_%=;\n"
      "ACQC_%=:\n"
      "mbarrier.try_wait.parity.acquire.cluster.shared::cta.b64 p, [%0], %1;\n"
      "@p bra DONEC_%=;\n"
      "bra ACQC_%=;\n"
      "DONEC_%=:\n"
      "}\n" ::"r"(smem_u32(bar)), "r"(parity)
      : "memory");
}
// ring load: CG = through L2 only (cluster form: the line may have been written by another SM since this SM's L1
// last saw it, and with 8 simulations per slot every 32-byte sector is consumed by one instruction anyway)
template <bool CG>
__device__ __forceinline__ float ring_ld(const float* p) { return CG ? __ldcg(p) : *p; }

// One batch of EBT edges [e, e + EBT) of a row for the chunk whose first step sits in ring slot `cur`: issue the
// ring loads of the first GCE slots of every edge (GCE = 2, 4 or 8 >= the chunk length) and return the values in
// v[EBT * GCE].  The loads are unconditional: a batch may run past the row (or past the CH slots a short chunk
// uses) -- it then reads other valid ring entries (the table index is clamped to e_last, rows are GC-1 mirror
// slots longer than the period) whose weight gather_add sets to zero.  The caller adds them with gather_add --
// later, when it wants the latency hidden.
// PADDED: the caller knows that the entries [e, e + EBT) exist (the pipelined batches of a chunk: the host pads every
// row of a packed-kernel table to >= K2_ROWMIN = 3 GC entries with zero weights), so the index needs no clamp.
template <int RS, int EBT, int GCE, bool CG, bool PADDED = false, typename EdgePtr>
__device__ __forceinline__ void gather_issue(EdgePtr edges, int e, int e_last, const float* ringg, int cur, int Hp, float* v) {
  // slot of the first read = (cur + back) mod Hp with back = Hp - d in [0, Hp]: wraps iff back >= Hp - cur.
  // The table stores pad = jbase + back * RS, so the element offset is pad + cur * RS - (wrap ? Hp * RS : 0).
  const uint32_t thr = (uint32_t)(Hp - cur), curRS = (uint32_t)cur * (uint32_t)RS, curRSw = curRS - (uint32_t)Hp * (uint32_t)RS;
#pragma unroll
  for (int b = 0; b < EBT; ++b) {
    const Edge<float> ed = edges[PADDED ? e + b : min(e + b, e_last)];
    const uint32_t off = ed.pad + (ed.back >= thr ? curRSw : curRS);      // (one select between two uniform values)
    const float* src = ringg + off;
#pragma unroll
    for (int j = 0; j < GCE; ++j) v[b * GCE + j] = ring_ld<CG>(src + j * RS);
  }
}
// acc[j] += w * (E(slot 2j), E(slot 2j+1)), j < GCE/2: the row's edges are added in ascending order into each
// slot, so a simulation's coupling sum does not depend on which other simulations share its CTA
// (PADDED: entries past the row's last edge carry zero weights themselves -- no test)
template <int EBT, int GCE, bool PADDED = false, typename EdgePtr>
__device__ __forceinline__ void gather_add(EdgePtr edges, int e, int e1, bool enable, const float* v, f2 acc[GC / 2]) {
#pragma unroll
  for (int b = 0; b < EBT; ++b) {
    const float w = PADDED ? edges[e + b].w : ((enable && e + b < e1) ? edges[e + b].w : 0.0f);
#pragma unroll
    for (int j = 0; j < GCE / 2; ++j) acc[j] = fma2(bc2(w), mk2(v[b * GCE + 2 * j], v[b * GCE + 2 * j + 1]), acc[j]);
  }
}
// the edges [e, e1) of a row in unpipelined rounds of 8 edges
template <int RS, int GCE, bool CG, typename EdgePtr>
__device__ __forceinline__ void gather_rounds(EdgePtr edges, int e, int e1, int e_last, const float* ringg, int cur, int Hp,
                                              f2 acc[GC / 2]) {
  for (; e < e1; e += 8) {
    float v[8 * GCE];
    gather_issue<RS, 8, GCE, CG>(edges, e, e_last, ringg, cur, Hp, v);
    gather_add<8, GCE>(edges, e, e1, true, v, acc);
  }
}

// ---- vector form of the gather (VEC: cluster kernels whose chunk length is GC = 8) ---------------------------
// Ring layout ring[group][region][slot / 4][sim][slot % 4] (Hp a multiple of 4, 8 mirror slots): the four
// consecutive time slots of a quad sit in one 16-byte word per simulation, so the 8 lanes that share a region fetch
// whole 128-byte lines with one LDG.128 each -- one L2 request per line instead of one per sector (the scalar cluster
// form is bound by the L1->XBAR request rate).  Chunks start at multiples of GC, so the alignment of an edge's 8-slot
// window inside its first quad, A = (Hp - d) mod 4, never changes, and the host sorts every row by it.
//
// SHIFTED WINDOWS.  An unaligned window (A != 0) spans three quads -- 48 bytes fetched for 32 used, and the gather
// of N = 360 is bound by exactly those bytes (L2 -> SM path saturated).  So an edge of class A
// fetches the TWO ALIGNED quads that start sh = (4 - A) mod 4 slots later: they hold its values for steps sh .. 7 of
// the chunk being gathered and for steps 0 .. sh - 1 of the chunk after it.  Every thread therefore keeps TWO rows
// of coupling sums in shared memory (16 slots, the 8-step block's parity selects the row): the gather for block b + 1
// completes block b + 1's slots (whose first sh_max = 3 slots hold partial sums from the previous gather) and leaves
// partial sums in the first three slots of block b + 2.  Reading sh slots further ahead needs the delay to be at
// least 8 LAG - 1 + sh steps; the few edges closer than that ("near": cfg 5 has 0.1 % of them) keep the
// unshifted three-quad window.  A row is stored as 7 segments: class 0 | classes 1, 2, 3 shifted | classes 1, 2, 3
// near, each padded to whole rounds of VR entries with zero-weight copies of its last edge (no clamps, no masks).
// Per slot j of a block the association is: the shifted classes with sh > j in class order (previous gather), then
// class 0 and the shifted classes with sh <= j in class order, then the near classes; inside a class the row's edges
// in ascending order.  gather_head_vec reproduces it with scalar loads for the first chunk of a launch.
enum { VR = 4 };                 // edges per round of the vector gather (segments are padded to multiples of it)
constexpr uint32_t VW = 4;                          // slots per ring word (a pair layout with LDG.64 was measured 4 % slower)
constexpr uint32_t VWS = 2;                         // log2
struct VecLd { typedef float4 word; };
// acc += w * (the 4 slots of word q): acc holds f2 pairs of consecutive slots
__device__ __forceinline__ void vec_fma(f2* acc, int i, float w, const VecLd::word& q) {
  acc[2 * i] = fma2(bc2(w), mk2(q.x, q.y), acc[2 * i]);
  acc[2 * i + 1] = fma2(bc2(w), mk2(q.z, q.w), acc[2 * i + 1]);
}
// 8-byte table entry of the vector kernels: w and, in one word, the word index Q = j * Hs/VW + back/VW in the low 20 bits
// and back/VW in the high 12 (back = Hp - d, plus the shift of a shifted class): half the shared memory of the 16-byte
// entries, which leaves the L1 the room it needs as landing space for the loads in flight.
struct __align__(8) Edge8 { float w; uint32_t qb; };
__device__ __forceinline__ Edge8 edge8_of(const Edge<float>& ed, uint32_t qdiv) {
  Edge8 e8;
  e8.w = ed.w; e8.qb = (ed.pad / qdiv) | ((ed.back >> VWS) << 20);
  return e8;
}
// One segment of a row: edges [e, e1) (whole rounds of VR), NQ aligned quads per edge from the entry's word index on;
// the products are accumulated unshifted over the NQ * 4 fetched slots in acc (NQ * 2 pairs).  get(e) -> Edge8.
template <int RS, int NQ, int NE, typename Get>
__device__ __forceinline__ void gather_round_vec(Get get, int e, const VecLd::word* ringw, uint32_t cur4, uint32_t thr4, uint32_t curW4, f2* acc) {
  VecLd::word q[NE][NQ];
  float w[NE];
#pragma unroll
  for (int b = 0; b < NE; ++b) {
    const Edge8 ed = get(e + b);
    const uint32_t idx = (ed.qb & 0xFFFFFu) + ((ed.qb >> 20) >= thr4 ? curW4 : cur4);
    const VecLd::word* src = ringw + (size_t)idx * RS;
#pragma unroll
    for (int i = 0; i < NQ; ++i) q[b][i] = __ldcg(src + i * RS);
    w[b] = ed.w;
  }
#pragma unroll
  for (int b = 0; b < NE; ++b) {
#pragma unroll
    for (int i = 0; i < NQ; ++i) vec_fma(acc, i, w[b], q[b][i]);
  }
}
// (two-quad segments run rounds of 2 VR edges while they last -- 16 LDG.128 in flight per thread: with 10 the gather fell
// from 10.4 to 6.4 TB/s on the L2 -> SM path -- then one round of VR)
template <int RS, int NQ, typename Get>
__device__ __forceinline__ void gather_seg_vec(Get get, int e, int e1, const VecLd::word* ringw, uint32_t cur4, uint32_t thr4,
                                               uint32_t curW4, f2* acc) {
#pragma unroll
  for (int i = 0; i < NQ * 2; ++i) acc[i] = mk2(0.0f, 0.0f);
  if (NQ == 2)
    for (; e + 2 * VR <= e1; e += 2 * VR) gather_round_vec<RS, NQ, 2 * VR>(get, e, ringw, cur4, thr4, curW4, acc);
  for (; e < e1; e += VR) gather_round_vec<RS, NQ, VR>(get, e, ringw, cur4, thr4, curW4, acc);
}
__device__ __forceinline__ float acc_slot(const f2* acc, int t) { return (t & 1) ? acc[t >> 1].y : acc[t >> 1].x; }

// S2 + S3 of one (simulation, region) node: the inputs of Eq. (5) (A5, A6, A10), both transfer functions with first
// and second derivatives (tf_closed2), Eqs. (1)-(3) (A7, A9, A22) and the forward-Euler update of
// nu = (E, I), Cs = (C_ee, C_ii), C_ei, W = (W_e, W_i).  cpl = the delayed coupling sum of this step, ou = the OU state
// (not advanced here); par(q) = the node's packed per-simulation parameter q (P2_*).  Shared by every form of the kernel.
template <typename ParF>
__device__ __forceinline__ void node_step2(const Integrate2Params& P, ParF par, float cpl, bool noise, float dt, f2 invN,
                                           f2& nu, f2& Cs, f2& W, float& Cei, float ou) {
  // ---- S2 inputs (Eq. 5; A5, A6, A10) ----
  const f2 gw = par(P2_GW);
  float drive = __fmaf_rn(gw.x, cpl, nu.x);
  if (noise) drive = __fmaf_rn(gw.y, ou, drive);
  const f2 xe = add2(bc2(drive), par(P2_CFE));
  const f2 xi_ = add2(bc2(nu.y), par(P2_CFI));
  const f2 se = mk2(xe.x > 0.0f ? P.kappa : 0.0f, xe.y > 0.0f ? P.kappa : 0.0f);      // A22 and the clamp of A10
  const f2 si = mk2(xi_.x > 0.0f ? P.kappa : 0.0f, xi_.y > 0.0f ? P.kappa : 0.0f);
  const f2 fe = add2(mk2(fmaxf(xe.x, 0.0f), fmaxf(xe.y, 0.0f)), bc2(P.tf.eps));
  const f2 fi = add2(mk2(fmaxf(xi_.x, 0.0f), fmaxf(xi_.y, 0.0f)), bc2(P.tf.eps));
  const f2 c0 = sub2(par(P2_GLEL), W);
  f2 muV;
  const Jet2 F = tf_closed2(P.tf, fe, fi, c0, &muV);
  if (P.muV_local) {                          // A9b alternative: mu_V of the local rates only
    const float le = fmaxf(nu.x, 0.0f) + P.tf.eps, li = fmaxf(nu.y, 0.0f) + P.tf.eps;
    const float den = __fmaf_rn(P.tf.ae, le, __fmaf_rn(P.tf.ai, li, P.tf.gL));
    const float base = __fmaf_rn(P.tf.aeEe, le, P.tf.aiEi * li);
    muV = mk2((base + c0.x) / den, (base + c0.y) / den);
  }
  // ---- S3 Eqs. (1)-(3), forward Euler (A7, A9) ----
  const f2 itp = par(P2_IT);                  // (1/T, dt/T)
  const f2 IT = bc2(itp.x), DT = bc2(itp.y);
  const f2 Fe = mul2(F.e, se), Fi = mul2(F.i, si);
  const f2 dF = sub2(F.v, nu);
  f2 a2nd = fma2(bc2(0.5f * Cs.x), mul2(F.ee, mul2(se, se)), dF);
  a2nd = fma2(bc2(Cei), mul2(F.ei, mul2(se, si)), a2nd);
  a2nd = fma2(bc2(0.5f * Cs.y), mul2(F.ii, mul2(si, si)), a2nd);
  const f2 Ca = mk2(Cs.x, Cei), Cb = mk2(Cei, Cs.y);            // row mu of the covariance matrix
  const f2 gC = fma2(Ca, Fe, fms2(Cb, Fi, Cs));                 // (C dF/dnu)_mu,mu - C_mu,mu
  const f2 dCs = fma2(mul2(F.v, sub2(IT, F.v)), invN, fma2(dF, dF, add2(gC, gC)));     // T dC/dt
  const f2 Co = mk2(Cei, Cs.x), Cp = mk2(Cs.y, Cei);            // the other row
  const f2 h2 = fma2(Co, Fe, mul2(Cp, Fi));
  const float dCei = __fmaf_rn(dF.x, dF.y, (h2.x + h2.y) - 2.0f * Cei);                 // T dC_ei/dt
  const f2 dW = fma2(par(P2_AT), muV, fms2(par(P2_B), nu, fma2(W, par(P2_ITW), par(P2_ATEL))));
  nu = fma2(DT, a2nd, nu);                    // y <- y + (dt / T) (T dy/dt)
  Cs = fma2(DT, dCs, Cs);
  Cei = __fmaf_rn(itp.y, dCei, Cei);
  W = fma2(bc2(dt), dW, W);
}

// SPC: simulations per CTA (1..8); SMEMTAB: the delay table of the group's speed is staged in shared memory;
// GCE: ring slots loaded per edge = 2, 4 or 8 >= the chunk length CH of the launched groups (P.group0 ...); 1 = the one-step
// form (with SRING; see gather_short).
// CLU: the group is integrated by a thread-block cluster; CTA r of the cluster owns the regions [r*NL, (r+1)*NL), NL =
// ceil(N / cluster size) (N = 360: 6 CTAs x 60 regions x 8 simulations -- lanes that share a region then read whole
// 32-byte sectors of the ring, which a single CTA of <= 480 threads cannot offer at N = 360).
// blockDim = (regions of the CTA)*SPC rounded up to whole warps (<= K2_MAXT); lanes past the last node replay it,
// stores suppressed.
// VEC (with CLU, GCE == 8): quad ring layout and vector gather, see gather_class_vec.
// SRING (short delays: the group's whole ring fits next to the table): the ring lives in SHARED memory for the
// launch -- copied in at the start, back at the end (resumable) -- so the per-chunk gathers that a short minimum
// delay leaves unpipelined (rows longer than PVN / GCE edges, every step when CH = 1) cost a shared-memory
// round trip instead of an L2 one (cfg 3, v >= 32 m/s).
// MAXT: the launch bound.  K2_MAXT = 480 threads leaves 128 registers per thread; CTAs of <= K2_SMALLT = 224 threads
// (small sweeps, few regions) are compiled with the bound 224 -> up to 255 registers (190 used): the scheduler of a
// CTA that has one or two warps per scheduler lives on the instruction-level parallelism the extra registers allow
// (cfg 4 +11 %, cfg 1 +14 %).
// ISAMP: the inhibitory 1-ms samples are stored as well (rate statistics of both populations, tvbx_rate_stats).
template <int SPC, bool SMEMTAB, int GCE, bool CLU, bool VEC = false, bool SRING = false, int MAXT = K2_MAXT, bool ISAMP = false>
__global__ void __launch_bounds__(MAXT, 1) integrate2_kernel(const __grid_constant__ Integrate2Params P) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  constexpr int RS = SPC;                         // simulation columns of a ring slot
  const uint32_t nrank = CLU ? cluster_nctarank() : 1u, crank = CLU ? cluster_ctarank() : 0u;
  const int g = (CLU ? (int)(blockIdx.x / nrank) : (int)blockIdx.x) + P.group0;
  const int N = P.N;
  const int tid = threadIdx.x, T = blockDim.x;
  const int NL = CLU ? (N + (int)nrank - 1) / (int)nrank : N;      // regions per CTA
  const int k0 = CLU ? (int)crank * NL : 0;
  const int NODES = min(NL, N - k0) * SPC;        // (the host picks a cluster size that leaves no CTA empty)
  const GroupDesc gd = P.groups[g];
  const TableDesc td = P.tables[gd.table];
  const int Hp = td.Hp, Hs = td.Hs, CH = td.CH, LAG = td.LAG;
  // shared memory: NBAR mbarriers | [GC][T] coupling sums (VEC: [2 GC][T]) | [GC][T] normals (private column per thread) |
  // [NP2][SPC] packed per-sim parameters | edge table + row pointers (SMEMTAB)
  uint64_t* bar_done = reinterpret_cast<uint64_t*>(smem_raw);
  float* const s_cpl = reinterpret_cast<float*>(smem_raw + NBAR * 8) + tid;
  constexpr int CPLROWS = VEC ? 2 * GC : GC;      // (VEC: two 8-step blocks of coupling sums, see SHIFTED WINDOWS)
  float* const s_xi = s_cpl + (size_t)CPLROWS * T;  // GCE == 8: the normals of the chunk's steps; GCE < 8: rows 0..3 = the current Philox quad
  float* const s_quad = s_xi;
  float2* s_ps = reinterpret_cast<float2*>(reinterpret_cast<float*>(smem_raw + NBAR * 8) + (size_t)(CPLROWS + GC) * T);
  // (16-byte aligned by construction: smem_raw is, 64 bytes of barriers, columns of 4 T bytes in multiples of 16 rows, and
  // the parameter block rounded up -- a run-time alignment of the pointer costs a dozen uniform instructions per step)
  unsigned char* const tab = smem_raw + NBAR * 8 + (size_t)(CPLROWS + GC) * T * sizeof(float) + ((NP2 * SPC * sizeof(float2) + 15) & ~(size_t)15);
  // the CTA's part of the delay table: all of it, or (CLU) the rows of its regions; edge indices below are relative
  // to rp0.  (Every table ends with one zero-weight entry that no row owns: a part is never empty.)
  const int32_t* const g_rowptr = P.rowptr + td.rowptr_off;
  const int rp0 = CLU ? g_rowptr[k0] : 0;
  const int n_stage = CLU ? g_rowptr[min(k0 + NL, N)] - rp0 + 1 : td.n_edges;
  Edge<float>* const s_edges = reinterpret_cast<Edge<float>*>(tab);
  Edge8* const s_edges8 = reinterpret_cast<Edge8*>(tab);           // (VEC: 8-byte entries instead)
  float2* const s_edges1 = reinterpret_cast<float2*>(tab);         // (GCE == 1: 8-byte entries (w, offset) instead)
  int32_t* const s_rowptr = reinterpret_cast<int32_t*>(s_edges + n_stage);
  const Edge<float>* const g_edges = P.edges + td.edge_off + rp0;
  float* s_ring = nullptr;                                          // SRING: [N][Hs][SPC] behind the row pointers
  if (SRING) {      // (offset arithmetic on smem_raw itself, so the compiler keeps the shared address space: LDS / STS)
    const size_t off = (size_t)(reinterpret_cast<unsigned char*>(s_rowptr + N + 1) - smem_raw);
    s_ring = reinterpret_cast<float*>(smem_raw + ((off + 15) & ~(size_t)15));
  }
  {
    if (tid < NBAR) mbar_init(bar_done + tid, (uint32_t)(T >> 5) * nrank);
    for (int i = tid; i < NP2 * SPC; i += T) s_ps[i] = P.psim2[(size_t)g * NP2 * SPC + i];
    if (SMEMTAB) {
      if (VEC) {
        const uint32_t qdiv = VW * (uint32_t)RS;
        for (int i = tid; i < n_stage; i += T) {
          const Edge<float> ed = g_edges[i];
          Edge8 e8;
          e8.w = ed.w; e8.qb = (ed.pad / qdiv) | ((ed.back >> VWS) << 20);
          s_edges8[i] = e8;
        }
      } else if (GCE == 1) {      // one-step form: (w, element offset of slot Hp - d of the source row) in 8 bytes
        for (int i = tid; i < n_stage; i += T) {
          const Edge<float> ed = g_edges[i];
          s_edges1[i] = make_float2(ed.w, __uint_as_float(ed.pad));
        }
      } else {
        for (int i = tid; i < n_stage; i += T) s_edges[i] = g_edges[i];
      }
      if (!CLU) for (int i = tid; i <= N; i += T) s_rowptr[i] = g_rowptr[i];
    }
    if (SRING) {
      const float* gr = P.ring + gd.ring_off;
      const int nr = N * Hs * RS;
      for (int i = tid; i < nr; i += T) s_ring[i] = gr[i];
    }
    if (CLU) cluster_sync_all(); else __syncthreads();      // (remote arrivals need the peers' barriers initialised)
  }
  // Scalar ring loads of the cluster forms go through L1 like those of a single CTA (RING_CG = false): a warp reads the
  // ring only after its acquire.cluster wait on the chunk barrier, which invalidates the SM's L1 (CCTL.IVALL), so a line
  // fetched afterwards cannot hold stale values of the slots that wait released; the 8 loads of an edge's window then
  // hit the one or two lines the first of them brought in (cfg 4 as 4-CTA clusters: 1.52e10 with L2-only loads, 1.61e10 so).
  constexpr bool RING_CG = false;
  constexpr int PV = PVN;                         // ring values in flight across one compute step
  const bool noise = P.noise_on != 0;
  const bool active = tid < NODES;
  const int node = active ? tid : NODES - 1;
  const int kl = node / SPC, sl = node - kl * SPC, k = k0 + kl;
  s_ps += sl;
  // the shared-memory address of the lane's parameter column, made opaque so that it stays in ONE register: left to
  // itself the compiler re-derives it every step from tid, N and SPC (7 instructions) to stay under the register bound
  uint32_t ps_a = (uint32_t)__cvta_generic_to_shared(s_ps);
  asm volatile("" : "+r"(ps_a));
  float* ringg = (SRING ? s_ring : P.ring + gd.ring_off) + (VEC ? (int)VW * sl : sl);   // this group's ring, the thread's simulation column
  // (global ring: the pointer is made opaque so that it lives in one register pair and an access is base + 4 * offset;
  // otherwise the compiler keeps the 64-bit element offset and re-adds it to the uniform base at every access)
  if (!SRING && !CLU) {
    asm volatile("" : "+l"(ringg));
    __builtin_assume(__isGlobal(ringg));          // (still LDG / STG, not generic LD / ST)
  }
  const int e_last = n_stage - 1;
  const uint32_t myrow = (uint32_t)(k * Hs) * (uint32_t)RS;
  const int loc = P.loc_id[(size_t)g * SPC + sl];
  const uint32_t ext = (uint32_t)P.ext_id[(size_t)g * SPC + sl];
  const float dt = P.dt;
  const float inv_ds = P.ds > 0 ? 1.0f / (float)P.ds : 0.0f;
  const f2 invN = mk2(P.inv_Ne, P.inv_Ni);
  const int pe0 = (SMEMTAB && !CLU ? s_rowptr[k] : g_rowptr[k]) - rp0, pe1 = (SMEMTAB && !CLU ? s_rowptr[k + 1] : g_rowptr[k + 1]) - rp0;   // this node's row

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

  // S1, not pipelined: coupling sums of the chunk that starts at ring slot cur0 into this thread's column
  // (unpipelined rounds stop at the row's last REAL edge: the zero-weight entries the host pads every row with -- to >= PVN,
  // an odd count -- serve the pipelined batches only; a row of <= 24 edges otherwise paid a round of 8 edges x GCE loads per
  // chunk for its 25th, empty entry: 8 of the 32 LDG per step of cfg 2)
  int pe1t = pe1;
  if (!VEC && GCE != 1)
    while (pe1t > pe0 && (SMEMTAB ? s_edges[pe1t - 1].w : g_edges[pe1t - 1].w) == 0.0f) --pe1t;
  auto gather_from = [&](int e, int cur0, f2 acc[GC / 2]) {
    if (SMEMTAB) gather_rounds<RS, GCE, RING_CG>(s_edges, e, pe1t, e_last, ringg, cur0, Hp, acc);
    else gather_rounds<RS, GCE, RING_CG>(g_edges, e, pe1t, e_last, ringg, cur0, Hp, acc);
  };
  // VEC: the row's seven segments (class 0 | classes 1-3 shifted | classes 1-3 near), ends relative to the staged part
  int seg[7] = {0, 0, 0, 0, 0, 0, 0};
  if (VEC) {
    const int4 sa = *reinterpret_cast<const int4*>(P.seg + td.seg_off + 8 * k), sb = *reinterpret_cast<const int4*>(P.seg + td.seg_off + 8 * k + 4);
    seg[0] = sa.x - rp0; seg[1] = sa.y - rp0; seg[2] = sa.z - rp0; seg[3] = sa.w - rp0;
    seg[4] = sb.x - rp0; seg[5] = sb.y - rp0; seg[6] = sb.z - rp0;
  }
  // the two rows of coupling sums of a VEC thread: block parity pb (0 / 1) -> row pb, 8 slots each, column stride T
  auto cpl_slot = [&](int pb, int j) -> float* { return s_cpl + (size_t)(pb * GC + j) * T; };
  // VEC: the gather for the 8-step block that starts at ring slot cur0 (a multiple of 4) and has parity pb1; completes
  // that block's sums and leaves the partial sums of the first three slots of the block after it (see SHIFTED WINDOWS)
  auto gather_vec = [&](int cur0, int pb1) {
    float cA[GC], cB[3] = {0.0f, 0.0f, 0.0f};
#pragma unroll
    for (int j = 0; j < GC; ++j) cA[j] = j < 3 ? *cpl_slot(pb1, j) : 0.0f;
    const VecLd::word* const ring4 = reinterpret_cast<const VecLd::word*>(ringg);
    const uint32_t thr4 = (uint32_t)(Hp - cur0) >> VWS, cur4 = (uint32_t)cur0 >> VWS, curW4 = cur4 - ((uint32_t)Hp >> VWS);
    const uint32_t qdiv = VW * (uint32_t)RS;
    auto get = [&](int e) -> Edge8 { return SMEMTAB ? s_edges8[e] : edge8_of(g_edges[e], qdiv); };
    f2 acc[6];
    gather_seg_vec<RS, 2>(get, pe0, seg[0], ring4, cur4, thr4, curW4, acc);          // class 0: aligned
#pragma unroll
    for (int t = 0; t < 8; ++t) cA[t] += acc_slot(acc, t);
    gather_seg_vec<RS, 2>(get, seg[0], seg[1], ring4, cur4, thr4, curW4, acc);       // class 1, shifted by 3
#pragma unroll
    for (int t = 0; t < 8; ++t) { if (t + 3 < 8) cA[t + 3] += acc_slot(acc, t); else cB[t - 5] += acc_slot(acc, t); }
    gather_seg_vec<RS, 2>(get, seg[1], seg[2], ring4, cur4, thr4, curW4, acc);       // class 2, shifted by 2
#pragma unroll
    for (int t = 0; t < 8; ++t) { if (t + 2 < 8) cA[t + 2] += acc_slot(acc, t); else cB[t - 6] += acc_slot(acc, t); }
    gather_seg_vec<RS, 2>(get, seg[2], seg[3], ring4, cur4, thr4, curW4, acc);       // class 3, shifted by 1
#pragma unroll
    for (int t = 0; t < 8; ++t) { if (t + 1 < 8) cA[t + 1] += acc_slot(acc, t); else cB[t - 7] += acc_slot(acc, t); }
    if (seg[6] > seg[3]) {                                                             // near edges: unshifted, three quads
      gather_seg_vec<RS, 3>(get, seg[3], seg[4], ring4, cur4, thr4, curW4, acc);
#pragma unroll
      for (int j = 0; j < GC; ++j) cA[j] += acc_slot(acc, 1 + j);
      gather_seg_vec<RS, 3>(get, seg[4], seg[5], ring4, cur4, thr4, curW4, acc);
#pragma unroll
      for (int j = 0; j < GC; ++j) cA[j] += acc_slot(acc, 2 + j);
      gather_seg_vec<RS, 3>(get, seg[5], seg[6], ring4, cur4, thr4, curW4, acc);
#pragma unroll
      for (int j = 0; j < GC; ++j) cA[j] += acc_slot(acc, 3 + j);
    }
#pragma unroll
    for (int j = 0; j < GC; ++j) *cpl_slot(pb1, j) = cA[j];
#pragma unroll
    for (int j = 0; j < 3; ++j) *cpl_slot(pb1 ^ 1, j) = cB[j];
  };
  // VEC, first chunk of a launch (starts at step n0 anywhere inside its 8-step block): the same sums with scalar loads
  // in the same association -- the block's slots from position n0 mod 8 on, and the partial sums of the next block
  auto gather_head_vec = [&](int cur0, int64_t n0) {
    const int o = (int)(n0 & 7), pb = (int)((n0 >> 3) & 1);
    int cb = cur0 - o; if (cb < 0) cb += Hp;                 // ring slot of the block's first step
    int cb2 = cb + GC; if (cb2 >= Hp) cb2 -= Hp;             // ... of the next block's
    // one segment's sum for block position j: edges in order, one FMA chain from zero; sh = the shift the table entry carries
    auto seg_sum = [&](int e0, int e1, int sh, int cbs, int j) -> float {
      float a = 0.0f;
      for (int e = e0; e < e1; ++e) {
        const Edge<float> ed = g_edges[e];
        uint32_t sj = (uint32_t)cbs + (ed.back - (uint32_t)sh) + (uint32_t)j;
        while (sj >= (uint32_t)Hp) sj -= (uint32_t)Hp;
        a = __fmaf_rn(ed.w, __ldcg(ringg + ed.jbase + (sj & ~(VW - 1u)) * (uint32_t)RS + (sj & (VW - 1u))), a);
      }
      return a;
    };
    const int sb[5] = {pe0, seg[0], seg[1], seg[2], seg[3]};      // segment c = [sb[c], sb[c + 1]): class c, shift (4 - c) mod 4
    for (int j = o; j < GC; ++j) {
      float v = 0.0f;
      for (int c = 1; c < 4; ++c) if (4 - c > j) v += seg_sum(sb[c], sb[c + 1], 4 - c, cb, j);        // previous gather's part
      v += seg_sum(sb[0], sb[1], 0, cb, j);
      for (int c = 1; c < 4; ++c) if (4 - c <= j) v += seg_sum(sb[c], sb[c + 1], 4 - c, cb, j);
      for (int c = 0; c < 3; ++c) v += seg_sum(seg[3 + c], seg[4 + c], 0, cb, j);                      // near classes 1, 2, 3
      *cpl_slot(pb, j) = v;
    }
    for (int j = 0; j < 3; ++j) {
      float v = 0.0f;
      for (int c = 1; c < 4; ++c) if (4 - c > j) v += seg_sum(sb[c], sb[c + 1], 4 - c, cb2, j);
      *cpl_slot(pb ^ 1, j) = v;
    }
  };
  // GCE == 1 (one-step chunks; the host mirrors EVERY slot of these rings, Hs = 2 Hp, and pads every row to whole rounds
  // of 4 edges with zero weights): the coupling sum of the step whose time index sits in ring slot cur0, straight from
  // the ring in shared memory -- per edge one table entry, one add (slot cur0 + Hp - d never wraps), one load, one FMA,
  // the row's edges in ascending order in one chain (the association of every other form of the gather).
  auto gather_short = [&](int cur0) -> float {
    const float* const base = ringg + (uint32_t)cur0 * (uint32_t)RS;
    float a = 0.0f;
    for (int e = pe0; e < pe1; e += 4) {      // (rows start at multiples of 4 entries: two 16-byte loads bring four edges)
      const float4 p01 = *reinterpret_cast<const float4*>(s_edges1 + e), p23 = *reinterpret_cast<const float4*>(s_edges1 + e + 2);
      const float v0 = base[__float_as_uint(p01.y)], v1 = base[__float_as_uint(p01.w)];
      const float v2 = base[__float_as_uint(p23.y)], v3 = base[__float_as_uint(p23.w)];
      a = __fmaf_rn(p23.z, v3, __fmaf_rn(p23.x, v2, __fmaf_rn(p01.z, v1, __fmaf_rn(p01.x, v0, a))));
    }
    return a;
  };
  auto gather_now = [&](int cur0) {
    if (GCE == 1) {
      s_cpl[0] = gather_short(cur0);      // (not used: the one-step form gathers inside its step loop)
    } else if (VEC) {
      gather_head_vec(cur0, n);
    } else {
      f2 acc[GC / 2];
#pragma unroll
      for (int j = 0; j < GC / 2; ++j) acc[j] = mk2(0.0f, 0.0f);
      gather_from(pe0, cur0, acc);
#pragma unroll
      for (int j = 0; j < GC / 2; ++j) { s_cpl[(2 * j) * T] = acc[j].x; s_cpl[(2 * j + 1) * T] = acc[j].y; }
    }
  };
  // S4: Philox (A12): one call per (sim, region) per 4 steps gives the normals of steps 4q .. 4q+3.
  // Long chunks (GCE == 8): the normals of a whole chunk are drawn next to its gather, into s_xi.
  // Short chunks (GCE < 8, small minimum delay): the quad lives in s_quad and is redrawn every 4th step.
  auto normals_now = [&](int64_t n0, int ch0) {
    float xi[4] = {0.f, 0.f, 0.f, 0.f};
    if (ch0 == GC && (n0 & 3) == 0) {       // the usual case, a whole chunk on a quad boundary: two Philox calls, eight plain stores
#pragma unroll
      for (int h = 0; h < GC / 4; ++h) {
        normals4<float>(P.seed, ext, (uint32_t)k, ((uint64_t)n0 >> 2) + (uint64_t)h, xi);
#pragma unroll
        for (int q = 0; q < 4; ++q) s_xi[(4 * h + q) * T] = xi[q];
      }
      return;
    }
    for (int i = 0; i < ch0; ++i) {
      const uint64_t nn = (uint64_t)(n0 + i);
      if (i == 0 || (nn & 3) == 0) normals4<float>(P.seed, ext, (uint32_t)k, nn >> 2, xi);
      const uint32_t q = (uint32_t)nn & 3u;
      s_xi[i * T] = q == 0 ? xi[0] : (q == 1 ? xi[1] : (q == 2 ? xi[2] : xi[3]));
    }
  };
  if (GCE < 8 && noise && (P.n_begin & 3)) {      // re-enter a partly used quad at the start of a launch
    float xi[4];
    normals4<float>(P.seed, ext, (uint32_t)k, (uint64_t)P.n_begin >> 2, xi);
#pragma unroll
    for (int q = 0; q < 4; ++q) s_quad[q * T] = xi[q];
  }
  // the gather of chunk m + 1 can overlap the compute of chunk m only if it does not need chunk m itself
  const bool LA = GCE != 1 && LAG >= 2;           // (one-step form: the row is gathered at the start of its own step; CH = 1 => LAG = d_min + 1)
  if (LA && n < P.n_end) {                        // chunk 0 of the launch has no predecessor to hide behind
    gather_now(c);
    if (GCE == 8 && noise) normals_now(n, (int)min((int64_t)(VEC ? CH - (int)(n % CH) : CH), P.n_end - n));
  }

  // per-simulation parameters: small CTAs (relaxed register bound) keep the 9 pairs in registers, the others read them
  // from shared memory where they are used
  constexpr bool PREG = MAXT <= K2_SMALLT;
  f2 ps_reg[NP2];
#pragma unroll
  for (int q = 0; q < NP2; ++q) ps_reg[q] = PREG ? s_ps[q * SPC] : mk2(0.0f, 0.0f);
  auto par = [&](int q) -> f2 {
    if (PREG) return ps_reg[q];
    f2 v;
    asm("ld.shared.v2.f32 {%0, %1}, [%2];" : "=f"(v.x), "=f"(v.y) : "r"(ps_a + (uint32_t)(q * SPC * 8)));
    return v;
  };
  auto wait_chunk = [&](uint32_t w) {              // all warps of the group have written chunk w
    if (CLU) mbar_wait_cluster(bar_done + (w & (NBAR - 1)), (w / NBAR) & 1u);
    else mbar_wait(bar_done + (w & (NBAR - 1)), (w / NBAR) & 1u);
  };
  // One-step form (GCE == 1): the bookkeeping block below is still up to GC steps long, but every step is its own
  // chunk of the rolling pipeline -- it waits for step m - LAG of all warps, gathers its row from the ring in shared
  // memory, computes, writes the ring and arrives -- inside the step loop; m counts steps.
  for (uint32_t m = 0; n < P.n_end; ) {
    // (VEC: a short first chunk brings the chunk starts to multiples of CH = GC, where every window alignment is fixed)
    const int ch = (int)min((int64_t)(GCE == 1 ? GC : (VEC ? CH - (int)(n % CH) : CH)), P.n_end - n);
    const bool has_next = n + ch < P.n_end;
    const int cur1 = c + ch >= Hp ? c + ch - Hp : c + ch;          // ring slot of the next chunk's first step
    if (!LA && GCE != 1) {                        // zero minimum delay: gather right before the chunk
      if (m >= (uint32_t)LAG) { const uint32_t w = m - (uint32_t)LAG; wait_chunk(w); }
      gather_now(c);
      if (GCE == 8 && noise) normals_now(n, ch);
    }
    // the ring writes of chunk m + 1 - LAG (all warps) must be visible before the loads for chunk m + 1
    const bool pipe = LA && has_next;
    if (pipe && m + 1 >= (uint32_t)LAG) { const uint32_t w = m + 1 - (uint32_t)LAG; wait_chunk(w); }
    f2 pacc[GC / 2];                              // coupling sums of chunk m + 1 in the making
#pragma unroll
    for (int j = 0; j < GC / 2; ++j) pacc[j] = mk2(0.0f, 0.0f);
    // step bookkeeping relative to the chunk start, in 32 bits (the 64-bit global step index n stays outside the step loop)
    const int64_t t_rel = n - P.traj_n0;                                             // trajectory row of the chunk's first step
    const bool traj_any = P.traj != nullptr && t_rel < P.traj_steps;                 // (uniform: one branch around the per-lane test)
    const bool traj_on = traj_any && loc >= 0 && active;
    const int traj_left = traj_on ? (int)min(P.traj_steps - t_rel, (int64_t)GC) : 0;     // steps of this chunk that are recorded
    float* const traj0 = traj_on ? P.traj + (((size_t)loc * P.traj_steps + (size_t)t_rel) * 7) * N + k : nullptr;
    const int keep_from = (int)max((int64_t)-1, min(P.discard_steps - n, (int64_t)GC));  // windows ending at step i are kept iff i >= keep_from
    const uint32_t n_lo = (uint32_t)n;
    const int cpl_row0 = VEC ? (int)(((n >> 3) & 1) * GC + (n & 7)) : 0;      // VEC: the block's row, from the chunk's position in it
    const float* cpl_p = s_cpl + cpl_row0 * T;    // running pointers into the thread's private columns (one add per step
    const float* xi_p = s_xi;                     // instead of the row index times the runtime column stride)
    // Steps per trip of the loop: 2 let the address arithmetic and parameter loads of step i + 1 overlap the arithmetic of
    // step i (round 1: cfg 2 +2.8 %; 4 is slower); after round 2's trimming of the loop 1 is ahead again on the one-CTA
    // forms (cfg 2 +1.0 %, cfg 3 +0.5 %), 2 stays ahead with the vector gather (cfg 5 +0.5 %).
    constexpr int STEP_UNROLL = VEC ? 2 : 1;
#pragma unroll STEP_UNROLL
    for (int i = 0; i < ch; ++i) {
      if (GCE == 1 && m + (uint32_t)i >= (uint32_t)LAG) wait_chunk(m + (uint32_t)i - (uint32_t)LAG);
      const float cpl = GCE == 1 ? gather_short(c) : *cpl_p;
      cpl_p += T;
      // ---- S1 for the next chunk: issue the loads of the next PVN / GCE edges now, add them below ----
      float pv[PV];
      if (VEC || GCE == 1) {}
      else if (SMEMTAB) gather_issue<RS, PV / GCE, GCE, RING_CG, true>(s_edges, pe0 + (PV / GCE) * i, e_last, ringg, cur1, Hp, pv);   // (a table has >= 1 entry)
      else gather_issue<RS, PV / GCE, GCE, RING_CG, true>(g_edges, pe0 + (PV / GCE) * i, e_last, ringg, cur1, Hp, pv);
      // ---- S2 + S3: inputs, both transfer functions with derivatives, Eqs. (1)-(3), forward Euler ----
      node_step2(P, par, cpl, noise, dt, invN, nu, Cs, W, Cei, ou);
      // ---- S4 OU (Eq. 4, A11) ----
      if (GCE == 8) {
        if (noise) ou = __fmaf_rn(P.ou_rho, ou, __fmaf_rn(P.ou_s, *xi_p, P.ou_m));
        xi_p += T;
      } else if (noise) {
        if (((n_lo + (uint32_t)i) & 3u) == 0) {   // a new quad of normals
          float xi[4];
          normals4<float>(P.seed, ext, (uint32_t)k, (uint64_t)(n + i) >> 2, xi);
#pragma unroll
          for (int q = 0; q < 4; ++q) s_quad[q * T] = xi[q];
        }
        ou = __fmaf_rn(P.ou_rho, ou, __fmaf_rn(P.ou_s, s_quad[((n_lo + (uint32_t)i) & 3u) * T], P.ou_m));
      }
      // ---- S1 for the next chunk: the loads issued above have had the whole step to arrive ----
      if (VEC || GCE == 1) {}
      else if (SMEMTAB) gather_add<PV / GCE, GCE, true>(s_edges, pe0 + (PV / GCE) * i, pe1, pipe, pv, pacc);
      else gather_add<PV / GCE, GCE, true>(g_edges, pe0 + (PV / GCE) * i, pe1, pipe, pv, pacc);
      // ---- S5 ring write: E at time nn+1 (mirror the first GC-1 slots behind the period) ----
      c = c + 1 == Hp ? 0 : c + 1;
      {     // (lanes past the last node replay it: they store the same value to the same address, no predicate needed)
        const uint32_t o = VEC ? myrow + ((uint32_t)c & ~(VW - 1u)) * (uint32_t)RS + ((uint32_t)c & (VW - 1u)) : myrow + (uint32_t)c * (uint32_t)RS;
        ringg[o] = nu.x;
        if (GCE == 1 || c < (VEC ? GC : GC - 1)) ringg[o + (uint32_t)Hp * (uint32_t)RS] = nu.x;
      }
      // ---- trajectory (tests / cfg 1) ----
      if (traj_any && i < traj_left) {
        float* t = traj0 + (size_t)i * 7 * N;
        t[0] = nu.x; t[N] = nu.y; t[2 * N] = Cs.x; t[3 * N] = Cei; t[4 * N] = Cs.y; t[5 * N] = W.x; t[6 * N] = W.y;
      }
      // ---- S6 temporal average (A17) ----
      win = add2(win, nu);
      if (--win_left == 0) {
        win_left = P.ds;
        if (i >= keep_from) {
          const f2 mm = scl2(inv_ds, win);
          P.xbar[(((size_t)g * P.chunk_samples + sidx) * N + k) * SPC + sl] = mm.x;
          if (ISAMP) P.xbar_i[(((size_t)g * P.chunk_samples + sidx) * N + k) * SPC + sl] = mm.y;
          sumE += (double)mm.x; sumI += (double)mm.y;
          ++sidx;
        }
        win = mk2(0.0f, 0.0f);
      }
      if (GCE == 1) {       // one-step form: this step is a chunk of its own -- publish it
        __syncwarp();
        if ((tid & 31) == 0) mbar_arrive(bar_done + ((m + (uint32_t)i) & (NBAR - 1)));
      }
    }
    if (pipe && VEC) {      // the whole row for chunk m + 1 with vector loads
      gather_vec(cur1, (int)(((n + ch) >> 3) & 1));
      if (noise) normals_now(n + ch, (int)min((int64_t)CH, P.n_end - (n + ch)));
    } else if (pipe) {      // the row's remaining edges (long rows, short chunks), then chunk m + 1 replaces chunk m
      gather_from(pe0 + (PV / GCE) * ch, cur1, pacc);   // (the registers of the transfer function are free here)
      if (GCE == 8 && noise) normals_now(n + ch, (int)min((int64_t)CH, P.n_end - (n + ch)));
#pragma unroll
      for (int j = 0; j < GC / 2; ++j) { s_cpl[(2 * j) * T] = pacc[j].x; s_cpl[(2 * j + 1) * T] = pacc[j].y; }
    }
    // chunk m is written: publish it
    if (GCE != 1) {
      __syncwarp();
      if ((tid & 31) == 0) {
        if (CLU) mbar_arrive_cluster(bar_done + (m & (NBAR - 1)), nrank);
        else mbar_arrive(bar_done + (m & (NBAR - 1)));
      }
    }
    n += ch;
    m += GCE == 1 ? (uint32_t)ch : 1u;
  }
  if (CLU) cluster_sync_all();                    // no CTA leaves while a peer may still arrive on its barriers
  if (SRING) {                                    // the ring goes back to global memory for the next launch
    __syncthreads();
    float* gr = P.ring + gd.ring_off;
    const int nr = N * Hs * RS;
    for (int i = tid; i < nr; i += T) gr[i] = s_ring[i];
  }
  if (active) {
    sp[0] = nu.x; sp[stride] = nu.y; sp[2 * stride] = Cs.x; sp[3 * stride] = Cei; sp[4 * stride] = Cs.y;
    sp[5 * stride] = W.x; sp[6 * stride] = W.y; sp[7 * stride] = ou; sp[8 * stride] = win.x; sp[9 * stride] = win.y;
    sump[0] = sumE; sump[stride] = sumI;
  }
}

}  // namespace tvbx
