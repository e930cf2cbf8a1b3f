// tvbx_device.cu -- the device side of a sweep (one instance per precision): delay tables and ring geometry per
// distinct speed, device memory, the integrator launches interleaved with the FC chunk reductions, readout, scores,
// rate statistics.  Host code plus the small FC / fill kernels; the integrator instances live in tvbx_k_*.cu.
#include "tvbx_host.h"

#include <cstring>
#include <type_traits>

#include "tvbx_fc.cuh"
#include "tvbx_fc_tc.cuh"
#include "tvbx_kernels.h"
#include "tvbx_tfconst.h"

namespace {

using namespace tvbx;
using namespace tvbx_host;
#define CU TVBX_CU

template <typename R>
__global__ void fill_kernel(R* p, size_t n, R v) {
  for (size_t i = blockIdx.x * (size_t)blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x) p[i] = v;
}

// state[g][q][i] = init[q] for the 7 model variables, 0 for OU and the two window sums
template <typename R>
struct InitVals { R v[NSV - 2]; };
template <typename R>
__global__ void state_init_kernel(R* p, size_t row, size_t total, InitVals<R> iv) {
  for (size_t i = blockIdx.x * (size_t)blockDim.x + threadIdx.x; i < total; i += (size_t)gridDim.x * blockDim.x)
    p[i] = iv.v[(i / row) % (NSV - 2)];
}

inline void set_pad(Edge<float>& e, uint32_t v) { e.pad = v; }
inline void set_pad(Edge<double>&, uint32_t) {}
struct Launch2 { int g0, count; Kernel2Fn fn; int smem; };   // consecutive groups whose tables share the slots-per-edge class

template <typename R>
struct DeviceImpl : DeviceSide {
  tvbx_sweep* sw;
  DevBuf<TableDesc> d_tables;
  DevBuf<GroupDesc> d_groups;
  DevBuf<Edge<R>> d_edges;
  DevBuf<int32_t> d_rowptr, d_seg, d_ext, d_loc;
  DevBuf<R> d_psim, d_ring, d_state, d_xbar;
  DevBuf<float> d_xc;                 // centred TF32 samples of the chunk, K-major (fc_tc)
  int64_t Kp = 0;
  DevBuf<double> d_sums, d_cmean, d_mean, d_M, d_M_scratch, d_mean_scratch;
  DevBuf<float> d_cmax, d_rmax, d_rmax_scratch;       // f4: chunk / running maximum of the excitatory samples
  DevBuf<int32_t> d_ccnt, d_rcnt, d_rcnt_scratch;     //     chunk / running count of samples above the threshold
  // f4, inhibitory population (optional): the chunk's samples and running (mean, M2, max, count), + scratch for readout
  DevBuf<R> d_xbar_i;
  DevBuf<double> d_imean, d_im2, d_imean_scratch, d_im2_scratch;
  DevBuf<float> d_imax, d_imax_scratch;
  DevBuf<int32_t> d_icnt, d_icnt_scratch;
  DevBuf<float> d_out_fc, d_out_me, d_out_mi;
  DevBuf<int32_t> d_ud, d_ud_scratch;                // f4: up / down-state episode state per column (UD_NSTATE planes)
  IntegrateParams<R> P;
  KernelPick<R> kp{nullptr};
  // packed FP32 product kernel (sw->packed)
  Integrate2Params P2;
  std::vector<Launch2> launches2;
  DevBuf<float2> d_psim2;
  DevBuf<uint32_t> d_grpcnt;                          // grouped low-latency form: chunk counters [group][NBAR]
  int threads = 0, smem = 0;
  int run_ds = 1;      // temporal-average window of the runs so far (sample spacing of the 1-ms series = run_ds * dt)
  bool single = true;
  size_t ring_count = 0, max_slice_edges = 0;

  explicit DeviceImpl(tvbx_sweep* s) : sw(s) { std::memset(&P, 0, sizeof P); std::memset(&P2, 0, sizeof P2); }

  int32_t start(double dt) override {
    const tvbx_connectome& c = sw->conn;
    const int N = c.n, SPC = sw->spc;
    const int G = (int)sw->groups.size();
    const double* dp = sw->defaults.p;
    const int RS = SPC;      // simulation columns of a ring slot
    if (sw->packed && sw->stats_i) {
      // the packed kernel stores the inhibitory samples in its 8-slot shared-memory-table instances only: a table with
      // a short minimum delay (chunks < 8 steps) or one too large for shared memory sends the sweep to the general kernel
      for (const HostTable& ht : sw->tables) {
        int32_t dmin = INT32_MAX;
        for (const HostEdge& e : c.edges) dmin = std::min(dmin, delay_steps(e.L, ht.v, dt));
        if (c.edges.empty()) dmin = GC;
        if (ring_geom(1, dmin, true).CH < GC) sw->packed = false;
      }
      const size_t threads2 = (size_t)(N * SPC + 31) / 32 * 32;
      const size_t need = (size_t)NBAR * 8 + 2 * GC * threads2 * sizeof(float) + (size_t)NP2 * SPC * sizeof(float2) + 16 +
                          (c.edges.size() + 1) * sizeof(Edge<float>) + (size_t)(N + 1) * 4;
      if (need > (size_t)200 * 1024) sw->packed = false;
    }
    // ---- delay tables per distinct speed (A13) and ring geometry ----
    std::vector<TableDesc> tds(sw->tables.size());
    std::vector<Edge<R>> edges;
    std::vector<int32_t> rowptr, seg;
    max_slice_edges = 0;
    for (size_t t = 0; t < sw->tables.size(); ++t) {
      HostTable& ht = sw->tables[t];
      ht.delays.clear();
      int32_t D = 0, dmin = INT32_MAX;
      for (const HostEdge& e : c.edges) {
        const int32_t d = delay_steps(e.L, ht.v, dt);
        if (d < 0 || d > 1000000) return fail(TVBX_EINVAL, "delay of %d steps out of range (v=%g, dt=%g)", d, ht.v, dt);
        ht.delays.push_back(d);
        D = std::max(D, d); dmin = std::min(dmin, d);
      }
      if (c.edges.empty()) dmin = GC;
      const RingGeom rg = ring_geom(D, dmin, sw->packed, sw->vec_ok);
      ht.D = D; ht.dmin = dmin; ht.B = rg.B; ht.Hp = rg.Hp; ht.vec = rg.vec;
      // one-step chunks (minimum delay <= 2 steps; cfg 3: v = 64, 128 m/s): the packed kernel keeps the group's ring in
      // shared memory with EVERY slot mirrored (row length 2 Hp), so a read at slot cur + (Hp - d) never wraps, and
      // gathers the row once per step from there (tvbx_integrate2.cuh, GCE == 1) -- if ring + table fit next to the rest
      bool short1 = false;
      if (sw->packed && sw->clu == 1 && rg.CH == 1 && !sw->stats_i && getenv("TVBX_NO_SRING") == nullptr) {
        const size_t thr2 = (size_t)(N * SPC + 31) / 32 * 32;
        const size_t need = (size_t)NBAR * 8 + 2 * GC * thr2 * sizeof(float) + (size_t)NP2 * SPC * sizeof(float2) + 64 +
                            (c.edges.size() + 4 * (size_t)N + 1) * sizeof(Edge<float>) + (size_t)(N + 1) * 4 + (size_t)N * 2 * rg.Hp * RS * sizeof(float);
        short1 = need <= (size_t)200 * 1024;
      }
      ht.short1 = short1;
      const int32_t Hs = short1 ? 2 * ht.Hp : ht.Hp + (rg.vec ? GC : GC - 1);
      if ((double)N * Hs * RS >= 4294967295.0) return fail(TVBX_EINVAL, "ring of one CTA exceeds 32-bit element offsets");
      tds[t].Hp = ht.Hp; tds[t].Hs = Hs; tds[t].B = ht.B; tds[t].n_edges = (int32_t)c.edges.size();
      tds[t].CH = rg.CH; tds[t].LAG = rg.LAG;
      tds[t].edge_off = (int64_t)edges.size(); tds[t].rowptr_off = (int64_t)rowptr.size();
      tds[t].vec = rg.vec; tds[t].seg_off = (int64_t)seg.size(); tds[t].pad0 = short1 ? 1 : 0;
      const int pad_to = short1 ? 4 : 1;      // rows padded with zero-weight copies of their first edge: whole rounds of 4 edges
      for (int k = 0; k < N; ++k) {
        rowptr.push_back((int32_t)(edges.size() - (size_t)tds[t].edge_off));
        const int r0 = c.rowptr[k], r1 = c.rowptr[k + 1];
        if (rg.vec) {
          // quad layout: the row as 7 segments by the alignment a = (Hp - d) mod 4 of an edge's 8-slot window, ascending j
          // inside -- class 0 | classes 1, 2, 3 with the window shifted forward to the next quad boundary (two aligned quads
          // instead of three; needs d >= 8 LAG - 1 + shift, tvbx_integrate2.cuh SHIFTED WINDOWS) | classes 1, 2, 3 "near"
          // (closer than that: unshifted).  Every segment is padded to whole rounds of VR entries.
          for (int sgm = 0; sgm < 7; ++sgm) {
            const int a = sgm == 0 ? 0 : (sgm <= 3 ? sgm : sgm - 3);
            const uint32_t sh = sgm >= 1 && sgm <= 3 ? (uint32_t)(4 - a) : 0u;
            int n_class = 0;
            for (int e = r0; e < r1; ++e) {
              const uint32_t back = (uint32_t)(ht.Hp - ht.delays[e]);
              if ((int)(back & 3u) != a) continue;
              if (a != 0) {
                const bool near_edge = ht.delays[e] < 8 * rg.LAG - 1 + (4 - a);
                if (near_edge != (sgm > 3)) continue;
              }
              Edge<R> ed;
              std::memset(&ed, 0, sizeof ed);
              ed.w = (R)c.edges[e].w;
              ed.jbase = (uint32_t)c.edges[e].j * (uint32_t)Hs * (uint32_t)RS;
              ed.back = back + sh;
              set_pad(ed, ed.jbase + (ed.back & ~(tvbx::VW - 1u)) * (uint32_t)RS);
              edges.push_back(ed);
              ++n_class;
            }
            for (; n_class % VR != 0; ++n_class) {      // whole rounds: zero-weight copies of the segment's last edge
              Edge<R> ed = edges.back();
              ed.w = R(0);
              edges.push_back(ed);
            }
            seg.push_back((int32_t)(edges.size() - (size_t)tds[t].edge_off));
          }
          seg.push_back(0);      // (8 ints per row: two 16-byte loads)
          continue;
        }
        // packed kernel: every row has at least kRowMin entries, so the pipelined batches of a chunk (PVN / GCE edges per
        // step) index the table without a clamp and add without a row-end test (tvbx_integrate2.cuh, PADDED)
        // -- and an ODD number of 16-byte entries: rows of equal even length would put the rows that the lanes of a warp
        // read at the same step into the same shared-memory banks (cfg 1, one region per lane: 32-way conflicts, -9 %).
        const int min_len = sw->packed && !short1 ? kRowMin : 0;
        for (int e = r0; e < r1 || (e - r0) % pad_to != 0 || e - r0 < min_len || (min_len > 0 && (e - r0) % 2 == 0); ++e) {
          Edge<R> ed;
          std::memset(&ed, 0, sizeof ed);
          if (r1 > r0) {      // zero-weight copies of the row's first edge behind its last one
            const int es = e < r1 ? e : r0;
            ed.w = e < r1 ? (R)c.edges[es].w : R(0);
            ed.jbase = (uint32_t)c.edges[es].j * (uint32_t)Hs * (uint32_t)RS;
            ed.back = (uint32_t)(ht.Hp - ht.delays[es]);
          } else {            // a region without afferents: region 0, one slot back
            ed.back = 1u;
          }
          set_pad(ed, ed.jbase + ed.back * (uint32_t)RS);
          edges.push_back(ed);
        }
      }
      rowptr.push_back((int32_t)(edges.size() - (size_t)tds[t].edge_off));
      {      // a table (and any run of its rows) is never empty: one zero-weight entry at the end that no row owns
        Edge<R> ed;
        std::memset(&ed, 0, sizeof ed);
        ed.back = rg.vec ? 4u : 1u;
        set_pad(ed, ed.back * (uint32_t)RS);
        edges.push_back(ed);
      }
      tds[t].n_edges = (int32_t)(edges.size() - (size_t)tds[t].edge_off);
      {      // cluster form: the largest run of rows one CTA stages in shared memory
        const int NLc = (N + sw->clu - 1) / sw->clu;
        const int32_t* rp = rowptr.data() + tds[t].rowptr_off;
        for (int r = 0; r * NLc < N; ++r)
          max_slice_edges = std::max<size_t>(max_slice_edges, (size_t)(rp[std::min(N, (r + 1) * NLc)] - rp[r * NLc] + 1));
      }
    }
    // ---- groups ----
    std::vector<GroupDesc> gds(G);
    std::vector<int32_t> ext((size_t)G * SPC), loc((size_t)G * SPC);
    std::vector<R> psim((size_t)G * NPS * SPC);
    std::vector<float2> psim2(sw->packed ? (size_t)G * NP2 * SPC : 0);
    size_t ring_elems = 0;
    for (int g = 0; g < G; ++g) {
      const HostGroup& hg = sw->groups[g];
      gds[g].table = hg.table; gds[g].pad = 0; gds[g].ring_off = (int64_t)ring_elems;
      ring_elems += (size_t)N * tds[hg.table].Hs * RS;
      ring_elems = (ring_elems + 31) / 32 * 32;      // every group's ring starts on a 128-byte line
      for (int sl = 0; sl < SPC; ++sl) {
        const int64_t s = hg.lanes[sl];
        const int64_t src = s >= 0 ? s : hg.lanes[0];      // padding lanes replay lane 0, never read back
        ext[(size_t)g * SPC + sl] = (int32_t)sw->ext_ids[src];
        loc[(size_t)g * SPC + sl] = s >= 0 ? (int32_t)s : -1;
        const double tw = sw->param(src, TVBX_P_TAU_W_E);
        const double vals[NPS] = {sw->param(src, TVBX_P_G), sw->param(src, TVBX_P_WNOISE), sw->param(src, TVBX_P_B_E),
                                  sw->param(src, TVBX_P_A_E) / tw, 1.0 / tw, sw->param(src, TVBX_P_EL_E),
                                  sw->param(src, TVBX_P_EL_I), 1.0 / sw->param(src, TVBX_P_T),
                                  sw->param(src, TVBX_P_CFEE), sw->param(src, TVBX_P_CFEI),
                                  sw->param(src, TVBX_P_CFIE), sw->param(src, TVBX_P_CFII)};
        for (int q = 0; q < NPS; ++q) psim[((size_t)g * NPS + q) * SPC + sl] = (R)vals[q];
        if (sw->packed) {     // the same scalars as (excitatory, inhibitory) pairs
          const double twi = dp[TVBX_P_TAU_W_I], ati = dp[TVBX_P_A_I] / twi, gL = dp[TVBX_P_GL];
          const double pr[NP2][2] = {{vals[0], vals[1]}, {vals[7], vals[7] * dt}, {vals[2], dp[TVBX_P_B_I]}, {vals[3], ati},
                                     {vals[4], 1.0 / twi}, {vals[3] * vals[5], ati * vals[6]}, {gL * vals[5], gL * vals[6]},
                                     {vals[8], vals[10]}, {vals[9], vals[11]}};
          for (int q = 0; q < NP2; ++q) psim2[((size_t)g * NP2 + q) * SPC + sl] = make_float2((float)pr[q][0], (float)pr[q][1]);
        }
      }
    }
    // ---- memory budget ----
    const size_t row = (size_t)N * SPC;
    size_t free_b = 0, total_b = 0;
    CU(dev_pool().mem_info(&free_b, &total_b));      // (cached: cudaMemGetInfo itself can take tens of ms, tvbx_host.h)
    free_b += dev_pool().cached_bytes();           // pooled buffers are reusable (or trimmed on demand)
    int64_t CS = sw->chunk_req;
    if (CS <= 0) {
      // sample chunk: up to 1/16 of the free device memory, at most 8 GiB (fewer, longer integrator launches)
      const size_t budget = std::min<size_t>((size_t)8 << 30, std::max<size_t>((size_t)1 << 28, free_b / 16));
      CS = (int64_t)(budget / std::max<size_t>(1, (size_t)G * row * sizeof(R)));
      CS = std::min<int64_t>(std::max<int64_t>(CS, 16), 4096);
    }
    Kp = (CS + tvbx::TC_BK - 1) / tvbx::TC_BK * tvbx::TC_BK;
    const size_t need = ring_elems * sizeof(R) + (size_t)G * CS * row * sizeof(R) + (sw->fc_tc ? (size_t)G * Kp * row * sizeof(float) : 0) + (sw->stats_i ? (size_t)G * CS * row * sizeof(R) : 0) +
                        (size_t)G * SPC * N * N * sizeof(double) * 2 + (size_t)G * 16 * row * sizeof(double);
    if (need > free_b)
      return fail(TVBX_ENOMEM, "sweep needs %.2f GB of device memory (ring %.2f GB), %.2f GB free",
                  need / 1e9, ring_elems * sizeof(R) / 1e9, free_b / 1e9);
    sw->CS = CS;
    int64_t* hb = &sw->h2d;
    CU(d_tables.upload(tds, hb)); CU(d_groups.upload(gds, hb)); CU(d_edges.upload(edges, hb)); CU(d_rowptr.upload(rowptr, hb));
    if (seg.empty()) seg.assign(8, 0);
    CU(d_seg.upload(seg, hb));
    CU(d_ext.upload(ext, hb)); CU(d_loc.upload(loc, hb)); CU(d_psim.upload(psim, hb));
    if (sw->packed) CU(d_psim2.upload(psim2, hb));
    CU(d_ring.alloc(ring_elems));
    CU(d_xbar.alloc((size_t)G * CS * row));
    if (sw->stats_i) {
      CU(d_xbar_i.alloc((size_t)G * CS * row));
      CU(cudaMemset(d_xbar_i.p, 0, d_xbar_i.n * sizeof(R)));
      CU(d_imean.alloc((size_t)G * row)); CU(d_im2.alloc((size_t)G * row)); CU(d_imax.alloc((size_t)G * row)); CU(d_icnt.alloc((size_t)G * row));
    }
    if (sw->ud_thr > 0.0) CU(d_ud.alloc((size_t)UD_NSTATE * G * row));
    if (sw->fc_tc) CU(d_xc.alloc((size_t)G * Kp * row));
    CU(d_cmean.alloc((size_t)G * row)); CU(d_mean.alloc((size_t)G * row));
    CU(d_cmax.alloc((size_t)G * row)); CU(d_rmax.alloc((size_t)G * row)); CU(d_ccnt.alloc((size_t)G * row)); CU(d_rcnt.alloc((size_t)G * row));
    CU(d_M.alloc((size_t)G * SPC * N * N));
    CU(d_state.alloc((size_t)G * (NSV - 2) * row));
    CU(d_sums.alloc((size_t)G * 2 * row));
    ring_count = ring_elems;
    CU(cudaMemset(d_xbar.p, 0, d_xbar.n * sizeof(R)));
    { int32_t rc = reset(0); if (rc) return rc; }

    // ---- uniform constants ----
    TFConst<R>& tf = P.tf;
    make_tf_const<R>(dp, tf);
    P.b_i = (R)dp[TVBX_P_B_I]; P.a_i_over_tau = (R)(dp[TVBX_P_A_I] / dp[TVBX_P_TAU_W_I]);
    P.inv_tau_w_i = (R)(1.0 / dp[TVBX_P_TAU_W_I]);
    P.inv_Ne = (R)(1.0 / (dp[TVBX_P_NTOT] * (1.0 - dp[TVBX_P_GINH])));
    P.inv_Ni = (R)(1.0 / (dp[TVBX_P_NTOT] * dp[TVBX_P_GINH]));
    P.kappa = (R)dp[TVBX_P_KAPPA];
    const double rho = std::exp(-dt / dp[TVBX_P_TAU_OU]);
    P.ou_rho = (R)rho; P.ou_s = (R)(dp[TVBX_P_SIGMA_OU] * std::sqrt(1.0 - rho * rho));
    P.ou_m = (R)(dp[TVBX_P_MU_OU] * (1.0 - rho));
    P.dt = (R)dt;
    P.muV_local = dp[TVBX_P_MUV_LOCAL] != 0.0;
    P.N = N; P.SPC = SPC; P.seed = sw->seed; P.chunk_samples = (int32_t)CS;
    P.tables = d_tables.p; P.groups = d_groups.p; P.edges = d_edges.p; P.rowptr = d_rowptr.p;
    P.psim = d_psim.p; P.ext_id = d_ext.p; P.loc_id = d_loc.p; P.ring = d_ring.p; P.state = d_state.p;
    P.sums = d_sums.p; P.xbar = d_xbar.p; P.xbar_i = sw->stats_i ? d_xbar_i.p : nullptr;

    // ---- launch geometry: two lanes per (sim, region) ----
    const int maxt = sw->threads_req > 0 ? std::min(sw->threads_req, MaxT<R>::v) : MaxT<R>::v;
    const int rt_max = std::max(1, maxt / (2 * SPC));           // regions per pass
    int rt;
    if (N <= rt_max) { single = true; rt = N; }
    else { single = false; const int passes = (N + rt_max - 1) / rt_max; rt = (N + passes - 1) / passes; }
    threads = 2 * SPC * rt;
    if constexpr (std::is_same<R, float>::value) kp = pick_kernel_f32(single, tf.same_tau != 0, SPC);
    else kp = pick_kernel_f64(single, tf.same_tau != 0);
    int32_t max_edges = 0;
    for (const TableDesc& td : tds) max_edges = std::max(max_edges, td.n_edges);      // (tables differ by their row padding)
    const size_t tbytes = (size_t)max_edges * sizeof(Edge<R>) + (size_t)(N + 1) * 4;
    const size_t base = ((size_t)(GC + 10) * (threads / 2) + (size_t)L_NPAR * threads + 20) * sizeof(R) + 16;
    P.smem_table = base + tbytes <= 200 * 1024;
    smem = (int)(base + (P.smem_table ? tbytes : 0));
    CU(raise_dynamic_smem((const void*)kp.fn, smem));
    cudaFuncAttributes fa;
    CU(cudaFuncGetAttributes(&fa, (const void*)kp.fn));
    sw->info[0] = G; sw->info[1] = threads; sw->info[2] = SPC; sw->info[3] = fa.numRegs; sw->info[4] = smem;
    sw->info[5] = single ? 1 : (N + rt - 1) / rt; sw->info[6] = (int32_t)CS; sw->info[7] = (int32_t)fa.localSizeBytes;
    if (sw->packed) { int32_t rc = start_packed(tbytes); if (rc) return rc; }
    CU(cudaDeviceSynchronize());
    return TVBX_OK;
  }

  // integrate2_kernel: one thread per (sim, region), both populations in packed FP32 pairs
  int32_t start_packed(size_t tbytes) {
    const int N = sw->conn.n, SPC = sw->spc;
    const double* dp = sw->defaults.p;
    make_tf2_const<R>(dp, P.tf, P2.tf);
    P2.kappa = (float)P.kappa; P2.inv_Ne = (float)P.inv_Ne; P2.inv_Ni = (float)P.inv_Ni;
    P2.ou_rho = (float)P.ou_rho; P2.ou_s = (float)P.ou_s; P2.ou_m = (float)P.ou_m; P2.dt = (float)P.dt;
    P2.muV_local = P.muV_local; P2.N = N; P2.SPC = SPC; P2.seed = P.seed; P2.chunk_samples = P.chunk_samples;
    P2.tables = P.tables; P2.groups = P.groups; P2.edges = (const Edge<float>*)P.edges; P2.rowptr = P.rowptr; P2.seg = d_seg.p;
    P2.psim2 = d_psim2.p; P2.ext_id = P.ext_id; P2.loc_id = P.loc_id; P2.ring = (float*)P.ring; P2.state = (float*)P.state;
    P2.sums = P.sums; P2.xbar = (float*)P.xbar; P2.xbar_i = (float*)P.xbar_i;
    const int CLU = sw->clu, NL = (N + CLU - 1) / CLU;      // regions per CTA
    threads = (NL * SPC + 31) / 32 * 32;
    single = true;
    // (vector-gather kernels keep two 8-step blocks of coupling sums per thread)
    const size_t base = (size_t)NBAR * 8 + (size_t)(sw->vec_ok ? 3 : 2) * GC * threads * sizeof(float) + (size_t)NP2 * SPC * sizeof(float2) + 16;
    // cluster form: the vector-gather kernels stage the rows of the CTA's regions as 8-byte entries; the scalar
    // cluster kernels read the table through L1/L2, except the small-CTA instance (16-byte entries in shared memory)
    const size_t slice_bytes = max_slice_edges * (sw->vec_ok ? sizeof(Edge8) : sizeof(Edge<float>));
    // (at most ~half of the SM's 256 KB: the L1 is the landing space of the ring loads in flight -- 15 warps x 15
    // LDG.128 = 115 KB; measured at N = 360: 212 KB of shared memory halves the throughput)
    bool clu_tab = CLU > 1 && base + slice_bytes <= (size_t)136 * 1024;
    for (const HostTable& ht : sw->tables)      // field widths of Edge8
      if (ht.vec && ((int64_t)N * ((ht.Hp + GC) / (int)tvbx::VW) >= (1 << 20) || ht.Hp / (int)tvbx::VW >= (1 << 12))) clu_tab = false;
    P2.smem_table = CLU == 1 ? base + tbytes <= 200 * 1024 : clu_tab;
    smem = (int)(base + (CLU == 1 ? (P2.smem_table ? tbytes : 0) : (clu_tab ? slice_bytes : 0)));
    // Low-latency form (tvbx_integrate2_ws.cuh): producer / consumer warp pairs.  It pays when the sweep leaves the warp
    // schedulers mostly idle -- all its CTAs resident at once with at most ~2 warps of nodes per scheduler -- and applies to
    // one-CTA groups of <= 160 nodes whose tables all run 8-step chunks from a shared-memory table.
    bool ws = false;
    {
      int n_sm = 148;
      cudaDeviceGetAttribute(&n_sm, cudaDevAttrMultiProcessorCount, sw->device);
      bool ok = CLU == 1 && !sw->stats_i && 2 * threads <= k2_ws_max_threads() && P2.smem_table != 0;
      for (const HostTable& ht : sw->tables) ok = ok && ring_geom(ht.D, ht.dmin, true).CH == GC && !ht.short1;
      const bool small_sweep = (int)sw->groups.size() <= 2 * n_sm;
      if (sw->ws_req == 2 && !ok)
        return fail(TVBX_EINVAL, "latency_form = 2 needs one-CTA groups of <= %d nodes, 8-step chunks (minimum delay >= 15 steps), no inhibitory samples",
                    k2_ws_max_threads() / 2);
      ws = ok && (sw->ws_req == 2 || (sw->ws_req == 0 && small_sweep && getenv("TVBX_NO_WS") == nullptr));
    }
    const size_t ws_base = (size_t)NBAR * 8 + (size_t)(threads / 32) * 4 * 8 + (size_t)4 * GC * threads * sizeof(float) +
                           (size_t)NP2 * SPC * sizeof(float2) + 16;
    // Grouped low-latency form: the mapping was chosen at tvbx_sweep_create (CLU CTAs per group, <= 4 consumer warps per
    // CTA); it runs if the tables qualify and the whole grid is resident at once, else the cluster form serves the mapping.
    bool grouped = false;
    if (sw->wsg && CLU > 1) {
      int n_sm = 148, coop = 0;
      cudaDeviceGetAttribute(&n_sm, cudaDevAttrMultiProcessorCount, sw->device);
      cudaDeviceGetAttribute(&coop, cudaDevAttrCooperativeLaunch, sw->device);
      // (two helper warps behind the warp pairs and NBAR more barriers: tvbx_integrate2_ws.cuh, GRP)
      const size_t wsg_smem = ws_base + (size_t)NBAR * 8 + tbytes;
      bool ok = coop != 0 && !sw->stats_i && !sw->vec_ok && 2 * threads + 64 <= k2_ws_max_threads() && wsg_smem <= (size_t)200 * 1024;
      for (const HostTable& ht : sw->tables) ok = ok && ring_geom(ht.D, ht.dmin, true).CH == GC && !ht.short1 && !ht.vec;
      if (ok) {
        const void* fn = (const void*)k2_wsg(SPC);
        CU(raise_dynamic_smem(fn, (int)wsg_smem));
        int occ = 0;
        CU(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, fn, 2 * threads + 64, wsg_smem));
        ok = (int64_t)sw->groups.size() * CLU <= (int64_t)occ * n_sm;
      }
      if (sw->ws_req == 3 && !ok)
        return fail(TVBX_EINVAL, "latency_form = 3 needs <= %d nodes per CTA, 8-step chunks (minimum delay >= 15 steps), no inhibitory samples and a grid that is resident at once",
                    k2_ws_max_threads() / 2);
      grouped = ok && getenv("TVBX_NO_WSG") == nullptr;
      if (grouped) {
        ws = true;
        P2.smem_table = 1;
        P2.grp_ctas = CLU;
        P2.grp_arrivals = CLU;      // one publication per CTA and chunk
        CU(d_grpcnt.alloc(sw->groups.size() * NBAR));
        P2.grp_cnt = d_grpcnt.p;
      }
    }
    sw->grouped = grouped;
    if (ws) smem = (int)(ws_base + (grouped ? (size_t)NBAR * 8 : 0) + tbytes);
    sw->split = ws ? 2 : 1;
    // one launch per run of groups whose chunk length falls in the same class (cfg 3: v <= 8 / 16 / >= 32 m/s)
    launches2.clear();
    cudaFuncAttributes fa;
    std::memset(&fa, 0, sizeof fa);
    for (int g = 0; g < (int)sw->groups.size(); ++g) {
      const HostTable& ht = sw->tables[sw->groups[g].table];
      const int ch = ring_geom(ht.D, ht.dmin, true).CH;
      const int gce = !P2.smem_table ? 8 : (ht.short1 ? 1 : (ch <= 2 ? 2 : (ch <= 4 ? 4 : 8)));
      // short delays: the group's ring ([N][Hp + GC - 1][SPC] floats) in shared memory next to the table
      const size_t ring_b = (size_t)N * (ht.short1 ? 2 * ht.Hp : ht.Hp + GC - 1) * SPC * sizeof(float) + 16;
      // (and, for CTAs small enough for the relaxed register bound, whenever it fits: cfg 1)
      const bool sring = ht.short1 || CLU == 1 && P2.smem_table && (gce < 8 || (threads <= K2_SMALLT && !sw->stats_i)) &&
                         smem + ring_b <= (size_t)200 * 1024 && getenv("TVBX_NO_SRING") == nullptr;
      const int lsmem = smem + (sring ? (int)ring_b : 0);
      Kernel2Key key;
      key.spc = SPC; key.smemtab = P2.smem_table != 0; key.gce = gce; key.clu = CLU > 1; key.vec = ht.vec != 0; key.sring = sring;
      key.small = !key.vec && !sring && key.smemtab && gce == 8 && threads <= K2_SMALLT;
      key.isamp = sw->stats_i; key.ws = ws; key.grp = grouped;
      if (grouped) { key.clu = false; key.sring = false; key.small = false; }
      Kernel2Fn fn = pick_kernel2(key);
      CU(raise_dynamic_smem((const void*)fn, lsmem));      // (per function, process-wide, raise-only)
      if (!launches2.empty() && launches2.back().fn == fn) {
        launches2.back().count++;
        launches2.back().smem = std::max(launches2.back().smem, lsmem);
        continue;
      }
      launches2.push_back({g, 1, fn, lsmem});
      cudaFuncAttributes f1;
      CU(cudaFuncGetAttributes(&f1, (const void*)fn));
      if (f1.numRegs >= fa.numRegs) fa = f1;
    }
    sw->info[0] = (int32_t)sw->groups.size() * CLU;
    sw->info[1] = ws ? 2 * threads + (grouped ? 64 : 0) : threads; sw->info[3] = fa.numRegs; sw->info[4] = smem; sw->info[5] = 1; sw->info[7] = (int32_t)fa.localSizeBytes;
    sw->info[8] = CLU;
    return TVBX_OK;
  }

  int32_t reset(cudaStream_t st) override {
    InitVals<R> iv;
    for (int q = 0; q < NSV - 2; ++q) iv.v[q] = q < 7 ? (R)sw->init[q] : R(0);
    sw->prof_begin(K_RESET, st);
    state_init_kernel<R><<<592, 256, 0, st>>>(d_state.p, (size_t)sw->conn.n * sw->spc, d_state.n, iv);
    fill_kernel<R><<<1184, 256, 0, st>>>(d_ring.p, ring_count, (R)sw->init[0]);    // A14
    fill_kernel<double><<<592, 256, 0, st>>>(d_sums.p, d_sums.n, 0.0);
    fill_kernel<double><<<592, 256, 0, st>>>(d_mean.p, d_mean.n, 0.0);
    fill_kernel<double><<<1184, 256, 0, st>>>(d_M.p, d_M.n, 0.0);
    if (sw->ud_thr > 0.0) {      // no state yet (-1) in plane 0, zeros elsewhere
      const size_t plane = d_ud.n / UD_NSTATE;
      fill_kernel<int32_t><<<592, 256, 0, st>>>(d_ud.p, plane, -1);
      fill_kernel<int32_t><<<592, 256, 0, st>>>(d_ud.p + plane, d_ud.n - plane, 0);
      sw->launches += 2;
    }
    sw->prof_end(st);
    sw->launches += 5;
    CU(cudaGetLastError());
    sw->n = 0; sw->cnt = 0; sw->fill = 0;
    return TVBX_OK;
  }

  // S7': centre + pack to K-major TF32, then the batched X^T X on tcgen05 with the FP64 Chan merge as epilogue
  int32_t comoment_tc(const FcParams<R>& F, cudaStream_t st) {
    if constexpr (std::is_same<R, float>::value) {
      FcTcParams T;
      T.xbar = F.xbar; T.xc = d_xc.p; T.cmean = F.cmean; T.mean = F.mean; T.M = F.M; T.cnt = F.cnt;
      T.n_c = F.n_c; T.CS = F.CS; T.Kp = (int32_t)Kp; T.N = F.N; T.SPC = F.SPC; T.G = F.G;
      T.Rt = (F.N + 127) / 128 * 128; T.Np = (F.N + 15) / 16 * 16;
      T.tmem_cols = 32;
      while (T.tmem_cols < T.Np) T.tmem_cols *= 2;
      const size_t smem_tc = tc_smem_bytes(T.Rt, T.Np);
      CU(raise_dynamic_smem((const void*)fc_xtx_tc_kernel, (int)smem_tc));
      dim3 gp(F.G, (F.N * F.SPC + 31) / 32, (F.n_c + PACK_Q - 1) / PACK_Q);
      fc_pack_tf32_kernel<<<gp, dim3(32, 8), 0, st>>>(T);
      dim3 gx(F.G * F.SPC, T.Rt / 128);
      fc_xtx_tc_kernel<<<gx, TC_THREADS, smem_tc, st>>>(T);
      return TVBX_OK;
    } else {
      return fail(TVBX_EINVAL, "tensor-core FC needs an FP32 sweep");
    }
  }

  int32_t accumulate(double* Mbuf, double* meanbuf, float* rmaxbuf, int32_t* rcntbuf, bool scratch_i, int64_t cnt, int n_c, cudaStream_t st) {
    const int N = sw->conn.n, SPC = sw->spc, G = (int)sw->groups.size();
    FcParams<R> F;
    F.xbar = d_xbar.p; F.cmean = d_cmean.p; F.mean = meanbuf; F.M = Mbuf; F.cnt = cnt; F.n_c = n_c;
    F.cmax = d_cmax.p; F.ccnt = d_ccnt.p; F.rmax = rmaxbuf; F.rcnt = rcntbuf; F.thr = (float)sw->rate_thr;
    F.CS = (int32_t)sw->CS; F.N = N; F.SPC = SPC; F.G = G;
    const int row = N * SPC;
    dim3 g1(G, (row + 127) / 128), g0(G, (row + 31) / 32);
    sw->prof_begin(K_FC, st);
    fc_chunk_mean_kernel<R><<<g0, 1024, 0, st>>>(F);
    if (sw->fc_tc) {
      int32_t rc = comoment_tc(F, st);
      if (rc) return rc;
    } else {
      const int nt = (N + 31) / 32;
      dim3 g2(G * SPC, nt, nt);
      fc_comoment_kernel<R><<<g2, 64, 0, st>>>(F);
    }
    fc_mean_update_kernel<R><<<g1, 128, 0, st>>>(F);
    if (sw->ud_thr > 0.0 && !scratch_i) {      // (readout merges the open chunk into its own scratch copy: state_durations)
      int32_t rc = updown_chunk(d_ud.p, n_c, st);
      if (rc) return rc;
    }
    if (sw->stats_i) {
      RateIParams<R> I;
      I.xbar_i = d_xbar_i.p;
      I.mean = scratch_i ? d_imean_scratch.p : d_imean.p; I.m2 = scratch_i ? d_im2_scratch.p : d_im2.p;
      I.rmax = scratch_i ? d_imax_scratch.p : d_imax.p; I.rcnt = scratch_i ? d_icnt_scratch.p : d_icnt.p;
      I.cnt = cnt; I.n_c = n_c; I.CS = (int32_t)sw->CS; I.N = N; I.SPC = SPC; I.G = G; I.thr = (float)sw->rate_thr;
      rate_i_chunk_kernel<R><<<g0, 1024, 0, st>>>(I);
      sw->launches += 1;
    }
    sw->prof_end(st);
    sw->launches += sw->fc_tc ? 4 : 3;
    CU(cudaGetLastError());
    return TVBX_OK;
  }

  int32_t run(int64_t steps, const tvbx_run_opts* o) override {
    cudaStream_t st = (cudaStream_t)o->cuda_stream;
    const int N = sw->conn.n;
    const int G = (int)sw->groups.size();
    DevBuf<R> tmp_traj;
    R* traj = nullptr;
    const int64_t tsteps = o->traj ? std::min<int64_t>(o->traj_steps, steps) : 0;
    const size_t traj_elems = (size_t)sw->n_sims * tsteps * 7 * N;
    if (tsteps > 0) {
      if (o->traj_on_device) traj = (R*)o->traj;
      else { CU(tmp_traj.alloc(traj_elems)); traj = tmp_traj.p; }
    }
    P.noise_on = o->noise_on != 0; P.ds = o->ds; P.discard_steps = o->discard_steps;
    if (o->ds > 0) run_ds = o->ds;
    P.traj = traj; P.traj_steps = o->traj_steps; P.traj_n0 = sw->n;
    if (tsteps > 0) P.traj_steps = tsteps;
    int64_t remaining = steps;
    const int64_t ds = o->ds;
    while (remaining > 0) {
      int64_t take = remaining;
      int64_t kept = 0;
      if (ds > 0) {
        const int64_t cap = sw->CS - sw->fill;                 // samples the chunk can still take
        const int64_t e1 = std::max((sw->n / ds + 1) * ds, (o->discard_steps / ds + 1) * ds);  // first kept window end > n
        const int64_t ec = e1 + (cap - 1) * ds;                // window end that fills the chunk
        take = std::min(remaining, ec - sw->n);
        const int64_t end = sw->n + take;
        kept = end >= e1 ? (end - e1) / ds + 1 : 0;
      }
      P.n_begin = sw->n; P.n_end = sw->n + take; P.sample_base = (int32_t)sw->fill;
      sw->prof_begin(K_INTEGRATE, st);
      if (sw->packed) {
        P2.noise_on = P.noise_on; P2.ds = P.ds; P2.discard_steps = P.discard_steps; P2.traj = (float*)P.traj;
        P2.traj_steps = P.traj_steps; P2.traj_n0 = P.traj_n0; P2.n_begin = P.n_begin; P2.n_end = P.n_end;
        P2.sample_base = P.sample_base;
        for (const Launch2& l : launches2) {
          P2.group0 = l.g0;
          if (sw->clu == 1) { l.fn<<<l.count, sw->split == 2 ? 2 * threads : threads, l.smem, st>>>(P2); continue; }
          if (sw->grouped) {     // grouped low-latency form: the CTAs of a group wait on one another -> all resident (cooperative launch)
            CU(cudaMemsetAsync(d_grpcnt.p, 0, d_grpcnt.bytes, st));
            void* args[1] = {(void*)&P2};
            CU(cudaLaunchCooperativeKernel((const void*)l.fn, dim3((unsigned)(l.count * sw->clu)), dim3((unsigned)(2 * threads + 64)), args, (size_t)l.smem, st));
            continue;
          }
          cudaLaunchConfig_t lc;
          std::memset(&lc, 0, sizeof lc);
          lc.gridDim = dim3((unsigned)(l.count * sw->clu)); lc.blockDim = dim3((unsigned)threads);
          lc.dynamicSmemBytes = (size_t)l.smem; lc.stream = st;
          cudaLaunchAttribute at;
          at.id = cudaLaunchAttributeClusterDimension;
          at.val.clusterDim.x = (unsigned)sw->clu; at.val.clusterDim.y = 1; at.val.clusterDim.z = 1;
          lc.attrs = &at; lc.numAttrs = 1;
          CU(cudaLaunchKernelEx(&lc, l.fn, P2));
        }
        sw->launches += (int64_t)launches2.size() - 1;
      } else {
        kp.fn<<<G, threads, smem, st>>>(P);
      }
      sw->prof_end(st);
      sw->launches += 1;
      CU(cudaGetLastError());
      sw->n += take; remaining -= take; sw->fill += kept;
      if (ds > 0 && sw->fill == sw->CS) {
        int32_t rc = accumulate(d_M.p, d_mean.p, d_rmax.p, d_rcnt.p, false, sw->cnt, (int)sw->fill, st);
        if (rc) return rc;
        sw->cnt += sw->fill; sw->fill = 0;
      }
    }
    if (tsteps > 0 && !o->traj_on_device) {
      CU(cudaMemcpyAsync(o->traj, traj, traj_elems * sizeof(R), cudaMemcpyDeviceToHost, st));
      sw->d2h += (int64_t)(traj_elems * sizeof(R));
      CU(cudaStreamSynchronize(st));
    }
    return TVBX_OK;
  }

  // co-moments including the open chunk: merged into a scratch copy, the accumulators stay untouched
  int32_t merged_M(const double** Msrc, cudaStream_t st) {
    DevBuf<double>& tM = d_M_scratch; DevBuf<double>& tmean = d_mean_scratch;   // allocated once, kept
    *Msrc = d_M.p;
    if (sw->fill > 0) {
      if (tM.n != d_M.n) { CU(tM.alloc(d_M.n)); CU(tmean.alloc(d_mean.n)); CU(d_rmax_scratch.alloc(d_rmax.n)); CU(d_rcnt_scratch.alloc(d_rcnt.n)); }
      CU(cudaMemcpyAsync(tM.p, d_M.p, d_M.n * sizeof(double), cudaMemcpyDeviceToDevice, st));
      CU(cudaMemcpyAsync(tmean.p, d_mean.p, d_mean.n * sizeof(double), cudaMemcpyDeviceToDevice, st));
      CU(cudaMemcpyAsync(d_rmax_scratch.p, d_rmax.p, d_rmax.n * sizeof(float), cudaMemcpyDeviceToDevice, st));
      CU(cudaMemcpyAsync(d_rcnt_scratch.p, d_rcnt.p, d_rcnt.n * sizeof(int32_t), cudaMemcpyDeviceToDevice, st));
      if (sw->stats_i) {
        if (d_imean_scratch.n != d_imean.n) { CU(d_imean_scratch.alloc(d_imean.n)); CU(d_im2_scratch.alloc(d_im2.n)); CU(d_imax_scratch.alloc(d_imax.n)); CU(d_icnt_scratch.alloc(d_icnt.n)); }
        CU(cudaMemcpyAsync(d_imean_scratch.p, d_imean.p, d_imean.n * sizeof(double), cudaMemcpyDeviceToDevice, st));
        CU(cudaMemcpyAsync(d_im2_scratch.p, d_im2.p, d_im2.n * sizeof(double), cudaMemcpyDeviceToDevice, st));
        CU(cudaMemcpyAsync(d_imax_scratch.p, d_imax.p, d_imax.n * sizeof(float), cudaMemcpyDeviceToDevice, st));
        CU(cudaMemcpyAsync(d_icnt_scratch.p, d_icnt.p, d_icnt.n * sizeof(int32_t), cudaMemcpyDeviceToDevice, st));
      }
      int32_t rc = accumulate(tM.p, tmean.p, d_rmax_scratch.p, d_rcnt_scratch.p, true, sw->cnt, (int)sw->fill, st);
      if (rc) return rc;
      *Msrc = tM.p;
    }
    return TVBX_OK;
  }

  // f3: FCSC, fitness against a reference FC, mean FC per simulation (fc_scores_kernel)
  DevBuf<double> d_sc, d_ref;
  DevBuf<float> d_out_sc[3];
  int32_t scores(const double* ref, float* fcsc, float* fitness, float* mean_fc, int on_device, cudaStream_t st) override {
    const int N = sw->conn.n, SPC = sw->spc, G = (int)sw->groups.size();
    const int64_t total = sw->cnt + sw->fill;
    if (total < 2) return fail(TVBX_ESTATE, "fewer than 2 samples kept (%lld)", (long long)total);
    const double* Msrc = nullptr;
    { int32_t rc = merged_M(&Msrc, st); if (rc) return rc; }
    const size_t nn = (size_t)N * N;
    if (d_sc.n != nn) {
      CU(d_sc.alloc(nn));
      CU(cudaMemcpyAsync(d_sc.p, sw->conn.W.data(), nn * sizeof(double), cudaMemcpyHostToDevice, st));
      sw->h2d += (int64_t)(nn * sizeof(double));
    }
    if (ref) {
      if (d_ref.n != nn) CU(d_ref.alloc(nn));
      CU(cudaMemcpyAsync(d_ref.p, ref, nn * sizeof(double), cudaMemcpyHostToDevice, st));
      sw->h2d += (int64_t)(nn * sizeof(double));
    }
    ScoreParams Q;
    Q.M = Msrc; Q.sc = d_sc.p; Q.ref = ref ? d_ref.p : nullptr; Q.loc_id = d_loc.p; Q.N = N; Q.SPC = SPC; Q.G = G;
    float* outs[3] = {fcsc, fitness, mean_fc};
    float* devs[3] = {fcsc, fitness, mean_fc};
    if (!on_device)
      for (int i = 0; i < 3; ++i)
        if (outs[i]) { if (d_out_sc[i].n != (size_t)sw->n_sims) CU(d_out_sc[i].alloc((size_t)sw->n_sims)); devs[i] = d_out_sc[i].p; }
    Q.fcsc = devs[0]; Q.fitness = devs[1]; Q.mean_fc = devs[2];
    sw->prof_begin(K_READOUT, st);
    Q.diag_in_smem = N <= 4096;
    fc_scores_kernel<<<G * SPC, 256, Q.diag_in_smem ? (size_t)N * sizeof(double) : 0, st>>>(Q);
    sw->prof_end(st);
    sw->launches += 1;
    CU(cudaGetLastError());
    if (!on_device) {
      for (int i = 0; i < 3; ++i)
        if (outs[i]) {
          CU(cudaMemcpyAsync(outs[i], devs[i], (size_t)sw->n_sims * sizeof(float), cudaMemcpyDeviceToHost, st));
          sw->d2h += (int64_t)((size_t)sw->n_sims * sizeof(float));
        }
      CU(cudaStreamSynchronize(st));
    } else if (ref) {
      CU(cudaStreamSynchronize(st));     // the host copy of ref must not be reused before the upload is done
    }
    return TVBX_OK;
  }

  // f4: variance, maximum and above-threshold count of the excitatory 1-ms samples per (simulation, region)
  DevBuf<float> d_out_var, d_out_max, d_out_var_i, d_out_max_i;
  DevBuf<int32_t> d_out_above, d_out_above_i;
  int32_t rate_stats(float* var_e, float* max_e, int32_t* above, float* var_i, float* max_i, int32_t* above_i, int on_device, cudaStream_t st) override {
    const int N = sw->conn.n, SPC = sw->spc, G = (int)sw->groups.size();
    const int64_t total = sw->cnt + sw->fill;
    if (total < 1) return fail(TVBX_ESTATE, "no sample kept yet");
    const double* Msrc = nullptr;
    { int32_t rc = merged_M(&Msrc, st); if (rc) return rc; }
    RateStatsParams Q;
    Q.M = Msrc; Q.rmax = sw->fill > 0 ? d_rmax_scratch.p : d_rmax.p; Q.rcnt = sw->fill > 0 ? d_rcnt_scratch.p : d_rcnt.p;
    Q.loc_id = d_loc.p; Q.cnt = total; Q.N = N; Q.SPC = SPC; Q.G = G;
    Q.var_e = var_e; Q.max_e = max_e; Q.above = above;
    const bool want_i = var_i || max_i || above_i;
    if (want_i && !sw->stats_i) return fail(TVBX_EINVAL, "inhibitory statistics need tvbx_sweep_opts.rate_stats_inhibitory");
    Q.m2_i = want_i ? (sw->fill > 0 ? d_im2_scratch.p : d_im2.p) : nullptr;
    Q.rmax_i = sw->fill > 0 ? d_imax_scratch.p : d_imax.p; Q.rcnt_i = sw->fill > 0 ? d_icnt_scratch.p : d_icnt.p;
    Q.var_i = var_i; Q.max_i = max_i; Q.above_i = above_i;
    const size_t n_out = (size_t)sw->n_sims * N;
    if (!on_device) {
      if (var_e) { if (d_out_var.n != n_out) CU(d_out_var.alloc(n_out)); Q.var_e = d_out_var.p; }
      if (max_e) { if (d_out_max.n != n_out) CU(d_out_max.alloc(n_out)); Q.max_e = d_out_max.p; }
      if (above) { if (d_out_above.n != n_out) CU(d_out_above.alloc(n_out)); Q.above = d_out_above.p; }
      if (var_i) { if (d_out_var_i.n != n_out) CU(d_out_var_i.alloc(n_out)); Q.var_i = d_out_var_i.p; }
      if (max_i) { if (d_out_max_i.n != n_out) CU(d_out_max_i.alloc(n_out)); Q.max_i = d_out_max_i.p; }
      if (above_i) { if (d_out_above_i.n != n_out) CU(d_out_above_i.alloc(n_out)); Q.above_i = d_out_above_i.p; }
    }
    sw->prof_begin(K_READOUT, st);
    rate_stats_kernel<<<dim3(G * SPC, (N + 127) / 128), 128, 0, st>>>(Q);
    sw->prof_end(st);
    sw->launches += 1;
    CU(cudaGetLastError());
    if (!on_device) {
      if (var_e) { CU(cudaMemcpyAsync(var_e, Q.var_e, n_out * sizeof(float), cudaMemcpyDeviceToHost, st)); sw->d2h += (int64_t)(n_out * sizeof(float)); }
      if (max_e) { CU(cudaMemcpyAsync(max_e, Q.max_e, n_out * sizeof(float), cudaMemcpyDeviceToHost, st)); sw->d2h += (int64_t)(n_out * sizeof(float)); }
      if (above) { CU(cudaMemcpyAsync(above, Q.above, n_out * sizeof(int32_t), cudaMemcpyDeviceToHost, st)); sw->d2h += (int64_t)(n_out * sizeof(int32_t)); }
      if (var_i) { CU(cudaMemcpyAsync(var_i, Q.var_i, n_out * sizeof(float), cudaMemcpyDeviceToHost, st)); sw->d2h += (int64_t)(n_out * sizeof(float)); }
      if (max_i) { CU(cudaMemcpyAsync(max_i, Q.max_i, n_out * sizeof(float), cudaMemcpyDeviceToHost, st)); sw->d2h += (int64_t)(n_out * sizeof(float)); }
      if (above_i) { CU(cudaMemcpyAsync(above_i, Q.above_i, n_out * sizeof(int32_t), cudaMemcpyDeviceToHost, st)); sw->d2h += (int64_t)(n_out * sizeof(int32_t)); }
      CU(cudaStreamSynchronize(st));
    }
    return TVBX_OK;
  }

  int32_t readout(float* fc, float* me, float* mi, int on_device, cudaStream_t st) override {
    const int N = sw->conn.n, SPC = sw->spc, G = (int)sw->groups.size();
    const int64_t total = sw->cnt + sw->fill;
    if (total < 2) return fail(TVBX_ESTATE, "fewer than 2 samples kept (%lld)", (long long)total);
    const double* Msrc = nullptr;
    { int32_t rc = merged_M(&Msrc, st); if (rc) return rc; }
    DevBuf<float>& dfc = d_out_fc; DevBuf<float>& dme = d_out_me; DevBuf<float>& dmi = d_out_mi;   // kept between calls
    ReadoutParams Q;
    Q.M = Msrc; Q.sums = d_sums.p; Q.loc_id = d_loc.p; Q.cnt = total; Q.N = N; Q.SPC = SPC; Q.G = G;
    Q.fc = fc; Q.mean_e = me; Q.mean_i = mi;
    if (!on_device) {
      if (fc) { if (dfc.n != (size_t)sw->n_sims * N * N) CU(dfc.alloc((size_t)sw->n_sims * N * N)); Q.fc = dfc.p; }
      if (me) { if (dme.n != (size_t)sw->n_sims * N) CU(dme.alloc((size_t)sw->n_sims * N)); Q.mean_e = dme.p; }
      if (mi) { if (dmi.n != (size_t)sw->n_sims * N) CU(dmi.alloc((size_t)sw->n_sims * N)); Q.mean_i = dmi.p; }
    }
    dim3 grid(G * SPC, (N + RO_ROWS - 1) / RO_ROWS);
    Q.diag_in_smem = N <= 4096;
    sw->prof_begin(K_READOUT, st);
    fc_readout_kernel<<<grid, 256, Q.diag_in_smem ? (size_t)N * sizeof(double) : 0, st>>>(Q);
    sw->prof_end(st);
    sw->launches += 1;
    CU(cudaGetLastError());
    if (!on_device) {
      if (fc) { CU(cudaMemcpyAsync(fc, dfc.p, dfc.n * sizeof(float), cudaMemcpyDeviceToHost, st)); sw->d2h += (int64_t)(dfc.n * sizeof(float)); }
      if (me) { CU(cudaMemcpyAsync(me, dme.p, dme.n * sizeof(float), cudaMemcpyDeviceToHost, st)); sw->d2h += (int64_t)(dme.n * sizeof(float)); }
      if (mi) { CU(cudaMemcpyAsync(mi, dmi.p, dmi.n * sizeof(float), cudaMemcpyDeviceToHost, st)); sw->d2h += (int64_t)(dmi.n * sizeof(float)); }
      CU(cudaStreamSynchronize(st));
    }
    return TVBX_OK;
  }

  int32_t updown_chunk(int32_t* stbuf, int n_c, cudaStream_t st) {
    const int N = sw->conn.n, SPC = sw->spc, G = (int)sw->groups.size();
    UpDownParams<R> U;
    U.xbar = d_xbar.p; U.st = stbuf; U.n_c = n_c; U.CS = (int32_t)sw->CS; U.N = N; U.SPC = SPC; U.G = G; U.thr = (float)sw->ud_thr;
    updown_chunk_kernel<R><<<dim3(G, (N * SPC + 127) / 128), 128, 0, st>>>(U);
    sw->launches += 1;
    CU(cudaGetLastError());
    return TVBX_OK;
  }

  // f4: up / down-state episode counts and mean durations per (simulation, region)
  DevBuf<int32_t> d_out_nup, d_out_ndn;
  DevBuf<float> d_out_mup, d_out_mdn;
  int32_t state_durations(int32_t* n_up, float* mean_up_ms, int32_t* n_down, float* mean_down_ms, int on_device, cudaStream_t st) override {
    const int N = sw->conn.n, SPC = sw->spc, G = (int)sw->groups.size();
    if (sw->cnt + sw->fill < 1) return fail(TVBX_ESTATE, "no sample kept yet");
    const int32_t* src = d_ud.p;
    if (sw->fill > 0) {      // the open chunk goes into a scratch copy of the state
      if (d_ud_scratch.n != d_ud.n) CU(d_ud_scratch.alloc(d_ud.n));
      CU(cudaMemcpyAsync(d_ud_scratch.p, d_ud.p, d_ud.n * sizeof(int32_t), cudaMemcpyDeviceToDevice, st));
      sw->prof_begin(K_FC, st);
      int32_t rc = updown_chunk(d_ud_scratch.p, (int)sw->fill, st);
      sw->prof_end(st);
      if (rc) return rc;
      src = d_ud_scratch.p;
    }
    UpDownReadParams Q;
    Q.st = src; Q.loc_id = d_loc.p; Q.n_up = n_up; Q.mean_up_ms = mean_up_ms; Q.n_down = n_down; Q.mean_down_ms = mean_down_ms;
    Q.sample_ms = (float)((double)run_ds * sw->dt); Q.N = N; Q.SPC = SPC; Q.G = G;
    const size_t n_out = (size_t)sw->n_sims * N;
    if (!on_device) {
      if (n_up) { if (d_out_nup.n != n_out) CU(d_out_nup.alloc(n_out)); Q.n_up = d_out_nup.p; }
      if (n_down) { if (d_out_ndn.n != n_out) CU(d_out_ndn.alloc(n_out)); Q.n_down = d_out_ndn.p; }
      if (mean_up_ms) { if (d_out_mup.n != n_out) CU(d_out_mup.alloc(n_out)); Q.mean_up_ms = d_out_mup.p; }
      if (mean_down_ms) { if (d_out_mdn.n != n_out) CU(d_out_mdn.alloc(n_out)); Q.mean_down_ms = d_out_mdn.p; }
    }
    sw->prof_begin(K_READOUT, st);
    updown_read_kernel<<<dim3(G * SPC, (N + 127) / 128), 128, 0, st>>>(Q);
    sw->prof_end(st);
    sw->launches += 1;
    CU(cudaGetLastError());
    if (!on_device) {
      if (n_up) { CU(cudaMemcpyAsync(n_up, Q.n_up, n_out * sizeof(int32_t), cudaMemcpyDeviceToHost, st)); sw->d2h += (int64_t)(n_out * 4); }
      if (n_down) { CU(cudaMemcpyAsync(n_down, Q.n_down, n_out * sizeof(int32_t), cudaMemcpyDeviceToHost, st)); sw->d2h += (int64_t)(n_out * 4); }
      if (mean_up_ms) { CU(cudaMemcpyAsync(mean_up_ms, Q.mean_up_ms, n_out * sizeof(float), cudaMemcpyDeviceToHost, st)); sw->d2h += (int64_t)(n_out * 4); }
      if (mean_down_ms) { CU(cudaMemcpyAsync(mean_down_ms, Q.mean_down_ms, n_out * sizeof(float), cudaMemcpyDeviceToHost, st)); sw->d2h += (int64_t)(n_out * 4); }
      CU(cudaStreamSynchronize(st));
    }
    return TVBX_OK;
  }

  // f3: the k best simulations by one of the FC scores
  DevBuf<float> d_topk_score[3], d_topk_val;
  DevBuf<int32_t> d_topk_idx;
  DevBuf<unsigned char> d_topk_taken;
  int32_t top_k(int which, const double* ref, int k, int64_t* sim_ids, float* scores_out, int32_t* n_out, cudaStream_t st) override {
    const size_t S = (size_t)sw->n_sims;
    for (int i = 0; i < 3; ++i) if (d_topk_score[i].n != S) CU(d_topk_score[i].alloc(S));
    int32_t rc = scores(ref, d_topk_score[0].p, ref ? d_topk_score[1].p : nullptr, d_topk_score[2].p, 1, st);
    if (rc) return rc;
    if (d_topk_taken.n != S) CU(d_topk_taken.alloc(S));
    if (d_topk_idx.n != 1024) { CU(d_topk_idx.alloc(1024)); CU(d_topk_val.alloc(1024)); }
    CU(cudaMemsetAsync(d_topk_taken.p, 0, S, st));
    sw->prof_begin(K_READOUT, st);
    topk_kernel<<<1, 1024, 0, st>>>(d_topk_score[which].p, d_topk_taken.p, (int)S, k, d_topk_idx.p, d_topk_val.p);
    sw->prof_end(st);
    sw->launches += 1;
    CU(cudaGetLastError());
    const int n = (int)std::min<size_t>((size_t)k, S);
    std::vector<int32_t> idx(n);
    CU(cudaMemcpyAsync(idx.data(), d_topk_idx.p, (size_t)n * sizeof(int32_t), cudaMemcpyDeviceToHost, st));
    CU(cudaMemcpyAsync(scores_out, d_topk_val.p, (size_t)n * sizeof(float), cudaMemcpyDeviceToHost, st));
    CU(cudaStreamSynchronize(st));
    sw->d2h += (int64_t)n * 8;
    for (int i = 0; i < n; ++i) sim_ids[i] = sw->ext_ids[idx[i]];
    if (n_out) *n_out = n;
    return TVBX_OK;
  }

  int32_t state(double* y, double* ou) override {
    const int N = sw->conn.n, SPC = sw->spc, G = (int)sw->groups.size();
    const size_t row = (size_t)N * SPC;
    std::vector<R> h((size_t)G * (NSV - 2) * row);
    CU(cudaDeviceSynchronize());
    CU(cudaMemcpy(h.data(), d_state.p, h.size() * sizeof(R), cudaMemcpyDeviceToHost));
    for (int64_t s = 0; s < sw->n_sims; ++s) {
      const int g = sw->sim_slot[s].first, sl = sw->sim_slot[s].second;
      for (int k = 0; k < N; ++k) {
        for (int q = 0; q < 7; ++q)
          if (y) y[((size_t)s * 7 + q) * N + k] = (double)h[((size_t)g * (NSV - 2) + q) * row + (size_t)k * SPC + sl];
        if (ou) ou[(size_t)s * N + k] = (double)h[((size_t)g * (NSV - 2) + 7) * row + (size_t)k * SPC + sl];
      }
    }
    return TVBX_OK;
  }
};

}  // namespace

namespace tvbx_host {
DeviceSide* make_device_side(tvbx_sweep* sw) {
  if (sw->precision == TVBX_F64) return new (std::nothrow) DeviceImpl<double>(sw);
  return new (std::nothrow) DeviceImpl<float>(sw);
}
}  // namespace tvbx_host
