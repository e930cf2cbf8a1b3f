// tvbx_api.cu -- the C ABI declared in include/tvbx.h and include/tvbx_diag.h: connectome, parameter grid, grouping
// of simulations by speed and the choice of the launch mapping; error text, device-buffer pool.
// No torch types, no CPU fallback: every compute entry point needs a CUDA device.
#include "tvbx_host.h"

#include <cstdarg>
#include <cstdio>
#include <cstring>
#include <new>

namespace tvbx_host {

namespace { thread_local std::string g_err; }
int32_t fail(int32_t code, const char* fmt, ...) {
  char buf[512];
  va_list ap;
  va_start(ap, fmt);
  vsnprintf(buf, sizeof buf, fmt, ap);
  va_end(ap);
  g_err = buf;
  return code;
}
const char* last_error() { return g_err.c_str(); }

size_t DevPool::capacity() {
  if (cap < 0) {
    if (const char* e = getenv("TVBX_POOL_BYTES")) cap = atoll(e);
    else { size_t f = 0, t = 0; cap = cudaMemGetInfo(&f, &t) == cudaSuccess ? (long long)(t / 4) : 0; }
  }
  return (size_t)cap;
}
static size_t trim_locked(DevPool& P) {
  size_t freed = P.cached;
  for (auto& kv : P.free_) { DeviceGuard guard(kv.first.first); cudaFree(kv.second); P.mem_[kv.first.first].delta -= (long long)kv.first.second; }
  P.free_.clear(); P.cached = 0;
  return freed;
}
size_t DevPool::trim() { std::lock_guard<std::mutex> g(mu); return trim_locked(*this); }
cudaError_t DevPool::get(void** p, size_t bytes, int* device) {
  int dev = 0;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) return e;
  *device = dev;
  std::lock_guard<std::mutex> g(mu);
  auto it = free_.find({dev, bytes});
  if (it != free_.end()) { *p = it->second; cached -= bytes; free_.erase(it); return cudaSuccess; }
  e = cudaMalloc(p, bytes);
  if (e != cudaSuccess && cached > 0) { cudaGetLastError(); trim_locked(*this); e = cudaMalloc(p, bytes); }
  if (e == cudaSuccess) mem_[dev].delta += (long long)bytes;
  else mem_[dev].t_ms = -1e300;      // (the figure was wrong: ask again next time)
  return e;
}
cudaError_t DevPool::mem_info(size_t* free_b, size_t* total_b) {
  int dev = 0;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) return e;
  std::lock_guard<std::mutex> g(mu);
  MemInfo& m = mem_[dev];
  const double now = std::chrono::duration<double, std::milli>(std::chrono::steady_clock::now().time_since_epoch()).count();
  if (now - m.t_ms > kMemInfoTtlMs) {
    e = cudaMemGetInfo(&m.free_b, &m.total_b);
    if (e != cudaSuccess) return e;
    m.t_ms = now; m.delta = 0;
  }
  const long long f = (long long)m.free_b - m.delta;
  *free_b = (size_t)std::max<long long>(f, 0);
  *total_b = m.total_b;
  return cudaSuccess;
}
void DevPool::put(void* p, size_t bytes, int device) {
  std::lock_guard<std::mutex> g(mu);
  if (cached + bytes > capacity()) { DeviceGuard guard(device); cudaFree(p); mem_[device].delta -= (long long)bytes; return; }
  free_.insert({{device, bytes}, p}); cached += bytes;
}
size_t DevPool::cached_bytes() { std::lock_guard<std::mutex> g(mu); return cached; }
DevPool& dev_pool() { static DevPool* P = new DevPool; return *P; }   // never destroyed: no cudaFree at process exit

cudaError_t raise_dynamic_smem(const void* fn, int bytes) {
  static std::map<std::pair<int, const void*>, int> fn_smem;     // (device, function) -> largest size set so far
  static std::mutex fn_mu;
  int dev = 0;
  cudaGetDevice(&dev);
  std::lock_guard<std::mutex> lock(fn_mu);
  int& fmax = fn_smem[{dev, fn}];
  if (bytes <= fmax) return cudaSuccess;
  cudaError_t e = cudaFuncSetAttribute(fn, cudaFuncAttributeMaxDynamicSharedMemorySize, std::max(bytes, 1024));
  if (e == cudaSuccess) fmax = bytes;
  return e;
}

DeviceSide* make_device_side(tvbx_sweep* sw);      // tvbx_device.cu
int32_t diag_tf_closed2(const tvbx_model_params* params, int32_t n, const double* fe, const double* fi, const double* w_e,
                        const double* w_i, double* out);      // tvbx_diag.cu

}  // namespace tvbx_host

namespace {

using namespace tvbx_host;
#define CU TVBX_CU

// library defaults
const double kPolyRS[10] = {-48.9, 5.1, -25.0, 1.4, -0.41, 10.5, -36.0, 7.4, 1.2, 40.7};
const double kPolyFS[10] = {-51.4, 0.4, -8.3, 0.2, -0.5, 1.4, -14.6, 4.5, 2.8, 15.3};

void default_params(tvbx_model_params* m) {
  double* p = m->p;
  for (int i = 0; i < TVBX_N_PARAMS; ++i) p[i] = 0.0;
  p[TVBX_P_G] = 0.0; p[TVBX_P_B_E] = 0.0; p[TVBX_P_A_E] = 0.0; p[TVBX_P_TAU_W_E] = 500.0;
  p[TVBX_P_V] = 4.0; p[TVBX_P_WNOISE] = 1e-6; p[TVBX_P_EL_E] = -64.0; p[TVBX_P_EL_I] = -64.0;
  p[TVBX_P_T] = 20.0;
  p[TVBX_P_CFEE] = 0.3e-3; p[TVBX_P_CFEI] = 0.0; p[TVBX_P_CFIE] = 0.3e-3; p[TVBX_P_CFII] = 0.0;
  p[TVBX_P_B_I] = 0.0; p[TVBX_P_A_I] = 0.0; p[TVBX_P_TAU_W_I] = 1.0;
  p[TVBX_P_GL] = 10.0; p[TVBX_P_CM] = 200.0;
  p[TVBX_P_QE] = 1.5; p[TVBX_P_TAUE] = 5.0; p[TVBX_P_EE] = 0.0;
  p[TVBX_P_QI] = 5.0; p[TVBX_P_TAUI] = 5.0; p[TVBX_P_EI] = -80.0;
  p[TVBX_P_NTOT] = 10000.0; p[TVBX_P_PCONN] = 0.05; p[TVBX_P_GINH] = 0.2;
  p[TVBX_P_TAU_OU] = 5.0; p[TVBX_P_MU_OU] = 0.0; p[TVBX_P_SIGMA_OU] = 1.0;
  p[TVBX_P_MUV0] = -60.0; p[TVBX_P_DMUV0] = 10.0; p[TVBX_P_SV0] = 4.0; p[TVBX_P_DSV0] = 6.0;
  p[TVBX_P_TVN0] = 0.5; p[TVBX_P_DTVN0] = 1.0;
  p[TVBX_P_EPS_NU] = 1e-6; p[TVBX_P_MUV_LOCAL] = 0.0; p[TVBX_P_KAPPA] = 1e-3;
  for (int i = 0; i < 10; ++i) { p[TVBX_P_POLY_E + i] = kPolyRS[i]; p[TVBX_P_POLY_I + i] = kPolyFS[i]; }
}

// A19: equally spaced, closed interval, last value forced to hi
double axis_value(double lo, double hi, int n, int i) {
  if (n <= 1) return lo;
  if (i == n - 1) return hi;
  const double step = (hi - lo) / (double)(n - 1);
  return lo + (double)i * step;
}
}  // namespace

// ====================================================================================================
//  extern "C" entry points
// ====================================================================================================
extern "C" {

const char* tvbx_last_error(void) { return tvbx_host::last_error(); }
int32_t tvbx_version(void) { return TVBX_VERSION; }
int32_t tvbx_trim_memory(int64_t* bytes_freed) {
  const size_t f = dev_pool().trim();
  if (bytes_freed) *bytes_freed = (int64_t)f;
  return TVBX_OK;
}

int32_t tvbx_default_params(tvbx_model_params* out) {
  if (!out) return fail(TVBX_EINVAL, "out is NULL");
  default_params(out);
  return TVBX_OK;
}

int32_t tvbx_create_connectome(int32_t n, const double* W, const double* L_mm, tvbx_connectome** out) {
  if (!out) return fail(TVBX_EINVAL, "out is NULL");
  *out = nullptr;
  if (n < 1 || n > 32767) return fail(TVBX_EINVAL, "n=%d out of range [1, 32767]", n);
  if (!W || !L_mm) return fail(TVBX_EINVAL, "W or L_mm is NULL");
  for (int64_t i = 0; i < (int64_t)n * n; ++i) {
    if (!std::isfinite(W[i]) || W[i] < 0.0) return fail(TVBX_EINVAL, "W[%lld] is negative or not finite", (long long)i);
    if (!std::isfinite(L_mm[i]) || L_mm[i] < 0.0) return fail(TVBX_EINVAL, "L_mm[%lld] is negative or not finite", (long long)i);
  }
  tvbx_connectome* c = new (std::nothrow) tvbx_connectome();
  if (!c) return fail(TVBX_ENOMEM, "host allocation failed");
  c->n = n;
  c->W.assign(W, W + (size_t)n * n);
  c->L.assign(L_mm, L_mm + (size_t)n * n);
  c->rowptr.assign(n + 1, 0);
  for (int k = 0; k < n; ++k) {
    for (int j = 0; j < n; ++j) {
      const double w = W[(size_t)k * n + j];
      if (w != 0.0) c->edges.push_back({j, w, L_mm[(size_t)k * n + j]});
    }
    c->rowptr[k + 1] = (int32_t)c->edges.size();
  }
  *out = c;
  return TVBX_OK;
}
int32_t tvbx_destroy_connectome(tvbx_connectome* c) { delete c; return TVBX_OK; }

// The mapping of the sweep onto CTAs: simulations per CTA, CTAs per group, which integrator serves it, and the groups
// themselves.  Run by tvbx_sweep_create; run AGAIN by the first tvbx_run with allow_wsg = false if the grouped low-latency
// mapping was chosen and dt then shows that a delay table cannot run it (chunks shorter than 8 steps): the delays are only
// known once dt is.
static int32_t choose_mapping(tvbx_sweep* sw, bool allow_wsg) {
  const double* dp = sw->defaults.p;
  sw->wsg = false; sw->clu = 1;
  sw->tables.clear(); sw->groups.clear(); sw->sim_table.clear(); sw->sim_slot.clear();
  // sims per CTA: any 1 .. floor(max threads / 2N).  Pick the count that minimises the number of
  // simulations the busiest SM has to integrate (148 SMs, CTAs of a sweep all resident or in waves).
  int spc = sw->spc_req;
  if (const char* e = getenv("TVBX_SPC")) if (spc == 0) spc = atoi(e);
  // the packed FP32 kernel (one thread per (sim, region), <= 480 of them, <= 8 simulations per CTA) serves
  // tau_e == tau_i and N <= 480; everything else runs the general kernel (two lanes per (sim, region))
  // (with rate_stats_inhibitory the packed kernel serves the one-CTA mapping, N <= 120; tvbx_run falls back to the general
  // kernel if a delay table then needs a short-chunk instance, which has no inhibitory-sample variant)
  const bool packed_ok = sw->precision == TVBX_F32 && dp[TVBX_P_TAUE] == dp[TVBX_P_TAUI] && sw->conn.n <= 480 &&
                         (!sw->stats_i || sw->conn.n <= 120) && getenv("TVBX_GENERAL_KERNEL") == nullptr;
  const int lanes_per_node = packed_ok ? 1 : 2;      // threads per (sim, region) node: the general kernel uses a lane pair
  const int maxt_sel = packed_ok ? 480 : (sw->precision == TVBX_F64 ? 384 : 1024);
  const int spc_max = std::max(1, std::min(packed_ok ? 8 : 32, maxt_sel / (lanes_per_node * sw->conn.n)));
  // CTAs per group (thread-block cluster): the packed kernel can split the regions of a group over up to 8 CTAs.
  // Chosen when one CTA of <= 480 threads would hold fewer than 4 simulations (N > 120; cfg 5: N = 360 ->
  // 6 CTAs x 60 regions x 8 simulations): lanes that share a region then read whole sectors of the ring.
  int clu = sw->clu_req;
  if (const char* e = getenv("TVBX_CLUSTER")) if (clu == 0) clu = atoi(e);
  if (clu < 0 || clu > 8) return fail(TVBX_EINVAL, "ctas_per_group=%d (valid: 0..8)", clu);
  if (clu > 1 && sw->stats_i) return fail(TVBX_EINVAL, "rate_stats_inhibitory needs ctas_per_group <= 1");
  if (clu > 1 && (!packed_ok || sw->threads_req != 0))
    return fail(TVBX_EINVAL, "ctas_per_group > 1 needs the packed FP32 kernel (tau_e == tau_i, N <= 480, no threads_per_cta)");
  auto clu_valid = [&](int c, int sp) {          // every CTA owns >= 1 region and fits 480 threads
    const int nl = (sw->conn.n + c - 1) / c;
    return (c - 1) * nl < sw->conn.n && nl * sp <= 480;
  };
  if (clu == 0 && spc == 0 && packed_ok && sw->threads_req == 0 && spc_max < 4) {
    std::map<double, int64_t> per_v;
    for (int64_t s = 0; s < sw->n_sims; ++s) per_v[sw->param(s, TVBX_P_V)]++;
    int64_t most = 1;
    for (auto& kv : per_v) most = std::max(most, kv.second);
    int want = 8;
    while (want > 1 && want / 2 >= most) want /= 2;       // no more lanes than the largest speed class can fill
    int best_thr = -1;
    for (int c = 1; c <= 8; ++c) {
      if (!clu_valid(c, want)) continue;
      const int thr = ((sw->conn.n + c - 1) / c) * want;
      if (thr > best_thr) { best_thr = thr; clu = c; }
    }
    if (best_thr > 0) spc = want; else clu = 0;
  }
  // Grouped low-latency form (tvbx_integrate2_ws.cuh, GRP): a consumer warp per scheduler is the unit of that form's speed,
  // and a one-CTA mapping of a few hundred simulations puts two on one scheduler (cfg 4: 2 x 68 nodes = 5 warps per SM, or
  // two CTAs of 3).  Splitting the regions of s simulations over c CTAs with <= 128 nodes each leaves one per scheduler if
  // the c * groups CTAs fit the SMs at once.  Taken by latency_form = 0 when no one-CTA mapping achieves that, and by 3.
  if (packed_ok && !sw->stats_i && sw->threads_req == 0 &&
      allow_wsg && (sw->ws_req == 3 || (sw->ws_req == 0 && clu == 0 && spc == 0 && getenv("TVBX_NO_WS") == nullptr && getenv("TVBX_NO_WSG") == nullptr))) {
    const int n_sm = 148;
    std::map<double, int64_t> per_v;
    for (int64_t s = 0; s < sw->n_sims; ++s) per_v[sw->param(s, TVBX_P_V)]++;
    auto n_groups = [&](int s) { int64_t g = 0; for (auto& kv : per_v) g += (kv.second + s - 1) / s; return g; };
    int best_plain = INT32_MAX;       // consumer warps on the busiest scheduler, best one-CTA mapping
    for (int s = 1; s <= 8 && sw->conn.n * s <= 160; ++s) {
      const int64_t ctas = n_groups(s);
      const int64_t per_sm = (ctas + n_sm - 1) / n_sm;
      best_plain = (int)std::min<int64_t>(best_plain, (((int64_t)sw->conn.n * s + 31) / 32 * per_sm + 3) / 4);
    }
    if (sw->ws_req == 3 || best_plain >= 2) {
      double best_fill = 0.0;
      int bc = 0, bs = 0;
      for (int c = 2; c <= 8; ++c) {
        if (clu != 0 && c != clu) continue;
        for (int s = 1; s <= 8; ++s) {
          if (spc != 0 && s != spc) continue;
          const int nl = (sw->conn.n + c - 1) / c;
          if (!clu_valid(c, s) || nl * s > 128) continue;
          const int64_t ctas = n_groups(s) * c;
          if (ctas > n_sm) continue;
          const double fill = (double)sw->n_sims * sw->conn.n / ((double)ctas * 128.0);
          if (fill > best_fill * 1.0001) { best_fill = fill; bc = c; bs = s; }      // (ties: fewer CTAs per group)
        }
      }
      if (bc > 0) { clu = bc; spc = bs; sw->wsg = true; }
      else if (sw->ws_req == 3)
        return fail(TVBX_EINVAL, "latency_form = 3: no split of the regions over 2 .. 8 CTAs with <= 128 nodes each fits %d SMs at once", n_sm);
    }
  }
  if (clu == 0) clu = 1;
  if (clu > 1) {
    if (spc == 0) { spc = 8; while (spc > 1 && !clu_valid(clu, spc)) --spc; }
    if (spc > 8 || !clu_valid(clu, spc))
      return fail(TVBX_EINVAL, "ctas_per_group=%d with sims_per_cta=%d does not fit (N=%d, <= 480 threads per CTA, no empty CTA)", clu, spc, sw->conn.n);
  }
  sw->clu = clu;
  if (spc == 0) {
    // simulations per distinct speed decide the CTA count; approximate with one table here
    std::map<double, int64_t> per_v;
    for (int64_t s = 0; s < sw->n_sims; ++s) per_v[sw->param(s, TVBX_P_V)]++;
    int64_t best_cost = INT64_MAX;
    for (int cand = 1; cand <= spc_max; ++cand) {
      int64_t ctas = 0;
      for (auto& kv : per_v) ctas += (kv.second + cand - 1) / cand;
      const int64_t resident = std::max<int64_t>(1, maxt_sel / (lanes_per_node * (int64_t)sw->conn.n * cand));
      const int64_t slots = 148 * resident;
      int64_t cost = ctas <= slots ? ((ctas + 147) / 148) * cand : ((ctas + slots - 1) / slots) * resident * cand;
      // an SM with fewer resident threads hides less latency: up to +60 % per simulation when nearly empty
      const int64_t thr_sm = std::min<int64_t>(maxt_sel, std::min<int64_t>(resident, (ctas + 147) / 148) * lanes_per_node * sw->conn.n * cand);
      cost = cost * (1000 + 600 * (maxt_sel - thr_sm) / maxt_sel);
      const bool tc = packed_ok || spc_is_templated(cand), ts = packed_ok || spc_is_templated(spc);
      if (cost < best_cost || (cost == best_cost && (tc || !ts))) { best_cost = cost; spc = cand; }
    }
  }
  if (spc < 1 || spc > 32) return fail(TVBX_EINVAL, "sims_per_cta=%d (valid: 1..32)", spc);
  sw->spc = spc;
  sw->packed = packed_ok && spc <= 8 && ((sw->conn.n + clu - 1) / clu) * spc <= 480 && (sw->threads_req == 0 || sw->threads_req >= sw->conn.n * spc);
  sw->vec_ok = sw->packed && clu > 1 && !sw->wsg && (spc == 8 || spc == 4) && getenv("TVBX_NO_VEC") == nullptr;
  if (!sw->packed) sw->wsg = false;
  if (sw->ws_req == 3 && !sw->wsg)
    return fail(TVBX_EINVAL, "latency_form = 3 needs the packed FP32 kernel (tau_e == tau_i), no threads_per_cta, no inhibitory samples");
  // group the simulations by speed (one delay table per distinct v), then into CTAs of spc lanes
  std::map<double, int32_t> vmap;
  sw->sim_table.resize(sw->n_sims);
  for (int64_t s = 0; s < sw->n_sims; ++s) {
    const double v = sw->param(s, TVBX_P_V);
    auto it = vmap.find(v);
    if (it == vmap.end()) {
      it = vmap.emplace(v, (int32_t)sw->tables.size()).first;
      HostTable t; t.v = v; sw->tables.push_back(t);
    }
    sw->sim_table[s] = it->second;
    sw->tables[it->second].sims.push_back(s);
  }
  sw->sim_slot.resize(sw->n_sims);
  for (size_t t = 0; t < sw->tables.size(); ++t) {
    const std::vector<int64_t>& v = sw->tables[t].sims;
    for (size_t i = 0; i < v.size(); i += spc) {
      HostGroup g; g.table = (int32_t)t; g.lanes.assign(spc, -1);
      for (int sl = 0; sl < spc && i + sl < v.size(); ++sl) {
        g.lanes[sl] = v[i + sl];
        sw->sim_slot[v[i + sl]] = {(int32_t)sw->groups.size(), sl};
      }
      sw->groups.push_back(std::move(g));
    }
  }
  return TVBX_OK;
}

int32_t tvbx_sweep_create(const tvbx_connectome* c, const tvbx_model_params* defaults, int32_t n_axes,
                          const tvbx_axis* axes, uint64_t seed, const tvbx_sweep_opts* opts, tvbx_sweep** out) {
  if (!out) return fail(TVBX_EINVAL, "out is NULL");
  *out = nullptr;
  if (!c) return fail(TVBX_EINVAL, "connectome is NULL");
  if (n_axes < 0 || n_axes > 16 || (n_axes > 0 && !axes)) return fail(TVBX_EINVAL, "bad axes");
  std::unique_ptr<tvbx_sweep> sw(new (std::nothrow) tvbx_sweep());
  if (!sw) return fail(TVBX_ENOMEM, "host allocation failed");
  sw->conn = *c;
  if (defaults) sw->defaults = *defaults; else default_params(&sw->defaults);
  sw->seed = seed;
  for (int a = 0; a < n_axes; ++a) {
    const tvbx_axis& ax = axes[a];
    if (ax.param_id < 0 || ax.param_id >= TVBX_N_SWEEPABLE) return fail(TVBX_EINVAL, "axis %d: parameter id %d is not sweepable", a, ax.param_id);
    if (ax.n < 1) return fail(TVBX_EINVAL, "axis %d: n=%d", a, ax.n);
    for (int b = 0; b < a; ++b) if (axes[b].param_id == ax.param_id) return fail(TVBX_EINVAL, "parameter id %d on two axes", ax.param_id);
    Axis h; h.id = ax.param_id;
    for (int i = 0; i < ax.n; ++i) {
      const double val = ax.values ? ax.values[i] : axis_value(ax.lo, ax.hi, ax.n, i);
      if (!std::isfinite(val)) return fail(TVBX_EINVAL, "axis %d: value %d not finite", a, i);
      h.vals.push_back(val);
    }
    if (sw->grid_size > (int64_t)2147483647 / ax.n) return fail(TVBX_EINVAL, "grid larger than 2^31-1 simulations");
    sw->grid_size *= ax.n;
    sw->axes.push_back(std::move(h));
  }
  if (opts && opts->n_sims > 0) {
    if (!opts->sim_ids) return fail(TVBX_EINVAL, "n_sims > 0 but sim_ids is NULL");
    for (int64_t i = 0; i < opts->n_sims; ++i) {
      if (opts->sim_ids[i] < 0 || opts->sim_ids[i] >= sw->grid_size) return fail(TVBX_EINVAL, "sim_ids[%lld]=%lld outside the grid", (long long)i, (long long)opts->sim_ids[i]);
      sw->ext_ids.push_back(opts->sim_ids[i]);      // (< grid_size <= 2^31 - 1: fits the 32-bit Philox counter word of A12)
    }
  } else {
    sw->ext_ids.resize(sw->grid_size);
    for (int64_t i = 0; i < sw->grid_size; ++i) sw->ext_ids[i] = i;
  }
  sw->n_sims = (int64_t)sw->ext_ids.size();
  sw->precision = opts ? opts->precision : TVBX_F32;
  if (sw->precision != TVBX_F32 && sw->precision != TVBX_F64) return fail(TVBX_EINVAL, "precision=%d", sw->precision);
  sw->threads_req = opts ? opts->threads_per_cta : 0;
  sw->ws_req = opts ? opts->latency_form : 0;
  if (sw->ws_req < 0 || sw->ws_req > 3) return fail(TVBX_EINVAL, "latency_form=%d (valid: 0 .. 3)", sw->ws_req);
  sw->chunk_req = opts ? opts->chunk_samples : 0;
  {
    sw->stats_i = opts && opts->rate_stats_inhibitory != 0;
    if (opts && opts->updown_threshold_khz != 0.0) {
      if (!(opts->updown_threshold_khz > 0.0) || !std::isfinite(opts->updown_threshold_khz)) return fail(TVBX_EINVAL, "updown_threshold_khz=%g", opts->updown_threshold_khz);
      sw->ud_thr = opts->updown_threshold_khz;
    }
    if (opts && opts->rate_threshold_khz != 0.0) {
      if (!(opts->rate_threshold_khz > 0.0)) return fail(TVBX_EINVAL, "rate_threshold_khz=%g", opts->rate_threshold_khz);
      sw->rate_thr = opts->rate_threshold_khz;
    }
    int fcm = opts ? opts->fc_mode : TVBX_FC_AUTO;
    if (const char* e = getenv("TVBX_FC_MODE")) if (fcm == TVBX_FC_AUTO) fcm = atoi(e);
    const bool tc_ok = sw->precision == TVBX_F32 && sw->conn.n <= kTcMaxN;
    if (fcm < TVBX_FC_AUTO || fcm > TVBX_FC_TF32) return fail(TVBX_EINVAL, "fc_mode=%d", fcm);
    if (fcm == TVBX_FC_TF32 && !tc_ok) return fail(TVBX_EINVAL, "fc_mode TVBX_FC_TF32 needs an FP32 sweep with N <= %d", kTcMaxN);
    sw->fc_tc = tc_ok && fcm != TVBX_FC_FP32;
  }
  // parameter sanity
  for (int64_t s = 0; s < sw->n_sims; ++s) {
    if (!(sw->param(s, TVBX_P_V) > 0.0)) return fail(TVBX_EINVAL, "speed v must be > 0 (sim %lld)", (long long)s);
    if (!(sw->param(s, TVBX_P_T) > 0.0) || !(sw->param(s, TVBX_P_TAU_W_E) > 0.0)) return fail(TVBX_EINVAL, "T and tau_w_e must be > 0 (sim %lld)", (long long)s);
  }
  const double* dp = sw->defaults.p;
  if (!(dp[TVBX_P_TAU_W_I] > 0) || !(dp[TVBX_P_TAU_OU] > 0) || !(dp[TVBX_P_GL] > 0) || !(dp[TVBX_P_CM] > 0) ||
      !(dp[TVBX_P_DMUV0] != 0) || !(dp[TVBX_P_DSV0] != 0) || !(dp[TVBX_P_DTVN0] != 0) || !(dp[TVBX_P_EPS_NU] > 0) ||
      !(dp[TVBX_P_GINH] > 0 && dp[TVBX_P_GINH] < 1) || !(dp[TVBX_P_NTOT] > 0) || !(dp[TVBX_P_PCONN] > 0))
    return fail(TVBX_EINVAL, "uniform model parameters out of range");
  sw->spc_req = opts ? opts->sims_per_cta : 0;
  sw->clu_req = opts ? opts->ctas_per_group : 0;
  {
    int32_t rc = choose_mapping(sw.get(), true);
    if (rc) return rc;
  }
  *out = sw.release();
  return TVBX_OK;
}

int32_t tvbx_sweep_destroy(tvbx_sweep* sw) { delete sw; return TVBX_OK; }

int32_t tvbx_sweep_set_initial(tvbx_sweep* sw, const double init[7]) {
  if (!sw || !init) return fail(TVBX_EINVAL, "NULL argument");
  if (sw->started) return fail(TVBX_ESTATE, "initial state can only be set before the first tvbx_run");
  for (int i = 0; i < 7; ++i) { if (!std::isfinite(init[i])) return fail(TVBX_EINVAL, "init[%d] not finite", i); sw->init[i] = init[i]; }
  return TVBX_OK;
}

int32_t tvbx_run(tvbx_sweep* sw, int64_t steps, double dt, const tvbx_run_opts* opts) {
  if (!sw) return fail(TVBX_EINVAL, "sweep is NULL");
  if (steps < 0) return fail(TVBX_EINVAL, "steps < 0");
  if (!(dt > 0.0) || !std::isfinite(dt)) return fail(TVBX_EINVAL, "dt must be > 0");
  tvbx_run_opts o;
  std::memset(&o, 0, sizeof o);
  if (opts) o = *opts;
  if (o.ds < 0 || o.discard_steps < 0 || o.traj_steps < 0) return fail(TVBX_EINVAL, "negative ds / discard_steps / traj_steps");
  DeviceGuard guard(sw->device);      // (a no-op before the first run: the sweep then adopts the current device)
  if (!sw->started) {
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev == 0) { cudaGetLastError(); return fail(TVBX_ECUDA, "no CUDA device"); }
    CU(cudaGetDevice(&sw->device));
    if (sw->wsg) {      // the grouped low-latency mapping needs 8-step chunks in every delay table: known only now, with dt
      bool ok = true;
      for (const HostTable& ht : sw->tables) {
        int32_t D = 0, dmin = INT32_MAX;
        for (const HostEdge& e : sw->conn.edges) {
          const int32_t d = delay_steps(e.L, ht.v, dt);
          D = std::max(D, d); dmin = std::min(dmin, d);
        }
        if (sw->conn.edges.empty()) dmin = kGC;
        ok = ok && ring_geom(D, dmin, true).CH == kGC;
      }
      if (!ok) {
        if (sw->ws_req == 3) return fail(TVBX_EINVAL, "latency_form = 3 needs 8-step chunks (minimum delay >= 15 steps)");
        int32_t rc = choose_mapping(sw, false);      // the mapping the sweep would have got without the grouped form
        if (rc) return rc;
      }
    }
    sw->dev.reset(make_device_side(sw));
    if (!sw->dev) return fail(TVBX_ENOMEM, "host allocation failed");
    int32_t rc = sw->dev->start(dt);
    if (rc) { sw->dev.reset(); sw->device = -1; return rc; }
    sw->dt = dt; sw->started = true;
  } else if (dt != sw->dt) {
    return fail(TVBX_EINVAL, "dt=%g differs from the dt of the first run (%g): the delay tables depend on it", dt, sw->dt);
  }
  if (steps == 0) return TVBX_OK;
  return sw->dev->run(steps, &o);
}

int32_t tvbx_fc_scores(tvbx_sweep* sw, const double* ref_fc, float* fcsc, float* fitness, float* mean_fc,
                       int32_t on_device, void* stream) {
  if (!sw) return fail(TVBX_EINVAL, "sweep is NULL");
  if (!sw->started) return fail(TVBX_ESTATE, "no run yet");
  if (fitness && !ref_fc) return fail(TVBX_EINVAL, "fitness needs a reference FC");
  if (ref_fc)
    for (size_t i = 0; i < (size_t)sw->conn.n * sw->conn.n; ++i)
      if (!std::isfinite(ref_fc[i])) return fail(TVBX_EINVAL, "reference FC entry %zu is not finite", i);
  DeviceGuard guard(sw->device);
  return sw->dev->scores(ref_fc, fcsc, fitness, mean_fc, on_device, (cudaStream_t)stream);
}
int32_t tvbx_rate_stats(tvbx_sweep* sw, float* var_e, float* max_e, int32_t* n_above_e, float* var_i, float* max_i,
                        int32_t* n_above_i, int32_t on_device, void* stream) {
  if (!sw) return fail(TVBX_EINVAL, "sweep is NULL");
  if (!sw->started) return fail(TVBX_ESTATE, "no run yet");
  DeviceGuard guard(sw->device);
  return sw->dev->rate_stats(var_e, max_e, n_above_e, var_i, max_i, n_above_i, on_device, (cudaStream_t)stream);
}
int32_t tvbx_state_durations(tvbx_sweep* sw, int32_t* n_up, float* mean_up_ms, int32_t* n_down, float* mean_down_ms,
                             int32_t on_device, void* stream) {
  if (!sw) return fail(TVBX_EINVAL, "sweep is NULL");
  if (!(sw->ud_thr > 0.0)) return fail(TVBX_ESTATE, "the sweep was created without tvbx_sweep_opts.updown_threshold_khz");
  if (!sw->started) return fail(TVBX_ESTATE, "no run yet");
  DeviceGuard guard(sw->device);
  return sw->dev->state_durations(n_up, mean_up_ms, n_down, mean_down_ms, on_device, (cudaStream_t)stream);
}
int32_t tvbx_top_k(tvbx_sweep* sw, int32_t which, const double* ref_fc, int32_t k, int64_t* sim_ids, float* scores,
                   int32_t* n_out, void* stream) {
  if (!sw || !sim_ids || !scores) return fail(TVBX_EINVAL, "NULL argument");
  if (which < 0 || which > 2 || k < 1 || k > 1024) return fail(TVBX_EINVAL, "which in 0..2, k in 1..1024");
  if (which == 1 && !ref_fc) return fail(TVBX_EINVAL, "fitness needs a reference FC");
  if (!sw->started) return fail(TVBX_ESTATE, "no run yet");
  if (ref_fc)
    for (size_t i = 0; i < (size_t)sw->conn.n * sw->conn.n; ++i)
      if (!std::isfinite(ref_fc[i])) return fail(TVBX_EINVAL, "reference FC entry %zu is not finite", i);
  DeviceGuard guard(sw->device);
  return sw->dev->top_k(which, ref_fc, k, sim_ids, scores, n_out, (cudaStream_t)stream);
}
int32_t tvbx_fc_readout(tvbx_sweep* sw, float* fc, float* mean_e, float* mean_i, int32_t on_device, void* stream) {
  if (!sw) return fail(TVBX_EINVAL, "sweep is NULL");
  if (!sw->started) return fail(TVBX_ESTATE, "no run yet");
  DeviceGuard guard(sw->device);
  return sw->dev->readout(fc, mean_e, mean_i, on_device, (cudaStream_t)stream);
}

int32_t tvbx_sweep_reset(tvbx_sweep* sw, void* stream) {
  if (!sw) return fail(TVBX_EINVAL, "sweep is NULL");
  if (!sw->started) return TVBX_OK;
  DeviceGuard guard(sw->device);
  return sw->dev->reset((cudaStream_t)stream);
}
int32_t tvbx_profile_enable(tvbx_sweep* sw, int32_t on) {
  if (!sw) return fail(TVBX_EINVAL, "sweep is NULL");
  sw->profiling = on != 0;
  return TVBX_OK;
}
int32_t tvbx_profile_read(tvbx_sweep* sw, double ms[4], int64_t launches[4]) {
  if (!sw || !ms || !launches) return fail(TVBX_EINVAL, "NULL argument");
  for (int i = 0; i < 4; ++i) { ms[i] = 0.0; launches[i] = 0; }
  DeviceGuard guard(sw->device);
  for (ProfEvent& e : sw->prof) {
    float t = 0.f;
    CU(cudaEventSynchronize(e.b));
    CU(cudaEventElapsedTime(&t, e.a, e.b));
    ms[e.kind] += (double)t;
    launches[e.kind] += e.kind == K_FC ? (sw->fc_tc ? 4 : 3) : (e.kind == K_RESET ? 5 : 1);
    cudaEventDestroy(e.a); cudaEventDestroy(e.b);
  }
  sw->prof.clear();
  return TVBX_OK;
}
int32_t tvbx_bytes_copied(const tvbx_sweep* sw, int64_t* h2d, int64_t* d2h) {
  if (!sw) return fail(TVBX_EINVAL, "sweep is NULL");
  if (h2d) *h2d = sw->h2d;
  if (d2h) *d2h = sw->d2h;
  return TVBX_OK;
}

int32_t tvbx_sweep_size(const tvbx_sweep* sw, int64_t* n_sims, int64_t* grid_size, int32_t* n_regions) {
  if (!sw) return fail(TVBX_EINVAL, "sweep is NULL");
  if (n_sims) *n_sims = sw->n_sims;
  if (grid_size) *grid_size = sw->grid_size;
  if (n_regions) *n_regions = sw->conn.n;
  return TVBX_OK;
}
int32_t tvbx_sweep_param(const tvbx_sweep* sw, int64_t sim, int32_t id, double* out) {
  if (!sw || !out) return fail(TVBX_EINVAL, "NULL argument");
  if (sim < 0 || sim >= sw->n_sims || id < 0 || id >= TVBX_N_PARAMS) return fail(TVBX_EINVAL, "sim or param id out of range");
  *out = sw->param(sim, id);
  return TVBX_OK;
}
int32_t tvbx_sweep_ext_id(const tvbx_sweep* sw, int64_t sim, int64_t* out) {
  if (!sw || !out || sim < 0 || sim >= sw->n_sims) return fail(TVBX_EINVAL, "bad argument");
  *out = sw->ext_ids[sim];
  return TVBX_OK;
}
int32_t tvbx_delay_index(const tvbx_sweep* sw, int64_t sim, int32_t k, int32_t j, double dt, int32_t* out) {
  if (!sw || !out) return fail(TVBX_EINVAL, "NULL argument");
  const int n = sw->conn.n;
  if (sim < 0 || sim >= sw->n_sims || k < 0 || k >= n || j < 0 || j >= n) return fail(TVBX_EINVAL, "index out of range");
  if (!(dt > 0.0)) { if (!sw->started) return fail(TVBX_ESTATE, "dt unknown before the first run"); dt = sw->dt; }
  *out = sw->conn.W[(size_t)k * n + j] == 0.0 ? -1 : delay_steps(sw->conn.L[(size_t)k * n + j], sw->param(sim, TVBX_P_V), dt);
  return TVBX_OK;
}
int32_t tvbx_ring_len(const tvbx_sweep* sw, int64_t sim, double dt, int32_t* H, int32_t* H_phys) {
  if (!sw) return fail(TVBX_EINVAL, "sweep is NULL");
  if (sim < 0 || sim >= sw->n_sims) return fail(TVBX_EINVAL, "sim out of range");
  if (!(dt > 0.0)) { if (!sw->started) return fail(TVBX_ESTATE, "dt unknown before the first run"); dt = sw->dt; }
  const double v = sw->param(sim, TVBX_P_V);
  int32_t D = 0, dmin = INT32_MAX;
  for (const HostEdge& e : sw->conn.edges) { const int32_t d = delay_steps(e.L, v, dt); D = std::max(D, d); dmin = std::min(dmin, d); }
  if (sw->conn.edges.empty()) dmin = kGC;
  if (H) *H = D + 1;
  if (H_phys) *H_phys = ring_geom(D, dmin, sw->packed, sw->vec_ok).Hp;
  return TVBX_OK;
}
int32_t tvbx_steps_done(const tvbx_sweep* sw, int64_t* n) {
  if (!sw || !n) return fail(TVBX_EINVAL, "NULL argument");
  *n = sw->n;
  return TVBX_OK;
}
int32_t tvbx_samples_kept(const tvbx_sweep* sw, int64_t* n) {
  if (!sw || !n) return fail(TVBX_EINVAL, "NULL argument");
  *n = sw->cnt + sw->fill;
  return TVBX_OK;
}
int32_t tvbx_sweep_state(tvbx_sweep* sw, double* y, double* ou) {
  if (!sw) return fail(TVBX_EINVAL, "sweep is NULL");
  if (!sw->started) return fail(TVBX_ESTATE, "no run yet");
  DeviceGuard guard(sw->device);
  return sw->dev->state(y, ou);
}
int32_t tvbx_launch_info(const tvbx_sweep* sw, int32_t info[10]) {
  if (!sw || !info) return fail(TVBX_EINVAL, "NULL argument");
  for (int i = 0; i < 9; ++i) info[i] = sw->info[i];
  info[9] = sw->split;
  return TVBX_OK;
}
int32_t tvbx_kernel_name(const tvbx_sweep* sw, char* buf, int32_t n) {
  if (!sw || !buf || n < 1) return fail(TVBX_EINVAL, "bad argument");
  snprintf(buf, (size_t)n, "%s", sw->packed ? "tvbx::integrate2_kernel" : "tvbx::integrate_kernel");
  return TVBX_OK;
}
int32_t tvbx_fc_kernel_name(const tvbx_sweep* sw, char* buf, int32_t n) {
  if (!sw || !buf || n < 1) return fail(TVBX_EINVAL, "bad argument");
  snprintf(buf, (size_t)n, "%s", sw->fc_tc ? "tvbx::fc_xtx_tc_kernel" : "tvbx::fc_comoment_kernel");
  return TVBX_OK;
}
int32_t tvbx_launch_count(const tvbx_sweep* sw, int64_t* n) {
  if (!sw || !n) return fail(TVBX_EINVAL, "NULL argument");
  *n = sw->launches;
  return TVBX_OK;
}

int32_t tvbx_diag_tf_closed2(const tvbx_model_params* params, int32_t n, const double* fe, const double* fi,
                             const double* w_e, const double* w_i, double* out) {
  if (n < 0 || (n > 0 && (!fe || !fi || !w_e || !w_i || !out))) return fail(TVBX_EINVAL, "bad argument");
  return diag_tf_closed2(params, n, fe, fi, w_e, w_i, out);
}

}  // extern "C"
