// tvbx_host.h -- host-side types shared by the translation units of libtvbx.so: error reporting, the
// connectome and sweep objects behind the opaque handles of include/tvbx.h, the ring geometry of a delay
// table, the device-buffer pool and the interface of the per-precision device side.  No kernels here.
#pragma once
#include "../../include/tvbx.h"
#include "../../include/tvbx_diag.h"

#include <cuda_runtime.h>

#include <algorithm>
#include <chrono>
#include <cmath>
#include <cstdint>
#include <cstdlib>
#include <map>
#include <memory>
#include <mutex>
#include <string>
#include <utility>
#include <vector>

namespace tvbx_host {

// thread-local message of the last failing call (tvbx_last_error); returns `code`
int32_t fail(int32_t code, const char* fmt, ...);
const char* last_error();

#define TVBX_CU(call)                                                                                           \
  do {                                                                                                          \
    cudaError_t e_ = (call);                                                                                    \
    if (e_ != cudaSuccess)                                                                                      \
      return ::tvbx_host::fail(e_ == cudaErrorMemoryAllocation ? TVBX_ENOMEM : TVBX_ECUDA, "%s: %s", #call,     \
                               cudaGetErrorString(e_));                                                         \
  } while (0)

// steps per gather chunk of the integrators (= mirror slots + 1), chunks a warp may run ahead (tvbx_integrate*.cuh)
constexpr int kGC = 8, kLagMax = 4;
// rows of a packed-kernel delay table are padded with zero-weight entries to at least this many (= PVN of
// tvbx_integrate2.cuh: the edges a thread gathers software-pipelined across the steps of one chunk)
constexpr int kRowMin = 24;
// largest N the tensor-core FC serves (tvbx_fc_tc.cuh TC_MAXN: the staged tile must fit 227 KB of shared memory)
constexpr int kTcMaxN = 384;

// compile-time simulations-per-CTA values of the general FP32 closed-form kernel (tvbx_k_general_f32.cu; else runtime SPC)
inline bool spc_is_templated(int spc) { return spc == 1 || spc == 2 || spc == 4 || spc == 7; }

// A13: d = nearbyint((L / v) / dt) in FP64, that operation order, round-half-to-even
inline int32_t delay_steps(double L_mm, double v, double dt) { return (int32_t)std::nearbyint((L_mm / v) / dt); }

// Ring geometry of one delay table.  integrate_kernel (general): B steps between CTA barriers, period
// D + B + 1.  integrate2_kernel (packed FP32): chunks of CH = clamp((d_min + 1)/2, 1, GC) steps; chunk m reads
// times <= CH m + CH - 1 - d_min, written by chunks <= m - LAG with LAG = ceil((d_min + 2)/CH) - 1 (>= 2 unless
// d_min = 0; capped at LAGMAX), so the gather of chunk m + 1 can precede the compute of chunk m, a warp may run
// LAG chunks ahead of the slowest one and the period is D + CH LAG + 1.
// vec_ok: the sweep runs the cluster form whose full-length chunks (CH == GC) use the quad ring layout and the
// vector gather (tvbx_integrate2.cuh, gather_class_vec): the period is then a multiple of 4.
struct RingGeom { int32_t B, CH, LAG, Hp, vec; };
inline RingGeom ring_geom(int32_t D, int32_t dmin, bool packed, bool vec_ok = false) {
  RingGeom g;
  const int32_t b = std::max(1, dmin);
  g.B = b >= kGC ? b / kGC * kGC : b;      // whole gather chunks when there is room for one
  g.CH = std::max(1, std::min<int32_t>(kGC, (std::max(0, dmin) + 1) / 2));
  g.LAG = std::max(1, std::min<int32_t>(kLagMax, (dmin + 2 + g.CH - 1) / g.CH - 1));
  g.Hp = packed ? D + g.CH * g.LAG + 1 : D + g.B + 1;
  g.vec = packed && vec_ok && g.CH == kGC;
  if (g.vec) g.Hp = (g.Hp + 3) / 4 * 4;
  return g;
}

struct HostEdge { int32_t j; double w; double L; };
struct Axis { int32_t id; std::vector<double> vals; };
struct HostTable {      // one per distinct speed
  double v = 0;
  int32_t D = 0, dmin = 0, B = 1, Hp = 2, vec = 0;
  bool short1 = false;           // one-step chunks with the fully mirrored ring in shared memory (packed kernel, GCE == 1)
  std::vector<int32_t> delays;   // per kept edge, CSR order
  std::vector<int64_t> sims;     // local sim indices
};
struct HostGroup { int32_t table; std::vector<int64_t> lanes; };  // lanes[sl] = local sim or -1

// RAII: make `device` current for the scope of a call, restore the previous device afterwards (a sweep lives on the
// device that was current at its first tvbx_run; its later calls may come with another device current)
struct DeviceGuard {
  int prev = -1;
  bool switched = false;
  explicit DeviceGuard(int device) {
    if (device < 0) return;
    if (cudaGetDevice(&prev) == cudaSuccess && prev != device) switched = cudaSetDevice(device) == cudaSuccess;
  }
  ~DeviceGuard() { if (switched) cudaSetDevice(prev); }
};

// Device-memory pool: buffers of destroyed sweeps are kept (per device, exact size) and handed to the next sweep
// that asks for the same size, so a create / run / destroy cycle of equal sweeps pays cudaMalloc / cudaFree
// once.  Capacity TVBX_POOL_BYTES (default: a quarter of the device memory; 0 disables); tvbx_trim_memory()
// returns everything to the driver; a failed cudaMalloc trims and retries.
struct DevPool {
  std::mutex mu;
  std::multimap<std::pair<int, size_t>, void*> free_;
  size_t cached = 0;
  long long cap = -1;
  size_t capacity();
  size_t trim();
  cudaError_t get(void** p, size_t bytes, int* device);
  void put(void* p, size_t bytes, int device);     // the caller has made sure no kernel still uses p
  size_t cached_bytes();
  // Free / total memory of the current device as the library knows it.  cudaMemGetInfo is a driver round trip that now
  // and then takes tens of milliseconds (measured: up to 80 ms inside the first tvbx_run of a sweep, on an idle GPU), so
  // it is asked at most once per kMemInfoTtlMs per device; in between the answer is corrected by the pool's own cudaMalloc /
  // cudaFree.  Allocations by others inside that window are not seen: a sweep sized on a stale figure fails in cudaMalloc
  // with TVBX_ENOMEM (which refreshes the figure) instead of in the budget check.
  struct MemInfo { double t_ms = -1e300; size_t free_b = 0, total_b = 0; long long delta = 0; };
  std::map<int, MemInfo> mem_;
  cudaError_t mem_info(size_t* free_b, size_t* total_b);
};
constexpr double kMemInfoTtlMs = 1000.0;
DevPool& dev_pool();

template <typename T>
struct DevBuf {
  T* p = nullptr;
  size_t n = 0, bytes = 0;
  int device = -1;                      // the device the buffer lives on (pool key)
  void release() {
    if (!p) return;
    DeviceGuard guard(device);
    cudaDeviceSynchronize();            // what cudaFree did implicitly: nothing in flight may still use p
    dev_pool().put(p, bytes, device);
    p = nullptr;
  }
  ~DevBuf() { release(); }
  cudaError_t alloc(size_t count) {
    release();
    n = count;
    bytes = (std::max<size_t>(count, 1) * sizeof(T) + 511) / 512 * 512;
    return dev_pool().get((void**)&p, bytes, &device);
  }
  cudaError_t upload(const std::vector<T>& h, int64_t* counter) {
    cudaError_t e = alloc(h.size());
    if (e != cudaSuccess) return e;
    *counter += (int64_t)(h.size() * sizeof(T));
    return cudaMemcpy(p, h.data(), h.size() * sizeof(T), cudaMemcpyHostToDevice);
  }
};

// The dynamic-shared-memory limit is an attribute of the FUNCTION, process-wide: several live sweeps may launch
// the same kernel instance with different sizes.  Raise-only: the attribute is kept at the largest request seen.
cudaError_t raise_dynamic_smem(const void* fn, int bytes);

// event pair around one kernel launch (tvbx_profile_*)
struct ProfEvent { cudaEvent_t a, b; int kind; };
enum { K_INTEGRATE = 0, K_FC = 1, K_READOUT = 2, K_RESET = 3 };

// polymorphic device side (float / double), tvbx_device.cu
struct DeviceSide {
  virtual ~DeviceSide() {}
  virtual int32_t start(double dt) = 0;
  virtual int32_t run(int64_t steps, const tvbx_run_opts* o) = 0;
  virtual int32_t readout(float* fc, float* me, float* mi, int on_device, cudaStream_t st) = 0;
  virtual int32_t scores(const double* ref, float* fcsc, float* fitness, float* mean_fc, int on_device, cudaStream_t st) = 0;
  virtual int32_t rate_stats(float* var_e, float* max_e, int32_t* above, float* var_i, float* max_i, int32_t* above_i, int on_device, cudaStream_t st) = 0;
  virtual int32_t state_durations(int32_t* n_up, float* mean_up_ms, int32_t* n_down, float* mean_down_ms, int on_device, cudaStream_t st) = 0;
  virtual int32_t top_k(int which, const double* ref, int k, int64_t* sim_ids, float* scores, int32_t* n_out, cudaStream_t st) = 0;
  virtual int32_t state(double* y, double* ou) = 0;
  virtual int32_t reset(cudaStream_t st) = 0;
};

}  // namespace tvbx_host

struct tvbx_connectome {
  int32_t n;
  std::vector<double> W, L;
  std::vector<int32_t> rowptr;       // CSR of the non-zero weights, ascending j
  std::vector<tvbx_host::HostEdge> edges;
};

struct tvbx_sweep {
  tvbx_connectome conn;
  tvbx_model_params defaults;
  std::vector<tvbx_host::Axis> axes;
  int64_t grid_size = 1, n_sims = 0;
  std::vector<int64_t> ext_ids;
  uint64_t seed = 0;
  int32_t precision = TVBX_F32, spc = 8, threads_req = 0;
  int32_t spc_req = 0, clu_req = 0;   // tvbx_sweep_opts.sims_per_cta / ctas_per_group as requested (0 = choose)
  int32_t clu = 1;        // CTAs (one thread-block cluster) per group: the regions are split over them
  bool vec_ok = false;    // cluster form with 4 or 8 simulations per group: vector gather where the chunk length allows
  bool packed = false;    // FP32 closed-form product kernel (integrate2_kernel)
  int32_t ws_req = 0;     // tvbx_sweep_opts.latency_form: 0 choose, 1 off, 2 on
  int32_t split = 1;      // 2 while the low-latency warp-pair form of the packed kernel runs (f1), else 1
  bool wsg = false;       // mapping chosen for the GROUPED low-latency form: `clu` CTAs per group, cooperative launch (else the cluster form)
  bool grouped = false;   // ... and it runs (decided at the first tvbx_run, when the delays are known)
  int64_t chunk_req = 0;
  bool fc_tc = false;     // FC co-moment on the tensor cores (tvbx_fc_tc.cuh)
  double rate_thr = 0.1;  // kHz: samples above it are counted (f4; 100 Hz)
  bool stats_i = false;   // keep the inhibitory 1-ms samples of the chunk too and their running statistics
  double ud_thr = 0.0;    // kHz: up / down-state threshold (f4, A25); 0 = the episode statistics are off
  double init[7] = {0.001, 0.001, 0, 0, 0, 0, 0};
  // grouping
  std::vector<tvbx_host::HostTable> tables;
  std::vector<int32_t> sim_table;    // local sim -> table
  std::vector<tvbx_host::HostGroup> groups;
  std::vector<std::pair<int32_t, int32_t>> sim_slot;   // local sim -> (group, lane)
  // run state
  bool started = false;
  double dt = 0;
  int64_t n = 0, cnt = 0, fill = 0, CS = 0, launches = 0;
  int32_t info[9] = {0, 0, 0, 0, 0, 0, 0, 0, 1};
  int64_t h2d = 0, d2h = 0;
  bool profiling = false;
  std::vector<tvbx_host::ProfEvent> prof;
  int device = -1;                   // the CUDA device the sweep lives on (current at its first tvbx_run)
  std::unique_ptr<tvbx_host::DeviceSide> dev;

  ~tvbx_sweep() {
    tvbx_host::DeviceGuard guard(device);
    for (tvbx_host::ProfEvent& e : prof) { cudaEventDestroy(e.a); cudaEventDestroy(e.b); }
    dev.reset();
  }
  // bracket a launch with events while profiling is on
  void prof_begin(int kind, cudaStream_t st) {
    if (!profiling) return;
    tvbx_host::ProfEvent e; e.kind = kind;
    cudaEventCreate(&e.a); cudaEventCreate(&e.b);
    cudaEventRecord(e.a, st);
    prof.push_back(e);
  }
  void prof_end(cudaStream_t st) { if (profiling) cudaEventRecord(prof.back().b, st); }

  // parameter value of local simulation `sim`: the axis digit of its external (grid) index, C order, first axis slowest (A19)
  double param(int64_t sim, int32_t id) const {
    int64_t s = ext_ids[sim];
    double val = defaults.p[id];
    for (int a = (int)axes.size() - 1; a >= 0; --a) {
      const int64_t na = (int64_t)axes[a].vals.size();
      const int64_t dig = s % na;
      s /= na;
      if (axes[a].id == id) val = axes[a].vals[dig];
    }
    return val;
  }
};
