// tvbx_kernels.h -- the integrator kernel instances live in their own translation units (tvbx_k_*.cu, compiled in
// parallel); the host side picks one through these functions and launches it through the returned pointer.
#pragma once
#include "tvbx_integrate.cuh"
#include "tvbx_integrate2.cuh"

namespace tvbx {

// ---- general kernel (tvbx_integrate.cuh): FP64 build mode, tau_e != tau_i, several region passes ----
template <typename R> struct KernelPick { void (*fn)(const IntegrateParams<R>); };
// MAXT bounds the registers per thread: 1024 threads -> 64 registers (FP32), 384 -> 168 (FP64).
template <typename R> struct MaxT;
template <> struct MaxT<float> { static constexpr int v = 1024; };
template <> struct MaxT<double> { static constexpr int v = 384; };
// (compile-time simulations-per-CTA values 1, 2, 4, 7 of the FP32 closed-form instances: tvbx_host::spc_is_templated)
KernelPick<float> pick_kernel_f32(bool single, bool closed, int spc);     // tvbx_k_general_f32.cu
KernelPick<double> pick_kernel_f64(bool single, bool closed);             // tvbx_k_general_f64.cu

// ---- packed FP32 product kernel (tvbx_integrate2.cuh) ----
typedef void (*Kernel2Fn)(const Integrate2Params);
struct Kernel2Key {
  int spc;          // simulations per CTA, 1..8
  bool smemtab;     // delay table staged in shared memory
  int gce;          // ring slots loaded per edge: 2, 4 or 8; 1 = the one-step form
  bool clu, vec;    // thread-block cluster form; quad ring layout + vector gather
  bool sring;       // history ring in shared memory (short delays)
  bool small;       // CTAs of <= K2_SMALLT threads: relaxed register bound
  bool isamp;       // also store the inhibitory 1-ms samples (rate statistics of both populations)
  bool ws;          // low-latency form: producer / consumer warp pairs (tvbx_integrate2_ws.cuh)
  bool grp;         // ... with the regions of a group split over several CTAs (cooperative launch)
};
Kernel2Fn pick_kernel2(const Kernel2Key& k);                              // tvbx_kernels.cu
// one function per instance family, each in its own translation unit
Kernel2Fn k2_g8(int spc, bool isamp);              // SMEMTAB, 8 slots
Kernel2Fn k2_g8_small(int spc, bool isamp);        // the same, launch bound K2_SMALLT
Kernel2Fn k2_g8_small_sring(int spc);              // the same with the ring in shared memory
Kernel2Fn k2_g4(int spc, bool sring);              // SMEMTAB, 4 slots (+ ring in shared memory)
Kernel2Fn k2_g2(int spc, bool sring);              // SMEMTAB, 2 slots (+ ring in shared memory)
Kernel2Fn k2_g1(int spc);                          // one-step chunks: fully mirrored ring in shared memory, row gathered per step
Kernel2Fn k2_nosmem(int spc);                      // table through L1/L2, 8 slots
Kernel2Fn k2_clu(int spc);                         // cluster, scalar gather
Kernel2Fn k2_clu_small(int spc);                   // cluster, scalar gather, the CTA's rows of the table in shared memory, launch bound K2_SMALLT
Kernel2Fn k2_ws(int spc, bool sring);               // low-latency warp-pair form (tvbx_integrate2_ws.cuh)
Kernel2Fn k2_wsg(int spc);                         // the same, grouped: a group's regions over several CTAs (tvbx_k_packed_wsg.cu)
int k2_ws_max_threads();                            // its launch bound (consumer + producer threads)
Kernel2Fn k2_vec(int spc, bool smemtab);           // cluster, vector gather (spc 4 or 8)

}  // namespace tvbx
