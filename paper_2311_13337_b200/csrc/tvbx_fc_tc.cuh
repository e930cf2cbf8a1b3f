// tvbx_fc_tc.cuh -- S7' of SURVEY.md section 8(a): the centred co-moment X^T X of a sample chunk as a batched
// dense contraction on the 5th-generation tensor cores (tcgen05.mma kind::tf32, FP32 accumulators in TMEM),
// fused with the Chan merge into the FP64 running co-moment.
// ("covariance of the resulting time-series for all concurrent simulations"), Eq. (6); BASELINE.json
// cfg 5 ("computed through a batched X^T X").
//
// Two kernels per chunk (after fc_chunk_mean_kernel, before fc_mean_update_kernel of tvbx_fc.cuh):
//   fc_pack_tf32_kernel : xbar[g][q][k][s] -> xc[g][s][k][q]  (sample index fastest = K-major operand rows),
//                         centred on the FP64 chunk mean BEFORE rounding to TF32 (the fluctuation is 1e-4 of
//                         the mean: uncentred TF32 products would lose everything), zero padded to a multiple
//                         of BK samples.
//   fc_xtx_tc_kernel    : one CTA per (simulation, block of 128 rows).  A = rows [128 mb, 128 mb + 128) and
//                         B = all N rows of the same K-major matrix, so ONE shared-memory tile per pipeline stage
//                         serves both operands (the A descriptor points into the B tile).  cp.async fills a
//                         4-stage ring in the canonical no-swizzle K-major core-matrix layout, one elected
//                         thread issues tcgen05.mma (M = 128, N <= 256 per instruction, K = 8 per instruction),
//                         tcgen05.commit on a per-stage mbarrier frees the stage; the epilogue reads TMEM with
//                         tcgen05.ld (thread = output row, 32 columns), transposes 32 x 32 blocks through the free
//                         stage memory and adds M_c + (delta_k delta_l) cnt n_c/(cnt + n_c) into the FP64
//                         accumulator rows the CTA owns -- one contiguous 256-byte run per warp instruction, every
//                         element written by exactly one thread (no mirrored or atomic writes).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include "tvbx_fc.cuh"

namespace tvbx {

constexpr int TC_BK = 32;        // samples per pipeline stage (4 MMAs of K = 8)
constexpr int TC_STAGES = 4;
constexpr int TC_THREADS = 256;
constexpr int TC_MAXN = 384;     // rows of the staged tile: 4 stages x 8 x (16 Rt + 16) B must fit 227 KB of shared memory
                                 // (Rt = 384: 197 KB; the 512 TMEM columns of a CTA would allow 512)

struct FcTcParams {
  const float* xbar;     // [G][CS][N][SPC]
  float* xc;             // [G][SPC][N][Kp]   centred, TF32-rounded, K-major
  const double* cmean;   // [G][N][SPC]
  const double* mean;    // [G][N][SPC] running mean (before this chunk)
  double* M;             // [G][SPC][N][N]
  int64_t cnt;
  int32_t n_c, CS, Kp, N, SPC, G;
  int32_t Rt;            // rows of the shared-memory tile: N rounded up to 128
  int32_t Np;            // MMA N extent: N rounded up to 16
  int32_t tmem_cols;     // power of two >= max(32, Np)
};

__device__ __forceinline__ float to_tf32(float x) {
  uint32_t r;
  asm("cvt.rna.tf32.f32 %0, %1;" : "=r"(r) : "f"(x));
  return __uint_as_float(r);
}

// grid (G, ceil(N SPC / 32), ceil(n_c / PACK_Q)), block (32, 8): a 32-column x PACK_Q-sample tile per block, all
// its loads in flight before the first store (16 per thread), 512-byte runs on the way out
constexpr int PACK_Q = 128;
__global__ void __launch_bounds__(256) fc_pack_tf32_kernel(FcTcParams P) {
  __shared__ float tile[PACK_Q][33];
  const int g = blockIdx.x;
  const int row = P.N * P.SPC;
  const int idx0 = blockIdx.y * 32, q0 = blockIdx.z * PACK_Q;
  const int tx = threadIdx.x, ty = threadIdx.y;
  {
    const int idx = idx0 + tx;
    const double cm = idx < row ? P.cmean[(size_t)g * row + idx] : 0.0;
    const float* x = P.xbar + (size_t)g * P.CS * row + idx;
    float v[PACK_Q / 8];
#pragma unroll
    for (int i = 0; i < PACK_Q / 8; ++i) {
      const int q = q0 + ty + 8 * i;
      v[i] = (idx < row && q < P.n_c) ? x[(size_t)q * row] : 0.0f;
    }
#pragma unroll
    for (int i = 0; i < PACK_Q / 8; ++i) {
      const int q = q0 + ty + 8 * i;
      tile[ty + 8 * i][tx] = (idx < row && q < P.n_c) ? to_tf32((float)((double)v[i] - cm)) : 0.0f;
    }
  }
  __syncthreads();
#pragma unroll
  for (int i = 0; i < 4; ++i) {
    const int c = ty + 8 * i, idx = idx0 + c;
    if (idx >= row) continue;
    const int k = idx / P.SPC, s = idx % P.SPC;
    float* dst = P.xc + (((size_t)g * P.SPC + s) * P.N + k) * P.Kp + q0;
#pragma unroll
    for (int t = 0; t < PACK_Q / 32; ++t)
      if (q0 + 32 * t < P.Kp) dst[32 * t + tx] = tile[32 * t + tx][c];
  }
}

// ---- PTX wrappers (sm_100a) ---------------------------------------------------------------------------------
namespace tc {
__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(uint32_t bar, uint32_t count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count));
}
__device__ __forceinline__ void mbar_wait(uint32_t bar, uint32_t parity) {
  asm volatile(
      "{\n\t.reg .pred p;\n\t"
      "W: mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n\t"
      "@p bra D;\n\tbra W;\n\tD:\n\t}" ::"r"(bar), "r"(parity) : "memory");
}
__device__ __forceinline__ void cp_async16(uint32_t dst, const void* src) {
  asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(dst), "l"(src) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
template <int NN>
__device__ __forceinline__ void cp_async_wait() { asm volatile("cp.async.wait_group %0;" ::"n"(NN) : "memory"); }
__device__ __forceinline__ void fence_proxy_async() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }
__device__ __forceinline__ void tc_fence_before() { asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void tc_fence_after() { asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory"); }
// shared-memory matrix descriptor, K-major, no swizzle: core matrix = 8 rows x 16 bytes stored contiguously
// (128 bytes); SBO = byte distance between 8-row groups, LBO = byte distance between the two 16-byte K halves
// of one K = 8 (TF32) instruction.  Bits: [0,14) address >> 4, [16,30) LBO >> 4, [32,46) SBO >> 4,
// [46,48) descriptor version 1 (Blackwell), [61,64) layout type 0 (no swizzle).
__device__ __forceinline__ uint64_t smem_desc(uint32_t addr, uint32_t lbo, uint32_t sbo) {
  return (uint64_t)((addr >> 4) & 0x3FFF) | ((uint64_t)((lbo >> 4) & 0x3FFF) << 16) |
         ((uint64_t)((sbo >> 4) & 0x3FFF) << 32) | ((uint64_t)1 << 46);
}
// instruction descriptor, kind::tf32: D = F32 (bits [4,6) = 1), A and B = TF32 (bits [7,10), [10,13) = 2),
// both K-major (bits 15, 16 = 0), N >> 3 in bits [17,23), M >> 4 in bits [24,29)
__device__ __forceinline__ uint32_t instr_desc_tf32(int M, int N) {
  return (1u << 4) | (2u << 7) | (2u << 10) | ((uint32_t)(N >> 3) << 17) | ((uint32_t)(M >> 4) << 24);
}
__device__ __forceinline__ void mma_tf32(uint32_t d_tmem, uint64_t adesc, uint64_t bdesc, uint32_t idesc, uint32_t acc) {
  asm volatile(
      "{\n\t.reg .pred p;\n\tsetp.ne.b32 p, %4, 0;\n\t"
      "tcgen05.mma.cta_group::1.kind::tf32 [%0], %1, %2, %3, p;\n\t}" ::"r"(d_tmem), "l"(adesc), "l"(bdesc),
      "r"(idesc), "r"(acc) : "memory");
}
__device__ __forceinline__ void mma_commit(uint32_t bar) {
  asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" ::"r"(bar) : "memory");
}
__device__ __forceinline__ void tmem_ld32(uint32_t taddr, uint32_t (&v)[32]) {
  asm volatile(
      "tcgen05.ld.sync.aligned.32x32b.x32.b32 {%0, %1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15, "
      "%16, %17, %18, %19, %20, %21, %22, %23, %24, %25, %26, %27, %28, %29, %30, %31}, [%32];"
      : "=r"(v[0]), "=r"(v[1]), "=r"(v[2]), "=r"(v[3]), "=r"(v[4]), "=r"(v[5]), "=r"(v[6]), "=r"(v[7]), "=r"(v[8]),
        "=r"(v[9]), "=r"(v[10]), "=r"(v[11]), "=r"(v[12]), "=r"(v[13]), "=r"(v[14]), "=r"(v[15]), "=r"(v[16]),
        "=r"(v[17]), "=r"(v[18]), "=r"(v[19]), "=r"(v[20]), "=r"(v[21]), "=r"(v[22]), "=r"(v[23]), "=r"(v[24]),
        "=r"(v[25]), "=r"(v[26]), "=r"(v[27]), "=r"(v[28]), "=r"(v[29]), "=r"(v[30]), "=r"(v[31])
      : "r"(taddr) : "memory");
  asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
}
}  // namespace tc

// Shared-memory tile of one stage: Rt rows x TC_BK samples as 8 K-columns of 16 bytes; within a K-column row r
// sits at byte 16 r (8-row core matrices back to back, SBO = 128), K-columns are LBO = 16 Rt + 16 bytes apart
// (the extra 16 bytes rotate the banks so the 8 lanes that copy one 128-byte global row do not collide).
__host__ __device__ inline uint32_t tc_lbo(int Rt) { return (uint32_t)Rt * 16u + 16u; }
__host__ __device__ inline uint32_t tc_stage_bytes(int Rt) { return 8u * tc_lbo(Rt); }
__host__ inline size_t tc_smem_bytes(int Rt, int Np) {
  return (size_t)TC_STAGES * tc_stage_bytes(Rt) + (size_t)Np * sizeof(double) + TC_STAGES * sizeof(uint64_t) + 16;
}

// grid (G SPC, Rt / 128), TC_THREADS threads
__global__ void __launch_bounds__(TC_THREADS) fc_xtx_tc_kernel(FcTcParams P) {
  extern __shared__ __align__(128) uint8_t smem[];
  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  const int mb = blockIdx.y, gs = blockIdx.x;
  const int g = gs / P.SPC, sl = gs % P.SPC;
  const int N = P.N;
  const uint32_t LBO = tc_lbo(P.Rt), SB = tc_stage_bytes(P.Rt);
  double* delta = reinterpret_cast<double*>(smem + (size_t)TC_STAGES * SB);
  uint64_t* mbar = reinterpret_cast<uint64_t*>(delta + P.Np);
  uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(mbar + TC_STAGES);
  const uint32_t sbase = tc::smem_u32(smem);
  const uint32_t bar0 = tc::smem_u32(mbar);

  // ---- one-time setup: TMEM columns, stage barriers, delta = chunk mean - running mean, zero rows >= N ----
  if (warp == 0) {
    asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(tc::smem_u32(tmem_slot)),
                 "r"((uint32_t)P.tmem_cols) : "memory");
    asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
  }
  if (tid == 32) {
    for (int i = 0; i < TC_STAGES; ++i) tc::mbar_init(bar0 + 8 * i, 1);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  {
    const size_t row = (size_t)N * P.SPC;
    const double* cm = P.cmean + (size_t)g * row + sl;
    const double* mean = P.mean + (size_t)g * row + sl;
    for (int l = tid; l < P.Np; l += TC_THREADS)
      delta[l] = (l < N && P.cnt > 0) ? cm[(size_t)l * P.SPC] - mean[(size_t)l * P.SPC] : 0.0;
    const int pad = P.Rt - N;
    for (int i = tid; i < TC_STAGES * 8 * pad; i += TC_THREADS) {
      const int st = i / (8 * pad), rem = i % (8 * pad), c = rem / pad, r = N + rem % pad;
      *reinterpret_cast<float4*>(smem + (size_t)st * SB + (size_t)c * LBO + (size_t)r * 16) = make_float4(0.f, 0.f, 0.f, 0.f);
    }
  }

  const float* xsrc = P.xc + (size_t)gs * N * P.Kp;
  const int nkb = (P.n_c + TC_BK - 1) / TC_BK;
  auto load_stage = [&](int kb) {
    const uint32_t dst0 = sbase + (uint32_t)(kb % TC_STAGES) * SB;
    const float* src0 = xsrc + (size_t)kb * TC_BK;
    for (int i = tid; i < N * 8; i += TC_THREADS) {
      const int r = i >> 3, c = i & 7;
      tc::cp_async16(dst0 + (uint32_t)c * LBO + (uint32_t)r * 16u, src0 + (size_t)r * P.Kp + c * 4);
    }
  };
  for (int p = 0; p < TC_STAGES - 1; ++p) {
    if (p < nkb) load_stage(p);
    tc::cp_async_commit();
  }
  tc::tc_fence_before();
  __syncthreads();
  tc::tc_fence_after();
  const uint32_t tmem = *tmem_slot;
  const int n1 = P.Np > 256 ? 256 : P.Np, n2 = P.Np - n1;
  const uint32_t id1 = tc::instr_desc_tf32(128, n1), id2 = tc::instr_desc_tf32(128, n2);

  // ---- main loop: wait for the stage, issue its MMAs, refill the stage the previous MMAs have released ----
  for (int kb = 0; kb < nkb; ++kb) {
    tc::cp_async_wait<TC_STAGES - 2>();
    tc::fence_proxy_async();
    __syncthreads();
    if (tid == 0) {
      tc::tc_fence_after();
      const uint32_t st0 = sbase + (uint32_t)(kb % TC_STAGES) * SB;
#pragma unroll
      for (int kk = 0; kk < TC_BK / 8; ++kk) {
        const uint32_t kbase = st0 + (uint32_t)(2 * kk) * LBO;
        const uint64_t ad = tc::smem_desc(kbase + (uint32_t)mb * 128u * 16u, LBO, 128);
        const uint32_t acc = (kb > 0 || kk > 0) ? 1u : 0u;
        tc::mma_tf32(tmem, ad, tc::smem_desc(kbase, LBO, 128), id1, acc);
        if (n2 > 0) tc::mma_tf32(tmem + 256u, ad, tc::smem_desc(kbase + 256u * 16u, LBO, 128), id2, acc);
      }
      tc::mma_commit(bar0 + 8 * (kb % TC_STAGES));
    }
    const int nk = kb + TC_STAGES - 1;
    if (nk < nkb) {
      if (kb >= 1) tc::mbar_wait(bar0 + 8 * ((kb - 1) % TC_STAGES), (uint32_t)(((kb - 1) / TC_STAGES) & 1));
      load_stage(nk);
    }
    tc::cp_async_commit();
  }
  tc::mbar_wait(bar0 + 8 * ((nkb - 1) % TC_STAGES), (uint32_t)(((nkb - 1) / TC_STAGES) & 1));
  tc::tc_fence_after();

  // ---- epilogue: TMEM -> registers (thread = output row, 32 columns per tcgen05.ld) -> a 32 x 32 transpose
  // through the (now free) stage memory -> lanes = 32 consecutive columns of one row, so every read-modify-write
  // of the FP64 accumulator is one contiguous 256-byte run per warp instruction; Chan merge in FP64 ----
  {
    const int lq = warp & 3, ch = warp >> 2;
    const int r0 = mb * 128 + lq * 32;                // first output row of this warp
    const int ng = (P.Np + 31) / 32, gh = (ng + 1) / 2;
    const int gbeg = ch == 0 ? 0 : gh, gend = ch == 0 ? gh : ng;
    if (r0 < N) {                                     // warp-uniform: some row of this warp exists
      float* tile = reinterpret_cast<float*>(smem) + warp * (32 * 33);
      const double f = P.cnt > 0 ? (double)P.cnt * (double)P.n_c / (double)(P.cnt + P.n_c) : 0.0;
      double* Mbase = P.M + (size_t)gs * N * N;
      const int nrow = min(32, N - r0);
      for (int cg = gbeg; cg < gend; ++cg) {
        uint32_t v[32];
        tc::tmem_ld32(tmem + ((uint32_t)(lq * 32) << 16) + (uint32_t)(cg * 32), v);
#pragma unroll
        for (int j = 0; j < 32; ++j) tile[lane * 33 + j] = __uint_as_float(v[j]);
        __syncwarp();
        const int l = cg * 32 + lane;
        if (l < N) {
          const double dl = delta[l];
          double* Mcol = Mbase + (size_t)r0 * N + l;
          for (int rb = 0; rb < nrow; rb += 8) {       // 8 independent loads in flight, then 8 stores
            double m[8];
#pragma unroll
            for (int u = 0; u < 8; ++u)
              if (rb + u < nrow) m[u] = __ldcs(Mcol + (size_t)(rb + u) * N);
#pragma unroll
            for (int u = 0; u < 8; ++u) {
              const int r = rb + u;
              // (dk dl) f: the same bits for (k, l) and (l, k), so M and FC stay symmetric
              if (r < nrow) __stcs(Mcol + (size_t)r * N, m[u] + ((double)tile[r * 33 + lane] + (delta[r0 + r] * dl) * f));
            }
          }
        }
        __syncwarp();
      }
    }
  }
  tc::tc_fence_before();
  __syncthreads();
  if (warp == 0) {
    asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(tmem), "r"((uint32_t)P.tmem_cols) : "memory");
  }
}

}  // namespace tvbx
