// bench_probes.cu -- MEASUREMENT ONLY (built and loaded by bench.py, not part of libtvbx.so and not exported from
// include/tvbx.h): micro-benchmarks for the peaks MEASURED_PEAKS.json does not carry and the rooflines of DESIGN.md
// section 7 need ("FP32 FMA issue peak ... must be measured by an FMA-chain microbenchmark on
// the box", "L2: measure with a read-only kernel over a 32-64 MB buffer").
//   probe_read_bandwidth : 16-byte ld.global.cg streaming reads of a buffer (the path of the delay gather): L2 -> SM
//                          bandwidth when the buffer fits the 126 MB L2, HBM read bandwidth when it is much larger
//   probe_alu            : FP32-lane throughput of the instruction forms integrate2_kernel is made of, as FP32 lane
//                          operations per clock per SM (nominal 128): packed FFMA2 with three distinct register-pair
//                          operands, FFMA2 with a scalar-broadcast operand, FMUL2, FADD2, scalar FFMA, MUFU.RCP
// Every kernel runs 148 x 4 CTAs of 256 threads (8 warps per scheduler), 8 independent chains per thread.
#include <cuda_runtime.h>
#include <stdint.h>

namespace {

__global__ void __launch_bounds__(512) read_probe_kernel(const float4* __restrict__ p, size_t n16, int passes, float* sink) {
  float acc = 0.f;
  const size_t stride = (size_t)gridDim.x * blockDim.x;
  for (int it = 0; it < passes; ++it) {
    size_t i = blockIdx.x * (size_t)blockDim.x + threadIdx.x;
    for (; i + 3 * stride < n16; i += 4 * stride) {
      const float4 a = __ldcg(p + i), b = __ldcg(p + i + stride), c = __ldcg(p + i + 2 * stride), d = __ldcg(p + i + 3 * stride);
      acc += (a.x + a.w) + (b.x + b.w) + (c.x + c.w) + (d.x + d.w);
    }
    for (; i < n16; i += stride) { const float4 a = __ldcg(p + i); acc += a.x + a.w; }
  }
  if (acc == 12345.678f) *sink = acc;
}

enum { ALU_FFMA2_3REG = 0, ALU_FFMA2_BCAST, ALU_FMUL2, ALU_FADD2, ALU_FFMA, ALU_MUFU_RCP, ALU_KINDS };
constexpr int CHAINS = 8, INNER = 64;

template <int KIND>
__global__ void __launch_bounds__(256) alu_probe_kernel(int iters, float seed, float* sink) {
  float2 x[CHAINS], y[CHAINS];
#pragma unroll
  for (int c = 0; c < CHAINS; ++c) {
    x[c] = make_float2(seed + 0.001f * (float)(threadIdx.x + c), seed - 0.002f * (float)c);
    y[c] = make_float2(0.999f + 1e-6f * (float)(threadIdx.x + c), 1.001f - 1e-6f * (float)(threadIdx.x + c));   // per thread: stays in registers
  }
  const float2 k = make_float2(1.0f + 1e-7f * seed, 1.0f - 1e-7f * seed);
  for (int it = 0; it < iters; ++it) {
#pragma unroll
    for (int u = 0; u < INNER; ++u) {
#pragma unroll
      for (int c = 0; c < CHAINS; ++c) {
        if (KIND == ALU_FFMA2_3REG) x[c] = __ffma2_rn(x[c], y[c], y[(c + 1) % CHAINS]);             // three distinct register pairs
        else if (KIND == ALU_FFMA2_BCAST) x[c] = __ffma2_rn(make_float2(k.x, k.x), x[c], y[c]);      // one scalar-broadcast operand
        else if (KIND == ALU_FMUL2) x[c] = __fmul2_rn(x[c], y[c]);
        else if (KIND == ALU_FADD2) x[c] = __fadd2_rn(x[c], y[c]);
        else if (KIND == ALU_FFMA) { x[c].x = __fmaf_rn(x[c].x, y[c].x, y[c].y); x[c].y = __fmaf_rn(x[c].y, y[c].y, y[c].x); }
        else { float r; asm volatile("rcp.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x[c].x)); x[c].x = r + y[c].x; }      // (+ y: ptxas folds rcp(rcp(x)); the FADD runs on the FMA pipe beside the MUFU)
      }
    }
  }
  float acc = 0.f;
#pragma unroll
  for (int c = 0; c < CHAINS; ++c) acc += x[c].x + x[c].y;
  if (acc == 12345.678f) *sink = acc;
}

// FP32 lane operations one loop body performs per thread
inline double lane_ops(int kind) {
  switch (kind) {
    case ALU_MUFU_RCP: return (double)CHAINS * INNER;            // one MUFU per chain
    default: return 2.0 * CHAINS * INNER;                        // two FP32 lanes per chain step (one packed or two scalar instructions)
  }
}

template <int KIND>
cudaError_t time_alu(int blocks, int iters, float* sink, float* ms) {
  cudaEvent_t a, b;
  cudaEventCreate(&a); cudaEventCreate(&b);
  alu_probe_kernel<KIND><<<blocks, 256>>>(iters / 8 + 1, 0.5f, sink);      // warm-up
  cudaEventRecord(a);
  alu_probe_kernel<KIND><<<blocks, 256>>>(iters, 0.5f, sink);
  cudaEventRecord(b);
  cudaError_t e = cudaEventSynchronize(b);
  cudaEventElapsedTime(ms, a, b);
  cudaEventDestroy(a); cudaEventDestroy(b);
  return e != cudaSuccess ? e : cudaGetLastError();
}

}  // namespace

extern "C" {

// GB/s of 16-byte ld.global.cg reads over a zeroed buffer of `bytes` bytes, `passes` times, after a warm-up pass.  0 = ok.
int probe_read_bandwidth(long long bytes, int passes, double* gb_per_s) {
  if (bytes < (1 << 20) || passes < 1 || !gb_per_s) return -1;
  float4* buf = nullptr;
  float* sink = nullptr;
  const size_t n16 = (size_t)bytes / 16;
  if (cudaMalloc(&buf, n16 * 16) != cudaSuccess || cudaMalloc(&sink, 4) != cudaSuccess) { cudaFree(buf); return -2; }
  cudaMemset(buf, 0, n16 * 16);
  int dev = 0, sms = 148;
  cudaGetDevice(&dev);
  cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
  cudaEvent_t a, b;
  cudaEventCreate(&a); cudaEventCreate(&b);
  read_probe_kernel<<<sms * 4, 512>>>(buf, n16, 2, sink);      // warm-up: the buffer is L2-resident afterwards if it fits
  cudaEventRecord(a);
  read_probe_kernel<<<sms * 4, 512>>>(buf, n16, passes, sink);
  cudaEventRecord(b);
  cudaError_t e = cudaEventSynchronize(b);
  float ms = 0.f;
  cudaEventElapsedTime(&ms, a, b);
  cudaEventDestroy(a); cudaEventDestroy(b);
  cudaFree(buf); cudaFree(sink);
  if (e != cudaSuccess || cudaGetLastError() != cudaSuccess) return -3;
  *gb_per_s = (double)n16 * 16.0 * passes / ((double)ms * 1e-3) / 1e9;
  return 0;
}

// kind: 0 FFMA2 (three register pairs), 1 FFMA2 (scalar-broadcast operand), 2 FMUL2, 3 FADD2, 4 scalar FFMA, 5 MUFU.RCP.
// Returns FP32 lane operations per second (all SMs); the caller divides by SMs x clock for lanes per clock per SM.
int probe_alu(int kind, int iters, double* lane_ops_per_s) {
  if (kind < 0 || kind >= ALU_KINDS || iters < 1 || !lane_ops_per_s) return -1;
  int dev = 0, sms = 148;
  cudaGetDevice(&dev);
  cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
  float* sink = nullptr;
  if (cudaMalloc(&sink, 4) != cudaSuccess) return -2;
  const int blocks = sms * 4;
  float ms = 0.f;
  cudaError_t e;
  switch (kind) {
    case ALU_FFMA2_3REG: e = time_alu<ALU_FFMA2_3REG>(blocks, iters, sink, &ms); break;
    case ALU_FFMA2_BCAST: e = time_alu<ALU_FFMA2_BCAST>(blocks, iters, sink, &ms); break;
    case ALU_FMUL2: e = time_alu<ALU_FMUL2>(blocks, iters, sink, &ms); break;
    case ALU_FADD2: e = time_alu<ALU_FADD2>(blocks, iters, sink, &ms); break;
    case ALU_FFMA: e = time_alu<ALU_FFMA>(blocks, iters, sink, &ms); break;
    default: e = time_alu<ALU_MUFU_RCP>(blocks, iters, sink, &ms); break;
  }
  cudaFree(sink);
  if (e != cudaSuccess) return -3;
  *lane_ops_per_s = lane_ops(kind) * (double)iters * 256.0 * (double)blocks / ((double)ms * 1e-3);
  return 0;
}

}  // extern "C"
