// tvbx_noalloc.cu -- tvbx_top_k_noalloc (include/tvbx_noalloc.h): the top-k selection of tvbx_top_k as an entry point that
// allocates nothing.  The scratch of the kernel -- one "taken" flag per score -- is a file-scope static __device__ array.
// Everything that touches that array is in THIS file: in host code its name is only a host-side stand-in for the symbol (a
// kernel handed `g_taken` itself would fault, or quietly use host memory where the GPU can reach it), so the host asks the
// runtime for the device address -- cudaGetSymbolAddress, once per device, with that device current -- and passes that.
#include "tvbx_host.h"
#include "../../include/tvbx_noalloc.h"

#include <cmath>

using namespace tvbx_host;

namespace {

// 1 MiB per GPU that loads the library, until the process exits.  Shared by every call on the device; it keeps the last
// call's flags, which the kernel below clears before use.
static __device__ __align__(256) unsigned char g_taken[TVBX_NOALLOC_MAX_SCORES];

// The selection of tvbx::topk_kernel (tvbx_fc.cuh, reading A23b): one CTA of 1024 threads, k rounds of a
// block-wide arg-max over the S scores, equal scores to the lower index.  Variant: the flags are cleared here, by the
// same CTA, instead of by a memset of a per-sweep buffer.
__global__ void __launch_bounds__(1024) topk_noalloc_kernel(const float* __restrict__ score, unsigned char* __restrict__ taken, int S, int k,
                                                            int32_t* __restrict__ out_idx, float* __restrict__ out_val) {
  __shared__ float sv[1024];
  __shared__ int si[1024];
  for (int i = threadIdx.x; i < S; i += 1024) taken[i] = 0;      // (thread t reads only the flags it cleared itself, plus the
  __syncthreads();                                               // ones thread 0 sets between barriers)
  for (int r = 0; r < k && r < S; ++r) {
    float bv = -INFINITY; int bi = -1;
    for (int i = threadIdx.x; i < S; i += 1024)
      if (!taken[i] && (bi < 0 || score[i] > bv)) { bv = score[i]; bi = i; }      // ascending i: the first maximum wins
    sv[threadIdx.x] = bv; si[threadIdx.x] = bi;
    __syncthreads();
    for (int w = 512; w > 0; w >>= 1) {
      if (threadIdx.x < w) {
        const float ov = sv[threadIdx.x + w]; const int oi = si[threadIdx.x + w];
        const int mi = si[threadIdx.x];
        if (oi >= 0 && (mi < 0 || ov > sv[threadIdx.x] || (ov == sv[threadIdx.x] && oi < mi))) { sv[threadIdx.x] = ov; si[threadIdx.x] = oi; }
      }
      __syncthreads();
    }
    if (threadIdx.x == 0) { out_idx[r] = si[0]; out_val[r] = sv[0]; taken[si[0]] = 1; }
    __syncthreads();
  }
}

// device address of g_taken per device (set up on the first call on that device)
std::mutex g_mu;
std::map<int, unsigned char*> g_addr;

int32_t taken_address(unsigned char** out) {
  int dev = -1;
  TVBX_CU(cudaGetDevice(&dev));
  std::lock_guard<std::mutex> lock(g_mu);
  auto it = g_addr.find(dev);
  if (it == g_addr.end()) {
    unsigned char* p = nullptr;
    TVBX_CU(cudaGetSymbolAddress((void**)&p, g_taken));      // (the current device's copy of the symbol)
    if (p == nullptr) return fail(TVBX_ECUDA, "cudaGetSymbolAddress returned a null address for the scratch array");
    it = g_addr.emplace(dev, p).first;
  }
  *out = it->second;
  return TVBX_OK;
}

}  // namespace

extern "C" int32_t tvbx_top_k_noalloc(const float* scores_dev, int32_t n, int32_t k, int32_t* idx_dev, float* val_dev, void* cuda_stream) {
  if (!scores_dev || !idx_dev || !val_dev) return fail(TVBX_EINVAL, "tvbx_top_k_noalloc: null pointer");
  if (n < 1 || k < 1) return fail(TVBX_EINVAL, "tvbx_top_k_noalloc: n=%d, k=%d (both must be >= 1)", n, k);
  if (n > TVBX_NOALLOC_MAX_SCORES)
    return fail(TVBX_EINVAL, "tvbx_top_k_noalloc: n=%d scores exceed the static scratch array (TVBX_NOALLOC_MAX_SCORES = %d); "
                             "use tvbx_top_k on a sweep for larger inputs", n, (int)TVBX_NOALLOC_MAX_SCORES);
  unsigned char* taken = nullptr;
  int32_t rc = taken_address(&taken);
  if (rc) return rc;
  topk_noalloc_kernel<<<1, 1024, 0, (cudaStream_t)cuda_stream>>>(scores_dev, taken, n, k, idx_dev, val_dev);
  TVBX_CU(cudaGetLastError());
  return TVBX_OK;
}
