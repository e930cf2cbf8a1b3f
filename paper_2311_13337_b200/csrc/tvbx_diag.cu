// tvbx_diag.cu -- test hook of include/tvbx_diag.h: the product kernel's packed transfer function tf_closed2
// (tvbx_tf2.cuh) evaluated on the device for a list of input points, so that every output of the jet -- the second
// derivatives included -- can be checked element by element from outside the library (tests/test_gpu_tf2.py).
#include "tvbx_host.h"
#include "tvbx_tfconst.h"

namespace {

using namespace tvbx;

// one thread per point: the same call the integrator makes (tvbx_integrate2.cuh, S2), c0 = g_L E_L,mu - W_mu
__global__ void tf_closed2_probe_kernel(TF2Const c, float2 gLEL, int n, const float* __restrict__ fe, const float* __restrict__ fi,
                                        const float* __restrict__ we, const float* __restrict__ wi, float* __restrict__ out) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  const f2 c0 = sub2(gLEL, mk2(we[i], wi[i]));
  f2 muV;
  const Jet2 F = tf_closed2(c, bc2(fe[i]), bc2(fi[i]), c0, &muV);
  float* o = out + (size_t)i * 14;
  o[0] = F.v.x; o[1] = F.e.x; o[2] = F.i.x; o[3] = F.ee.x; o[4] = F.ei.x; o[5] = F.ii.x; o[6] = muV.x;
  o[7] = F.v.y; o[8] = F.e.y; o[9] = F.i.y; o[10] = F.ee.y; o[11] = F.ei.y; o[12] = F.ii.y; o[13] = muV.y;
}

}  // namespace

namespace tvbx_host {

int32_t diag_tf_closed2(const tvbx_model_params* params, int32_t n, const double* fe, const double* fi, const double* w_e,
                        const double* w_i, double* out) {
  tvbx_model_params mp;
  if (params) mp = *params; else tvbx_default_params(&mp);
  const double* dp = mp.p;
  if (dp[TVBX_P_TAUE] != dp[TVBX_P_TAUI]) return fail(TVBX_EINVAL, "the closed-form transfer function needs tau_e == tau_i");
  int ndev = 0;
  if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev == 0) { cudaGetLastError(); return fail(TVBX_ECUDA, "no CUDA device"); }
  if (n == 0) return TVBX_OK;
  TFConst<float> tf;
  TF2Const t2;
  make_tf_const<float>(dp, tf);
  make_tf2_const<float>(dp, tf, t2);
  std::vector<float> h((size_t)4 * n);
  for (int i = 0; i < n; ++i) { h[i] = (float)fe[i]; h[n + i] = (float)fi[i]; h[2 * n + i] = (float)w_e[i]; h[3 * n + i] = (float)w_i[i]; }
  DevBuf<float> din, dout;
  int64_t dummy = 0;
  TVBX_CU(din.upload(h, &dummy));
  TVBX_CU(dout.alloc((size_t)14 * n));
  const float2 gLEL = make_float2((float)(dp[TVBX_P_GL] * dp[TVBX_P_EL_E]), (float)(dp[TVBX_P_GL] * dp[TVBX_P_EL_I]));
  tf_closed2_probe_kernel<<<(n + 127) / 128, 128>>>(t2, gLEL, n, din.p, din.p + n, din.p + 2 * n, din.p + 3 * n, dout.p);
  TVBX_CU(cudaGetLastError());
  std::vector<float> ho((size_t)14 * n);
  TVBX_CU(cudaMemcpy(ho.data(), dout.p, ho.size() * sizeof(float), cudaMemcpyDeviceToHost));
  for (size_t i = 0; i < ho.size(); ++i) out[i] = (double)ho[i];
  return TVBX_OK;
}

}  // namespace tvbx_host
