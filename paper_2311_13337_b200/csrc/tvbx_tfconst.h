// tvbx_tfconst.h -- host side: the uniform constants of the transfer function, computed once per sweep in FP64 from
// the model parameters (include/tvbx.h, enum tvbx_param_id) and cast to the kernels' arithmetic type.
// PAPER.md Eq. (5), Table 1; readings A1, A2, A4; closed form: DESIGN.md section 6.3.
#pragma once
#include "../../include/tvbx.h"
#include "tvbx_tf.cuh"
#include "tvbx_tf2.cuh"

namespace tvbx_host {

template <typename R>
inline void make_tf_const(const double* dp, tvbx::TFConst<R>& tf) {
  const double Ke = dp[TVBX_P_PCONN] * dp[TVBX_P_NTOT] * (1.0 - dp[TVBX_P_GINH]);
  const double Ki = dp[TVBX_P_PCONN] * dp[TVBX_P_NTOT] * dp[TVBX_P_GINH];
  tf.gL = (R)dp[TVBX_P_GL]; tf.Cm = (R)dp[TVBX_P_CM];
  tf.ae = (R)(dp[TVBX_P_QE] * dp[TVBX_P_TAUE] * Ke); tf.ai = (R)(dp[TVBX_P_QI] * dp[TVBX_P_TAUI] * Ki);
  tf.aeEe = (R)(dp[TVBX_P_QE] * dp[TVBX_P_TAUE] * Ke * dp[TVBX_P_EE]);
  tf.aiEi = (R)(dp[TVBX_P_QI] * dp[TVBX_P_TAUI] * Ki * dp[TVBX_P_EI]);
  tf.Ee = (R)dp[TVBX_P_EE]; tf.Ei = (R)dp[TVBX_P_EI]; tf.Qe = (R)dp[TVBX_P_QE]; tf.Qi = (R)dp[TVBX_P_QI];
  tf.cAe = (R)(Ke * dp[TVBX_P_TAUE] * dp[TVBX_P_TAUE]); tf.cAi = (R)(Ki * dp[TVBX_P_TAUI] * dp[TVBX_P_TAUI]);
  tf.Te = (R)dp[TVBX_P_TAUE]; tf.Ti = (R)dp[TVBX_P_TAUI];
  tf.gL_over_Cm = (R)(dp[TVBX_P_GL] / dp[TVBX_P_CM]);
  tf.m_s = (R)(1.0 / dp[TVBX_P_DMUV0]); tf.m_o = (R)(-dp[TVBX_P_MUV0] / dp[TVBX_P_DMUV0]);
  tf.s_s = (R)(1.0 / dp[TVBX_P_DSV0]);  tf.s_o = (R)(-dp[TVBX_P_SV0] / dp[TVBX_P_DSV0]);
  tf.t_s = (R)(1.0 / dp[TVBX_P_DTVN0]); tf.t_o = (R)(-dp[TVBX_P_TVN0] / dp[TVBX_P_DTVN0]);
  for (int i = 0; i < 10; ++i) { tf.P[0][i] = (R)dp[TVBX_P_POLY_E + i]; tf.P[1][i] = (R)dp[TVBX_P_POLY_I + i]; }
  tf.eps = (R)dp[TVBX_P_EPS_NU];
  tf.same_tau = dp[TVBX_P_TAUE] == dp[TVBX_P_TAUI];
  // closed form (tau_e == tau_i); all in FP64, then cast
  const double tau = dp[TVBX_P_TAUE], gL = dp[TVBX_P_GL], Cm = dp[TVBX_P_CM], Ee = dp[TVBX_P_EE], Ei = dp[TVBX_P_EI];
  const double ae = dp[TVBX_P_QE] * tau * Ke, ai = dp[TVBX_P_QI] * tau * Ki;
  const double de = ai * (Ee - Ei), di = ae * (Ei - Ee);
  const double ke = Ke * tau * tau * dp[TVBX_P_QE] * dp[TVBX_P_QE], ki = Ki * tau * tau * dp[TVBX_P_QI] * dp[TVBX_P_QI];
  tf.EegL = (R)(Ee * gL); tf.EigL = (R)(Ei * gL); tf.de = (R)de; tf.di = (R)di; tf.ke = (R)ke; tf.ki = (R)ki;
  tf.cq_e = (R)(2 * ki * di); tf.cq_i = (R)(2 * ke * de); tf.cq_ee = (R)(2 * ki * di * di); tf.cq_ii = (R)(2 * ke * de * de);
  tf.tau_ae = (R)(tau * ae); tf.tau_ai = (R)(tau * ai); tf.ae2 = (R)(ae * ae); tf.aeai = (R)(ae * ai); tf.ai2 = (R)(ai * ai);
  // polynomial variables: m = (mu_V - muV0)/dmuV0, s = (sigma_V - sV0)/dsV0,
  // t = (tau_V g_L/C_m - tvn0)/dtvn0 = (g_L/dtvn0) (r - r0) with tau_V = tau + C_m r
  const double ms = 1.0 / dp[TVBX_P_DMUV0], ss = 1.0 / dp[TVBX_P_DSV0], ts = gL / dp[TVBX_P_DTVN0];
  tf.muV0 = (R)dp[TVBX_P_MUV0]; tf.sV0 = (R)dp[TVBX_P_SV0]; tf.r0 = (R)((dp[TVBX_P_TVN0] - tau * gL / Cm) / gL);
  const double sc[10] = {1.0, ms, ss, ts, ms * ms, ss * ss, ts * ts, ms * ss, ms * ts, ss * ts};
  for (int i = 0; i < 10; ++i) { tf.C[0][i] = (R)(dp[TVBX_P_POLY_E + i] * sc[i]); tf.C[1][i] = (R)(dp[TVBX_P_POLY_I + i] * sc[i]); }
}

// the same constants for the packed pairs of tvbx_tf2.cuh (.x = excitatory / RS row, .y = inhibitory / FS row)
template <typename R>
inline void make_tf2_const(const double* dp, const tvbx::TFConst<R>& f, tvbx::TF2Const& t) {
  t.gL = (float)f.gL; t.Cm = (float)f.Cm; t.ae = (float)f.ae; t.ai = (float)f.ai; t.aeEe = (float)f.aeEe; t.aiEi = (float)f.aiEi;
  t.Te = (float)f.Te; t.de = (float)f.de; t.di = (float)f.di; t.ke = (float)f.ke; t.ki = (float)f.ki;
  t.EegL = (float)f.EegL; t.EigL = (float)f.EigL; t.cq_e = (float)f.cq_e; t.cq_i = (float)f.cq_i;
  t.cq_ee = (float)f.cq_ee; t.cq_ii = (float)f.cq_ii; t.tau_ae = (float)f.tau_ae; t.tau_ai = (float)f.tau_ai;
  t.ae2 = (float)f.ae2; t.aeai = (float)f.aeai; t.ai2 = (float)f.ai2; t.muV0 = (float)f.muV0; t.sV0 = (float)f.sV0;
  t.r0 = (float)f.r0; t.eps = (float)f.eps; t.m2Te = (float)(-2.0 * dp[TVBX_P_TAUE]); t.pad0 = 0.f;
  for (int i = 0; i < 10; ++i) t.C[i] = make_float2((float)f.C[0][i], (float)f.C[1][i]);
  t.D4 = make_float2(2.f * t.C[4].x, 2.f * t.C[4].y); t.D5 = make_float2(2.f * t.C[5].x, 2.f * t.C[5].y);
  t.D6 = make_float2(2.f * t.C[6].x, 2.f * t.C[6].y);
}

}  // namespace tvbx_host
