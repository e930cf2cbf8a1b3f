// tvbx_tf.cuh -- device-side transfer function of the TVB-AdEx mean field with exact first and
// second partial derivatives (DESIGN.md section 2 steps 3-4; Eq. (5), Table 1 P:68-73,
// section 2.2; readings A1, A2, A8).  Templated on the arithmetic type R (float = product
// path, double = the 1e-9 parity build mode).  Everything lives in registers.
#pragma once
#include <cuda_runtime.h>

namespace tvbx {

// ---- uniform (per-sweep) constants, precomputed on the host in FP64 and cast to R --------------
template <typename R>
struct TFConst {
  R gL, Cm;
  R ae, ai;          // Q_e tau_e K_e, Q_i tau_i K_i          (mu_G = gL + ae*fe + ai*fi)
  R aeEe, aiEi;      // ae*E_e, ai*E_i
  R Ee, Ei, Qe, Qi;
  R cAe, cAi;        // K_e tau_e^2, K_i tau_i^2              (A_x = cA_x f_x U_x^2)
  R Te, Ti;
  R gL_over_Cm;
  R m_s, m_o, s_s, s_o, t_s, t_o;  // normalised variable = raw * _s + _o (A2)
  R P[2][10];        // Table 1 rows (RS, FS)
  R eps;             // input floor (A10)
  int same_tau;      // tau_e == tau_i
};

// ---- second-order jets in (x, y) = (f_e, f_i) ---------------------------------------------------
template <typename R> struct Jet { R v, e, i, ee, ei, ii; };   // full
template <typename R> struct Aff { R v, e, i; };               // affine: second derivatives are 0

template <typename R> __device__ __forceinline__ R tfma(R a, R b, R c);
template <> __device__ __forceinline__ float tfma<float>(float a, float b, float c) { return __fmaf_rn(a, b, c); }
template <> __device__ __forceinline__ double tfma<double>(double a, double b, double c) { return __fma_rn(a, b, c); }

template <typename R> __device__ __forceinline__ Jet<R> jadd(const Jet<R>& a, const Jet<R>& b) {
  return {a.v + b.v, a.e + b.e, a.i + b.i, a.ee + b.ee, a.ei + b.ei, a.ii + b.ii};
}
template <typename R> __device__ __forceinline__ Jet<R> jsub(const Jet<R>& a, const Jet<R>& b) {
  return {a.v - b.v, a.e - b.e, a.i - b.i, a.ee - b.ee, a.ei - b.ei, a.ii - b.ii};
}
template <typename R> __device__ __forceinline__ Jet<R> jscale(const Jet<R>& a, R c) {
  return {a.v * c, a.e * c, a.i * c, a.ee * c, a.ei * c, a.ii * c};
}
// c - a
template <typename R> __device__ __forceinline__ Jet<R> jrsub(R c, const Jet<R>& a) {
  return {c - a.v, -a.e, -a.i, -a.ee, -a.ei, -a.ii};
}
// full x full
template <typename R> __device__ __forceinline__ Jet<R> jmul(const Jet<R>& a, const Jet<R>& b) {
  Jet<R> r;
  r.v = a.v * b.v;
  r.e = tfma(a.e, b.v, a.v * b.e);
  r.i = tfma(a.i, b.v, a.v * b.i);
  R t = a.e * b.e;
  r.ee = tfma(a.ee, b.v, tfma(a.v, b.ee, t + t));
  r.ei = tfma(a.ei, b.v, tfma(a.e, b.i, tfma(a.i, b.e, a.v * b.ei)));
  R u = a.i * b.i;
  r.ii = tfma(a.ii, b.v, tfma(a.v, b.ii, u + u));
  return r;
}
// affine x full
template <typename R> __device__ __forceinline__ Jet<R> jmul(const Aff<R>& a, const Jet<R>& b) {
  Jet<R> r;
  r.v = a.v * b.v;
  r.e = tfma(a.e, b.v, a.v * b.e);
  r.i = tfma(a.i, b.v, a.v * b.i);
  R t = a.e * b.e;
  r.ee = tfma(a.v, b.ee, t + t);
  r.ei = tfma(a.e, b.i, tfma(a.i, b.e, a.v * b.ei));
  R u = a.i * b.i;
  r.ii = tfma(a.v, b.ii, u + u);
  return r;
}
template <typename R> __device__ __forceinline__ Jet<R> jsqr(const Jet<R>& a) {
  Jet<R> r;
  R v2 = a.v + a.v;
  r.v = a.v * a.v;
  r.e = v2 * a.e;
  r.i = v2 * a.i;
  r.ee = tfma(v2, a.ee, (a.e + a.e) * a.e);
  r.ei = tfma(v2, a.ei, (a.e + a.e) * a.i);
  r.ii = tfma(v2, a.ii, (a.i + a.i) * a.i);
  return r;
}
// g(u) given g0 = g(u), g1 = g'(u), g2 = g''(u)
template <typename R> __device__ __forceinline__ Jet<R> jchain(const Jet<R>& u, R g0, R g1, R g2) {
  Jet<R> r;
  r.v = g0;
  r.e = g1 * u.e;
  r.i = g1 * u.i;
  R ge = g2 * u.e, gi = g2 * u.i;
  r.ee = tfma(ge, u.e, g1 * u.ee);
  r.ei = tfma(ge, u.i, g1 * u.ei);
  r.ii = tfma(gi, u.i, g1 * u.ii);
  return r;
}
template <typename R> __device__ __forceinline__ R t_rcp(R x) { return R(1) / x; }
template <typename R> __device__ __forceinline__ R t_sqrt(R x);
template <> __device__ __forceinline__ float t_sqrt<float>(float x) { return sqrtf(x); }
template <> __device__ __forceinline__ double t_sqrt<double>(double x) { return sqrt(x); }
template <typename R> __device__ __forceinline__ R t_erfc(R x);
template <> __device__ __forceinline__ float t_erfc<float>(float x) { return erfcf(x); }
template <> __device__ __forceinline__ double t_erfc<double>(double x) { return erfc(x); }
template <typename R> __device__ __forceinline__ R t_exp(R x);
template <> __device__ __forceinline__ float t_exp<float>(float x) { return expf(x); }
template <> __device__ __forceinline__ double t_exp<double>(double x) { return exp(x); }

template <typename R> __device__ __forceinline__ Jet<R> jrecip(const Jet<R>& u) {
  R r = t_rcp(u.v);
  R r2 = r * r;
  return jchain(u, r, -r2, (r2 + r2) * r);
}

// mu_V alone (value), for the A9b option
template <typename R>
__device__ __forceinline__ R mu_V_only(const TFConst<R>& c, R fe, R fi, R gLEL_mW) {
  return tfma(c.aeEe, fe, tfma(c.aiEi, fi, gLEL_mW)) / tfma(c.ae, fe, tfma(c.ai, fi, c.gL));
}

// F_mu(f_e, f_i, W) as a jet in (f_e, f_i); pop selects (E_L, Table-1 row).  gLEL_mW = g_L*E_L - W.
// Follows DESIGN.md section 2 step 3 line by line.  *muV_out = mu_V.
template <typename R>
__device__ __forceinline__ Jet<R> transfer_function(const TFConst<R>& c, int pop, R fe, R fi,
                                                    R gLEL_mW, R* muV_out) {
  // mu_G = g_L + mu_Ge + mu_Gi (affine), r = 1/mu_G
  const R G = tfma(c.ae, fe, tfma(c.ai, fi, c.gL));
  const R r0 = t_rcp(G);
  const R r2 = r0 * r0, r3 = (r2 + r2) * r0;
  Jet<R> r = {r0, -c.ae * r2, -c.ai * r2, c.ae * c.ae * r3, c.ae * c.ai * r3, c.ai * c.ai * r3};
  // mu_V = (mu_Ge E_e + mu_Gi E_i + g_L E_L - W) / mu_G
  Aff<R> num = {tfma(c.aeEe, fe, tfma(c.aiEi, fi, gLEL_mW)), c.aeEe, c.aiEi};
  Jet<R> muV = jmul(num, r);
  // U_e = Q_e (E_e - mu_V)/mu_G, U_i likewise;  A_x = K_x f_x (U_x tau_x)^2
  Jet<R> Ue = jmul(jrsub(c.Ee, muV), r);
  Jet<R> Ui = jmul(jrsub(c.Ei, muV), r);
  Aff<R> xe = {c.cAe * c.Qe * c.Qe * fe, c.cAe * c.Qe * c.Qe, R(0)};
  Aff<R> xi = {c.cAi * c.Qi * c.Qi * fi, R(0), c.cAi * c.Qi * c.Qi};
  Jet<R> Ae = jmul(xe, jsqr(Ue));
  Jet<R> Ai = jmul(xi, jsqr(Ui));
  // tau_m = C_m / mu_G
  Jet<R> Tm = jscale(r, c.Cm);
  Jet<R> sV, TV, iTV;   // sigma_V, tau_V, 1/tau_V
  if (c.same_tau) {
    // tau_e == tau_i  =>  tau_V = tau_e + tau_m identically, sigma_V^2 = (A_e + A_i) / (2 tau_V)
    TV = Tm; TV.v += c.Te;
    iTV = jrecip(TV);
    Jet<R> S = jadd(Ae, Ai);
    Jet<R> var = jscale(jmul(S, iTV), R(0.5));
    R s = t_sqrt(var.v);
    R is = t_rcp(s);
    sV = jchain(var, s, R(0.5) * is, R(-0.25) * is * t_rcp(var.v));
  } else {
    Jet<R> qe = Tm; qe.v += c.Te; qe = jrecip(qe);
    Jet<R> qi = Tm; qi.v += c.Ti; qi = jrecip(qi);
    Jet<R> D = jadd(jmul(Ae, qe), jmul(Ai, qi));        // = 2 sigma_V^2
    Jet<R> var = jscale(D, R(0.5));
    R s = t_sqrt(var.v);
    R is = t_rcp(s);
    sV = jchain(var, s, R(0.5) * is, R(-0.25) * is * t_rcp(var.v));
    TV = jmul(jadd(Ae, Ai), jrecip(D));
    iTV = jrecip(TV);
  }
  // normalised variables (A2) and the Table-1 polynomial
  const R* P = c.P[pop];
  Jet<R> m = jscale(muV, c.m_s); m.v += c.m_o;
  Jet<R> s = jscale(sV, c.s_s);  s.v += c.s_o;
  Jet<R> t = jscale(TV, c.gL_over_Cm * c.t_s); t.v += c.t_o;
  // gradient of the quadratic form
  const R gm = tfma(R(2) * P[4], m.v, tfma(P[7], s.v, tfma(P[8], t.v, P[1])));
  const R gs = tfma(R(2) * P[5], s.v, tfma(P[7], m.v, tfma(P[9], t.v, P[2])));
  const R gt = tfma(R(2) * P[6], t.v, tfma(P[8], m.v, tfma(P[9], s.v, P[3])));
  Jet<R> V;
  V.v = P[0] + m.v * tfma(P[4], m.v, tfma(P[7], s.v, tfma(P[8], t.v, P[1]))) +
        s.v * tfma(P[5], s.v, tfma(P[9], t.v, P[2])) + t.v * tfma(P[6], t.v, P[3]);
  V.e = tfma(gm, m.e, tfma(gs, s.e, gt * t.e));
  V.i = tfma(gm, m.i, tfma(gs, s.i, gt * t.i));
  // H a_x : rows of the constant Hessian applied to the first derivatives
  const R hme = tfma(R(2) * P[4], m.e, tfma(P[7], s.e, P[8] * t.e));
  const R hse = tfma(R(2) * P[5], s.e, tfma(P[7], m.e, P[9] * t.e));
  const R hte = tfma(R(2) * P[6], t.e, tfma(P[8], m.e, P[9] * s.e));
  const R hmi = tfma(R(2) * P[4], m.i, tfma(P[7], s.i, P[8] * t.i));
  const R hsi = tfma(R(2) * P[5], s.i, tfma(P[7], m.i, P[9] * t.i));
  const R hti = tfma(R(2) * P[6], t.i, tfma(P[8], m.i, P[9] * s.i));
  V.ee = tfma(gm, m.ee, tfma(gs, s.ee, tfma(gt, t.ee, tfma(hme, m.e, tfma(hse, s.e, hte * t.e)))));
  V.ei = tfma(gm, m.ei, tfma(gs, s.ei, tfma(gt, t.ei, tfma(hme, m.i, tfma(hse, s.i, hte * t.i)))));
  V.ii = tfma(gm, m.ii, tfma(gs, s.ii, tfma(gt, t.ii, tfma(hmi, m.i, tfma(hsi, s.i, hti * t.i)))));
  // F = erfc((V_thr - mu_V) / (sqrt(2) sigma_V)) / (2 tau_V)
  Jet<R> isV = jrecip(sV);
  Jet<R> z = jscale(jmul(jsub(V, muV), isV), R(0.70710678118654752440));
  const R g = t_exp(-z.v * z.v) * R(1.1283791670955125739);   // 2/sqrt(pi) e^{-z^2}
  Jet<R> ec = jchain(z, t_erfc(z.v), -g, (g + g) * z.v);
  Jet<R> F = jscale(jmul(ec, iTV), R(0.5));
  *muV_out = muV.v;
  return F;
}

}  // namespace tvbx
