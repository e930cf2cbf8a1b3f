// tvbx_tf.cuh -- device-side transfer function of the TVB-AdEx mean field with exact first and
// second partial derivatives (DESIGN.md section 2 steps 3-4; Eq. (5), Table 1 P:68-73,
// section 2.2; readings A1, A2, A8).  Templated on the arithmetic type R (float = product
// path, double = the 1e-9 parity build mode).  Everything lives in registers.
//
// Two formulations of the same function:
//   tf_closed   tau_e == tau_i (the default): mu_G = A, tau_V = B/A with B = tau*A + C_m,
//               sigma_V^2 = Q / (2 A^3 B) with Q a cubic polynomial of (f_e, f_i); derivatives by
//               closed forms / logarithmic differentiation.
//   tf_jet      general tau_e != tau_i: second-order forward-mode jets through the formulas as written.
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
  // ---- closed form (same_tau) ----
  R EegL, EigL;      // E_e g_L, E_i g_L
  R de, di;          // ai (E_e - E_i) = d p_e / d f_i ;  ae (E_i - E_e) = d p_i / d f_e
  R ke, ki;          // K_e tau^2 Q_e^2, K_i tau^2 Q_i^2
  R cq_e, cq_i;      // 2 ki di, 2 ke de
  R cq_ee, cq_ii;    // 2 ki di^2, 2 ke de^2
  R tau_ae, tau_ai;  // tau ae, tau ai
  R ae2, aeai, ai2;  // ae^2, ae ai, ai^2
  R muV0, sV0, r0;   // centres of the polynomial variables (mu_V, sigma_V, r = 1/mu_G)
  R C[2][10];        // Table 1 rows rescaled to the centred raw variables (mu_V - muV0, sigma_V - sV0, r - r0)
};

template <typename R> struct Jet { R v, e, i, ee, ei, ii; };   // value, d/dfe, d/dfi, second derivatives
template <typename R> struct Aff { R v, e, i; };               // affine: second derivatives are 0

template <typename R> __device__ __forceinline__ R tfma(R a, R b, R c);
template <> __device__ __forceinline__ float tfma<float>(float a, float b, float c) { return __fmaf_rn(a, b, c); }
template <> __device__ __forceinline__ double tfma<double>(double a, double b, double c) { return __fma_rn(a, b, c); }

// ---- scalar helpers.  FP32 uses the SFU approximations (rcp/sqrt/ex2, <= 2 ulp) -- the FP32 parity
// budget is 1e-3; FP64 uses the IEEE operations. ----------------------------------------------------
template <typename R> __device__ __forceinline__ R t_rcp(R x);
template <> __device__ __forceinline__ float t_rcp<float>(float x) {
  float y;
  asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
  return y;
}
template <> __device__ __forceinline__ double t_rcp<double>(double x) { return 1.0 / x; }
template <typename R> __device__ __forceinline__ R t_sqrt(R x);
template <> __device__ __forceinline__ float t_sqrt<float>(float x) {
  float y;
  asm("sqrt.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
  return y;
}
template <> __device__ __forceinline__ double t_sqrt<double>(double x) { return sqrt(x); }
template <typename R> __device__ __forceinline__ R t_erfc(R x);
template <> __device__ __forceinline__ float t_erfc<float>(float x) { return erfcf(x); }
template <> __device__ __forceinline__ double t_erfc<double>(double x) { return erfc(x); }
template <typename R> __device__ __forceinline__ R t_exp(R x);
template <> __device__ __forceinline__ float t_exp<float>(float x) { return __expf(x); }
template <> __device__ __forceinline__ double t_exp<double>(double x) { return exp(x); }

// E0 = erfc(z)/2 and ex = exp(-z^2) together.  FP32: erfc(z) = exp(-z^2) * erfcx(z) with
// erfcx(a) = t R(t), t = 1/(1 + 0.4 a), a = |z|; R is a degree-8 least-squares fit of erfcx(a)/t on
// t in (0, 1] (coefficients from csrc/gen_erfcx_coeffs.py; relative error of t R(t) evaluated in
// FP32 <= 4.7e-7 for all a >= 0), and erfc(-a) = 2 - erfc(a).  FP64: libm.
template <typename R> __device__ __forceinline__ R half_erfc(R z, R* ex);
template <> __device__ __forceinline__ float half_erfc<float>(float z, float* ex) {
  const float e = __expf(-z * z);
  const float t = t_rcp(tfma(0.4f, fabsf(z), 1.0f));
  float p = 5.018728834e-02f;
  p = tfma(p, t, -1.826153469e-01f);
  p = tfma(p, t, 1.686438582e-01f);
  p = tfma(p, t, -5.255410161e-03f);
  p = tfma(p, t, 1.412773411e-01f);
  p = tfma(p, t, 1.685781716e-01f);
  p = tfma(p, t, 2.078385839e-01f);
  p = tfma(p, t, 2.256697733e-01f);
  p = tfma(p, t, 2.256758607e-01f);
  const float h = 0.5f * e * t * p;
  *ex = e;
  return z >= 0.0f ? h : 1.0f - h;
}
template <> __device__ __forceinline__ double half_erfc<double>(double z, double* ex) {
  *ex = exp(-z * z);
  return 0.5 * erfc(z);
}

// mu_V alone (value), for the A9b option
template <typename R>
__device__ __forceinline__ R mu_V_only(const TFConst<R>& c, R fe, R fi, R gLEL_mW) {
  return tfma(c.aeEe, fe, tfma(c.aiEi, fi, gLEL_mW)) / tfma(c.ae, fe, tfma(c.ai, fi, c.gL));
}

// ====================================================================================================
//  Closed form (tau_e == tau_i = tau).  With A = mu_G, r = 1/A, B = tau A + C_m, c0 = g_L E_L - W:
//    mu_V  = (aeEe fe + aiEi fi + c0) r
//    p_e   = (E_e - mu_V) A = (E_e g_L - c0) + de fi          (affine in fi only: the fe terms cancel)
//    p_i   = (E_i - mu_V) A = (E_i g_L - c0) + di fe
//    Q     = ke fe p_e^2 + ki fi p_i^2                         (A_e + A_i = Q r^4)
//    tau_V = B r,  sigma_V^2 = Q r^3 / (2 B),  tau_V^N - tvn0 = g_L (r - r0)
//    F     = erfc(z) / (2 tau_V) = (1/2) erfc(z) * A / B,  z = (V_thr - mu_V) / (sqrt 2 sigma_V)
//  L = ln sigma_V = (ln Q - 3 ln A - ln B)/2 + const gives sigma_x = sigma L_x, sigma_xy = sigma (L_xy + L_x L_y).
//  Cpop = the population's rescaled Table-1 row (TFConst::C[pop]).
// ====================================================================================================
template <typename R>
__device__ __forceinline__ Jet<R> tf_closed(const TFConst<R>& c, const R* __restrict__ Cpop, R fe, R fi,
                                            R c0, R* muV_out) {
  const R A = tfma(c.ae, fe, tfma(c.ai, fi, c.gL));
  const R r = t_rcp(A);
  const R B = tfma(c.Te, A, c.Cm);
  const R iB = t_rcp(B);
  const R muV = tfma(c.aeEe, fe, tfma(c.aiEi, fi, c0)) * r;
  const R pe = tfma(c.de, fi, c.EegL - c0);
  const R pi = tfma(c.di, fe, c.EigL - c0);
  const R t1 = c.ke * pe * pe, t2 = c.ki * pi * pi;
  const R Q = tfma(fe, t1, fi * t2);
  const R Qe = tfma(c.cq_e, fi * pi, t1);
  const R Qi = tfma(c.cq_i, fe * pe, t2);
  const R Qee = c.cq_ee * fi, Qii = c.cq_ii * fe;
  const R Qei = tfma(c.cq_i, pe, c.cq_e * pi);
  const R iQ = t_rcp(Q);
  const R a1 = c.ae * r, a2 = c.ai * r, b1 = c.tau_ae * iB, b2 = c.tau_ai * iB;
  const R q1 = Qe * iQ, q2 = Qi * iQ;
  // L = ln sigma_V
  const R Le = R(0.5) * (q1 - tfma(R(3), a1, b1));
  const R Li = R(0.5) * (q2 - tfma(R(3), a2, b2));
  const R Lee = R(0.5) * tfma(Qee, iQ, tfma(R(3) * a1, a1, tfma(b1, b1, -q1 * q1)));
  const R Lei = R(0.5) * tfma(Qei, iQ, tfma(R(3) * a1, a2, tfma(b1, b2, -q1 * q2)));
  const R Lii = R(0.5) * tfma(Qii, iQ, tfma(R(3) * a2, a2, tfma(b2, b2, -q2 * q2)));
  const R sig = t_sqrt(R(0.5) * (r * r) * (r * Q) * iB);
  const R s_e = sig * Le, s_i = sig * Li;
  const R s_ee = sig * tfma(Le, Le, Lee), s_ei = sig * tfma(Le, Li, Lei), s_ii = sig * tfma(Li, Li, Lii);
  // mu_V: mu_e = ae (E_e - mu_V) r, mu_i = ai (E_i - mu_V) r; second derivatives from (mu_V A)_xy = 0
  const R m_e = a1 * (pe * r), m_i = a2 * (pi * r);
  const R m_ee = R(-2) * a1 * m_e, m_ei = -tfma(a1, m_i, a2 * m_e), m_ii = R(-2) * a2 * m_i;
  // r = 1/A
  const R r_e = -a1 * r, r_i = -a2 * r;
  const R r_ee = R(-2) * a1 * r_e, r_ei = R(-2) * a1 * r_i, r_ii = R(-2) * a2 * r_i;
  // Table-1 polynomial in the centred variables (x, y, w) = (mu_V - muV0, sigma_V - sV0, r - r0)
  const R x = muV - c.muV0, y = sig - c.sV0, w = r - c.r0;
  const R C1 = Cpop[1], C2 = Cpop[2], C3 = Cpop[3], C4 = Cpop[4], C5 = Cpop[5], C6 = Cpop[6], C7 = Cpop[7],
          C8 = Cpop[8], C9 = Cpop[9];
  const R C4x = C4 * x, C5y = C5 * y, C6w = C6 * w;
  const R lm = tfma(C7, y, tfma(C8, w, C1)), ls = tfma(C9, w, C2);     // partial sums reused by V and grad
  const R V = tfma(x, lm + C4x, tfma(y, ls + C5y, tfma(w, C3 + C6w, Cpop[0])));
  const R gm = lm + (C4x + C4x);
  const R gs = tfma(C7, x, ls) + (C5y + C5y);
  const R gt = tfma(C8, x, tfma(C9, y, C3)) + (C6w + C6w);
  const R D4 = C4 + C4, D5 = C5 + C5, D6 = C6 + C6;
  const R hm_e = tfma(D4, m_e, tfma(C7, s_e, C8 * r_e)), hs_e = tfma(D5, s_e, tfma(C7, m_e, C9 * r_e)),
          ht_e = tfma(D6, r_e, tfma(C8, m_e, C9 * s_e));
  const R hm_i = tfma(D4, m_i, tfma(C7, s_i, C8 * r_i)), hs_i = tfma(D5, s_i, tfma(C7, m_i, C9 * r_i)),
          ht_i = tfma(D6, r_i, tfma(C8, m_i, C9 * s_i));
  // u = V_thr - mu_V
  const R u = V - muV;
  const R u_e = tfma(gm, m_e, tfma(gs, s_e, gt * r_e)) - m_e;
  const R u_i = tfma(gm, m_i, tfma(gs, s_i, gt * r_i)) - m_i;
  const R u_ee = tfma(gm, m_ee, tfma(gs, s_ee, tfma(gt, r_ee, tfma(hm_e, m_e, tfma(hs_e, s_e, ht_e * r_e))))) - m_ee;
  const R u_ei = tfma(gm, m_ei, tfma(gs, s_ei, tfma(gt, r_ei, tfma(hm_e, m_i, tfma(hs_e, s_i, ht_e * r_i))))) - m_ei;
  const R u_ii = tfma(gm, m_ii, tfma(gs, s_ii, tfma(gt, r_ii, tfma(hm_i, m_i, tfma(hs_i, s_i, ht_i * r_i))))) - m_ii;
  // z = u / (sqrt2 sigma): with W = 1/(sqrt2 sigma), W_x = -W L_x, W_xy = W (L_x L_y - L_xy)
  const R Wz = R(0.70710678118654752440) * t_rcp(sig);
  const R z = u * Wz;
  const R z_e = Wz * tfma(-u, Le, u_e), z_i = Wz * tfma(-u, Li, u_i);
  const R z_ee = Wz * tfma(u, tfma(Le, Le, -Lee), tfma(R(-2) * u_e, Le, u_ee));
  const R z_ei = Wz * tfma(u, tfma(Le, Li, -Lei), tfma(-u_e, Li, tfma(-u_i, Le, u_ei)));
  const R z_ii = Wz * tfma(u, tfma(Li, Li, -Lii), tfma(R(-2) * u_i, Li, u_ii));
  // E = erfc(z)/2:  E' = -exp(-z^2)/sqrt(pi),  E'' = -2 z E'
  R ex;
  const R E0 = half_erfc<R>(z, &ex);
  const R g0 = R(-0.56418958354775628695) * ex;
  const R zz = -(z + z);
  const R E_e = g0 * z_e, E_i = g0 * z_i;
  const R E_ee = g0 * tfma(zz * z_e, z_e, z_ee), E_ei = g0 * tfma(zz * z_e, z_i, z_ei), E_ii = g0 * tfma(zz * z_i, z_i, z_ii);
  // 1/(2 tau_V) = A/(2B):  Rv = A/B, dRv/dA = C_m/B^2, d2Rv/dA2 = -2 tau C_m / B^3
  const R Rv = A * iB;
  const R RA = c.Cm * iB * iB;
  const R RAA = R(-2) * c.Te * RA * iB;
  const R R_e = RA * c.ae, R_i = RA * c.ai;
  Jet<R> F;
  F.v = E0 * Rv;
  F.e = tfma(E_e, Rv, E0 * R_e);
  F.i = tfma(E_i, Rv, E0 * R_i);
  const R E0RAA = E0 * RAA;
  F.ee = tfma(E_ee, Rv, tfma(E_e + E_e, R_e, E0RAA * c.ae2));
  F.ei = tfma(E_ei, Rv, tfma(E_e, R_i, tfma(E_i, R_e, E0RAA * c.aeai)));
  F.ii = tfma(E_ii, Rv, tfma(E_i + E_i, R_i, E0RAA * c.ai2));
  *muV_out = muV;
  return F;
}

// ====================================================================================================
//  General case: second-order jets in (f_e, f_i) through the formulas as written
// ====================================================================================================
template <typename R> __device__ __forceinline__ Jet<R> jadd(const Jet<R>& a, const Jet<R>& b) {
  return {a.v + b.v, a.e + b.e, a.i + b.i, a.ee + b.ee, a.ei + b.ei, a.ii + b.ii};
}
template <typename R> __device__ __forceinline__ Jet<R> jsub(const Jet<R>& a, const Jet<R>& b) {
  return {a.v - b.v, a.e - b.e, a.i - b.i, a.ee - b.ee, a.ei - b.ei, a.ii - b.ii};
}
template <typename R> __device__ __forceinline__ Jet<R> jscale(const Jet<R>& a, R c) {
  return {a.v * c, a.e * c, a.i * c, a.ee * c, a.ei * c, a.ii * c};
}
template <typename R> __device__ __forceinline__ Jet<R> jrsub(R c, const Jet<R>& a) {   // c - a
  return {c - a.v, -a.e, -a.i, -a.ee, -a.ei, -a.ii};
}
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
template <typename R> __device__ __forceinline__ Jet<R> jrecip(const Jet<R>& u) {
  R r = R(1) / u.v;
  R r2 = r * r;
  return jchain(u, r, -r2, (r2 + r2) * r);
}

// F_mu(f_e, f_i, W) as a jet in (f_e, f_i); P = the population's Table-1 row (TFConst::P[pop]).
// gLEL_mW = g_L*E_L - W.  Follows DESIGN.md section 2 step 3 line by line.  *muV_out = mu_V.
template <typename R>
__device__ __noinline__ Jet<R> tf_jet(const TFConst<R>& c, const R* __restrict__ P, R fe, R fi, R gLEL_mW,
                                      R* muV_out) {
  const R G = tfma(c.ae, fe, tfma(c.ai, fi, c.gL));
  const R r0 = R(1) / G;
  const R r2 = r0 * r0, r3 = (r2 + r2) * r0;
  Jet<R> r = {r0, -c.ae * r2, -c.ai * r2, c.ae * c.ae * r3, c.ae * c.ai * r3, c.ai * c.ai * r3};
  Aff<R> num = {tfma(c.aeEe, fe, tfma(c.aiEi, fi, gLEL_mW)), c.aeEe, c.aiEi};
  Jet<R> muV = jmul(num, r);
  Jet<R> Ue = jmul(jrsub(c.Ee, muV), r);
  Jet<R> Ui = jmul(jrsub(c.Ei, muV), r);
  Aff<R> xe = {c.cAe * c.Qe * c.Qe * fe, c.cAe * c.Qe * c.Qe, R(0)};
  Aff<R> xi = {c.cAi * c.Qi * c.Qi * fi, R(0), c.cAi * c.Qi * c.Qi};
  Jet<R> Ae = jmul(xe, jsqr(Ue));
  Jet<R> Ai = jmul(xi, jsqr(Ui));
  Jet<R> Tm = jscale(r, c.Cm);
  Jet<R> qe = Tm; qe.v += c.Te; qe = jrecip(qe);
  Jet<R> qi = Tm; qi.v += c.Ti; qi = jrecip(qi);
  Jet<R> D = jadd(jmul(Ae, qe), jmul(Ai, qi));        // = 2 sigma_V^2
  Jet<R> var = jscale(D, R(0.5));
  R s0 = sqrt(var.v);
  R is = R(1) / s0;
  Jet<R> sV = jchain(var, s0, R(0.5) * is, R(-0.25) * is / var.v);
  Jet<R> TV = jmul(jadd(Ae, Ai), jrecip(D));
  Jet<R> iTV = jrecip(TV);
  Jet<R> m = jscale(muV, c.m_s); m.v += c.m_o;
  Jet<R> s = jscale(sV, c.s_s);  s.v += c.s_o;
  Jet<R> t = jscale(TV, c.gL_over_Cm * c.t_s); t.v += c.t_o;
  const R gm = tfma(R(2) * P[4], m.v, tfma(P[7], s.v, tfma(P[8], t.v, P[1])));
  const R gs = tfma(R(2) * P[5], s.v, tfma(P[7], m.v, tfma(P[9], t.v, P[2])));
  const R gt = tfma(R(2) * P[6], t.v, tfma(P[8], m.v, tfma(P[9], s.v, P[3])));
  Jet<R> V;
  V.v = P[0] + m.v * tfma(P[4], m.v, tfma(P[7], s.v, tfma(P[8], t.v, P[1]))) +
        s.v * tfma(P[5], s.v, tfma(P[9], t.v, P[2])) + t.v * tfma(P[6], t.v, P[3]);
  V.e = tfma(gm, m.e, tfma(gs, s.e, gt * t.e));
  V.i = tfma(gm, m.i, tfma(gs, s.i, gt * t.i));
  const R hme = tfma(R(2) * P[4], m.e, tfma(P[7], s.e, P[8] * t.e));
  const R hse = tfma(R(2) * P[5], s.e, tfma(P[7], m.e, P[9] * t.e));
  const R hte = tfma(R(2) * P[6], t.e, tfma(P[8], m.e, P[9] * s.e));
  const R hmi = tfma(R(2) * P[4], m.i, tfma(P[7], s.i, P[8] * t.i));
  const R hsi = tfma(R(2) * P[5], s.i, tfma(P[7], m.i, P[9] * t.i));
  const R hti = tfma(R(2) * P[6], t.i, tfma(P[8], m.i, P[9] * s.i));
  V.ee = tfma(gm, m.ee, tfma(gs, s.ee, tfma(gt, t.ee, tfma(hme, m.e, tfma(hse, s.e, hte * t.e)))));
  V.ei = tfma(gm, m.ei, tfma(gs, s.ei, tfma(gt, t.ei, tfma(hme, m.i, tfma(hse, s.i, hte * t.i)))));
  V.ii = tfma(gm, m.ii, tfma(gs, s.ii, tfma(gt, t.ii, tfma(hmi, m.i, tfma(hsi, s.i, hti * t.i)))));
  Jet<R> isV = jrecip(sV);
  Jet<R> z = jscale(jmul(jsub(V, muV), isV), R(0.70710678118654752440));
  const R g = exp(-z.v * z.v) * R(1.1283791670955125739);   // 2/sqrt(pi) e^{-z^2}
  Jet<R> ec = jchain(z, t_erfc(z.v), -g, (g + g) * z.v);
  Jet<R> F = jscale(jmul(ec, iTV), R(0.5));
  *muV_out = muV.v;
  return F;
}

}  // namespace tvbx
