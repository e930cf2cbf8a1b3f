// tvbx_tf2.cuh -- the closed-form transfer function of tvbx_tf.cuh (tau_e == tau_i) evaluated for BOTH
// populations at once in packed FP32 pairs: every quantity is a float2 whose .x belongs to the
// excitatory population and .y to the inhibitory one, and every arithmetic instruction is one of
// Blackwell's two-wide FP32 operations (FFMA2 / FMUL2 / FADD2, PTX fma/mul/add.rn.f32x2).  The two
// populations run the same formulas on different constants (Table-1 row, E_L, c_F, W), so one
// instruction stream serves both and the FP32 work of a region-step takes half the issue slots.
//
// Same mathematics as tf_closed (Eq. (5), Table 1 P:68-73,
// P:84; readings A1, A2, A8): value, first and second partial derivatives with respect to the two
// input rates (f_e, f_i).
#pragma once
#include <cuda_runtime.h>

namespace tvbx {

typedef float2 f2;

__device__ __forceinline__ f2 mk2(float a, float b) { return make_float2(a, b); }
__device__ __forceinline__ f2 bc2(float a) { return make_float2(a, a); }          // scalar broadcast (free: .F32 operand form)
__device__ __forceinline__ f2 neg2(f2 a) { return make_float2(-a.x, -a.y); }      // folds into an operand modifier
__device__ __forceinline__ f2 fma2(f2 a, f2 b, f2 c) { return __ffma2_rn(a, b, c); }
__device__ __forceinline__ f2 mul2(f2 a, f2 b) { return __fmul2_rn(a, b); }
__device__ __forceinline__ f2 add2(f2 a, f2 b) { return __fadd2_rn(a, b); }
__device__ __forceinline__ f2 sub2(f2 a, f2 b) { return add2(a, neg2(b)); }
__device__ __forceinline__ f2 fms2(f2 a, f2 b, f2 c) { return fma2(a, b, neg2(c)); }    // a*b - c
__device__ __forceinline__ f2 fnma2(f2 a, f2 b, f2 c) { return fma2(neg2(a), b, c); }   // c - a*b
__device__ __forceinline__ f2 scl2(float s, f2 a) { return mul2(bc2(s), a); }

__device__ __forceinline__ float sfu_rcp(float x) { float y; asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x)); return y; }
__device__ __forceinline__ float sfu_sqrt(float x) { float y; asm("sqrt.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x)); return y; }
__device__ __forceinline__ float sfu_ex2(float x) { float y; asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x)); return y; }
__device__ __forceinline__ f2 rcp2(f2 a) { return mk2(sfu_rcp(a.x), sfu_rcp(a.y)); }
__device__ __forceinline__ f2 sqrt2(f2 a) { return mk2(sfu_sqrt(a.x), sfu_sqrt(a.y)); }

// uniform constants of the closed form (scalars are broadcast into both halves by the instruction;
// the Table-1 rows are true pairs: .x = RS row / excitatory, .y = FS row / inhibitory)
struct TF2Const {
  float gL, Cm, ae, ai, aeEe, aiEi, Te, de, di, ke, ki, EegL, EigL, cq_e, cq_i, cq_ee, cq_ii;
  float tau_ae, tau_ai, ae2, aeai, ai2, muV0, sV0, r0, eps;
  float m2Te;          // -2 tau
  float pad0;
  f2 C[10];            // Table-1 rows rescaled to the centred raw variables (mu_V - muV0, sigma_V - sV0, r - r0)
  f2 D4, D5, D6;       // 2 C4, 2 C5, 2 C6
};

struct Jet2 { f2 v, e, i, ee, ei, ii; };

// erfc(z)/2 and exp(-z^2) per half (tvbx_tf.cuh half_erfc<float>: erfc(z) = exp(-z^2) t R(t),
// t = 1/(1 + 0.4|z|), degree-8 fit from csrc/gen_erfcx_coeffs.py, relative error <= 4.7e-7)
__device__ __forceinline__ f2 half_erfc2(f2 z, f2* ex) {
  const f2 zz = mul2(z, z);
  const f2 ez = scl2(-1.4426950408889634f, zz);
  const f2 e = mk2(sfu_ex2(ez.x), sfu_ex2(ez.y));
  const f2 az = mk2(fabsf(z.x), fabsf(z.y));
  const f2 td = fma2(bc2(0.4f), az, bc2(1.0f));
  const f2 t = mk2(sfu_rcp(td.x), sfu_rcp(td.y));
  f2 p = bc2(5.018728834e-02f);
  p = fma2(p, t, bc2(-1.826153469e-01f));
  p = fma2(p, t, bc2(1.686438582e-01f));
  p = fma2(p, t, bc2(-5.255410161e-03f));
  p = fma2(p, t, bc2(1.412773411e-01f));
  p = fma2(p, t, bc2(1.685781716e-01f));
  p = fma2(p, t, bc2(2.078385839e-01f));
  p = fma2(p, t, bc2(2.256697733e-01f));
  p = fma2(p, t, bc2(2.256758607e-01f));
  const f2 h = mul2(mul2(scl2(0.5f, e), t), p);
  *ex = e;
  // erfc(-a)/2 = 1 - erfc(a)/2: result = off + sgn h with sgn = +-1 carrying the sign bit of z and off = (1 - sgn)/2
  const f2 sgn = mk2(__uint_as_float(0x3f800000u | (__float_as_uint(z.x) & 0x80000000u)),
                     __uint_as_float(0x3f800000u | (__float_as_uint(z.y) & 0x80000000u)));
  return fma2(sgn, h, fma2(bc2(-0.5f), sgn, bc2(0.5f)));
}

// F_mu(f_e, f_i, W_mu) for mu = e (.x) and mu = i (.y).  c0 = g_L E_L,mu - W_mu.  *muV_out = mu_V.
__device__ __forceinline__ Jet2 tf_closed2(const TF2Const& c, f2 fe, f2 fi, f2 c0, f2* muV_out) {
  const f2 A = fma2(bc2(c.ae), fe, fma2(bc2(c.ai), fi, bc2(c.gL)));
  const f2 r = rcp2(A);
  const f2 B = fma2(bc2(c.Te), A, bc2(c.Cm));
  const f2 iB = rcp2(B);
  const f2 muV = mul2(fma2(bc2(c.aeEe), fe, fma2(bc2(c.aiEi), fi, c0)), r);
  const f2 pe = fma2(bc2(c.de), fi, sub2(bc2(c.EegL), c0));
  const f2 pi = fma2(bc2(c.di), fe, sub2(bc2(c.EigL), c0));
  const f2 t1 = mul2(scl2(c.ke, pe), pe), t2 = mul2(scl2(c.ki, pi), pi);
  const f2 Q = fma2(fe, t1, mul2(fi, t2));
  const f2 Qe = fma2(bc2(c.cq_e), mul2(fi, pi), t1);
  const f2 Qi = fma2(bc2(c.cq_i), mul2(fe, pe), t2);
  const f2 Qee = scl2(c.cq_ee, fi), Qii = scl2(c.cq_ii, fe);
  const f2 Qei = fma2(bc2(c.cq_i), pe, scl2(c.cq_e, pi));
  const f2 iQ = rcp2(Q);
  const f2 a1 = scl2(c.ae, r), a2 = scl2(c.ai, r), b1 = scl2(c.tau_ae, iB), b2 = scl2(c.tau_ai, iB);
  const f2 q1 = mul2(Qe, iQ), q2 = mul2(Qi, iQ);
  // L = ln sigma_V
  const f2 Le = scl2(0.5f, sub2(q1, fma2(bc2(3.0f), a1, b1)));
  const f2 Li = scl2(0.5f, sub2(q2, fma2(bc2(3.0f), a2, b2)));
  const f2 a1_3 = scl2(3.0f, a1);
  const f2 Lee = scl2(0.5f, fma2(Qee, iQ, fma2(a1_3, a1, fms2(b1, b1, mul2(q1, q1)))));
  const f2 Lei = scl2(0.5f, fma2(Qei, iQ, fma2(a1_3, a2, fms2(b1, b2, mul2(q1, q2)))));
  const f2 Lii = scl2(0.5f, fma2(Qii, iQ, fma2(scl2(3.0f, a2), a2, fms2(b2, b2, mul2(q2, q2)))));
  const f2 sig = sqrt2(mul2(mul2(scl2(0.5f, mul2(r, r)), mul2(r, Q)), iB));
  const f2 s_e = mul2(sig, Le), s_i = mul2(sig, Li);
  const f2 s_ee = mul2(sig, fma2(Le, Le, Lee)), s_ei = mul2(sig, fma2(Le, Li, Lei)), s_ii = mul2(sig, fma2(Li, Li, Lii));
  // mu_V: mu_e = ae (E_e - mu_V) r, mu_i = ai (E_i - mu_V) r, and r = 1/A: r_e = -a1 r, r_i = -a2 r.
  // Their second derivatives are multiples of the first ones -- (mu_V A)_xy = 0 gives m_ee = -2 a1 m_e,
  // m_ei = -(a1 m_i + a2 m_e), m_ii = -2 a2 m_i, and r_ee = -2 a1 r_e, r_ei = -(a1 r_i + a2 r_e), r_ii = -2 a2 r_i --
  // so they are never formed: they enter u_xy below through t_x = (g_m - 1) m_x + g_t r_x.
  const f2 m_e = mul2(a1, mul2(pe, r)), m_i = mul2(a2, mul2(pi, r));
  const f2 r_e = neg2(mul2(a1, r)), r_i = neg2(mul2(a2, r));
  // Table-1 polynomial in the centred variables (x, y, w) = (mu_V - muV0, sigma_V - sV0, r - r0)
  const f2 x = sub2(muV, bc2(c.muV0)), y = sub2(sig, bc2(c.sV0)), w = sub2(r, bc2(c.r0));
  // gradient first; the value then follows from Euler's identity for a quadratic form:
  // V - C0 = lin + quad and x gm + y gs + w gt = lin + 2 quad  =>  V = C0 + (x (gm + C1) + y (gs + C2) + w (gt + C3)) / 2
  const f2 gm = fma2(c.D4, x, fma2(c.C[7], y, fma2(c.C[8], w, c.C[1])));
  const f2 gs = fma2(c.D5, y, fma2(c.C[7], x, fma2(c.C[9], w, c.C[2])));
  const f2 gt = fma2(c.D6, w, fma2(c.C[8], x, fma2(c.C[9], y, c.C[3])));
  const f2 V = fma2(bc2(0.5f), fma2(x, add2(gm, c.C[1]), fma2(y, add2(gs, c.C[2]), mul2(w, add2(gt, c.C[3])))), c.C[0]);
  const f2 hm_e = fma2(c.D4, m_e, fma2(c.C[7], s_e, mul2(c.C[8], r_e))), hs_e = fma2(c.D5, s_e, fma2(c.C[7], m_e, mul2(c.C[9], r_e))),
           ht_e = fma2(c.D6, r_e, fma2(c.C[8], m_e, mul2(c.C[9], s_e)));
  const f2 hm_i = fma2(c.D4, m_i, fma2(c.C[7], s_i, mul2(c.C[8], r_i))), hs_i = fma2(c.D5, s_i, fma2(c.C[7], m_i, mul2(c.C[9], r_i))),
           ht_i = fma2(c.D6, r_i, fma2(c.C[8], m_i, mul2(c.C[9], s_i)));
  // u = V_thr - mu_V
  const f2 u = sub2(V, muV);
  const f2 gm1 = sub2(gm, bc2(1.0f));             // d(V_thr - mu_V)/d mu_V
  // u_x = t_x + g_s s_x;  u_xy = g_m1 m_xy + g_t r_xy + g_s s_xy + (grad_x)^T H (grad_y)
  //      with g_m1 m_xy + g_t r_xy = -2 a1 t_e (ee), -(a1 t_i + a2 t_e) (ei), -2 a2 t_i (ii)
  const f2 t_e = fma2(gm1, m_e, mul2(gt, r_e)), t_i = fma2(gm1, m_i, mul2(gt, r_i));
  const f2 u_e = fma2(gs, s_e, t_e), u_i = fma2(gs, s_i, t_i);
  const f2 q_ee = fma2(hm_e, m_e, fma2(hs_e, s_e, mul2(ht_e, r_e)));
  const f2 q_ei = fma2(hm_e, m_i, fma2(hs_e, s_i, mul2(ht_e, r_i)));
  const f2 q_ii = fma2(hm_i, m_i, fma2(hs_i, s_i, mul2(ht_i, r_i)));
  const f2 u_ee = fma2(scl2(-2.0f, a1), t_e, fma2(gs, s_ee, q_ee));
  const f2 u_ei = fnma2(a1, t_i, fnma2(a2, t_e, fma2(gs, s_ei, q_ei)));
  const f2 u_ii = fma2(scl2(-2.0f, a2), t_i, fma2(gs, s_ii, q_ii));
  // z = u Wz with Wz = 1/(sqrt2 sigma), Wz_x = -Wz L_x, Wz_xy = Wz (L_x L_y - L_xy):  z_x = Wz zh_x, z_xy = Wz zh_xy with
  // zh_x = u_x - u L_x,  zh_xy = u (L_x L_y - L_xy) - u_x L_y - u_y L_x + u_xy   (Wz is applied once, in G1 below)
  const f2 Wz = scl2(0.70710678118654752440f, rcp2(sig));
  const f2 z = mul2(u, Wz);
  const f2 zh_e = fnma2(u, Le, u_e), zh_i = fnma2(u, Li, u_i);
  const f2 zh_ee = fma2(u, fms2(Le, Le, Lee), fma2(scl2(-2.0f, u_e), Le, u_ee));
  const f2 zh_ei = fma2(u, fms2(Le, Li, Lei), fnma2(u_e, Li, fnma2(u_i, Le, u_ei)));
  const f2 zh_ii = fma2(u, fms2(Li, Li, Lii), fma2(scl2(-2.0f, u_i), Li, u_ii));
  // E = erfc(z)/2:  E' = -exp(-z^2)/sqrt(pi),  E'' = -2 z E'
  // E_x = E' z_x = G1 zh_x,  E_xy = E'' z_x z_y + E' z_xy = G1 (K zh_x zh_y + zh_xy)  with G1 = E' Wz, K = -2 z Wz
  f2 ex;
  const f2 E0 = half_erfc2(z, &ex);
  const f2 G1 = mul2(scl2(-0.56418958354775628695f, ex), Wz);
  const f2 K = mul2(scl2(-2.0f, z), Wz);
  const f2 kze = mul2(K, zh_e), kzi = mul2(K, zh_i);
  const f2 E_e = mul2(G1, zh_e), E_i = mul2(G1, zh_i);
  const f2 E_ee = mul2(G1, fma2(kze, zh_e, zh_ee)), E_ei = mul2(G1, fma2(kze, zh_i, zh_ei)), E_ii = mul2(G1, fma2(kzi, zh_i, zh_ii));
  // 1/(2 tau_V) = A/(2B):  Rv = A/B, dRv/dA = C_m/B^2, d2Rv/dA2 = -2 tau C_m / B^3
  const f2 Rv = mul2(A, iB);
  const f2 RA = mul2(scl2(c.Cm, iB), iB);
  const f2 RAA = mul2(scl2(c.m2Te, RA), iB);
  const f2 R_e = scl2(c.ae, RA), R_i = scl2(c.ai, RA);
  Jet2 F;
  F.v = mul2(E0, Rv);
  F.e = fma2(E_e, Rv, mul2(E0, R_e));
  F.i = fma2(E_i, Rv, mul2(E0, R_i));
  const f2 E0RAA = mul2(E0, RAA);
  F.ee = fma2(E_ee, Rv, fma2(add2(E_e, E_e), R_e, scl2(c.ae2, E0RAA)));
  F.ei = fma2(E_ei, Rv, fma2(E_e, R_i, fma2(E_i, R_e, scl2(c.aeai, E0RAA))));
  F.ii = fma2(E_ii, Rv, fma2(add2(E_i, E_i), R_i, scl2(c.ai2, E0RAA)));
  *muV_out = muV;
  return F;
}

}  // namespace tvbx
