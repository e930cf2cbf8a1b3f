// ============================================================================
//  oracle/tvb_adex_oracle.cpp  --  TEST INFRASTRUCTURE, NOT PRODUCT CODE.
//
//  Plain, slow, scalar FP64 CPU statement of what the hot path computes: the
//  batched forward-Euler time stepping of the TVB-AdEx second-order mean-field
//  model with delayed connectome coupling, OU noise, temporal-average
//  downsampling, per-region mean rates and the Pearson FC matrix.
//
//  Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
//  --impl reference legs may load this file.  It shares NO code, header,
//  table or constant generator with the CUDA path (paper_2311_13337_b200/csrc).
//
//  Citations "P:NN" are lines of /root/reference/PAPER.md; "A<n>" are the
//  readings listed in DESIGN.md section 3 (taken from SURVEY.md section 8(c)),
//  used where PAPER.md is silent or garbled.
//
//  PARITY UNPINNED (absolute values only): PAPER.md prints no worked numerical
//  example; the transfer-function internals and default constants (A1-A4) come
//  from the works the paper cites, not from PAPER.md.  Every function below IS
//  pinned by tests/test_oracle_*.py against independent evaluation (mpmath
//  numerical differentiation, closed forms, invariants, an independent Philox),
//  but not against the authors' code, which is not available.
//
//  No blocking, fusion or reordering: loops are sim -> step -> region -> source.
//  OpenMP is used over simulations only (they are independent).
// ============================================================================
#include <cmath>
#include <cstdint>
#include <cstring>
#include <vector>
#include <new>
#ifdef _OPENMP
#include <omp.h>
#endif

namespace {

// ---- parameter vector layout (one vector of NP doubles per simulation) ------
enum Pid {
  P_G = 0, P_B_E, P_A_E, P_TAU_W_E, P_V, P_WNOISE, P_EL_E, P_EL_I, P_T,
  P_CFEE, P_CFEI, P_CFIE, P_CFII,              // c_{F mu,lambda}
  P_B_I, P_A_I, P_TAU_W_I,
  P_GL, P_CM, P_QE, P_TAUE, P_EE, P_QI, P_TAUI, P_EI,
  P_NTOT, P_PCONN, P_GINH,
  P_TAU_OU, P_MU_OU, P_SIGMA_OU,
  P_MUV0, P_DMUV0, P_SV0, P_DSV0, P_TVN0, P_DTVN0,
  P_EPS_NU, P_MUV_LOCAL,
  P_KAPPA,                  // unit of the rates in dF/dnu relative to kHz (A22)
  P_POLY_E,                 // 10 coefficients, Table 1 RS-cell
  P_POLY_I = P_POLY_E + 10, // 10 coefficients, Table 1 FS-cell
  NP = P_POLY_I + 10
};

// ---- second-order forward-mode jet in the two local rates (A8) --------------
// v, d/de, d/di, d2/dede, d2/dedi, d2/didi
struct Jet { double v, e, i, ee, ei, ii; };

inline Jet jconst(double c) { return {c, 0, 0, 0, 0, 0}; }
inline Jet operator+(const Jet& a, const Jet& b) {
  return {a.v + b.v, a.e + b.e, a.i + b.i, a.ee + b.ee, a.ei + b.ei, a.ii + b.ii};
}
inline Jet operator-(const Jet& a, const Jet& b) {
  return {a.v - b.v, a.e - b.e, a.i - b.i, a.ee - b.ee, a.ei - b.ei, a.ii - b.ii};
}
inline Jet operator+(const Jet& a, double c) { Jet r = a; r.v += c; return r; }
inline Jet operator+(double c, const Jet& a) { return a + c; }
inline Jet operator-(const Jet& a, double c) { Jet r = a; r.v -= c; return r; }
inline Jet operator-(double c, const Jet& a) {
  return {c - a.v, -a.e, -a.i, -a.ee, -a.ei, -a.ii};
}
inline Jet operator*(const Jet& a, double c) {
  return {a.v * c, a.e * c, a.i * c, a.ee * c, a.ei * c, a.ii * c};
}
inline Jet operator*(double c, const Jet& a) { return a * c; }
inline Jet operator/(const Jet& a, double c) {
  return {a.v / c, a.e / c, a.i / c, a.ee / c, a.ei / c, a.ii / c};
}
// product rule to second order
inline Jet operator*(const Jet& a, const Jet& b) {
  Jet r;
  r.v  = a.v * b.v;
  r.e  = a.e * b.v + a.v * b.e;
  r.i  = a.i * b.v + a.v * b.i;
  r.ee = a.ee * b.v + 2.0 * a.e * b.e + a.v * b.ee;
  r.ei = a.ei * b.v + a.e * b.i + a.i * b.e + a.v * b.ei;
  r.ii = a.ii * b.v + 2.0 * a.i * b.i + a.v * b.ii;
  return r;
}
// chain rule for a scalar function g(u) with g0=g(u), g1=g'(u), g2=g''(u)
inline Jet jchain(const Jet& u, double g0, double g1, double g2) {
  Jet r;
  r.v  = g0;
  r.e  = g1 * u.e;
  r.i  = g1 * u.i;
  r.ee = g2 * u.e * u.e + g1 * u.ee;
  r.ei = g2 * u.e * u.i + g1 * u.ei;
  r.ii = g2 * u.i * u.i + g1 * u.ii;
  return r;
}
inline Jet jrecip(const Jet& u) {
  double r = 1.0 / u.v;
  return jchain(u, r, -r * r, 2.0 * r * r * r);
}
inline Jet operator/(const Jet& a, const Jet& b) { return a * jrecip(b); }
inline Jet operator/(double c, const Jet& b) { return jrecip(b) * c; }
inline Jet jsqrt(const Jet& u) {
  double s = std::sqrt(u.v);
  return jchain(u, s, 0.5 / s, -0.25 / (s * u.v));
}
inline Jet jerfc(const Jet& u) {
  const double two_over_sqrt_pi = 1.1283791670955125738961589031215;
  double g = std::exp(-u.v * u.v);
  return jchain(u, std::erfc(u.v), -two_over_sqrt_pi * g, 2.0 * two_over_sqrt_pi * u.v * g);
}

// ---- transfer function, A1 (template of [25],[5]; P:84 names mu_V, sigma_V, ---
// tau_V, the 2nd-order polynomial threshold and the Gaussian assumption) ------
// pop: 0 = excitatory (RS, E_L,e, P_e), 1 = inhibitory (FS, E_L,i, P_i).
// fe, fi are the already clamped inputs (A10) carried as jets; Wad = W_mu.
// Returns F_mu as a jet; *muV_out receives the value of mu_V.
Jet transfer_function(const double* p, int pop, const Jet& fe, const Jet& fi, double Wad,
                      double* muV_out) {
  const double gL = p[P_GL], Cm = p[P_CM];
  const double Qe = p[P_QE], Te = p[P_TAUE], Ee = p[P_EE];
  const double Qi = p[P_QI], Ti = p[P_TAUI], Ei = p[P_EI];
  const double Ke = p[P_PCONN] * p[P_NTOT] * (1.0 - p[P_GINH]);
  const double Ki = p[P_PCONN] * p[P_NTOT] * p[P_GINH];
  const double EL = pop == 0 ? p[P_EL_E] : p[P_EL_I];
  const double* P = pop == 0 ? p + P_POLY_E : p + P_POLY_I;

  Jet muGe = (Qe * Te * Ke) * fe;
  Jet muGi = (Qi * Ti * Ki) * fi;
  Jet muG  = gL + muGe + muGi;
  Jet Tm   = Cm / muG;
  Jet muV  = (muGe * Ee + muGi * Ei + (gL * EL - Wad)) / muG;
  Jet Ue   = Qe * (Ee - muV) / muG;
  Jet Ui   = Qi * (Ei - muV) / muG;
  Jet UeTe = Ue * Te, UiTi = Ui * Ti;
  Jet Ae   = Ke * fe * (UeTe * UeTe);
  Jet Ai   = Ki * fi * (UiTi * UiTi);
  Jet TeTm = Te + Tm, TiTm = Ti + Tm;
  Jet sV   = jsqrt(Ae / (2.0 * TeTm) + Ai / (2.0 * TiTm));
  Jet TV   = (Ae + Ai) / (Ae / TeTm + Ai / TiTm);
  Jet TVN  = TV * (gL / Cm);

  Jet m = (muV - p[P_MUV0]) / p[P_DMUV0];
  Jet s = (sV - p[P_SV0]) / p[P_DSV0];
  Jet t = (TVN - p[P_TVN0]) / p[P_DTVN0];
  // Table 1 column order: P0, mu, sigma, tau, mu^2, sigma^2, tau^2, mu.sigma, mu.tau, sigma.tau
  Jet Vthr = P[0] + P[1] * m + P[2] * s + P[3] * t + P[4] * (m * m) + P[5] * (s * s) +
             P[6] * (t * t) + P[7] * (m * s) + P[8] * (m * t) + P[9] * (s * t);

  const double sqrt2 = 1.4142135623730950488016887242097;
  Jet F = jerfc((Vthr - muV) / (sqrt2 * sV)) / (2.0 * TV);
  if (muV_out) *muV_out = muV.v;
  return F;
}

// clamped input as a jet seeded in direction `dir` (0 = e, 1 = i), A10
inline Jet clamp_input(double x, double eps, int dir) {
  const bool pos = x > 0.0;
  Jet j = jconst((pos ? x : double(0.0)) + eps);
  double seed = pos ? 1.0 : 0.0;
  if (dir == 0) j.e = seed; else j.i = seed;
  return j;
}

// ---- Philox4x32-10 and the normal variates, A12 -----------------------------
inline void philox4x32_10(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4]) {
  uint32_t c0 = ctr[0], c1 = ctr[1], c2 = ctr[2], c3 = ctr[3];
  uint32_t k0 = key[0], k1 = key[1];
  for (int r = 0; r < 10; ++r) {
    uint64_t p0 = (uint64_t)0xD2511F53u * c0;
    uint64_t p1 = (uint64_t)0xCD9E8D57u * c2;
    uint32_t n0 = (uint32_t)(p1 >> 32) ^ c1 ^ k0;
    uint32_t n1 = (uint32_t)p1;
    uint32_t n2 = (uint32_t)(p0 >> 32) ^ c3 ^ k1;
    uint32_t n3 = (uint32_t)p0;
    c0 = n0; c1 = n1; c2 = n2; c3 = n3;
    k0 += 0x9E3779B9u; k1 += 0xBB67AE85u;
  }
  out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}
// u(x) = ((x >> 9) + 0.5) * 2^-23: (2k+1)/2^24 with k < 2^23 is exact in FP32 and FP64 (A12 as
// amended in DESIGN.md: 24 bits + 0.5 would need a 25-bit significand).
inline double u23(uint32_t x) { return (double((double)(x >> 9)) + 0.5) * (1.0 / 8388608.0); }

// xi_{s,k,n}: counter = (q_lo, q_hi, region, sim), q = n/4; key = (seed_lo, seed_hi)
double normal_variate(uint64_t seed, int64_t sim, int32_t region, int64_t step) {
  uint64_t q = (uint64_t)step >> 2;
  uint32_t ctr[4] = {(uint32_t)q, (uint32_t)(q >> 32), (uint32_t)region, (uint32_t)sim};
  uint32_t key[2] = {(uint32_t)seed, (uint32_t)(seed >> 32)};
  uint32_t x[4];
  philox4x32_10(ctr, key, x);
  const double two_pi = 6.2831853071795864769252867665590;
  int w = (int)(step & 3);
  uint32_t xa = w < 2 ? x[0] : x[2], xb = w < 2 ? x[1] : x[3];
  double r = std::sqrt(-2.0 * std::log(u23(xa)));
  double th = two_pi * u23(xb);
  return (w & 1) ? r * std::sin(th) : r * std::cos(th);
}

// ---- delay index, A13: d = nearbyint((L/v)/dt), IEEE double, half-to-even ---
inline int32_t delay_index(double L_mm, double v, double dt) {
  return (int32_t)std::nearbyint((L_mm / v) / dt);
}

}  // namespace

// ============================================================================
//  The simulation object (one sweep of S independent simulations)
// ============================================================================
namespace {

struct Edge { int32_t j; double w; int32_t d; };

struct Sim {
  std::vector<double> p;                 // NP parameters
  int64_t ext_id = 0;                    // external sim index (Philox counter word 3)
  int32_t D = 0, H = 1;                  // max delay (steps), ring length D+1
  std::vector<std::vector<Edge>> rows;   // non-zero W_kj in ascending j (A16)
  std::vector<double> y;                 // state [7][N]: E,I,C_ee,C_ei,C_ii,W_e,W_i
  std::vector<double> ou;                // OU state [N]
  std::vector<double> hist;              // ring [H][N] or unwrapped history [(n+1)][N]
  std::vector<double> win_e, win_i;      // running window sums [N]
  std::vector<double> xe, xi;            // kept samples [n_s][N]
};

struct Sweep {
  int32_t N = 0;
  int64_t S = 0;
  std::vector<double> W, L;
  std::vector<Sim> sims;
  double init[7] = {0.001, 0.001, 0, 0, 0, 0, 0};
  uint64_t seed = 0;
  int64_t n = 0;          // global step counter
  double dt = 0.0;        // fixed by the first run
  int32_t unwrapped = 0;  // test variant (pin P6): keep the whole history, no modulo
  bool started = false;
};

void build_tables(Sweep& sw, Sim& sm, double dt) {
  const int N = sw.N;
  sm.rows.assign(N, {});
  int32_t D = 0;
  for (int k = 0; k < N; ++k)
    for (int j = 0; j < N; ++j) {
      double w = sw.W[(size_t)k * N + j];      // u_kj: source j into target k
      if (w == 0.0) continue;                  // zero-weight edges are dropped
      int32_t d = delay_index(sw.L[(size_t)k * N + j], sm.p[P_V], dt);
      sm.rows[k].push_back({j, w, d});
      if (d > D) D = d;
    }
  sm.D = D;
  sm.H = D + 1;
}

void start(Sweep& sw, double dt) {
  const int N = sw.N;
  sw.dt = dt;
  for (auto& sm : sw.sims) {
    build_tables(sw, sm, dt);
    sm.y.assign((size_t)7 * N, 0.0);
    for (int c = 0; c < 7; ++c)
      for (int k = 0; k < N; ++k) sm.y[(size_t)c * N + k] = sw.init[c];
    sm.ou.assign(N, 0.0);                                  // OU_0 = 0 (A11)
    sm.hist.assign((size_t)(sw.unwrapped ? 1 : sm.H) * N, sw.init[0]);  // A14
    sm.win_e.assign(N, 0.0);
    sm.win_i.assign(N, 0.0);
    sm.xe.clear(); sm.xi.clear();
  }
  sw.started = true;
}

// E_j at time index m (m may be negative: constant initial history, A14)
inline double ehist(const Sweep& sw, const Sim& sm, int64_t m, int j) {
  if (m < 0) return sw.init[0];
  if (sw.unwrapped) return sm.hist[(size_t)m * sw.N + j];
  return sm.hist[(size_t)(m % sm.H) * sw.N + j];
}

// one forward-Euler step n -> n+1 of one simulation (A20: all derivatives from
// the state at step n, then all updates)
void step_sim(Sweep& sw, Sim& sm, int64_t n, double dt, int noise_on, int ds,
              int64_t discard_steps, double* traj_row /* [7][N] or null */) {
  const int N = sw.N;
  const double* p = sm.p.data();
  double* E = &sm.y[0 * (size_t)N];  double* I = &sm.y[1 * (size_t)N];
  double* Cee = &sm.y[2 * (size_t)N]; double* Cei = &sm.y[3 * (size_t)N];
  double* Cii = &sm.y[4 * (size_t)N]; double* We = &sm.y[5 * (size_t)N];
  double* Wi = &sm.y[6 * (size_t)N];
  const double T = p[P_T];
  const double Ne = p[P_NTOT] * (1.0 - p[P_GINH]);   // N_lambda of Eq. (2)
  const double Ni = p[P_NTOT] * p[P_GINH];
  std::vector<double> ynew((size_t)7 * N);
  std::vector<double> ounew(N);

  for (int k = 0; k < N; ++k) {
    // 1. coupling, P:82 (ascending j, A16)
    double c = 0.0;
    for (const Edge& e : sm.rows[k]) c += double(e.w) * ehist(sw, sm, n - e.d, e.j);
    // 2. inputs, Eq. (5) P:79 with A5/A6
    const double eta = noise_on ? p[P_WNOISE] * (sm.ou[k]) : double(0.0);
    const double drive = E[k] + p[P_G] * c + eta;
    Jet F[2]; double muV[2];
    for (int mu = 0; mu < 2; ++mu) {
      const double xe = drive + (mu == 0 ? p[P_CFEE] : p[P_CFIE]);
      const double xi = double(I[k]) + (mu == 0 ? p[P_CFEI] : p[P_CFII]);
      Jet fe = clamp_input(xe, p[P_EPS_NU], 0);
      Jet fi = clamp_input(xi, p[P_EPS_NU], 1);
      // 3.-4. transfer function and its exact derivatives (A1, A8)
      F[mu] = transfer_function(p, mu, fe, fi, mu == 0 ? We[k] : Wi[k], &muV[mu]);
      if (p[P_MUV_LOCAL] != 0.0) {   // A9b literal alternative: mu_V(nu_e, nu_i, W) of local rates
        Jet le = clamp_input(E[k], p[P_EPS_NU], 0), li = clamp_input(I[k], p[P_EPS_NU], 1);
        transfer_function(p, mu, le, li, mu == 0 ? We[k] : Wi[k], &muV[mu]);
      }
    }
    // A22: the derivatives of Eqs. (1)-(2) are taken per (1/kappa) kHz: kappa = 1 is the
    // unit-consistent reading, kappa = 1e-3 (default) measures the differentiated rate in Hz.
    const double kap = p[P_KAPPA];
    for (int mu = 0; mu < 2; ++mu) {
      F[mu].e *= double(kap); F[mu].i *= double(kap);
      F[mu].ee *= double(kap * kap); F[mu].ei *= double(kap * kap); F[mu].ii *= double(kap * kap);
    }
    const Jet& Fe = F[0]; const Jet& Fi = F[1];
    // 5. Eq. (1), sums over lambda,eta written out (A7)
    double dE = ((Fe.v - E[k]) + 0.5 * Cee[k] * Fe.ee + Cei[k] * Fe.ei + 0.5 * Cii[k] * Fe.ii) / T;
    double dI = ((Fi.v - I[k]) + 0.5 * Cee[k] * Fi.ee + Cei[k] * Fi.ei + 0.5 * Cii[k] * Fi.ii) / T;
    // 6. Eq. (2)
    double dCee = (Fe.v * (1.0 / T - Fe.v) / Ne + (Fe.v - E[k]) * (Fe.v - E[k]) +
                   2.0 * (Cee[k] * Fe.e + Cei[k] * Fe.i) - 2.0 * Cee[k]) / T;
    double dCii = (Fi.v * (1.0 / T - Fi.v) / Ni + (Fi.v - I[k]) * (Fi.v - I[k]) +
                   2.0 * (Cei[k] * Fi.e + Cii[k] * Fi.i) - 2.0 * Cii[k]) / T;
    double dCei = ((Fe.v - E[k]) * (Fi.v - I[k]) + (Cei[k] * Fe.e + Cii[k] * Fe.i) +
                   (Cee[k] * Fi.e + Cei[k] * Fi.i) - 2.0 * Cei[k]) / T;
    // 7. Eq. (3), with A9 (a-term divided by tau_w)
    double dWe = -We[k] / p[P_TAU_W_E] + p[P_B_E] * E[k] +
                 p[P_A_E] * (muV[0] - p[P_EL_E]) / p[P_TAU_W_E];
    double dWi = -Wi[k] / p[P_TAU_W_I] + p[P_B_I] * I[k] +
                 p[P_A_I] * (muV[1] - p[P_EL_I]) / p[P_TAU_W_I];
    // 8. forward Euler
    ynew[0 * (size_t)N + k] = (E[k] + dt * dE);
    ynew[1 * (size_t)N + k] = (I[k] + dt * dI);
    ynew[2 * (size_t)N + k] = (Cee[k] + dt * dCee);
    ynew[3 * (size_t)N + k] = (Cei[k] + dt * dCei);
    ynew[4 * (size_t)N + k] = (Cii[k] + dt * dCii);
    ynew[5 * (size_t)N + k] = (We[k] + dt * dWe);
    ynew[6 * (size_t)N + k] = (Wi[k] + dt * dWi);
    // 9. exact one-step OU update, Eq. (4) P:58 with A11
    if (noise_on) {
      const double rho = std::exp(-dt / p[P_TAU_OU]);
      const double xi = normal_variate(sw.seed, sm.ext_id, k, n);
      ounew[k] = (p[P_MU_OU] + ((sm.ou[k]) - p[P_MU_OU]) * rho +
                     (p[P_SIGMA_OU] * std::sqrt(1.0 - rho * rho)) * xi);
    } else {
      ounew[k] = sm.ou[k];
    }
  }
  sm.y = ynew;
  sm.ou = ounew;
  // 10. history write: Ehist_k(n+1) = new E_k
  if (sw.unwrapped) {
    sm.hist.resize((size_t)(n + 2) * N);
    for (int k = 0; k < N; ++k) sm.hist[(size_t)(n + 1) * N + k] = sm.y[k];
  } else {
    for (int k = 0; k < N; ++k) sm.hist[(size_t)((n + 1) % sm.H) * N + k] = sm.y[k];
  }
  if (traj_row) std::memcpy(traj_row, sm.y.data(), sizeof(double) * 7 * N);
  // 11. temporal-average downsample of the post-update values (A17)
  if (ds > 0) {
    for (int k = 0; k < N; ++k) {
      sm.win_e[k] = ((sm.win_e[k]) + sm.y[k]);
      sm.win_i[k] = ((sm.win_i[k]) + sm.y[(size_t)N + k]);
    }
    if ((n + 1) % ds == 0) {
      if (n + 1 > discard_steps) {
        for (int k = 0; k < N; ++k) {
          sm.xe.push_back(((sm.win_e[k]) / (double)ds));
          sm.xi.push_back(((sm.win_i[k]) / (double)ds));
        }
      }
      for (int k = 0; k < N; ++k) { sm.win_e[k] = 0.0; sm.win_i[k] = 0.0; }
    }
  }
}

}  // namespace

// ============================================================================
//  C interface (loaded with ctypes by tests/ and bench.py's CPU-baseline leg)
// ============================================================================
extern "C" {

int orc_num_params() { return NP; }

// Equally spaced axis value i of n on [lo, hi] ("values equally spaced within the defined
// range"; A19): lo + i*((hi-lo)/(n-1)), last value forced to hi, n == 1 -> lo.
double orc_axis_value(double lo, double hi, int n, int i) {
  if (n <= 1) return lo;
  if (i == n - 1) return hi;
  double step = (hi - lo) / (double)(n - 1);
  return lo + (double)i * step;
}

// C-order Cartesian product, first axis slowest (A19): digit of axis a for sim index s.
void orc_grid_digits(int n_axes, const int* n_per_axis, long long s, int* digits) {
  for (int a = n_axes - 1; a >= 0; --a) { digits[a] = (int)(s % n_per_axis[a]); s /= n_per_axis[a]; }
}

int orc_delay_index(double L_mm, double v, double dt) { return delay_index(L_mm, v, dt); }

void orc_philox4x32_10(const unsigned* ctr, const unsigned* key, unsigned* out) {
  philox4x32_10(ctr, key, out);
}
double orc_uniform23(unsigned x) { return (u23(x)); }
double orc_normal(unsigned long long seed, long long sim, int region, long long step) {
  return (normal_variate(seed, sim, region, step));
}

// F_mu and derivatives at raw inputs (x_e, x_i) (clamp A10 applied inside), out6 =
// {F, dF/de, dF/di, d2F/dede, d2F/dedi, d2F/didi}; *muV = mu_V.
void orc_tf(const double* params, int pop, double x_e, double x_i, double W, double* out6,
            double* muV) {
  Jet fe = clamp_input(x_e, params[P_EPS_NU], 0), fi = clamp_input(x_i, params[P_EPS_NU], 1);
  double mv;
  Jet F = transfer_function(params, pop, fe, fi, W, &mv);
  if (muV) *muV = (mv);
  out6[0] = (F.v); out6[1] = (F.e); out6[2] = (F.i); out6[3] = (F.ee); out6[4] = (F.ei);
  out6[5] = (F.ii);
}

void* orc_create(int N, const double* W, const double* L_mm, long long S, const double* params,
                 const long long* ext_ids, unsigned long long seed) {
  if (N < 1 || S < 1) return nullptr;
  Sweep* sw = new (std::nothrow) Sweep();
  if (!sw) return nullptr;
  sw->N = N; sw->S = S; sw->seed = seed;
  sw->W.assign(W, W + (size_t)N * N);
  sw->L.assign(L_mm, L_mm + (size_t)N * N);
  sw->sims.resize(S);
  for (long long s = 0; s < S; ++s) {
    sw->sims[s].p.assign(params + (size_t)s * NP, params + (size_t)(s + 1) * NP);
    sw->sims[s].ext_id = ext_ids ? ext_ids[s] : s;
  }
  return sw;
}
void orc_destroy(void* h) { delete (Sweep*)h; }

int orc_set_initial(void* h, const double* init7) {
  Sweep* sw = (Sweep*)h;
  if (sw->started) return -1;
  for (int c = 0; c < 7; ++c) sw->init[c] = init7[c];
  return 0;
}
int orc_set_unwrapped_history(void* h, int on) {
  Sweep* sw = (Sweep*)h;
  if (sw->started) return -1;
  sw->unwrapped = on;
  return 0;
}

// Advance every simulation `steps` steps.  traj (optional): [S][traj_steps][7][N] doubles, the
// post-update state of the first traj_steps steps of THIS call.  Returns 0, or -1 on bad input.
int orc_run(void* h, long long steps, double dt, int noise_on, int ds, long long discard_steps,
            double* traj, long long traj_steps, int n_threads) {
  Sweep* sw = (Sweep*)h;
  if (steps < 0 || !(dt > 0.0) || ds < 0) return -1;
  if (!sw->started) start(*sw, dt);
  else if (dt != sw->dt) return -1;     // delay tables depend on dt
  const int N = sw->N;
  const int64_t n0 = sw->n;
#ifdef _OPENMP
  if (n_threads > 0) omp_set_num_threads(n_threads);
#pragma omp parallel for schedule(dynamic, 1)
#endif
  for (long long s = 0; s < sw->S; ++s) {
    Sim& sm = sw->sims[s];
    for (long long q = 0; q < steps; ++q) {
      double* row = (traj && q < traj_steps)
                        ? traj + ((size_t)s * traj_steps + q) * 7 * N : nullptr;
      step_sim(*sw, sm, n0 + q, dt, noise_on, ds, discard_steps, row);
    }
  }
  sw->n = n0 + steps;
  return 0;
}

long long orc_num_samples(void* h) {
  Sweep* sw = (Sweep*)h;
  return sw->sims.empty() ? 0 : (long long)(sw->sims[0].xe.size() / sw->N);
}
// kept downsampled series of one sim: xe, xi [n_s][N]
void orc_samples(void* h, long long s, double* xe, double* xi) {
  Sweep* sw = (Sweep*)h;
  const Sim& sm = sw->sims[s];
  if (xe) std::memcpy(xe, sm.xe.data(), sizeof(double) * sm.xe.size());
  if (xi) std::memcpy(xi, sm.xi.data(), sizeof(double) * sm.xi.size());
}
void orc_state(void* h, long long s, double* y7N, double* ouN) {
  Sweep* sw = (Sweep*)h;
  const Sim& sm = sw->sims[s];
  if (y7N) std::memcpy(y7N, sm.y.data(), sizeof(double) * sm.y.size());
  if (ouN) std::memcpy(ouN, sm.ou.data(), sizeof(double) * sm.ou.size());
}
int orc_ring_len(void* h, long long s) { return ((Sweep*)h)->sims[s].H; }
long long orc_steps_done(void* h) { return ((Sweep*)h)->n; }

// 12. per-region means and the Pearson matrix of the kept excitatory samples (Eq. (6) P:161;
// "Pearson corr. of time-series firing rate" P:129), plain two-pass definition.
// fc [S][N][N], mean_e/mean_i [S][N].  Degenerate rule A18.  Returns -2 if fewer than 2 samples.
int orc_fc_readout(void* h, double* fc, double* mean_e, double* mean_i) {
  Sweep* sw = (Sweep*)h;
  const int N = sw->N;
  for (long long s = 0; s < sw->S; ++s) {
    const Sim& sm = sw->sims[s];
    const size_t ns = sm.xe.size() / N;
    if (ns < 2) return -2;
    std::vector<double> me(N, 0.0), mi(N, 0.0);
    for (size_t q = 0; q < ns; ++q)
      for (int k = 0; k < N; ++k) { me[k] += sm.xe[q * N + k]; mi[k] += sm.xi[q * N + k]; }
    for (int k = 0; k < N; ++k) { me[k] /= (double)ns; mi[k] /= (double)ns; }
    if (mean_e) std::memcpy(mean_e + (size_t)s * N, me.data(), sizeof(double) * N);
    if (mean_i) std::memcpy(mean_i + (size_t)s * N, mi.data(), sizeof(double) * N);
    if (!fc) continue;
    double* out = fc + (size_t)s * N * N;
    std::vector<double> M((size_t)N * N, 0.0);
    for (int k = 0; k < N; ++k)
      for (int l = 0; l < N; ++l) {
        double acc = 0.0;
        for (size_t q = 0; q < ns; ++q) acc += (sm.xe[q * N + k] - me[k]) * (sm.xe[q * N + l] - me[l]);
        M[(size_t)k * N + l] = acc;
      }
    for (int k = 0; k < N; ++k)
      for (int l = 0; l < N; ++l) {
        if (k == l) { out[(size_t)k * N + l] = 1.0; continue; }
        double den = M[(size_t)k * N + k] * M[(size_t)l * N + l];
        double r = (den > 0.0 && std::isfinite(den)) ? M[(size_t)k * N + l] / std::sqrt(den) : 0.0;
        out[(size_t)k * N + l] = std::isfinite(r) ? r : 0.0;
      }
  }
  return 0;
}


int orc_max_threads() {
#ifdef _OPENMP
  return omp_get_max_threads();
#else
  return 1;
#endif
}

}  // extern "C"
