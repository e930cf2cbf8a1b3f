"""Independent arbitrary-precision statement of the model, for pinning the oracle (tests only).

Written from the equations as listed in DESIGN.md section 2 / PAPER.md Eqs. (1)-(5): the transfer
function is evaluated with mpmath at 40 digits and its derivatives are obtained by *numerical*
differentiation (mpmath.diff), not by the jet algebra the oracle uses; Eqs. (1)-(2) are written as
literal index sums over the populations, not in the expanded form the oracle uses.
"""
import mpmath as mp

import workloads as wl

mp.mp.dps = 40


def P(params, name):
    return mp.mpf(float(params[wl.PARAM_NAMES.index(name)]))


def poly(params, pop):
    base = len(wl.PARAM_NAMES) + (0 if pop == 0 else 10)
    return [mp.mpf(float(params[base + q])) for q in range(10)]


def tf_parts(params, pop, fe, fi, W):
    """(F, mu_V, sigma_V, tau_V, V_thr) at already-clamped inputs fe, fi (kHz)."""
    gL, Cm = P(params, "g_L"), P(params, "C_m")
    Qe, Te, Ee = P(params, "Q_e"), P(params, "tau_e"), P(params, "E_e")
    Qi, Ti, Ei = P(params, "Q_i"), P(params, "tau_i"), P(params, "E_i")
    Ke = P(params, "p_conn") * P(params, "N_tot") * (1 - P(params, "g_inh"))
    Ki = P(params, "p_conn") * P(params, "N_tot") * P(params, "g_inh")
    EL = P(params, "E_L_e") if pop == 0 else P(params, "E_L_i")
    c = poly(params, pop)
    muGe, muGi = Qe * Te * Ke * fe, Qi * Ti * Ki * fi
    muG = gL + muGe + muGi
    Tm = Cm / muG
    muV = (muGe * Ee + muGi * Ei + gL * EL - W) / muG
    Ue, Ui = Qe * (Ee - muV) / muG, Qi * (Ei - muV) / muG
    Ae, Ai = Ke * fe * (Ue * Te) ** 2, Ki * fi * (Ui * Ti) ** 2
    sV = mp.sqrt(Ae / (2 * (Te + Tm)) + Ai / (2 * (Ti + Tm)))
    TV = (Ae + Ai) / (Ae / (Te + Tm) + Ai / (Ti + Tm))
    TVN = TV * gL / Cm
    m = (muV - P(params, "muV0")) / P(params, "dmuV0")
    s = (sV - P(params, "sV0")) / P(params, "dsV0")
    t = (TVN - P(params, "tauVN0")) / P(params, "dtauVN0")
    Vthr = (c[0] + c[1] * m + c[2] * s + c[3] * t + c[4] * m * m + c[5] * s * s + c[6] * t * t
            + c[7] * m * s + c[8] * m * t + c[9] * s * t)
    F = mp.erfc((Vthr - muV) / (mp.sqrt(2) * sV)) / (2 * TV)
    return F, muV, sV, TV, Vthr


def tf(params, pop, fe, fi, W):
    return tf_parts(params, pop, mp.mpf(fe), mp.mpf(fi), mp.mpf(W))[0]


def tf_derivs(params, pop, fe, fi, W):
    """F and its numerical partial derivatives [F, F_e, F_i, F_ee, F_ei, F_ii] (per kHz)."""
    f = lambda a, b: tf_parts(params, pop, a, b, mp.mpf(W))[0]
    fe, fi = mp.mpf(fe), mp.mpf(fi)
    h = mp.mpf(10) ** -12
    return [f(fe, fi),
            mp.diff(f, (fe, fi), (1, 0), h=h), mp.diff(f, (fe, fi), (0, 1), h=h),
            mp.diff(f, (fe, fi), (2, 0), h=h), mp.diff(f, (fe, fi), (1, 1), h=h),
            mp.diff(f, (fe, fi), (0, 2), h=h)]


def rhs_node(params, y, drive_extra=0):
    """dy/dt of one isolated node, y = [E, I, C_ee, C_ei, C_ii, W_e, W_i] (mpf), Eqs. (1)-(3) as
    literal sums.  drive_extra = G*c_k + wNoise*OU added to the excitatory input (Eq. (5))."""
    E, I, Cee, Cei, Cii, We, Wi = y
    T = P(params, "T")
    kap = P(params, "kappa")
    eps = P(params, "eps_nu")
    nu = [E, I]
    c = [[Cee, Cei], [Cei, Cii]]
    Npop = [P(params, "N_tot") * (1 - P(params, "g_inh")), P(params, "N_tot") * P(params, "g_inh")]
    cF = [[P(params, "c_Fee"), P(params, "c_Fei")], [P(params, "c_Fie"), P(params, "c_Fii")]]
    Wad = [We, Wi]
    F, dF, d2F, muV = [], [], [], []
    for mu in range(2):
        xe = E + drive_extra + cF[mu][0]
        xi = I + cF[mu][1]
        se, si = (1 if xe > 0 else 0), (1 if xi > 0 else 0)
        fe, fi = max(xe, 0) + eps, max(xi, 0) + eps
        d = tf_derivs(params, mu, fe, fi, Wad[mu])
        F.append(d[0])
        dF.append([kap * se * d[1], kap * si * d[2]])
        d2F.append([[kap * kap * se * se * d[3], kap * kap * se * si * d[4]],
                    [kap * kap * se * si * d[4], kap * kap * si * si * d[5]]])
        muV.append(tf_parts(params, mu, fe, fi, Wad[mu])[1])
    dnu = []
    for mu in range(2):    # Eq. (1)
        acc = F[mu] - nu[mu]
        for lam in range(2):
            for eta in range(2):
                acc += mp.mpf(1) / 2 * c[lam][eta] * d2F[mu][lam][eta]
        dnu.append(acc / T)
    dc = [[0, 0], [0, 0]]
    for lam in range(2):   # Eq. (2)
        for eta in range(2):
            acc = (F[lam] * (1 / T - F[eta]) / Npop[lam] if lam == eta else 0)
            acc += (F[lam] - nu[lam]) * (F[eta] - nu[eta])
            for mu in range(2):
                acc += dF[lam][mu] * c[eta][mu] + dF[eta][mu] * c[lam][mu]
            acc -= 2 * c[lam][eta]
            dc[lam][eta] = acc / T
    twe, twi = P(params, "tau_w_e"), P(params, "tau_w_i")
    dWe = -We / twe + P(params, "b_e") * E + P(params, "a_e") * (muV[0] - P(params, "E_L_e")) / twe   # Eq. (3), A9
    dWi = -Wi / twi + P(params, "b_i") * I + P(params, "a_i") * (muV[1] - P(params, "E_L_i")) / twi
    return [dnu[0], dnu[1], dc[0][0], dc[0][1], dc[1][1], dWe, dWi]
