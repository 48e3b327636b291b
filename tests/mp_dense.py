"""Independent high-precision restatement of the hot path, used ONLY to validate pins.

mpmath at 50 digits, dense stoichiometric matrices nu' and nu'' (K x I), mp.power for every
power, the equations typed from PAPER.md Eq. 2, 4-9 and SURVEY.md O1-O11.  It shares nothing
with oracle/ or with the CUDA path: a mistake in either shows up as a disagreement here.
"""
from mpmath import mp, mpf, exp, log, log10, power

mp.dps = 50

RGAS = mpf("8.31446261815324e7")
RCAL = mpf("8.31446261815324") / mpf("4.184")
PATM = mpf("1.01325e6")


def dense_nu(mech):
    K, I = mech.n_species, mech.n_reactions
    nup = [[0] * I for _ in range(K)]
    nupp = [[0] * I for _ in range(K)]
    for k in range(I):
        for j in range(mech.reac_ptr[k], mech.reac_ptr[k + 1]):
            nup[int(mech.reac_sp[j])][k] += int(mech.reac_nu[j])
        for j in range(mech.prod_ptr[k], mech.prod_ptr[k + 1]):
            nupp[int(mech.prod_sp[j])][k] += int(mech.prod_nu[j])
    return nup, nupp


def evaluate(mech, T, P, Y, Yin=None, tau=None, Tset=None, lindemann_only=False, M_scale=None, Tin=None):
    """Returns dict with mp values: Wbar, rho, C, Ctot, per-reaction kinf,k0,Pr,Fcent,F,M,Kp,Kc,kf,kr,q,
    wdot, F (K+1 entries, row 0 = T - Tset).  With Tin: also h (erg/g), cp_mix and the energy row F_T
    (steady Eq. 3 of the paper, Qdot = 0, dP/dt = 0, as a residual: F_T = -dT/dt)."""
    K, I = mech.n_species, mech.n_reactions
    T, P = mpf(T), mpf(P)
    Y = [mpf(float(y)) for y in Y]
    W = [mpf(float(w)) for w in mech.W]
    nup, nupp = dense_nu(mech)
    Wbar = 1 / sum(Y[i] / W[i] for i in range(K))
    rho = P * Wbar / (RGAS * T)
    C = [rho * Y[i] / W[i] for i in range(K)]
    Ctot = sum(C)
    hRT, sR = [], []
    for i in range(K):
        a = [mpf(float(v)) for v in mech.nasa[i]]
        hRT.append(a[0] + a[1] * T / 2 + a[2] * T**2 / 3 + a[3] * T**3 / 4 + a[4] * T**4 / 5 + a[5] / T)
        sR.append(a[0] * log(T) + a[1] * T + a[2] * T**2 / 2 + a[3] * T**3 / 3 + a[4] * T**4 / 4 + a[6])
    out = dict(Wbar=Wbar, rho=rho, C=C, Ctot=Ctot, rx=[])
    wdot = [mpf(0)] * K
    for k in range(I):
        arr = lambda A, b, E: mpf(float(A)) * power(T, mpf(float(b))) * exp(-mpf(float(E)) / (RCAL * T))
        kinf = arr(mech.A[k], mech.b[k], mech.Ea[k])
        nu = [nupp[i][k] - nup[i][k] for i in range(K)]
        Kp = exp(sum(nu[i] * sR[i] for i in range(K)) - sum(nu[i] * hRT[i] for i in range(K)))
        Kc = Kp * power(PATM / (RGAS * T), sum(nu))
        alpha = [mpf(1)] * K
        for j in range(mech.eff_ptr[k], mech.eff_ptr[k + 1]):
            alpha[int(mech.eff_sp[j])] = mpf(float(mech.eff_val[j]))
        M = sum(alpha[i] * C[i] for i in range(K))
        if M_scale is not None:
            M = M * mpf(M_scale)
        rt = int(mech.rtype[k])
        kf, k0, Pr, Fcent, F = kinf, mpf(0), mpf(0), mpf(1), mpf(1)
        if rt >= 2:
            k0 = arr(mech.A0[k], mech.b0[k], mech.Ea0[k])
            Pr = k0 * M / kinf
            if rt == 3 and not lindemann_only:
                al, T3, T1, T2 = [mpf(float(v)) for v in mech.troe[k]]
                Fcent = (1 - al) * exp(-T / T3) + al * exp(-T / T1) + exp(-T2 / T)
                c = mpf("-0.4") - mpf("0.67") * log10(Fcent)
                n = mpf("0.75") - mpf("1.27") * log10(Fcent)
                d = mpf("0.14")
                f1 = (log10(Pr) + c) / (n - d * (log10(Pr) + c))
                F = power(10, log10(Fcent) / (1 + f1**2))
            kf = kinf * (Pr / (1 + Pr)) * F
        kr = kf / Kc if mech.reversible[k] else mpf(0)
        pf = mpf(1)
        pr = mpf(1)
        for i in range(K):
            pf *= power(C[i], nup[i][k])
            pr *= power(C[i], nupp[i][k])
        q = kf * pf - kr * pr
        if rt == 1:
            q *= M
        for i in range(K):
            wdot[i] = wdot[i] + nu[i] * q
        out["rx"].append(dict(kinf=kinf, k0=k0, Pr=Pr, Fcent=Fcent, F=F, M=M, Kp=Kp, Kc=Kc, kf=kf, kr=kr, q=q))
    out["wdot"] = wdot
    if Yin is not None:
        Yin = [mpf(float(y)) for y in Yin]
        tau = mpf(float(tau))
        Tset = T if Tset is None else mpf(Tset)
        out["F"] = [T - Tset] + [(Y[i] - Yin[i]) / tau - wdot[i] * W[i] / rho for i in range(K)]
        if Tin is not None:
            Tin = mpf(Tin)
            h, hin, cp = [], [], []
            for i in range(K):
                a = [mpf(float(v)) for v in mech.nasa[i]]
                enth = lambda t: (a[0] + a[1] * t / 2 + a[2] * t**2 / 3 + a[3] * t**3 / 4 + a[4] * t**4 / 5 + a[5] / t) * RGAS * t / W[i]
                h.append(enth(T))
                hin.append(enth(Tin))
                cp.append((a[0] + a[1] * T + a[2] * T**2 + a[3] * T**3 + a[4] * T**4) * RGAS / W[i])
            cp_mix = sum(Y[i] * cp[i] for i in range(K))
            rhs = sum(Yin[i] * (hin[i] - h[i]) for i in range(K)) / tau - sum(h[i] * wdot[i] * W[i] for i in range(K)) / rho
            out.update(h=h, cp_mix=cp_mix, FT=-rhs / cp_mix)
    return out


def roundoff_scale(mech, T, P, Y, Yin, tau, Tin=None):
    """The round-off scale S of SURVEY.md 8(c)-J, typed from its definition (not from the oracle):
        S_i = |Y_i - Yin_i|/tau + (W_i/rho) sum_k (nu'_ik + nu''_ik) (|k_f prod C^nu'| + |k_r prod C^nu''|) [x |[M]_k| if three-body]
    for the species rows i = 1..K; S_0 = 0 for the fixed-temperature row, and with Tin the energy row's
        S_0 = [ (1/tau) sum_i |Yin_i (h_in,i - h_i)| + sum_i |h_i| (W_i/rho) sum_k (...)_ik ] / cp_mix .
    Returns K+1 mp values."""
    K, I = mech.n_species, mech.n_reactions
    ev = evaluate(mech, T, P, Y, Yin=Yin, tau=tau, Tin=Tin)
    nup, nupp = dense_nu(mech)
    W = [mpf(float(w)) for w in mech.W]
    C, rho = ev["C"], ev["rho"]
    acc = [mpf(0)] * K
    for k in range(I):
        rx = ev["rx"][k]
        pf, pr = mpf(1), mpf(1)
        for i in range(K):
            pf *= power(C[i], nup[i][k])
            pr *= power(C[i], nupp[i][k])
        mag = abs(rx["kf"] * pf) + abs(rx["kr"] * pr)
        if int(mech.rtype[k]) == 1:
            mag *= abs(rx["M"])
        for i in range(K):
            acc[i] = acc[i] + (nup[i][k] + nupp[i][k]) * mag
    Yv = [mpf(float(y)) for y in Y]
    Yi = [mpf(float(y)) for y in Yin]
    tau = mpf(float(tau))
    S = [mpf(0)] + [abs(Yv[i] - Yi[i]) / tau + W[i] / rho * acc[i] for i in range(K)]
    if Tin is not None:
        Tm, Tinm = mpf(T), mpf(Tin)
        st = mpf(0)
        for i in range(K):
            a = [mpf(float(v)) for v in mech.nasa[i]]
            enth = lambda t: (a[0] + a[1] * t / 2 + a[2] * t**2 / 3 + a[3] * t**3 / 4 + a[4] * t**4 / 5 + a[5] / t) * RGAS * t / W[i]
            st += abs(Yi[i] * (enth(Tinm) - enth(Tm))) / tau + abs(enth(Tm)) * W[i] / rho * acc[i]
        S[0] = st / ev["cp_mix"]
    return S
