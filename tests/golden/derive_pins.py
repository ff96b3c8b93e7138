"""Re-derives, in 40-digit arithmetic (mpmath), the worked examples SURVEY.md section 8(c)-iii prints,
and writes them as text fixtures next to this script.  It calls neither oracle/ nor the CUDA path: it is
a third, independent evaluation of the textbook formulas (Toro, ch. 10; Jiang & Shu 1996; Einfeldt 1988;
Shu & Osher 1988) used to pin the oracle.  Run:  python tests/golden/derive_pins.py
"""
import os

from mpmath import mp, mpf, sqrt

mp.dps = 40
HERE = os.path.dirname(os.path.abspath(__file__))


def weno5(a, b, c, d, e, eps):
    a, b, c, d, e, eps = map(mpf, (a, b, c, d, e, eps))
    p = [(2 * a - 7 * b + 11 * c) / 6, (-b + 5 * c + 2 * d) / 6, (2 * c + 5 * d - e) / 6]
    beta = [mpf(13) / 12 * (a - 2 * b + c) ** 2 + (a - 4 * b + 3 * c) ** 2 / 4,
            mpf(13) / 12 * (b - 2 * c + d) ** 2 + (b - d) ** 2 / 4,
            mpf(13) / 12 * (c - 2 * d + e) ** 2 + (3 * c - 4 * d + e) ** 2 / 4]
    g = [mpf(1) / 10, mpf(6) / 10, mpf(3) / 10]
    al = [g[k] / (eps + beta[k]) ** 2 for k in range(3)]
    return sum(al[k] * p[k] for k in range(3)) / sum(al)


def riemann(WL, WR, gamma, solver, speeds="einfeldt"):
    """1-D states (rho, u, p) -> flux (mass, momentum, energy)."""
    gamma = mpf(gamma)

    def side(W):
        r, u, p = W
        E = p / (gamma - 1) + r * u * u / 2
        return dict(r=r, u=u, p=p, c=sqrt(gamma * p / r), E=E, H=(E + p) / r,
                    U=[r, r * u, E], F=[r * u, r * u * u + p, u * (E + p)])

    L, R = side(WL), side(WR)
    if speeds == "einfeldt":
        sl, sr = sqrt(L["r"]), sqrt(R["r"])
        ut = (sl * L["u"] + sr * R["u"]) / (sl + sr)
        Ht = (sl * L["H"] + sr * R["H"]) / (sl + sr)
        ct = sqrt((gamma - 1) * (Ht - ut * ut / 2))
        SL, SR = min(L["u"] - L["c"], ut - ct), max(R["u"] + R["c"], ut + ct)
    else:
        SL = min(L["u"] - L["c"], R["u"] - R["c"])
        SR = max(L["u"] + L["c"], R["u"] + R["c"])
    if SL >= 0:
        return L["F"]
    if SR <= 0:
        return R["F"]
    if solver == "hlle":
        return [(SR * L["F"][v] - SL * R["F"][v] + SL * SR * (R["U"][v] - L["U"][v])) / (SR - SL) for v in range(3)]
    aL, aR = L["r"] * (SL - L["u"]), R["r"] * (SR - R["u"])
    Ss = (R["p"] - L["p"] + aL * L["u"] - aR * R["u"]) / (aL - aR)
    K, S, a = (L, SL, aL) if Ss >= 0 else (R, SR, aR)
    f = a / (S - Ss)
    Us = [f, f * Ss, f * (K["E"] / K["r"] + (Ss - K["u"]) * (Ss + K["p"] / a))]
    return [K["F"][v] + S * (Us[v] - K["U"][v]) for v in range(3)]


def minmod(a, b):
    if a > 0 and b > 0:
        return min(a, b)
    if a < 0 and b < 0:
        return max(a, b)
    return mpf(0)


def spatial(U, gamma, solver, lam):
    """lam * (F_{i+1/2} - F_{i-1/2}) for a 1-D line with 2 zero-gradient guard cells per side."""
    n = len(U)
    Ug = [U[0], U[0]] + U + [U[-1], U[-1]]
    W = []
    for r, m, E in Ug:
        u = m / r
        W.append((r, u, (mpf(gamma) - 1) * (E - m * u / 2)))
    sl = [[mpf(0)] * 3] + [[minmod(W[i][v] - W[i - 1][v], W[i + 1][v] - W[i][v]) for v in range(3)]
                           for i in range(1, n + 3)] + [[mpf(0)] * 3]
    F = []
    for f in range(n + 1):
        iL, iR = f + 1, f + 2
        WL = [W[iL][v] + sl[iL][v] / 2 for v in range(3)]
        WR = [W[iR][v] - sl[iR][v] / 2 for v in range(3)]
        F.append(riemann(WL, WR, gamma, solver))
    return [[lam * (F[i + 1][v] - F[i][v]) for v in range(3)] for i in range(n)]


def sod_step(solver):
    """One SSP-RK2 step of config 1 (N = 256, cfl 0.8); only a window around the jump is evolved
    (the state is uniform elsewhere, so zero-gradient ends are exact)."""
    gamma, N = mpf(14) / 10, 256
    dx = mpf(1) / N
    dt = mpf(8) / 10 * dx / sqrt(gamma)  # max (|u|+c) is c_L = sqrt(1.4)
    lo, hi = 112, 144
    U0 = []
    for i in range(lo, hi):
        r, p = (mpf(1), mpf(1)) if i < N // 2 else (mpf(1) / 8, mpf(1) / 10)
        U0.append([r, mpf(0), p / (gamma - 1)])
    lam = dt / dx
    S0 = spatial(U0, gamma, solver, lam)
    U1 = [[U0[i][v] - S0[i][v] for v in range(3)] for i in range(len(U0))]
    S1 = spatial(U1, gamma, solver, lam)
    U2 = [[U0[i][v] + ((U1[i][v] - U0[i][v]) - S1[i][v]) / 2 for v in range(3)] for i in range(len(U0))]
    return dt, lo, U0, U1, U2


def fmt(x):
    return mp.nstr(x, 20)


def main():
    with open(os.path.join(HERE, "weno5_pins.txt"), "w") as f:
        f.write("# WENO5-JS worked values, eps = 1e-6 (SURVEY.md 8(c)-iii row 'O3 WENO5'; Jiang & Shu 1996).\n")
        f.write("# a b c d e eps value\n")
        for args in [(1.0, 1.5, 1.2, 0.9, 1.4, 1e-6), (1.4, 0.9, 1.2, 1.5, 1.0, 1e-6), (0, 0, 0, 1, 1, 1e-6),
                     (1.0, 1.5, 1.2, 0.9, 1.4, 1e30)]:
            sa = [mpf(str(a)) for a in args]
            f.write(" ".join(str(a) for a in args) + " " + fmt(weno5(*sa)) + "\n")
    L, R = (mpf(1), mpf(0), mpf(1)), (mpf(1) / 8, mpf(0), mpf(1) / 10)
    with open(os.path.join(HERE, "sod_interface_flux.txt"), "w") as f:
        f.write("# Sod interface, gamma = 1.4, L = (1,0,1), R = (0.125,0,0.1): flux (mass, momentum, energy)\n")
        f.write("# (SURVEY.md 8(c)-iii row 'O4 worked example'; Toro ch. 10, Einfeldt 1988).  solver speeds F0 F1 F2\n")
        for solver in ("hlle", "hllc"):
            for speeds in ("einfeldt", "davis"):
                F = riemann(L, R, 1.4 if False else mpf(14) / 10, solver, speeds)
                f.write(f"{solver} {speeds} " + " ".join(fmt(x) for x in F) + "\n")
    with open(os.path.join(HERE, "sod_single_step.txt"), "w") as f:
        f.write("# Config 1 (N = 256, PLM-minmod, SSP-RK2, cfl 0.8), one step from t = 0: dt and (rho, m, E) of the\n")
        f.write("# zones the step changes (SURVEY.md 8(c)-iii row 'O5+O6+O7 1D hand-computed single step').\n")
        f.write("# rows: 'dt value' | 'solver stage zone rho m E'; stage 1 = U1, stage 2 = U^{n+1}\n")
        for solver in ("hlle", "hllc"):
            dt, lo, U0, U1, U2 = sod_step(solver)
            if solver == "hlle":
                f.write("dt " + fmt(dt) + "\n")
            for stage, U in ((1, U1), (2, U2)):
                for i in range(len(U)):
                    if any(U[i][v] != U0[i][v] for v in range(3)):
                        f.write(f"{solver} {stage} {lo + i} " + " ".join(fmt(x) for x in U[i]) + "\n")


if __name__ == "__main__":
    main()
