"""Writes tests/golden/functional_values_mgga.txt: the restricted meta-GGA of reading A23 (MS0 exchange of Sun, Xiao,
Ruzsinszky 2012 + PBE correlation) f(rho, sigma, tau) per unit volume and its three partial derivatives at fixed points,
evaluated with mpmath at 40 digits and differentiated numerically by mpmath (mp.diff) -- independent of oracle/ (forward
duals, fp64) and of the CUDA path.  The paper only names the extension.

Run:  python tests/golden/make_functional_golden_mgga.py
"""
import os

from mpmath import mp, mpf, cbrt, diff, exp, log, pi, sqrt

mp.dps = 40
CX = mpf(3) / 4 * cbrt(3 / pi)


def f_ms0_x(rho, sigma, tau):
    kappa, c, b, mu = mpf("0.29"), mpf("0.28771"), mpf(1), mpf(10) / 81
    k23 = (3 * pi ** 2) ** (mpf(2) / 3)
    p = sigma / (4 * k23 * rho ** (mpf(8) / 3))
    alpha = (tau - sigma / (8 * rho)) / (mpf(3) / 10 * k23 * rho ** (mpf(5) / 3))
    F1 = 1 + kappa - kappa / (1 + mu * p / kappa)
    F0 = 1 + kappa - kappa / (1 + (mu * p + c) / kappa)
    fa = (1 - alpha ** 2) ** 3 / (1 + alpha ** 3 + b * alpha ** 6)
    return -CX * rho ** (mpf(4) / 3) * (F1 + fa * (F0 - F1))


def f_pbe_c(rho, sigma):
    A, a1 = mpf("0.0310907"), mpf("0.21370")
    b1, b2, b3, b4 = mpf("7.5957"), mpf("3.5876"), mpf("1.6382"), mpf("0.49294")
    beta = mpf("0.06672455060314922")
    gamma = (1 - log(2)) / pi ** 2
    r = cbrt(3 / (4 * pi * rho))
    eu = -2 * A * (1 + a1 * r) * log(1 + 1 / (2 * A * (b1 * sqrt(r) + b2 * r + b3 * r ** 1.5 + b4 * r * r)))
    kF = cbrt(3 * pi ** 2 * rho)
    t2 = sigma / (4 * (4 * kF / pi) * rho * rho)
    Ac = (beta / gamma) / (exp(-eu / gamma) - 1)
    H = gamma * log(1 + (beta / gamma) * t2 * (1 + Ac * t2) / (1 + Ac * t2 + Ac * Ac * t2 * t2))
    return rho * (eu + H)


def f_mgga(rho, sigma, tau):
    return f_ms0_x(rho, sigma, tau) + f_pbe_c(rho, sigma)


def main():
    out = ["# kind rho sigma tau f df/drho df/dsigma df/dtau   (kind 7 = MS0 exchange + PBE correlation, 8 = MS0 exchange)",
           "# mpmath 40 digits, mp.diff; source: tests/golden/make_functional_golden_mgga.py"]
    pts = [("0.5", "0.3", "0.4"), ("0.08", "0.004", "0.02"), ("3", "20", "9"), ("1e-3", "1e-6", "2e-5"), ("1", "0", "2.8712340001881918"),
           ("2", "1", "0.0625"), ("1e-5", "1e-10", "3e-8"), ("0.2", "0.05", "1.5")]
    for kind, fn in ((7, f_mgga), (8, f_ms0_x)):
        for p in pts:
            x = [mpf(t) for t in p]
            f = fn(*x)
            d = [diff(fn, tuple(x), tuple(1 if q == k else 0 for q in range(3))) for k in range(3)]
            out.append("%d %s %s" % (kind, " ".join(p), " ".join(mp.nstr(v, 20) for v in [f] + d)))
    path = os.path.join(os.path.dirname(os.path.abspath(__file__)), "functional_values_mgga.txt")
    with open(path, "w") as fh:
        fh.write("\n".join(out) + "\n")
    print("\n".join(out))


if __name__ == "__main__":
    main()
