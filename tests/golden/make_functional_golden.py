"""Writes tests/golden/functional_values.txt: f = rho*eps, v_rho = df/drho, v_sigma = df/dsigma of
Slater+VWN5 (LDA) and PBE at fixed (rho, sigma), evaluated with mpmath at 40 digits and differentiated
numerically by mpmath (mp.diff) -- an evaluation independent of oracle/ (dual numbers, fp64) and of
the CUDA path (hand-derived derivatives, fp64).  Formulas: DESIGN.md "Functional definitions"
(the paper gives none).  The same numbers are listed in SURVEY.md section 8(c) pin P6.

Run:  python tests/golden/make_functional_golden.py
"""
import os

from mpmath import mp, mpf, atan, cbrt, diff, exp, log, pi, sqrt

mp.dps = 40


def rs(rho):
    return cbrt(3 / (4 * pi * rho))


CX = mpf(3) / 4 * cbrt(3 / pi)


def f_slater(rho):
    return -CX * rho ** (mpf(4) / 3)


def eps_vwn5(rho):
    A, x0, b, c = mpf("0.0310907"), mpf("-0.10498"), mpf("3.72744"), mpf("12.9352")
    Q = sqrt(4 * c - b * b)
    x = sqrt(rs(rho))
    X = lambda y: y * y + b * y + c  # noqa: E731
    return A * (log(x * x / X(x)) + 2 * b / Q * atan(Q / (2 * x + b))
                - b * x0 / X(x0) * (log((x - x0) ** 2 / X(x)) + 2 * (b + 2 * x0) / Q * atan(Q / (2 * x + b))))


def eps_pw92(rho):
    A, a1 = mpf("0.0310907"), mpf("0.21370")
    b1, b2, b3, b4 = mpf("7.5957"), mpf("3.5876"), mpf("1.6382"), mpf("0.49294")
    r = rs(rho)
    return -2 * A * (1 + a1 * r) * log(1 + 1 / (2 * A * (b1 * sqrt(r) + b2 * r + b3 * r ** 1.5 + b4 * r * r)))


def f_lda(rho, sigma=0):
    return f_slater(rho) + rho * eps_vwn5(rho)


def f_pbe(rho, sigma):
    kappa = mpf("0.804")
    beta = mpf("0.06672455060314922")
    gamma = (1 - log(2)) / pi ** 2
    mu = beta * pi ** 2 / 3
    s2 = sigma / (4 * (3 * pi ** 2) ** (mpf(2) / 3) * rho ** (mpf(8) / 3))
    F = 1 + kappa - kappa / (1 + mu * s2 / kappa)
    fx = -CX * rho ** (mpf(4) / 3) * F
    eu = eps_pw92(rho)
    kF = cbrt(3 * pi ** 2 * rho)
    ks2 = 4 * kF / pi
    t2 = sigma / (4 * ks2 * rho * rho)
    Ac = (beta / gamma) / (exp(-eu / gamma) - 1)
    H = gamma * log(1 + (beta / gamma) * t2 * (1 + Ac * t2) / (1 + Ac * t2 + Ac * Ac * t2 * t2))
    return fx + rho * (eu + H)


def main():
    out = ["# kind rho sigma f v_rho v_sigma   (kind 0 = Slater+VWN5, 1 = PBE); mpmath 40 digits, mp.diff",
           "# source: tests/golden/make_functional_golden.py; formulas DESIGN.md 'Functional definitions'"]
    lda_pts = ["1e-3", "0.1", "1", "10", "3.7e-6", "250"]
    for r in lda_pts:
        rho = mpf(r)
        f = f_lda(rho)
        vr = diff(lambda x: f_lda(x), rho)
        out.append("0 %s 0 %s %s 0" % (r, mp.nstr(f, 20), mp.nstr(vr, 20)))
    pbe_pts = [("0.1", "0.01"), ("1", "0.5"), ("1", "100"), ("10", "50"), ("1e-3", "1e-6"), ("0.3", "0"),
               ("2e-5", "3e-9"), ("40", "1e4")]
    for r, s in pbe_pts:
        rho, sig = mpf(r), mpf(s)
        f = f_pbe(rho, sig)
        vr = diff(lambda x: f_pbe(x, sig), rho)
        vs = diff(lambda x: f_pbe(rho, x), sig)
        out.append("1 %s %s %s %s %s" % (r, s, mp.nstr(f, 20), mp.nstr(vr, 20), mp.nstr(vs, 20)))
    # uniform-gas correlation energies per particle at r_s = 1,2,5,10 (pin P7 / SURVEY F4)
    out.append("# eps_c(r_s): kind 3 = VWN5, 4 = PW92 ; columns: kind r_s eps_c")
    for r in (1, 2, 5, 10):
        rho = 3 / (4 * pi * mpf(r) ** 3)
        out.append("3 %d %s" % (r, mp.nstr(eps_vwn5(rho), 20)))
        out.append("4 %d %s" % (r, mp.nstr(eps_pw92(rho), 20)))
    path = os.path.join(os.path.dirname(os.path.abspath(__file__)), "functional_values.txt")
    with open(path, "w") as fh:
        fh.write("\n".join(out) + "\n")
    print("\n".join(out))


if __name__ == "__main__":
    main()
