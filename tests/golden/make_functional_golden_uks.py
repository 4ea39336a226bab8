"""Writes tests/golden/functional_values_uks.txt: the spin-polarised Slater+VWN5 (LDA) and PBE energy densities
f(rho_a, rho_b, s_aa, s_ab, s_bb) per unit volume and their five partial derivatives at fixed points, evaluated with
mpmath at 40 digits and differentiated numerically by mpmath (mp.diff) -- independent of oracle/ (forward-mode duals,
fp64) and of the CUDA path.  Formulas: DESIGN.md "Functional definitions, spin-polarised" (reading A20); the paper gives
none and only names the extension.

Run:  python tests/golden/make_functional_golden_uks.py
"""
import os

from mpmath import mp, mpf, atan, cbrt, diff, exp, log, pi, sqrt

mp.dps = 40
CX = mpf(3) / 4 * cbrt(3 / pi)
FPP0 = mpf(4) / (9 * (cbrt(2) - 1))


def fz(z):
    return ((1 + z) ** (mpf(4) / 3) + (1 - z) ** (mpf(4) / 3) - 2) / (2 ** (mpf(4) / 3) - 2)


def vwn_G(x, A, x0, b, c):
    Q = sqrt(4 * c - b * b)
    X = lambda y: y * y + b * y + c  # noqa: E731
    return A * (log(x * x / X(x)) + 2 * b / Q * atan(Q / (2 * x + b))
                - b * x0 / X(x0) * (log((x - x0) ** 2 / X(x)) + 2 * (b + 2 * x0) / Q * atan(Q / (2 * x + b))))


def eps_vwn5(rho, z):
    x = sqrt(cbrt(3 / (4 * pi * rho)))
    eP = vwn_G(x, mpf("0.0310907"), mpf("-0.10498"), mpf("3.72744"), mpf("12.9352"))
    eF = vwn_G(x, mpf("0.01554535"), mpf("-0.32500"), mpf("7.06042"), mpf("18.0578"))
    ac = vwn_G(x, -1 / (6 * pi ** 2), mpf("-0.0047584"), mpf("1.13107"), mpf("13.0045"))
    return eP + ac * fz(z) / FPP0 * (1 - z ** 4) + (eF - eP) * fz(z) * z ** 4


def pw_G(r, A, a1, b1, b2, b3, b4):
    return -2 * A * (1 + a1 * r) * log(1 + 1 / (2 * A * (b1 * sqrt(r) + b2 * r + b3 * r ** 1.5 + b4 * r * r)))


def eps_pw92(rho, z):
    r = cbrt(3 / (4 * pi * rho))
    e0 = pw_G(r, mpf("0.0310907"), mpf("0.21370"), mpf("7.5957"), mpf("3.5876"), mpf("1.6382"), mpf("0.49294"))
    e1 = pw_G(r, mpf("0.01554535"), mpf("0.20548"), mpf("14.1189"), mpf("6.1977"), mpf("3.3662"), mpf("0.62517"))
    mac = pw_G(r, mpf("0.0168869"), mpf("0.11125"), mpf("10.357"), mpf("3.6231"), mpf("0.88026"), mpf("0.49671"))
    return e0 - mac * fz(z) / FPP0 * (1 - z ** 4) + (e1 - e0) * fz(z) * z ** 4


def f_lda(ra, rb, saa, sab, sbb):
    rho = ra + rb
    z = (ra - rb) / rho
    fx = -CX * ((2 * ra) ** (mpf(4) / 3) + (2 * rb) ** (mpf(4) / 3)) / 2
    return fx + rho * eps_vwn5(rho, z)


def fx_pbe_unpol(rho, sigma):
    kappa = mpf("0.804")
    mu = mpf("0.06672455060314922") * pi ** 2 / 3
    s2 = sigma / (4 * (3 * pi ** 2) ** (mpf(2) / 3) * rho ** (mpf(8) / 3))
    return -CX * rho ** (mpf(4) / 3) * (1 + kappa - kappa / (1 + mu * s2 / kappa))


def f_pbe(ra, rb, saa, sab, sbb):
    beta = mpf("0.06672455060314922")
    gamma = (1 - log(2)) / pi ** 2
    rho = ra + rb
    z = (ra - rb) / rho
    sigma = saa + 2 * sab + sbb
    fx = (fx_pbe_unpol(2 * ra, 4 * saa) + fx_pbe_unpol(2 * rb, 4 * sbb)) / 2
    eu = eps_pw92(rho, z)
    phi = ((1 + z) ** (mpf(2) / 3) + (1 - z) ** (mpf(2) / 3)) / 2
    kF = cbrt(3 * pi ** 2 * rho)
    t2 = sigma / (4 * phi ** 2 * (4 * kF / pi) * rho * rho)
    Ac = (beta / gamma) / (exp(-eu / (gamma * phi ** 3)) - 1)
    H = gamma * phi ** 3 * log(1 + (beta / gamma) * t2 * (1 + Ac * t2) / (1 + Ac * t2 + Ac * Ac * t2 * t2))
    return fx + rho * (eu + H)


def main():
    out = ["# kind rho_a rho_b s_aa s_ab s_bb f df/drho_a df/drho_b df/ds_aa df/ds_ab df/ds_bb  (kind 0 = Slater+VWN5, 1 = PBE)",
           "# mpmath 40 digits, mp.diff; source: tests/golden/make_functional_golden_uks.py"]
    pts = [("0.6", "0.4", "0.2", "0.1", "0.15"), ("0.08", "0.02", "0.004", "-0.001", "0.0007"), ("3", "1", "20", "5", "4"),
           ("1e-3", "4e-4", "1e-6", "2e-7", "3e-7"), ("0.5", "0.5", "0.125", "0.125", "0.125"), ("2", "1e-3", "1", "1e-3", "1e-5"),
           ("1e-5", "3e-5", "1e-9", "-2e-10", "4e-9")]
    for kind, fn in ((0, f_lda), (1, f_pbe)):
        for p in pts:
            x = [mpf(t) for t in p]
            if kind == 0:
                x[2:] = [mpf(0)] * 3
            f = fn(*x)
            d = []
            for k in range(5):
                if kind == 0 and k >= 2:
                    d.append(mpf(0))
                    continue
                order = tuple(1 if q == k else 0 for q in range(5))
                d.append(diff(fn, tuple(x), order))
            out.append("%d %s %s" % (kind, " ".join(p if kind == 1 else (p[0], p[1], "0", "0", "0")),
                                     " ".join(mp.nstr(v, 20) for v in [f] + d)))
    # ferromagnetic uniform gas: eps_c(r_s, zeta = 1), kind 3 = VWN5, 4 = PW92
    out.append("# eps_c(r_s, zeta = 1): kind r_s eps_c")
    for r in (1, 2, 5, 10):
        rho = 3 / (4 * pi * mpf(r) ** 3)
        out.append("3 %d %s" % (r, mp.nstr(eps_vwn5(rho, mpf(1)), 20)))
        out.append("4 %d %s" % (r, mp.nstr(eps_pw92(rho, mpf(1)), 20)))
    path = os.path.join(os.path.dirname(os.path.abspath(__file__)), "functional_values_uks.txt")
    with open(path, "w") as fh:
        fh.write("\n".join(out) + "\n")
    print("\n".join(out))


if __name__ == "__main__":
    main()
