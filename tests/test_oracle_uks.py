"""Pins of the oracle's spin-unrestricted path and of the meta-GGA intermediate tau (SURVEY 8(f) item 3,
PAPER.md:L49-L51; readings A20-A22).  CPU only."""
import math
import os

import numpy as np
import pytest

from workloads import make_workload, overlap_matrix, spin_density_matrices

HERE = os.path.dirname(os.path.abspath(__file__))


def _basis(w):
    return (w.shell_atom, w.shell_L, w.shell_nprim, w.shell_prim_off, w.exps, w.coefs)


def _golden():
    pts, eps = [], []
    with open(os.path.join(HERE, "golden", "functional_values_uks.txt")) as fh:
        for line in fh:
            if line.startswith("#"):
                continue
            t = line.split()
            if len(t) == 12:
                pts.append([float(x) for x in t])
            else:
                eps.append((int(t[0]), float(t[1]), float(t[2])))
    return np.array(pts), eps


def test_polarised_functionals_vs_mpmath_golden(orc):
    """Every value and partial derivative against the 40-digit mpmath evaluation (independent script in tests/golden)."""
    g, _ = _golden()
    for row in g:
        kind = int(row[0])
        f, v = orc.functional_pol(kind, [row[1]], [row[2]], [row[3]], [row[4]], [row[5]])
        assert f[0] == pytest.approx(row[6], rel=2e-13)
        nder = 5 if kind == 1 else 2
        for k in range(nder):
            assert v[0, k] == pytest.approx(row[7 + k], rel=5e-12, abs=1e-13 * abs(row[7])), (kind, row[1:6], k)
        if kind == 0:
            assert np.all(v[0, 2:] == 0.0)


def test_ferromagnetic_uniform_gas(orc):
    """eps_c(r_s, zeta = 1) of VWN5 and PW92 (mpmath golden; the Ceperley-Alder ferromagnetic values -0.0316, -0.0239,
    -0.0154, -0.0105 Ha at r_s = 1, 2, 5, 10 within 3e-4)."""
    _, eps = _golden()
    lit = {1: -0.0316, 2: -0.0239, 5: -0.0154, 10: -0.0105}
    for kind, rs, val in eps:
        rho = 3.0 / (4.0 * math.pi * rs ** 3)
        # rho_b = 1e-15 rho: zeta = 1 to rounding, still a regular point of the interpolation
        f, _ = orc.functional_pol(kind, [rho], [1e-15 * rho], rho_tol=1e-300)
        assert f[0] / rho == pytest.approx(val, rel=1e-9)
        assert abs(val - lit[int(rs)]) < 3e-4


@pytest.mark.parametrize("kind", [0, 1])
def test_zeta_zero_is_the_unpolarised_functional(orc, kind):
    """f_pol(rho/2, rho/2, s/4, s/4, s/4) = f(rho, s); d/d rho_a = d/d rho_b = v_rho; (v_aa + v_ab + v_bb)/4 = v_sigma;
    v_aa = v_bb by symmetry.  The unpolarised functional is itself pinned to mpmath (P6)."""
    rng = np.random.default_rng(3)
    rho = np.exp(rng.uniform(np.log(1e-6), np.log(50.0), 200))
    sig = rho ** (8.0 / 3.0) * np.exp(rng.uniform(np.log(1e-4), np.log(30.0), 200)) if kind == 1 else np.zeros(200)
    f0, vr, vs = orc.functional(kind, rho, sig)
    f, v = orc.functional_pol(kind, rho / 2, rho / 2, sig / 4, sig / 4, sig / 4)
    assert np.max(np.abs(f - f0) / np.abs(f0)) < 1e-13
    assert np.max(np.abs(v[:, 0] - vr) / np.abs(vr)) < 1e-12 and np.max(np.abs(v[:, 1] - vr) / np.abs(vr)) < 1e-12
    if kind == 1:
        # (the exchange parts of v_aa, v_bb and the cross term cancel to a few digits: the error scales with the terms)
        assert np.max(np.abs((v[:, 2] + v[:, 3] + v[:, 4]) / 4 - vs) / (np.abs(v[:, 2]) + np.abs(v[:, 3]) + np.abs(vs))) < 1e-12
        assert np.max(np.abs(v[:, 2] - v[:, 4]) / np.abs(v[:, 2])) < 1e-11


def test_exchange_spin_scaling(orc):
    """E_x[rho_a, rho_b] = (E_x[2 rho_a] + E_x[2 rho_b]) / 2 for Slater (kind 2) and PBE exchange (kind 5, sigma -> 4 s_ss),
    against the unpolarised kinds; no dependence on s_ab."""
    rng = np.random.default_rng(4)
    ra, rb = np.exp(rng.uniform(-8, 3, 100)), np.exp(rng.uniform(-8, 3, 100))
    saa, sbb = ra ** (8 / 3) * rng.uniform(0.01, 5, 100), rb ** (8 / 3) * rng.uniform(0.01, 5, 100)
    sab = rng.normal(size=100) * np.sqrt(saa * sbb)
    for kp, ku in ((2, 2), (5, 5)):
        f, v = orc.functional_pol(kp, ra, rb, saa, sab, sbb)
        fa, vra, vsa = orc.functional(ku, 2 * ra, 4 * saa)
        fb, vrb, vsb = orc.functional(ku, 2 * rb, 4 * sbb)
        assert np.max(np.abs(f - 0.5 * (fa + fb)) / np.abs(f)) < 1e-13
        assert np.max(np.abs(v[:, 0] - vra) / np.abs(vra)) < 1e-12 and np.max(np.abs(v[:, 1] - vrb) / np.abs(vrb)) < 1e-12
        assert np.all(v[:, 3] == 0.0)
        if kp == 5:
            assert np.max(np.abs(v[:, 2] - 2 * vsa) / np.abs(vsa)) < 1e-12


def _setup(orc, name, n_rad=None, n_ang=None, angular=0):
    w = make_workload(name)
    pts, wq, par = orc.build_grid(w.atoms_xyz, n_rad or w.n_rad, n_ang or w.n_ang, angular)
    rc = orc.rcut(w.shell_nprim, w.shell_prim_off, w.exps)
    plan = orc.plan_paper(w.atoms_xyz, pts, wq, par, w.shell_atom, rc)
    wts = orc.partition_weights(w.atoms_xyz, plan.pts, plan.wq, plan.parent, 0, True)
    return w, plan, wts


@pytest.mark.parametrize("kind", [0, 1])
def test_closed_shell_limit_equals_restricted(orc, kind):
    """P_a = P_b = P/2: E_xc, N_el and V_a = V_b = V of the restricted evaluation (itself pinned by P1-P5)."""
    w, plan, wts = _setup(orc, "c1")
    r = orc.evaluate(plan, wts, _basis(w), w.atoms_xyz, w.P, kind, want_rho=True)
    u = orc.evaluate_uks(plan, wts, _basis(w), w.atoms_xyz, 0.5 * w.P, 0.5 * w.P, kind, want_rho=True)
    vmax = np.max(np.abs(r.V))
    assert abs(u.E_xc - r.E_xc) <= 1e-12 * abs(r.E_xc)
    assert abs(u.N_a + u.N_b - r.N_el) <= 1e-12 * r.N_el and u.N_a == pytest.approx(u.N_b, rel=1e-14)
    assert np.max(np.abs(u.Va - r.V)) <= 1e-12 * vmax and np.max(np.abs(u.Vb - r.V)) <= 1e-12 * vmax
    assert np.max(np.abs(u.rho[0] + u.rho[1] - r.rho)) <= 1e-13 * np.max(r.rho)


@pytest.mark.parametrize("kind", [0, 1])
def test_open_shell_trace_symmetry_and_finite_difference(orc, kind):
    """Monomer with 6 alpha / 4 beta orbitals on the product grid: N_s = tr(P_s S) = n_s, V_s symmetric, and
    dE/dP^s_mu,nu = V^s_mu,nu by central differences for both spins (pins the cross term v_s_ab and the factors of A21)."""
    w, plan, wts = _setup(orc, "c1", 100, 1152, 1)
    Pa, Pb = spin_density_matrices(w, 6, 4)
    S = overlap_matrix(w)
    assert float(np.trace(Pa @ S)) == pytest.approx(6.0, abs=1e-11) and float(np.trace(Pb @ S)) == pytest.approx(4.0, abs=1e-11)
    basis = _basis(w)
    u = orc.evaluate_uks(plan, wts, basis, w.atoms_xyz, Pa, Pb, kind)
    assert abs(u.N_a - 6.0) < 1e-5 and abs(u.N_b - 4.0) < 1e-5
    vmax = max(np.max(np.abs(u.Va)), np.max(np.abs(u.Vb)))
    assert np.max(np.abs(u.Va - u.Va.T)) <= 1e-15 * vmax and np.max(np.abs(u.Vb - u.Vb.T)) <= 1e-15 * vmax
    assert np.max(np.abs(u.Va - u.Vb)) > 1e-3 * vmax          # genuinely spin-polarised
    h = 2e-5                                                  # truncation error h^2 f'''/6 well below 1e-7 vmax
    rng = np.random.default_rng(11)
    pairs = [(int(a), int(b)) for a, b in rng.integers(0, w.n_basis, (8, 2))] + [(3, 3), (14, 14)]
    for spin in (0, 1):
        for (m, n) in pairs:
            D = np.zeros_like(Pa)
            D[m, n] = D[n, m] = 1.0
            Pp = (Pa + h * D, Pb) if spin == 0 else (Pa, Pb + h * D)
            Pm = (Pa - h * D, Pb) if spin == 0 else (Pa, Pb - h * D)
            ep = orc.evaluate_uks(plan, wts, basis, w.atoms_xyz, Pp[0], Pp[1], kind, want_V=False).E_xc
            em = orc.evaluate_uks(plan, wts, basis, w.atoms_xyz, Pm[0], Pm[1], kind, want_V=False).E_xc
            V = u.Va if spin == 0 else u.Vb
            expect = V[m, m] if m == n else 2.0 * V[m, n]
            assert abs((ep - em) / (2 * h) - expect) < 1e-7 * vmax, (spin, m, n)


@pytest.mark.parametrize("L,factor", [(0, 1.5), (1, 2.5)])
def test_tau_integrates_to_the_kinetic_energy_of_a_gaussian(orc, L, factor):
    """tau = 1/2 sum grad Phi . grad X: for one normalised primitive with one electron, int tau = <phi|-1/2 lap|phi> =
    (2L + 3) alpha / 2 (closed form), on the Mura-Knowles x product grid."""
    alpha = 0.8
    xyz = np.array([[0.1, 0.2, -0.3]])
    norm = (2 * alpha / math.pi) ** 0.75 * (4 * alpha) ** (L / 2.0)
    basis = (np.array([0], np.int32), np.array([L], np.int32), np.array([1], np.int32), np.array([0], np.int32),
             np.array([alpha]), np.array([norm]))
    nf = 1 if L == 0 else 3
    Pa = np.zeros((nf, nf))
    Pa[nf - 1, nf - 1] = 1.0                                    # one electron in the last component (s, or p_z)
    pts, wq, par = orc.build_grid(xyz, 100, 1152, 1)
    plan = orc.plan_paper(xyz, pts, wq, par, basis[0], orc.rcut(basis[2], basis[3], basis[4]))
    u = orc.evaluate_uks(plan, plan.wq, basis, xyz, Pa, np.zeros_like(Pa), 0, want_V=False, want_rho=True, want_tau=True)
    assert float(np.sum(plan.wq * u.rho[0])) == pytest.approx(1.0, rel=1e-12)
    assert float(np.sum(plan.wq * u.tau[0])) == pytest.approx(factor * alpha, rel=1e-11)
    assert np.all(u.tau[1] == 0.0)


def test_tau_pointwise_definition(orc):
    """tau_s,i = 1/2 sum_mu,nu P^s_mu,nu grad phi_mu . grad phi_nu from the collocation gradients (einsum over all shells,
    no screening) on the monomer."""
    w, plan, wts = _setup(orc, "c1")
    Pa, Pb = spin_density_matrices(w, 6, 4)
    u = orc.evaluate_uks(plan, wts, _basis(w), w.atoms_xyz, Pa, Pb, 1, want_V=False, want_rho=True, want_tau=True)
    sel = np.random.default_rng(2).choice(len(plan.pts), 300, replace=False)
    sh = np.arange(len(w.shell_L), dtype=np.int32)
    phi, gx, gy, gz = orc.collocation(sh, _basis(w), w.atoms_xyz, plan.pts[sel])
    for s, P in enumerate((Pa, Pb)):
        tau = 0.5 * sum(np.einsum("mi,mn,ni->i", g, P, g) for g in (gx, gy, gz))
        assert np.max(np.abs(tau - u.tau[s][sel])) <= 1e-10 * np.max(np.abs(tau))
        assert np.all(u.tau[s] >= -1e-18)


# ---- restricted meta-GGA (reading A23: MS0 exchange + PBE correlation), PAPER.md:L51 -----------------------------------
def test_mgga_functional_vs_mpmath_golden(orc):
    rows = []
    with open(os.path.join(HERE, "golden", "functional_values_mgga.txt")) as fh:
        for line in fh:
            if not line.startswith("#"):
                rows.append([float(x) for x in line.split()])
    assert len(rows) == 16
    for row in rows:
        f, v = orc.functional_mgga(int(row[0]), [row[1]], [row[2]], [row[3]])
        assert f[0] == pytest.approx(row[4], rel=2e-13)
        for k in range(3):
            assert v[0, k] == pytest.approx(row[5 + k], rel=5e-11, abs=1e-13 * abs(row[5])), (row[:4], k)


def test_mgga_limits(orc):
    """alpha = 1, sigma = 0 (uniform gas): MS0 exchange = Slater exactly (kind 2, pinned); tau = tau_W (one orbital, alpha = 0):
    F_x = F_int(p; c), typed out; f(alpha) -> 0 like alpha^-... for large alpha: F_x -> F1(p) from above."""
    rho = np.exp(np.random.default_rng(1).uniform(-9, 3, 50))
    k23 = (3 * math.pi ** 2) ** (2.0 / 3.0)
    tau_u = 0.3 * k23 * rho ** (5.0 / 3.0)
    f, v = orc.functional_mgga(8, rho, np.zeros_like(rho), tau_u)
    f0, _, _ = orc.functional(2, rho)
    assert np.max(np.abs(f - f0) / np.abs(f0)) < 1e-14
    sig = rho ** (8.0 / 3.0) * 3.0
    f, _ = orc.functional_mgga(8, rho, sig, sig / (8 * rho))
    p = sig / (4 * k23 * rho ** (8.0 / 3.0))
    F0 = 1 + 0.29 - 0.29 / (1 + (10.0 / 81.0 * p + 0.28771) / 0.29)
    assert np.max(np.abs(f / (f0 * F0) - 1.0)) < 1e-13
    # correlation part of kind 7 = PBE correlation (kind 6, pinned)
    f7, v7 = orc.functional_mgga(7, rho, sig, 1.7 * tau_u)
    f8, v8 = orc.functional_mgga(8, rho, sig, 1.7 * tau_u)
    fc, vrc, vsc = orc.functional(6, rho, sig)
    assert np.max(np.abs(f7 - f8 - fc) / np.abs(fc)) < 1e-11
    assert np.max(np.abs(v7[:, 2] - v8[:, 2])) == 0.0 and np.max(np.abs(v7[:, 1] - v8[:, 1] - vsc) / np.abs(vsc)) < 1e-9


def test_mgga_tau_equals_weizsaecker_for_one_orbital(orc):
    """One doubly occupied orbital: tau = |grad rho|^2 / (8 rho) at every point (alpha = 0), from the oracle's own tau and
    grad rho on the monomer with P = 2 c c^T."""
    w, plan, wts = _setup(orc, "c1")
    S = overlap_matrix(w)
    c = np.random.default_rng(4).normal(size=w.n_basis)
    c /= math.sqrt(c @ S @ c)
    P = 2.0 * np.outer(c, c)
    r = orc.evaluate_mgga(plan, wts, _basis(w), w.atoms_xyz, P, 7, want_V=False, want_rho=True)
    m = r.rho > 1e-8
    sigma = np.sum(r.grad_rho ** 2, axis=1)
    assert np.max(np.abs(r.tau[m] - sigma[m] / (8 * r.rho[m])) / r.tau[m]) < 1e-7   # (cancellation in sum c phi near the orbital nodes)


def test_mgga_symmetry_and_finite_difference(orc):
    """dE/dP = V for the meta-GGA on the product grid: pins the factor 1/2 of the tau term and the three partials."""
    w, plan, wts = _setup(orc, "c1", 100, 1152, 1)
    basis = _basis(w)
    r = orc.evaluate_mgga(plan, wts, basis, w.atoms_xyz, w.P, 7, want_rho=True)
    assert abs(r.N_el - 10.0) < 1e-5
    vmax = np.max(np.abs(r.V))
    assert np.max(np.abs(r.V - r.V.T)) <= 1e-15 * vmax
    g = orc.evaluate(plan, wts, basis, w.atoms_xyz, w.P, 1)
    assert np.max(np.abs(r.V - g.V)) > 1e-3 * vmax and r.N_el == pytest.approx(g.N_el, rel=1e-14)   # not PBE, same density
    h = 2e-5
    rng = np.random.default_rng(12)
    pairs = [(int(a), int(b)) for a, b in rng.integers(0, w.n_basis, (10, 2))] + [(3, 3), (14, 14), (24, 24)]
    for (m, n) in pairs:
        D = np.zeros_like(w.P)
        D[m, n] = D[n, m] = 1.0
        ep = orc.evaluate_mgga(plan, wts, basis, w.atoms_xyz, w.P + h * D, 7, want_V=False).E_xc
        em = orc.evaluate_mgga(plan, wts, basis, w.atoms_xyz, w.P - h * D, 7, want_V=False).E_xc
        expect = r.V[m, m] if m == n else 2.0 * r.V[m, n]
        assert abs((ep - em) / (2 * h) - expect) < 1e-7 * vmax, (m, n)
