"""Pins of the CPU oracle against what the paper and the mathematics fix (P1-P10).
All CPU-only (-m "not gpu").  Nothing here calls the CUDA path."""
import math
import os

import numpy as np
import pytest

from workloads import make_workload, overlap_matrix, ncart

HERE = os.path.dirname(os.path.abspath(__file__))


def _basis(w):
    return (w.shell_atom, w.shell_L, w.shell_nprim, w.shell_prim_off, w.exps, w.coefs)


def _one_atom_one_s(alpha):
    norm = (2.0 * alpha / math.pi) ** 0.75
    xyz = np.array([[0.3, -0.2, 0.1]])
    basis = (np.array([0], np.int32), np.array([0], np.int32), np.array([1], np.int32), np.array([0], np.int32),
             np.array([alpha]), np.array([norm]))
    return xyz, basis


# ---- quadrature rules (O1, O2) ------------------------------------------------------------------
def test_table2_grid_sizes():
    # PAPER.md:L298-L304 Table 2: N_g^A = N_ang * N_rad
    assert 302 * 75 == 22650 and 590 * 99 == 58410 and 974 * 175 == 170450


@pytest.mark.parametrize("n_rad", [50, 75, 100])
def test_mk_radial_integrates_gaussians(orc, n_rad):
    # int_0^inf r^2 exp(-a r^2) dr = sqrt(pi)/(4 a^1.5)
    r, w = orc.radial_mk(n_rad, 5.0)
    for a in (0.4, 1.0, 6.0, 60.0):  # density exponents 2*alpha for alpha = 0.2 ... 30
        exact = math.sqrt(math.pi) / (4.0 * a ** 1.5)
        assert abs(np.sum(w * np.exp(-a * r * r)) / exact - 1.0) < 1e-13
    assert np.all(np.diff(r) > 0) and r[0] > 0


def test_mk_first_node_formula(orc):
    r, w = orc.radial_mk(3, 5.0)
    x = 0.25
    assert r[0] == pytest.approx(-5.0 * math.log(1 - x ** 3), rel=1e-15)
    assert w[0] == pytest.approx(r[0] ** 2 * 3 * 5.0 * x * x / (1 - x ** 3) / 4.0, rel=1e-15)


@pytest.mark.parametrize("kind,n", [(0, 194), (0, 302), (1, 288), (1, 1152)])
def test_angular_rules(orc, kind, n):
    u, w = orc.angular(kind, n)
    assert np.allclose(np.linalg.norm(u, axis=1), 1.0, atol=1e-15)
    assert np.sum(w) == pytest.approx(4 * math.pi, rel=1e-14)
    x, y, z = u.T
    if kind == 1:  # product rule is exact for low-order polynomials on the sphere
        assert np.sum(w * x * x) == pytest.approx(4 * math.pi / 3, rel=1e-13)
        assert np.sum(w * z ** 4) == pytest.approx(4 * math.pi / 5, rel=1e-13)
        assert np.sum(w * x * x * y * y) == pytest.approx(4 * math.pi / 15, rel=1e-13)
        assert abs(np.sum(w * x * y * z)) < 1e-14
        assert abs(np.sum(w * x ** 3)) < 1e-14
    else:  # Fibonacci: equal weights, z_k = 1 - (2k+1)/n, quasi-uniform
        assert np.allclose(w, 4 * math.pi / n)
        assert np.allclose(z, 1 - (2 * np.arange(n) + 1) / n, atol=1e-15)
        assert abs(np.sum(w * x * x) / (4 * math.pi / 3) - 1) < 2e-2


def test_grid_order_and_base_weights(orc):
    xyz = np.array([[0.0, 0.0, 0.0], [1.0, 2.0, 3.0]])
    pts, wq, par = orc.build_grid(xyz, 7, 10)
    r, wr = orc.radial_mk(7)
    u, wa = orc.angular(0, 10)
    assert np.all(par == np.repeat([0, 1], 70))
    k = 70 + 3 * 10 + 4  # atom 1, radial 3, angular 4
    assert np.allclose(pts[k], xyz[1] + r[3] * u[4], atol=1e-15)
    assert wq[k] == pytest.approx(wr[3] * wa[4], rel=1e-15)


# ---- partition (O4) ------------------------------------------------------------------------------
def test_partition_brute_force_and_unity(orc):
    w = make_workload("w8", with_P=False)
    rng = np.random.default_rng(5)
    xyz = w.atoms_xyz
    n = 400
    pts = xyz[rng.integers(0, len(xyz), n)] + rng.normal(size=(n, 3)) * rng.choice([0.05, 0.8, 4.0], size=(n, 1))
    wq = np.ones(n)
    for kind in (0, 1):
        tot = np.zeros(n)
        for A in range(len(xyz)):  # the same point replicated with every parent: weights sum to w^q
            tot += orc.partition_weights(xyz, pts, wq, np.full(n, A, np.int32), kind, prune=False)
        assert np.allclose(tot, 1.0, atol=1e-13)
    # SSF exact pruning == unpruned O(N_A^2) product
    par = rng.integers(0, len(xyz), n).astype(np.int32)
    a = orc.partition_weights(xyz, pts, wq, par, 0, prune=True)
    b = orc.partition_weights(xyz, pts, wq, par, 0, prune=False)
    assert np.max(np.abs(a - b)) < 1e-14
    # independent numpy restatement of Becke's scheme with the SSF cell function on a few points
    def ssf(mu, aa=0.64):
        z = np.clip(mu / aa, -1, 1)
        return 0.5 * (1 - (35 * z - 35 * z ** 3 + 21 * z ** 5 - 5 * z ** 7) / 16)
    for i in range(0, n, 37):
        rr = np.linalg.norm(pts[i] - xyz, axis=1)
        R = np.linalg.norm(xyz[:, None] - xyz[None], axis=-1)
        np.fill_diagonal(R, 1.0)
        s = ssf((rr[:, None] - rr[None, :]) / R)
        np.fill_diagonal(s, 1.0)
        PB = s.prod(axis=1)
        assert b[i] == pytest.approx(PB[par[i]] / PB.sum(), abs=1e-13)


def test_partition_near_nucleus_is_one_and_two_atom_midplane(orc):
    xyz = np.array([[0.0, 0.0, 0.0], [0.0, 0.0, 2.0]])
    pts = np.array([[0.0, 0.1, 0.05], [0.3, -0.2, 1.0], [0.0, 0.0, 1.9]])
    for kind in (0, 1):
        w0 = orc.partition_weights(xyz, pts, np.ones(3), np.zeros(3, np.int32), kind, True)
        assert w0[1] == pytest.approx(0.5, abs=1e-15)        # mid-plane: mu = 0, s = 1/2
    w0 = orc.partition_weights(xyz, pts, np.ones(3), np.zeros(3, np.int32), 0, True)
    assert w0[0] == 1.0 and w0[2] == 0.0                      # SSF compact support
    # Becke-88 midpoint polynomial value: mu = 0.25 -> p iterated three times
    pt = np.array([[0.0, 0.0, 1.25]])                         # r_A - r_B = 0.5, R = 2 -> mu_AB = 0.25
    p = 0.25
    for _ in range(3):
        p = 1.5 * p - 0.5 * p ** 3
    wb = orc.partition_weights(xyz, pt, np.ones(1), np.zeros(1, np.int32), 1, True)
    assert wb[0] == pytest.approx(0.5 * (1 - p), abs=1e-15)


# ---- screening (O5, Alg. 1) ------------------------------------------------------------------
def test_rcut_eq10(orc):
    ex = np.array([2.0, 0.5, 100.0])
    rc = orc.rcut(np.array([2, 1]), np.array([0, 2]), ex, 1e-10)
    f = lambda a: math.sqrt((0.5 * math.log(a) - math.log(1e-10)) / a)  # noqa: E731
    assert rc[0] == pytest.approx(max(f(2.0), f(0.5)), rel=1e-15)
    assert rc[1] == pytest.approx(f(100.0), rel=1e-15)
    # Eq. (10) is the radius at which sqrt(alpha) exp(-alpha r^2) = eta
    assert math.sqrt(2.0) * math.exp(-2.0 * f(2.0) ** 2) == pytest.approx(1e-10, rel=1e-9)


def test_alg1_cuboid_sphere_vs_brute_force(orc):
    rng = np.random.default_rng(11)
    for _ in range(300):
        V = rng.uniform(-2, 2, 3)
        W = V + rng.uniform(0.01, 3, 3)
        R = rng.uniform(-5, 5, 3)
        rc = rng.uniform(0.1, 4)
        closest = np.clip(R, V, W)
        expect = np.linalg.norm(closest - R) <= rc
        assert orc.cuboid_sphere(R, rc, V, W) == expect


# ---- collocation (O7), pin P8 ---------------------------------------------------------------
def test_collocation_gradient_vs_finite_difference(orc):
    w = make_workload("c1", with_P=False)
    rng = np.random.default_rng(3)
    pts = rng.normal(size=(40, 3)) * 1.5
    sh = np.arange(len(w.shell_L), dtype=np.int32)
    phi, gx, gy, gz = orc.collocation(sh, _basis(w), w.atoms_xyz, pts)
    h = 1e-5
    for c, g in enumerate((gx, gy, gz)):
        d = np.zeros(3)
        d[c] = h
        fd = (orc.collocation(sh, _basis(w), w.atoms_xyz, pts + d, grad=False)
              - orc.collocation(sh, _basis(w), w.atoms_xyz, pts - d, grad=False)) / (2 * h)
        scale = np.max(np.abs(g), axis=1, keepdims=True) + 1e-30
        assert np.max(np.abs(fd - g) / scale) < 1e-7


def test_collocation_explicit_values(orc):
    # Eq. (7) PAPER.md:L78 typed out for one d shell and one p shell at one point, order A5
    xyz = np.array([[0.5, -1.0, 0.25]])
    basis = (np.array([0, 0], np.int32), np.array([2, 1], np.int32), np.array([2, 1], np.int32),
             np.array([0, 2], np.int32), np.array([0.7, 0.2, 1.3]), np.array([0.4, 0.9, 1.1]))
    pt = np.array([[1.0, 0.5, -0.75]])
    phi = orc.collocation(np.array([0, 1], np.int32), basis, xyz, pt, grad=False)[:, 0]
    dx, dy, dz = (pt - xyz)[0]
    r2 = dx * dx + dy * dy + dz * dz
    Rd = 0.4 * math.exp(-0.7 * r2) + 0.9 * math.exp(-0.2 * r2)
    Rp = 1.1 * math.exp(-1.3 * r2)
    expect = [dx * dx * Rd, dx * dy * Rd, dx * dz * Rd, dy * dy * Rd, dy * dz * Rd, dz * dz * Rd, dx * Rp, dy * Rp, dz * Rp]
    assert np.allclose(phi, expect, rtol=1e-15)


def test_collocation_overlap_on_fine_atom_grid(orc):
    # int phi_mu phi_nu on a fine one-centre grid == closed-form S for same-centre pairs (O atom)
    w = make_workload("c1", with_P=False)
    S = overlap_matrix(w)
    xyz = w.atoms_xyz[:1]
    pts, wq, _ = orc.build_grid(xyz, 150, 1152, angular_kind=1)
    sh = np.where(w.shell_atom == 0)[0].astype(np.int32)
    phi = orc.collocation(sh, _basis(w), w.atoms_xyz, pts, grad=False)
    Sq = (phi * wq) @ phi.T
    assert np.max(np.abs(Sq - S[:15, :15])) < 1e-10


# ---- functionals (O9), pins P6 / P7 ------------------------------------------------------------
def _golden():
    rows = []
    with open(os.path.join(HERE, "golden", "functional_values.txt")) as fh:
        for line in fh:
            if line.startswith("#"):
                continue
            rows.append(line.split())
    return rows


def test_functional_values_vs_mpmath(orc):
    n = 0
    for row in _golden():
        kind = int(row[0])
        if kind > 1:
            continue
        rho, sig, f, vr, vs = (float(x) for x in row[1:6])
        of, ovr, ovs = orc.functional(kind, rho, sig)
        assert of[0] == pytest.approx(f, rel=1e-13)
        assert ovr[0] == pytest.approx(vr, rel=1e-13)
        assert ovs[0] == pytest.approx(vs, rel=1e-12, abs=1e-15)  # abs: x/c cancellation at sigma=0
        n += 1
    assert n >= 14


def test_survey_p6_values(orc):
    # SURVEY.md section 8(c) pin P6 (values computed with mpmath in the survey session)
    f, vr, _ = orc.functional(0, np.array([1e-3, 0.1, 1.0, 10.0]))
    assert np.allclose(f, [-9.8720671567184165e-5, -0.039620590148651224, -0.81015137868881307, -16.828163327030209], rtol=1e-13)
    assert np.allclose(vr, [-0.12819269645829555, -0.51789018006534478, -1.0646834050186822, -2.2222372449403902], rtol=1e-13)
    f, vr, vs = orc.functional(1, np.array([1.0]), np.array([100.0]))
    assert f[0] == pytest.approx(-0.99206728967694423, rel=1e-13)
    assert vr[0] == pytest.approx(-0.95959515944823391, rel=1e-13)
    assert vs[0] == pytest.approx(-1.3534784532723082e-3, rel=1e-13)


def test_functional_limits(orc):
    rho = np.array([1e-4, 0.01, 0.3, 2.0, 50.0])
    zero = np.zeros_like(rho)
    # PBE(sigma = 0) = Slater + PW92, v_sigma(sigma -> 0) = 0 (mu = beta pi^2/3 cancels)
    fp, vp, vs = orc.functional(1, rho, zero)
    fs, vsl, _ = orc.functional(2, rho)
    fw, vw, _ = orc.functional(4, rho)
    assert np.allclose(fp, fs + fw, rtol=1e-13)
    assert np.allclose(vp, vsl + vw, rtol=1e-13)
    assert np.max(np.abs(vs) * rho ** (4.0 / 3.0)) < 1e-12
    # LDA = Slater + VWN5
    f0, v0, _ = orc.functional(0, rho)
    f3, v3, _ = orc.functional(3, rho)
    assert np.allclose(f0, fs + f3, rtol=1e-14)
    # Slater closed form
    cx = 0.75 * (3 / math.pi) ** (1 / 3)
    assert np.allclose(fs, -cx * rho ** (4 / 3), rtol=1e-14)
    assert np.allclose(vsl, -(4 / 3) * cx * rho ** (1 / 3), rtol=1e-14)
    # F_x -> 1 + kappa as s -> inf
    fx, _, _ = orc.functional(5, np.array([1.0]), np.array([1e14]))
    assert fx[0] / (-cx) == pytest.approx(1.804, rel=1e-9)
    # eps_c(r_s): both fits match the mpmath values (1e-13) and each other within 3e-4 Ha (Ceperley-Alder data)
    for row in _golden():
        if int(row[0]) in (3, 4):
            r_s = float(row[1])
            rho1 = 3 / (4 * math.pi * r_s ** 3)
            f, _, _ = orc.functional(int(row[0]), np.array([rho1]))
            assert f[0] / rho1 == pytest.approx(float(row[2]), rel=1e-13)
    for r_s, ref in ((1, -0.0600), (2, -0.0448), (5, -0.0282), (10, -0.0186)):
        rho1 = 3 / (4 * math.pi * r_s ** 3)
        for k in (3, 4):
            f, _, _ = orc.functional(k, np.array([rho1]))
            assert abs(f[0] / rho1 - ref) < 3e-4
    # rho <= rho_tol contributes nothing (A12)
    f, vr, vs = orc.functional(1, np.array([1e-16, 0.0]), np.array([1e-3, 0.0]))
    assert np.all(f == 0) and np.all(vr == 0) and np.all(vs == 0)


def test_functional_derivatives_vs_finite_difference(orc):
    rng = np.random.default_rng(9)
    rho = np.exp(rng.uniform(np.log(1e-4), np.log(20), 50))
    sig = rho ** (8 / 3) * np.exp(rng.uniform(np.log(1e-3), np.log(30), 50))
    for kind in (0, 1):
        f, vr, vs = orc.functional(kind, rho, sig)
        h = 1e-5 * rho
        fd = (orc.functional(kind, rho + h, sig)[0] - orc.functional(kind, rho - h, sig)[0]) / (2 * h)
        assert np.allclose(fd, vr, rtol=2e-8)
        if kind == 1:
            hs = 1e-5 * sig
            fds = (orc.functional(kind, rho, sig + hs)[0] - orc.functional(kind, rho, sig - hs)[0]) / (2 * hs)
            assert np.all(np.abs(fds - vs) <= 2e-7 * np.abs(vs) + 1e-9 * np.abs(f) / sig)  # + FD cancellation noise


# ---- whole quadrature ---------------------------------------------------------------------------
def _setup(orc, name, n_rad=None, n_ang=None, angular_kind=0, partition=0, max_pts=512):
    w = make_workload(name)
    pts, wq, par = orc.build_grid(w.atoms_xyz, n_rad or w.n_rad, n_ang or w.n_ang, angular_kind)
    rc = orc.rcut(w.shell_nprim, w.shell_prim_off, w.exps)
    plan = orc.plan_paper(w.atoms_xyz, pts, wq, par, w.shell_atom, rc, max_pts)
    wts = orc.partition_weights(w.atoms_xyz, plan.pts, plan.wq, plan.parent, partition, True)
    return w, plan, wts, rc


@pytest.mark.parametrize("alpha", [0.5, 1.0, 3.0])
def test_p1_one_primitive_closed_form(orc, alpha):
    # E_x^Slater = -C_x (2 N^2)^(4/3) (3 pi/(8 alpha))^(3/2), N^2 = (2 alpha/pi)^(3/2); V_11 = (2/3) E_x; N_el = 2
    xyz, basis = _one_atom_one_s(alpha)
    P = np.array([[2.0]])
    cx = 0.75 * (3 / math.pi) ** (1 / 3)
    N2 = (2 * alpha / math.pi) ** 1.5
    Ex = -cx * (2 * N2) ** (4 / 3) * (3 * math.pi / (8 * alpha)) ** 1.5
    for n_rad in (50, 100):
        pts, wq, par = orc.build_grid(xyz, n_rad, 194)
        rc = orc.rcut(basis[2], basis[3], basis[4])
        plan = orc.plan_paper(xyz, pts, wq, par, basis[0], rc)
        wts = orc.partition_weights(xyz, plan.pts, plan.wq, plan.parent, 0, True)
        assert np.array_equal(wts, plan.wq)
        r = orc.evaluate(plan, wts, basis, xyz, P, kind=2)
        assert r.E_xc == pytest.approx(Ex, rel=1e-13)
        assert r.N_el == pytest.approx(2.0, rel=1e-13)
        assert r.V[0, 0] == pytest.approx(2.0 / 3.0 * Ex, rel=1e-13)


def test_p2_electron_count_vs_trace_PS(orc):
    w = make_workload("c1")
    S = overlap_matrix(w)
    n_exact = float(np.trace(w.P @ S))
    assert n_exact == pytest.approx(10.0, abs=1e-11)
    errs = {}
    for label, (nr, na, ak, part) in {"fib_stated": (50, 194, 0, 0), "fib_302": (75, 302, 0, 0),
                                      "fib_1202": (75, 1202, 0, 0), "fib_5810": (100, 5810, 0, 0),
                                      "prod_1152_ssf": (100, 1152, 1, 0), "prod_1152_becke": (100, 1152, 1, 1),
                                      "prod_512": (75, 512, 1, 0)}.items():
        _, plan, wts, _ = _setup(orc, "c1", nr, na, ak, part)
        r = orc.evaluate(plan, wts, _basis(w), w.atoms_xyz, w.P, kind=0, want_V=False)
        errs[label] = abs(r.N_el - n_exact) / n_exact
    # north_star pin restated (reading F1): 1e-6 on the product rule; <= 2e-4 at the stated
    # Fibonacci 50x194 / 75x302 grids; error shrinks under refinement
    # (observed: 3.2e-8 SSF / 3.4e-8 Becke-88 at 100x1152 product; 9.6e-7 at 75x512 product;
    #  Fibonacci 1.5e-4 at 50x194, 1.1e-5 at 75x302, 8.8e-6 at 75x1202, 6.2e-7 at 100x5810)
    assert errs["prod_1152_ssf"] < 1e-6 and errs["prod_1152_becke"] < 1e-6 and errs["prod_512"] < 3e-6
    assert errs["fib_stated"] < 2e-4 and errs["fib_302"] < 2e-4
    assert errs["fib_1202"] < 2e-5 and errs["fib_5810"] < 1e-6
    assert errs["fib_stated"] > errs["fib_302"] > errs["fib_1202"] > errs["fib_5810"]


@pytest.mark.parametrize("kind", [0, 1])
def test_p3_p4_symmetry_and_finite_difference(orc, kind):
    w, plan, wts, _ = _setup(orc, "c1")
    basis = _basis(w)
    r = orc.evaluate(plan, wts, basis, w.atoms_xyz, w.P, kind)
    vmax = np.max(np.abs(r.V))
    assert np.max(np.abs(r.V - r.V.T)) <= 1e-15 * vmax
    rng = np.random.default_rng(17)
    h = 1e-4
    pairs = [(int(a), int(b)) for a, b in rng.integers(0, w.n_basis, (20, 2))] + [(3, 3), (10, 10), (24, 24)]
    for (m, n) in pairs:
        D = np.zeros_like(w.P)
        if m == n:
            D[m, m] = 1.0
        else:
            D[m, n] = D[n, m] = 1.0
        ep = orc.evaluate(plan, wts, basis, w.atoms_xyz, w.P + h * D, kind, want_V=False).E_xc
        em = orc.evaluate(plan, wts, basis, w.atoms_xyz, w.P - h * D, kind, want_V=False).E_xc
        fd = (ep - em) / (2 * h)
        expect = r.V[m, m] if m == n else 2.0 * r.V[m, n]
        assert abs(fd - expect) < 1e-7 * vmax, (m, n, fd, expect)


@pytest.mark.parametrize("name,kind", [("c1", 0), ("c1", 1), ("w8", 1)])
def test_p5_screened_vs_unscreened(orc, name, kind):
    w, plan, wts, _ = _setup(orc, name)
    basis = _basis(w)
    a = orc.evaluate(plan, wts, basis, w.atoms_xyz, w.P, kind)
    b = orc.evaluate_unscreened(plan.pts, wts, basis, w.atoms_xyz, w.P, kind)
    vmax = np.max(np.abs(b.V))
    assert np.max(np.abs(a.V - b.V)) <= 1e-10 * vmax
    assert abs(a.E_xc - b.E_xc) <= 1e-11 * abs(b.E_xc)
    assert abs(a.N_el - b.N_el) <= 1e-11 * abs(b.N_el)


def test_mode_b_is_the_plain_definition(orc):
    # independent numpy restatement of the unscreened quadrature sum on a tiny grid (LDA, Slater only)
    w = make_workload("c1")
    pts, wq, par = orc.build_grid(w.atoms_xyz, 12, 26)
    wts = orc.partition_weights(w.atoms_xyz, pts, wq, par, 1, False)
    basis = _basis(w)
    sh = np.arange(len(w.shell_L), dtype=np.int32)
    phi = orc.collocation(sh, basis, w.atoms_xyz, pts, grad=False)
    rho = np.einsum("mi,mn,ni->i", phi, w.P, phi)
    cx = 0.75 * (3 / math.pi) ** (1 / 3)
    E = np.sum(wts * (-cx) * rho ** (4 / 3))
    V = np.einsum("i,mi,ni->mn", wts * (-(4 / 3) * cx * rho ** (1 / 3)), phi, phi)
    b = orc.evaluate_unscreened(pts, wts, basis, w.atoms_xyz, w.P, 2)
    assert b.E_xc == pytest.approx(E, rel=1e-13)
    assert b.N_el == pytest.approx(np.sum(wts * rho), rel=1e-13)
    assert np.max(np.abs(b.V - V)) < 1e-13 * np.max(np.abs(V))


def test_gga_mode_b_vs_numpy(orc):
    # PBE: the V formula of Mode B typed with einsum, using the oracle's own functional values
    w = make_workload("c1")
    pts, wq, par = orc.build_grid(w.atoms_xyz, 10, 26)
    wts = orc.partition_weights(w.atoms_xyz, pts, wq, par, 0, False)
    basis = _basis(w)
    sh = np.arange(len(w.shell_L), dtype=np.int32)
    phi, gx, gy, gz = orc.collocation(sh, basis, w.atoms_xyz, pts)
    X = w.P @ phi
    rho = np.sum(phi * X, 0)
    gr = 2 * np.stack([np.sum(g * X, 0) for g in (gx, gy, gz)])
    f, vr, vs = orc.functional(1, rho, np.sum(gr * gr, 0))
    Z = 0.5 * wts * vr * phi + 2 * wts * vs * (gr[0] * gx + gr[1] * gy + gr[2] * gz)
    V = Z @ phi.T + phi @ Z.T
    b = orc.evaluate_unscreened(pts, wts, basis, w.atoms_xyz, w.P, 1)
    assert b.E_xc == pytest.approx(np.sum(wts * f), rel=1e-13)
    assert np.max(np.abs(b.V - V)) < 1e-13 * np.max(np.abs(V))


def test_p9_plan_validity_and_validator_catches_errors(orc):
    w, plan, wts, rc = _setup(orc, "w8", max_pts=512)
    assert orc.validate_plan(plan, w.atoms_xyz, w.shell_atom, rc) == 0
    nq = np.diff(plan.batch_off)
    assert nq.min() >= 1 and nq.max() <= 512 and nq.sum() == len(plan.pts)
    assert np.array_equal(np.sort(plan.orig), np.arange(len(plan.pts)))
    import copy
    bad = copy.deepcopy(plan)
    bad.orig[5] = bad.orig[6]
    assert orc.validate_plan(bad, w.atoms_xyz, w.shell_atom, rc) == 1
    bad = copy.deepcopy(plan)
    j = int(np.argmax(np.diff(bad.shell_off)))
    s0, s1 = bad.shell_off[j], bad.shell_off[j + 1]
    bad.shells = np.concatenate([bad.shells[:s0 + 1], bad.shells[s0 + 2:]])  # drop a needed shell
    bad.shell_off = bad.shell_off.copy()
    bad.shell_off[j + 1:] -= 1
    assert orc.validate_plan(bad, w.atoms_xyz, w.shell_atom, rc) == 4
    assert orc.validate_plan(plan, w.atoms_xyz, w.shell_atom, rc, max_pts=100) == 2
    # outside r_cut a primitive is below eta times its norm-free prefactor (Eq. (10) derivation)
    for s in range(len(w.shell_L)):
        a = w.exps[w.shell_prim_off[s]:w.shell_prim_off[s] + w.shell_nprim[s]]
        assert np.all(np.sqrt(a) * np.exp(-a * rc[s] ** 2) <= 1e-10 * (1 + 1e-9))


def test_p10_translation_invariance(orc):
    w = make_workload("c1")
    basis = _basis(w)
    res = []
    for shift in (np.zeros(3), np.array([3.25, -1.5, 7.125])):
        xyz = w.atoms_xyz + shift
        pts, wq, par = orc.build_grid(xyz, w.n_rad, w.n_ang)
        rc = orc.rcut(w.shell_nprim, w.shell_prim_off, w.exps)
        plan = orc.plan_paper(xyz, pts, wq, par, w.shell_atom, rc)
        wts = orc.partition_weights(xyz, plan.pts, plan.wq, plan.parent, 0, True)
        res.append(orc.evaluate(plan, wts, basis, xyz, w.P, 1))
    assert res[0].E_xc == pytest.approx(res[1].E_xc, rel=1e-12)
    assert res[0].N_el == pytest.approx(res[1].N_el, rel=1e-12)
    assert np.max(np.abs(res[0].V - res[1].V)) < 1e-11 * np.max(np.abs(res[0].V))


def test_subset_and_batch_partials(orc):
    w, plan, wts, _ = _setup(orc, "c1")
    basis = _basis(w)
    full = orc.evaluate(plan, wts, basis, w.atoms_xyz, w.P, 1, want_batch=True, want_rho=True)
    assert full.E_xc == pytest.approx(full.E_batch.sum(), rel=1e-13)
    assert full.N_el == pytest.approx(full.N_batch.sum(), rel=1e-13)
    sub = np.arange(0, plan.n_batches, 3)
    rest = np.setdiff1d(np.arange(plan.n_batches), sub)
    a = orc.evaluate(plan, wts, basis, w.atoms_xyz, w.P, 1, subset=sub)
    b = orc.evaluate(plan, wts, basis, w.atoms_xyz, w.P, 1, subset=rest)
    assert a.E_xc + b.E_xc == pytest.approx(full.E_xc, rel=1e-13)
    assert np.max(np.abs(a.V + b.V - full.V)) < 1e-13 * np.max(np.abs(full.V))
    assert full.N_el == pytest.approx(np.sum(wts * full.rho), rel=1e-13)


def test_workload_generator_shapes():
    w = make_workload("c1")
    assert w.n_basis == 25 and len(w.atoms_Z) == 3 and sum(ncart(int(L)) for L in w.shell_L) == 25
    w2 = make_workload("c2", with_P=False)
    assert w2.n_basis == 1600 and len(w2.atoms_Z) == 192
    a, b = make_workload("c1"), make_workload("c1", cache=False)
    assert np.array_equal(a.P, b.P) and np.allclose(a.P, a.P.T)


def test_next_workload_shapes():
    """SURVEY 8(f) item 2 workloads: u2 = the c2 cluster on a 99 x 590 grid (Table 2: 99 * 590 = 58410 per atom);
    g1 = irregular 410-water cluster (1230 atoms, 10250 functions), seeded and reproducible, O-O distances >= 2.6 A."""
    u2, c2 = make_workload("u2", with_P=False), make_workload("c2", with_P=False)
    assert np.array_equal(u2.atoms_xyz, c2.atoms_xyz) and np.array_equal(u2.exps, c2.exps)
    assert (u2.n_rad, u2.n_ang) == (99, 590) and u2.n_rad * u2.n_ang == 58410 and u2.functional == 1
    g1, g1b = make_workload("g1", with_P=False), make_workload("g1", with_P=False)
    assert np.array_equal(g1.atoms_xyz, g1b.atoms_xyz)
    assert len(g1.atoms_Z) == 1230 and g1.n_basis == 10250 and list(g1.atoms_Z[:3]) == [8, 1, 1]
    O = g1.atoms_xyz[::3]
    d2 = np.sum((O[:, None, :] - O[None, :, :]) ** 2, axis=2) + 1e9 * np.eye(len(O))
    assert np.sqrt(d2.min()) >= 2.6 * 1.8897261246257702 - 1e-9
    # O-H bond lengths are the monomer's
    assert np.allclose(np.linalg.norm(g1.atoms_xyz[1::3] - O, axis=1), np.linalg.norm(c2.atoms_xyz[1] - c2.atoms_xyz[0]))
    ext = O.max(0) - O.min(0)
    assert ext[0] > 1.8 * ext[2]          # elongated: not a cube


# ---- pure (real solid harmonic) d shells, SURVEY 8(f) item 4 (reading A19) -----------
def _one_atom_pure_d(alpha=0.9):
    # one centre: s, p and a pure d shell, one primitive each; the d radial part has unit norm on xx (A6)
    from workloads import PURE
    xyz = np.array([[0.2, -0.1, 0.3]])
    ns = (2 * alpha / math.pi) ** 0.75
    npp = ns * (4 * alpha) ** 0.5
    nd = ns * (4 * alpha) / math.sqrt(3.0)
    basis = (np.array([0, 0, 0], np.int32), np.array([0, 1, 2 | PURE], np.int32), np.array([1, 1, 1], np.int32),
             np.array([0, 1, 2], np.int32), np.array([alpha, alpha, alpha]), np.array([ns, npp, nd]))
    return xyz, basis


def test_pure_d_explicit_values_and_gradient(orc):
    """The five pure d functions typed out from the real solid harmonics of degree 2 (m = -2..2), and their gradients
    against central finite differences."""
    xyz, basis = _one_atom_pure_d()
    pt = np.array([[1.0, 0.5, -0.75], [-0.4, 0.9, 0.2]])
    sh = np.array([2], np.int32)
    phi, gx, gy, gz = orc.collocation(sh, basis, xyz, pt)
    assert phi.shape == (5, 2)
    for i in range(2):
        x, y, z = pt[i] - xyz[0]
        R = basis[5][2] * math.exp(-basis[4][2] * (x * x + y * y + z * z))
        s3 = math.sqrt(3.0)
        expect = [s3 * x * y * R, s3 * y * z * R, (z * z - 0.5 * (x * x + y * y)) * R, s3 * x * z * R, 0.5 * s3 * (x * x - y * y) * R]
        assert np.allclose(phi[:, i], expect, rtol=1e-14, atol=1e-300)
    h = 1e-5
    for c, g in enumerate((gx, gy, gz)):
        d = np.zeros(3)
        d[c] = h
        fd = (orc.collocation(sh, basis, xyz, pt + d, grad=False) - orc.collocation(sh, basis, xyz, pt - d, grad=False)) / (2 * h)
        assert np.max(np.abs(fd - g)) < 1e-8 * np.max(np.abs(g))


def test_pure_d_orthonormal_and_orthogonal_to_s_and_p(orc):
    """int phi_mu phi_nu over a fine one-centre grid: the 1 + 3 + 5 functions are orthonormal.  (A Cartesian zz overlaps
    with s; the trace-free d(0) must not; wrong coefficients break the unit norms.)"""
    xyz, basis = _one_atom_pure_d()
    pts, wq, _ = orc.build_grid(xyz, 150, 1152, angular_kind=1)
    phi = orc.collocation(np.array([0, 1, 2], np.int32), basis, xyz, pts, grad=False)
    S = (phi * wq) @ phi.T
    assert S.shape == (9, 9)
    assert np.max(np.abs(S - np.eye(9))) < 1e-10


def test_pure_d_unsold_theorem(orc):
    """sum_m d_m(r)^2 depends on |r| only (Unsold): equal on random directions of one sphere; pins the relative
    normalisation of the five components."""
    xyz, basis = _one_atom_pure_d()
    rng = np.random.default_rng(5)
    u = rng.normal(size=(200, 3))
    u /= np.linalg.norm(u, axis=1, keepdims=True)
    for rad in (0.3, 1.7):
        phi = orc.collocation(np.array([2], np.int32), basis, xyz, xyz + rad * u, grad=False)
        tot = np.sum(phi * phi, axis=0)
        assert np.max(np.abs(tot - tot[0])) < 1e-14 * tot[0]
        # = (3/4) r^4 R(r)^2 ... checked against the closed form: sum_m d_m^2 = r^4 R^2 (x,y,z on the unit sphere)
        R = basis[5][2] * math.exp(-basis[4][2] * rad * rad)
        assert tot[0] == pytest.approx(rad ** 4 * R * R, rel=1e-13)


def test_pure_d_workload_trace_and_finite_difference(orc):
    """p1 (monomer, O d shell pure: 24 functions): closed-form S of the generator vs quadrature, tr(PS) = 10, N_el on
    the product grid, V symmetric and V = dE/dP by central differences (PBE)."""
    w = make_workload("p1")
    assert w.n_basis == 24
    S = overlap_matrix(w)
    assert float(np.trace(w.P @ S)) == pytest.approx(10.0, abs=1e-11)
    basis = _basis(w)
    ptsO, wqO, _ = orc.build_grid(w.atoms_xyz[:1], 150, 1152, angular_kind=1)
    shO = np.where(w.shell_atom == 0)[0].astype(np.int32)
    phi = orc.collocation(shO, basis, w.atoms_xyz, ptsO, grad=False)
    assert np.max(np.abs((phi * wqO) @ phi.T - S[:14, :14])) < 1e-10
    pts, wq, par = orc.build_grid(w.atoms_xyz, 100, 1152, 1)
    rc = orc.rcut(w.shell_nprim, w.shell_prim_off, w.exps)
    plan = orc.plan_paper(w.atoms_xyz, pts, wq, par, w.shell_atom, rc)
    wts = orc.partition_weights(w.atoms_xyz, plan.pts, plan.wq, plan.parent, 0, True)
    r = orc.evaluate(plan, wts, basis, w.atoms_xyz, w.P, 1)
    assert abs(r.N_el - 10.0) < 1e-5
    vmax = np.max(np.abs(r.V))
    assert np.max(np.abs(r.V - r.V.T)) <= 1e-15 * vmax
    b = orc.evaluate_unscreened(plan.pts, wts, basis, w.atoms_xyz, w.P, 1)
    assert np.max(np.abs(r.V - b.V)) <= 1e-10 * vmax and abs(r.E_xc - b.E_xc) <= 1e-11 * abs(b.E_xc)
    h = 1e-4
    for (m, n) in [(9, 9), (11, 13), (2, 10), (12, 20), (13, 13), (10, 23)]:   # 9..13 = the pure d functions of O
        D = np.zeros_like(w.P)
        D[m, n] = D[n, m] = 1.0
        ep = orc.evaluate(plan, wts, basis, w.atoms_xyz, w.P + h * D, 1, want_V=False).E_xc
        em = orc.evaluate(plan, wts, basis, w.atoms_xyz, w.P - h * D, 1, want_V=False).E_xc
        expect = r.V[m, m] if m == n else 2.0 * r.V[m, n]
        assert abs((ep - em) / (2 * h) - expect) < 1e-7 * vmax
