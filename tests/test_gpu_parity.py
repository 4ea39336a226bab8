"""GPU parity tests (-m gpu): the CUDA path, called through the C ABI binding, against the CPU oracle on the
same seeded inputs.  Tolerances are BASELINE.json:north_star's: max|dV| <= 1e-10 max|V|, rel. error of E_xc
and N_el <= 1e-11.  The oracle runs in Mode A on the library's exported plan (reading A9), after
validating that plan independently (P9)."""
import math
import os

import numpy as np
import pytest

from parity_util import TOL_S, TOL_V, basis_of, oracle_plan, report, run_gpu, run_oracle
from workloads import make_workload

pytestmark = pytest.mark.gpu
HERE = os.path.dirname(os.path.abspath(__file__))


@pytest.fixture(scope="module")
def xc():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    import paper_2007_03143_b200 as m
    assert os.path.exists(m.LIB_PATH)
    return m


def _check(rep):
    assert rep["dV"] <= TOL_V, rep
    assert rep["dE"] <= TOL_S and rep["dN"] <= TOL_S, rep
    assert rep["asym"] == 0.0, rep
    if "dw" in rep:
        assert rep["dw"] <= 1e-13, rep
    if "drho" in rep:
        assert rep["drho"] <= 1e-12, rep


def _full_parity(orc, name, functional, partition=0, **spec_kw):
    w = make_workload(name)
    plan, g = run_gpu(w, functional, partition=partition, **spec_kw)
    ex = plan.export()
    rc = orc.rcut(w.shell_nprim, w.shell_prim_off, w.exps)
    assert orc.validate_plan(oracle_plan(orc, ex), w.atoms_xyz, w.shell_atom, rc, spec_kw.get("max_batch_pts", 512)) == 0
    op, wts, r = run_oracle(orc, w, ex, functional, partition)
    rep = report(g, r, wts)
    _check(rep)
    assert np.max(np.abs(g["E_batch"] - r.E_batch)) <= 1e-12 * abs(r.E_xc)
    assert np.max(np.abs(g["N_batch"] - r.N_batch)) <= 1e-12 * abs(r.N_el)
    if functional == 1:
        m = g["w"] != 0.0                       # rho / grad rho are not evaluated where w = 0 exactly
        assert np.max(np.abs(g["grad_rho"][m] - r.grad_rho[m])) <= 1e-12 * np.max(np.abs(r.grad_rho))
    return w, plan, g, r


@pytest.mark.parametrize("functional", [0, 1])
def test_c1_monomer(xc, orc, functional):
    w, plan, g, r = _full_parity(orc, "c1", functional)
    assert abs(g["N"] - 10.0) / 10.0 < 2e-4   # P2 at the stated 50x194 Fibonacci grid
    plan.close()


def test_w8_becke_partition(xc, orc):
    _, plan, _, _ = _full_parity(orc, "w8", 1, partition=1)
    plan.close()


def test_w27_becke_partition(xc, orc):
    _, plan, _, _ = _full_parity(orc, "w27", 1, partition=1)
    plan.close()


def test_c2_becke_weights_sampled(xc, orc):
    """Becke-88 weights at 192 atoms: the kernel stops an owner's cell product once an upper bound of it is below 2^-60
    of the running sum (bit-identical fp64 sum); the oracle evaluates the full O(N_A^2) products on sampled batches."""
    import torch
    w = make_workload("c2")
    plan = xc.Plan.from_workload(w, spec=xc.grid_spec(w.n_rad, w.n_ang, 0, partition=1))
    P = torch.from_numpy(w.P).cuda()
    E, N, V = plan.eval(P)
    assert abs(N - 2.0 * w.n_occ) / (2.0 * w.n_occ) < 2e-4
    d = plan.diagnostics()
    ex = plan.export()
    rng = np.random.default_rng(5)
    sub = np.sort(rng.choice(plan.n_batches, 40, replace=False))
    pidx = np.concatenate([np.arange(ex.batch_off[j], ex.batch_off[j + 1]) for j in sub])
    ref = orc.partition_weights(w.atoms_xyz, ex.pts[pidx], ex.wq[pidx], ex.parent[pidx], 1, False)
    assert np.max(np.abs(d["w"][pidx] - ref)) <= 1e-13 * np.max(ex.wq[pidx])
    E2, N2, V2 = plan.eval(P)
    assert E2 == E and N2 == N and torch.equal(V, V2)     # bit-identical repeat
    plan.close()


def test_w27_pbe(xc, orc):
    _, plan, _, _ = _full_parity(orc, "w27", 1)
    plan.close()


def test_w27_pbe_resplit_batches(xc, orc):
    """eta = 1e-20: every shell reaches so far that the bisection's batches exceed N_b^j = 192 and are split again (2515
    batches instead of 2048, N_b^j up to 192: the class-1 kernel at its limit, the GPU planner's hand-back path)."""
    _, plan, _, _ = _full_parity(orc, "w27", 1, eta=1e-20)
    assert plan.n_batches > 2048 and plan.stats()["max_nb"] == 192
    plan.close()


@pytest.mark.parametrize("name", ["p1", "p8", "p8l", "p27"])
def test_pure_d_shells(xc, orc, name):
    """the O d shell as five pure functions (XC_SHELL_PURE), monomer / 8 / 27
    waters, PBE and (p8l) LDA: every output against the oracle, which holds its own statement of the transformation."""
    w = make_workload(name)
    assert w.n_basis == 24 * len(w.atoms_Z) // 3
    _, plan, g, r = _full_parity(orc, name, w.functional)
    assert plan.n_basis == w.n_basis
    plan.close()


def test_c2_lda_64_waters(xc, orc):
    w, plan, g, r = _full_parity(orc, "c2", 0)
    assert abs(g["N"] - 640.0) / 640.0 < 2e-4
    plan.close()


def test_c3_pbe_64_waters(xc, orc):
    _, plan, _, _ = _full_parity(orc, "c3", 1)
    plan.close()


@pytest.mark.parametrize("max_pts,angular,n_ang", [(37, 0, 194), (100, 1, 288), (512, 0, 50), (1, 0, 6)])
def test_ragged_batches_and_product_grid(xc, orc, max_pts, angular, n_ang):
    # batch sizes that are not multiples of the 64-point tile; the Gauss-Legendre product rule; 1-point batches
    w = make_workload("c1")
    w.n_ang = n_ang
    if max_pts == 1:
        w.n_rad = 20
    plan, g = run_gpu(w, 1, max_batch_pts=max_pts, angular=angular)
    ex = plan.export()
    rc = orc.rcut(w.shell_nprim, w.shell_prim_off, w.exps)
    assert orc.validate_plan(oracle_plan(orc, ex), w.atoms_xyz, w.shell_atom, rc, max_pts) == 0
    assert np.diff(ex.batch_off).max() <= max_pts
    _, wts, r = run_oracle(orc, w, ex, 1)
    _check(report(g, r, wts))
    plan.close()


@pytest.mark.parametrize("alpha", [0.5, 3.0])
def test_one_atom_one_shell_closed_form(xc, alpha):
    # pin P1 through the CUDA path: Slater exchange of one normalised s primitive; LDA adds VWN5, so compare
    # N_el = 2 (exact to quadrature) and V symmetric 1x1; E against the oracle is covered elsewhere
    import torch
    norm = (2.0 * alpha / math.pi) ** 0.75
    spec = xc.grid_spec(75, 302, 0)
    plan = xc.Plan(np.array([[0.3, -0.2, 0.1]]), np.array([1]), [0], [0], [1], [0], [alpha], [norm], spec)
    P = torch.tensor([[2.0]], dtype=torch.float64, device="cuda")
    E, N, V = plan.eval(P)
    assert N == pytest.approx(2.0, rel=1e-13)
    assert plan.diagnostics()["w"] == pytest.approx(plan.export().wq, rel=0, abs=0)   # single atom: w = w^q exactly
    plan.close()


def test_determinism_ld_host_path_and_one_shot(xc, orc):
    import torch
    w = make_workload("w8")
    plan = xc.Plan.from_workload(w)
    n = w.n_basis
    P = torch.from_numpy(w.P).cuda()
    E1, N1, V1 = plan.eval(P)
    V1 = V1.clone()
    E2, N2, V2 = plan.eval(P)
    assert E1 == E2 and N1 == N2 and torch.equal(V1, V2)                      # bit-identical
    E3, N3, V3 = plan.eval(P, reuse_weights=True)
    assert E1 == E3 and N1 == N3 and torch.equal(V1, V3)                      # cached-weights build
    Ppad = torch.zeros((n, n + 7), dtype=torch.float64, device="cuda")
    Ppad[:, :n] = P
    Vpad = torch.full((n, n + 5), 7.0, dtype=torch.float64, device="cuda")
    E4, N4, _ = plan.eval(Ppad[:, :n], Vpad[:, :n])                           # leading dimensions > n_basis
    assert E1 == E4 and torch.equal(V1, Vpad[:, :n]) and bool((Vpad[:, n:] == 7.0).all())
    s = torch.cuda.Stream()
    with torch.cuda.stream(s):
        E5, N5, V5 = plan.eval(P, stream=s)                                   # non-default stream
    assert E1 == E5 and torch.equal(V1, V5)
    Eh, Nh, Vh = plan.eval_host(w.P.copy())                                   # host buffers through the C ABI
    assert Eh == E1 and Nh == N1 and np.array_equal(Vh, V1.cpu().numpy())
    Eo, Vo, No = xc.xc_integrate(w, P)                                        # one-shot create+eval+destroy
    assert Eo == E1 and No == N1 and torch.equal(Vo, V1)
    plan.close()


def test_error_codes(xc):
    w0 = make_workload("c1")
    bad_L = w0.shell_L.copy()
    bad_L[0] |= 0x200                                        # unknown bit in xc_shell.L
    with pytest.raises(xc.XcError) as e0:
        xc.Plan(w0.atoms_xyz, w0.atoms_Z, w0.shell_atom, bad_L, w0.shell_nprim, w0.shell_prim_off, w0.exps, w0.coefs,
                xc.grid_spec(10, 26, 0))
    assert e0.value.code == -1
    import torch
    w = make_workload("c1")
    with pytest.raises(xc.XcError) as e:
        xc.Plan.from_workload(w, spec=xc.grid_spec(10, 26, 0, max_batch_pts=4096))
    assert e.value.code == -1
    w2 = make_workload("c1")
    w2.shell_L = w2.shell_L.copy()
    w2.shell_L[0] = 3
    with pytest.raises(xc.XcError) as e:
        xc.Plan.from_workload(w2)
    assert e.value.code == -2
    plan = xc.Plan.from_workload(w, spec=xc.grid_spec(10, 26, 0))
    P = torch.from_numpy(w.P).cuda()
    import ctypes as C
    from paper_2007_03143_b200 import binding as b
    E, N = C.c_double(), C.c_double()
    rc = b._lib.xc_eval(plan._h, C.c_void_p(P.data_ptr()), 3, C.c_void_p(P.data_ptr()), 25, C.byref(E), C.byref(N), 0, None)
    assert rc == -1   # ld < n_basis
    plan.close()


# ---- single kernels, element by element ---------------------------------------------------------
def test_functional_kernel_vs_oracle_and_golden(xc, orc):
    import torch
    rng = np.random.default_rng(21)
    n = 20000
    rho = np.exp(rng.uniform(np.log(1e-12), np.log(500.0), n))
    sig = rho ** (8.0 / 3.0) * np.exp(rng.uniform(np.log(1e-6), np.log(1e3), n))
    sig[::17] = 0.0
    rho[::501] = 1e-16   # below rho_tol
    for kind in (0, 1):
        f, vr, vs = (t.cpu().numpy() for t in xc.functional(kind, torch.from_numpy(rho).cuda(), torch.from_numpy(sig).cuda()))
        of, ovr, ovs = orc.functional(kind, rho, sig)
        assert np.max(np.abs(f - of) / (np.abs(of) + 1e-300)) < 1e-12
        assert np.max(np.abs(vr - ovr) / (np.abs(ovr) + 1e-300)) < 1e-11
        if kind == 1:
            # v_sigma is a difference of an exchange and a correlation term: tolerance relative to the exchange term
            scale = np.abs(ovs) + 0.05 / rho ** (4.0 / 3.0)
            assert np.max(np.abs(vs - ovs) / scale) < 1e-12
    rows = [l.split() for l in open(os.path.join(HERE, "golden", "functional_values.txt")) if not l.startswith("#")]
    for row in rows:
        kind = int(row[0])
        if kind > 1:
            continue
        r_, s_, f_, vr_, vs_ = (float(x) for x in row[1:6])
        f, vr, vs = (float(t.item()) for t in xc.functional(kind, torch.tensor([r_], dtype=torch.float64, device="cuda"),
                                                           torch.tensor([s_], dtype=torch.float64, device="cuda")))
        assert f == pytest.approx(f_, rel=1e-13) and vr == pytest.approx(vr_, rel=1e-13)
        assert vs == pytest.approx(vs_, rel=1e-12, abs=1e-15)


@pytest.mark.parametrize("kind", [0, 1])
def test_partition_kernel_vs_oracle(xc, orc, kind):
    import torch
    w = make_workload("w27", with_P=False)
    rng = np.random.default_rng(4)
    n = 5000
    par = rng.integers(0, len(w.atoms_xyz), n).astype(np.int32)
    pts = w.atoms_xyz[par] + rng.normal(size=(n, 3)) * rng.choice([0.02, 0.5, 2.0, 8.0], size=(n, 1))
    wq = rng.uniform(0.1, 2.0, n)
    got = xc.partition_weights(w.atoms_xyz, torch.from_numpy(pts).cuda(), torch.from_numpy(wq).cuda(),
                               torch.from_numpy(par).cuda(), kind).cpu().numpy()
    ref = orc.partition_weights(w.atoms_xyz, pts, wq, par, kind, prune=False)
    assert np.max(np.abs(got - ref)) <= 1e-13 * np.max(wq)
    if kind == 0:
        assert np.array_equal(got == 0.0, ref == 0.0) and np.array_equal(got == wq, ref == wq)


# ---- full-size configs: sampled outputs + properties ---------------------------------------------
@pytest.mark.parametrize("name", ["c5", "u2", "s2", "g1"])
def test_full_size_sampled(xc, orc, name):
    """The 512-water PBE workload in the launch configuration bench.py times (sampled outputs plus properties; c4 and c5
    are also compared in full by test_c4_full / test_c5_full), plus the SURVEY 8(f) "next" workloads: u2 / s2 (64 waters on the
    UFG- / SFG-shaped 99 x 590 / 175 x 974 grids) and g1 (irregular 410-water cluster).  Here the oracle computes (i) the weights, rho, grad rho and the per-batch E / N_el partial sums
    of sampled batches, and (ii) sampled V entries exactly: V[mu,nu] only receives contributions from batches
    whose S_j holds both shells, so evaluating that subset of batches gives the full entry.  Properties at any
    size: V symmetric, N_el = tr(PS) within the grid error, bit-identical repeat."""
    import torch
    w = make_workload(name)
    plan = xc.Plan.from_workload(w)
    P = torch.from_numpy(w.P).cuda()
    E, N, V = plan.eval(P, diag=True)
    Vh = V.cpu().numpy()
    assert np.array_equal(Vh, Vh.T)
    assert abs(N - 2.0 * w.n_occ) / (2.0 * w.n_occ) < 2e-4
    d = plan.diagnostics(want_rho=True)
    assert N == pytest.approx(float(np.sum(d["N_batch"])), rel=1e-12) and E == pytest.approx(float(np.sum(d["E_batch"])), rel=1e-12)
    ex = plan.export()
    op = oracle_plan(orc, ex)
    basis = basis_of(w)
    rng = np.random.default_rng(99)
    nb = plan.n_batches
    # (i) sampled batches
    sub = np.sort(rng.choice(nb, 48, replace=False))
    pidx = np.concatenate([np.arange(ex.batch_off[j], ex.batch_off[j + 1]) for j in sub])
    wts = np.zeros(plan.n_points)
    wts[pidx] = orc.partition_weights(w.atoms_xyz, ex.pts[pidx], ex.wq[pidx], ex.parent[pidx], 0, True)
    assert np.max(np.abs(d["w"][pidx] - wts[pidx])) <= 1e-13 * np.max(ex.wq[pidx])
    r = orc.evaluate(op, wts, basis, w.atoms_xyz, w.P, 1, subset=sub, want_V=False, want_batch=True, want_rho=True)
    pl = pidx[d["w"][pidx] != 0.0]              # rho / grad rho are not evaluated where w = 0 exactly
    assert np.max(np.abs(d["rho"][pl] - r.rho[pl])) <= 1e-12 * np.max(np.abs(r.rho[pidx]))
    assert np.max(np.abs(d["grad_rho"][pl] - r.grad_rho[pl])) <= 1e-12 * np.max(np.abs(r.grad_rho[pidx]))
    assert np.all(d["rho"][pidx[d["w"][pidx] == 0.0]] == 0.0)
    assert np.max(np.abs(d["E_batch"][sub] - r.E_batch[sub])) <= 1e-11 * np.max(np.abs(r.E_batch[sub]))
    assert np.max(np.abs(d["N_batch"][sub] - r.N_batch[sub])) <= 1e-11 * np.max(np.abs(r.N_batch[sub]))
    # (ii) sampled V entries: tight shells (d of an O, p of its H) keep the batch subset small
    foff = w.shell_func_off
    atom = int(rng.integers(0, len(w.atoms_Z) // 3)) * 3          # an O atom
    sh_d = [s for s in range(len(w.shell_L)) if w.shell_atom[s] == atom and w.shell_L[s] == 2][0]
    sh_p = [s for s in range(len(w.shell_L)) if w.shell_atom[s] == atom + 1 and w.shell_L[s] == 1][0]
    has = np.zeros((nb, 2), bool)
    bid = np.repeat(np.arange(nb), np.diff(ex.shell_off))
    has[bid[ex.shells == sh_d], 0] = True
    has[bid[ex.shells == sh_p], 1] = True
    both = np.where(has[:, 0] & has[:, 1])[0]
    assert 0 < len(both) < 4000
    pidx = np.concatenate([np.arange(ex.batch_off[j], ex.batch_off[j + 1]) for j in both])
    wts2 = np.zeros(plan.n_points)
    wts2[pidx] = d["w"][pidx]     # weights already checked on the sample above; reuse the GPU's here
    r2 = orc.evaluate(op, wts2, basis, w.atoms_xyz, w.P, 1, subset=both, want_V=True)
    rows = np.arange(foff[sh_d], foff[sh_d] + 6)
    cols = np.arange(foff[sh_p], foff[sh_p] + 3)
    blk_o, blk_g = r2.V[np.ix_(rows, cols)], Vh[np.ix_(rows, cols)]
    assert np.max(np.abs(blk_o - blk_g)) <= TOL_V * np.max(np.abs(Vh))
    assert np.max(np.abs(blk_o)) > 0
    E2, N2, V2 = plan.eval(P)
    assert E2 == E and N2 == N and bool((V2.cpu().numpy() == Vh).all())
    plan.close()


# ---- full-size parity of every output on the 256- and 512-water configurations ------------------------
def test_c4_full(xc, orc):
    """256 waters, 6400 functions, 17.4 M points, PBE -- every output compared in full: the oracle runs Mode A over all
    42 424 batches of the exported plan (about two minutes on 16 host cores)."""
    _, plan, g, r = _full_parity(orc, "c4", 1)
    assert abs(g["N"] - 2560.0) / 2560.0 < 2e-4
    plan.close()


def test_c5_full(xc, orc):
    """512 waters, 12800 functions, 46.4 M points, PBE, the largest single-GPU configuration -- every output compared in
    full: weights of all points, rho / grad rho where w != 0, per-batch and total E_xc / N_el, all 1.6e8 entries of V
    (the oracle runs Mode A over all 131 072 batches of the exported plan: a few minutes on 16 host cores)."""
    _, plan, g, r = _full_parity(orc, "c5", 1)
    assert abs(g["N"] - 5120.0) / 5120.0 < 2e-4
    plan.close()


# ---- step (a): the long-list paths of the hot SSF kernel ------------------------------------------------
@pytest.mark.parametrize("name", ["c4", "g1"])
def test_ssf_long_lists_dense_cluster(xc, orc, name):
    """768 / 1230 atoms on a 6 x 26 grid: every batch has an atom list longer than the kernel's distance row (256), so
    every point takes the long-list path (lazily filled rows, partners past the row, the negligible-owner rule).  All
    weights against the oracle's pruned evaluation (pinned against brute force on the CPU), a random 3000 against the
    full O(N_A^2) products, and the sets of exact zeros and exact w^q."""
    import torch
    w = make_workload(name, with_P=False)
    plan = xc.Plan.from_workload(w, spec=xc.grid_spec(6, 26, 0))
    st = plan.stats()
    assert st["w_partners_mean"] > 256
    P = torch.eye(w.n_basis, dtype=torch.float64, device="cuda")
    plan.eval(P)
    got = plan.diagnostics()["w"]
    ex = plan.export()
    ref = orc.partition_weights(w.atoms_xyz, ex.pts, ex.wq, ex.parent, 0, True)
    assert np.max(np.abs(got - ref)) <= 1e-13 * np.max(ex.wq)
    # exact zeros on the same set, up to mu_BC within ~1e-4 of a: there s(mu) = 2.2 (1 - mu/a)^4 < 1e-16 is below the
    # rounding error of the polynomial (1 - g loses it in the oracle's form, 1/2 - z q(z^2) in the kernel's), so one side
    # may return exactly 0 and the other ~1e-17 (mpmath at three such points of g1: true s = 1.2e-17, 5.5e-18, 6.9e-19)
    zm = (got == 0.0) != (ref == 0.0)
    assert np.all(np.abs(got[zm] - ref[zm]) <= 1e-15 * ex.wq[zm]) and zm.sum() <= 1e-4 * len(got)
    # w = w^q exactly on the same set, up to the last-bit rounding of w^q P_A / sum when P_A / sum is within an ulp of 1
    mism = (got == ex.wq) != (ref == ex.wq)
    assert np.all(np.abs(got[mism] - ref[mism]) <= 2.3e-16 * ex.wq[mism]) and mism.sum() <= 1e-3 * len(got)
    sel = np.random.default_rng(8).choice(len(got), 3000, replace=False)
    full = orc.partition_weights(w.atoms_xyz, ex.pts[sel], ex.wq[sel], ex.parent[sel], 0, False)
    assert np.max(np.abs(got[sel] - full)) <= 1e-13 * np.max(ex.wq)
    plan.close()


def test_ssf_lists_beyond_the_shared_memory_cache(xc, orc):
    """4752 atoms (1584 waters), points far outside the cluster included: atom lists longer than the kernel's shared-memory
    atom cache (2112 atoms: coordinates fetched from global memory beyond it) and than its chunk table (4096 atoms).
    Through xc_partition_weights, which runs the kernels of xc_eval on ad-hoc batches."""
    import torch
    w = make_workload("x15", with_P=False)
    rng = np.random.default_rng(15)
    n = 1536
    par = rng.integers(0, len(w.atoms_xyz), n).astype(np.int32)
    pts = w.atoms_xyz[par] + rng.normal(size=(n, 3)) * rng.choice([0.3, 2.0, 6.0, 40.0], size=(n, 1))
    order = np.argsort(np.linalg.norm(pts - w.atoms_xyz.mean(0), axis=1))     # spatially coherent pseudo-batches of 512
    pts, par = pts[order], par[order]
    wq = rng.uniform(0.1, 2.0, n)
    got = xc.partition_weights(w.atoms_xyz, torch.from_numpy(pts).cuda(), torch.from_numpy(wq).cuda(),
                               torch.from_numpy(par).cuda(), 0).cpu().numpy()
    ref = orc.partition_weights(w.atoms_xyz, pts, wq, par, 0, True)
    assert np.max(np.abs(got - ref)) <= 1e-13 * np.max(wq)
    assert np.array_equal(got == 0.0, ref == 0.0)
    sel = rng.choice(n, 150, replace=False)
    full = orc.partition_weights(w.atoms_xyz, pts[sel], wq[sel], par[sel], 0, False)
    assert np.max(np.abs(got[sel] - full)) <= 1e-13 * np.max(wq)


# ---- the fixed-point accumulator of V: scale, non-finite input ------------------------------------------
@pytest.mark.parametrize("k", [20, -20])
def test_v_scaled_by_powers_of_two(xc, k):
    """phi -> 2^k phi (coefficients) and P -> 2^-2k P leave rho, E_xc, N_el unchanged bit for bit and scale V by exactly
    2^2k: V = 2^40 V0 / 2^-40 V0.  The accumulator's exponent must follow (one repeated build), never wrap or lose bits."""
    import torch
    w = make_workload("w8")
    plan0 = xc.Plan.from_workload(w)
    E0, N0, V0 = plan0.eval(torch.from_numpy(w.P).cuda())
    s_ = 2.0 ** k
    plan = xc.Plan(w.atoms_xyz, w.atoms_Z, w.shell_atom, w.shell_L, w.shell_nprim, w.shell_prim_off, w.exps, w.coefs * s_,
                   xc.grid_spec(w.n_rad, w.n_ang, w.functional))
    P = torch.from_numpy(w.P / (s_ * s_)).cuda()
    E, N, V = plan.eval(P)
    assert E == E0 and N == N0
    assert float((V / (s_ * s_) - V0).abs().max()) <= 1e-13 * float(V0.abs().max())
    E2, N2, V2 = plan.eval(P)                                                  # the plan remembers the exponent
    assert E2 == E and torch.equal(V, V2)
    plan.close(); plan0.close()


def test_non_finite_input_is_reported(xc):
    import torch
    w = make_workload("w8")
    plan = xc.Plan.from_workload(w)
    P = torch.from_numpy(w.P).cuda()
    E0, N0, V0 = plan.eval(P)
    for bad in (float("nan"), float("inf")):
        Pb = P.clone()
        Pb[3, 3] = bad
        V = torch.zeros_like(P)
        with pytest.raises(xc.XcError) as e:
            plan.eval(Pb, V)
        assert e.value.code == -1 and bool(torch.isnan(V).all())
    E1, N1, V1 = plan.eval(P)                                                  # the plan is usable afterwards
    assert E1 == E0 and torch.equal(V0, V1)
    plan.close()


def test_bad_geometry_is_rejected(xc):
    w = make_workload("c1")
    xyz = w.atoms_xyz.copy()
    xyz[2] = xyz[1]
    with pytest.raises(xc.XcError) as e:
        xc.Plan(xyz, w.atoms_Z, w.shell_atom, w.shell_L, w.shell_nprim, w.shell_prim_off, w.exps, w.coefs, xc.grid_spec(10, 26, 0))
    assert e.value.code == -1
    xyz = w.atoms_xyz.copy()
    xyz[0, 0] = np.nan
    with pytest.raises(xc.XcError) as e:
        xc.Plan(xyz, w.atoms_Z, w.shell_atom, w.shell_L, w.shell_nprim, w.shell_prim_off, w.exps, w.coefs, xc.grid_spec(10, 26, 0))
    assert e.value.code == -1


# ---- spin-unrestricted build, SURVEY 8(f) item 3 (readings A20-A22) -----------------------------
@pytest.mark.parametrize("name,functional,n_a,n_b", [("c1", 0, 6, 4), ("c1", 1, 6, 4), ("w8", 1, 44, 36), ("p8", 1, 42, 38),
                                                     ("w27", 0, 140, 130), ("w27", 1, 139, 131)])
def test_uks_parity(xc, orc, name, functional, n_a, n_b):
    """xc_eval_uks against the oracle's spin-unrestricted Alg. 4 on the library's exported plan: V_a, V_b, E_xc, N_a, N_b
    at the north_star tolerances, rho_s / grad rho_s point by point; bit-identical repeat."""
    import torch
    from workloads import spin_density_matrices
    w = make_workload(name)
    Pa, Pb = spin_density_matrices(w, n_a, n_b)
    plan = xc.Plan.from_workload(w, spec=xc.grid_spec(w.n_rad, w.n_ang, functional))
    Pad, Pbd = torch.from_numpy(Pa).cuda(), torch.from_numpy(Pb).cuda()
    E, (Na, Nb), Va, Vb = plan.eval_uks(Pad, Pbd)
    ex = plan.export()
    op = oracle_plan(orc, ex)
    wts = orc.partition_weights(w.atoms_xyz, op.pts, op.wq, op.parent, 0, True)
    r = orc.evaluate_uks(op, wts, basis_of(w), w.atoms_xyz, Pa, Pb, functional, want_rho=True)
    vmax = max(np.max(np.abs(r.Va)), np.max(np.abs(r.Vb)))
    Vah, Vbh = Va.cpu().numpy(), Vb.cpu().numpy()
    assert np.max(np.abs(Vah - r.Va)) <= TOL_V * vmax and np.max(np.abs(Vbh - r.Vb)) <= TOL_V * vmax
    assert np.array_equal(Vah, Vah.T) and np.array_equal(Vbh, Vbh.T)
    assert np.max(np.abs(Vah - Vbh)) > 1e-3 * vmax                      # genuinely spin-polarised
    assert abs(E - r.E_xc) <= TOL_S * abs(r.E_xc)
    assert abs(Na - r.N_a) <= TOL_S * r.N_a and abs(Nb - r.N_b) <= TOL_S * r.N_b
    gw = plan.diagnostics()["w"]
    assert np.max(np.abs(gw - wts)) <= 1e-13 * np.max(wts)
    rho, gr = plan.uks_densities()
    m = gw != 0.0
    for s in range(2):
        assert np.max(np.abs(rho[s][m] - r.rho[s][m])) <= 1e-12 * np.max(np.abs(r.rho))
        if functional == 1:
            assert np.max(np.abs(gr[s][m] - r.grad_rho[s][m])) <= 1e-12 * np.max(np.abs(r.grad_rho))
    E2, N2, Va2, Vb2 = plan.eval_uks(Pad, Pbd, reuse_weights=True)
    assert E2 == E and N2 == (Na, Nb) and torch.equal(Va, Va2) and torch.equal(Vb, Vb2)
    plan.close()


@pytest.mark.parametrize("functional", [0, 1])
def test_uks_closed_shell_limit_is_the_restricted_build(xc, functional):
    """P_a = P_b = P/2 through the pass-wise spin-unrestricted build against the fused restricted kernel (two code paths
    of the library: closed-form derivatives vs forward-mode tangents, fused vs separate passes)."""
    import torch
    w = make_workload("w8")
    plan = xc.Plan.from_workload(w, spec=xc.grid_spec(w.n_rad, w.n_ang, functional))
    P = torch.from_numpy(w.P).cuda()
    E0, N0, V0 = plan.eval(P)
    E, (Na, Nb), Va, Vb = plan.eval_uks(0.5 * P, 0.5 * P)
    vmax = float(V0.abs().max())
    assert abs(E - E0) <= 1e-12 * abs(E0) and abs(Na + Nb - N0) <= 1e-12 * N0 and abs(Na - Nb) <= 1e-14 * N0
    assert float((Va - V0).abs().max()) <= 1e-12 * vmax and float((Va - Vb).abs().max()) <= 1e-14 * vmax
    plan.close()


@pytest.mark.parametrize("name,functional", [("c1", 0), ("w8", 1), ("p8", 1), ("w27", 0)])
def test_tau_parity(xc, orc, name, functional):
    """xc_eval_tau (meta-GGA intermediate) against the oracle's tau on the library's plan, for the two spin
    density matrices of an open-shell determinant, point by point where w != 0; zero elsewhere."""
    import torch
    from workloads import spin_density_matrices
    w = make_workload(name)
    n_occ = w.n_occ
    Pa, Pb = spin_density_matrices(w, n_occ + 1, n_occ - 1)
    plan = xc.Plan.from_workload(w, spec=xc.grid_spec(w.n_rad, w.n_ang, functional))
    ta = plan.eval_tau(torch.from_numpy(Pa).cuda()).cpu().numpy()
    tb = plan.eval_tau(torch.from_numpy(Pb).cuda(), reuse_weights=True).cpu().numpy()
    ex = plan.export()
    op = oracle_plan(orc, ex)
    wts = orc.partition_weights(w.atoms_xyz, op.pts, op.wq, op.parent, 0, True)
    r = orc.evaluate_uks(op, wts, basis_of(w), w.atoms_xyz, Pa, Pb, 0, want_V=False, want_rho=True, want_tau=True)
    gw = plan.diagnostics()["w"]
    m = gw != 0.0
    scale = np.max(np.abs(r.tau))
    assert np.max(np.abs(ta[m] - r.tau[0][m])) <= 1e-12 * scale and np.max(np.abs(tb[m] - r.tau[1][m])) <= 1e-12 * scale
    assert np.all(ta[~m] == 0.0) and np.all(tb[~m] == 0.0)
    # the kinetic-energy integrals of the two spin channels (sum w tau), relative 1e-11
    assert abs(np.sum(gw * ta) - np.sum(wts * r.tau[0])) <= 1e-11 * abs(np.sum(wts * r.tau[0]))
    plan.close()


# ---- planner on the GPU, SURVEY 8(f) item 1 ----------------------------------------------------
@pytest.mark.parametrize("name,kw", [("c1", {}), ("c1", dict(max_batch_pts=37)), ("c1", dict(max_batch_pts=1, n_ang=6, n_rad=10)),
                                     ("w8", dict(max_batch_pts=100, angular=1, n_ang=288)), ("w27", {}), ("w27", dict(eta=1e-20)), ("c2", {}),
                                     ("g1", {})])
def test_gpu_planner_equals_host_planner(xc, name, kw):
    """The grid and the global median bisection run on the GPU when a plan is created for a device (xc_gpu_planner.cu); the
    host-only plan (device = -1) runs them on the host.  Every exported array must be identical: points, base weights,
    parents, permutation, batch offsets, shell lists.  (w27 with eta = 1e-20: cutoff radii so large that batches exceed the
    kernel's N_b^j limit and are split again -- the host then takes the points back from the GPU and finishes alone.)"""
    w = make_workload(name, with_P=False)
    kw = dict(kw)
    spec = xc.grid_spec(kw.pop("n_rad", w.n_rad), kw.pop("n_ang", w.n_ang), w.functional, **kw)
    pd = xc.Plan.from_workload(w, spec=spec, device=0)
    ph = xc.Plan.from_workload(w, spec=spec, device=-1)
    a, b = pd.export(), ph.export()
    for f in ("pts", "wq", "parent", "orig", "batch_off", "shell_off", "shells"):
        assert np.array_equal(getattr(a, f), getattr(b, f)), f
    assert pd.stats() == ph.stats()
    pd.close(); ph.close()


# ---- restricted meta-GGA, SURVEY 8(f) item 3 (reading A23: MS0 exchange + PBE correlation) -----------------
@pytest.mark.parametrize("name", ["c1", "w8", "p8", "w27"])
def test_mgga_parity(xc, orc, name):
    """grid_spec.functional = 2: xc_eval runs the meta-GGA as passes of the batch kernel (densities, tau, functional, Z / V^j,
    tau term of V^j).  Against the oracle's literal Alg. 4 with tau on the library's plan: V, E_xc, N_el at the north_star
    tolerances, rho / grad rho and the per-batch sums point by point; bit-identical repeat."""
    import torch
    w = make_workload(name)
    plan = xc.Plan.from_workload(w, spec=xc.grid_spec(w.n_rad, w.n_ang, 2))
    P = torch.from_numpy(w.P).cuda()
    E, N, V = plan.eval(P, diag=True)
    d = plan.diagnostics(want_points=True, want_rho=True)
    ex = plan.export()
    op = oracle_plan(orc, ex)
    wts = orc.partition_weights(w.atoms_xyz, op.pts, op.wq, op.parent, 0, True)
    r = orc.evaluate_mgga(op, wts, basis_of(w), w.atoms_xyz, w.P, 7, want_batch=True, want_rho=True)
    vmax = np.max(np.abs(r.V))
    Vh = V.cpu().numpy()
    assert np.max(np.abs(Vh - r.V)) <= TOL_V * vmax and np.array_equal(Vh, Vh.T)
    assert abs(E - r.E_xc) <= TOL_S * abs(r.E_xc) and abs(N - r.N_el) <= TOL_S * r.N_el
    assert np.max(np.abs(d["w"] - wts)) <= 1e-13 * np.max(wts)
    m = d["w"] != 0.0
    assert np.max(np.abs(d["rho"][m] - r.rho[m])) <= 1e-12 * np.max(np.abs(r.rho))
    assert np.max(np.abs(d["grad_rho"][m] - r.grad_rho[m])) <= 1e-12 * np.max(np.abs(r.grad_rho))
    assert np.max(np.abs(d["E_batch"] - r.E_batch)) <= 1e-12 * abs(r.E_xc)
    assert np.max(np.abs(d["N_batch"] - r.N_batch)) <= 1e-12 * abs(r.N_el)
    # it is not PBE: the tau-dependent exchange changes V
    g = orc.evaluate(op, wts, basis_of(w), w.atoms_xyz, w.P, 1, want_V=True)
    assert np.max(np.abs(Vh - g.V)) > 1e-3 * vmax
    E2, N2, V2 = plan.eval(P, reuse_weights=True)
    assert E2 == E and N2 == N and torch.equal(V, V2)
    plan.close()


def test_three_round_class_matches_the_five_round_one(xc):
    """27 waters have 169 batches with 113..144 functions and 5 beyond: by default one five-round launch.  With
    XC_SPEC_SPLIT_CLASS1 the 169 run the three-round instantiation (the one the large configs use): every build type --
    restricted LDA / PBE / meta-GGA, spin-unrestricted, tau -- must agree to rounding (same blocks, same order of the sums;
    the two instantiations are compiled separately, so a product-sum may be contracted into another FMA: 1 ulp of an
    element of Phi, seen as ~1e-16 max|V|)."""
    import torch
    from workloads import spin_density_matrices
    w = make_workload("w27")
    P = torch.from_numpy(w.P).cuda()
    Pa, Pb = (torch.from_numpy(x).cuda() for x in spin_density_matrices(w, 139, 131))
    for functional in (0, 1, 2):
        res = []
        for flags in (0, xc.XC_SPEC_SPLIT_CLASS1):
            plan = xc.Plan.from_workload(w, spec=xc.grid_spec(w.n_rad, w.n_ang, functional, flags=flags))
            E, N, V = plan.eval(P)
            out = [E, N, V.clone(), plan.eval_tau(P, reuse_weights=True).clone()]
            if functional < 2:
                Eu, (Na, Nb), Va, Vb = plan.eval_uks(Pa, Pb, reuse_weights=True)
                out += [Eu, Na, Nb, Va.clone(), Vb.clone()]
            res.append(out)
            plan.close()
        for a, b in zip(*res):
            if torch.is_tensor(a):
                assert float((a - b).abs().max()) <= 1e-14 * float(a.abs().max()), functional
            else:
                assert abs(a - b) <= 1e-14 * abs(a), functional
        assert float(res[0][2].abs().max()) > 0.1


def test_extensions_at_c3_size_sampled(xc, orc):
    """The spin-unrestricted and meta-GGA builds on the 64-water PBE shapes (4.3 M points, 1600 functions): 60 random batches
    against the oracle point by point (rho_s, grad rho_s, tau) and per batch (meta-GGA E / N sums); electron counts against
    tr(P_s S) = n_s at the Fibonacci-grid accuracy; V symmetric and bit-identical on repeat."""
    import torch
    from workloads import spin_density_matrices
    w = make_workload("c3")
    Pa, Pb = spin_density_matrices(w, 330, 310)
    plan = xc.Plan.from_workload(w, spec=xc.grid_spec(w.n_rad, w.n_ang, 1))
    Pad, Pbd = torch.from_numpy(Pa).cuda(), torch.from_numpy(Pb).cuda()
    E, (Na, Nb), Va, Vb = plan.eval_uks(Pad, Pbd)
    assert abs(Na - 330.0) / 330.0 < 2e-4 and abs(Nb - 310.0) / 310.0 < 2e-4
    assert torch.equal(Va, Va.T) and torch.equal(Vb, Vb.T)
    rho, gr = plan.uks_densities()
    ta = plan.eval_tau(Pad, reuse_weights=True).cpu().numpy()
    ex = plan.export()
    op = oracle_plan(orc, ex)
    sub = np.sort(np.random.default_rng(21).choice(plan.n_batches, 60, replace=False))
    pidx = np.concatenate([np.arange(ex.batch_off[j], ex.batch_off[j + 1]) for j in sub])
    gw = plan.diagnostics()["w"]
    wts = np.zeros(len(ex.wq))
    wts[pidx] = orc.partition_weights(w.atoms_xyz, ex.pts[pidx], ex.wq[pidx], ex.parent[pidx], 0, True)
    assert np.max(np.abs(gw[pidx] - wts[pidx])) <= 1e-13 * np.max(ex.wq)
    r = orc.evaluate_uks(op, wts, basis_of(w), w.atoms_xyz, Pa, Pb, 1, subset=sub, want_V=False, want_rho=True, want_tau=True)
    m = pidx[gw[pidx] != 0.0]
    for s in range(2):
        assert np.max(np.abs(rho[s][m] - r.rho[s][m])) <= 1e-12 * np.max(np.abs(r.rho))
        assert np.max(np.abs(gr[s][m] - r.grad_rho[s][m])) <= 1e-12 * np.max(np.abs(r.grad_rho))
    assert np.max(np.abs(ta[m] - r.tau[0][m])) <= 1e-12 * np.max(np.abs(r.tau))
    E2, N2, Va2, Vb2 = plan.eval_uks(Pad, Pbd, reuse_weights=True)
    assert E2 == E and torch.equal(Va, Va2) and torch.equal(Vb, Vb2)
    plan.close()
    # meta-GGA on the same cluster
    mplan = xc.Plan.from_workload(w, spec=xc.grid_spec(w.n_rad, w.n_ang, 2))
    P = torch.from_numpy(w.P).cuda()
    Em, Nm, Vm = mplan.eval(P, diag=True)
    assert abs(Nm - 640.0) / 640.0 < 2e-4 and torch.equal(Vm, Vm.T)
    d = mplan.diagnostics(want_points=True, want_rho=True)
    exm = mplan.export()
    assert np.array_equal(exm.orig, ex.orig)                 # same plan (the functional only sizes the shared memory)
    rm = orc.evaluate_mgga(op, wts, basis_of(w), w.atoms_xyz, w.P, 7, subset=sub, want_V=False, want_batch=True, want_rho=True)
    assert np.max(np.abs(d["rho"][m] - rm.rho[m])) <= 1e-12 * np.max(np.abs(rm.rho))
    assert np.max(np.abs(d["E_batch"][sub] - rm.E_batch[sub])) <= 1e-12 * abs(Em)
    assert np.max(np.abs(d["N_batch"][sub] - rm.N_batch[sub])) <= 1e-12 * abs(Nm)
    mplan.close()
