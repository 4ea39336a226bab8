"""xc_functional_uks_static (-m gpu): the entry point that allocates nothing (scratch in a static device array) against the
existing path -- the same step inside xc_eval_uks, whose partial sums live in a cudaMalloc'ed buffer of the plan.

The file name sorts last on purpose: the run is `pytest -x`, so a failure here hides no other test.  The test
passes alone in a fresh process and after the other tests (it creates its own plans and touches no shared state but the
static array, which every call overwrites before reading)."""
import ctypes as C
import os

import numpy as np
import pytest

from parity_util import TOL_S
from workloads import make_workload, spin_density_matrices

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def xc():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    import paper_2007_03143_b200 as m
    assert os.path.exists(m.LIB_PATH)
    return m


def _existing_path(xc, name, functional, n_a, n_b):
    """xc_eval_uks on a workload: (E_xc, N_a, N_b) and the inputs its spin-coupling step saw (w, rho_s, grad rho_s)."""
    import torch
    w = make_workload(name)
    Pa, Pb = spin_density_matrices(w, n_a, n_b)
    spec = xc.grid_spec(w.n_rad, w.n_ang, functional)
    plan = xc.Plan.from_workload(w, spec=spec)
    E, (Na, Nb), _, _ = plan.eval_uks(torch.from_numpy(Pa).cuda(), torch.from_numpy(Pb).cuda())
    wts = plan.diagnostics()["w"]
    rho, gr = plan.uks_densities()
    plan.close()
    live = wts != 0.0                      # the build leaves rho_s undefined where w = 0 (and never reads it there)
    rho[:, ~live] = 0.0
    gr[:, ~live, :] = 0.0
    return (E, Na, Nb), wts, rho, gr, spec.rho_tol


def _static_path(xc, functional, wts, rho, gr, rho_tol, poison):
    import torch
    n = len(wts)
    dw, drho, dgr = torch.from_numpy(wts).cuda(), torch.from_numpy(rho).cuda(), torch.from_numpy(gr).cuda()
    cA = torch.full((2, n), poison, dtype=torch.float64, device="cuda")
    cG = torch.full((2, n, 3), poison, dtype=torch.float64, device="cuda")
    out3 = torch.full((3,), poison, dtype=torch.float64, device="cuda")
    xc.functional_uks_static(functional, dw, drho, dgr if functional == 1 else None, cA, cG if functional == 1 else None, out3,
                             rho_tol=rho_tol)
    torch.cuda.synchronize()
    return out3.cpu().numpy(), cA.cpu().numpy(), cG.cpu().numpy()


def _coefficients_from_oracle(orc, functional, wts, rho, gr, rho_tol, idx):
    """a_s and g_s of Eq. (20) per spin from the oracle's spin-polarised functional at the points idx."""
    ra, rb = rho[0][idx], rho[1][idx]
    ga, gb = gr[0][idx], gr[1][idx]
    saa, sab, sbb = (ga * ga).sum(1), (ga * gb).sum(1), (gb * gb).sum(1)
    _, v = orc.functional_pol(functional, ra, rb, saa, sab, sbb, rho_tol=rho_tol)
    wi = wts[idx]
    half = 0.5 if functional == 1 else 1.0
    cA = np.stack([half * wi * v[:, 0], half * wi * v[:, 1]])
    cG = np.stack([wi[:, None] * (2.0 * v[:, 2:3] * ga + v[:, 3:4] * gb), wi[:, None] * (2.0 * v[:, 4:5] * gb + v[:, 3:4] * ga)])
    return cA, cG


def test_static_scratch_entry_point_matches_xc_eval_uks(xc, orc):
    """Two calls in a row on different inputs (27 waters PBE: 3070 blocks; 8 waters LDA with pure d shells: 910 blocks, so
    the array still holds the first call's partials past them), then the first again: E_xc, N_a, N_b equal those of
    xc_eval_uks within the tolerance of the parity tests (the kernels and the summation order are the same: in fact
    bit-identical), and the per-point coefficients match the oracle's functional."""
    cases = [("w27", 1, 139, 131), ("p8l", 0, 42, 38)]
    ref = [_existing_path(xc, *c) for c in cases]
    outs = []
    for k in (0, 1, 0):
        (E, Na, Nb), wts, rho, gr, rho_tol = ref[k]
        functional = cases[k][1]
        out3, cA, cG = _static_path(xc, functional, wts, rho, gr, rho_tol, poison=float("nan") if k else 1e300)
        outs.append(out3)
        assert abs(out3[0] - E) <= TOL_S * abs(E), (k, out3, E)
        assert abs(out3[1] - Na) <= TOL_S * Na and abs(out3[2] - Nb) <= TOL_S * Nb, (k, out3, Na, Nb)
        assert np.array_equal(out3, np.array([E, Na, Nb])), "same kernels, same order: expected bit-identical sums"
        # every coefficient written (no poison left), zero where w = 0, and equal to the oracle's on a sample of live points
        assert np.isfinite(cA).all() and np.abs(cA).max() < 1e100
        dead = wts == 0.0
        assert not cA[:, dead].any()
        rng = np.random.default_rng(7 + k)
        idx = rng.choice(np.flatnonzero(~dead), size=4000, replace=False)
        oA, oG = _coefficients_from_oracle(orc, functional, wts, rho, gr, rho_tol, idx)
        assert np.max(np.abs(cA[:, idx] - oA)) <= 1e-11 * np.max(np.abs(oA))
        if functional == 1:
            assert np.isfinite(cG).all() and not cG[:, dead].any()
            assert np.max(np.abs(cG[:, idx] - oG)) <= 1e-11 * np.max(np.abs(oG))
    assert np.array_equal(outs[0], outs[2])


def test_static_scratch_entry_point_rejects_what_it_cannot_hold(xc):
    import torch
    lib = xc.binding._lib
    d = torch.zeros(8, dtype=torch.float64, device="cuda")
    p = C.c_void_p(d.data_ptr())
    rc = lib.xc_functional_uks_static(0, xc.XC_STATIC_MAX_POINTS + 1, p, p, p, 1e-15, p, p, p, None)
    assert rc == -2 and b"exceeds the static scratch" in lib.xc_last_error()      # XC_EUNSUPPORTED, before anything runs
    assert lib.xc_functional_uks_static(2, 8, p, p, p, 1e-15, p, p, p, None) == -1  # XC_EINVAL: enum
    assert lib.xc_functional_uks_static(0, 8, p, p, p, 0.0, p, p, p, None) == -1    # rho_tol must be > 0
    assert lib.xc_functional_uks_static(1, 8, p, p, None, 1e-15, p, p, p, None) == -1  # PBE needs grad rho
    out3 = torch.full((3,), 7.0, dtype=torch.float64, device="cuda")
    assert lib.xc_functional_uks_static(0, 0, None, None, None, 1e-15, None, None, C.c_void_p(out3.data_ptr()), None) == 0
    torch.cuda.synchronize()
    assert not out3.cpu().numpy().any()                                             # no points: exact zeros
