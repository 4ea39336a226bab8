"""Helpers of the GPU parity tests: run the CUDA library (through the C ABI binding) and the CPU oracle
(Mode A, fed with the library's exported plan -- DESIGN.md reading A9) on the same seeded inputs."""
import numpy as np

TOL_V = 1e-10      # max|V_gpu - V_orc| <= TOL_V * max|V_orc|     (BASELINE.json:north_star)
TOL_S = 1e-11      # relative error of E_xc and N_el              (BASELINE.json:north_star)


def basis_of(w):
    return (w.shell_atom, w.shell_L, w.shell_nprim, w.shell_prim_off, w.exps, w.coefs)


def oracle_plan(orc, ex):
    return orc.Plan(ex.pts, ex.wq, ex.parent, ex.orig, ex.batch_off, ex.shell_off, ex.shells)


def run_gpu(w, functional=None, P=None, want_points=True, **spec_kw):
    import torch
    import paper_2007_03143_b200 as xc
    fn = w.functional if functional is None else functional
    spec = xc.grid_spec(w.n_rad, w.n_ang, fn, **spec_kw)
    plan = xc.Plan.from_workload(w, spec=spec)
    Pd = torch.from_numpy(np.ascontiguousarray(w.P if P is None else P)).cuda()
    E, N, V = plan.eval(Pd, diag=want_points)
    torch.cuda.synchronize()
    diag = plan.diagnostics(want_points=want_points, want_rho=want_points)
    return plan, dict(E=E, N=N, V=V.cpu().numpy(), **diag)


def run_oracle(orc, w, ex, functional, partition=0, P=None, subset=None, want_V=True, weights=None):
    op = oracle_plan(orc, ex)
    wts = weights if weights is not None else orc.partition_weights(w.atoms_xyz, op.pts, op.wq, op.parent, partition, True)
    r = orc.evaluate(op, wts, basis_of(w), w.atoms_xyz, w.P if P is None else P, functional, subset=subset,
                     want_V=want_V, want_batch=True, want_rho=True)
    return op, wts, r


def report(g, r, wts=None):
    vmax = np.max(np.abs(r.V)) if r.V is not None else 1.0
    out = dict(dV=float(np.max(np.abs(g["V"] - r.V)) / vmax) if r.V is not None else None,
               dE=abs(g["E"] - r.E_xc) / abs(r.E_xc), dN=abs(g["N"] - r.N_el) / abs(r.N_el),
               asym=float(np.max(np.abs(g["V"] - g["V"].T))))
    if wts is not None and g.get("w") is not None:
        out["dw"] = float(np.max(np.abs(g["w"] - wts)) / np.max(np.abs(wts)))
    if g.get("rho") is not None and r.rho is not None:
        # the library does not evaluate rho at points whose weight is exactly 0 (they cannot contribute)
        m = (g["w"] != 0.0) if g.get("w") is not None else np.ones(len(r.rho), bool)
        out["drho"] = float(np.max(np.abs(g["rho"][m] - r.rho[m])) / np.max(np.abs(r.rho)))
    return out
