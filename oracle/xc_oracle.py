"""ctypes binding of oracle/xc_oracle.cpp (argument marshalling only; no arithmetic here)."""
from __future__ import annotations

import ctypes as C
import dataclasses

import numpy as np

from . import build as _build

_lib = None

_dp = C.POINTER(C.c_double)
_ip = C.POINTER(C.c_int32)
_lp = C.POINTER(C.c_int64)


def lib():
    global _lib
    if _lib is None:
        _lib = C.CDLL(_build.build())
        _lib.orc_plan_flops.restype = C.c_double
        _lib.orc_plan_paper.restype = C.c_int64
    return _lib


def _d(a):
    return None if a is None else a.ctypes.data_as(_dp)


def _i(a):
    return None if a is None else a.ctypes.data_as(_ip)


def _l(a):
    return None if a is None else a.ctypes.data_as(_lp)


def _f64(a):
    return np.ascontiguousarray(a, dtype=np.float64)


def _i32(a):
    return np.ascontiguousarray(a, dtype=np.int32)


def _i64(a):
    return np.ascontiguousarray(a, dtype=np.int64)


def num_threads() -> int:
    return int(lib().orc_num_threads())


def radial_mk(n_rad, alpha=5.0):
    r = np.empty(n_rad)
    w = np.empty(n_rad)
    lib().orc_radial_mk(C.c_int(n_rad), C.c_double(alpha), _d(r), _d(w))
    return r, w


def angular(kind, n_ang):
    u = np.empty((n_ang, 3))
    w = np.empty(n_ang)
    rc = lib().orc_angular(C.c_int(kind), C.c_int(n_ang), _d(u), _d(w))
    if rc:
        raise ValueError("bad angular rule (kind=%d, n_ang=%d)" % (kind, n_ang))
    return u, w


def build_grid(xyz, n_rad, n_ang, angular_kind=0, mk_alpha=5.0):
    xyz = _f64(xyz)
    na = xyz.shape[0]
    n = na * n_rad * n_ang
    pts = np.empty((n, 3))
    wq = np.empty(n)
    parent = np.empty(n, np.int32)
    rc = lib().orc_build_grid(C.c_int(na), _d(xyz), C.c_int(n_rad), C.c_int(n_ang), C.c_int(angular_kind),
                              C.c_double(mk_alpha), _d(pts), _d(wq), _i(parent))
    if rc:
        raise ValueError("bad grid spec")
    return pts, wq, parent


def partition_weights(xyz, pts, wq, parent, kind=0, prune=True):
    xyz, pts, wq, parent = _f64(xyz), _f64(pts), _f64(wq), _i32(parent)
    w = np.empty(len(wq))
    lib().orc_partition_weights(C.c_int(xyz.shape[0]), _d(xyz), C.c_int64(len(wq)), _d(pts), _d(wq), _i(parent),
                                C.c_int(kind), C.c_int(1 if prune else 0), _d(w))
    return w


def rcut(shell_nprim, shell_prim_off, exps, eta=1e-10):
    shell_nprim, shell_prim_off, exps = _i32(shell_nprim), _i32(shell_prim_off), _f64(exps)
    out = np.empty(len(shell_nprim))
    lib().orc_rcut(C.c_int(len(shell_nprim)), _i(shell_nprim), _i(shell_prim_off), _d(exps), C.c_double(eta), _d(out))
    return out


def cuboid_sphere(R, rc, V, W) -> bool:
    R, V, W = _f64(R), _f64(V), _f64(W)
    return bool(lib().orc_cuboid_sphere(_d(R), C.c_double(rc), _d(V), _d(W)))


@dataclasses.dataclass
class Plan:
    """A batch plan as DATA: points in batch-contiguous order + per-batch shell lists."""
    pts: np.ndarray         # (N_g,3) batch-contiguous
    wq: np.ndarray          # (N_g,) base quadrature weights, same order
    parent: np.ndarray      # (N_g,) int32
    orig: np.ndarray        # (N_g,) int64 index into the canonical (atom-major) grid
    batch_off: np.ndarray   # (N_batch+1,) int64
    shell_off: np.ndarray   # (N_batch+1,) int64
    shells: np.ndarray      # int32 shell ids, ascending inside a batch

    @property
    def n_batches(self):
        return len(self.batch_off) - 1


def plan_paper(xyz, pts, wq, parent, shell_atom, rcuts, max_pts=512) -> Plan:
    """The paper's literal per-atom 27-/8-split batching + Alg. 1 screening (oracle's own planner, O6)."""
    xyz, pts, parent, shell_atom, rcuts = _f64(xyz), _f64(pts), _i32(parent), _i32(shell_atom), _f64(rcuts)
    n = len(parent)
    perm = np.empty(n, np.int64)
    boff = np.empty(n + 1, np.int64)
    soff = np.empty(n + 1, np.int64)
    cap = 64 * 1024 * 1024
    while True:
        shells = np.empty(cap, np.int32)
        nb = lib().orc_plan_paper(C.c_int(xyz.shape[0]), _d(xyz), C.c_int64(n), _d(pts), _i(parent), C.c_int(max_pts),
                                  C.c_int(len(shell_atom)), _i(shell_atom), _d(rcuts), _l(perm), _l(boff), _l(soff),
                                  _i(shells), C.c_int64(cap))
        if nb >= 0:
            break
        cap *= 4
    boff = boff[:nb + 1].copy()
    soff = soff[:nb + 1].copy()
    return Plan(pts[perm], _f64(wq)[perm], parent[perm], perm, boff, soff, shells[:soff[-1]].copy())


def validate_plan(plan: Plan, xyz, shell_atom, rcuts, max_pts=512) -> int:
    xyz, shell_atom, rcuts = _f64(xyz), _i32(shell_atom), _f64(rcuts)
    pts = _f64(plan.pts)
    orig = _i64(plan.orig)
    boff, soff, sh = _i64(plan.batch_off), _i64(plan.shell_off), _i32(plan.shells)
    return int(lib().orc_validate_plan(C.c_int64(len(pts)), _d(pts), _l(orig), C.c_int64(len(boff) - 1), _l(boff),
                                       _l(soff), _i(sh), C.c_int(max_pts), C.c_int(xyz.shape[0]), _d(xyz),
                                       C.c_int(len(shell_atom)), _i(shell_atom), _d(rcuts)))


def collocation(sh_list, basis, xyz, pts, grad=True):
    """basis = (shell_atom, shell_L, shell_nprim, shell_prim_off, exps, coefs). Returns phi (nf,npts)[, gx, gy, gz]."""
    sa, sL, sn, so, ex, co = basis
    sa, sL, sn, so, ex, co = _i32(sa), _i32(sL), _i32(sn), _i32(so), _f64(ex), _f64(co)
    sh_list = _i32(sh_list)
    xyz, pts = _f64(xyz), _f64(pts)
    nf = int(sum(_nfun(int(sL[s])) for s in sh_list))
    n = len(pts)
    phi = np.empty((nf, n))
    g = [np.empty((nf, n)) for _ in range(3)] if grad else [None] * 3
    lib().orc_collocation(C.c_int(len(sh_list)), _i(sh_list), _i(sa), _i(sL), _i(sn), _i(so), _d(ex), _d(co), _d(xyz),
                          C.c_int64(n), _d(pts), _d(phi), _d(g[0]), _d(g[1]), _d(g[2]))
    return (phi, g[0], g[1], g[2]) if grad else phi


def functional(kind, rho, sigma=None, rho_tol=1e-15):
    rho = _f64(np.atleast_1d(rho))
    sigma = _f64(np.atleast_1d(sigma)) if sigma is not None else np.zeros_like(rho)
    f, vr, vs = np.empty_like(rho), np.empty_like(rho), np.empty_like(rho)
    lib().orc_functional(C.c_int(kind), C.c_int64(len(rho)), _d(rho), _d(sigma), C.c_double(rho_tol), _d(f), _d(vr), _d(vs))
    return f, vr, vs


def _nfun(code):
    """Functions of a shell code (low byte L; bit 8: pure d shell = 5 functions): sizes the output arrays."""
    L = code & 0xff
    return 5 if (code & 0x100) and L == 2 else (L + 1) * (L + 2) // 2


def _func_off(shell_L):
    nc = np.array([_nfun(int(c)) for c in np.asarray(shell_L)], dtype=np.int64)
    return np.concatenate([[0], np.cumsum(nc)[:-1]]).astype(np.int32), int(nc.sum())


@dataclasses.dataclass
class Result:
    E_xc: float
    N_el: float
    V: np.ndarray | None
    E_batch: np.ndarray | None = None
    N_batch: np.ndarray | None = None
    rho: np.ndarray | None = None
    grad_rho: np.ndarray | None = None


def evaluate(plan: Plan, w, basis, xyz, P, kind, rho_tol=1e-15, subset=None, want_V=True, want_batch=False,
             want_rho=False) -> Result:
    """Mode A (plan-conditioned) evaluation of Alg. 4 over `subset` of batches (None = all)."""
    sa, sL, sn, so, ex, co = basis
    sa, sL, sn, so, ex, co = _i32(sa), _i32(sL), _i32(sn), _i32(so), _f64(ex), _f64(co)
    foff, nbf = _func_off(sL)
    xyz, P, w = _f64(xyz), _f64(P), _f64(w)
    pts = _f64(plan.pts)
    boff, soff, sh = _i64(plan.batch_off), _i64(plan.shell_off), _i32(plan.shells)
    nbat = len(boff) - 1
    sub = _i64(subset) if subset is not None else None
    V = np.zeros((nbf, nbf)) if want_V else None
    Eb = np.zeros(nbat) if want_batch else None
    Nb = np.zeros(nbat) if want_batch else None
    rho = np.zeros(len(pts)) if want_rho else None
    gr = np.zeros((len(pts), 3)) if want_rho else None
    E = C.c_double(0.0)
    N = C.c_double(0.0)
    lib().orc_eval(C.c_int64(nbat), _l(boff), _l(soff), _i(sh), _l(sub), C.c_int64(0 if sub is None else len(sub)),
                   _d(pts), _d(w), _i(sa), _i(sL), _i(sn), _i(so), _i(foff), _d(ex), _d(co), _d(xyz), C.c_int(nbf),
                   _d(P), C.c_int64(P.shape[1]), C.c_int(kind), C.c_double(rho_tol), _d(V), C.byref(E), C.byref(N),
                   _d(Eb), _d(Nb), _d(rho), _d(gr))
    return Result(E.value, N.value, V, Eb, Nb, rho, gr)


def evaluate_unscreened(pts, w, basis, xyz, P, kind, rho_tol=1e-15, want_V=True) -> Result:
    """Mode B: the plain quadrature sum, every shell at every point."""
    sa, sL, sn, so, ex, co = basis
    sa, sL, sn, so, ex, co = _i32(sa), _i32(sL), _i32(sn), _i32(so), _f64(ex), _f64(co)
    _, nbf = _func_off(sL)
    xyz, P, w, pts = _f64(xyz), _f64(P), _f64(w), _f64(pts)
    V = np.zeros((nbf, nbf)) if want_V else None
    E = C.c_double(0.0)
    N = C.c_double(0.0)
    lib().orc_eval_unscreened(C.c_int64(len(pts)), _d(pts), _d(w), C.c_int(len(sL)), _i(sa), _i(sL), _i(sn), _i(so),
                              _d(ex), _d(co), _d(xyz), C.c_int(nbf), _d(P), C.c_int64(P.shape[1]), C.c_int(kind),
                              C.c_double(rho_tol), _d(V), C.byref(E), C.byref(N))
    return Result(E.value, N.value, V)


def plan_flops(plan: Plan, shell_L) -> float:
    boff, soff, sh, sL = _i64(plan.batch_off), _i64(plan.shell_off), _i32(plan.shells), _i32(shell_L)
    return float(lib().orc_plan_flops(C.c_int64(len(boff) - 1), _l(boff), _l(soff), _i(sh), _i(sL)))


def functional_pol(kind, ra, rb, saa=None, sab=None, sbb=None, rho_tol=1e-15):
    """Spin-polarised functional (reading A20): f and d f / d (rho_a, rho_b, s_aa, s_ab, s_bb), shape (n, 5)."""
    ra, rb = _f64(np.atleast_1d(ra)), _f64(np.atleast_1d(rb))
    z = np.zeros_like(ra)
    saa = z if saa is None else _f64(np.atleast_1d(saa))
    sab = z if sab is None else _f64(np.atleast_1d(sab))
    sbb = z if sbb is None else _f64(np.atleast_1d(sbb))
    f = np.empty_like(ra)
    v = np.empty((len(ra), 5))
    lib().orc_functional_pol(C.c_int(kind), C.c_int64(len(ra)), _d(ra), _d(rb), _d(saa), _d(sab), _d(sbb),
                             C.c_double(rho_tol), _d(f), _d(v))
    return f, v


@dataclasses.dataclass
class ResultUks:
    E_xc: float
    N_a: float
    N_b: float
    Va: np.ndarray | None
    Vb: np.ndarray | None
    rho: np.ndarray | None = None        # (2, npts)
    grad_rho: np.ndarray | None = None   # (2, npts, 3)
    tau: np.ndarray | None = None        # (2, npts)


def evaluate_uks(plan: Plan, w, basis, xyz, Pa, Pb, kind, rho_tol=1e-15, subset=None, want_V=True, want_rho=False,
                 want_tau=False) -> ResultUks:
    """Mode A evaluation for spin-unrestricted densities (rho_s = sum P^s phi phi) and the meta-GGA intermediate tau."""
    sa, sL, sn, so, ex, co = basis
    sa, sL, sn, so, ex, co = _i32(sa), _i32(sL), _i32(sn), _i32(so), _f64(ex), _f64(co)
    foff, nbf = _func_off(sL)
    xyz, Pa, Pb, w = _f64(xyz), _f64(Pa), _f64(Pb), _f64(w)
    pts = _f64(plan.pts)
    boff, soff, sh = _i64(plan.batch_off), _i64(plan.shell_off), _i32(plan.shells)
    nbat = len(boff) - 1
    sub = _i64(subset) if subset is not None else None
    Va = np.zeros((nbf, nbf)) if want_V else None
    Vb = np.zeros((nbf, nbf)) if want_V else None
    n = len(pts)
    rho = np.zeros((2, n)) if want_rho else None
    gr = np.zeros((2, n, 3)) if want_rho else None
    tau = np.zeros((2, n)) if want_tau else None
    E = C.c_double(0.0)
    N = (C.c_double * 2)(0.0, 0.0)
    lib().orc_eval_uks(C.c_int64(nbat), _l(boff), _l(soff), _i(sh), _l(sub), C.c_int64(0 if sub is None else len(sub)),
                       C.c_int64(n), _d(pts), _d(w), _i(sa), _i(sL), _i(sn), _i(so), _i(foff), _d(ex), _d(co), _d(xyz),
                       C.c_int(nbf), _d(Pa), _d(Pb), C.c_int64(Pa.shape[1]), C.c_int(kind), C.c_double(rho_tol), _d(Va), _d(Vb),
                       C.byref(E), N, _d(rho), _d(gr), _d(tau))
    return ResultUks(E.value, N[0], N[1], Va, Vb, rho, gr, tau)


def functional_mgga(kind, rho, sigma, tau, rho_tol=1e-15):
    """meta-GGA functional (reading A23; kind 7 = MS0 exchange + PBE correlation, 8 = MS0 exchange): f and
    d f / d (rho, sigma, tau), shape (n, 3)."""
    rho, sigma, tau = _f64(np.atleast_1d(rho)), _f64(np.atleast_1d(sigma)), _f64(np.atleast_1d(tau))
    f = np.empty_like(rho)
    v = np.empty((len(rho), 3))
    lib().orc_functional_mgga(C.c_int(kind), C.c_int64(len(rho)), _d(rho), _d(sigma), _d(tau), C.c_double(rho_tol), _d(f), _d(v))
    return f, v


@dataclasses.dataclass
class ResultMgga(Result):
    tau: np.ndarray | None = None


def evaluate_mgga(plan: Plan, w, basis, xyz, P, kind=7, rho_tol=1e-15, subset=None, want_V=True, want_batch=False,
                  want_rho=False) -> ResultMgga:
    """Mode A evaluation of a restricted meta-GGA (tau = 1/2 sum grad Phi . grad X and its potential term)."""
    sa, sL, sn, so, ex, co = basis
    sa, sL, sn, so, ex, co = _i32(sa), _i32(sL), _i32(sn), _i32(so), _f64(ex), _f64(co)
    foff, nbf = _func_off(sL)
    xyz, P, w = _f64(xyz), _f64(P), _f64(w)
    pts = _f64(plan.pts)
    boff, soff, sh = _i64(plan.batch_off), _i64(plan.shell_off), _i32(plan.shells)
    nbat = len(boff) - 1
    sub = _i64(subset) if subset is not None else None
    V = np.zeros((nbf, nbf)) if want_V else None
    Eb = np.zeros(nbat) if want_batch else None
    Nb = np.zeros(nbat) if want_batch else None
    rho = np.zeros(len(pts)) if want_rho else None
    gr = np.zeros((len(pts), 3)) if want_rho else None
    tau = np.zeros(len(pts)) if want_rho else None
    E = C.c_double(0.0)
    N = C.c_double(0.0)
    lib().orc_eval_mgga(C.c_int64(nbat), _l(boff), _l(soff), _i(sh), _l(sub), C.c_int64(0 if sub is None else len(sub)),
                        _d(pts), _d(w), _i(sa), _i(sL), _i(sn), _i(so), _i(foff), _d(ex), _d(co), _d(xyz), C.c_int(nbf),
                        _d(P), C.c_int64(P.shape[1]), C.c_int(kind), C.c_double(rho_tol), _d(V), C.byref(E), C.byref(N),
                        _d(Eb), _d(Nb), _d(rho), _d(gr), _d(tau))
    return ResultMgga(E.value, N.value, V, Eb, Nb, rho, gr, tau)
