"""Thin ctypes binding of libxc_b200.so (include/xc_b200.h): argument marshalling only -- every step of
the hot path runs in the library's CUDA kernels.  torch is used for device memory and streams.
There is no fallback: if the shared library is missing or cannot be loaded, importing this module fails."""
from __future__ import annotations

import ctypes as C
import dataclasses
import os

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(HERE, "libxc_b200.so")

XC_OK, XC_EINVAL, XC_EUNSUPPORTED, XC_ENOMEM, XC_ECUDA = 0, -1, -2, -3, -4
XC_EVAL_REUSE_WEIGHTS, XC_EVAL_DIAG, XC_EVAL_COUNT_PAIRS = 1, 2, 4


class XcAtom(C.Structure):
    _fields_ = [("x", C.c_double), ("y", C.c_double), ("z", C.c_double), ("Z", C.c_int32), ("_pad", C.c_int32)]


class XcShell(C.Structure):
    _fields_ = [("atom", C.c_int32), ("L", C.c_int32), ("nprim", C.c_int32), ("prim_off", C.c_int32)]


class XcGridSpec(C.Structure):
    _fields_ = [("n_rad", C.c_int32), ("n_ang", C.c_int32), ("radial", C.c_int32), ("angular", C.c_int32),
                ("partition", C.c_int32), ("functional", C.c_int32), ("max_batch_pts", C.c_int32), ("flags", C.c_int32),
                ("eta", C.c_double), ("mk_alpha", C.c_double), ("rho_tol", C.c_double)]


XC_SPEC_SPLIT_CLASS1 = 2


def grid_spec(n_rad, n_ang, functional, angular=0, partition=0, max_batch_pts=512, eta=1e-10, mk_alpha=5.0,
              rho_tol=1e-15, flags=0) -> XcGridSpec:
    return XcGridSpec(n_rad, n_ang, 0, angular, partition, functional, max_batch_pts, flags, eta, mk_alpha, rho_tol)


class XcError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__("libxc_b200: %s (%d): %s" % (_lib.xc_strerror(code).decode(), code, msg))
        self.code = code


def _load():
    if not os.path.exists(LIB_PATH):
        raise ImportError("libxc_b200.so not built (run `python -m paper_2007_03143_b200.build` or __graft_entry__.build()); "
                          "there is no CPU fallback")
    lib = C.CDLL(LIB_PATH)
    vp, dp, ip, lp = C.c_void_p, C.POINTER(C.c_double), C.POINTER(C.c_int32), C.POINTER(C.c_int64)
    lib.xc_strerror.restype = C.c_char_p
    lib.xc_strerror.argtypes = [C.c_int]
    lib.xc_last_error.restype = C.c_char_p
    lib.xc_plan_create.argtypes = [C.POINTER(XcAtom), C.c_int32, C.POINTER(XcShell), C.c_int32, dp, dp, C.c_int32,
                                   C.POINTER(XcGridSpec), C.c_int32, C.POINTER(vp)]
    lib.xc_plan_info.argtypes = [vp, lp, lp, ip, lp, dp]
    lib.xc_plan_stats.argtypes = [vp, dp]
    lib.xc_plan_export.argtypes = [vp, dp, dp, ip, lp, lp, lp, ip]
    lib.xc_eval.argtypes = [vp, vp, C.c_int64, vp, C.c_int64, dp, dp, C.c_int32, vp]
    lib.xc_eval_host.argtypes = [vp, vp, C.c_int64, vp, C.c_int64, dp, dp, C.c_int32]
    lib.xc_eval_uks.argtypes = [vp, vp, vp, C.c_int64, vp, vp, C.c_int64, dp, dp, C.c_int32, vp]
    lib.xc_eval_uks_densities.argtypes = [vp, dp, dp]
    lib.xc_eval_tau.argtypes = [vp, vp, C.c_int64, vp, C.c_int32, vp]
    lib.xc_eval_diagnostics.argtypes = [vp, dp, dp, dp, dp, dp]
    lib.xc_eval_timings.argtypes = [vp, C.POINTER(C.c_float), ip]
    lib.xc_eval_counters.argtypes = [vp, lp, lp]
    lib.xc_plan_destroy.argtypes = [vp]
    lib.xc_integrate.argtypes = [C.POINTER(XcAtom), C.c_int32, C.POINTER(XcShell), C.c_int32, dp, dp, C.c_int32,
                                 C.POINTER(XcGridSpec), C.c_int32, vp, C.c_int64, vp, C.c_int64, dp, dp, vp]
    lib.xc_partition_weights.argtypes = [C.POINTER(XcAtom), C.c_int32, C.c_int32, C.c_int64, vp, vp, vp, vp, vp, vp, vp]
    lib.xc_functional.argtypes = [C.c_int32, C.c_int64, vp, vp, C.c_double, vp, vp, vp, vp]
    lib.xc_functional_uks_static.argtypes = [C.c_int32, C.c_int64, vp, vp, vp, C.c_double, vp, vp, vp, vp]
    lib.xc_measure_fp64_peak.argtypes = [C.c_int32, C.c_int32, C.c_int32, dp, dp]
    for name in EXPORTED:
        getattr(lib, name)  # fail loudly if a declared symbol is missing
    return lib


EXPORTED = ["xc_plan_create", "xc_plan_info", "xc_plan_export", "xc_eval", "xc_eval_host", "xc_eval_uks", "xc_eval_uks_densities", "xc_eval_tau", "xc_eval_diagnostics",
            "xc_eval_timings", "xc_eval_counters", "xc_plan_stats", "xc_plan_destroy", "xc_integrate", "xc_partition_weights",
            "xc_functional", "xc_functional_uks_static", "xc_measure_fp64_peak", "xc_strerror", "xc_last_error"]

_lib = _load()


def _check(rc):
    if rc != XC_OK:
        raise XcError(rc, _lib.xc_last_error().decode())


def _dp(a):
    return None if a is None else a.ctypes.data_as(C.POINTER(C.c_double))


def _atoms(xyz, Z):
    xyz = np.ascontiguousarray(xyz, np.float64)
    arr = (XcAtom * len(xyz))()
    for i in range(len(xyz)):
        arr[i] = XcAtom(xyz[i, 0], xyz[i, 1], xyz[i, 2], int(Z[i]) if Z is not None else 0, 0)
    return arr


def _shells(atom, L, nprim, off):
    arr = (XcShell * len(atom))()
    for i in range(len(atom)):
        arr[i] = XcShell(int(atom[i]), int(L[i]), int(nprim[i]), int(off[i]))
    return arr


def _stream_ptr(stream):
    if stream is None:
        import torch
        return C.c_void_p(torch.cuda.current_stream().cuda_stream)
    return C.c_void_p(int(stream) if isinstance(stream, int) else stream.cuda_stream)


@dataclasses.dataclass
class PlanExport:
    pts: np.ndarray
    wq: np.ndarray
    parent: np.ndarray
    orig: np.ndarray
    batch_off: np.ndarray
    shell_off: np.ndarray
    shells: np.ndarray


class Plan:
    """xc_plan: grid + batches + screening + device workspaces for one molecule/basis/grid."""

    def __init__(self, atoms_xyz, atoms_Z, shell_atom, shell_L, shell_nprim, shell_prim_off, exps, coefs,
                 spec: XcGridSpec, device: int = 0):
        exps = np.ascontiguousarray(exps, np.float64)
        coefs = np.ascontiguousarray(coefs, np.float64)
        at = _atoms(atoms_xyz, atoms_Z)
        sh = _shells(shell_atom, shell_L, shell_nprim, shell_prim_off)
        h = C.c_void_p()
        _check(_lib.xc_plan_create(at, len(at), sh, len(sh), _dp(exps), _dp(coefs), len(exps), C.byref(spec), device,
                                   C.byref(h)))
        self._h = h
        self.spec = spec
        self.device = device
        npts, nbat, nsh = C.c_int64(), C.c_int64(), C.c_int64()
        nbas = C.c_int32()
        fl = C.c_double()
        _check(_lib.xc_plan_info(h, C.byref(npts), C.byref(nbat), C.byref(nbas), C.byref(nsh), C.byref(fl)))
        self.n_points, self.n_batches, self.n_basis = npts.value, nbat.value, nbas.value
        self.n_shell_entries, self.algorithmic_flops = nsh.value, fl.value

    @classmethod
    def from_workload(cls, w, spec=None, device=0, **kw):
        if spec is None:
            spec = grid_spec(w.n_rad, w.n_ang, w.functional, **kw)
        return cls(w.atoms_xyz, w.atoms_Z, w.shell_atom, w.shell_L, w.shell_nprim, w.shell_prim_off, w.exps, w.coefs,
                   spec, device)

    def stats(self):
        s = (C.c_double * 12)()
        _check(_lib.xc_plan_stats(self._h, s))
        return dict(sum_nb_nq=s[0], sum_nb2=s[1], flops=s[2], max_nb=int(s[3]), mean_nq=s[4], workspace_bytes=s[5],
                    w_partners_mean=s[6], w_partners_max=int(s[7]), w_owners_mean=s[8], w_owners_max=int(s[9]),
                    max_ns=int(s[10]))

    def export(self) -> PlanExport:
        n, nb = self.n_points, self.n_batches
        pts = np.empty((n, 3))
        wq = np.empty(n)
        parent = np.empty(n, np.int32)
        orig = np.empty(n, np.int64)
        boff = np.empty(nb + 1, np.int64)
        soff = np.empty(nb + 1, np.int64)
        shells = np.empty(self.n_shell_entries, np.int32)
        _check(_lib.xc_plan_export(self._h, _dp(pts), _dp(wq), parent.ctypes.data_as(C.POINTER(C.c_int32)),
                                   orig.ctypes.data_as(C.POINTER(C.c_int64)), boff.ctypes.data_as(C.POINTER(C.c_int64)),
                                   soff.ctypes.data_as(C.POINTER(C.c_int64)),
                                   shells.ctypes.data_as(C.POINTER(C.c_int32))))
        return PlanExport(pts, wq, parent, orig, boff, soff, shells)

    def eval(self, P, V=None, reuse_weights=False, stream=None, diag=False, count_pairs=False):
        """P, V: torch CUDA float64 tensors (n_basis x n_basis). Returns (E_xc, N_el, V).
        diag: also keep rho / grad rho of every point for diagnostics() (XC_EVAL_DIAG)."""
        import torch
        assert P.is_cuda and P.dtype == torch.float64 and P.dim() == 2 and P.stride(1) == 1
        if V is None:
            V = torch.empty((self.n_basis, self.n_basis), dtype=torch.float64, device=P.device)
        assert V.is_cuda and V.dtype == torch.float64 and V.stride(1) == 1
        E, N = C.c_double(), C.c_double()
        _check(_lib.xc_eval(self._h, C.c_void_p(P.data_ptr()), P.stride(0), C.c_void_p(V.data_ptr()), V.stride(0),
                            C.byref(E), C.byref(N), (XC_EVAL_REUSE_WEIGHTS if reuse_weights else 0) | (XC_EVAL_DIAG if diag else 0) | (XC_EVAL_COUNT_PAIRS if count_pairs else 0),
                            _stream_ptr(stream)))
        return E.value, N.value, V

    def eval_uks(self, Pa, Pb, Va=None, Vb=None, reuse_weights=False, stream=None):
        """Spin-unrestricted build (xc_eval_uks): Pa, Pb torch CUDA float64 (n_basis x n_basis, same row stride).
        Returns (E_xc, (N_a, N_b), Va, Vb)."""
        import torch
        for t in (Pa, Pb):
            assert t.is_cuda and t.dtype == torch.float64 and t.dim() == 2 and t.stride(1) == 1
        assert Pa.stride(0) == Pb.stride(0)
        if Va is None:
            Va = torch.empty((self.n_basis, self.n_basis), dtype=torch.float64, device=Pa.device)
        if Vb is None:
            Vb = torch.empty((self.n_basis, self.n_basis), dtype=torch.float64, device=Pa.device)
        assert Va.stride(1) == 1 and Vb.stride(1) == 1 and Va.stride(0) == Vb.stride(0)
        E = C.c_double()
        N = (C.c_double * 2)()
        _check(_lib.xc_eval_uks(self._h, C.c_void_p(Pa.data_ptr()), C.c_void_p(Pb.data_ptr()), Pa.stride(0),
                                C.c_void_p(Va.data_ptr()), C.c_void_p(Vb.data_ptr()), Va.stride(0), C.byref(E), N,
                                XC_EVAL_REUSE_WEIGHTS if reuse_weights else 0, _stream_ptr(stream)))
        return E.value, (N[0], N[1]), Va, Vb

    def eval_tau(self, P, reuse_weights=False, stream=None):
        """tau_i = 1/2 sum grad Phi . grad X for the density matrix P (torch CUDA float64): tensor of n_points, plan order."""
        import torch
        assert P.is_cuda and P.dtype == torch.float64 and P.dim() == 2 and P.stride(1) == 1
        tau = torch.empty(self.n_points, dtype=torch.float64, device=P.device)
        _check(_lib.xc_eval_tau(self._h, C.c_void_p(P.data_ptr()), P.stride(0), C.c_void_p(tau.data_ptr()),
                                XC_EVAL_REUSE_WEIGHTS if reuse_weights else 0, _stream_ptr(stream)))
        return tau

    def uks_densities(self, want_grad=True):
        """rho_s (2, n_points) and grad rho_s (2, n_points, 3) of the last eval_uks (undefined where w = 0)."""
        n = self.n_points
        rho = np.empty((2, n))
        gr = np.empty((2, n, 3)) if want_grad else None
        _check(_lib.xc_eval_uks_densities(self._h, _dp(rho), _dp(gr)))
        return rho, gr

    def eval_host(self, P, V=None, reuse_weights=False):
        """P, V: host buffers (numpy arrays or pinned torch CPU tensors), float64, row-major."""
        Pp, ldp = _host_ptr(P)
        if V is None:
            V = np.empty((self.n_basis, self.n_basis))
        Vp, ldv = _host_ptr(V)
        E, N = C.c_double(), C.c_double()
        _check(_lib.xc_eval_host(self._h, Pp, ldp, Vp, ldv, C.byref(E), C.byref(N), 1 if reuse_weights else 0))
        return E.value, N.value, V

    def diagnostics(self, want_points=True, want_rho=False):
        """w (want_points), rho / grad_rho (want_rho: the last eval must have run with diag=True), per-batch E / N_el partials."""
        n, nb = self.n_points, self.n_batches
        w = np.empty(n) if want_points else None
        rho = np.empty(n) if want_rho else None
        gr = np.empty((n, 3)) if want_rho else None
        Eb, Nb = np.empty(nb), np.empty(nb)
        _check(_lib.xc_eval_diagnostics(self._h, _dp(w), _dp(rho), _dp(gr), _dp(Eb), _dp(Nb)))
        return dict(w=w, rho=rho, grad_rho=gr, E_batch=Eb, N_batch=Nb)

    def counters(self):
        """(pair factors evaluated by step (a) in the last eval(count_pairs=True), points the SSF kernel visits)."""
        a, b = C.c_int64(), C.c_int64()
        _check(_lib.xc_eval_counters(self._h, C.byref(a), C.byref(b)))
        return a.value, b.value

    def timings(self):
        ms = (C.c_float * 5)()
        n = C.c_int32()
        _check(_lib.xc_eval_timings(self._h, ms, C.byref(n)))
        return dict(weights_ms=ms[0], pack_ms=ms[1], batch_ms=ms[2], finalize_ms=ms[3], total_ms=ms[4],
                    launches=n.value)

    def close(self):
        if getattr(self, "_h", None):
            _lib.xc_plan_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


def _host_ptr(a):
    if isinstance(a, np.ndarray):
        assert a.dtype == np.float64 and a.ndim == 2 and a.strides[1] == 8
        return C.c_void_p(a.ctypes.data), a.strides[0] // 8
    assert (not a.is_cuda) and a.dim() == 2 and a.stride(1) == 1  # torch CPU tensor
    return C.c_void_p(a.data_ptr()), a.stride(0)


def xc_integrate(w, P, spec=None, device=0, stream=None):
    """One-shot form of BASELINE.json:north_star: (atoms, shells, grid_spec, P) -> (E_xc, V_xc, N_el)."""
    import torch
    if spec is None:
        spec = grid_spec(w.n_rad, w.n_ang, w.functional)
    exps = np.ascontiguousarray(w.exps, np.float64)
    coefs = np.ascontiguousarray(w.coefs, np.float64)
    at = _atoms(w.atoms_xyz, w.atoms_Z)
    sh = _shells(w.shell_atom, w.shell_L, w.shell_nprim, w.shell_prim_off)
    V = torch.empty_like(P)
    E, N = C.c_double(), C.c_double()
    _check(_lib.xc_integrate(at, len(at), sh, len(sh), _dp(exps), _dp(coefs), len(exps), C.byref(spec), device,
                             C.c_void_p(P.data_ptr()), P.stride(0), C.c_void_p(V.data_ptr()), V.stride(0), C.byref(E),
                             C.byref(N), _stream_ptr(stream)))
    return E.value, V, N.value


def partition_weights(atoms_xyz, pts, wq, parent, partition=0, stream=None):
    """Step (a) alone on torch CUDA tensors; pts (n,3)."""
    import torch
    at = _atoms(atoms_xyz, None)
    x, y, z = (pts[:, k].contiguous() for k in range(3))
    out = torch.empty_like(wq)
    _check(_lib.xc_partition_weights(at, len(at), partition, wq.numel(), C.c_void_p(x.data_ptr()),
                                     C.c_void_p(y.data_ptr()), C.c_void_p(z.data_ptr()), C.c_void_p(wq.data_ptr()),
                                     C.c_void_p(parent.data_ptr()), C.c_void_p(out.data_ptr()), _stream_ptr(stream)))
    return out


def functional(kind, rho, sigma, rho_tol=1e-15, stream=None):
    """Step (f) point values on torch CUDA tensors: returns f, v_rho, v_sigma."""
    import torch
    f, vr, vs = torch.empty_like(rho), torch.empty_like(rho), torch.empty_like(rho)
    _check(_lib.xc_functional(kind, rho.numel(), C.c_void_p(rho.data_ptr()), C.c_void_p(sigma.data_ptr()), rho_tol,
                              C.c_void_p(f.data_ptr()), C.c_void_p(vr.data_ptr()), C.c_void_p(vs.data_ptr()),
                              _stream_ptr(stream)))
    return f, vr, vs


XC_STATIC_MAX_POINTS = 1 << 23


def functional_uks_static(kind, w, rho, grho, cA, cG, out3, rho_tol=1e-15, stream=None):
    """xc_functional_uks_static: the spin-coupling step without any allocation (the scratch is a static device array).
    Every tensor is a caller-owned torch CUDA float64 tensor of the current device: w (n), rho (2, n), grho (2, n, 3) or
    None for kind 0, outputs cA (2, n), cG (2, n, 3) or None, out3 (3) = E_xc, N_a, N_b.  Stream-ordered, no sync."""
    ptr = lambda t: C.c_void_p(t.data_ptr() if t is not None else 0)
    for t in (w, rho, grho, cA, cG, out3):
        assert t is None or (t.is_cuda and t.is_contiguous() and t.element_size() == 8)
    _check(_lib.xc_functional_uks_static(kind, w.numel(), ptr(w), ptr(rho), ptr(grho), rho_tol, ptr(cA), ptr(cG), ptr(out3),
                                         _stream_ptr(stream)))


def measure_fp64_peak(kind=1, device=0, reps=5):
    """FP64 pipe rate of `device` in TFLOP/s (kind 0 = DFMA, 1 = DMMA) and the SM clock it implies (MHz)."""
    t, c = C.c_double(), C.c_double()
    _check(_lib.xc_measure_fp64_peak(kind, device, reps, C.byref(t), C.byref(c)))
    return t.value, c.value
