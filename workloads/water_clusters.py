"""Synthetic water-cluster workloads shaped like BASELINE.json:configs (stand-ins for the paper's
Taxol/Valinomycin/Olestra/Ubiquitin inputs, Tables 1-2, whose geometries and
basis-set tables are not available here).

Recipe:
  * basis: one synthetic contracted Cartesian basis per ELEMENT, drawn once from BASIS_SEED
    (the same for every config, like a real basis set).  O: s(6) s(3) s(1) p(3) p(1) d(1) = 15
    functions; H: s(3) s(1) p(1) = 5 functions.  Exponents log-uniform (O [0.2,5000], H [0.1,30]),
    sorted descending inside a shell; raw contraction weights U[0.2,1], multiplied by the primitive
    norm and scaled so that the (L,0,0) component has unit self-overlap.
  * geometry: nx*ny*nz cubic lattice, 3.1 A spacing, each molecule rotated by a uniform random
    rotation about its O atom (normalised 4-Gaussian quaternion) and translated rigidly by a uniform
    jitter in [-0.2,0.2]^3 A.  Monomer: O(0,0,0), H(+-0.757, 0.586, 0) A, no rotation/jitter.
  * P = 2 C C^T with C (N_b x N_occ) standard normal, S-orthonormalised (M = C^T S C = L L^T,
    C <- C L^-T); tr(P S) = 2 N_occ.
Units: bohr.
"""
from __future__ import annotations

import dataclasses
import hashlib
import os
from math import pi

import numpy as np

ANGSTROM = 1.8897261246257702  # bohr per Angstrom
BASIS_SEED = 200703143
LATTICE_A = 3.1

# (L, nprim) per shell, in function order
O_SHELLS = [(0, 6), (0, 3), (0, 1), (1, 3), (1, 1), (2, 1)]
H_SHELLS = [(0, 3), (0, 1), (1, 1)]
O_EXP_RANGE = (0.2, 5000.0)
H_EXP_RANGE = (0.1, 30.0)


PURE = 0x100  # shell code bit: pure (real solid harmonic) shell; only changes d shells (5 functions instead of 6)


@dataclasses.dataclass(frozen=True)
class Config:
    name: str
    lattice: tuple
    n_occ: int
    n_rad: int
    n_ang: int
    functional: int  # 0 = LDA Slater+VWN5, 1 = GGA PBE
    geom_seed: int
    pure_d: bool = False  # the O d shell as 5 pure functions (cc-pVDZ-style)


CONFIGS = {
    "c1": Config("c1", (1, 1, 1), 5, 50, 194, 0, BASIS_SEED + 1),
    "c2": Config("c2", (4, 4, 4), 320, 75, 302, 0, BASIS_SEED + 2),
    "c3": Config("c3", (4, 4, 4), 320, 75, 302, 1, BASIS_SEED + 2),  # same geometry/basis/P as c2
    "c4": Config("c4", (8, 8, 4), 1280, 75, 302, 1, BASIS_SEED + 4),
    "c5": Config("c5", (8, 8, 8), 2560, 100, 302, 1, BASIS_SEED + 5),
    # SURVEY.md section 8(f) item 2 ("next" workloads, not in BASELINE.json): u2 = the c2 cluster on a UFG-shaped
    # 99 x 590 grid (Table 2); g1 = an irregular, surface-heavy cluster of 410 waters (1230 atoms,
    # 10250 functions: the shape of the paper's Ubiquitin runs, Table 1) -- lattice (0, 0, n)
    # means n molecules placed by random sequential addition in an ellipsoid
    "u2": Config("u2", (4, 4, 4), 320, 99, 590, 1, BASIS_SEED + 2),
    "g1": Config("g1", (0, 0, 410), 2050, 75, 302, 1, BASIS_SEED + 11),
    # s2 = the c2 cluster on an SFG-shaped 175 x 974 grid (Table 2), PBE
    "s2": Config("s2", (4, 4, 4), 320, 175, 974, 1, BASIS_SEED + 2),
    # geometry-only shape for the weights kernels (never used with a density matrix): 1584 waters, 4752 atoms -- atom
    # lists longer than the SSF kernel's shared-memory cache (2112) and chunk table (4096)
    "x15": Config("x15", (12, 12, 11), 7920, 6, 26, 1, BASIS_SEED + 15),
    # small extra shapes for tests (not in BASELINE.json): 8 and 27 waters
    "w8": Config("w8", (2, 2, 2), 40, 50, 194, 1, BASIS_SEED + 8),
    # pure (spherical) d shells on O: monomer, 8 and 27 waters; 14 functions per O
    "p1": Config("p1", (1, 1, 1), 5, 50, 194, 1, BASIS_SEED + 1, True),
    "p8": Config("p8", (2, 2, 2), 40, 50, 194, 1, BASIS_SEED + 8, True),
    "p8l": Config("p8l", (2, 2, 2), 40, 50, 194, 0, BASIS_SEED + 8, True),
    "p27": Config("p27", (3, 3, 3), 135, 50, 194, 1, BASIS_SEED + 27, True),
    "w27": Config("w27", (3, 3, 3), 135, 50, 194, 1, BASIS_SEED + 27),
}


def ncart(L: int) -> int:
    return (L + 1) * (L + 2) // 2


def nfun(code: int) -> int:
    """Functions of a shell code: low byte L, bit PURE = pure d shell (5 functions)."""
    L = code & 0xff
    return 5 if (code & PURE) and L == 2 else ncart(L)


def cart_components(L: int):
    """(l,m,n) in the order l descending, then m descending: p = x,y,z; d = xx,xy,xz,yy,yz,zz."""
    return [(l, m, L - l - m) for l in range(L, -1, -1) for m in range(L - l, -1, -1)]


def _dfact(n: int) -> int:
    """(n)!! with (-1)!! = 1."""
    r = 1
    while n > 1:
        r *= n
        n -= 2
    return r


def _draw_element_basis(rng, shells, exp_range):
    lo, hi = np.log(exp_range[0]), np.log(exp_range[1])
    out = []
    for (L, nprim) in shells:
        a = np.sort(np.exp(rng.uniform(lo, hi, size=nprim)))[::-1].copy()
        c = rng.uniform(0.2, 1.0, size=nprim)
        norm = (2.0 * a / pi) ** 0.75 * (4.0 * a) ** (L / 2.0) / np.sqrt(_dfact(2 * L - 1))
        d = c * norm
        # self overlap of the (L,0,0) component
        ap = a[:, None] + a[None, :]
        self_ov = np.sum(d[:, None] * d[None, :] * (pi / ap) ** 1.5 * _dfact(2 * L - 1) / (2.0 * ap) ** L)
        d = d / np.sqrt(self_ov)
        out.append((L, a, d))
    return out


def element_basis():
    rng = np.random.default_rng(BASIS_SEED)
    o = _draw_element_basis(rng, O_SHELLS, O_EXP_RANGE)
    h = _draw_element_basis(rng, H_SHELLS, H_EXP_RANGE)
    return {8: o, 1: h}


def _quat_to_rot(q):
    q = q / np.linalg.norm(q)
    w, x, y, z = q
    return np.array([
        [1 - 2 * (y * y + z * z), 2 * (x * y - z * w), 2 * (x * z + y * w)],
        [2 * (x * y + z * w), 1 - 2 * (x * x + z * z), 2 * (y * z - x * w)],
        [2 * (x * z - y * w), 2 * (y * z + x * w), 1 - 2 * (x * x + y * y)]])


_MONOMER = np.array([[0.0, 0.0, 0.0], [0.757, 0.586, 0.0], [-0.757, 0.586, 0.0]])  # Angstrom
_MONOMER_Z = np.array([8, 1, 1], dtype=np.int32)


def _geometry(rng, lattice):
    nx, ny, nz = lattice
    coords, zs = [], []
    if lattice == (1, 1, 1):
        return _MONOMER * ANGSTROM, _MONOMER_Z.copy()
    if nx == 0:
        # irregular cluster: nz molecules, O centres by random sequential addition (min O-O distance 2.6 A) in an
        # ellipsoid with semi-axes (1.6, 1.0, 0.7) R sized for one molecule per (3.3 A)^3; random rotations
        n = nz
        axes = np.array([1.6, 1.0, 0.7]) * (n * 3.3 ** 3 / (4.0 / 3.0 * np.pi * 1.6 * 0.7)) ** (1.0 / 3.0)
        centres = np.zeros((0, 3))
        while len(centres) < n:
            c = rng.uniform(-1.0, 1.0, size=3)
            if c @ c > 1.0:
                continue
            c = c * axes
            if len(centres) and np.min(np.sum((centres - c) ** 2, axis=1)) < 2.6 ** 2:
                continue
            centres = np.vstack([centres, c])
        for c in centres:
            R = _quat_to_rot(rng.standard_normal(4))
            coords.append(_MONOMER @ R.T + c)
            zs.append(_MONOMER_Z)
        return np.concatenate(coords) * ANGSTROM, np.concatenate(zs)
    for i in range(nx):
        for j in range(ny):
            for k in range(nz):
                q = rng.standard_normal(4)
                jit = rng.uniform(-0.2, 0.2, size=3)
                R = _quat_to_rot(q)
                mol = _MONOMER @ R.T + np.array([i, j, k]) * LATTICE_A + jit
                coords.append(mol)
                zs.append(_MONOMER_Z)
    return np.concatenate(coords) * ANGSTROM, np.concatenate(zs)


@dataclasses.dataclass
class Workload:
    name: str
    atoms_xyz: np.ndarray      # (N_A,3) bohr
    atoms_Z: np.ndarray        # (N_A,) int32
    shell_atom: np.ndarray     # (N_s,) int32
    shell_L: np.ndarray        # (N_s,) int32
    shell_nprim: np.ndarray    # (N_s,) int32
    shell_prim_off: np.ndarray  # (N_s,) int32
    exps: np.ndarray           # (nprim_total,)
    coefs: np.ndarray          # (nprim_total,)  (norms included)
    n_basis: int
    n_occ: int
    n_rad: int
    n_ang: int
    functional: int
    P: np.ndarray | None       # (N_b,N_b) symmetric

    @property
    def shell_func_off(self):
        nc = np.array([nfun(int(L)) for L in self.shell_L], dtype=np.int64)
        return np.concatenate([[0], np.cumsum(nc)[:-1]]).astype(np.int32)


def _build_basis(atoms_Z, pure_d=False):
    eb = element_basis()
    shell_atom, shell_L, shell_nprim, shell_off, exps, coefs = [], [], [], [], [], []
    off = 0
    for ia, Z in enumerate(atoms_Z):
        for (L, a, d) in eb[int(Z)]:
            shell_atom.append(ia)
            shell_L.append(L | PURE if (pure_d and L == 2) else L)
            shell_nprim.append(len(a))
            shell_off.append(off)
            exps.append(a)
            coefs.append(d)
            off += len(a)
    return (np.array(shell_atom, np.int32), np.array(shell_L, np.int32), np.array(shell_nprim, np.int32),
            np.array(shell_off, np.int32), np.concatenate(exps), np.concatenate(coefs))


def _int1d_table(p, PA, PB, la, lb):
    """1-D overlap factor  int (x-A)^la (x-B)^lb exp(-p (x-P)^2) dx / sqrt(pi/p)  (binomial expansion
    about the product centre P; int u^{2m} e^{-p u^2} du = (2m-1)!!/(2p)^m sqrt(pi/p))."""
    from math import comb
    out = np.zeros_like(p)
    for s in range(la + 1):
        for t in range(lb + 1):
            if (s + t) % 2:
                continue
            m = (s + t) // 2
            out = out + comb(la, s) * comb(lb, t) * PA ** (la - s) * PB ** (lb - t) * _dfact(2 * m - 1) / (2.0 * p) ** m
    return out


# rows: the five pure d functions (m = -2..2) in terms of xx, xy, xz, yy, yz, zz (all with the radial part whose xx
# component has unit norm): sqrt3 xy, sqrt3 yz, zz - (xx + yy)/2, sqrt3 xz, (sqrt3/2)(xx - yy)
_PURE_D = np.array([[0, 3 ** 0.5, 0, 0, 0, 0], [0, 0, 0, 0, 3 ** 0.5, 0], [-0.5, 0, 0, -0.5, 0, 1.0],
                    [0, 0, 3 ** 0.5, 0, 0, 0], [0.5 * 3 ** 0.5, 0, 0, -0.5 * 3 ** 0.5, 0, 0]])


def overlap_matrix(w: "Workload") -> np.ndarray:
    """Closed-form overlap S of the contracted basis (Gaussian product theorem); pure d shells: T S_cart T^T."""
    if np.any(np.asarray(w.shell_L) & PURE):
        wc = dataclasses.replace(w, shell_L=(np.asarray(w.shell_L) & 0xff).astype(np.int32), P=None)
        wc.n_basis = int(sum(ncart(int(L)) for L in wc.shell_L))
        Sc = overlap_matrix(wc)
        T = np.zeros((w.n_basis, wc.n_basis))
        fo, fc = w.shell_func_off, wc.shell_func_off
        for s_, code in enumerate(w.shell_L):
            n_ = ncart(int(code) & 0xff)
            if int(code) & PURE and (int(code) & 0xff) == 2:
                T[fo[s_]:fo[s_] + 5, fc[s_]:fc[s_] + 6] = _PURE_D
            else:
                T[fo[s_]:fo[s_] + n_, fc[s_]:fc[s_] + n_] = np.eye(n_)
        return T @ Sc @ T.T
    nb = w.n_basis
    S = np.zeros((nb, nb))
    foff = w.shell_func_off
    # group shells by (L, nprim)
    classes = {}
    for s in range(len(w.shell_L)):
        classes.setdefault((int(w.shell_L[s]), int(w.shell_nprim[s])), []).append(s)
    cl = {}
    for key, idx in classes.items():
        idx = np.array(idx)
        L, npr = key
        prim = w.shell_prim_off[idx][:, None] + np.arange(npr)[None, :]
        cl[key] = dict(idx=idx, R=w.atoms_xyz[w.shell_atom[idx]], a=w.exps[prim], d=w.coefs[prim], f0=foff[idx])
    keys = sorted(cl.keys())
    for ka in keys:
        A = cl[ka]
        La = ka[0]
        compsA = cart_components(La)
        for kb in keys:
            B = cl[kb]
            Lb = kb[0]
            compsB = cart_components(Lb)
            nA, nB = len(A["idx"]), len(B["idx"])
            chunk = max(1, int(4e6 // max(1, nB * ka[1] * kb[1])))
            for c0 in range(0, nA, chunk):
                sl = slice(c0, min(nA, c0 + chunk))
                a = A["a"][sl][:, None, :, None]
                b = B["a"][None, :, None, :]
                da = A["d"][sl][:, None, :, None]
                db = B["d"][None, :, None, :]
                RA = A["R"][sl][:, None, None, None, :]
                RB = B["R"][None, :, None, None, :]
                p = a + b
                AB2 = np.sum((RA - RB) ** 2, axis=-1)
                K = np.exp(-a * b / p * AB2) * (pi / p) ** 1.5 * da * db
                Pc = (a[..., None] * RA + b[..., None] * RB) / p[..., None]
                PA = Pc - RA
                PB = Pc - RB
                for ia, (l1, m1, n1) in enumerate(compsA):
                    for ib, (l2, m2, n2) in enumerate(compsB):
                        v = (K * _int1d_table(p, PA[..., 0], PB[..., 0], l1, l2)
                               * _int1d_table(p, PA[..., 1], PB[..., 1], m1, m2)
                               * _int1d_table(p, PA[..., 2], PB[..., 2], n1, n2)).sum(axis=(2, 3))
                        S[np.ix_(A["f0"][sl] + ia, B["f0"] + ib)] = v
    return 0.5 * (S + S.T)


def _cache_dir():
    d = os.environ.get("XC_WORKLOAD_CACHE", "/tmp/xc_workload_cache")
    os.makedirs(d, exist_ok=True)
    return d


def make_workload(name: str, with_P: bool = True, cache: bool = True) -> Workload:
    cfg = CONFIGS[name]
    rng = np.random.default_rng(cfg.geom_seed)
    xyz, Z = _geometry(rng, cfg.lattice)
    sa, sL, sn, so, exps, coefs = _build_basis(Z, cfg.pure_d)
    nb = int(sum(nfun(int(L)) for L in sL))
    w = Workload(name, xyz, Z.astype(np.int32), sa, sL, sn, so, exps, coefs, nb, cfg.n_occ, cfg.n_rad, cfg.n_ang,
                 cfg.functional, None)
    if not with_P:
        return w
    key = hashlib.sha1(("v1|%d|%s|%d|%d%s" % (cfg.geom_seed, cfg.lattice, cfg.n_occ, BASIS_SEED, "|pure" if cfg.pure_d else "")).encode()).hexdigest()[:16]
    path = os.path.join(_cache_dir(), "P_%s_%s.npy" % (cfg.name if cfg.name not in ("c3", "u2", "s2") else "c2", key))
    if cache and os.path.exists(path):
        P = np.load(path)
        if P.shape == (nb, nb):
            w.P = P
            return w
    C = rng.standard_normal((nb, cfg.n_occ))
    S = overlap_matrix(w)
    M = C.T @ (S @ C)
    Lc = np.linalg.cholesky(0.5 * (M + M.T))
    C = np.linalg.solve(Lc, C.T).T  # C L^-T
    P = 2.0 * (C @ C.T)
    P = 0.5 * (P + P.T)
    w.P = P
    if cache:
        tmp = path + ".tmp%d.npy" % os.getpid()
        np.save(tmp, P)
        os.replace(tmp, path)
    return w


def spin_density_matrices(w: Workload, n_a: int, n_b: int, seed: int = 7):
    """(P_a, P_b) of a spin-unrestricted determinant: P_s = C[:, :n_s] C[:, :n_s]^T with C random, S-orthonormal
    (C^T S C = 1), so tr(P_s S) = n_s; n_b <= n_a (the first n_b orbitals are doubly occupied)."""
    rng = np.random.default_rng(BASIS_SEED + 1000 + seed)
    C = rng.standard_normal((w.n_basis, max(n_a, n_b)))
    S = overlap_matrix(w)
    M = C.T @ (S @ C)
    Lc = np.linalg.cholesky(0.5 * (M + M.T))
    C = np.linalg.solve(Lc, C.T).T
    Pa, Pb = C[:, :n_a] @ C[:, :n_a].T, C[:, :n_b] @ C[:, :n_b].T
    return 0.5 * (Pa + Pa.T), 0.5 * (Pb + Pb.T)
