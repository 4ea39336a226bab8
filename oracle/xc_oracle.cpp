// xc_oracle.cpp -- CPU ORACLE for the XC quadrature of arxiv 2007.03143.   TEST INFRASTRUCTURE ONLY.
//
// Plain, slow, fp64, obviously-correct restatement of what the hot path computes, written from
// /root/reference/PAPER.md (cited as PAPER.md:L<line>) and the readings listed in DESIGN.md
// ("Readings of the paper", A1..A18).  It shares NO code with the CUDA path
// (paper_2007_03143_b200/csrc): no common headers, helpers, tables or constants.  Only tests/,
// __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may load it.
//
// No blocking, fusion or reordering beyond what the paper's equations state: every contraction is
// the literal loop nest of the equation it cites.  OpenMP is used only for "parallel for B_j in B"
// (Alg. 4) -- batches are independent -- never inside a formula.
//
// Pins (tests/test_oracle_*.py, all -m "not gpu"): closed-form one-primitive Slater energy (P1),
// sum w rho = tr(P S) (P2), V symmetric (P3), finite-difference dE/dP = V (P4), unscreened brute
// force (P5), functional values vs 40-digit mpmath (P6), functional limits (P7), collocation vs
// finite differences and closed-form overlaps (P8), plan validity (P9), translation invariance (P10);
// spin-unrestricted path and tau (readings A20-A22; tests/test_oracle_uks.py): polarised functionals vs 40-digit mpmath,
// ferromagnetic uniform gas, zeta = 0 and spin-scaling reductions to the pinned unpolarised forms, P_a = P_b limit,
// tr(P_s S), dE/dP^s = V^s, int tau = (2L+3) alpha/2 for one primitive, tau against the einsum definition;
// meta-GGA MS0x+PBEc (reading A23; tests/test_oracle_uks.py): mpmath golden, Slater limit at alpha = 1, alpha = 0 for one
// orbital, dE/dP = V with the tau term;
// pure d shells (reading A19): typed values, orthonormality with s and p on a fine grid, Unsold's theorem, tr(PS), dE/dP = V.
// Parity UNPINNED against the paper itself: the paper prints no E_xc / V_xc / N_el value.
//
// Build: g++ -O2 -fopenmp -shared -fPIC -o libxc_oracle.so xc_oracle.cpp   (oracle/build.py)

#include <algorithm>
#include <cmath>
#include <cstdint>
#include <cstdlib>
#include <cstring>
#include <vector>
#ifdef _OPENMP
#include <omp.h>
#endif

namespace {

const double kPi = 3.14159265358979323846264338327950288;

// ---------------------------------------------------------------------------------------------
// Forward-mode dual numbers in (rho, sigma): value + d/drho + d/dsigma.  The oracle differentiates
// the ENERGY expression f(rho,sigma) mechanically (A11: v_rho = d(rho eps)/d rho,
// v_sigma = d(rho eps)/d sigma); the CUDA path uses hand-derived closed forms instead.
// ---------------------------------------------------------------------------------------------
struct D2 {
  double v, a, b;  // value, d/drho, d/dsigma
};
inline D2 mk(double v) { return {v, 0.0, 0.0}; }
inline D2 operator+(D2 x, D2 y) { return {x.v + y.v, x.a + y.a, x.b + y.b}; }
inline D2 operator-(D2 x, D2 y) { return {x.v - y.v, x.a - y.a, x.b - y.b}; }
inline D2 operator-(D2 x) { return {-x.v, -x.a, -x.b}; }
inline D2 operator*(D2 x, D2 y) { return {x.v * y.v, x.a * y.v + x.v * y.a, x.b * y.v + x.v * y.b}; }
inline D2 operator/(D2 x, D2 y) {
  double q = x.v / y.v;
  return {q, (x.a - q * y.a) / y.v, (x.b - q * y.b) / y.v};
}
inline D2 operator+(D2 x, double c) { return {x.v + c, x.a, x.b}; }
inline D2 operator+(double c, D2 x) { return {x.v + c, x.a, x.b}; }
inline D2 operator-(D2 x, double c) { return {x.v - c, x.a, x.b}; }
inline D2 operator-(double c, D2 x) { return {c - x.v, -x.a, -x.b}; }
inline D2 operator*(D2 x, double c) { return {x.v * c, x.a * c, x.b * c}; }
inline D2 operator*(double c, D2 x) { return {x.v * c, x.a * c, x.b * c}; }
inline D2 operator/(D2 x, double c) { return {x.v / c, x.a / c, x.b / c}; }
inline D2 operator/(double c, D2 x) { return mk(c) / x; }
inline D2 dlog(D2 x) { return {std::log(x.v), x.a / x.v, x.b / x.v}; }
inline D2 dexp(D2 x) {
  double e = std::exp(x.v);
  return {e, e * x.a, e * x.b};
}
inline D2 dexpm1(D2 x) {
  double e = std::exp(x.v);
  return {std::expm1(x.v), e * x.a, e * x.b};
}
inline D2 dlog1p(D2 x) { return {std::log1p(x.v), x.a / (1.0 + x.v), x.b / (1.0 + x.v)}; }
inline D2 datan(D2 x) {
  double d = 1.0 / (1.0 + x.v * x.v);
  return {std::atan(x.v), x.a * d, x.b * d};
}
inline D2 dsqrt(D2 x) {
  double s = std::sqrt(x.v);
  return {s, 0.5 * x.a / s, 0.5 * x.b / s};
}
inline D2 dcbrt(D2 x) {
  double c = std::cbrt(x.v);
  double d = c / (3.0 * x.v);
  return {c, x.a * d, x.b * d};
}

// ---- functional energy densities per unit volume f(rho, sigma), spin-unpolarised ------------
// DESIGN.md "Functional definitions" (the paper defers to LIBXC/ExchCXX).

const double kCx = 0.7385587663820224058842300326808360;  // (3/4)(3/pi)^(1/3)

inline D2 rs_of(D2 rho) { return dcbrt(mk(3.0 / (4.0 * kPi)) / rho); }

// Slater exchange: f_x = -C_x rho^(4/3)
inline D2 f_slater(D2 rho) { return -kCx * rho * dcbrt(rho); }

// VWN5 paramagnetic correlation energy per particle, Vosko-Wilk-Nusair 1980 fit "V".
inline D2 eps_vwn5(D2 rho) {
  const double A = 0.0310907, x0 = -0.10498, b = 3.72744, c = 12.9352;
  const double Q = std::sqrt(4.0 * c - b * b);
  const double Xx0 = x0 * x0 + b * x0 + c;
  D2 x = dsqrt(rs_of(rho));
  D2 X = x * x + b * x + c;
  D2 at = datan(Q / (2.0 * x + b));
  D2 t1 = dlog(x * x / X);
  D2 t2 = (2.0 * b / Q) * at;
  D2 t3 = dlog((x - x0) * (x - x0) / X) + (2.0 * (b + 2.0 * x0) / Q) * at;
  return A * (t1 + t2 - (b * x0 / Xx0) * t3);
}

// PW92 uniform-gas correlation energy per particle (unpolarised), "modified" A (A12).
inline D2 eps_pw92(D2 rho) {
  const double A = 0.0310907, a1 = 0.21370, b1 = 7.5957, b2 = 3.5876, b3 = 1.6382, b4 = 0.49294;
  D2 rs = rs_of(rho);
  D2 srs = dsqrt(rs);
  D2 den = 2.0 * A * (b1 * srs + b2 * rs + b3 * rs * srs + b4 * rs * rs);
  return -2.0 * A * (1.0 + a1 * rs) * dlog1p(1.0 / den);
}

// PBE exchange: f_x = -C_x rho^(4/3) F(s^2), F = 1 + kappa - kappa/(1 + mu s^2/kappa)
inline D2 f_pbe_x(D2 rho, D2 sigma) {
  const double kappa = 0.804, mu = 0.2195149727645171;
  const double c = 4.0 * std::pow(3.0 * kPi * kPi, 2.0 / 3.0);
  D2 r13 = dcbrt(rho);
  D2 r83 = rho * rho * r13 * r13;
  D2 s2 = sigma / (c * r83);
  D2 F = (1.0 + kappa) - kappa / (1.0 + (mu / kappa) * s2);
  return -kCx * rho * r13 * F;
}

// PBE correlation: f_c = rho (eps_unif + H)
inline D2 f_pbe_c(D2 rho, D2 sigma) {
  const double gamma = 0.031090690869654895, beta = 0.06672455060314922;
  D2 eu = eps_pw92(rho);
  D2 kF = dcbrt(3.0 * kPi * kPi * rho);
  D2 ks2 = 4.0 * kF / kPi;
  D2 t2 = sigma / (4.0 * ks2 * rho * rho);
  D2 Ac = (beta / gamma) / dexpm1(-eu / gamma);
  D2 At2 = Ac * t2;
  D2 H = gamma * dlog1p((beta / gamma) * t2 * (1.0 + At2) / (1.0 + At2 + At2 * At2));
  return rho * (eu + H);
}

// functional kind: 0 = LDA Slater+VWN5, 1 = GGA PBE; extra kinds for pins: 2 = Slater only,
// 3 = VWN5 only, 4 = PW92 only (rho eps), 5 = PBE x only, 6 = PBE c only.
inline D2 f_xc(int kind, D2 rho, D2 sigma) {
  switch (kind) {
    case 0: return f_slater(rho) + rho * eps_vwn5(rho);
    case 1: return f_pbe_x(rho, sigma) + f_pbe_c(rho, sigma);
    case 2: return f_slater(rho);
    case 3: return rho * eps_vwn5(rho);
    case 4: return rho * eps_pw92(rho);
    case 5: return f_pbe_x(rho, sigma);
    default: return f_pbe_c(rho, sigma);
  }
}

inline bool is_gga(int kind) { return kind == 1 || kind == 5 || kind == 6; }

// O9 (A12): points with rho <= rho_tol contribute nothing.
inline void eval_point(int kind, double rho, double sigma, double rho_tol, double* f, double* vr, double* vs) {
  if (!(rho > rho_tol)) {
    *f = 0.0; *vr = 0.0; *vs = 0.0;
    return;
  }
  D2 r = {rho, 1.0, 0.0};
  D2 s = {sigma, 0.0, 1.0};
  D2 e = f_xc(kind, r, s);
  *f = e.v; *vr = e.a; *vs = is_gga(kind) ? e.b : 0.0;
}

inline int ncart(int L) { return (L + 1) * (L + 2) / 2; }
// Shell code (reading A19): low byte = angular momentum L; bit 8 (0x100) set = "pure" shell, whose functions are
// the 2L+1 real solid harmonics instead of the (L+1)(L+2)/2 Cartesian monomials ("spherical Gaussian
// functions"; L323 cc-pVDZ).  Only d shells change: a pure s or p shell has the same functions as the Cartesian one.
inline int sh_L(int code) { return code & 0xff; }
inline bool sh_pure(int code) { return (code & 0x100) != 0 && sh_L(code) == 2; }
inline int nfun(int code) { return sh_pure(code) ? 5 : ncart(sh_L(code)); }

// ---- partition cell functions ------------------------------------------------------------------
// SSF (Stratmann-Scuseria-Frisch 1996), a = 0.64 (A1/A2): s = (1 - g)/2,
// g = -1 (mu <= -a), +1 (mu >= a), else (35 z - 35 z^3 + 21 z^5 - 5 z^7)/16, z = mu/a.
inline double s_ssf(double mu) {
  const double a = 0.64;
  if (mu <= -a) return 1.0;
  if (mu >= a) return 0.0;
  double z = mu / a, z2 = z * z;
  double g = z * (35.0 + z2 * (-35.0 + z2 * (21.0 - 5.0 * z2))) / 16.0;
  return 0.5 * (1.0 - g);
}
// Becke 1988: s = (1 - p(p(p(mu))))/2, p(t) = 1.5 t - 0.5 t^3, no atomic-size adjustment.
inline double s_becke(double mu) {
  double p = mu;
  for (int k = 0; k < 3; ++k) p = 1.5 * p - 0.5 * p * p * p;
  return 0.5 * (1.0 - p);
}

inline double dist3(const double* a, const double* b) {
  double dx = a[0] - b[0], dy = a[1] - b[1], dz = a[2] - b[2];
  return std::sqrt(dx * dx + dy * dy + dz * dz);
}

// Alg. 1 with reading A7: the cuboid [V,W] and the sphere (R, rcut) intersect
// iff the squared distance from R to the cuboid is <= rcut^2.
inline bool cuboid_sphere_intersect(const double* R, double rcut, const double* V, const double* W) {
  double d = rcut * rcut;
  for (int p = 0; p < 3; ++p) {
    if (R[p] < V[p]) d -= (R[p] - V[p]) * (R[p] - V[p]);
    else if (R[p] > W[p]) d -= (R[p] - W[p]) * (R[p] - W[p]);
  }
  return d >= 0.0;
}

// O7: one contracted Cartesian shell at one point (Eq. (7)); components in the order
// l descending then m descending (A5).  phi[c], and if grad != nullptr grad[3*c + {0,1,2}].
inline double ipow(double x, int n) {
  double r = 1.0;
  for (int k = 0; k < n; ++k) r *= x;
  return r;
}
inline void shell_at_point(int code, int nprim, const double* alpha, const double* d, const double* R, const double* r,
                           double* phi, double* grad) {
  const int L = sh_L(code);
  double dx = r[0] - R[0], dy = r[1] - R[1], dz = r[2] - R[2];
  double r2 = dx * dx + dy * dy + dz * dz;
  double R0 = 0.0, R1 = 0.0;
  for (int k = 0; k < nprim; ++k) {
    double e = d[k] * std::exp(-alpha[k] * r2);
    R0 += e;
    R1 += -2.0 * alpha[k] * e;
  }
  int c = 0;
  for (int l = L; l >= 0; --l)
    for (int m = L - l; m >= 0; --m) {
      int n = L - l - m;
      double mono = ipow(dx, l) * ipow(dy, m) * ipow(dz, n);
      phi[c] = mono * R0;
      if (grad) {
        // d/dx [dx^l dy^m dz^n R0(r^2)] = l dx^(l-1) dy^m dz^n R0 + dx^(l+1) dy^m dz^n R1   (A18)
        grad[3 * c + 0] = (l ? l * ipow(dx, l - 1) * ipow(dy, m) * ipow(dz, n) * R0 : 0.0) + dx * mono * R1;
        grad[3 * c + 1] = (m ? m * ipow(dx, l) * ipow(dy, m - 1) * ipow(dz, n) * R0 : 0.0) + dy * mono * R1;
        grad[3 * c + 2] = (n ? n * ipow(dx, l) * ipow(dy, m) * ipow(dz, n - 1) * R0 : 0.0) + dz * mono * R1;
      }
      ++c;
    }
  if (sh_pure(code)) {
    // Pure d shell (A19): the five real solid harmonics of degree 2, m = -2 .. 2, as combinations of the Cartesian
    // functions xx, xy, xz, yy, yz, zz (which share one radial part whose xx component has unit norm, A6):
    //   d(-2) = sqrt3 xy,  d(-1) = sqrt3 yz,  d(0) = zz - (xx + yy)/2,  d(+1) = sqrt3 xz,  d(+2) = (sqrt3/2)(xx - yy).
    // Each has unit norm and they are mutually orthogonal (pinned by the overlap and Unsold tests).
    const double s3 = std::sqrt(3.0);
    const int nv = grad ? 4 : 1;
    for (int v = 0; v < nv; ++v) {   // v = 0: values, 1..3: x, y, z derivatives (the transformation is linear)
      double cart[6], pure[5];
      for (int q = 0; q < 6; ++q) cart[q] = v == 0 ? phi[q] : grad[3 * q + v - 1];
      pure[0] = s3 * cart[1];
      pure[1] = s3 * cart[4];
      pure[2] = cart[5] - 0.5 * (cart[0] + cart[3]);
      pure[3] = s3 * cart[2];
      pure[4] = 0.5 * s3 * (cart[0] - cart[3]);
      for (int q = 0; q < 5; ++q) {
        if (v == 0) phi[q] = pure[q];
        else grad[3 * q + v - 1] = pure[q];
      }
    }
  }
}


// =============================================================================================================
// Spin-unrestricted densities and the meta-GGA intermediate tau ("may be
// extended to both spin-unrestricted ... as well as ... the meta-GGA with the addition of only a few intermediates").
// DESIGN.md readings A20-A22.  Variables: rho_a, rho_b, s_aa = |grad rho_a|^2, s_ab = grad rho_a . grad rho_b,
// s_bb = |grad rho_b|^2.  f = energy per unit volume; the five partial derivatives come from forward-mode duals.
// =============================================================================================================
struct D5 {
  double v;
  double d[5];
};
inline D5 mk5(double v) { return {v, {0, 0, 0, 0, 0}}; }
inline D5 var5(double v, int k) { D5 r = mk5(v); r.d[k] = 1.0; return r; }
inline D5 lin5(const D5& x, double fv, double fp) {   // g(x) with value fv and derivative fp at x.v
  D5 r; r.v = fv;
  for (int k = 0; k < 5; ++k) r.d[k] = fp * x.d[k];
  return r;
}
inline D5 operator+(D5 x, D5 y) { D5 r; r.v = x.v + y.v; for (int k = 0; k < 5; ++k) r.d[k] = x.d[k] + y.d[k]; return r; }
inline D5 operator-(D5 x, D5 y) { D5 r; r.v = x.v - y.v; for (int k = 0; k < 5; ++k) r.d[k] = x.d[k] - y.d[k]; return r; }
inline D5 operator-(D5 x) { D5 r; r.v = -x.v; for (int k = 0; k < 5; ++k) r.d[k] = -x.d[k]; return r; }
inline D5 operator*(D5 x, D5 y) { D5 r; r.v = x.v * y.v; for (int k = 0; k < 5; ++k) r.d[k] = x.d[k] * y.v + x.v * y.d[k]; return r; }
inline D5 operator/(D5 x, D5 y) {
  D5 r; r.v = x.v / y.v;
  for (int k = 0; k < 5; ++k) r.d[k] = (x.d[k] - r.v * y.d[k]) / y.v;
  return r;
}
inline D5 operator+(D5 x, double c) { x.v += c; return x; }
inline D5 operator+(double c, D5 x) { x.v += c; return x; }
inline D5 operator-(D5 x, double c) { x.v -= c; return x; }
inline D5 operator-(double c, D5 x) { return mk5(c) - x; }
inline D5 operator*(D5 x, double c) { x.v *= c; for (int k = 0; k < 5; ++k) x.d[k] *= c; return x; }
inline D5 operator*(double c, D5 x) { return x * c; }
inline D5 operator/(D5 x, double c) { return x * (1.0 / c); }
inline D5 operator/(double c, D5 x) { return mk5(c) / x; }
inline D5 dlog(D5 x) { return lin5(x, std::log(x.v), 1.0 / x.v); }
inline D5 dexp(D5 x) { double e = std::exp(x.v); return lin5(x, e, e); }
inline D5 datan(D5 x) { return lin5(x, std::atan(x.v), 1.0 / (1.0 + x.v * x.v)); }
inline D5 dsqrt(D5 x) { double s = std::sqrt(x.v); return lin5(x, s, 0.5 / s); }
inline D5 dcbrt(D5 x) { double c = std::cbrt(x.v); return lin5(x, c, c / (3.0 * x.v)); }
inline D5 dpow(D5 x, double p) { double w = std::pow(x.v, p); return lin5(x, w, p * w / x.v); }   // x.v > 0

// f(zeta) = ((1+z)^(4/3) + (1-z)^(4/3) - 2) / (2^(4/3) - 2) and f''(0) = 4 / (9 (2^(1/3) - 1))   (von Barth-Hedin form)
inline D5 f_zeta(D5 z) { return (dpow(1.0 + z, 4.0 / 3.0) + dpow(1.0 - z, 4.0 / 3.0) - 2.0) / (std::pow(2.0, 4.0 / 3.0) - 2.0); }
const double kFpp0 = 4.0 / (9.0 * (std::cbrt(2.0) - 1.0));

// VWN 1980 fit "V" interpolation G(x; A, x0, b, c), x = sqrt(r_s): paramagnetic, ferromagnetic and spin-stiffness sets
inline D5 vwn_G(D5 x, double A, double x0, double b, double c) {
  const double Q = std::sqrt(4.0 * c - b * b);
  const double X0 = x0 * x0 + b * x0 + c;
  D5 X = x * x + b * x + c;
  D5 at = datan(Q / (2.0 * x + b));
  return A * (dlog(x * x / X) + (2.0 * b / Q) * at - (b * x0 / X0) * (dlog((x - x0) * (x - x0) / X) + (2.0 * (b + 2.0 * x0) / Q) * at));
}
// Slater exchange, spin-scaled: E_x[ra, rb] = (E_x[2 ra] + E_x[2 rb]) / 2
inline D5 f_slater_pol(D5 ra, D5 rb) { return -kCx * 0.5 * (2.0 * ra * dcbrt(2.0 * ra) + 2.0 * rb * dcbrt(2.0 * rb)); }
// VWN5 correlation energy per particle at (r_s, zeta):
// eps = eps_P + alpha_c f(z)/f''(0) (1 - z^4) + (eps_F - eps_P) f(z) z^4
inline D5 eps_vwn5_pol(D5 rho, D5 zeta) {
  D5 x = dsqrt(dcbrt(mk5(3.0 / (4.0 * kPi)) / rho));
  D5 eP = vwn_G(x, 0.0310907, -0.10498, 3.72744, 12.9352);
  D5 eF = vwn_G(x, 0.01554535, -0.32500, 7.06042, 18.0578);
  D5 ac = vwn_G(x, -1.0 / (6.0 * kPi * kPi), -0.0047584, 1.13107, 13.0045);
  D5 fz = f_zeta(zeta), z4 = zeta * zeta * zeta * zeta;
  return eP + ac * (fz / kFpp0) * (1.0 - z4) + (eF - eP) * fz * z4;
}
// PW92 G(r_s; A, a1, b1..b4) and the interpolation in zeta (the third set fits -alpha_c)
inline D5 pw92_G(D5 r, double A, double a1, double b1, double b2, double b3, double b4) {
  D5 sr = dsqrt(r);
  D5 q = 2.0 * A * (b1 * sr + b2 * r + b3 * r * sr + b4 * r * r);
  return -2.0 * A * (1.0 + a1 * r) * dlog(1.0 + 1.0 / q);
}
inline D5 eps_pw92_pol(D5 rho, D5 zeta) {
  D5 r = dcbrt(mk5(3.0 / (4.0 * kPi)) / rho);
  D5 e0 = pw92_G(r, 0.0310907, 0.21370, 7.5957, 3.5876, 1.6382, 0.49294);
  D5 e1 = pw92_G(r, 0.01554535, 0.20548, 14.1189, 6.1977, 3.3662, 0.62517);
  D5 mac = pw92_G(r, 0.0168869, 0.11125, 10.357, 3.6231, 0.88026, 0.49671);   // = -alpha_c
  D5 fz = f_zeta(zeta), z4 = zeta * zeta * zeta * zeta;
  return e0 - mac * (fz / kFpp0) * (1.0 - z4) + (e1 - e0) * fz * z4;
}
// PBE exchange of one spin channel at density 2 r, sigma 4 s (spin scaling), per unit volume
inline D5 f_pbe_x_channel(D5 r2, D5 s4) {
  const double kappa = 0.804, mu = 0.2195149727645171;
  D5 s2 = s4 / (4.0 * std::pow(3.0 * kPi * kPi, 2.0 / 3.0) * dpow(r2, 8.0 / 3.0));
  D5 F = 1.0 + kappa - kappa / (1.0 + mu * s2 / kappa);
  return -kCx * r2 * dcbrt(r2) * F;
}
inline D5 f_pbe_x_pol(D5 ra, D5 rb, D5 saa, D5 sbb) {
  return 0.5 * (f_pbe_x_channel(2.0 * ra, 4.0 * saa) + f_pbe_x_channel(2.0 * rb, 4.0 * sbb));
}
// PBE correlation at (rho, zeta, sigma = |grad rho|^2): rho (eps_unif + H), phi = ((1+z)^(2/3) + (1-z)^(2/3)) / 2,
// t^2 = sigma / (4 phi^2 k_s^2 rho^2), A = (beta/gamma) / (exp(-eps/(gamma phi^3)) - 1)
inline D5 f_pbe_c_pol(D5 rho, D5 zeta, D5 sigma) {
  const double gamma = (1.0 - std::log(2.0)) / (kPi * kPi), beta = 0.06672455060314922;
  D5 eu = eps_pw92_pol(rho, zeta);
  D5 phi = 0.5 * (dpow(1.0 + zeta, 2.0 / 3.0) + dpow(1.0 - zeta, 2.0 / 3.0));
  D5 phi3 = phi * phi * phi;
  D5 kF = dcbrt(3.0 * kPi * kPi * rho);
  D5 ks2 = 4.0 * kF / kPi;
  D5 t2 = sigma / (4.0 * phi * phi * ks2 * rho * rho);
  D5 Ac = (beta / gamma) / (dexp(-eu / (gamma * phi3)) - 1.0);
  D5 At2 = Ac * t2;
  D5 H = gamma * phi3 * dlog(1.0 + (beta / gamma) * t2 * (1.0 + At2) / (1.0 + At2 + At2 * At2));
  return rho * (eu + H);
}
// kind: 0 = LDA Slater+VWN5, 1 = GGA PBE; pin kinds 2 = Slater, 3 = VWN5 (rho eps), 4 = PW92 (rho eps), 5 = PBE x, 6 = PBE c
inline D5 f_xc_pol(int kind, D5 ra, D5 rb, D5 saa, D5 sab, D5 sbb) {
  D5 rho = ra + rb, zeta = (ra - rb) / rho, sigma = saa + 2.0 * sab + sbb;
  switch (kind) {
    case 0: return f_slater_pol(ra, rb) + rho * eps_vwn5_pol(rho, zeta);
    case 1: return f_pbe_x_pol(ra, rb, saa, sbb) + f_pbe_c_pol(rho, zeta, sigma);
    case 2: return f_slater_pol(ra, rb);
    case 3: return rho * eps_vwn5_pol(rho, zeta);
    case 4: return rho * eps_pw92_pol(rho, zeta);
    case 5: return f_pbe_x_pol(ra, rb, saa, sbb);
    default: return f_pbe_c_pol(rho, zeta, sigma);
  }
}
// Reading A20: a point contributes nothing when rho_a + rho_b <= rho_tol; otherwise a spin density below rho_tol is
// raised to rho_tol before the functional is evaluated (zeta = +-1 is a singular point of the zeta interpolation), and
// the derivative with respect to it is the one at the raised value.
inline void eval_point_pol(int kind, double ra, double rb, double saa, double sab, double sbb, double rho_tol, double* f, double* v) {
  *f = 0.0;
  for (int k = 0; k < 5; ++k) v[k] = 0.0;
  if (ra + rb <= rho_tol) return;
  D5 r = f_xc_pol(kind, var5(std::max(ra, rho_tol), 0), var5(std::max(rb, rho_tol), 1), var5(saa, 2), var5(sab, 3), var5(sbb, 4));
  *f = r.v;
  for (int k = 0; k < 5; ++k) v[k] = r.d[k];
}


// ---- meta-GGA (reading A23): f(rho, sigma, tau), restricted -----------------
// Exchange "MS0" (Sun, Xiao, Ruzsinszky 2012): F_x = F1(p) + f(alpha) (F0(p) - F1(p)),
//   F_int(p; c) = 1 + kappa - kappa / (1 + (mu_GE p + c)/kappa),  F1 = F_int(p; 0),  F0 = F_int(p; c),
//   f(alpha) = (1 - alpha^2)^3 / (1 + alpha^3 + b alpha^6),  p = s^2 = sigma / (4 (3 pi^2)^(2/3) rho^(8/3)),
//   alpha = (tau - tau_W) / tau_unif,  tau_W = sigma / (8 rho),  tau_unif = (3/10) (3 pi^2)^(2/3) rho^(5/3),
//   kappa = 0.29, c = 0.28771, b = 1, mu_GE = 10/81;  f_x = -C_x rho^(4/3) F_x.
// Correlation: PBE (the unpolarised limit of f_pbe_c_pol).  D5 slots: 0 = rho, 1 = sigma, 2 = tau.
inline D5 f_ms0_x(D5 rho, D5 sigma, D5 tau) {
  const double kappa = 0.29, c = 0.28771, b = 1.0, muGE = 10.0 / 81.0;
  const double k23 = std::pow(3.0 * kPi * kPi, 2.0 / 3.0);
  D5 p = sigma / (4.0 * k23 * dpow(rho, 8.0 / 3.0));
  D5 tauW = sigma / (8.0 * rho);
  D5 tauU = 0.3 * k23 * dpow(rho, 5.0 / 3.0);
  D5 al = (tau - tauW) / tauU;
  D5 F1 = 1.0 + kappa - kappa / (1.0 + muGE * p / kappa);
  D5 F0 = 1.0 + kappa - kappa / (1.0 + (muGE * p + c) / kappa);
  D5 a2 = al * al, a3 = a2 * al;
  D5 om = 1.0 - a2;
  D5 fa = om * om * om / (1.0 + a3 + b * a3 * a3);
  return -kCx * rho * dcbrt(rho) * (F1 + fa * (F0 - F1));
}
// kind 7 = MS0 exchange + PBE correlation, 8 = MS0 exchange alone (pins)
inline bool is_mgga(int kind) { return kind == 7 || kind == 8; }
inline void eval_point_mgga(int kind, double rho, double sigma, double tau, double rho_tol, double* f, double* v3) {
  *f = 0.0; v3[0] = v3[1] = v3[2] = 0.0;
  if (!(rho > rho_tol)) return;
  D5 r = var5(rho, 0), s = var5(sigma, 1), t = var5(tau, 2);
  D5 e = f_ms0_x(r, s, t);
  if (kind == 7) e = e + f_pbe_c_pol(r, mk5(0.0), s);
  *f = e.v; v3[0] = e.d[0]; v3[1] = e.d[1]; v3[2] = e.d[2];
}

}  // namespace

extern "C" {

int orc_num_threads() {
#ifdef _OPENMP
  return omp_get_max_threads();
#else
  return 1;
#endif
}

// O1 Mura-Knowles radial rule, m = 3 (A3): x_i = i/(n+1), r = -alpha ln(1 - x^3),
// w = r^2 dr/dx /(n+1), dr/dx = 3 alpha x^2/(1 - x^3).
void orc_radial_mk(int n_rad, double alpha, double* r, double* w) {
  for (int i = 1; i <= n_rad; ++i) {
    double x = (double)i / (double)(n_rad + 1);
    double x3 = x * x * x;
    double ri = -alpha * std::log(1.0 - x3);
    r[i - 1] = ri;
    w[i - 1] = ri * ri * (3.0 * alpha * x * x / (1.0 - x3)) / (double)(n_rad + 1);
  }
}

// O2 angular rules (A4).  kind 0: Fibonacci sphere, equal weights 4 pi/n.
// kind 1: Gauss-Legendre(cos theta, n_theta nodes) x trapezoid(phi, 2 n_theta nodes), n_ang = 2 n_theta^2.
int orc_angular(int kind, int n_ang, double* u, double* w) {
  if (kind == 0) {
    const double golden = kPi * (3.0 - std::sqrt(5.0));
    for (int k = 0; k < n_ang; ++k) {
      double z = 1.0 - (2.0 * k + 1.0) / (double)n_ang;
      double s = std::sqrt(1.0 - z * z);
      double ph = k * golden;
      u[3 * k + 0] = s * std::cos(ph);
      u[3 * k + 1] = s * std::sin(ph);
      u[3 * k + 2] = z;
      w[k] = 4.0 * kPi / (double)n_ang;
    }
    return 0;
  }
  if (kind == 1) {
    int nt = (int)std::lround(std::sqrt(n_ang / 2.0));
    if (2 * nt * nt != n_ang) return -1;
    // Gauss-Legendre nodes by Newton iteration on P_nt
    std::vector<double> x(nt), gw(nt);
    for (int i = 0; i < nt; ++i) {
      double z = std::cos(kPi * (i + 0.75) / (nt + 0.5));
      double pp = 0.0;
      for (int it = 0; it < 100; ++it) {
        double p0 = 1.0, p1 = z;
        for (int k = 2; k <= nt; ++k) {
          double p2 = ((2.0 * k - 1.0) * z * p1 - (k - 1.0) * p0) / k;
          p0 = p1; p1 = p2;
        }
        if (nt == 1) { p0 = 1.0; p1 = z; }
        pp = nt * (z * p1 - p0) / (z * z - 1.0);
        double dz = p1 / pp;
        z -= dz;
        if (std::fabs(dz) < 1e-16) break;
      }
      // recompute derivative at converged node
      double p0 = 1.0, p1 = z;
      for (int k = 2; k <= nt; ++k) {
        double p2 = ((2.0 * k - 1.0) * z * p1 - (k - 1.0) * p0) / k;
        p0 = p1; p1 = p2;
      }
      pp = nt * (z * p1 - p0) / (z * z - 1.0);
      x[i] = z;
      gw[i] = 2.0 / ((1.0 - z * z) * pp * pp);
    }
    int k = 0;
    for (int i = 0; i < nt; ++i)
      for (int m = 0; m < 2 * nt; ++m) {
        double ph = (m + 0.5) * kPi / nt;
        double s = std::sqrt(1.0 - x[i] * x[i]);
        u[3 * k + 0] = s * std::cos(ph);
        u[3 * k + 1] = s * std::sin(ph);
        u[3 * k + 2] = x[i];
        w[k] = gw[i] * kPi / nt;
        ++k;
      }
    return 0;
  }
  return -1;
}

// O3 (Eq. (9)): r = R_A + r_i u_k, w^q = w_i^rad w_k^ang, parent A.
// Order: atom-major, then radial, then angular.
int orc_build_grid(int natoms, const double* xyz, int n_rad, int n_ang, int angular_kind, double mk_alpha,
                   double* pts, double* wq, int32_t* parent) {
  std::vector<double> r(n_rad), wr(n_rad), u(3 * (size_t)n_ang), wa(n_ang);
  orc_radial_mk(n_rad, mk_alpha, r.data(), wr.data());
  if (orc_angular(angular_kind, n_ang, u.data(), wa.data())) return -1;
  size_t p = 0;
  for (int A = 0; A < natoms; ++A)
    for (int i = 0; i < n_rad; ++i)
      for (int k = 0; k < n_ang; ++k) {
        for (int c = 0; c < 3; ++c) pts[3 * p + c] = xyz[3 * A + c] + r[i] * u[3 * k + c];
        wq[p] = wr[i] * wa[k];
        parent[p] = A;
        ++p;
      }
  return 0;
}

// O4 (Eqs. (8),(9); L107): w_i = w_i^q P_A(r_i)/sum_B P_B(r_i),
// P_B = prod_{C != B} s(mu_BC), mu_BC = (|r-R_B| - |r-R_C|)/|R_B-R_C|.
// kind 0 = SSF, 1 = Becke-88.  prune = 1 uses the exact SSF compact-support pruning (DESIGN.md,
// "SSF pruning"): P_B = 0 if r_B >= kappa r_min, and s(mu_BC) = 1 if r_C >= kappa r_B,
// kappa = (1+a)/(1-a); pinned against prune = 0 by tests (P5).  prune is ignored for Becke-88.
void orc_partition_weights(int natoms, const double* xyz, int64_t npts, const double* pts, const double* wq,
                           const int32_t* parent, int kind, int prune, double* w_out) {
  const double a = 0.64, kappa = (1.0 + a) / (1.0 - a);
  std::vector<double> RAB((size_t)natoms * natoms);
  for (int A = 0; A < natoms; ++A)
    for (int B = 0; B < natoms; ++B) RAB[(size_t)A * natoms + B] = dist3(xyz + 3 * A, xyz + 3 * B);
#pragma omp parallel
  {
    std::vector<double> rr(natoms);
#pragma omp for schedule(dynamic, 256)
    for (int64_t i = 0; i < npts; ++i) {
      double rmin = 1e300;
      for (int B = 0; B < natoms; ++B) {
        rr[B] = dist3(pts + 3 * i, xyz + 3 * B);
        rmin = std::min(rmin, rr[B]);
      }
      double sum = 0.0, PA = 0.0;
      for (int B = 0; B < natoms; ++B) {
        double PB = 1.0;
        if (kind == 0 && prune && rr[B] >= kappa * rmin && natoms > 1 && rr[B] > rmin) {
          PB = 0.0;
        } else {
          for (int C = 0; C < natoms; ++C) {
            if (C == B) continue;
            if (kind == 0 && prune && rr[C] >= kappa * rr[B]) continue;  // factor is exactly 1
            double mu = (rr[B] - rr[C]) / RAB[(size_t)B * natoms + C];
            PB *= (kind == 0) ? s_ssf(mu) : s_becke(mu);
            if (PB == 0.0) break;
          }
        }
        sum += PB;
        if (B == parent[i]) PA = PB;
      }
      w_out[i] = wq[i] * PA / sum;
    }
  }
}

// O5 (Eq. (10)): rcut = max_xi sqrt((ln(alpha)/2 - ln(eta))/alpha)
void orc_rcut(int nshells, const int32_t* shell_nprim, const int32_t* shell_prim_off, const double* exps, double eta,
              double* rcut) {
  for (int s = 0; s < nshells; ++s) {
    double m = 0.0;
    for (int k = 0; k < shell_nprim[s]; ++k) {
      double al = exps[shell_prim_off[s] + k];
      double v = (0.5 * std::log(al) - std::log(eta)) / al;
      if (v > 0.0) m = std::max(m, std::sqrt(v));
    }
    rcut[s] = m;
  }
}

// Alg. 1 exposed for tests.
int orc_cuboid_sphere(const double* R, double rcut, const double* V, const double* W) {
  return cuboid_sphere_intersect(R, rcut, V, W) ? 1 : 0;
}

// Shell list of one batch: S_j = shells whose cutoff sphere meets the tight bounding box of the
// batch's points (Alg. 3 l.3.7; reading A8).  Returns count; list ascending.
static int screen_batch(int nshells, const int32_t* shell_atom, const double* xyz, const double* rcut,
                        const double* pts, const int64_t* idx, int64_t n, int32_t* out) {
  double V[3] = {1e300, 1e300, 1e300}, W[3] = {-1e300, -1e300, -1e300};
  for (int64_t q = 0; q < n; ++q) {
    const double* p = pts + 3 * (idx ? idx[q] : q);
    for (int c = 0; c < 3; ++c) {
      V[c] = std::min(V[c], p[c]);
      W[c] = std::max(W[c], p[c]);
    }
  }
  int cnt = 0;
  for (int s = 0; s < nshells; ++s)
    if (cuboid_sphere_intersect(xyz + 3 * shell_atom[s], rcut[s], V, W)) out[cnt++] = s;
  return cnt;
}

// O6: the paper's literal batching (Fig. 1; Alg. 3 l.3.5-3.7; reading A8).
// Per atom: cube of half-side r_max (largest radial node) centred on R_A; a cuboid with <= max_pts
// points is emitted; otherwise it is split 3x3x3 if the closed cuboid holds an atomic centre, else
// 2x2x2 (equal splits; half-open cells, the last one closed); empty cells are dropped.
// Outputs (caller allocates: perm npts, batch_off npts+1, shell_off npts+1, shells cap):
//   perm[k] = index (into pts) of the k-th point in batch-contiguous order.
// Returns number of batches, or -1 if the shell-list capacity is too small.
struct PaperPlanCtx {
  int natoms; const double* xyz; const double* pts; int max_pts;
  std::vector<int64_t>* perm; std::vector<int64_t>* batch_off;
};
static void split_cuboid(PaperPlanCtx& c, std::vector<int64_t>& idx, const double* lo, const double* hi, int depth) {
  if (idx.empty()) return;
  if ((int64_t)idx.size() <= c.max_pts || depth > 40) {
    for (int64_t i : idx) c.perm->push_back(i);
    c.batch_off->push_back((int64_t)c.perm->size());
    return;
  }
  bool has_centre = false;
  for (int A = 0; A < c.natoms && !has_centre; ++A) {
    const double* R = c.xyz + 3 * A;
    has_centre = R[0] >= lo[0] && R[0] <= hi[0] && R[1] >= lo[1] && R[1] <= hi[1] && R[2] >= lo[2] && R[2] <= hi[2];
  }
  int ns = has_centre ? 3 : 2;
  std::vector<std::vector<int64_t>> cells((size_t)ns * ns * ns);
  for (int64_t i : idx) {
    int cell[3];
    for (int p = 0; p < 3; ++p) {
      double t = (c.pts[3 * i + p] - lo[p]) / (hi[p] - lo[p]) * ns;
      int k = (int)std::floor(t);
      if (k < 0) k = 0;
      if (k >= ns) k = ns - 1;  // last cell closed
      cell[p] = k;
    }
    cells[((size_t)cell[0] * ns + cell[1]) * ns + cell[2]].push_back(i);
  }
  std::vector<int64_t>().swap(idx);
  for (int a = 0; a < ns; ++a)
    for (int b = 0; b < ns; ++b)
      for (int d = 0; d < ns; ++d) {
        int k[3] = {a, b, d};
        double l2[3], h2[3];
        for (int p = 0; p < 3; ++p) {
          l2[p] = lo[p] + (hi[p] - lo[p]) * k[p] / ns;
          h2[p] = lo[p] + (hi[p] - lo[p]) * (k[p] + 1) / ns;
        }
        split_cuboid(c, cells[((size_t)a * ns + b) * ns + d], l2, h2, depth + 1);
      }
}

int64_t orc_plan_paper(int natoms, const double* xyz, int64_t npts, const double* pts, const int32_t* parent,
                       int max_pts, int nshells, const int32_t* shell_atom, const double* rcut, int64_t* perm,
                       int64_t* batch_off, int64_t* shell_off, int32_t* shells, int64_t shells_cap) {
  std::vector<int64_t> vperm, voff;
  vperm.reserve(npts);
  voff.push_back(0);
  PaperPlanCtx c{natoms, xyz, pts, max_pts, &vperm, &voff};
  // points are atom-major (O3): gather each atom's points
  std::vector<std::vector<int64_t>> by_atom(natoms);
  for (int64_t i = 0; i < npts; ++i) by_atom[parent[i]].push_back(i);
  for (int A = 0; A < natoms; ++A) {
    double rmax = 0.0;
    for (int64_t i : by_atom[A]) rmax = std::max(rmax, dist3(pts + 3 * i, xyz + 3 * A));
    double lo[3], hi[3];
    for (int p = 0; p < 3; ++p) {
      lo[p] = xyz[3 * A + p] - rmax;
      hi[p] = xyz[3 * A + p] + rmax;
    }
    split_cuboid(c, by_atom[A], lo, hi, 0);
  }
  int64_t nb = (int64_t)voff.size() - 1;
  std::copy(vperm.begin(), vperm.end(), perm);
  std::copy(voff.begin(), voff.end(), batch_off);
  // screening per batch (tight bounding box)
  std::vector<int64_t> cnt(nb);
  std::vector<std::vector<int32_t>> lists(nb);
#pragma omp parallel for schedule(dynamic, 16)
  for (int64_t j = 0; j < nb; ++j) {
    std::vector<int32_t> tmp(nshells);
    int n = screen_batch(nshells, shell_atom, xyz, rcut, pts, perm + batch_off[j], batch_off[j + 1] - batch_off[j],
                         tmp.data());
    lists[j].assign(tmp.begin(), tmp.begin() + n);
  }
  int64_t tot = 0;
  shell_off[0] = 0;
  for (int64_t j = 0; j < nb; ++j) {
    if (tot + (int64_t)lists[j].size() > shells_cap) return -1;
    std::copy(lists[j].begin(), lists[j].end(), shells + tot);
    tot += (int64_t)lists[j].size();
    shell_off[j + 1] = tot;
  }
  return nb;
}

// P9: validate ANY plan (the oracle's or one exported by the CUDA library) against the three rules
// of reading A8: (1) Eq. (11): batches partition Q -- here: points are given in
// batch-contiguous order and `orig` maps each to its index in the canonical O3 grid, which must be a
// permutation; (2) every batch has 1..max_pts points; (3) S_j contains every shell whose cutoff
// sphere meets the batch's tight bounding box (Alg. 1), is strictly ascending and in range.
// Returns 0 if valid, else a positive code (1: not a permutation, 2: batch size, 3: shell list order,
// 4: missing shell, 5: offsets).
int orc_validate_plan(int64_t npts, const double* pts_plan, const int64_t* orig, int64_t nbatch,
                      const int64_t* batch_off, const int64_t* shell_off, const int32_t* shells, int max_pts,
                      int natoms, const double* xyz, int nshells, const int32_t* shell_atom, const double* rcut) {
  (void)natoms;
  if (batch_off[0] != 0 || batch_off[nbatch] != npts || shell_off[0] != 0) return 5;
  if (orig) {
    std::vector<char> seen(npts, 0);
    for (int64_t k = 0; k < npts; ++k) {
      if (orig[k] < 0 || orig[k] >= npts || seen[orig[k]]) return 1;
      seen[orig[k]] = 1;
    }
  }
  int bad = 0;
#pragma omp parallel for schedule(dynamic, 16)
  for (int64_t j = 0; j < nbatch; ++j) {
    int64_t n = batch_off[j + 1] - batch_off[j];
    if (n < 1 || n > max_pts) {
#pragma omp critical
      bad = std::max(bad, 2);
      continue;
    }
    std::vector<int32_t> need(nshells);
    int nn = screen_batch(nshells, shell_atom, xyz, rcut, pts_plan + 3 * batch_off[j], nullptr, n, need.data());
    const int32_t* L = shells + shell_off[j];
    int64_t nl = shell_off[j + 1] - shell_off[j];
    int err = 0;
    for (int64_t k = 0; k < nl; ++k)
      if (L[k] < 0 || L[k] >= nshells || (k && L[k] <= L[k - 1])) err = 3;
    if (!err) {
      int64_t k = 0;
      for (int q = 0; q < nn && !err; ++q) {
        while (k < nl && L[k] < need[q]) ++k;
        if (k >= nl || L[k] != need[q]) err = 4;
      }
    }
    if (err) {
#pragma omp critical
      bad = std::max(bad, err);
    }
  }
  return bad;
}

// O7 exposed: collocation of a shell list at a point list.  phi[f*npts + i]; grad (may be null)
// gx,gy,gz each [nf*npts].  Returns number of functions.
int orc_collocation(int nsh, const int32_t* sh_list, const int32_t* shell_atom, const int32_t* shell_L,
                    const int32_t* shell_nprim, const int32_t* shell_prim_off, const double* exps,
                    const double* coefs, const double* xyz, int64_t npts, const double* pts, double* phi,
                    double* gx, double* gy, double* gz) {
  int nf = 0;
  for (int k = 0; k < nsh; ++k) nf += nfun(shell_L[sh_list[k]]);
  for (int64_t i = 0; i < npts; ++i) {
    int f = 0;
    for (int k = 0; k < nsh; ++k) {
      int s = sh_list[k];
      double ph[6], gr[18];
      shell_at_point(shell_L[s], shell_nprim[s], exps + shell_prim_off[s], coefs + shell_prim_off[s],
                     xyz + 3 * shell_atom[s], pts + 3 * i, ph, gx ? gr : nullptr);
      for (int c = 0; c < nfun(shell_L[s]); ++c, ++f) {
        phi[(size_t)f * npts + i] = ph[c];
        if (gx) {
          gx[(size_t)f * npts + i] = gr[3 * c + 0];
          gy[(size_t)f * npts + i] = gr[3 * c + 1];
          gz[(size_t)f * npts + i] = gr[3 * c + 2];
        }
      }
    }
  }
  return nf;
}

// O9 exposed: f, v_rho, v_sigma at n points.
void orc_functional(int kind, int64_t n, const double* rho, const double* sigma, double rho_tol, double* f,
                    double* vrho, double* vsigma) {
  for (int64_t i = 0; i < n; ++i) eval_point(kind, rho[i], sigma ? sigma[i] : 0.0, rho_tol, f + i, vrho + i, vsigma + i);
}

// O7-O12, Mode A (plan-conditioned; A9): Alg. 4 for the batches listed in
// `subset` (nsub entries; null = all batches), with the per-batch shell lists S_j given as data.
//   pts, w           points (batch-contiguous order) and FINAL weights w_i (after O4)
//   func_off[s]      first global function index of shell s
//   P                N_b x N_b, leading dimension ldp
//   V (may be null)  N_b x N_b (ld = nbasis), INCREMENTED (caller zeroes)
//   E_b, N_b_out     per-batch partial sums (size nbatch; entries of skipped batches untouched); may be null
//   rho_out, grho_out per-point rho (npts) and grad rho (3*npts), may be null
// Returns E_xc and N_el summed over the processed batches in batch order in long double.
void orc_eval(int64_t nbatch, const int64_t* batch_off, const int64_t* shell_off, const int32_t* shells,
              const int64_t* subset, int64_t nsub, const double* pts, const double* w, const int32_t* shell_atom,
              const int32_t* shell_L, const int32_t* shell_nprim, const int32_t* shell_prim_off,
              const int32_t* func_off, const double* exps, const double* coefs, const double* xyz, int nbasis,
              const double* P, int64_t ldp, int kind, double rho_tol, double* V, double* E_out, double* N_out,
              double* E_b, double* N_b_out, double* rho_out, double* grho_out) {
  const bool gga = is_gga(kind);
  int64_t njobs = subset ? nsub : nbatch;
  std::vector<long double> Eb(njobs, 0.0L), Nb(njobs, 0.0L);
#pragma omp parallel for schedule(dynamic, 1)
  for (int64_t job = 0; job < njobs; ++job) {
    int64_t j = subset ? subset[job] : job;
    int64_t q0 = batch_off[j], nq = batch_off[j + 1] - q0;
    const int32_t* S = shells + shell_off[j];
    int ns = (int)(shell_off[j + 1] - shell_off[j]);
    // S_j function index list
    std::vector<int> fidx;
    for (int k = 0; k < ns; ++k)
      for (int c = 0; c < nfun(shell_L[S[k]]); ++c) fidx.push_back(func_off[S[k]] + c);
    size_t nb = fidx.size();
    if (nb == 0 || nq == 0) continue;
    // O7: Phi^j (nb x nq) and gradients, Eq. (12a)
    std::vector<double> Phi(nb * nq), Gx, Gy, Gz;
    if (gga) { Gx.resize(nb * nq); Gy.resize(nb * nq); Gz.resize(nb * nq); }
    orc_collocation(ns, S, shell_atom, shell_L, shell_nprim, shell_prim_off, exps, coefs, xyz, nq, pts + 3 * q0,
                    Phi.data(), gga ? Gx.data() : nullptr, gga ? Gy.data() : nullptr, gga ? Gz.data() : nullptr);
    // Eq. (12b): P^j
    std::vector<double> Pj(nb * nb);
    for (size_t m = 0; m < nb; ++m)
      for (size_t n = 0; n < nb; ++n) Pj[m * nb + n] = P[(size_t)fidx[m] * ldp + fidx[n]];
    // Eq. (15): X^j = P^j Phi^j
    std::vector<double> X(nb * nq, 0.0);
    for (size_t m = 0; m < nb; ++m)
      for (size_t n = 0; n < nb; ++n) {
        double p = Pj[m * nb + n];
        const double* ph = &Phi[n * nq];
        double* x = &X[m * nq];
        for (int64_t i = 0; i < nq; ++i) x[i] += p * ph[i];
      }
    // Eqs. (13),(14) PAPER.md:L141-L144: rho_i = sum_mu Phi X ; grad rho_i = 2 sum_mu grad Phi X
    std::vector<double> rho(nq, 0.0), gx(nq, 0.0), gy(nq, 0.0), gz(nq, 0.0);
    for (size_t m = 0; m < nb; ++m)
      for (int64_t i = 0; i < nq; ++i) {
        rho[i] += Phi[m * nq + i] * X[m * nq + i];
        if (gga) {
          gx[i] += 2.0 * Gx[m * nq + i] * X[m * nq + i];
          gy[i] += 2.0 * Gy[m * nq + i] * X[m * nq + i];
          gz[i] += 2.0 * Gz[m * nq + i] * X[m * nq + i];
        }
      }
    // Eq. (19) PAPER.md:L159 (O9) and Eq. (16) PAPER.md:L150 (O10)
    std::vector<double> wvr(nq), wvs(nq);
    long double e = 0.0L, nel = 0.0L;
    for (int64_t i = 0; i < nq; ++i) {
      double sigma = gx[i] * gx[i] + gy[i] * gy[i] + gz[i] * gz[i];
      double f, vr, vs;
      eval_point(kind, rho[i], sigma, rho_tol, &f, &vr, &vs);
      wvr[i] = w[q0 + i] * vr;
      wvs[i] = w[q0 + i] * vs;
      e += (long double)w[q0 + i] * (long double)f;
      nel += (long double)w[q0 + i] * (long double)rho[i];
      if (rho_out) rho_out[q0 + i] = rho[i];
      if (grho_out) { grho_out[3 * (q0 + i) + 0] = gx[i]; grho_out[3 * (q0 + i) + 1] = gy[i]; grho_out[3 * (q0 + i) + 2] = gz[i]; }
    }
    Eb[job] = e;
    Nb[job] = nel;
    if (E_b) E_b[j] = (double)e;
    if (N_b_out) N_b_out[j] = (double)nel;
    if (!V) continue;
    // Eq. (20) PAPER.md:L162 (O11): Z = 1/2 (w v_rho) Phi + 2 (w v_sigma) grad rho . grad Phi
    std::vector<double> Z(nb * nq);
    for (size_t m = 0; m < nb; ++m)
      for (int64_t i = 0; i < nq; ++i) {
        double z = 0.5 * wvr[i] * Phi[m * nq + i];
        if (gga) z += 2.0 * wvs[i] * (gx[i] * Gx[m * nq + i] + gy[i] * Gy[m * nq + i] + gz[i] * Gz[m * nq + i]);
        Z[m * nq + i] = z;
      }
    // Eq. (18): V^j = Z Phi^T + Phi Z^T
    std::vector<double> Vj(nb * nb, 0.0);
    for (size_t m = 0; m < nb; ++m)
      for (size_t n = 0; n < nb; ++n) {
        double acc = 0.0;
        for (int64_t i = 0; i < nq; ++i) acc += Z[m * nq + i] * Phi[n * nq + i] + Phi[m * nq + i] * Z[n * nq + i];
        Vj[m * nb + n] = acc;
      }
    // Eq. (17) PAPER.md:L152, L168-L174 (O12): increment the blocks of V by V^j
#pragma omp critical(orc_v_increment)
    for (size_t m = 0; m < nb; ++m)
      for (size_t n = 0; n < nb; ++n) V[(size_t)fidx[m] * nbasis + fidx[n]] += Vj[m * nb + n];
  }
  long double E = 0.0L, N = 0.0L;
  for (int64_t job = 0; job < njobs; ++job) { E += Eb[job]; N += Nb[job]; }
  if (E_out) *E_out = (double)E;
  if (N_out) *N_out = (double)N;
}

// Mode B (A9; the plain definition of the quadrature sum, no screening): every shell at
// every point, rho_i = phi_i^T P phi_i,
// V = sum_i [ (w v_rho)_i phi_i phi_i^T + 2 (w v_sigma)_i (phi_i (grad rho_i . grad phi_i)^T + (...) phi_i^T) ].
void orc_eval_unscreened(int64_t npts, const double* pts, const double* w, int nshells, const int32_t* shell_atom,
                         const int32_t* shell_L, const int32_t* shell_nprim, const int32_t* shell_prim_off,
                         const double* exps, const double* coefs, const double* xyz, int nbasis, const double* P,
                         int64_t ldp, int kind, double rho_tol, double* V, double* E_out, double* N_out) {
  const bool gga = is_gga(kind);
  int nthr = orc_num_threads();
  std::vector<std::vector<double>> Vt(nthr);
  std::vector<long double> Et(nthr, 0.0L), Nt(nthr, 0.0L);
#pragma omp parallel
  {
#ifdef _OPENMP
    int tid = omp_get_thread_num();
#else
    int tid = 0;
#endif
    std::vector<double>& Vl = Vt[tid];
    if (V) Vl.assign((size_t)nbasis * nbasis, 0.0);
    std::vector<double> phi(nbasis), g(3 * (size_t)nbasis), x(nbasis), z(nbasis);
    long double e = 0.0L, nel = 0.0L;
#pragma omp for schedule(static)
    for (int64_t i = 0; i < npts; ++i) {
      int f = 0;
      for (int s = 0; s < nshells; ++s) {
        shell_at_point(shell_L[s], shell_nprim[s], exps + shell_prim_off[s], coefs + shell_prim_off[s],
                       xyz + 3 * shell_atom[s], pts + 3 * i, &phi[f], &g[3 * f]);
        f += nfun(shell_L[s]);
      }
      double rho = 0.0, gr[3] = {0.0, 0.0, 0.0};
      for (int m = 0; m < nbasis; ++m) {
        double xm = 0.0;
        for (int n = 0; n < nbasis; ++n) xm += P[(size_t)m * ldp + n] * phi[n];
        x[m] = xm;
        rho += phi[m] * xm;
        for (int c = 0; c < 3; ++c) gr[c] += 2.0 * g[3 * m + c] * xm;
      }
      double sigma = gr[0] * gr[0] + gr[1] * gr[1] + gr[2] * gr[2];
      double fv, vr, vs;
      eval_point(kind, rho, gga ? sigma : 0.0, rho_tol, &fv, &vr, &vs);
      e += (long double)w[i] * (long double)fv;
      nel += (long double)w[i] * (long double)rho;
      if (!V) continue;
      for (int m = 0; m < nbasis; ++m) {
        double zz = 0.5 * w[i] * vr * phi[m];
        if (gga) zz += 2.0 * w[i] * vs * (gr[0] * g[3 * m] + gr[1] * g[3 * m + 1] + gr[2] * g[3 * m + 2]);
        z[m] = zz;
      }
      for (int m = 0; m < nbasis; ++m)
        for (int n = 0; n < nbasis; ++n) Vl[(size_t)m * nbasis + n] += z[m] * phi[n] + phi[m] * z[n];
    }
    Et[tid] = e;
    Nt[tid] = nel;
  }
  long double E = 0.0L, N = 0.0L;
  for (int t = 0; t < nthr; ++t) {
    E += Et[t];
    N += Nt[t];
    if (V && !Vt[t].empty())
      for (size_t k = 0; k < (size_t)nbasis * nbasis; ++k) V[k] += Vt[t][k];
  }
  if (E_out) *E_out = (double)E;
  if (N_out) *N_out = (double)N;
}

// Work model of the paper, Eq. (22), and the contraction flop count used by bench.py
// for a plan: sum_j 4 (N_b^j)^2 N_q^j (X GEMM + SYR2K, each MAC = 2 flop).
double orc_plan_flops(int64_t nbatch, const int64_t* batch_off, const int64_t* shell_off, const int32_t* shells,
                      const int32_t* shell_L) {
  double tot = 0.0;
  for (int64_t j = 0; j < nbatch; ++j) {
    double nb = 0.0;
    for (int64_t k = shell_off[j]; k < shell_off[j + 1]; ++k) nb += nfun(shell_L[shells[k]]);
    tot += 4.0 * nb * nb * (double)(batch_off[j + 1] - batch_off[j]);
  }
  return tot;
}

// Spin-polarised functional exposed (A20): f and the five partials at n points.
void orc_functional_pol(int kind, int64_t n, const double* ra, const double* rb, const double* saa, const double* sab,
                        const double* sbb, double rho_tol, double* f, double* v5 /* [n][5]: d/d ra, rb, saa, sab, sbb */) {
  for (int64_t i = 0; i < n; ++i)
    eval_point_pol(kind, ra[i], rb[i], saa ? saa[i] : 0.0, sab ? sab[i] : 0.0, sbb ? sbb[i] : 0.0, rho_tol, f + i, v5 + 5 * i);
}

// Alg. 4, Mode A, for spin-unrestricted densities (readings A20-A22):
//   X^s = P^s,j Phi^j;  rho_s,i = sum_mu Phi X^s;  grad rho_s,i = 2 sum_mu grad Phi X^s          (Eqs. (13)-(15) per spin)
//   tau_s,i = 1/2 sum_mu grad Phi_mu,i . grad X^s_mu,i,  grad X^s = P^s,j grad Phi^j              (meta-GGA intermediate)
//   Z^s = 1/2 (w v_rho_s) Phi + w (2 v_s_ss grad rho_s + v_s_ab grad rho_s') . grad Phi;  V^s,j = Z^s Phi^T + Phi Z^s^T
// P_a, P_b: N_b x N_b (ld = ldp) with rho_s = sum P^s phi phi (no factor 2).  Va, Vb (may be null) are INCREMENTED.
// rho_out [2][npts], grho_out [2][npts][3], tau_out [2][npts] may be null.  N_out[2] = (N_a, N_b).
void orc_eval_uks(int64_t nbatch, const int64_t* batch_off, const int64_t* shell_off, const int32_t* shells,
                  const int64_t* subset, int64_t nsub, int64_t npts, const double* pts, const double* w, const int32_t* shell_atom,
                  const int32_t* shell_L, const int32_t* shell_nprim, const int32_t* shell_prim_off,
                  const int32_t* func_off, const double* exps, const double* coefs, const double* xyz, int nbasis,
                  const double* Pa, const double* Pb, int64_t ldp, int kind, double rho_tol, double* Va, double* Vb,
                  double* E_out, double* N_out, double* rho_out, double* grho_out, double* tau_out) {
  const bool gga = is_gga(kind);
  int64_t njobs = subset ? nsub : nbatch;
  std::vector<long double> Eb(njobs, 0.0L), Na(njobs, 0.0L), Nb(njobs, 0.0L);
#pragma omp parallel for schedule(dynamic, 1)
  for (int64_t job = 0; job < njobs; ++job) {
    int64_t j = subset ? subset[job] : job;
    int64_t q0 = batch_off[j], nq = batch_off[j + 1] - q0;
    const int32_t* S = shells + shell_off[j];
    int ns = (int)(shell_off[j + 1] - shell_off[j]);
    std::vector<int> fidx;
    for (int k = 0; k < ns; ++k)
      for (int c = 0; c < nfun(shell_L[S[k]]); ++c) fidx.push_back(func_off[S[k]] + c);
    size_t nb = fidx.size();
    if (nb == 0 || nq == 0) continue;
    const bool need_grad = gga || tau_out;
    std::vector<double> Phi(nb * nq), G[3];
    if (need_grad) for (int c = 0; c < 3; ++c) G[c].resize(nb * nq);
    orc_collocation(ns, S, shell_atom, shell_L, shell_nprim, shell_prim_off, exps, coefs, xyz, nq, pts + 3 * q0,
                    Phi.data(), need_grad ? G[0].data() : nullptr, need_grad ? G[1].data() : nullptr, need_grad ? G[2].data() : nullptr);
    // per spin: P^s,j, X^s, rho_s, grad rho_s, tau_s
    std::vector<double> rho[2], gr[2][3], tau[2];
    for (int s = 0; s < 2; ++s) {
      const double* P = s == 0 ? Pa : Pb;
      std::vector<double> X(nb * nq, 0.0);
      for (size_t m = 0; m < nb; ++m)
        for (size_t n = 0; n < nb; ++n) {
          double p = P[(size_t)fidx[m] * ldp + fidx[n]];
          for (int64_t i = 0; i < nq; ++i) X[m * nq + i] += p * Phi[n * nq + i];
        }
      rho[s].assign(nq, 0.0);
      for (int c = 0; c < 3; ++c) gr[s][c].assign(nq, 0.0);
      for (size_t m = 0; m < nb; ++m)
        for (int64_t i = 0; i < nq; ++i) {
          rho[s][i] += Phi[m * nq + i] * X[m * nq + i];
          if (need_grad)
            for (int c = 0; c < 3; ++c) gr[s][c][i] += 2.0 * G[c][m * nq + i] * X[m * nq + i];
        }
      if (tau_out) {
        tau[s].assign(nq, 0.0);
        for (int c = 0; c < 3; ++c) {
          std::vector<double> GX(nb * nq, 0.0);   // grad_c X^s = P^s,j grad_c Phi^j
          for (size_t m = 0; m < nb; ++m)
            for (size_t n = 0; n < nb; ++n) {
              double p = P[(size_t)fidx[m] * ldp + fidx[n]];
              for (int64_t i = 0; i < nq; ++i) GX[m * nq + i] += p * G[c][n * nq + i];
            }
          for (size_t m = 0; m < nb; ++m)
            for (int64_t i = 0; i < nq; ++i) tau[s][i] += 0.5 * G[c][m * nq + i] * GX[m * nq + i];
        }
      }
    }
    // functional (A20), energy and electron counts
    std::vector<double> a[2], gz[2][3];   // Z^s = a_s Phi + gz_s . grad Phi
    for (int s = 0; s < 2; ++s) { a[s].resize(nq); for (int c = 0; c < 3; ++c) gz[s][c].assign(nq, 0.0); }
    long double e = 0.0L, na = 0.0L, nbl = 0.0L;
    for (int64_t i = 0; i < nq; ++i) {
      double saa = 0.0, sab = 0.0, sbb = 0.0;
      if (gga)
        for (int c = 0; c < 3; ++c) { saa += gr[0][c][i] * gr[0][c][i]; sab += gr[0][c][i] * gr[1][c][i]; sbb += gr[1][c][i] * gr[1][c][i]; }
      double f, v[5];
      eval_point_pol(kind, rho[0][i], rho[1][i], saa, sab, sbb, rho_tol, &f, v);
      const double wi = w[q0 + i];
      a[0][i] = 0.5 * wi * v[0];
      a[1][i] = 0.5 * wi * v[1];
      if (gga)
        for (int c = 0; c < 3; ++c) {
          gz[0][c][i] = wi * (2.0 * v[2] * gr[0][c][i] + v[3] * gr[1][c][i]);
          gz[1][c][i] = wi * (2.0 * v[4] * gr[1][c][i] + v[3] * gr[0][c][i]);
        }
      e += (long double)wi * (long double)f;
      na += (long double)wi * (long double)rho[0][i];
      nbl += (long double)wi * (long double)rho[1][i];
      for (int s = 0; s < 2; ++s) {
        if (rho_out) rho_out[(size_t)s * npts + q0 + i] = rho[s][i];
        if (grho_out && need_grad) for (int c = 0; c < 3; ++c) grho_out[((size_t)s * npts + q0 + i) * 3 + c] = gr[s][c][i];
        if (tau_out) tau_out[(size_t)s * npts + q0 + i] = tau[s][i];
      }
    }
    Eb[job] = e; Na[job] = na; Nb[job] = nbl;
    for (int s = 0; s < 2; ++s) {
      double* V = s == 0 ? Va : Vb;
      if (!V) continue;
      std::vector<double> Z(nb * nq);
      for (size_t m = 0; m < nb; ++m)
        for (int64_t i = 0; i < nq; ++i) {
          double z = a[s][i] * Phi[m * nq + i];
          if (gga) for (int c = 0; c < 3; ++c) z += gz[s][c][i] * G[c][m * nq + i];
          Z[m * nq + i] = z;
        }
      std::vector<double> Vj(nb * nb, 0.0);
      for (size_t m = 0; m < nb; ++m)
        for (size_t n = 0; n < nb; ++n) {
          double acc = 0.0;
          for (int64_t i = 0; i < nq; ++i) acc += Z[m * nq + i] * Phi[n * nq + i] + Phi[m * nq + i] * Z[n * nq + i];
          Vj[m * nb + n] = acc;
        }
#pragma omp critical(orc_v_increment_uks)
      for (size_t m = 0; m < nb; ++m)
        for (size_t n = 0; n < nb; ++n) V[(size_t)fidx[m] * nbasis + fidx[n]] += Vj[m * nb + n];
    }
  }
  long double E = 0.0L, A = 0.0L, B = 0.0L;
  for (int64_t job = 0; job < njobs; ++job) { E += Eb[job]; A += Na[job]; B += Nb[job]; }
  if (E_out) *E_out = (double)E;
  if (N_out) { N_out[0] = (double)A; N_out[1] = (double)B; }
}

// meta-GGA functional exposed (A23): f and d f / d (rho, sigma, tau) at n points, v3 [n][3].
void orc_functional_mgga(int kind, int64_t n, const double* rho, const double* sigma, const double* tau, double rho_tol, double* f,
                         double* v3) {
  for (int64_t i = 0; i < n; ++i) eval_point_mgga(kind, rho[i], sigma[i], tau[i], rho_tol, f + i, v3 + 3 * i);
}

// Alg. 4, Mode A, for a restricted meta-GGA ("with the addition of only a few
// intermediates"; reading A23).  Besides Eqs. (13)-(15):
//   tau_i = 1/2 sum_mu grad Phi_mu,i . grad X_mu,i,   grad X = P^j grad Phi^j
//   Z = 1/2 (w v_rho) Phi + 2 (w v_sigma) grad rho . grad Phi                                   (Eq. (20))
//   V^j = Z Phi^T + Phi Z^T + sum_c 1/2 (w v_tau) (d_c Phi) (d_c Phi)^T                          (d tau / d P_mu,nu = 1/2 grad phi_mu . grad phi_nu)
// Arguments as orc_eval; tau_out (may be null) [npts].
void orc_eval_mgga(int64_t nbatch, const int64_t* batch_off, const int64_t* shell_off, const int32_t* shells,
                   const int64_t* subset, int64_t nsub, const double* pts, const double* w, const int32_t* shell_atom,
                   const int32_t* shell_L, const int32_t* shell_nprim, const int32_t* shell_prim_off,
                   const int32_t* func_off, const double* exps, const double* coefs, const double* xyz, int nbasis,
                   const double* P, int64_t ldp, int kind, double rho_tol, double* V, double* E_out, double* N_out,
                   double* E_b, double* N_b_out, double* rho_out, double* grho_out, double* tau_out) {
  int64_t njobs = subset ? nsub : nbatch;
  std::vector<long double> Eb(njobs, 0.0L), Nb(njobs, 0.0L);
#pragma omp parallel for schedule(dynamic, 1)
  for (int64_t job = 0; job < njobs; ++job) {
    int64_t j = subset ? subset[job] : job;
    int64_t q0 = batch_off[j], nq = batch_off[j + 1] - q0;
    const int32_t* S = shells + shell_off[j];
    int ns = (int)(shell_off[j + 1] - shell_off[j]);
    std::vector<int> fidx;
    for (int k = 0; k < ns; ++k)
      for (int c = 0; c < nfun(shell_L[S[k]]); ++c) fidx.push_back(func_off[S[k]] + c);
    size_t nb = fidx.size();
    if (nb == 0 || nq == 0) continue;
    std::vector<double> Phi(nb * nq), G[3];
    for (int c = 0; c < 3; ++c) G[c].resize(nb * nq);
    orc_collocation(ns, S, shell_atom, shell_L, shell_nprim, shell_prim_off, exps, coefs, xyz, nq, pts + 3 * q0, Phi.data(),
                    G[0].data(), G[1].data(), G[2].data());
    std::vector<double> Pj(nb * nb);
    for (size_t m = 0; m < nb; ++m)
      for (size_t n = 0; n < nb; ++n) Pj[m * nb + n] = P[(size_t)fidx[m] * ldp + fidx[n]];
    std::vector<double> X(nb * nq, 0.0);
    for (size_t m = 0; m < nb; ++m)
      for (size_t n = 0; n < nb; ++n)
        for (int64_t i = 0; i < nq; ++i) X[m * nq + i] += Pj[m * nb + n] * Phi[n * nq + i];
    std::vector<double> rho(nq, 0.0), gr[3], tau(nq, 0.0);
    for (int c = 0; c < 3; ++c) gr[c].assign(nq, 0.0);
    for (size_t m = 0; m < nb; ++m)
      for (int64_t i = 0; i < nq; ++i) {
        rho[i] += Phi[m * nq + i] * X[m * nq + i];
        for (int c = 0; c < 3; ++c) gr[c][i] += 2.0 * G[c][m * nq + i] * X[m * nq + i];
      }
    for (int c = 0; c < 3; ++c) {
      std::vector<double> GX(nb * nq, 0.0);
      for (size_t m = 0; m < nb; ++m)
        for (size_t n = 0; n < nb; ++n)
          for (int64_t i = 0; i < nq; ++i) GX[m * nq + i] += Pj[m * nb + n] * G[c][n * nq + i];
      for (size_t m = 0; m < nb; ++m)
        for (int64_t i = 0; i < nq; ++i) tau[i] += 0.5 * G[c][m * nq + i] * GX[m * nq + i];
    }
    std::vector<double> wvr(nq), wvs(nq), wvt(nq);
    long double e = 0.0L, nel = 0.0L;
    for (int64_t i = 0; i < nq; ++i) {
      double sigma = gr[0][i] * gr[0][i] + gr[1][i] * gr[1][i] + gr[2][i] * gr[2][i];
      double f, v[3];
      eval_point_mgga(kind, rho[i], sigma, tau[i], rho_tol, &f, v);
      wvr[i] = w[q0 + i] * v[0]; wvs[i] = w[q0 + i] * v[1]; wvt[i] = w[q0 + i] * v[2];
      e += (long double)w[q0 + i] * (long double)f;
      nel += (long double)w[q0 + i] * (long double)rho[i];
      if (rho_out) rho_out[q0 + i] = rho[i];
      if (grho_out) for (int c = 0; c < 3; ++c) grho_out[3 * (q0 + i) + c] = gr[c][i];
      if (tau_out) tau_out[q0 + i] = tau[i];
    }
    Eb[job] = e; Nb[job] = nel;
    if (E_b) E_b[j] = (double)e;
    if (N_b_out) N_b_out[j] = (double)nel;
    if (!V) continue;
    std::vector<double> Z(nb * nq);
    for (size_t m = 0; m < nb; ++m)
      for (int64_t i = 0; i < nq; ++i)
        Z[m * nq + i] = 0.5 * wvr[i] * Phi[m * nq + i] +
                        2.0 * wvs[i] * (gr[0][i] * G[0][m * nq + i] + gr[1][i] * G[1][m * nq + i] + gr[2][i] * G[2][m * nq + i]);
    std::vector<double> Vj(nb * nb, 0.0);
    for (size_t m = 0; m < nb; ++m)
      for (size_t n = 0; n < nb; ++n) {
        double acc = 0.0;
        for (int64_t i = 0; i < nq; ++i) {
          acc += Z[m * nq + i] * Phi[n * nq + i] + Phi[m * nq + i] * Z[n * nq + i];
          for (int c = 0; c < 3; ++c) acc += 0.5 * wvt[i] * G[c][m * nq + i] * G[c][n * nq + i];
        }
        Vj[m * nb + n] = acc;
      }
#pragma omp critical(orc_v_increment_mgga)
    for (size_t m = 0; m < nb; ++m)
      for (size_t n = 0; n < nb; ++n) V[(size_t)fidx[m] * nbasis + fidx[n]] += Vj[m * nb + n];
  }
  long double E = 0.0L, N = 0.0L;
  for (int64_t job = 0; job < njobs; ++job) { E += Eb[job]; N += Nb[job]; }
  if (E_out) *E_out = (double)E;
  if (N_out) *N_out = (double)N;
}

}  // extern "C"
