// xc_kernels.cu -- CUDA kernels (sm_100a) of libxc_b200: the hot path of Alg. 4.
//
//   k_weights   step (a)   partition weights, Eq. (9), Alg. 4 l.4.1
//   k_pack_P    step (d1) gather: P^j Eq. (12b), packed once per batch in DMMA fragment order
//   k_xc_batch  steps (c)-(g) fused, one CTA per batch: collocation Eq. (7)/(12a), X = P^j Phi^j Eq. (15),
//               rho / grad rho Eqs. (13),(14), functional Eq. (19), E/N Eq. (16), Z Eq. (20),
//               V^j = Z Phi^T + Phi Z^T Eq. (18) in registers, increment Eq. (17)
//   k_finalize  fixed point -> fp64, mirror to the full symmetric V
//
// The dense contractions run on the FP64 tensor path (mma.sync m8n8k4 f64 -> DMMA.8x8x4 SASS), which on
// B200 reaches the full FP64 rate (37.2 TFLOP/s measured) while leaving issue slots for the collocation
// and epilogue arithmetic; tcgen05 has no f64 kind.  (Product code; shares nothing with oracle/.)
#include <cuda_runtime.h>

#include <algorithm>
#include <cstdint>

#include "xc_internal.h"
#include "xc_kernels.h"

namespace xcb {

// Optional per-phase cycle counters of the batch kernel (thread 0 of every CTA; development builds only:
// compile with -DXC_PHASE_TIMING, read with xc_debug_phase).  Compiled out of the product library.
#ifdef XC_PHASE_TIMING
__device__ unsigned long long g_phase[16];
#define PH_DECL long long _pt = clock64();
#define PH(k) do { if (threadIdx.x == 0) { long long _n = clock64(); atomicAdd(&g_phase[k], (unsigned long long)(_n - _pt)); _pt = _n; } } while (0)
extern "C" void xc_debug_phase(unsigned long long* out, int reset) {
  if (reset) { unsigned long long z[16] = {0}; cudaMemcpyToSymbol(g_phase, z, sizeof(z)); }
  else { cudaDeviceSynchronize(); cudaMemcpyFromSymbol(out, g_phase, sizeof(unsigned long long) * 16); }
}
#else
#define PH_DECL
#define PH(k)
#endif

// ------------------------------------------------------------------------------------------------
// small device helpers
// ------------------------------------------------------------------------------------------------
__device__ __forceinline__ void dmma884(double& c0, double& c1, double a, double b) {
  asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};\n"
               : "+d"(c0), "+d"(c1)
               : "d"(a), "d"(b));
}
__device__ __forceinline__ double pw012(double v, int n) { return n == 0 ? 1.0 : (n == 1 ? v : v * v); }
__device__ __forceinline__ double dpw012(double v, int n) { return n == 0 ? 0.0 : (n == 1 ? 1.0 : 2.0 * v); }

// exp(-arg) for 0 <= arg < 708 (the result stays a normal number), <= 1 ulp: arg = -(n ln2/64 + r), n = 64 k + j,
// exp(-arg) = 2^k 2^(j/64) (1 + p(r)), |r| <= ln2/128, p of degree 5 in Estrin form.  The dependent FP64 chain is 9
// operations (the library exp: ~25), which is what the collocation stage waits on when the FP64 pipe is shared
// with another CTA's DMMAs.  tab = 2^(j/64), j = 0..63, correctly rounded (shared-memory copy of kExp2Tab).
__device__ const double kExp2Tab[64] = {
    0x1.0000000000000p+0, 0x1.02c9a3e778061p+0, 0x1.059b0d3158574p+0, 0x1.0874518759bc8p+0,
    0x1.0b5586cf9890fp+0, 0x1.0e3ec32d3d1a2p+0, 0x1.11301d0125b51p+0, 0x1.1429aaea92de0p+0,
    0x1.172b83c7d517bp+0, 0x1.1a35beb6fcb75p+0, 0x1.1d4873168b9aap+0, 0x1.2063b88628cd6p+0,
    0x1.2387a6e756238p+0, 0x1.26b4565e27cddp+0, 0x1.29e9df51fdee1p+0, 0x1.2d285a6e4030bp+0,
    0x1.306fe0a31b715p+0, 0x1.33c08b26416ffp+0, 0x1.371a7373aa9cbp+0, 0x1.3a7db34e59ff7p+0,
    0x1.3dea64c123422p+0, 0x1.4160a21f72e2ap+0, 0x1.44e086061892dp+0, 0x1.486a2b5c13cd0p+0,
    0x1.4bfdad5362a27p+0, 0x1.4f9b2769d2ca7p+0, 0x1.5342b569d4f82p+0, 0x1.56f4736b527dap+0,
    0x1.5ab07dd485429p+0, 0x1.5e76f15ad2148p+0, 0x1.6247eb03a5585p+0, 0x1.6623882552225p+0,
    0x1.6a09e667f3bcdp+0, 0x1.6dfb23c651a2fp+0, 0x1.71f75e8ec5f74p+0, 0x1.75feb564267c9p+0,
    0x1.7a11473eb0187p+0, 0x1.7e2f336cf4e62p+0, 0x1.82589994cce13p+0, 0x1.868d99b4492edp+0,
    0x1.8ace5422aa0dbp+0, 0x1.8f1ae99157736p+0, 0x1.93737b0cdc5e5p+0, 0x1.97d829fde4e50p+0,
    0x1.9c49182a3f090p+0, 0x1.a0c667b5de565p+0, 0x1.a5503b23e255dp+0, 0x1.a9e6b5579fdbfp+0,
    0x1.ae89f995ad3adp+0, 0x1.b33a2b84f15fbp+0, 0x1.b7f76f2fb5e47p+0, 0x1.bcc1e904bc1d2p+0,
    0x1.c199bdd85529cp+0, 0x1.c67f12e57d14bp+0, 0x1.cb720dcef9069p+0, 0x1.d072d4a07897cp+0,
    0x1.d5818dcfba487p+0, 0x1.da9e603db3285p+0, 0x1.dfc97337b9b5fp+0, 0x1.e502ee78b3ff6p+0,
    0x1.ea4afa2a490dap+0, 0x1.efa1bee615a27p+0, 0x1.f50765b6e4540p+0, 0x1.fa7c1819e90d8p+0};

__device__ __forceinline__ double exp_neg(double arg, const double* __restrict__ tab) {
  const double kMagic = 6755399441055744.0;                 // 1.5 * 2^52: the low word of (t + kMagic) is round(t)
  double kd = fma(arg, -92.332482616893656768, kMagic);     // -64 / ln2
  const int n = __double2loint(kd);
  kd -= kMagic;
  double r = fma(-kd, 0x1.62e42feep-7, -arg);               // ln2 / 64, high part (32 significant bits: exact product)
  r = fma(-kd, 0x1.a39ef358p-39, r);
  const double r2 = r * r;
  const double qa = fma(r, 1.0 / 6.0, 0.5), qb = fma(r, 1.0 / 120.0, 1.0 / 24.0);
  const double pr = fma(r2, fma(r2, qb, qa), r);
  const double tj = tab[n & 63];
  const double res = fma(tj, pr, tj);
  return __hiloint2double(__double2hiint(res) + ((n >> 6) << 20), __double2loint(res));
}

// gradient of  x^l y^m z^n R0(r^2)  given R1 = dR0/d(r^2) * 2  (i.e. d/dx R0 = x R1)
__device__ __forceinline__ void grad_cart(int info, double dx, double dy, double dz, double R0, double R1,
                                          double& gx, double& gy, double& gz) {
  int l = (info >> 4) & 3, m = (info >> 2) & 3, n = info & 3;
  double xl = pw012(dx, l), ym = pw012(dy, m), zn = pw012(dz, n);
  double mono = xl * ym * zn, mr1 = mono * R1;
  gx = fma(dpw012(dx, l) * ym * zn, R0, dx * mr1);
  gy = fma(xl * dpw012(dy, m) * zn, R0, dy * mr1);
  gz = fma(xl * ym * dpw012(dz, n), R0, dz * mr1);
}

// ------------------------------------------------------------------------------------------------
// XC functionals (spin-unpolarised), closed-form derivatives.  f = energy per unit volume,
// vr = df/drho, vs = df/dsigma, sigma = |grad rho|^2 (A10-A12).
// ------------------------------------------------------------------------------------------------
#define XC_PI 3.14159265358979323846264338327950288
#define XC_CX 0.7385587663820224058842300326808360  // (3/4)(3/pi)^(1/3)
#define XC_RSFAC 0.6203504908994000166680068120477781  // (3/(4 pi))^(1/3)

// The point functional is evaluated by ONE warp per tile while the other warps wait, so its dependent chain is kept
// short: one rcbrt and one rsqrt give every power of rho and r_s, and the reciprocals are merged (4 divisions each).
__device__ __forceinline__ void lda_slater_vwn5(double rho, double& f, double& vr) {
  const double A = 0.0310907, x0 = -0.10498, b = 3.72744, c = 12.9352;
  const double Q = 6.1519908197590802321728722658;         // sqrt(4c - b^2)
  const double Xx0 = x0 * x0 + b * x0 + c;
  const double bx0 = b * x0 / Xx0;
  const double ir13 = rcbrt(rho);
  const double r13 = rho * ir13 * ir13;
  const double rs = XC_RSFAC * ir13;
  const double isx = rsqrt(rs);
  const double x = rs * isx;                                // sqrt(r_s)
  const double X = fma(x, x + b, c);
  const double tb = 2.0 * x + b;
  const double xm = x - x0;
  const double iX = 1.0 / X, itb = 1.0 / tb, ixm = 1.0 / xm;
  const double at = atan(Q * itb);
  const double eps = A * (log(x * x * iX) + (2.0 * b / Q) * at - bx0 * (log(xm * xm * iX) + (2.0 * (b + 2.0 * x0) / Q) * at));
  const double q2 = 1.0 / (Q * Q + tb * tb);
  const double deps = A * (2.0 * isx - tb * iX - 4.0 * b * q2 - bx0 * (2.0 * ixm - tb * iX - 4.0 * (2.0 * x0 + b) * q2));
  const double vc = eps - (x / 6.0) * deps;
  f = rho * (eps - XC_CX * r13);
  vr = vc - (4.0 / 3.0) * XC_CX * r13;
}

__device__ __forceinline__ void gga_pbe(double rho, double sigma, double& f, double& vr, double& vs) {
  const double kappa = 0.804, mu = 0.2195149727645171;
  const double gamma = 0.031090690869654895, beta = 0.06672455060314922;
  const double A = 0.0310907, a1 = 0.21370, b1 = 7.5957, b2 = 3.5876, b3 = 1.6382, b4 = 0.49294;
  const double c_s2 = 38.283120002509214;      // 4 (3 pi^2)^(2/3)
  const double c_t2 = 0.06346820609770369;     // pi / (16 (3 pi^2)^(1/3))
  const double ir13 = rcbrt(rho);
  const double ir23 = ir13 * ir13;
  const double r13 = rho * ir23;
  const double r43 = rho * r13;
  const double ir43 = ir23 * ir23, irho = ir23 * ir13;
  // exchange
  const double s2 = sigma * (ir43 * ir43) * (1.0 / c_s2);
  const double den = 1.0 / (kappa + mu * s2);
  const double F = 1.0 + kappa - kappa * kappa * den;
  const double dF = kappa * kappa * mu * den * den;
  const double fx = -XC_CX * r43 * F;
  const double vxr = -(4.0 / 3.0) * XC_CX * r13 * (F - 2.0 * s2 * dF);
  const double vxs = -XC_CX * dF * ir43 * (1.0 / c_s2);
  // PW92
  const double rs = XC_RSFAC * ir13;
  const double isrs = rsqrt(rs);
  const double srs = rs * isrs;
  const double q = 2.0 * A * (srs * (b1 + b3 * rs) + rs * (b2 + b4 * rs));
  const double dq = 2.0 * A * (0.5 * b1 * isrs + b2 + 1.5 * b3 * srs + 2.0 * b4 * rs);
  const double tq = 1.0 / (q * (q + 1.0));
  const double lg = log1p(tq * (q + 1.0));     // log(1 + 1/q)
  const double eu = -2.0 * A * (1.0 + a1 * rs) * lg;
  const double deu_drs = -2.0 * A * a1 * lg + 2.0 * A * (1.0 + a1 * rs) * dq * tq;
  const double deu = -deu_drs * rs * irho * (1.0 / 3.0);    // d eps_unif / d rho
  // H
  const double yfac = c_t2 * ir43 * irho;      // c_t2 / rho^(7/3)
  const double y = sigma * yfac;
  const double Em1 = expm1(-eu * (1.0 / gamma));
  const double Ac = (beta / gamma) / Em1;
  const double Ay = Ac * y;
  const double N = 1.0 + Ay, D = 1.0 + Ay + Ay * Ay;
  const double cyN = (beta / gamma) * y * N;
  const double Du = D + cyN;                   // D (1 + G)
  const double iDDu = 1.0 / (D * Du);          // 1 / (D^2 (1 + G))
  const double G = cyN * (iDDu * Du);
  const double H = gamma * log1p(G);
  const double dHdy = beta * (1.0 + 2.0 * Ay) * iDDu;
  const double dHdA = -beta * y * Ay * y * (2.0 + Ay) * iDDu;
  const double dAde = Ac * Ac * (Em1 + 1.0) * (1.0 / beta);
  const double vcs = rho * dHdy * yfac;
  const double vcr = eu + H + rho * (deu + dHdy * (-(7.0 / 3.0) * y * irho) + dHdA * dAde * deu);
  f = fx + rho * (eu + H);
  vr = vxr + vcr;
  vs = vxs + vcs;
}

template <bool GGA>
__device__ __forceinline__ void xc_point(double rho, double sigma, double rho_tol, double& f, double& vr, double& vs) {
  f = 0.0; vr = 0.0; vs = 0.0;
  if (!(rho > rho_tol)) return;
  if (GGA) gga_pbe(rho, sigma, f, vr, vs);
  else lda_slater_vwn5(rho, f, vr);
}

__global__ void k_functional(int kind, int64_t n, const double* rho, const double* sigma, double rho_tol, double* f,
                             double* vr, double* vs) {
  int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  double a, b, c;
  if (kind == 1) xc_point<true>(rho[i], sigma[i], rho_tol, a, b, c);
  else xc_point<false>(rho[i], 0.0, rho_tol, a, b, c);
  f[i] = a; vr[i] = b; vs[i] = c;
}

// ------------------------------------------------------------------------------------------------
// step (a): partition weights.  One thread per point (points are batch-contiguous, so a warp is
// spatially compact and its loops over atoms stay uniform).  SSF uses its exact compact support:
//   * r_A < (1-a)/2 * R_nn(A)            => w = w^q               (all mu_AC <= -a)
//   * r_B >= kappa r_min, kappa=(1+a)/(1-a) => P_B = 0
//   * r_C >= kappa r_B                     => s(mu_BC) = 1
// ------------------------------------------------------------------------------------------------
__device__ __forceinline__ double s_ssf(double mu) {
  const double a = 0.64;
  if (mu <= -a) return 1.0;
  if (mu >= a) return 0.0;
  double z = mu * (1.0 / a), z2 = z * z;
  double g = z * (35.0 + z2 * (-35.0 + z2 * (21.0 - 5.0 * z2))) * (1.0 / 16.0);
  return 0.5 * (1.0 - g);
}
__device__ __forceinline__ double s_becke(double mu) {
  double p = mu;
#pragma unroll
  for (int k = 0; k < 3; ++k) p = 1.5 * p - 0.5 * p * p * p;
  return 0.5 * (1.0 - p);
}

template <int PART>
__global__ void __launch_bounds__(128) k_weights(int natoms, const double* __restrict__ atoms,
                                                 const double* __restrict__ invR, const double* __restrict__ rnn,
                                                 int64_t npts, const double* __restrict__ px,
                                                 const double* __restrict__ py, const double* __restrict__ pz,
                                                 const double* __restrict__ wq, const int32_t* __restrict__ parent,
                                                 double* __restrict__ w) {
  const unsigned FULL = 0xffffffffu;
  int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  bool act = i < npts;
  int64_t ii = act ? i : npts - 1;
  double x = px[ii], y = py[ii], z = pz[ii];
  int A = parent[ii];
  double base = wq[ii];
  bool done = !act;
  double result = base;
  auto dist = [&](int C) {
    double dx = x - __ldg(atoms + 3 * C), dy = y - __ldg(atoms + 3 * C + 1), dz = z - __ldg(atoms + 3 * C + 2);
    return sqrt(dx * dx + dy * dy + dz * dz);
  };
  if (natoms == 1) done = true;
  if (PART == 0 && !done) {
    double rA = dist(A);
    if (rA < 0.5 * (1.0 - 0.64) * __ldg(rnn + A)) done = true;
  }
  if (__all_sync(FULL, done)) {
    if (act) w[i] = result;
    return;
  }
  const double kappa = (1.0 + 0.64) / (1.0 - 0.64);
  double rmin = 1e300;
  int m = 0;
  if (PART == 0) {
    for (int C = 0; C < natoms; ++C) {
      double r = dist(C);
      if (r < rmin) { rmin = r; m = C; }
    }
  }
  double sum = 0.0, PA = 0.0;
  for (int B = 0; B < natoms; ++B) {
    double rB = dist(B);
    bool cand = !done;
    if (PART == 0) cand = cand && !(rB >= kappa * rmin && rB > rmin);
    if (!__any_sync(FULL, cand)) continue;
    double PB = cand ? 1.0 : 0.0;
    const double* iR = invR + (size_t)B * natoms;
    if (PART == 0) {
      // the nearest atom first: it zeroes most candidates at once
      if (cand && m != B) PB *= s_ssf((rB - rmin) * __ldg(iR + m));
      if (__any_sync(FULL, PB != 0.0)) {
        for (int C = 0; C < natoms; ++C) {
          double rC = dist(C);
          if (PB != 0.0 && C != B && C != m && rC < kappa * rB) PB *= s_ssf((rB - rC) * __ldg(iR + C));
          if ((C & 7) == 7 && !__any_sync(FULL, PB != 0.0)) break;
        }
      }
    } else {
      for (int C = 0; C < natoms; ++C) {
        double rC = dist(C);
        if (C != B) PB *= s_becke((rB - rC) * __ldg(iR + C));
      }
    }
    if (cand) {
      sum += PB;
      if (B == A) PA = PB;
    }
  }
  if (!done) result = base * PA / sum;
  if (act) w[i] = result;
}

// ------------------------------------------------------------------------------------------------
// step (a), hot path: one CTA per batch, one WARP per point.  The batch's atom list (planner: exact SSF support,
// sorted by distance to the batch box; owners = the first nB, partners = all nC) sits in shared memory; the
// lanes of a warp split the partners, so there is no divergence between points, and the products are
// combined with an xor butterfly (same value in every lane, fixed order => deterministic).
// ------------------------------------------------------------------------------------------------
template <int PART>
__global__ void __launch_bounds__(kWeightThreads) k_weights_batched(WeightArgs a, const int32_t* __restrict__ batch_ids, int nwarps) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  const unsigned FULL = 0xffffffffu;
  const BatchRec b = a.batches[batch_ids[blockIdx.x]];
  const int nC = b.wa_nC, nB = PART == 0 ? b.wa_nB : b.wa_nC;
  double* sXYZ = (double*)smem_raw;                 // [nC][3]
  double* sDall = sXYZ + (size_t)3 * nC;            // [nwarps][nC]
  int* sAt = (int*)(sDall + (size_t)nwarps * nC);   // [nC]
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  if (warp >= nwarps) return;
  for (int c = threadIdx.x; c < nC; c += nwarps * 32) {
    int at = a.watoms[b.wa_off + c];
    sAt[c] = at;
    sXYZ[3 * c] = a.atoms[3 * at]; sXYZ[3 * c + 1] = a.atoms[3 * at + 1]; sXYZ[3 * c + 2] = a.atoms[3 * at + 2];
  }
  // nwarps*32 threads take part (the others returned): named barrier over the active threads
  asm volatile("bar.sync 1, %0;" ::"r"(nwarps * 32));
  double* sD = sDall + (size_t)warp * nC;
  const double kappa = (1.0 + 0.64) / (1.0 - 0.64);
  for (int p = warp; p < b.nq; p += nwarps) {
    const int64_t gi = (int64_t)b.pt_off + p;
    const double x = a.px[gi], y = a.py[gi], z = a.pz[gi], base = a.wq[gi];
    const int A = a.parent[gi];
    double result = base;
    bool trivial = a.natoms == 1;
    if (PART == 0 && !trivial) {
      double dx = x - a.atoms[3 * A], dy = y - a.atoms[3 * A + 1], dz = z - a.atoms[3 * A + 2];
      trivial = sqrt(dx * dx + dy * dy + dz * dz) < 0.5 * (1.0 - 0.64) * a.rnn[A];
    }
    if (!trivial) {
      double dmin = 1e300;
      int imin = 0x7fffffff;
      for (int c = lane; c < nC; c += 32) {
        double dx = x - sXYZ[3 * c], dy = y - sXYZ[3 * c + 1], dz = z - sXYZ[3 * c + 2];
        double d = sqrt(dx * dx + dy * dy + dz * dz);
        sD[c] = d;
        if (d < dmin) { dmin = d; imin = c; }
      }
#pragma unroll
      for (int o = 16; o >= 1; o >>= 1) {
        double od = __shfl_xor_sync(FULL, dmin, o);
        int oi = __shfl_xor_sync(FULL, imin, o);
        if (od < dmin || (od == dmin && oi < imin)) { dmin = od; imin = oi; }
      }
      __syncwarp();
      double sum = 0.0, PA = 0.0;
      const int nsteps = (nC + 31) >> 5;
      // Becke-88: the parent first (always in full), then the owners nearest to the batch first.  An owner's product is
      // abandoned as soon as one lane's partial product (an upper bound of P_B: every factor is <= 1) is below 2^-60 of
      // the sum so far: adding such a term would not change the fp64 sum, so w is bit-identical to the full
      // O(N_A^2) evaluation in this order.  (k_weights_ssf applies the same rule on its long-list path.)
      int ia = -1;
      if (PART == 1) {
        for (int c0 = 0; c0 < nC && ia < 0; c0 += 32) {
          const unsigned m = __ballot_sync(FULL, c0 + lane < nC && sAt[c0 + lane] == A);
          if (m) ia = c0 + __ffs(m) - 1;
        }
      }
      unsigned premask = 0xffffffffu;
      for (int ib = (PART == 1 ? -1 : 0); ib < nB; ++ib) {
        if (PART == 1 && ib >= 0 && (ib & 31) == 0) {
          // 32 owners at a time, one per lane: the product of the factors against the 8 atoms nearest to the batch is an
          // upper bound of P_B; below 2^-60 of the sum so far (which only grows) the owner cannot change the sum
          const int ob = ib + lane;
          bool keep = ob < nB;
          if (keep && ob != ia) {
            const double rO = sD[ob];
            const double* iRo = a.invR + (size_t)sAt[ob] * a.natoms;
            double bound = 1.0;
            const int npre = min(8, nC);
            for (int k = 0; k < npre; ++k)
              if (k != ob) bound *= s_becke((rO - sD[k]) * __ldg(iRo + sAt[k]));
            keep = !(bound < sum * 8.673617379884035e-19);
          }
          premask = __ballot_sync(FULL, keep);
        }
        const int bb = ib < 0 ? ia : ib;
        if (PART == 1 && (bb < 0 || (ib >= 0 && bb == ia))) continue;
        if (PART == 1 && ib >= 0 && !((premask >> (ib & 31)) & 1u)) continue;
        const double thresh = (PART == 1 && ib >= 0) ? sum * 8.673617379884035e-19 : 0.0;   // 2^-60
        const double rB = sD[bb];
        if (PART == 0 && rB >= kappa * dmin && rB > dmin) continue;           // P_B = 0 exactly
        const int Bid = sAt[bb];
        const double* iR = a.invR + (size_t)Bid * a.natoms;
        double PB = 1.0;
        if (PART == 0 && bb != imin) {
          PB = s_ssf((rB - dmin) * __ldg(iR + sAt[imin]));                     // nearest atom first
          if (PB == 0.0) continue;
        }
        double part = 1.0;
        for (int k = 0; k < nsteps; ++k) {
          const int c = (k << 5) + lane;
          if (c < nC && c != bb && (PART == 1 || c != imin)) {
            const double rC = sD[c];
            if (PART == 1) part *= s_becke((rB - rC) * __ldg(iR + sAt[c]));
            else if (rC < kappa * rB) part *= s_ssf((rB - rC) * __ldg(iR + sAt[c]));  // else the factor is exactly 1
          }
          if (PART == 0 && (k & 3) == 3 && !__any_sync(FULL, part != 0.0)) break;
          if (PART == 1 && thresh > 0.0) {                                       // negligible owner?
            // log2 of the product over the lanes bounded from above by one integer warp reduction (see ssf_cell_product)
            const int ub = __reduce_add_sync(FULL, __double2hiint(part) >> 10) - 32 * (1023 << 10) + 32 * (1 + 89);
            if (ub < (__double2hiint(thresh) >> 10) - (1023 << 10)) { part = -1.0; break; }
          }
        }
        if (PART == 1 && part < 0.0) continue;                                  // warp-uniform
#pragma unroll
        for (int o = 16; o >= 1; o >>= 1) part *= __shfl_xor_sync(FULL, part, o);
        PB *= part;
        sum += PB;
        if (Bid == A) PA = PB;
      }
      result = base * PA / sum;
      __syncwarp();
    }
    if (lane == 0) a.w[gi] = result;
  }
}

// ------------------------------------------------------------------------------------------------
// step (a), hot path for SSF: one CTA (16 warps) per batch, one WARP per non-trivial point, the lanes split the
// atoms.  Exact pruning only.  The batch's atom list (planner) is sorted by dmin(atom, batch box)
// <= r_atom, so every scan stops as soon as dmin reaches its bound, and all control flow is warp-uniform.
//
// Per batch (once): the first kLcap list atoms (x, y, z, dmin) and the dmin of every chunk of 32 in shared memory;
//   a table 1 / (a R_BC) for the first kTabB (owner) x kTabC (partner) list positions.
// Per point (one warp, points handed out dynamically):
//   0. r_A < (1-a)/2 R_nn(A)  =>  w = w^q (decided per thread before; the other points are compacted in order).
//   1. nearest atom m, r_min (32 atoms per step, scan while dmin < r_min).  Every distance r_C computed on the way
//      is kept in a per-warp shared-memory row (filled lazily, chunk by chunk) and reused by all cell products.
//   2. P_A first: P_A = 0 => w = 0 and the point is done.
//   3. owner candidates B, 32 per step, one per lane (scan while dmin < kappa r_min): r_B < kappa r_min, and not
//      already zeroed by one of the kPre atoms nearest to the batch box or by m (mu_BC >= a <=> r_B - r_C >= a R_BC);
//      each survivor's cell product P_B is then evaluated by the whole warp.
//   Cell product: partners C in chunks of 32 while dmin < kappa r_B (beyond, s(mu_BC) = 1 exactly); a chunk whose
//   32 distances are all >= kappa r_B is skipped; mu_BC / a = (r_B - r_C) / (a R_BC) with 1 / (a R_BC) from the table
//   or from the coordinates, clamped below at -1 (where the polynomial is exactly 1); the scan stops as soon as one
//   mu_BC >= a (P_B = 0).  In the table path the factor s(0) = 1/2 of the pair (B, B) is multiplied in and undone by
//   an exact factor 2.
//   Lane products are combined by an xor butterfly (same value in every lane) and the owners are summed in
//   list order, so w is bit-identical from run to run.
// ------------------------------------------------------------------------------------------------
constexpr int kSsfThreads = 512, kSsfWarps = kSsfThreads / 32;
constexpr int kRcap = 256;                  // per-warp distance row: first kRcap list positions
constexpr int kTabC = 320;                  // 1/(a R_BC) table: partners (list positions) per owner row
constexpr int kMaxCh = 128;                 // chunk-start dmin values held in shared memory
constexpr int kPre = 8;                     // partners used by the lane-parallel owner pre-filter
constexpr size_t kSsfSmem = 112 * 1024;     // two CTAs per SM
// shared-memory split (launch_weights_batched): lcap list atoms (28 B each) + fixed parts + tabB table rows
constexpr size_t kSsfFixed = (size_t)kSsfWarps * kRcap * 8 + (size_t)kMaxCh * 8 + 512 * 2;
constexpr int kSsfMaxLcap = (int)((kSsfSmem - kSsfFixed - (size_t)8 * kTabC * 8) / 28) / 32 * 32;

struct SsfCtx {
  const double* sX; const double* sY; const double* sZ; const int* sId; const double* sTab; const double* sDm; double* sRC;
  const WeightArgs* a; const double* box; int64_t wa_off;
  int nC, nch, lane, lcap, tabB;
  double x, y, z;
  int filled;     // list positions [0, filled) of sRC hold r_C of this point
};

__device__ __forceinline__ double ssf_poly(double zz) {   // s(mu) for zz = mu / a in [-1, 1]; exactly 1 at -1, 0 at +1
  const double z2 = zz * zz;
  return fma(-zz, fma(z2, fma(z2, fma(z2, -5.0 / 32.0, 21.0 / 32.0), -35.0 / 32.0), 35.0 / 32.0), 0.5);
}

__device__ __forceinline__ double ssf_dmin_box(double cx, double cy, double cz, const double* box) {
  const double tx = cx < box[0] ? box[0] - cx : (cx > box[3] ? cx - box[3] : 0.0);
  const double ty = cy < box[1] ? box[1] - cy : (cy > box[4] ? cy - box[4] : 0.0);
  const double tz = cz < box[2] ? box[2] - cz : (cz > box[5] ? cz - box[5] : 0.0);
  // a hair below the true distance: the early exits must never cut an atom that matters
  return sqrt(tx * tx + ty * ty + tz * tz) * (1.0 - 1e-12) - 1e-12;
}

// coordinates of list entry c: shared memory for c < lcap, global beyond (systems with more atoms than fit)
__device__ __forceinline__ void ssf_atom(const SsfCtx& s, int c, double& cx, double& cy, double& cz) {
  if (c < s.lcap) { cx = s.sX[c]; cy = s.sY[c]; cz = s.sZ[c]; return; }
  const int at = s.a->watoms[s.wa_off + c];
  cx = s.a->atoms[3 * at]; cy = s.a->atoms[3 * at + 1]; cz = s.a->atoms[3 * at + 2];
}
__device__ __forceinline__ double ssf_chunk_dmin(const SsfCtx& s, int ch) {
  if (ch < kMaxCh) return s.sDm[ch];
  double cx, cy, cz;
  ssf_atom(s, ch * 32, cx, cy, cz);
  return ssf_dmin_box(cx, cy, cz, s.box);
}
// number of leading chunks whose first (smallest) dmin is below `bound`
__device__ __forceinline__ int ssf_nscan(const SsfCtx& s, double bound) {
  for (int base = 0; base < s.nch; base += 32) {
    const int ch = base + s.lane;
    const double v = ch < s.nch ? ssf_chunk_dmin(s, ch) : 1e300;
    const unsigned m = __ballot_sync(0xffffffffu, v >= bound);
    if (m) return base + __ffs(m) - 1;
  }
  return s.nch;
}

// r_C of this lane's list position c = c0 + lane (c0 warp-uniform); fills the warp's row on first touch
__device__ __forceinline__ double ssf_dist(SsfCtx& s, int c0) {
  const int c = c0 + s.lane;
  if (c0 < s.filled) return s.sRC[c];
  double r = 1e300;
  if (c < s.nC) {
    double cx, cy, cz;
    ssf_atom(s, c, cx, cy, cz);
    const double dx = s.x - cx, dy = s.y - cy, dz = s.z - cz;
    r = sqrt(dx * dx + dy * dy + dz * dz);
  }
  if (c0 < kRcap && c0 == s.filled) { s.sRC[c] = r; s.filled = c0 + 32; __syncwarp(); }
  return r;
}

// P_B = prod_C s(mu_BC).  bb = list position of B (warp-uniform, -1: not in the list), rB = r_B.
// (Bx, By, Bz) is only read for bb < 0; a list atom's coordinates are fetched where the table does not reach.
// thresh: an owner other than the parent is abandoned (returns 0) as soon as the product over the partners visited so far --
// an upper bound of P_B, every factor being <= 1 -- is below thresh = 2^-61 of the running sum of the owners before it:
// adding such a P_B would not change the fp64 sum, so w stays bit-identical.  The bound is formed (one integer warp reduction) after
// every visited chunk of the long-list path only; the short-list path is too cheap to pay for it.
__device__ __forceinline__ double ssf_cell_product(SsfCtx& s, int bb, double Bx, double By, double Bz, double rB, double thresh) {
  const unsigned FULL = 0xffffffffu;
  const double kappa = (1.0 + 0.64) / (1.0 - 0.64);
  const double krB = kappa * rB;
  const int nscan = ssf_nscan(s, krB);                     // every later C has r_C >= kappa r_B: factor 1
  const bool tab = bb >= 0 && bb < s.tabB;
  double part = 1.0;
  if (tab && s.filled >= s.nC) {
    // short list (the whole row was filled up front and every partner is in the table): no chunk tests; a factor
    // that is exactly 1 comes out of the clamped polynomial as exactly 1
    const double* trow = s.sTab + bb * kTabC + s.lane;
    const double* rrow = s.sRC + s.lane;
    for (int ch = 0; ch < nscan; ++ch) {
      double zz = (rB - rrow[ch << 5]) * trow[ch << 5];     // (B, B): 0, factor 1/2; c >= nC: r_C = 1e300, entry 1
      if (__any_sync(FULL, zz >= 1.0)) return 0.0;         // s = 0: P_B = 0
      zz = zz < -1.0 ? -1.0 : zz;
      part *= ssf_poly(zz);
    }
#pragma unroll
    for (int o = 16; o >= 1; o >>= 1) part *= __shfl_xor_sync(FULL, part, o);
    return part * 2.0;
  }
  if (bb >= 0) ssf_atom(s, bb, Bx, By, Bz);
  int nvis = 0;                                            // chunks that contributed factors
  auto negligible = [&]() {
    if (!(thresh > 0.0)) return false;
    // log2 of the product over the 32 lanes, bounded from ABOVE in fixed point with 10 fractional bits, by one integer
    // warp reduction: for x = m 2^e, m in [1, 2):  e + (m - 1) <= log2 x <= e + (m - 1) + 0.0861.  The high word >> 10 is
    // (e + 1023) 2^10 + the top 10 mantissa bits (truncated: + 1).  The bound is within 2^2.8 of the product; thresh is
    // bounded from BELOW the same way, so `true` implies product < thresh rigorously.
    const int I = __double2hiint(part) >> 10;
    const int ub = __reduce_add_sync(FULL, I) - 32 * (1023 << 10) + 32 * (1 + 89);   // 89 = ceil(0.0861 * 1024)
    const int lt = (__double2hiint(thresh) >> 10) - (1023 << 10);
    return ub < lt;                                        // same value in every lane
  };
  const int nrow = min(nscan, kRcap >> 5);                 // chunks served by the distance row
  for (int ch = 0; ch < nrow; ++ch) {
    const int c0 = ch << 5, c = c0 + s.lane;
    const double rC = ssf_dist(s, c0);
    if (!__any_sync(FULL, rC < krB)) continue;             // 32 factors exactly 1
    double zz;
    if (tab && c0 < kTabC) {
      zz = (rB - rC) * s.sTab[bb * kTabC + c];             // (B, B): 0, factor 1/2; c >= nC: r_C = 1e300, entry 1
    } else {
      zz = -1.0;                                           // factor exactly 1
      if (c < s.nC && c != bb) {
        double cx, cy, cz;
        ssf_atom(s, c, cx, cy, cz);
        const double ex = Bx - cx, ey = By - cy, ez = Bz - cz;
        zz = (rB - rC) * (rsqrt(ex * ex + ey * ey + ez * ez) * (1.0 / 0.64));   // mu_BC / a
      }
    }
    if (__any_sync(FULL, zz >= 1.0)) return 0.0;           // s = 0: P_B = 0
    zz = zz < -1.0 ? -1.0 : zz;
    part *= ssf_poly(zz);
    ++nvis;
    if (negligible()) return 0.0;
  }
  // partners past the row: r_C and R_BC from one fetch of the coordinates
  for (int ch = nrow; ch < nscan; ++ch) {
    const int c0 = ch << 5, c = c0 + s.lane;
    const bool valid = c < s.nC;
    double cx = 0.0, cy = 0.0, cz = 0.0, rC = 1e300;
    if (valid) {
      ssf_atom(s, c, cx, cy, cz);
      const double dx = s.x - cx, dy = s.y - cy, dz = s.z - cz;
      rC = sqrt(dx * dx + dy * dy + dz * dz);
    }
    if (!__any_sync(FULL, rC < krB)) continue;             // 32 factors exactly 1
    double zz = -1.0;                                      // factor exactly 1
    if (tab && c0 < kTabC) {
      zz = (rB - rC) * s.sTab[bb * kTabC + c];
    } else if (valid && c != bb) {
      const double ex = Bx - cx, ey = By - cy, ez = Bz - cz;
      zz = (rB - rC) * (rsqrt(ex * ex + ey * ey + ez * ez) * (1.0 / 0.64));   // mu_BC / a
    }
    if (__any_sync(FULL, zz >= 1.0)) return 0.0;           // s = 0: P_B = 0
    zz = zz < -1.0 ? -1.0 : zz;
    part *= ssf_poly(zz);
    ++nvis;
    if (negligible()) return 0.0;
  }
#pragma unroll
  for (int o = 16; o >= 1; o >>= 1) part *= __shfl_xor_sync(FULL, part, o);
  // table path: the chunk of B itself is always visited (dmin_B <= r_B < kappa r_B) and contributed s(0) = 1/2
  if (tab) part *= 2.0;
  return part;
}

__global__ void __launch_bounds__(kSsfThreads, 2) k_weights_ssf(WeightArgs a, const int32_t* __restrict__ batch_ids, int lcap, int tabB) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  __shared__ int sCnt[kSsfWarps];
  __shared__ int sNext;
  const unsigned FULL = 0xffffffffu;
  const int bid = batch_ids[blockIdx.x];
  const BatchRec b = a.batches[bid];
  const int nC = b.wa_nC, nB = b.wa_nB;
  double* sX = (double*)smem_raw;                        // [lcap] x 3
  double* sY = sX + lcap;
  double* sZ = sY + lcap;
  double* sRCall = sZ + lcap;                            // [kSsfWarps][kRcap]
  double* sDm = sRCall + kSsfWarps * kRcap;              // [kMaxCh]
  double* sTab = sDm + kMaxCh;                           // [tabB][kTabC]
  int* sId = (int*)(sTab + tabB * kTabC);                // [lcap]
  short* sList = (short*)(sId + lcap);                   // compacted non-trivial points of the batch (<= 512)
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const double aa = 0.64, kappa = (1.0 + aa) / (1.0 - aa);
  const double* box = a.wbox + (size_t)6 * bid;

  // ---- 0. trivial points, ordered compaction of the others ----
  bool live = false;
  {
    const int p = threadIdx.x;
    if (p < b.nq) {
      const int64_t gi = (int64_t)b.pt_off + p;
      const int A = a.parent[gi];
      bool trivial = a.natoms == 1;
      if (!trivial) {
        const double dx = a.px[gi] - a.atoms[3 * A], dy = a.py[gi] - a.atoms[3 * A + 1], dz = a.pz[gi] - a.atoms[3 * A + 2];
        trivial = sqrt(dx * dx + dy * dy + dz * dz) < 0.5 * (1.0 - aa) * a.rnn[A];
      }
      if (trivial) a.w[gi] = a.wq[gi];
      live = !trivial;
    }
  }
  const unsigned lmask = __ballot_sync(FULL, live);
  if (lane == 0) sCnt[warp] = __popc(lmask);
  if (threadIdx.x == 0) sNext = kSsfWarps;
  __syncthreads();
  int total = 0, off = 0;
#pragma unroll
  for (int k = 0; k < kSsfWarps; ++k) {
    if (k < warp) off += sCnt[k];
    total += sCnt[k];
  }
  if (live) sList[off + __popc(lmask & ((1u << lane) - 1u))] = (short)threadIdx.x;
  if (total == 0) return;
  const int nS = min(nC, lcap), nch = (nC + 31) >> 5;
  for (int c = threadIdx.x; c < nS; c += kSsfThreads) {
    const int at = a.watoms[b.wa_off + c];
    const double cx = a.atoms[3 * at], cy = a.atoms[3 * at + 1], cz = a.atoms[3 * at + 2];
    sX[c] = cx; sY[c] = cy; sZ[c] = cz;
    sId[c] = at;
    if ((c & 31) == 0 && (c >> 5) < kMaxCh) sDm[c >> 5] = ssf_dmin_box(cx, cy, cz, box);
  }
  for (int ch = (lcap >> 5) + threadIdx.x; ch < min(nch, kMaxCh); ch += kSsfThreads) {
    const int at = a.watoms[b.wa_off + ch * 32];
    sDm[ch] = ssf_dmin_box(a.atoms[3 * at], a.atoms[3 * at + 1], a.atoms[3 * at + 2], box);
  }
  __syncthreads();
  if (total < 8) tabB = 0;                                 // too few points to pay for the table
  {
    const int tb = min(nS, tabB), tc = min((nC + 31) & ~31, kTabC);
    for (int e = threadIdx.x; e < tb * tc; e += kSsfThreads) {
      const int bb = e / tc, c = e - bb * tc;
      double v = 1.0;                                      // neutral entry for c >= nC (r_C = 1e300 there)
      if (c < nC) {
        double cx, cy, cz;
        if (c < lcap) { cx = sX[c]; cy = sY[c]; cz = sZ[c]; }
        else { const int at = a.watoms[b.wa_off + c]; cx = a.atoms[3 * at]; cy = a.atoms[3 * at + 1]; cz = a.atoms[3 * at + 2]; }
        const double ex = sX[bb] - cx, ey = sY[bb] - cy, ez = sZ[bb] - cz;
        v = bb == c ? 0.0 : rsqrt(ex * ex + ey * ey + ez * ez) * (1.0 / 0.64);
      }
      sTab[bb * kTabC + c] = v;
    }
    tabB = tb;
    __syncthreads();
  }
  const int tcols = tabB > 0 ? min((nC + 31) & ~31, kTabC) : 0;   // table columns that were built

  SsfCtx s;
  s.sX = sX; s.sY = sY; s.sZ = sZ; s.sId = sId; s.sTab = sTab; s.sDm = sDm; s.sRC = sRCall + warp * kRcap; s.a = &a; s.box = box;
  s.wa_off = b.wa_off; s.nC = nC; s.nch = nch; s.lane = lane; s.lcap = lcap; s.tabB = tabB;
  for (int n = warp; n < total;) {
    const int64_t gi = (int64_t)b.pt_off + sList[n];
    s.x = a.px[gi]; s.y = a.py[gi]; s.z = a.pz[gi];
    s.filled = 0;
    const int A = a.parent[gi];
    __syncwarp();                                          // the previous point's readers of the row are done
    // ---- 1. nearest atom ----
    double rmin = 1e300;
    int im = 0;
    for (int c0 = 0; c0 < nC; c0 += 32) {
      if (ssf_chunk_dmin(s, c0 >> 5) >= rmin) break;
      const double r = ssf_dist(s, c0);
      // argmin over the lanes: r >= 0, so the bit patterns order like the values
      const unsigned hi = (unsigned)__double2hiint(r);
      const unsigned mhi = __reduce_min_sync(FULL, hi);
      const unsigned lo = hi == mhi ? (unsigned)__double2loint(r) : 0xffffffffu;
      const unsigned mlo = __reduce_min_sync(FULL, lo);
      const double rm = __hiloint2double((int)mhi, (int)mlo);
      if (rm < rmin) { rmin = rm; im = c0 + __ffs(__ballot_sync(FULL, hi == mhi && lo == mlo)) - 1; }
    }
    const double own_lim = kappa * rmin;
    if (nC <= kRcap) {                                     // short list: complete the row now (fast cell products)
      for (int c0 = s.filled; c0 < nC; c0 += 32) ssf_dist(s, c0);
    }
    // ---- 2. the parent's cell product ----
    const double Ax = a.atoms[3 * A], Ay = a.atoms[3 * A + 1], Az = a.atoms[3 * A + 2];
    double rA;
    { const double dx = s.x - Ax, dy = s.y - Ay, dz = s.z - Az; rA = sqrt(dx * dx + dy * dy + dz * dz); }
    double result = 0.0;
    if (!(rA >= own_lim && rA > rmin)) {
      int ia = -1;                                         // list position of the parent
      for (int c0 = 0; c0 < nC && ia < 0; c0 += 32) {
        const int c = c0 + lane;
        const unsigned m = __ballot_sync(FULL, c < nC && (c < lcap ? sId[c] : a.watoms[b.wa_off + c]) == A);
        if (m) ia = c0 + __ffs(m) - 1;
      }
      const double PA = ssf_cell_product(s, ia, Ax, Ay, Az, rA, 0.0);
      if (PA != 0.0) {
        // ---- 3. the other owners ----
        double sum = PA;
        double mx, my, mz;
        ssf_atom(s, im, mx, my, mz);
        const int nown = min(ssf_nscan(s, own_lim) << 5, nB);
        for (int b0 = 0; b0 < nown; b0 += 32) {
          const int bb = b0 + lane;
          const double rB = ssf_dist(s, b0);
          bool cand = bb < nB && bb != ia && rB < own_lim;   // else r_B >= kappa r_min: P_B = 0 exactly
          // pre-filter: mu_BC >= a for one of the first kPre list atoms or the nearest atom  =>  P_B = 0
          const int npre = min(kPre, nC);
          if (tabB >= npre && b0 + 32 <= tcols) {
            // 1 / (a R_Bk) = table entry (k, B): row k is warp-uniform, the lanes read consecutive columns;
            // the entry (B, B) is 0, so k = B never fires
            for (int k = 0; k < npre; ++k)                   // positions < 32 of the row are always filled (scan 1)
              if ((rB - s.sRC[k]) * sTab[k * kTabC + bb] >= 1.0) cand = false;
            if (im >= npre && __any_sync(FULL, cand)) {
              double bx = 0.0, by = 0.0, bz = 0.0;
              if (cand) ssf_atom(s, bb, bx, by, bz);
              const double u = rB - rmin;
              const double ex = bx - mx, ey = by - my, ez = bz - mz;
              if (im != bb && u > 0.0 && u * u >= (aa * aa) * (ex * ex + ey * ey + ez * ez)) cand = false;
            }
          } else {
            double bx = 0.0, by = 0.0, bz = 0.0;
            if (cand) ssf_atom(s, bb, bx, by, bz);
            for (int k = 0; k < npre; ++k) {
              const double u = rB - s.sRC[k];
              const double ex = bx - sX[k], ey = by - sY[k], ez = bz - sZ[k];
              if (k != bb && u > 0.0 && u * u >= (aa * aa) * (ex * ex + ey * ey + ez * ez)) cand = false;
            }
            if (im >= npre) {
              const double u = rB - rmin;
              const double ex = bx - mx, ey = by - my, ez = bz - mz;
              if (im != bb && u > 0.0 && u * u >= (aa * aa) * (ex * ex + ey * ey + ez * ez)) cand = false;
            }
          }
          unsigned mask = __ballot_sync(FULL, cand);
          while (mask) {
            const int src = __ffs(mask) - 1;
            mask &= mask - 1;
            const int bs = b0 + src;
            sum += ssf_cell_product(s, bs, 0.0, 0.0, 0.0, __shfl_sync(FULL, rB, src), sum * 4.3368086899420177e-19);   // 2^-61
          }
        }
        result = a.wq[gi] * PA / sum;
      }
    }
    if (lane == 0) { a.w[gi] = result; n = atomicAdd(&sNext, 1); }
    n = __shfl_sync(FULL, n, 0);
  }
}

// ------------------------------------------------------------------------------------------------
// P^j pack (Eq. (12b), Alg. 4 l.4.2): gathers the batch's block of P ONCE per build into the
// DMMA B-fragment order the batch kernel consumes: for k-step ks (4 nu) and column tile nt (8 mu), 32
// contiguous doubles, lane (g4 = lane >> 2, t4 = lane & 3) holding P[nu = 4 ks + t4][mu = 8 nt + g4];
// zero padded to nb4 x nb8.  One warp-wide 256-byte load per fragment in the batch kernel, no index math there.
// ------------------------------------------------------------------------------------------------
// tri (LDA): rho = phi^T P phi = 2 phi^T L phi with L = strict lower triangle of P^j + half its diagonal, so only
// L is packed (entries nu > mu are zero) and the X GEMM skips the k-steps above the diagonal.
__global__ void __launch_bounds__(256) k_pack_P(BatchArgs a, const int32_t* __restrict__ batch_ids, int tri) {
  const BatchRec b = a.batches[batch_ids[blockIdx.x]];
  const int nb = b.nb, ntile = (nb + 7) >> 3, nks = (nb + 3) >> 2;
  const int32_t* fidx = a.bfidx + b.f_off;
  double* out = a.ppk + b.ppk_off;
  const int total = nks * ntile * 32;
  for (int e = threadIdx.x; e < total; e += 256) {
    const int lane = e & 31, frag = e >> 5;
    const int ks = frag / ntile, nt = frag - ks * ntile;
    const int nu = 4 * ks + (lane & 3), mu = 8 * nt + (lane >> 2);
    double v = 0.0;
    if (nu < nb && mu < nb) v = __ldg(a.P + (size_t)fidx[mu] * a.ldp + fidx[nu]);   // P symmetric: row mu is read along nu
    if (tri) v = nu < mu ? v : (nu == mu ? 0.5 * v : 0.0);
    out[e] = v;
  }
}

// ------------------------------------------------------------------------------------------------
// exact, order-independent accumulation: 96-bit fixed point (two 64-bit integer atomics) => V is
// bit-identical from run to run whatever the order in which the batches arrive.
// ------------------------------------------------------------------------------------------------
__device__ __forceinline__ void fixed_add(unsigned long long* hi, unsigned long long* lo, double v) {
  // x = round(v * 2^64) as a signed 128-bit integer; lo = low 32 bits, hi = x >> 32
  long long bits = __double_as_longlong(v);
  int eb = (int)((bits >> 52) & 0x7ff);
  unsigned long long man = (unsigned long long)(bits & 0xfffffffffffffLL);
  if (eb) man |= 1ull << 52; else eb = 1;
  int s = eb - 1075 + 64;                       // x = man * 2^s
  __int128 x;
  if (s >= 0) x = (__int128)man << (s > 74 ? 74 : s);
  else if (s <= -54) x = 0;
  else x = (__int128)((man + (1ull << (-s - 1))) >> (-s));
  if (bits < 0) x = -x;
  unsigned long long l = (unsigned long long)x & 0xffffffffull;
  unsigned long long h = (unsigned long long)(long long)(x >> 32);
  if (l | h) {
    atomicAdd(lo, l);
    atomicAdd(hi, h);
  }
}

// ------------------------------------------------------------------------------------------------
// batch kernel: ONE CTA = one batch B_j, Alg. 4 l.4.3-4.10 fused.  The CTA walks over the batch's points in
// tiles of T; nothing but the packed P^j is read from and nothing but the final V^j increment is written to
// global memory:
//   per batch  0  shell records, primitive table (alpha, d), collocation order, 2^(j/64) table -> shared memory
//   per tile   1  collocation per (shell, point): R0, R1 -> sR (GGA); Phi -> sPhi[nu][i]              Eq. (7)
//              2  X^T = Phi^T P^j on DMMA (M = points, N = mu, K = nu): A from sPhi, B = packed P^j    Eq. (15)
//                 LDA: rho_i += Phi X in the epilogue, straight from the accumulator registers          Eq. (13)
//                 GGA: X^T -> shared memory (the Z buffer), then one pass per (shell, point):          Eqs. (13),(14)
//                      with m_c the monomials of the shell, S0 = sum_c X_c m_c, G = sum_c X_c grad m_c:
//                      rho_i += R0 S0, grad rho_i += R0 G + R1 S0 (r_i - R)
//              3  functional at the T points; E / N_el partials                                     Eqs. (19),(16)
//              4  GGA: Z_c = m_c (a R0 + R1 g.(r_i - R)) + R0 g.grad m_c per (shell, point) -> sZ       Eq. (20)
//              5  V^j += Z Phi^T + Phi Z^T on DMMA, lower-triangle 16x16 blocks, accumulators in     Eq. (18)
//                 REGISTERS over all tiles of the batch.  LDA: Z = 1/2 a Phi, so V^j = (a Phi) Phi^T is one
//                 symmetric product (half the flops); the scaling by a_i is applied to the A fragment.
//   per batch  6  increment of V (Eq. (17)): one fixed-point add per lower-triangle element.
// ------------------------------------------------------------------------------------------------
// X^T tile of one warp: C[u][v] += A_u(16 points x 4 nu) * B_v(4 nu x 8 mu) over all k-steps; NV mu-tiles (compile
// time), B fragments (packed P^j, global/L1) loaded one k-step ahead into registers and kPfDist k-steps ahead
// into L1 (the fragments of a batch are re-read for every tile, from L2 once they have left L1).
constexpr int kPfDist = 4;
template <int NV, int NTW, int BS>
__device__ __forceinline__ void xgemm_tile(double (&C)[2][NTW][2], const double* __restrict__ Ap, const double* __restrict__ Bp,
                                           int nks, int astep, int bstep) {
  double Bn[NV];
#pragma unroll
  for (int v = 0; v < NV; ++v) Bn[v] = __ldg(Bp + v * BS);
#pragma unroll
  for (int d = 1; d < kPfDist; ++d)
    if (d < nks) {
#pragma unroll
      for (int v = 0; v < NV; ++v) asm volatile("prefetch.global.L1 [%0];" ::"l"(Bp + (size_t)d * bstep + v * BS));
    }
  for (int ks = 0; ks < nks; ++ks) {
    const double A0 = Ap[0], A1 = Ap[8];
    double Bc[NV];
#pragma unroll
    for (int v = 0; v < NV; ++v) Bc[v] = Bn[v];
    Ap += astep;
    Bp += bstep;
    if (ks + kPfDist < nks) {
#pragma unroll
      for (int v = 0; v < NV; ++v) asm volatile("prefetch.global.L1 [%0];" ::"l"(Bp + (size_t)(kPfDist - 1) * bstep + v * BS));
    }
    if (ks + 1 < nks) {
#pragma unroll
      for (int v = 0; v < NV; ++v) Bn[v] = __ldg(Bp + v * BS);
    }
#pragma unroll
    for (int v = 0; v < NV; ++v) {
      dmma884(C[0][v][0], C[0][v][1], A0, Bc[v]);
      dmma884(C[1][v][0], C[1][v][1], A1, Bc[v]);
    }
  }
}

// LDA: X' = L Phi (k_pack_P, tri).  mu-tile mt only has non-zero fragments for the k-steps ks < 2 mt + 2, so the tiles of
// a warp (mt0, mt0 + WM, ...) drop in one after the other: k-steps [lim_{v-1}, lim_v) run the tiles v .. NV-1, each range
// with its own fully unrolled loop (no predicated-off DMMA).
template <int V0, int NV, int NTW, int BS>
__device__ __forceinline__ void xgemm_seg(double (&C)[2][NTW][2], const double*& Ap, const double*& Bp, int ks_lo, int ks_hi,
                                          int astep, int bstep) {
  if (ks_lo >= ks_hi) return;
  double Bn[NV];
#pragma unroll
  for (int v = V0; v < NV; ++v) Bn[v] = __ldg(Bp + v * BS);
  for (int ks = ks_lo; ks < ks_hi; ++ks) {
    const double A0 = Ap[0], A1 = Ap[8];
    double Bc[NV];
#pragma unroll
    for (int v = V0; v < NV; ++v) Bc[v] = Bn[v];
    Ap += astep;
    Bp += bstep;
    if (ks + kPfDist < ks_hi) {
#pragma unroll
      for (int v = V0; v < NV; ++v) asm volatile("prefetch.global.L1 [%0];" ::"l"(Bp + (size_t)(kPfDist - 1) * bstep + v * BS));
    }
    if (ks + 1 < ks_hi) {
#pragma unroll
      for (int v = V0; v < NV; ++v) Bn[v] = __ldg(Bp + v * BS);
    }
#pragma unroll
    for (int v = V0; v < NV; ++v) {
      dmma884(C[0][v][0], C[0][v][1], A0, Bc[v]);
      dmma884(C[1][v][0], C[1][v][1], A1, Bc[v]);
    }
  }
}
template <int NV, int NTW, int BS>
__device__ __forceinline__ void xgemm_tri(double (&C)[2][NTW][2], const double* Ap, const double* Bp, int nks, int mt0, int wmstep,
                                          int astep, int bstep) {
  int lim[4];
#pragma unroll
  for (int v = 0; v < 4; ++v) lim[v] = v < NV ? min(nks, 2 * (mt0 + v * wmstep) + 2) : nks;
  xgemm_seg<0, NV, NTW, BS>(C, Ap, Bp, 0, lim[0], astep, bstep);
  if (NV > 1) xgemm_seg<(NV > 1 ? 1 : 0), NV, NTW, BS>(C, Ap, Bp, lim[0], lim[1], astep, bstep);
  if (NV > 2) xgemm_seg<(NV > 2 ? 2 : 0), NV, NTW, BS>(C, Ap, Bp, lim[1], lim[2], astep, bstep);
  if (NV > 3) xgemm_seg<(NV > 3 ? 3 : 0), NV, NTW, BS>(C, Ap, Bp, lim[2], lim[3], astep, bstep);
}

template <int NT, int T>
struct BatchCfg {
  static constexpr int NW = NT / 32;           // warps per CTA
  static constexpr int WP = T / 16;            // warps along points in the X GEMM
  static constexpr int WM = NW / WP;           // warps along mu
  static constexpr int LD = T + 4;             // == 4 (mod 16) doubles: conflict-free fragment reads
  static constexpr int NG = NT / T;            // thread groups of the per-(shell, point) passes
};

template <int NT, int T, bool GGA, int NTW, int ROUNDS, int MINB>
__global__ void __launch_bounds__(NT, MINB) k_xc_batch(BatchArgs a, const int32_t* __restrict__ batch_ids) {
  using Cfg = BatchCfg<NT, T>;
  constexpr int LD = Cfg::LD;
  extern __shared__ __align__(16) unsigned char smem_raw[];
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int g4 = lane >> 2, t4 = lane & 3;
  const int bidx = batch_ids[blockIdx.x];
  const BatchRec b = a.batches[bidx];
  const int nb = b.nb, ns = b.ns;
  const int nb16 = (nb + 15) & ~15, ntile = (nb + 7) >> 3, nks = (nb + 3) >> 2;
  const int nbk = nb16 >> 4, nblocks = nbk * (nbk + 1) / 2;

  // ---- carve shared memory (mirrored by batch_smem_bytes in the planner) ----
  unsigned char* sp = smem_raw;
  double* sPhi = (double*)sp; sp += (size_t)nb16 * LD * 8;
  double* sZ = (double*)sp; if (GGA) sp += (size_t)nb16 * LD * 8;
  double* sR = (double*)sp; if (GGA) sp += (size_t)ns * T * 16;
  double* sPt = (double*)sp; sp += (size_t)16 * T * 8;  // points x, y, z, w of two tiles (double buffer) + 8 T scratch
  double* sRed = (double*)sp; sp += (size_t)NT * 4 * 8; // partial rho / grad rho: [groups][4][T]
  double* sExpT = (double*)sp; sp += (size_t)64 * 8;    // 2^(j/64)
  ShellRec* sSh = (ShellRec*)sp; sp += (size_t)ns * sizeof(ShellRec);
  int* sInfo = (int*)sp; sp += (size_t)nb16 * 4;
  int* sIdx = (int*)sp; sp += (size_t)nb16 * 4;
  int* sOrd = (int*)sp; sp += (size_t)((ns + 3) & ~3) * 4;   // [ns] shell slots, most primitives first
  double2* sPrim = (double2*)sp;                        // (alpha, d) of the batch's primitives, shell by shell
  double *sE = sPt + 8 * T, *sN = sPt + 9 * T;
  double *sA = sPt + 10 * T, *sG0 = sPt + 11 * T, *sG1 = sPt + 12 * T, *sG2 = sPt + 13 * T;

  // ---- points with w_i = 0 exactly (SSF zeroes ~10-20 % of them) add exact zeros to E, N_el and V^j: the tiles walk
  //      over the ordered list of the others (rho / grad rho of the skipped points are not evaluated) ----
  __shared__ short sLive[kBatchThreads];
  __shared__ int sLiveCnt[NT / 32];
  int nqe;
  {
    const bool live = tid < b.nq && a.w[(int64_t)b.pt_off + tid] != 0.0;   // N_q^j <= 512 = NT
    const unsigned lm = __ballot_sync(0xffffffffu, live);
    if (lane == 0) sLiveCnt[warp] = __popc(lm);
    __syncthreads();
    int off = 0;
    nqe = 0;
#pragma unroll
    for (int k = 0; k < NT / 32; ++k) {
      if (k < warp) off += sLiveCnt[k];
      nqe += sLiveCnt[k];
    }
    if (live) sLive[off + __popc(lm & ((1u << lane) - 1u))] = (short)tid;
    __syncthreads();
    if (nqe == 0) {                              // block-uniform
      if (tid == 0) { a.Epart[bidx] = 0.0; a.Npart[bidx] = 0.0; }
      return;
    }
  }

  // ---- per batch: metadata, zero padding rows, V^j block assignment ----
  {
    const int32_t* fidx = a.bfidx + b.f_off;
    const int32_t* finfo = a.bfinfo + b.f_off;
    for (int k = tid; k < ns; k += NT) {
      ShellRec r = a.shells[a.bshells[b.sh_off + k]];
      r._pad = a.bsfoff[b.sh_off + k];         // first local function of the shell
      r.atom = r.prim_off;                     // global primitive offset (the atom index is not used here)
      sSh[k] = r;
    }
    for (int f = tid; f < nb16; f += NT) {
      sIdx[f] = f < nb ? fidx[f] : 0;
      sInfo[f] = f < nb ? finfo[f] : 0;
    }
    for (int e = tid; e < (nb16 - nb) * LD; e += NT) {
      sPhi[(size_t)nb * LD + e] = 0.0;
      if (GGA) sZ[(size_t)nb * LD + e] = 0.0;
    }
    for (int k = tid; k < 64; k += NT) sExpT[k] = kExp2Tab[k];
    if (tid < T) {                               // points of the first tile
      const int64_t gi = (int64_t)b.pt_off + sLive[min(tid, nqe - 1)];
      sPt[tid] = a.px[gi]; sPt[T + tid] = a.py[gi]; sPt[2 * T + tid] = a.pz[gi];
      sPt[3 * T + tid] = tid < nqe ? a.w[gi] : 0.0;
    }
    __syncthreads();
    // collocation order (shells with the most primitives first, dealt round-robin to the warps) and the
    // primitive table: shell k's primitives start at the sum of the counts before it
    for (int k = tid; k < ns; k += NT) {
      const int ck = sSh[k].nprim * 4 + sSh[k].L;
      int rank = 0, loc = 0;
      for (int j = 0; j < ns; ++j) {
        const int cj = sSh[j].nprim * 4 + sSh[j].L;
        rank += (cj > ck || (cj == ck && j < k)) ? 1 : 0;
        loc += j < k ? sSh[j].nprim : 0;
      }
      sOrd[rank] = k;
      const int goff = sSh[k].atom, np = sSh[k].nprim;
      for (int q = 0; q < np; ++q) sPrim[loc + q] = make_double2(__ldg(a.exps + goff + q), __ldg(a.coefs + goff + q));
      sSh[k].prim_off = loc;                   // only thread k reads or writes this field from here on ... until the barrier
    }
  }
  int blk_m[ROUNDS], blk_n[ROUNDS];
  double V[ROUNDS][2][2][2];
#pragma unroll
  for (int r = 0; r < ROUNDS; ++r) {
    const int q = warp + Cfg::NW * r;
    int bm = (int)((sqrtf(8.0f * q + 1.0f) - 1.0f) * 0.5f);
    while ((bm + 1) * (bm + 2) / 2 <= q) ++bm;
    while (bm * (bm + 1) / 2 > q) --bm;
    blk_m[r] = q < nblocks ? bm : -1;
    blk_n[r] = q - bm * (bm + 1) / 2;
#pragma unroll
    for (int u = 0; u < 2; ++u)
#pragma unroll
      for (int v = 0; v < 2; ++v) V[r][u][v][0] = V[r][u][v][1] = 0.0;
  }
  const double* __restrict__ ppk = a.ppk + b.ppk_off;
  const int wp = warp % Cfg::WP, wm = warp / Cfg::WP;
  double Eacc = 0.0, Nacc = 0.0;
  PH_DECL
  PH(0);
  for (int t0 = 0, it = 0; t0 < nqe; t0 += T, ++it) {
    const int npt = min(T, nqe - t0);          // valid points in this tile
    const double* sx = sPt + (size_t)(it & 1) * 4 * T;   // this tile's points (written one tile ahead)
    const double *sy = sx + T, *sz = sx + 2 * T, *sw = sx + 3 * T;
    __syncthreads();                           // previous tile's readers of sPhi / sZ are done; tables / points visible
    PH(1);

    // ---- 1. collocation (Eq. (7); same shell across a warp) ----
    for (int q = warp; q < ns * (T / 32); q += Cfg::NW) {
      const int slot = sOrd[q / (T / 32)], i = (q % (T / 32)) * 32 + lane;
      const ShellRec sh = sSh[slot];
      const double dx = sx[i] - sh.x, dy = sy[i] - sh.y, dz = sz[i] - sh.z;
      const double r2 = dx * dx + dy * dy + dz * dz;
      const double2* pr = sPrim + sh.prim_off;
      double R0 = 0.0, R1 = 0.0;
      for (int k = 0; k < sh.nprim; ++k) {
        const double2 ad = pr[k];
        const double arg = ad.x * r2;
        if (arg < 708.0) {                     // beyond, exp(-arg) < 3.3e-308: dropped (it cannot change any result)
#ifdef XC_EXP_STUB
          const double ev = ad.y * (1.0 - 1e-3 * arg);
#else
          const double ev = ad.y * exp_neg(arg, sExpT);
#endif
          R0 += ev;
          R1 = fma(-2.0 * ad.x, ev, R1);
        }
      }
      if (GGA) *reinterpret_cast<double2*>(sR + ((size_t)slot * T + i) * 2) = make_double2(R0, R1);
      double* dst = sPhi + (size_t)sh._pad * LD + i;
      if (sh.L == 0) {
        dst[0] = R0;
      } else if (sh.L == 1) {
        dst[0] = dx * R0; dst[LD] = dy * R0; dst[2 * LD] = dz * R0;
      } else {
        const double xr = dx * R0, yr = dy * R0;
        dst[0] = dx * xr; dst[LD] = dy * xr; dst[2 * LD] = dz * xr;
        dst[3 * LD] = dy * yr; dst[4 * LD] = dz * yr; dst[5 * LD] = dz * dz * R0;
      }
    }
    __syncthreads();
    PH(2);

    // ---- 2. X^T = Phi^T P^j and the density reductions ----
    {
      double C[2][NTW][2];
#pragma unroll
      for (int u = 0; u < 2; ++u)
#pragma unroll
        for (int v = 0; v < NTW; ++v) C[u][v][0] = C[u][v][1] = 0.0;
      const double* Ap = sPhi + (size_t)t4 * LD + wp * 16 + g4;
      const double* Bp = ppk + (size_t)wm * 32 + lane;
      // number of mu-tiles of this warp (warp-uniform): one fully unrolled loop per count, so that no DMMA is
      // ever issued predicated-off (a predicated-off DMMA still takes its slot in the FP64 tensor pipe)
      const int nv = wm < ntile ? min(NTW, (ntile - wm + Cfg::WM - 1) / Cfg::WM) : 0;
      if (GGA) {
        switch (nv) {
          case 1: xgemm_tile<1, NTW, Cfg::WM * 32>(C, Ap, Bp, nks, 4 * LD, ntile * 32); break;
          case 2: xgemm_tile<(NTW >= 2 ? 2 : 1), NTW, Cfg::WM * 32>(C, Ap, Bp, nks, 4 * LD, ntile * 32); break;
          case 3: xgemm_tile<(NTW >= 3 ? 3 : 1), NTW, Cfg::WM * 32>(C, Ap, Bp, nks, 4 * LD, ntile * 32); break;
          case 4: xgemm_tile<(NTW >= 4 ? 4 : 1), NTW, Cfg::WM * 32>(C, Ap, Bp, nks, 4 * LD, ntile * 32); break;
          default: break;
        }
      } else {                                 // LDA: lower triangle only, rho = 2 Phi . (L Phi)
        switch (nv) {
          case 1: xgemm_tri<1, NTW, Cfg::WM * 32>(C, Ap, Bp, nks, wm, Cfg::WM, 4 * LD, ntile * 32); break;
          case 2: xgemm_tri<(NTW >= 2 ? 2 : 1), NTW, Cfg::WM * 32>(C, Ap, Bp, nks, wm, Cfg::WM, 4 * LD, ntile * 32); break;
          case 3: xgemm_tri<(NTW >= 3 ? 3 : 1), NTW, Cfg::WM * 32>(C, Ap, Bp, nks, wm, Cfg::WM, 4 * LD, ntile * 32); break;
          case 4: xgemm_tri<(NTW >= 4 ? 4 : 1), NTW, Cfg::WM * 32>(C, Ap, Bp, nks, wm, Cfg::WM, 4 * LD, ntile * 32); break;
          default: break;
        }
      }
      if (GGA) {
        // X^T -> shared memory (the Z buffer, [mu][i]); rows >= nb receive exact zeros (zero padding of the packed P^j)
#pragma unroll
        for (int v = 0; v < NTW; ++v) {
          if (v < nv) {
#pragma unroll
            for (int u = 0; u < 2; ++u)
#pragma unroll
              for (int h = 0; h < 2; ++h)
                sZ[(size_t)((wm + v * Cfg::WM) * 8 + t4 * 2 + h) * LD + wp * 16 + u * 8 + g4] = C[u][v][h];
          }
        }
      } else {
        // epilogue: Eq. (13)
        double rho_acc[2] = {0.0, 0.0};
#pragma unroll
        for (int u = 0; u < 2; ++u) {
          const int i = wp * 16 + u * 8 + g4;
#pragma unroll
          for (int v = 0; v < NTW; ++v) {
            if (v < nv) {
#pragma unroll
              for (int h = 0; h < 2; ++h) {
                const int mu = (wm + v * Cfg::WM) * 8 + t4 * 2 + h;    // rows >= nb of sPhi are zero
                rho_acc[u] = fma(sPhi[(size_t)mu * LD + i], C[u][v][h], rho_acc[u]);
              }
            }
          }
        }
        // reduce over the 4 lanes sharing a point, then over the WM warps (fixed order => deterministic)
#pragma unroll
        for (int u = 0; u < 2; ++u) {
          rho_acc[u] += __shfl_xor_sync(0xffffffffu, rho_acc[u], 1);
          rho_acc[u] += __shfl_xor_sync(0xffffffffu, rho_acc[u], 2);
          if (t4 == 0) sRed[(size_t)(wm * 4) * T + wp * 16 + u * 8 + g4] = rho_acc[u];
        }
      }
    }
    __syncthreads();
    if (GGA) {
      // density pass per (shell, point): thread = (group, point); a group walks over the shells group, group + NG, ...
      const int i = tid % T, grp = tid / T;
      const double xi = sx[i], yi = sy[i], zi = sz[i];
      double rho = 0.0, gx = 0.0, gy = 0.0, gz = 0.0;
      for (int slot = grp; slot < ns; slot += Cfg::NG) {
        const ShellRec sh = sSh[slot];
        const double dx = xi - sh.x, dy = yi - sh.y, dz = zi - sh.z;
        const double2 R = *reinterpret_cast<const double2*>(sR + ((size_t)slot * T + i) * 2);
        const double* xp = sZ + (size_t)sh._pad * LD + i;
        double S0, Gx, Gy, Gz;
        if (sh.L == 0) {
          S0 = xp[0]; Gx = Gy = Gz = 0.0;
        } else if (sh.L == 1) {
          Gx = xp[0]; Gy = xp[LD]; Gz = xp[2 * LD];
          S0 = fma(Gx, dx, fma(Gy, dy, Gz * dz));
        } else {
          const double Xxx = xp[0], Xxy = xp[LD], Xxz = xp[2 * LD], Xyy = xp[3 * LD], Xyz = xp[4 * LD], Xzz = xp[5 * LD];
          Gx = fma(2.0 * Xxx, dx, fma(Xxy, dy, Xxz * dz));
          Gy = fma(Xxy, dx, fma(2.0 * Xyy, dy, Xyz * dz));
          Gz = fma(Xxz, dx, fma(Xyz, dy, 2.0 * Xzz * dz));
          S0 = 0.5 * fma(Gx, dx, fma(Gy, dy, Gz * dz));
        }
        rho = fma(R.x, S0, rho);
        const double t = R.y * S0;
        gx = fma(R.x, Gx, fma(t, dx, gx));
        gy = fma(R.x, Gy, fma(t, dy, gy));
        gz = fma(R.x, Gz, fma(t, dz, gz));
      }
      sRed[(size_t)(grp * 4 + 0) * T + i] = rho;
      sRed[(size_t)(grp * 4 + 1) * T + i] = gx;
      sRed[(size_t)(grp * 4 + 2) * T + i] = gy;
      sRed[(size_t)(grp * 4 + 3) * T + i] = gz;
      __syncthreads();
    }
    PH(3);

    // ---- 3. functional (Eq. (19)), E and N_el partials (Eq. (16)); the warps after the first T threads fetch
    //         the next tile's points into the other buffer ----
    if (tid >= T && tid < 2 * T && t0 + T < nqe) {
      const int li = tid - T, nn = min(T, nqe - t0 - T);
      const int64_t gi = (int64_t)b.pt_off + sLive[t0 + T + min(li, nn - 1)];
      double* nx = sPt + (size_t)((it + 1) & 1) * 4 * T;
      nx[li] = a.px[gi]; nx[T + li] = a.py[gi]; nx[2 * T + li] = a.pz[gi];
      nx[3 * T + li] = li < nn ? a.w[gi] : 0.0;
    }
    if (tid < T) {
      double rho = 0.0, gx = 0.0, gy = 0.0, gz = 0.0;
      for (int q = 0; q < (GGA ? Cfg::NG : Cfg::WM); ++q) {
        rho += sRed[(size_t)(q * 4 + 0) * T + tid];
        if (GGA) {
          gx += sRed[(size_t)(q * 4 + 1) * T + tid];
          gy += sRed[(size_t)(q * 4 + 2) * T + tid];
          gz += sRed[(size_t)(q * 4 + 3) * T + tid];
        }
      }
      if (!GGA) rho *= 2.0;                      // LDA: the X GEMM ran over the lower triangle of P^j (half the diagonal)
      gx *= 2.0; gy *= 2.0; gz *= 2.0;
      const double sigma = gx * gx + gy * gy + gz * gz;
      const double wi = sw[tid];
      double f, vr, vs;
      xc_point<GGA>(rho, sigma, a.rho_tol, f, vr, vs);
      sA[tid] = GGA ? 0.5 * wi * vr : wi * vr;   // LDA: V^j = sum_i (w v_rho)_i Phi_mu,i Phi_nu,i
      const double gs = 2.0 * wi * vs;
      sG0[tid] = gs * gx; sG1[tid] = gs * gy; sG2[tid] = gs * gz;
      if (tid < npt && a.rho_out) {
        const int64_t gi = (int64_t)b.pt_off + sLive[t0 + tid];
        a.rho_out[gi] = rho;
        if (a.grho_out) { a.grho_out[3 * gi] = gx; a.grho_out[3 * gi + 1] = gy; a.grho_out[3 * gi + 2] = gz; }
      }
      double e = wi * f, n = wi * rho;
#pragma unroll
      for (int o = 16; o >= 1; o >>= 1) {
        e += __shfl_xor_sync(0xffffffffu, e, o);
        n += __shfl_xor_sync(0xffffffffu, n, o);
      }
      if (lane == 0) { sE[warp] = e; sN[warp] = n; }
    }
    __syncthreads();
    PH(4);
    if (tid == 0) {
      for (int q = 0; q < T / 32; ++q) { Eacc += sE[q]; Nacc += sN[q]; }
    }

    // ---- 4. GGA: Z (Eq. (20)) per (shell, point); overwrites X^T ----
    if (GGA) {
      const int i = tid % T, grp = tid / T;
      const double xi = sx[i], yi = sy[i], zi = sz[i];
      const double ai = sA[i], g0 = sG0[i], g1 = sG1[i], g2 = sG2[i];
      for (int slot = grp; slot < ns; slot += Cfg::NG) {
        const ShellRec sh = sSh[slot];
        const double dx = xi - sh.x, dy = yi - sh.y, dz = zi - sh.z;
        const double2 R = *reinterpret_cast<const double2*>(sR + ((size_t)slot * T + i) * 2);
        const double base = fma(ai, R.x, R.y * fma(g0, dx, fma(g1, dy, g2 * dz)));   // a R0 + R1 g.(r - R)
        double* zp = sZ + (size_t)sh._pad * LD + i;
        if (sh.L == 0) {
          zp[0] = base;
        } else if (sh.L == 1) {
          zp[0] = fma(dx, base, R.x * g0); zp[LD] = fma(dy, base, R.x * g1); zp[2 * LD] = fma(dz, base, R.x * g2);
        } else {
          const double bx = dx * base, by = dy * base;
          const double r0 = R.x;
          zp[0] = fma(dx, bx, 2.0 * r0 * dx * g0);
          zp[LD] = fma(dy, bx, r0 * fma(dy, g0, dx * g1));
          zp[2 * LD] = fma(dz, bx, r0 * fma(dz, g0, dx * g2));
          zp[3 * LD] = fma(dy, by, 2.0 * r0 * dy * g1);
          zp[4 * LD] = fma(dz, by, r0 * fma(dz, g1, dy * g2));
          zp[5 * LD] = fma(dz * dz, base, 2.0 * r0 * dz * g2);
        }
      }
      __syncthreads();
      PH(5);
    }

    // ---- 5. V^j += Z Phi^T + Phi Z^T (lower-triangle 16x16 blocks; Eq. (18)) ----
    // block by block (one block's fragment addresses live at a time), all T/4 k-steps of the tile per block
#pragma unroll
    for (int r = 0; r < ROUNDS; ++r) {
      if (blk_m[r] < 0) continue;
      const int om = (blk_m[r] * 16 + g4) * LD + t4, on = (blk_n[r] * 16 + g4) * LD + t4;
      const bool diag = blk_m[r] == blk_n[r];
      if (GGA) {
#pragma unroll 4
        for (int kk = 0; kk < T / 4; ++kk) {
          const double Pm0 = sPhi[om + 4 * kk], Pm1 = sPhi[om + 8 * LD + 4 * kk], Zm0 = sZ[om + 4 * kk], Zm1 = sZ[om + 8 * LD + 4 * kk];
          const double Pn0 = sPhi[on + 4 * kk], Pn1 = sPhi[on + 8 * LD + 4 * kk], Zn0 = sZ[on + 4 * kk], Zn1 = sZ[on + 8 * LD + 4 * kk];
          dmma884(V[r][0][0][0], V[r][0][0][1], Zm0, Pn0); dmma884(V[r][0][0][0], V[r][0][0][1], Pm0, Zn0);
          dmma884(V[r][1][0][0], V[r][1][0][1], Zm1, Pn0); dmma884(V[r][1][0][0], V[r][1][0][1], Pm1, Zn0);
          dmma884(V[r][1][1][0], V[r][1][1][1], Zm1, Pn1); dmma884(V[r][1][1][0], V[r][1][1][1], Pm1, Zn1);
          if (!diag) { dmma884(V[r][0][1][0], V[r][0][1][1], Zm0, Pn1); dmma884(V[r][0][1][0], V[r][0][1][1], Pm0, Zn1); }
        }
      } else {
#pragma unroll 4
        for (int kk = 0; kk < T / 4; ++kk) {
          const double ai = sA[4 * kk + t4];
          const double Pm0 = sPhi[om + 4 * kk], Pm1 = sPhi[om + 8 * LD + 4 * kk];
          const double Pn0 = sPhi[on + 4 * kk], Pn1 = sPhi[on + 8 * LD + 4 * kk];
          const double Zm0 = ai * Pm0, Zm1 = ai * Pm1;
          dmma884(V[r][0][0][0], V[r][0][0][1], Zm0, Pn0);
          dmma884(V[r][1][0][0], V[r][1][0][1], Zm1, Pn0);
          dmma884(V[r][1][1][0], V[r][1][1][1], Zm1, Pn1);
          if (!diag) dmma884(V[r][0][1][0], V[r][0][1][1], Zm0, Pn1);
        }
      }
    }
    PH(6);
  }

  PH(7);
  // ---- 6. increment of V (Eq. (17)), lower triangle; global indices ascend with local ones ----
  if (tid == 0) { a.Epart[bidx] = Eacc; a.Npart[bidx] = Nacc; }
#pragma unroll
  for (int r = 0; r < ROUNDS; ++r) {
    if (blk_m[r] < 0) continue;
#pragma unroll
    for (int u = 0; u < 2; ++u) {
      const int mu = blk_m[r] * 16 + u * 8 + g4;
      if (mu >= nb) continue;
      const size_t row = (size_t)sIdx[mu] * a.nbasis;
#pragma unroll
      for (int v = 0; v < 2; ++v)
#pragma unroll
        for (int h = 0; h < 2; ++h) {
          const int nu = blk_n[r] * 16 + v * 8 + t4 * 2 + h;
          if (nu <= mu) {
            const size_t o = row + sIdx[nu];
            fixed_add(a.vhi + o, a.vlo + o, V[r][u][v][h]);
          }
        }
    }
  }
  PH(8);
}

// fixed point -> fp64, mirrored.  32x32 tiles, tm >= tn.
__global__ void __launch_bounds__(256) k_finalize(int nbasis, const unsigned long long* __restrict__ vhi,
                                                  const unsigned long long* __restrict__ vlo, double* __restrict__ V,
                                                  int64_t ldv) {
  __shared__ double tile[32][33];
  // decode the linear lower-triangle tile index
  int t = blockIdx.x;
  int tm = (int)((sqrt(8.0 * t + 1.0) - 1.0) * 0.5);
  while ((tm + 1) * (tm + 2) / 2 <= t) ++tm;
  while (tm * (tm + 1) / 2 > t) --tm;
  int tn = t - tm * (tm + 1) / 2;
  const int tx = threadIdx.x & 31, ty = threadIdx.x >> 5;
  for (int r = ty; r < 32; r += 8) {
    int mu = tm * 32 + r, nu = tn * 32 + tx;
    double v = 0.0;
    if (mu < nbasis && nu < nbasis && nu <= mu) {
      size_t o = (size_t)mu * nbasis + nu;
      long long h = (long long)vhi[o];
      unsigned long long l = vlo[o];
      // value = (h * 2^32 + l) * 2^-64
      v = (double)h * 2.3283064365386962890625e-10 + (double)l * 5.42101086242752217003726400434970855712890625e-20;
      V[(size_t)mu * ldv + nu] = v;
    }
    tile[r][tx] = v;
  }
  __syncthreads();
  for (int r = ty; r < 32; r += 8) {
    int nu = tn * 32 + r, mu = tm * 32 + tx;   // write V[nu][mu] = tile[mu_local][nu_local]
    if (mu < nbasis && nu < nbasis && nu < mu) V[(size_t)nu * ldv + mu] = tile[tx][r];
  }
}

// deterministic sum of the per-tile partials: one block, fixed strided order then a fixed tree
__global__ void __launch_bounds__(1024) k_reduce2(int64_t n, const double* __restrict__ ep, const double* __restrict__ np,
                                                  double* __restrict__ out) {
  __shared__ double se[1024], sn[1024];
  double e = 0.0, m = 0.0;
  for (int64_t i = threadIdx.x; i < n; i += 1024) { e += ep[i]; m += np[i]; }
  se[threadIdx.x] = e; sn[threadIdx.x] = m;
  __syncthreads();
  for (int s = 512; s >= 1; s >>= 1) {
    if ((int)threadIdx.x < s) { se[threadIdx.x] += se[threadIdx.x + s]; sn[threadIdx.x] += sn[threadIdx.x + s]; }
    __syncthreads();
  }
  if (threadIdx.x == 0) { out[0] = se[0]; out[1] = sn[0]; }
}

// ------------------------------------------------------------------------------------------------
// launchers
// ------------------------------------------------------------------------------------------------
cudaError_t launch_weights(int partition, int natoms, const double* atoms, const double* invR, const double* rnn,
                           int64_t npts, const double* px, const double* py, const double* pz, const double* wq,
                           const int32_t* parent, double* w, cudaStream_t st) {
  if (npts <= 0) return cudaSuccess;
  unsigned grid = (unsigned)((npts + 127) / 128);
  if (partition == 0) k_weights<0><<<grid, 128, 0, st>>>(natoms, atoms, invR, rnn, npts, px, py, pz, wq, parent, w);
  else k_weights<1><<<grid, 128, 0, st>>>(natoms, atoms, invR, rnn, npts, px, py, pz, wq, parent, w);
  return cudaGetLastError();
}

cudaError_t launch_weights_batched(int partition, const WeightArgs& a, const int32_t* batch_ids, int nbatches, int nwarps,
                                   int max_list, cudaStream_t st) {
  if (nbatches <= 0) return cudaSuccess;
  size_t smem = weights_smem_bytes(max_list, nwarps);
  cudaError_t e;
  if (partition == 0) {
    // shared-memory split: the whole atom list if it fits (28 B per atom), the rest for rows of the 1/(a R_BC) table
    const int lcap = std::min((max_list + 31) / 32 * 32, kSsfMaxLcap);
    const int tabB = std::min(32, (int)((kSsfSmem - kSsfFixed - (size_t)lcap * 28) / ((size_t)kTabC * 8)));
    e = cudaFuncSetAttribute(k_weights_ssf, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kSsfSmem);
    if (e != cudaSuccess) return e;
    k_weights_ssf<<<nbatches, kSsfThreads, kSsfSmem, st>>>(a, batch_ids, lcap, tabB);
  } else {
    e = cudaFuncSetAttribute(k_weights_batched<1>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)std::max<size_t>(smem, 1024));
    if (e != cudaSuccess) return e;
    k_weights_batched<1><<<nbatches, kWeightThreads, smem, st>>>(a, batch_ids, nwarps);
  }
  return cudaGetLastError();
}

cudaError_t launch_functional(int kind, int64_t n, const double* rho, const double* sigma, double rho_tol, double* f,
                              double* vr, double* vs, cudaStream_t st) {
  if (n <= 0) return cudaSuccess;
  k_functional<<<(unsigned)((n + 255) / 256), 256, 0, st>>>(kind, n, rho, sigma, rho_tol, f, vr, vs);
  return cudaGetLastError();
}

cudaError_t launch_pack(const BatchArgs& a, const int32_t* batch_ids, int nbatches, bool tri, cudaStream_t st) {
  if (nbatches <= 0) return cudaSuccess;
  k_pack_P<<<nbatches, 256, 0, st>>>(a, batch_ids, tri ? 1 : 0);
  return cudaGetLastError();
}

template <int NT, int T, bool GGA, int NTW, int ROUNDS, int MINB>
static cudaError_t launch_batch_t(const BatchArgs& a, const int32_t* batch_ids, int nbatches, size_t smem, cudaStream_t st) {
  cudaError_t e = cudaFuncSetAttribute(k_xc_batch<NT, T, GGA, NTW, ROUNDS, MINB>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
  if (e != cudaSuccess) return e;
  k_xc_batch<NT, T, GGA, NTW, ROUNDS, MINB><<<nbatches, NT, smem, st>>>(a, batch_ids);
  return cudaGetLastError();
}

// cls 0: N_b^j <= kSmallNb, tiles of 64 points; cls 1: N_b^j <= kMaxNb, tiles of 32 points; 16 warps, one CTA per SM
cudaError_t launch_batch(int cls, bool gga, const BatchArgs& a, const int32_t* batch_ids, int nbatches, size_t smem,
                         cudaStream_t st) {
  if (nbatches <= 0) return cudaSuccess;
  if (cls == 0) return gga ? launch_batch_t<512, 64, true, 4, 2, 1>(a, batch_ids, nbatches, smem, st)
                           : launch_batch_t<512, 64, false, 4, 2, 1>(a, batch_ids, nbatches, smem, st);
  return gga ? launch_batch_t<512, 32, true, 3, 5, 1>(a, batch_ids, nbatches, smem, st)
             : launch_batch_t<512, 32, false, 3, 5, 1>(a, batch_ids, nbatches, smem, st);
}

cudaError_t launch_finalize(int nbasis, const unsigned long long* vhi, const unsigned long long* vlo, double* V,
                            int64_t ldv, cudaStream_t st) {
  int nt = (nbasis + 31) / 32;
  k_finalize<<<(unsigned)(nt * (nt + 1) / 2), 256, 0, st>>>(nbasis, vhi, vlo, V, ldv);
  return cudaGetLastError();
}

cudaError_t launch_reduce(int64_t n, const double* ep, const double* np, double* out, cudaStream_t st) {
  k_reduce2<<<1, 1024, 0, st>>>(n, ep, np, out);
  return cudaGetLastError();
}

}  // namespace xcb
