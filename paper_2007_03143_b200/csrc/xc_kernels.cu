// xc_kernels.cu -- CUDA kernels (sm_100a) of libxc_b200: the hot path of Alg. 4.
//
//   (step (a), the partition weights of Eq. (9) PAPER.md:L96 / Alg. 4 l.4.1, lives in xc_weights.cu)
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
#include <cmath>
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

// R0 = sum_k d_k exp(-alpha_k r^2) and R1 = sum_k -2 alpha_k d_k exp(-alpha_k r^2) of one shell (Eq. (7)), the
// primitives three at a time: the three exponentials are independent chains with no branch between them (a collocation
// warp is bound by the latency of its own dependent chain), the sums run in primitive order.  A primitive with
// alpha r^2 >= 708 (exp < 3.3e-308) adds an exact 0: it cannot change any result.  Measured: c4 41.1 -> 40.3 ms; two or six
// at a time are slower, and so is the same code written operation by operation across the three chains.
template <int W>
__device__ __forceinline__ void radial_group(const double2* __restrict__ pr, int& k, int np, double r2,
                                             const double* __restrict__ tab, double& s0, double& s1) {
#pragma unroll 1
  for (; k + W <= np; k += W) {
    double ev[W], al[W];
#pragma unroll
    for (int u = 0; u < W; ++u) {
      const double2 ad = pr[k + u];
      const double arg = ad.x * r2;
      const double e = ad.y * exp_neg(arg, tab);
      al[u] = ad.x;
      ev[u] = __double2hiint(arg) < 0x40862000 ? e : 0.0;   // arg < 708 (arg >= 0: the high word decides; no FP64 compare)
    }
#pragma unroll
    for (int u = 0; u < W; ++u) { s0 += ev[u]; s1 = fma(al[u], ev[u], s1); }
  }
}
__device__ __forceinline__ void radial(const double2* __restrict__ pr, int np, double r2, const double* __restrict__ tab,
                                       double& R0, double& R1) {
  double s0 = 0.0, s1 = 0.0;                   // s1 = sum alpha d exp: the factor -2 is exact, applied once
  int k = 0;
  radial_group<3>(pr, k, np, r2, tab, s0, s1);
  radial_group<1>(pr, k, np, r2, tab, s0, s1);
  R0 = s0;
  R1 = -2.0 * s1;
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
constexpr double kSqrt3 = 1.7320508075688772935274463415058724;
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
  if (rho <= rho_tol) return;              // a NaN density is not skipped: it propagates to E_xc and V
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
// P^j pack (Eq. (12b), Alg. 4 l.4.2): gathers the batch's block of P ONCE per build into the
// DMMA B-fragment order the batch kernel consumes: for k-step ks (4 nu) and column tile nt (8 mu), 32
// contiguous doubles, lane (g4 = lane >> 2, t4 = lane & 3) holding P[nu = 4 ks + t4][mu = 8 nt + g4];
// zero padded to nb4 x nb8.  One warp-wide 256-byte load per fragment in the batch kernel, no index math there.
// ------------------------------------------------------------------------------------------------
// tri (LDA): rho = phi^T P phi = 2 phi^T L phi with L = strict lower triangle of P^j + half its diagonal, so only
// L is packed (entries nu > mu are zero) and the X GEMM skips the k-steps above the diagonal.
__global__ void __launch_bounds__(256) k_pack_P(BatchArgs a, const int32_t* __restrict__ batch_ids, int tri) {
  __shared__ int64_t sRow[kMaxNb];             // row offsets fidx[mu] * ldp
  __shared__ int sCol[kMaxNb];
  const BatchRec b = a.batches[batch_ids[blockIdx.x]];
  const int nb = b.nb, ntile = (nb + 7) >> 3, nks = (nb + 3) >> 2;
  const int32_t* fidx = a.bfidx + b.f_off;
  for (int f = threadIdx.x; f < nb; f += 256) { const int g = fidx[f]; sCol[f] = g; sRow[f] = (int64_t)g * a.ldp; }
  __syncthreads();
  double* out = a.ppk + b.ppk_off;
  const int total = nks * ntile * 32;
  const int lane = threadIdx.x & 31, t4 = lane & 3, g4 = lane >> 2;
  // four fragments in flight per thread (independent loads)
  for (int e0 = threadIdx.x; e0 < total; e0 += 4 * 256) {
    double v[4];
#pragma unroll
    for (int u = 0; u < 4; ++u) {
      const int e = e0 + u * 256, frag = e >> 5;
      const int ks = frag / ntile, nt = frag - ks * ntile;
      const int nu = 4 * ks + t4, mu = 8 * nt + g4;
      v[u] = 0.0;
      if (e < total && nu < nb && mu < nb && !(tri && nu > mu)) v[u] = __ldg(a.P + sRow[mu] + sCol[nu]);   // P symmetric: row mu is read along nu
      if (tri && nu == mu) v[u] *= 0.5;
    }
#pragma unroll
    for (int u = 0; u < 4; ++u) if (e0 + u * 256 < total) out[e0 + u * 256] = v[u];
  }
}

// ------------------------------------------------------------------------------------------------
// exact, order-independent accumulation: 96-bit fixed point (two 64-bit integer atomics) => V is
// bit-identical from run to run whatever the order in which the batches arrive.  An increment v is added as
// round(v 2^(64 - vexp)): resolution 2^(vexp - 64), range |sum| < 2^(vexp + 31).  vexp belongs to the plan
// (xc_api.cu); the kernel reports the largest |v| it met (high word, `vmax`) so that the host can tell whether
// vexp suited this build, and whether some v was not finite (`bad`): neither is ever dropped silently.
// ------------------------------------------------------------------------------------------------
__device__ __forceinline__ void fixed_add(unsigned long long* hi, unsigned long long* lo, double v, int vexp, unsigned& vmax, bool& bad) {
  // x = round(v * 2^(64 - vexp)) as a signed 128-bit integer; lo = low 32 bits, hi = x >> 32
  long long bits = __double_as_longlong(v);
  int eb = (int)((bits >> 52) & 0x7ff);
  unsigned long long man = (unsigned long long)(bits & 0xfffffffffffffLL);
  vmax = max(vmax, (unsigned)(bits >> 32) & 0x7fffffffu);
  if (eb == 0x7ff) { bad = true; return; }
  if (eb) man |= 1ull << 52; else eb = 1;
  int s = eb - 1075 + 64 - vexp;                // x = man * 2^s
  __int128 x;
  if (s > 41) return;                           // |x| >= 2^94: out of range -- vmax tells the host, which repeats the build with a larger vexp
  if (s >= 0) x = (__int128)man << s;
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
// ------------------------------------------------------------------------------------------------
// P^j staging (north_star (d): "P_sub gathered through TMA or shared-memory staging"; PAPER.md:L379-L385 names the P^j
// pack as the paper's own bottleneck).  The packed P^j of the batch is streamed through a ring of kRingStages
// shared-memory slots of G k-steps each (G = BatchRec::ring_g: what the batch's tiles leave of the SM's shared memory) by the bulk asynchronous copy engine (cp.async.bulk, one elected thread),
// each slot guarded by a full / empty mbarrier pair: every fragment crosses L2 -> SM once per tile pass for the whole
// CTA (it used to be fetched by each of the four warps that share a mu-tile, through an L1 that the 200+ KB
// shared-memory carve-out leaves almost empty), the copies run kRingStages - 1 slots ahead of the DMMAs across tile
// boundaries, and the GEMM warps issue no global loads at all.
// ------------------------------------------------------------------------------------------------
__device__ __forceinline__ unsigned smem_u32(const void* p) { return (unsigned)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(unsigned long long* bar, int count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count));
}
__device__ __forceinline__ void mbar_arrive(unsigned long long* bar) {
  asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(unsigned long long* bar, unsigned bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(unsigned long long* bar, unsigned parity) {
  unsigned done = 0;
  for (unsigned spin = 0; !done; ++spin) {
    asm volatile("{\n .reg .pred p;\n mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n selp.u32 %0, 1, 0, p;\n}"
                 : "=r"(done) : "r"(smem_u32(bar)), "r"(parity) : "memory");
    if (spin > (1u << 28)) __trap();           // a copy or an arrival was lost: fail loudly instead of hanging the device
  }
}
__device__ __forceinline__ void bulk_g2s(void* dst, const void* src, unsigned bytes, unsigned long long* bar) {
  asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
               ::"r"(smem_u32(dst)), "l"(src), "r"(bytes), "r"(smem_u32(bar)) : "memory");
}
struct PRing {
  const double* ppk;            // packed P^j of the batch (global)
  double* buf;                  // [kRingStages][G * ntile * 32]
  unsigned long long* full;     // [kRingStages]
  unsigned long long* empty;    // [kRingStages]
  int ntile, nks, G, spp;       // mu-tiles, k-steps, k-steps per stage, stages per pass over P^j (= ceil(nks / G))
  unsigned total;               // stages the whole batch consumes
  unsigned n;                   // next stage this thread consumes (same value in every thread of the CTA)
};
// the elected thread: start the copy of stage number q (P^j k-steps [kb G, ...) of pass q / spp) into its slot
__device__ __forceinline__ void ring_issue(const PRing& r, unsigned q) {
  const int slot = q % kRingStages, kb = (q % r.spp) * r.G;
  const unsigned bytes = (unsigned)(min(r.G, r.nks - kb) * r.ntile) * 256u;
  mbar_expect_tx(r.full + slot, bytes);
  bulk_g2s(r.buf + (size_t)slot * (r.G * r.ntile * 32), r.ppk + (size_t)kb * r.ntile * 32, bytes, r.full + slot);
}

// X^T tile of one warp over one pass of P^j: C[u][v] += A_u(16 points x 4 nu) * B_v(4 nu x 8 mu) over all k-steps; NV
// mu-tiles (compile time: mt0, mt0 + wmstep, ...), A fragments from sPhi, B fragments from the ring.  TRI (LDA): only the
// lower triangle of P^j is packed non-zero, so mu-tile mt skips the k-steps ks >= 2 mt + 2 (warp-uniform branch: a
// predicated-off DMMA would still take its slot in the FP64 tensor pipe).  Every warp of the CTA walks every stage
// (warps without tiles included): the slot is handed back when all NW warps have arrived.
template <int NV, int NTW, bool TRI>
__device__ __forceinline__ void xgemm_ring(double (&C)[2][NTW][2], const double* __restrict__ Ap, int astep, PRing& r, int mt0,
                                           int wmstep, int lane, bool elected) {
  int lim[4];
#pragma unroll
  for (int v = 0; v < 4; ++v) lim[v] = (TRI && v < NV) ? min(r.nks, 2 * (mt0 + v * wmstep) + 2) : r.nks;
  for (int kb = 0; kb < r.nks; kb += r.G) {
    const unsigned q = r.n;
    const int slot = q % kRingStages;
    if (elected) {
      // keep the ring kRingStages - 1 stages ahead: the slot of stage q - 1 is refilled once every warp has left it
      const unsigned nxt = q + kRingStages - 1;
      if (nxt < r.total) {
        if (q >= 1) mbar_wait(r.empty + (q - 1) % kRingStages, ((q - 1) / kRingStages) & 1);
        ring_issue(r, nxt);
      }
    }
    mbar_wait(r.full + slot, (q / kRingStages) & 1);
    const double* Bs = r.buf + (size_t)slot * (r.G * r.ntile * 32) + (size_t)mt0 * 32 + lane;
    const int gend = min(r.G, r.nks - kb);
    for (int g = 0; g < gend; ++g) {
      const int ks = kb + g;
      {
        const double A0 = Ap[0], A1 = Ap[8];
        Ap += astep;
#pragma unroll
        for (int v = 0; v < NV; ++v) {
          if (!TRI || ks < lim[v]) {
            const double Bv = Bs[(size_t)(g * r.ntile + v * wmstep) * 32];
            dmma884(C[0][v][0], C[0][v][1], A0, Bv);
            dmma884(C[1][v][0], C[1][v][1], A1, Bv);
          }
        }
      }
    }
    __syncwarp();
    if (lane == 0) mbar_arrive(r.empty + slot);
    r.n = q + 1;
  }
}

// LDA (and the tau passes): the packed lower triangle is read straight from global memory, one k-step ahead in registers
// and kPfDist k-steps ahead in L1 -- each mu-tile stops at its diagonal, so a ring that every warp has to walk in step would
// make the warps with short k-ranges wait (measured: 7 % slower on c2 than this path).
constexpr int kPfDist = 4;
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

// MODE 0: the fused restricted build (all stages).  The spin-unrestricted build (xc_eval_uks, readings
// A20-A22) runs the same stages as separate passes, once per spin: MODE 1 = stages 1-2 only, rho_s (and grad rho_s) of the
// live points written to rho_out / grho_out; then k_functional_uks couples the spins; MODE 2 = stages 1, 4-6 with the
// per-point coefficients of Z^s read from cA / cG instead of a functional evaluation.  MODE 3 (xc_eval_tau): the meta-GGA
// intermediate tau = 1/2 sum_mu grad Phi_mu . grad X_mu: stages 1-2 once per gradient component with
// d_c Phi in the Phi buffer, tau = sum_c (d_c Phi)^T L (d_c Phi) from the LDA epilogue, written to rho_out.  MODE 4 (restricted
// meta-GGA, reading A23): stages 1, 5, 6 once per gradient component, V^j += sum_i (1/2 w v_tau)_i d_c Phi_mu,i d_c Phi_nu,i
// with the coefficient read from cA, accumulated in the same registers over the three components.
template <int NT, int T, bool GGA, int NTW, int ROUNDS, int MINB, int MODE>
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
  double* sRing = (double*)sp; sp += (size_t)kRingStages * b.ring_g * ntile * 32 * 8;   // P^j staging ring (16-byte aligned)
  double* sExpT = (double*)sp; sp += (size_t)64 * 8;    // 2^(j/64)
  ShellRec* sSh = (ShellRec*)sp; sp += (size_t)ns * sizeof(ShellRec);
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
      if (tid == 0 && MODE == 0) { a.Epart[bidx] = 0.0; a.Npart[bidx] = 0.0; }
      return;
    }
  }

  // ---- per batch: metadata, zero padding rows, V^j block assignment ----
  {
    const int32_t* fidx = a.bfidx + b.f_off;
    for (int k = tid; k < ns; k += NT) {
      ShellRec r = a.shells[a.bshells[b.sh_off + k]];
      r._pad = a.bsfoff[b.sh_off + k];         // first local function of the shell
      r.atom = r.prim_off;                     // global primitive offset (the atom index is not used here)
      sSh[k] = r;
    }
    for (int f = tid; f < nb16; f += NT) {
      sIdx[f] = f < nb ? fidx[f] : 0;
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
  // ---- P^j staging ring: barriers, and the first kRingStages - 1 stages on their way before the first tile ----
  __shared__ __align__(8) unsigned long long sBar[2 * kRingStages];
  PRing ring;
  ring.ppk = a.ppk + b.ppk_off; ring.buf = sRing; ring.full = sBar; ring.empty = sBar + kRingStages;
  ring.ntile = ntile; ring.nks = nks; ring.G = max(1, b.ring_g); ring.spp = (nks + ring.G - 1) / ring.G;
  ring.total = (MODE == 2 || MODE == 4 || !GGA) ? 0u : (unsigned)(((nqe + T - 1) / T) * ring.spp);   // GGA X GEMM only
  ring.n = 0;
  if (MODE != 2 && MODE != 4 && GGA && tid == 0) {
    for (int k = 0; k < kRingStages; ++k) { mbar_init(ring.full + k, 1); mbar_init(ring.empty + k, Cfg::NW); }
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
    for (unsigned q = 0; q < (unsigned)(kRingStages - 1) && q < ring.total; ++q) ring_issue(ring, q);
  }
  const int wp = warp % Cfg::WP, wm = warp / Cfg::WP;
  double Eacc = 0.0, Nacc = 0.0;
  PH_DECL
  PH(0);
  // MODE 4 visits every tile three times (c4 = gradient component), the other modes once
  for (int t0 = 0, it = 0, c4 = 0; t0 < nqe; (MODE == 4 && c4 < 2) ? (void)++c4 : (void)(c4 = 0, t0 += T, ++it)) {
    const int npt = min(T, nqe - t0);          // valid points in this tile
    const double* sx = sPt + (size_t)(it & 1) * 4 * T;   // this tile's points (written one tile ahead)
    const double *sy = sx + T, *sz = sx + 2 * T, *sw = sx + 3 * T;
    __syncthreads();                           // previous tile's readers of sPhi / sZ are done; tables / points visible
    PH(1);

    double tau_acc = 0.0;                        // MODE 3: tau of this thread's point
    for (int comp = 0; comp < (MODE == 3 ? 3 : 1); ++comp) {   // MODE 3: one pass per gradient component
    // ---- 1. collocation (Eq. (7); same shell across a warp) ----
    for (int q = warp; q < ns * (T / 32); q += Cfg::NW) {
      const int slot = sOrd[q / (T / 32)], i = (q % (T / 32)) * 32 + lane;
      const ShellRec sh = sSh[slot];
      const double dx = sx[i] - sh.x, dy = sy[i] - sh.y, dz = sz[i] - sh.z;
      const double r2 = dx * dx + dy * dy + dz * dz;
      const double2* pr = sPrim + sh.prim_off;
      double R0, R1;
      radial(pr, sh.nprim, r2, sExpT, R0, R1);
      if (GGA) *reinterpret_cast<double2*>(sR + ((size_t)slot * T + i) * 2) = make_double2(R0, R1);
      double* dst = sPhi + (size_t)sh._pad * LD + i;
      if (MODE == 3 || MODE == 4) {
        // d/dr_c of the shell's functions: d_c (m R0) = (d_c m) R0 + m (r - R)_c R1
        const int dcomp = MODE == 4 ? c4 : comp;
        const double dc = dcomp == 0 ? dx : (dcomp == 1 ? dy : dz);
        const double base = dc * R1;
        const double ex = dcomp == 0 ? R0 : 0.0, ey = dcomp == 1 ? R0 : 0.0, ez = dcomp == 2 ? R0 : 0.0;   // R0 d(r - R)_k / dr_c
        if (sh.L == 0) {
          dst[0] = base;
        } else if (sh.L == 1) {
          dst[0] = fma(dx, base, ex); dst[LD] = fma(dy, base, ey); dst[2 * LD] = fma(dz, base, ez);
        } else {
          const double bx = dx * base, by = dy * base;
          const double Dxx = fma(dx, bx, 2.0 * dx * ex), Dxy = fma(dy, bx, fma(dy, ex, dx * ey)), Dxz = fma(dz, bx, fma(dz, ex, dx * ez));
          const double Dyy = fma(dy, by, 2.0 * dy * ey), Dyz = fma(dz, by, fma(dz, ey, dy * ez)), Dzz = fma(dz * dz, base, 2.0 * dz * ez);
          if (sh.L == 2) {
            dst[0] = Dxx; dst[LD] = Dxy; dst[2 * LD] = Dxz; dst[3 * LD] = Dyy; dst[4 * LD] = Dyz; dst[5 * LD] = Dzz;
          } else {
            dst[0] = kSqrt3 * Dxy; dst[LD] = kSqrt3 * Dyz; dst[2 * LD] = Dzz - 0.5 * (Dxx + Dyy);
            dst[3 * LD] = kSqrt3 * Dxz; dst[4 * LD] = (0.5 * kSqrt3) * (Dxx - Dyy);
          }
        }
      } else if (sh.L == 0) {
        dst[0] = R0;
      } else if (sh.L == 1) {
        dst[0] = dx * R0; dst[LD] = dy * R0; dst[2 * LD] = dz * R0;
      } else if (sh.L == 2) {
        const double xr = dx * R0, yr = dy * R0;
        dst[0] = dx * xr; dst[LD] = dy * xr; dst[2 * LD] = dz * xr;
        dst[3 * LD] = dy * yr; dst[4 * LD] = dz * yr; dst[5 * LD] = dz * dz * R0;
      } else {
        // pure d (reading A19), m = -2..2: sqrt3 xy, sqrt3 yz, zz - (xx + yy)/2, sqrt3 xz, (sqrt3/2)(xx - yy)
        const double xr = dx * R0, yr = dy * R0, zr = dz * R0;
        dst[0] = kSqrt3 * dy * xr; dst[LD] = kSqrt3 * dz * yr; dst[2 * LD] = fma(dz, zr, -0.5 * fma(dx, xr, dy * yr));
        dst[3 * LD] = kSqrt3 * dz * xr; dst[4 * LD] = (0.5 * kSqrt3) * fma(dx, xr, -dy * yr);
      }
    }
    __syncthreads();
    PH(2);

    // ---- 2. X^T = Phi^T P^j and the density reductions ----
    if (MODE != 2 && MODE != 4) {
      double C[2][NTW][2];
#pragma unroll
      for (int u = 0; u < 2; ++u)
#pragma unroll
        for (int v = 0; v < NTW; ++v) C[u][v][0] = C[u][v][1] = 0.0;
      const double* Ap = sPhi + (size_t)t4 * LD + wp * 16 + g4;
      // number of mu-tiles of this warp (warp-uniform): one fully unrolled loop per count
      const int nv = wm < ntile ? min(NTW, (ntile - wm + Cfg::WM - 1) / Cfg::WM) : 0;
      if (GGA) {
        const bool elected = tid == 0;
        switch (nv) {
          case 1: xgemm_ring<1, NTW, false>(C, Ap, 4 * LD, ring, wm, Cfg::WM, lane, elected); break;
          case 2: xgemm_ring<(NTW >= 2 ? 2 : 1), NTW, false>(C, Ap, 4 * LD, ring, wm, Cfg::WM, lane, elected); break;
          case 3: xgemm_ring<(NTW >= 3 ? 3 : 1), NTW, false>(C, Ap, 4 * LD, ring, wm, Cfg::WM, lane, elected); break;
          case 4: xgemm_ring<(NTW >= 4 ? 4 : 1), NTW, false>(C, Ap, 4 * LD, ring, wm, Cfg::WM, lane, elected); break;
          default: xgemm_ring<0, NTW, false>(C, Ap, 4 * LD, ring, 0, Cfg::WM, lane, elected); break;   // no tile: walk the stages
        }
      } else {                                 // LDA: lower triangle only, rho = 2 Phi . (L Phi)
        const double* Bp = ring.ppk + (size_t)wm * 32 + lane;
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
    if (MODE != 2 && MODE != 4) __syncthreads();
    if (MODE == 3 && tid < T) {                  // (grad_c Phi)^T L (grad_c Phi) = 1/2 (grad_c Phi)^T P (grad_c Phi): tau's share
      for (int q = 0; q < Cfg::WM; ++q) tau_acc += sRed[(size_t)(q * 4) * T + tid];
    }
    }                                            // component loop (one pass unless MODE 3)
    if (GGA && MODE != 2 && MODE != 4) {
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
          double Xxx, Xxy, Xxz, Xyy, Xyz, Xzz;
          if (sh.L == 2) {
            Xxx = xp[0]; Xxy = xp[LD]; Xxz = xp[2 * LD]; Xyy = xp[3 * LD]; Xyz = xp[4 * LD]; Xzz = xp[5 * LD];
          } else {
            // pure d: sum_q X_q d_q = sum_c (T^T X)_c (Cartesian d)_c
            const double X0 = xp[0], X1 = xp[LD], X2 = xp[2 * LD], X3 = xp[3 * LD], X4 = xp[4 * LD];
            Xxx = fma(0.5 * kSqrt3, X4, -0.5 * X2); Xyy = fma(-0.5 * kSqrt3, X4, -0.5 * X2); Xzz = X2;
            Xxy = kSqrt3 * X0; Xyz = kSqrt3 * X1; Xxz = kSqrt3 * X3;
          }
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
    if (tid < T && (MODE == 2 || MODE == 4)) {
      // per-point coefficients of Z^s from the functional kernel: a (LDA: w v_rho_s; GGA: 1/2 w v_rho_s), g (GGA)
      const int64_t gi = (int64_t)b.pt_off + sLive[t0 + min(tid, npt - 1)];
      const bool ok = tid < npt;
      sA[tid] = ok ? a.cA[gi] : 0.0;
      if (GGA) { sG0[tid] = ok ? a.cG[3 * gi] : 0.0; sG1[tid] = ok ? a.cG[3 * gi + 1] : 0.0; sG2[tid] = ok ? a.cG[3 * gi + 2] : 0.0; }
    }
    if (tid < T && MODE != 2 && MODE != 4) {
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
      if (MODE == 3) {                           // tau_s = 1/2 sum_mu grad Phi . grad X^s, to rho_out
        if (tid < npt) a.rho_out[(int64_t)b.pt_off + sLive[t0 + tid]] = tau_acc;
      } else if (MODE == 1) {
        if (tid < npt) {
          const int64_t gi = (int64_t)b.pt_off + sLive[t0 + tid];
          a.rho_out[gi] = rho;
          if (GGA) { a.grho_out[3 * gi] = gx; a.grho_out[3 * gi + 1] = gy; a.grho_out[3 * gi + 2] = gz; }
        }
      } else {
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
    }
    __syncthreads();
    PH(4);
    if (tid == 0 && MODE == 0) {
      for (int q = 0; q < T / 32; ++q) { Eacc += sE[q]; Nacc += sN[q]; }
    }
    if (MODE == 1 || MODE == 3) continue;        // densities only: next tile (the barrier at the top of the loop orders the buffers)

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
          const double Zxx = fma(dx, bx, 2.0 * r0 * dx * g0);
          const double Zxy = fma(dy, bx, r0 * fma(dy, g0, dx * g1));
          const double Zxz = fma(dz, bx, r0 * fma(dz, g0, dx * g2));
          const double Zyy = fma(dy, by, 2.0 * r0 * dy * g1);
          const double Zyz = fma(dz, by, r0 * fma(dz, g1, dy * g2));
          const double Zzz = fma(dz * dz, base, 2.0 * r0 * dz * g2);
          if (sh.L == 2) {
            zp[0] = Zxx; zp[LD] = Zxy; zp[2 * LD] = Zxz; zp[3 * LD] = Zyy; zp[4 * LD] = Zyz; zp[5 * LD] = Zzz;
          } else {                                  // pure d: Z_q = sum_c T_qc (Cartesian Z)_c
            zp[0] = kSqrt3 * Zxy; zp[LD] = kSqrt3 * Zyz; zp[2 * LD] = Zzz - 0.5 * (Zxx + Zyy);
            zp[3 * LD] = kSqrt3 * Zxz; zp[4 * LD] = (0.5 * kSqrt3) * (Zxx - Zyy);
          }
        }
      }
      __syncthreads();
      PH(5);
    }

    // ---- 5. V^j += Z Phi^T + Phi Z^T (lower-triangle 16x16 blocks; Eq. (18)) ----
    // block by block (one block's fragment addresses live at a time), all k-steps of the tile per block; the last tile of a
    // batch stops at its last point (columns past npt hold zeros: they would add nothing)
    const int kkn = (npt + 3) >> 2;
#pragma unroll
    for (int r = 0; r < ROUNDS; ++r) {
      if (blk_m[r] < 0) continue;
      const int om = (blk_m[r] * 16 + g4) * LD + t4, on = (blk_n[r] * 16 + g4) * LD + t4;
      const bool diag = blk_m[r] == blk_n[r];
      if (GGA) {
#pragma unroll 4
        for (int kk = 0; kk < kkn; ++kk) {
          const double Pm0 = sPhi[om + 4 * kk], Pm1 = sPhi[om + 8 * LD + 4 * kk], Zm0 = sZ[om + 4 * kk], Zm1 = sZ[om + 8 * LD + 4 * kk];
          const double Pn0 = sPhi[on + 4 * kk], Pn1 = sPhi[on + 8 * LD + 4 * kk], Zn0 = sZ[on + 4 * kk], Zn1 = sZ[on + 8 * LD + 4 * kk];
          // the two DMMAs of one accumulator are kept apart (a dependent DMMA waits for the result of the one before)
          dmma884(V[r][0][0][0], V[r][0][0][1], Zm0, Pn0);
          dmma884(V[r][1][0][0], V[r][1][0][1], Zm1, Pn0);
          dmma884(V[r][1][1][0], V[r][1][1][1], Zm1, Pn1);
          if (!diag) dmma884(V[r][0][1][0], V[r][0][1][1], Zm0, Pn1);
          dmma884(V[r][0][0][0], V[r][0][0][1], Pm0, Zn0);
          dmma884(V[r][1][0][0], V[r][1][0][1], Pm1, Zn0);
          dmma884(V[r][1][1][0], V[r][1][1][1], Pm1, Zn1);
          if (!diag) dmma884(V[r][0][1][0], V[r][0][1][1], Pm0, Zn1);
        }
      } else {
#pragma unroll 4
        for (int kk = 0; kk < kkn; ++kk) {
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
  if (MODE == 1 || MODE == 3) return;
  if (tid == 0 && MODE == 0) { a.Epart[bidx] = Eacc; a.Npart[bidx] = Nacc; }
  unsigned vmax = 0;
  bool bad = false;
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
            fixed_add(a.vhi + o, a.vlo + o, V[r][u][v][h], a.vexp, vmax, bad);
          }
        }
    }
  }
  vmax = __reduce_max_sync(0xffffffffu, vmax);
  bad = __any_sync(0xffffffffu, bad);
  if (lane == 0) {
    if (vmax) atomicMax(a.vflags, vmax);
    if (bad) atomicOr(a.vflags + 1, 1u);
  }
  PH(8);
}

// fixed point -> fp64, mirrored.  32x32 tiles, tm >= tn.  value = (hi 2^32 + lo) 2^(vexp - 64); poison: NaN everywhere.
__global__ void __launch_bounds__(256) k_finalize(int nbasis, const unsigned long long* __restrict__ vhi,
                                                  const unsigned long long* __restrict__ vlo, double* __restrict__ V,
                                                  int64_t ldv, double shi, double slo, int poison) {
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
      v = poison ? __longlong_as_double(0x7ff8000000000000LL) : (double)h * shi + (double)l * slo;
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

template <int NT, int T, bool GGA, int NTW, int ROUNDS, int MINB, int MODE>
static cudaError_t launch_batch_t(const BatchArgs& a, const int32_t* batch_ids, int nbatches, size_t smem, cudaStream_t st) {
  cudaError_t e = cudaFuncSetAttribute(k_xc_batch<NT, T, GGA, NTW, ROUNDS, MINB, MODE>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
  if (e != cudaSuccess) return e;
  k_xc_batch<NT, T, GGA, NTW, ROUNDS, MINB, MODE><<<nbatches, NT, smem, st>>>(a, batch_ids);
  return cudaGetLastError();
}
// one class of batches; cls 0: T = 64, two rounds of V^j blocks; cls 1: T = 32, three rounds (N_b^j <= kMidNb); cls 2: T = 32, five
template <int MODE, bool GGA>
static cudaError_t launch_batch_c(int cls, const BatchArgs& a, const int32_t* batch_ids, int nbatches, size_t smem, cudaStream_t st) {
  if (cls == 0) return launch_batch_t<512, 64, GGA, 4, 2, 1, MODE>(a, batch_ids, nbatches, smem, st);
  if (cls == 1) return launch_batch_t<512, 32, GGA, 3, 3, 1, MODE>(a, batch_ids, nbatches, smem, st);
  return launch_batch_t<512, 32, GGA, 3, 5, 1, MODE>(a, batch_ids, nbatches, smem, st);
}
static cudaError_t launch_batch_1(int cls, bool gga, int mode, const BatchArgs& a, const int32_t* batch_ids, int nbatches, size_t smem,
                                  cudaStream_t st) {
  switch (mode) {
    case 1: return gga ? launch_batch_c<1, true>(cls, a, batch_ids, nbatches, smem, st) : launch_batch_c<1, false>(cls, a, batch_ids, nbatches, smem, st);
    case 2: return gga ? launch_batch_c<2, true>(cls, a, batch_ids, nbatches, smem, st) : launch_batch_c<2, false>(cls, a, batch_ids, nbatches, smem, st);
    // tau (3) and the tau term of a meta-GGA potential (4) run the LDA GEMMs per gradient component, whatever the plan's functional
    case 3: return launch_batch_c<3, false>(cls, a, batch_ids, nbatches, smem, st);
    case 4: return launch_batch_c<4, false>(cls, a, batch_ids, nbatches, smem, st);
    default: return gga ? launch_batch_c<0, true>(cls, a, batch_ids, nbatches, smem, st) : launch_batch_c<0, false>(cls, a, batch_ids, nbatches, smem, st);
  }
}

cudaError_t launch_batch(int cls, bool gga, int mode, const BatchArgs& a, const int32_t* batch_ids, int nbatches, size_t smem,
                         cudaStream_t st, int n_heavy, int* launched) {
  if (launched) *launched = 0;
  if (nbatches <= 0) return cudaSuccess;
  if (cls == 0) {
    if (launched) *launched = 1;
    return launch_batch_1(0, gga, mode, a, batch_ids, nbatches, smem, st);
  }
  n_heavy = n_heavy < 0 ? 0 : (n_heavy > nbatches ? nbatches : n_heavy);
  if (n_heavy > 0) {
    const cudaError_t e = launch_batch_1(2, gga, mode, a, batch_ids, n_heavy, smem, st);
    if (e != cudaSuccess) return e;
    if (launched) ++*launched;
  }
  if (n_heavy < nbatches) {
    const cudaError_t e = launch_batch_1(1, gga, mode, a, batch_ids + n_heavy, nbatches - n_heavy, smem, st);
    if (e != cudaSuccess) return e;
    if (launched) ++*launched;
  }
  return cudaSuccess;
}

cudaError_t launch_finalize(int nbasis, const unsigned long long* vhi, const unsigned long long* vlo, double* V,
                            int64_t ldv, int vexp, bool poison, cudaStream_t st) {
  int nt = (nbasis + 31) / 32;
  k_finalize<<<(unsigned)(nt * (nt + 1) / 2), 256, 0, st>>>(nbasis, vhi, vlo, V, ldv, std::ldexp(1.0, vexp - 32), std::ldexp(1.0, vexp - 64), poison ? 1 : 0);
  return cudaGetLastError();
}

cudaError_t launch_reduce(int64_t n, const double* ep, const double* np, double* out, cudaStream_t st) {
  k_reduce2<<<1, 1024, 0, st>>>(n, ep, np, out);
  return cudaGetLastError();
}

}  // namespace xcb
