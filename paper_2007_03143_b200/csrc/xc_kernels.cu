// xc_kernels.cu -- CUDA kernels (sm_100a) of libxc_b200: the hot path of Alg. 4.
//
//   k_weights   step (a)   partition weights, Eq. (9), Alg. 4 l.4.1
//   k_density   steps (c),(d1),(e),(f) + Z of (d2): collocation Eq. (7)/(12a), X = P^j Phi^j Eq. (15),
//               rho / grad rho Eqs. (13),(14), functional Eq. (19), E/N Eq. (16), Z Eq. (20)
//   k_potential step (d2),(g): V^j = Z Phi^T + Phi Z^T Eq. (18) and the increment Eq. (17)
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

// ------------------------------------------------------------------------------------------------
// small device helpers
// ------------------------------------------------------------------------------------------------
__device__ __forceinline__ void dmma884(double& c0, double& c1, double a, double b) {
  asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};\n"
               : "+d"(c0), "+d"(c1)
               : "d"(a), "d"(b));
}
__device__ __forceinline__ void cp_async8(void* smem, const void* gmem) {
  unsigned s = (unsigned)__cvta_generic_to_shared(smem);
  asm volatile("cp.async.ca.shared.global [%0], [%1], 8;\n" ::"r"(s), "l"(gmem));
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;\n" ::); }
template <int N>
__device__ __forceinline__ void cp_async_wait() { asm volatile("cp.async.wait_group %0;\n" ::"n"(N)); }

__device__ __forceinline__ double pw012(double v, int n) { return n == 0 ? 1.0 : (n == 1 ? v : v * v); }
__device__ __forceinline__ double dpw012(double v, int n) { return n == 0 ? 0.0 : (n == 1 ? 1.0 : 2.0 * v); }

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

__device__ __forceinline__ void lda_slater_vwn5(double rho, double& f, double& vr) {
  const double A = 0.0310907, x0 = -0.10498, b = 3.72744, c = 12.9352;
  const double Q = 6.1519908197590802321728722658;         // sqrt(4c - b^2)
  const double Xx0 = x0 * x0 + b * x0 + c;
  const double bx0 = b * x0 / Xx0;
  double r13 = cbrt(rho);
  double rs = XC_RSFAC / r13;
  double x = sqrt(rs);
  double X = fma(x, x + b, c);
  double tb = 2.0 * x + b;
  double at = atan(Q / tb);
  double xm = x - x0;
  double eps = A * (log(x * x / X) + (2.0 * b / Q) * at - bx0 * (log(xm * xm / X) + (2.0 * (b + 2.0 * x0) / Q) * at));
  double q2 = 1.0 / (Q * Q + tb * tb);
  double deps = A * (2.0 / x - tb / X - 4.0 * b * q2 - bx0 * (2.0 / xm - tb / X - 4.0 * (2.0 * x0 + b) * q2));
  double vc = eps - (x / 6.0) * deps;
  f = rho * (eps - XC_CX * r13);
  vr = vc - (4.0 / 3.0) * XC_CX * r13;
}

__device__ __forceinline__ void gga_pbe(double rho, double sigma, double& f, double& vr, double& vs) {
  const double kappa = 0.804, mu = 0.2195149727645171;
  const double gamma = 0.031090690869654895, beta = 0.06672455060314922;
  const double A = 0.0310907, a1 = 0.21370, b1 = 7.5957, b2 = 3.5876, b3 = 1.6382, b4 = 0.49294;
  const double c_s2 = 38.283120002509214;      // 4 (3 pi^2)^(2/3)
  const double c_t2 = 0.06346820609770369;     // pi / (16 (3 pi^2)^(1/3))
  double r13 = cbrt(rho);
  double r43 = rho * r13;
  // exchange
  double s2 = sigma / (c_s2 * r43 * r43);
  double den = 1.0 / (kappa + mu * s2);
  double F = 1.0 + kappa - kappa * kappa * den;
  double dF = kappa * kappa * mu * den * den;
  double fx = -XC_CX * r43 * F;
  double vxr = -(4.0 / 3.0) * XC_CX * r13 * (F - 2.0 * s2 * dF);
  double vxs = -XC_CX * dF / (c_s2 * r43);
  // PW92
  double rs = XC_RSFAC / r13;
  double srs = sqrt(rs);
  double q = 2.0 * A * (srs * (b1 + b3 * rs) + rs * (b2 + b4 * rs));
  double dq = 2.0 * A * (0.5 * b1 / srs + b2 + 1.5 * b3 * srs + 2.0 * b4 * rs);
  double lg = log1p(1.0 / q);
  double eu = -2.0 * A * (1.0 + a1 * rs) * lg;
  double deu_drs = -2.0 * A * a1 * lg + 2.0 * A * (1.0 + a1 * rs) * dq / (q * (q + 1.0));
  double deu = -deu_drs * rs / (3.0 * rho);    // d eps_unif / d rho
  // H
  double r73 = r43 * rho;
  double yfac = c_t2 / r73;
  double y = sigma * yfac;
  double Em1 = expm1(-eu / gamma);
  double Ac = (beta / gamma) / Em1;
  double Ay = Ac * y;
  double N = 1.0 + Ay, D = 1.0 + Ay + Ay * Ay;
  double G = (beta / gamma) * y * N / D;
  double H = gamma * log1p(G);
  double iD2G = 1.0 / (D * D * (1.0 + G));
  double dHdy = beta * (1.0 + 2.0 * Ay) * iD2G;
  double dHdA = -beta * y * Ay * y * (2.0 + Ay) * iD2G;
  double dAde = Ac * Ac * (Em1 + 1.0) / beta;
  double vcs = rho * dHdy * yfac;
  double vcr = eu + H + rho * (deu + dHdy * (-(7.0 / 3.0) * y / rho) + dHdA * dAde * deu);
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
      for (int bb = 0; bb < nB; ++bb) {
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
        }
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
// step (a), hot path for SSF: one CTA per batch, one WARP per point, the lanes split the atom list.
// Exact pruning only; the batch's atom list (planner) is sorted by
// dmin(atom, batch box) <= r_atom, so every scan stops as soon as dmin reaches its bound, and all control
// flow is warp-uniform:
//   0. r_A < (1-a)/2 R_nn(A)  =>  w = w^q.  The other points of the batch are compacted (in order); a batch
//      of core points never touches the atom list.
//   1. nearest atom m, r_min                 (32 atoms per step, scan while dmin < r_min)
//   2. P_A first: P_A = 0 => w = 0 and the point is done.
//   3. owner candidates B, 32 per step (scan while dmin < kappa r_min): r_B < kappa r_min and mu_Bm < a;
//      each surviving candidate's cell product P_B is then evaluated by the whole warp.
//   A cell product scans the partners C, 32 per step (while dmin < kappa r_B): s(mu_BC) = 1 exactly when
//   r_C >= r_B + a R_BC (tested on squares, no sqrt), and the scan stops as soon as one mu_BC >= a (P_B = 0).
//   Lane products are combined by an xor butterfly (same value in every lane) and the owners are summed in
//   list order, so w is bit-identical from run to run.
// ------------------------------------------------------------------------------------------------
__device__ __forceinline__ double ssf_cell_product(const double4* __restrict__ sAt, const int* __restrict__ sId, int nC, int lane,
                                                   double x, double y, double z, double Bx, double By, double Bz, int Bid,
                                                   double rB, double rB2) {
  const unsigned FULL = 0xffffffffu;
  const double kappa = (1.0 + 0.64) / (1.0 - 0.64);
  const double krB = kappa * rB, f4 = (4.0 * 0.64 * 0.64) * rB2;
  double part = 1.0;
  for (int c0 = 0; c0 < nC; c0 += 32) {
    if (sAt[c0].w >= krB) break;                          // every later C has r_C >= kappa r_B: factor 1
    const int c = c0 + lane;
    bool dead = false;
    if (c < nC) {
      const double4 at = sAt[c];
      if (at.w < krB && sId[c] != Bid) {
        const double dx = x - at.x, dy = y - at.y, dz = z - at.z;
        const double d2 = dx * dx + dy * dy + dz * dz;                 // r_C^2
        const double ex = Bx - at.x, ey = By - at.y, ez = Bz - at.z;
        const double R2 = ex * ex + ey * ey + ez * ez;                 // R_BC^2
        // s(mu_BC) = 1 exactly  <=>  r_C >= r_B + a R_BC  <=>  t >= 0 and t^2 >= 4 a^2 r_B^2 R_BC^2,
        // t = r_C^2 - r_B^2 - a^2 R_BC^2   (no square root)
        const double t = d2 - rB2 - (0.64 * 0.64) * R2;
        if (!(t >= 0.0 && t * t >= f4 * R2)) {
          const double zz = (rB - sqrt(d2)) * rsqrt(R2) * (1.0 / 0.64);   // mu_BC / a
          if (zz >= 1.0) {
            dead = true;                                               // s = 0: P_B = 0
          } else if (zz > -1.0) {
            const double z2 = zz * zz;
            part *= 0.5 - zz * (35.0 + z2 * (-35.0 + z2 * (21.0 - 5.0 * z2))) * (1.0 / 32.0);
          }
        }
      }
    }
    if (__any_sync(FULL, dead)) return 0.0;
  }
#pragma unroll
  for (int o = 16; o >= 1; o >>= 1) part *= __shfl_xor_sync(FULL, part, o);
  return part;
}

__global__ void __launch_bounds__(kWeightThreads, 4) k_weights_ssf(WeightArgs a, const int32_t* __restrict__ batch_ids) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  __shared__ int sCnt[2 * (kWeightThreads / 32)];
  const unsigned FULL = 0xffffffffu;
  const int bid = batch_ids[blockIdx.x];
  const BatchRec b = a.batches[bid];
  const int nC = b.wa_nC, nB = b.wa_nB;
  double4* sAt = (double4*)smem_raw;                     // x, y, z, dmin
  int* sId = (int*)(sAt + nC);
  short* sList = (short*)(sId + nC);                     // compacted non-trivial points of the batch (<= 512)
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const double aa = 0.64, kappa = (1.0 + aa) / (1.0 - aa);

  // ---- 0. trivial points, ordered compaction of the others ----
  int rank[2];
  bool live[2];
#pragma unroll
  for (int r = 0; r < 2; ++r) {
    const int p = r * kWeightThreads + threadIdx.x;
    live[r] = false;
    if (p < b.nq) {
      const int64_t gi = (int64_t)b.pt_off + p;
      const int A = a.parent[gi];
      bool trivial = a.natoms == 1;
      if (!trivial) {
        double dx = a.px[gi] - a.atoms[3 * A], dy = a.py[gi] - a.atoms[3 * A + 1], dz = a.pz[gi] - a.atoms[3 * A + 2];
        trivial = sqrt(dx * dx + dy * dy + dz * dz) < 0.5 * (1.0 - aa) * a.rnn[A];
      }
      if (trivial) a.w[gi] = a.wq[gi];
      live[r] = !trivial;
    }
    const unsigned mask = __ballot_sync(FULL, live[r]);
    rank[r] = __popc(mask & ((1u << lane) - 1u));
    if (lane == 0) sCnt[r * (kWeightThreads / 32) + warp] = __popc(mask);
  }
  __syncthreads();
  int total = 0;
#pragma unroll
  for (int r = 0; r < 2; ++r) {
    int off = 0;
    for (int k = 0; k < 2 * (kWeightThreads / 32); ++k) {
      if (k < r * (kWeightThreads / 32) + warp) off += sCnt[k];
      if (r == 0) total += sCnt[k];
    }
    if (live[r]) sList[off + rank[r]] = (short)(r * kWeightThreads + threadIdx.x);
  }
  if (total == 0) return;
  {
    const double* box = a.wbox + (size_t)6 * bid;
    for (int c = threadIdx.x; c < nC; c += kWeightThreads) {
      int at = a.watoms[b.wa_off + c];
      double cx = a.atoms[3 * at], cy = a.atoms[3 * at + 1], cz = a.atoms[3 * at + 2];
      double tx = cx < box[0] ? box[0] - cx : (cx > box[3] ? cx - box[3] : 0.0);
      double ty = cy < box[1] ? box[1] - cy : (cy > box[4] ? cy - box[4] : 0.0);
      double tz = cz < box[2] ? box[2] - cz : (cz > box[5] ? cz - box[5] : 0.0);
      // a hair below the true distance: the early exits must never cut an atom that matters
      sAt[c] = make_double4(cx, cy, cz, sqrt(tx * tx + ty * ty + tz * tz) * (1.0 - 1e-12) - 1e-12);
      sId[c] = at;
    }
  }
  __syncthreads();

  for (int n = warp; n < total; n += kWeightThreads / 32) {
    const int64_t gi = (int64_t)b.pt_off + sList[n];
    const double x = a.px[gi], y = a.py[gi], z = a.pz[gi];
    const int A = a.parent[gi];
    // ---- 1. nearest atom ----
    double rmin2 = 1e300;
    int im = 0;
    for (int c0 = 0; c0 < nC; c0 += 32) {
      const double dm = sAt[c0].w;
      if (dm > 0.0 && dm * dm >= rmin2) break;
      const int c = c0 + lane;
      double d2 = 1e300;
      if (c < nC) { const double4 at = sAt[c]; const double dx = x - at.x, dy = y - at.y, dz = z - at.z; d2 = dx * dx + dy * dy + dz * dz; }
      int ci = c;
#pragma unroll
      for (int o = 16; o >= 1; o >>= 1) {
        const double od = __shfl_xor_sync(FULL, d2, o);
        const int oi = __shfl_xor_sync(FULL, ci, o);
        if (od < d2 || (od == d2 && oi < ci)) { d2 = od; ci = oi; }
      }
      if (d2 < rmin2) { rmin2 = d2; im = ci; }
    }
    const double rmin = sqrt(rmin2), own_lim = kappa * rmin, own_lim2 = own_lim * own_lim;
    const double4 atm = sAt[im];
    const int mid = sId[im];
    // ---- 2. the parent's cell product ----
    const double Ax = a.atoms[3 * A], Ay = a.atoms[3 * A + 1], Az = a.atoms[3 * A + 2];
    double rA2;
    { const double dx = x - Ax, dy = y - Ay, dz = z - Az; rA2 = dx * dx + dy * dy + dz * dz; }
    const double rA = sqrt(rA2);
    double PA = 0.0;
    if (!(rA >= own_lim && rA > rmin)) PA = ssf_cell_product(sAt, sId, nC, lane, x, y, z, Ax, Ay, Az, A, rA, rA2);
    double result = 0.0;
    if (PA != 0.0) {
      // ---- 3. the other owners ----
      double sum = PA;
      for (int b0 = 0; b0 < nB; b0 += 32) {
        if (sAt[b0].w >= own_lim) break;
        const int bb = b0 + lane;
        bool cand = false;
        double4 at = make_double4(0.0, 0.0, 0.0, 0.0);
        double d2 = 0.0;
        int cid = -1;
        if (bb < nB) {
          at = sAt[bb]; cid = sId[bb];
          const double dx = x - at.x, dy = y - at.y, dz = z - at.z;
          d2 = dx * dx + dy * dy + dz * dz;
          cand = at.w < own_lim && cid != A && d2 < own_lim2;          // else r_B >= kappa r_min: P_B = 0 exactly
          if (cand && cid != mid) {                                    // mu_Bm >= a  =>  P_B = 0
            const double ex = at.x - atm.x, ey = at.y - atm.y, ez = at.z - atm.z;
            cand = (sqrt(d2) - rmin) * rsqrt(ex * ex + ey * ey + ez * ez) < aa;
          }
        }
        unsigned mask = __ballot_sync(FULL, cand);
        while (mask) {
          const int src = __ffs(mask) - 1;
          mask &= mask - 1;
          const double Bx = __shfl_sync(FULL, at.x, src), By = __shfl_sync(FULL, at.y, src), Bz = __shfl_sync(FULL, at.z, src);
          const double rB2 = __shfl_sync(FULL, d2, src);
          const int Bid = __shfl_sync(FULL, cid, src);
          sum += ssf_cell_product(sAt, sId, nC, lane, x, y, z, Bx, By, Bz, Bid, sqrt(rB2), rB2);
        }
      }
      result = a.wq[gi] * PA / sum;
    }
    if (lane == 0) a.w[gi] = result;
  }
}

// ------------------------------------------------------------------------------------------------
// density kernel.  One CTA (512 threads) = one tile of T points of one batch.
//   phase 0  metadata -> smem
//   phase 1  collocation: radial sums R0,R1 per (shell, point) -> sR; Phi -> sPhi[nu][i]
//   phase 2  X^T = Phi^T P  on DMMA (M = points, N = mu, K = nu): A from sPhi, B = P gathered through a
//            cp.async double buffer; epilogue: rho_i += Phi X, grad rho_i += grad Phi X
//   phase 3  functional at the T points, E / N_el partials
//   phase 4  Z = 1/2 a Phi + g . grad Phi; Phi and Z stored fragment-blocked for k_potential
// ------------------------------------------------------------------------------------------------
template <int T>
struct DensityCfg {
  static constexpr int WP = T / 16;            // warps along points
  static constexpr int WM = 16 / WP;           // warps along mu
  static constexpr int NTMAX = kMuPass / (8 * WM);
  static constexpr int LD = T + 4;             // == 4 (mod 16): conflict-free A-fragment reads
};

template <int T, bool GGA>
__global__ void __launch_bounds__(kDensityThreads, 1) k_density(DensityArgs a, const DensityItem* __restrict__ items, int item0) {
  using Cfg = DensityCfg<T>;
  constexpr int LD = Cfg::LD;
  extern __shared__ __align__(16) unsigned char smem_raw[];
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const DensityItem it = items[blockIdx.x];
  const BatchRec b = a.batches[it.batch];
  const int nb = b.nb, ns = b.ns, nb4 = (nb + 3) & ~3;
  const int npass = (nb + kMuPass - 1) / kMuPass;
  const int mbmax = min((nb + 8 * Cfg::WM - 1) / (8 * Cfg::WM) * (8 * Cfg::WM), kMuPass);
  const int LDP = mbmax + 4;

  // ---- carve shared memory ----
  unsigned char* sp = smem_raw;
  double* sPhi = (double*)sp; sp += (size_t)nb4 * LD * 8;
  double* sR = (double*)sp; if (GGA) sp += (size_t)ns * T * 16;
  double* sP = (double*)sp; sp += (size_t)2 * kKC * LDP * 8;
  double* sPt = (double*)sp; sp += (size_t)12 * T * 8;
  double* sRed = (double*)sp; sp += (size_t)1024 * 8;   // [WM][4][T], WM*4*T == 1024
  ShellRec* sSh = (ShellRec*)sp; sp += (size_t)ns * sizeof(ShellRec);
  int* sIdxMu = (int*)sp; sp += (size_t)npass * kMuPass * 4;
  int* sIdxNu = (int*)sp; sp += (size_t)nb4 * 4;
  int* sInfo = (int*)sp;
  double *sx = sPt, *sy = sPt + T, *sz = sPt + 2 * T, *sw = sPt + 3 * T;
  double *sRho = sPt + 4 * T, *sGx = sPt + 5 * T, *sGy = sPt + 6 * T, *sGz = sPt + 7 * T;
  double *sA = sPt + 8 * T, *sG0 = sPt + 9 * T, *sG1 = sPt + 10 * T, *sG2 = sPt + 11 * T;

  // ---- phase 0 ----
  const int32_t* fidx = a.bfidx + b.f_off;
  const int32_t* finfo = a.bfinfo + b.f_off;
  for (int k = tid; k < ns; k += kDensityThreads) {
    ShellRec r = a.shells[a.bshells[b.sh_off + k]];
    r._pad = a.bsfoff[b.sh_off + k];
    sSh[k] = r;
  }
  const int idx0 = fidx[0];
  for (int f = tid; f < nb4; f += kDensityThreads) {
    sIdxNu[f] = f < nb ? fidx[f] : idx0;
    sInfo[f] = f < nb ? finfo[f] : 0;
  }
  for (int f = tid; f < npass * kMuPass; f += kDensityThreads) sIdxMu[f] = f < nb ? fidx[f] : idx0;
  const int npt = min(T, b.nq - it.tile_start);  // valid points in this tile
  if (tid < T) {
    int li = min(tid, npt - 1);
    int64_t gi = (int64_t)b.pt_off + it.tile_start + li;
    sx[tid] = a.px[gi]; sy[tid] = a.py[gi]; sz[tid] = a.pz[gi];
    sw[tid] = tid < npt ? a.w[gi] : 0.0;
  }
  __syncthreads();

  // ---- phase 1: collocation (Eq. (7); same shell across a warp) ----
  for (int e = tid; e < ns * T; e += kDensityThreads) {
    int slot = e / T, i = e - slot * T;
    const ShellRec sh = sSh[slot];
    double dx = sx[i] - sh.x, dy = sy[i] - sh.y, dz = sz[i] - sh.z;
    double r2 = dx * dx + dy * dy + dz * dz;
    double R0 = 0.0, R1 = 0.0;
    for (int k = 0; k < sh.nprim; ++k) {
      double al = __ldg(a.exps + sh.prim_off + k), c = __ldg(a.coefs + sh.prim_off + k);
      double ev = c * exp(-al * r2);
      R0 += ev;
      R1 = fma(-2.0 * al, ev, R1);
    }
    if (GGA) *reinterpret_cast<double2*>(sR + ((size_t)slot * T + i) * 2) = make_double2(R0, R1);
    double* dst = sPhi + (size_t)sh._pad * LD + i;
    if (sh.L == 0) {
      dst[0] = R0;
    } else if (sh.L == 1) {
      dst[0] = dx * R0; dst[LD] = dy * R0; dst[2 * LD] = dz * R0;
    } else {
      double xr = dx * R0, yr = dy * R0;
      dst[0] = dx * xr; dst[LD] = dy * xr; dst[2 * LD] = dz * xr;
      dst[3 * LD] = dy * yr; dst[4 * LD] = dz * yr; dst[5 * LD] = dz * dz * R0;
    }
  }
  for (int e = tid; e < (nb4 - nb) * T; e += kDensityThreads) sPhi[(size_t)(nb + e / T) * LD + (e % T)] = 0.0;
  __syncthreads();

  // ---- phase 2: X^T = Phi^T P and the density reductions ----
  const int wp = warp % Cfg::WP, wm = warp / Cfg::WP;
  const int g4 = lane >> 2, t4 = lane & 3;
  double rho_acc[2] = {0.0, 0.0}, gx_acc[2] = {0.0, 0.0}, gy_acc[2] = {0.0, 0.0}, gz_acc[2] = {0.0, 0.0};
  const int nchunk = (nb4 + kKC - 1) / kKC;
  for (int pass = 0; pass < npass; ++pass) {
    const int mu0 = pass * kMuPass;
    const int mb = min((nb - mu0 + 8 * Cfg::WM - 1) / (8 * Cfg::WM) * (8 * Cfg::WM), kMuPass);
    const int mbw = mb / Cfg::WM;     // mu columns per warp (multiple of 8)
    const int nt = mbw >> 3;
    double C[2][Cfg::NTMAX][2];
#pragma unroll
    for (int u = 0; u < 2; ++u)
#pragma unroll
      for (int v = 0; v < Cfg::NTMAX; ++v) C[u][v][0] = C[u][v][1] = 0.0;

    auto stage_load = [&](int chunk, int stage) {
      double* dstS = sP + (size_t)stage * kKC * LDP;
      const int rows = min(kKC, nb4 - chunk * kKC);
      for (int e = tid; e < rows * mb; e += kDensityThreads) {
        int k = e / mb, mcol = e - k * mb;
        const double* src = a.P + (size_t)sIdxNu[chunk * kKC + k] * a.ldp + sIdxMu[mu0 + mcol];
        cp_async8(dstS + (size_t)k * LDP + mcol, src);
      }
      cp_async_commit();
    };
    stage_load(0, 0);
    for (int chunk = 0; chunk < nchunk; ++chunk) {
      const int stage = chunk & 1;
      if (chunk + 1 < nchunk) { stage_load(chunk + 1, stage ^ 1); cp_async_wait<1>(); }
      else cp_async_wait<0>();
      __syncthreads();
      const double* Ps = sP + (size_t)stage * kKC * LDP + wm * mbw + g4;
      const int steps = min(kKC, nb4 - chunk * kKC) >> 2;
      for (int ks = 0; ks < steps; ++ks) {
        const int kk = chunk * kKC + ks * 4 + t4;
        const double* Ap = sPhi + (size_t)kk * LD + wp * 16 + g4;
        double A0 = Ap[0], A1 = Ap[8];
        const double* Bp = Ps + (size_t)(ks * 4 + t4) * LDP;
#pragma unroll
        for (int v = 0; v < Cfg::NTMAX; ++v) {
          if (v < nt) {
            double Bv = Bp[v * 8];
            dmma884(C[0][v][0], C[0][v][1], A0, Bv);
            dmma884(C[1][v][0], C[1][v][1], A1, Bv);
          }
        }
      }
      __syncthreads();
    }
    // epilogue of this pass: Eqs. (13),(14)
#pragma unroll
    for (int u = 0; u < 2; ++u) {
      const int i = wp * 16 + u * 8 + g4;
      const double xi = sx[i], yi = sy[i], zi = sz[i];
#pragma unroll
      for (int v = 0; v < Cfg::NTMAX; ++v) {
        if (v < nt) {
#pragma unroll
          for (int h = 0; h < 2; ++h) {
            const int mu = mu0 + wm * mbw + v * 8 + t4 * 2 + h;
            if (mu < nb) {
              const double X = C[u][v][h];
              rho_acc[u] = fma(sPhi[(size_t)mu * LD + i], X, rho_acc[u]);
              if (GGA) {
                const int info = sInfo[mu];
                const int slot = info >> 8;
                const double2 R = *reinterpret_cast<const double2*>(sR + ((size_t)slot * T + i) * 2);
                double gx, gy, gz;
                grad_cart(info, xi - sSh[slot].x, yi - sSh[slot].y, zi - sSh[slot].z, R.x, R.y, gx, gy, gz);
                gx_acc[u] = fma(gx, X, gx_acc[u]);
                gy_acc[u] = fma(gy, X, gy_acc[u]);
                gz_acc[u] = fma(gz, X, gz_acc[u]);
              }
            }
          }
        }
      }
    }
  }
  // reduce over the 4 lanes sharing a point, then over the WM warps (fixed order => deterministic)
#pragma unroll
  for (int u = 0; u < 2; ++u) {
#pragma unroll
    for (int o = 1; o <= 2; o <<= 1) {
      rho_acc[u] += __shfl_xor_sync(0xffffffffu, rho_acc[u], o);
      if (GGA) {
        gx_acc[u] += __shfl_xor_sync(0xffffffffu, gx_acc[u], o);
        gy_acc[u] += __shfl_xor_sync(0xffffffffu, gy_acc[u], o);
        gz_acc[u] += __shfl_xor_sync(0xffffffffu, gz_acc[u], o);
      }
    }
    if (t4 == 0) {
      const int i = wp * 16 + u * 8 + g4;
      sRed[(size_t)(wm * 4 + 0) * T + i] = rho_acc[u];
      if (GGA) {
        sRed[(size_t)(wm * 4 + 1) * T + i] = gx_acc[u];
        sRed[(size_t)(wm * 4 + 2) * T + i] = gy_acc[u];
        sRed[(size_t)(wm * 4 + 3) * T + i] = gz_acc[u];
      }
    }
  }
  __syncthreads();

  // ---- phase 3: functional (Eq. (19)), E and N_el partials (Eq. (16)) ----
  if (tid < T) {
    double rho = 0.0, gx = 0.0, gy = 0.0, gz = 0.0;
    for (int q = 0; q < Cfg::WM; ++q) {
      rho += sRed[(size_t)(q * 4 + 0) * T + tid];
      if (GGA) {
        gx += sRed[(size_t)(q * 4 + 1) * T + tid];
        gy += sRed[(size_t)(q * 4 + 2) * T + tid];
        gz += sRed[(size_t)(q * 4 + 3) * T + tid];
      }
    }
    gx *= 2.0; gy *= 2.0; gz *= 2.0;
    const double sigma = gx * gx + gy * gy + gz * gz;
    const double wi = sw[tid];
    double f, vr, vs;
    xc_point<GGA>(rho, sigma, a.rho_tol, f, vr, vs);
    sA[tid] = 0.5 * wi * vr;
    const double gs = 2.0 * wi * vs;
    sG0[tid] = gs * gx; sG1[tid] = gs * gy; sG2[tid] = gs * gz;
    if (tid < npt && a.rho_out) {
      int64_t gi = (int64_t)b.pt_off + it.tile_start + tid;
      a.rho_out[gi] = rho;
      if (a.grho_out) { a.grho_out[3 * gi] = gx; a.grho_out[3 * gi + 1] = gy; a.grho_out[3 * gi + 2] = gz; }
    }
    double e = wi * f, n = wi * rho;
#pragma unroll
    for (int o = 16; o >= 1; o >>= 1) {
      e += __shfl_xor_sync(0xffffffffu, e, o);
      n += __shfl_xor_sync(0xffffffffu, n, o);
    }
    if (lane == 0) { sRho[warp] = e; sGx[warp] = n; }
  }
  __syncthreads();
  if (tid == 0) {
    double e = 0.0, n = 0.0;
    for (int q = 0; q < T / 32; ++q) { e += sRho[q]; n += sGx[q]; }
    a.Epart[item0 + blockIdx.x] = e;
    a.Npart[item0 + blockIdx.x] = n;
  }

  // ---- phase 4: Z (Eq. (20)); store Phi and Z in 8x4 fragment blocks ----
  {
    const int nkq = b.nq_pad >> 2;             // 4-point chunks per row tile of the batch
    const int q0 = it.tile_start >> 2;
    const int nq4 = min(T / 4, nkq - q0);      // chunks of this tile that exist in the workspace
    const int nmt = b.nb_pad8 >> 3;
    double* phi_out = a.phi_scr + b.scr_off;
    double* z_out = a.z_scr + b.scr_off;
    for (int blk = warp; blk < nmt * nq4; blk += kDensityThreads / 32) {
      const int mt = blk / nq4, q = blk - mt * nq4;
      const int mu = mt * 8 + g4, i = q * 4 + t4;
      double phi = 0.0, zv = 0.0;
      if (mu < nb && i < npt) {
        phi = sPhi[(size_t)mu * LD + i];
        zv = sA[i] * phi;
        if (GGA) {
          const int info = sInfo[mu];
          const int slot = info >> 8;
          const double2 R = *reinterpret_cast<const double2*>(sR + ((size_t)slot * T + i) * 2);
          double gx, gy, gz;
          grad_cart(info, sx[i] - sSh[slot].x, sy[i] - sSh[slot].y, sz[i] - sSh[slot].z, R.x, R.y, gx, gy, gz);
          zv = fma(sG0[i], gx, fma(sG1[i], gy, fma(sG2[i], gz, zv)));
        }
      }
      const size_t o = ((size_t)mt * nkq + q0 + q) * 32 + lane;
      phi_out[o] = phi;
      z_out[o] = zv;
    }
  }
}

// ------------------------------------------------------------------------------------------------
// potential kernel.  One WARP = one work item: a 32x32 lower-triangle tile of V^j over a range of points.
// Fragments are read straight from the fragment-blocked workspace (one coalesced 256-byte line per
// fragment); tiles of the same batch run in the same CTA so the panels are shared through L1.
// The increment Eq. (17) is done in exact 96-bit fixed point (two 64-bit integer atomics), which is
// associative: V is bit-identical from run to run whatever the order of arrival.
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

__global__ void __launch_bounds__(kPotThreads, 2) k_potential(PotArgs a) {
  const int lane = threadIdx.x & 31;
  const int64_t item = (int64_t)blockIdx.x * (kPotThreads / 32) + (threadIdx.x >> 5);
  if (item >= a.nitems) return;
  const PotItem it = a.items[item];
  const BatchRec b = a.batches[it.batch];
  const int nkq = b.nq_pad >> 2;
  const int nmt = b.nb_pad8 >> 3;
  const double* phi = a.phi_scr + b.scr_off;
  const double* zz = a.z_scr + b.scr_off;
  const bool diag = it.tm == it.tn;
  double C[4][4][2];
#pragma unroll
  for (int u = 0; u < 4; ++u)
#pragma unroll
    for (int v = 0; v < 4; ++v) C[u][v][0] = C[u][v][1] = 0.0;
  bool vm[4], vn[4];
  size_t om[4], on[4];
#pragma unroll
  for (int u = 0; u < 4; ++u) {
    vm[u] = it.tm * 4 + u < nmt;
    vn[u] = it.tn * 4 + u < nmt;
    om[u] = (size_t)(it.tm * 4 + u) * nkq * 32 + lane;
    on[u] = (size_t)(it.tn * 4 + u) * nkq * 32 + lane;
  }
  for (int kc = it.k0 >> 2; kc < (it.k1 >> 2); ++kc) {
    double Zm[4], Pm[4], Zn[4], Pn[4];
#pragma unroll
    for (int u = 0; u < 4; ++u) {
      Zm[u] = vm[u] ? __ldg(zz + om[u] + (size_t)kc * 32) : 0.0;
      Pm[u] = vm[u] ? __ldg(phi + om[u] + (size_t)kc * 32) : 0.0;
    }
    if (diag) {
#pragma unroll
      for (int u = 0; u < 4; ++u) { Zn[u] = Zm[u]; Pn[u] = Pm[u]; }
    } else {
#pragma unroll
      for (int u = 0; u < 4; ++u) {
        Zn[u] = vn[u] ? __ldg(zz + on[u] + (size_t)kc * 32) : 0.0;
        Pn[u] = vn[u] ? __ldg(phi + on[u] + (size_t)kc * 32) : 0.0;
      }
    }
#pragma unroll
    for (int u = 0; u < 4; ++u)
#pragma unroll
      for (int v = 0; v < 4; ++v) {
        dmma884(C[u][v][0], C[u][v][1], Zm[u], Pn[v]);
        dmma884(C[u][v][0], C[u][v][1], Pm[u], Zn[v]);
      }
  }
  // scatter: lower triangle (mu >= nu) only; global indices ascend with local ones
  const int32_t* fidx = a.bfidx + b.f_off;
  const int g4 = lane >> 2, t4 = lane & 3;
#pragma unroll
  for (int u = 0; u < 4; ++u) {
    const int mu = it.tm * 32 + u * 8 + g4;
    if (mu >= b.nb) continue;
    const size_t row = (size_t)fidx[mu] * a.nbasis;
#pragma unroll
    for (int v = 0; v < 4; ++v)
#pragma unroll
      for (int h = 0; h < 2; ++h) {
        const int nu = it.tn * 32 + v * 8 + t4 * 2 + h;
        if (nu <= mu && nu < b.nb) {
          const size_t o = row + fidx[nu];
          fixed_add(a.vhi + o, a.vlo + o, C[u][v][h]);
        }
      }
  }
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
    smem = (size_t)max_list * 36 + 1024 + 64;   // list: x,y,z,dmin,id; compacted point list
    e = cudaFuncSetAttribute(k_weights_ssf, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)std::max<size_t>(smem, 1024));
    if (e != cudaSuccess) return e;
    k_weights_ssf<<<nbatches, kWeightThreads, smem, st>>>(a, batch_ids);
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

template <int T, bool GGA>
static cudaError_t launch_density_t(const DensityArgs& a, const DensityItem* items, int nitems, int item0, size_t smem,
                                    cudaStream_t st) {
  if (nitems <= 0) return cudaSuccess;
  cudaError_t e = cudaFuncSetAttribute(k_density<T, GGA>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
  if (e != cudaSuccess) return e;
  k_density<T, GGA><<<nitems, kDensityThreads, smem, st>>>(a, items, item0);
  return cudaGetLastError();
}

cudaError_t launch_density(int T, bool gga, const DensityArgs& a, const DensityItem* items, int nitems, int item0,
                           size_t smem, cudaStream_t st) {
  if (T == 64) return gga ? launch_density_t<64, true>(a, items, nitems, item0, smem, st)
                          : launch_density_t<64, false>(a, items, nitems, item0, smem, st);
  return gga ? launch_density_t<32, true>(a, items, nitems, item0, smem, st)
             : launch_density_t<32, false>(a, items, nitems, item0, smem, st);
}

cudaError_t launch_potential(const PotArgs& a, cudaStream_t st) {
  if (a.nitems <= 0) return cudaSuccess;
  int wpb = kPotThreads / 32;
  k_potential<<<(unsigned)((a.nitems + wpb - 1) / wpb), kPotThreads, 0, st>>>(a);
  return cudaGetLastError();
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
