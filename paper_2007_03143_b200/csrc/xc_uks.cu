// xc_uks.cu -- the spin-coupling step of the spin-unrestricted build (xc_eval_uks; "may be extended to
// ... spin-unrestricted ... with the addition of only a few intermediates"; readings A20-A22).
//
//   k_functional_uks   per grid point: f(rho_a, rho_b, s_aa, s_ab, s_bb) and its five partials (spin-polarised
//                      Slater+VWN5 or PBE), then the per-point coefficients of Z^s (Eq. (20) PAPER.md:L162 per spin):
//                        a_s = 1/2 w v_rho_s (GGA) | w v_rho_s (LDA),  g_s = w (2 v_ss grad rho_s + v_ab grad rho_s')
//                      and deterministic per-block partial sums of E_xc, N_a, N_b (Eq. (16)).
//
// The partial derivatives are taken by forward-mode differentiation of the energy expression in device code (five
// tangents per value).  This is an element-wise kernel over the grid, < 1 % of a build; the restricted hot path
// (xc_kernels.cu) keeps its hand-derived closed forms.  (Product code; shares nothing with oracle/.)
#include <cuda_runtime.h>

#include <cstdint>
#include <mutex>

#include "xc_internal.h"
#include "xc_kernels.h"

namespace xcb {

namespace {

struct T5 {           // value and tangents with respect to (rho_a, rho_b, s_aa, s_ab, s_bb)
  double v, t[5];
};
__device__ __forceinline__ T5 cst(double v) { T5 r; r.v = v; for (int k = 0; k < 5; ++k) r.t[k] = 0.0; return r; }
__device__ __forceinline__ T5 seed(double v, int k) { T5 r = cst(v); r.t[k] = 1.0; return r; }
__device__ __forceinline__ T5 chain(const T5& x, double g, double dg) { T5 r; r.v = g; for (int k = 0; k < 5; ++k) r.t[k] = dg * x.t[k]; return r; }
__device__ __forceinline__ T5 operator+(const T5& a, const T5& b) { T5 r; r.v = a.v + b.v; for (int k = 0; k < 5; ++k) r.t[k] = a.t[k] + b.t[k]; return r; }
__device__ __forceinline__ T5 operator-(const T5& a, const T5& b) { T5 r; r.v = a.v - b.v; for (int k = 0; k < 5; ++k) r.t[k] = a.t[k] - b.t[k]; return r; }
__device__ __forceinline__ T5 operator*(const T5& a, const T5& b) { T5 r; r.v = a.v * b.v; for (int k = 0; k < 5; ++k) r.t[k] = fma(a.t[k], b.v, a.v * b.t[k]); return r; }
__device__ __forceinline__ T5 operator/(const T5& a, const T5& b) {
  T5 r; const double ib = 1.0 / b.v; r.v = a.v * ib;
  for (int k = 0; k < 5; ++k) r.t[k] = (a.t[k] - r.v * b.t[k]) * ib;
  return r;
}
__device__ __forceinline__ T5 operator+(const T5& a, double c) { T5 r = a; r.v += c; return r; }
__device__ __forceinline__ T5 operator-(const T5& a, double c) { T5 r = a; r.v -= c; return r; }
__device__ __forceinline__ T5 operator*(const T5& a, double c) { T5 r; r.v = a.v * c; for (int k = 0; k < 5; ++k) r.t[k] = a.t[k] * c; return r; }
__device__ __forceinline__ T5 operator*(double c, const T5& a) { return a * c; }
__device__ __forceinline__ T5 operator+(double c, const T5& a) { return a + c; }
__device__ __forceinline__ T5 operator-(double c, const T5& a) { T5 r; r.v = c - a.v; for (int k = 0; k < 5; ++k) r.t[k] = -a.t[k]; return r; }
__device__ __forceinline__ T5 operator/(double c, const T5& a) { const double i = 1.0 / a.v; return chain(a, c * i, -c * i * i); }
__device__ __forceinline__ T5 tlog(const T5& x) { return chain(x, log(x.v), 1.0 / x.v); }
__device__ __forceinline__ T5 tlog1p(const T5& x) { return chain(x, log1p(x.v), 1.0 / (1.0 + x.v)); }
__device__ __forceinline__ T5 texpm1(const T5& x) { const double e = expm1(x.v); return chain(x, e, e + 1.0); }
__device__ __forceinline__ T5 tatan(const T5& x) { return chain(x, atan(x.v), 1.0 / fma(x.v, x.v, 1.0)); }
__device__ __forceinline__ T5 tsqrt(const T5& x) { const double s = sqrt(x.v); return chain(x, s, 0.5 / s); }
__device__ __forceinline__ T5 tcbrt(const T5& x) { const double c = cbrt(x.v); return chain(x, c, c / (3.0 * x.v)); }
__device__ __forceinline__ T5 tpow(const T5& x, double p) { const double w = pow(x.v, p); return chain(x, w, p * w / x.v); }   // x.v > 0

constexpr double kPi = 3.14159265358979323846264338327950288;
constexpr double kCx = 0.7385587663820224058842300326808360;          // (3/4)(3/pi)^(1/3)
constexpr double kRs = 0.6203504908994000166680068120477781;          // (3/(4 pi))^(1/3)
constexpr double kFz = 1.9236610509315363197779613852955;             // 1 / (2^(4/3) - 2)
constexpr double kFpp0 = 1.7099209341613656175639627762446;           // f''(0) = 4 / (9 (2^(1/3) - 1))

// spin interpolation f(zeta) = ((1+z)^(4/3) + (1-z)^(4/3) - 2) / (2^(4/3) - 2)
__device__ __forceinline__ T5 spin_f(const T5& z) { return (tpow(1.0 + z, 4.0 / 3.0) + tpow(1.0 - z, 4.0 / 3.0) - 2.0) * kFz; }

// VWN (1980) fit V: G(x) with x = sqrt(r_s)
__device__ __forceinline__ T5 vwn_fit(const T5& x, double A, double x0, double b, double c) {
  const double Q = sqrt(4.0 * c - b * b), X0 = fma(x0, x0 + b, c);
  const T5 X = x * (x + b) + c;
  const T5 at = tatan(Q / (2.0 * x + b));
  const T5 xm = x - x0;
  return A * (tlog(x * x / X) + (2.0 * b / Q) * at - (b * x0 / X0) * (tlog(xm * xm / X) + (2.0 * (b + 2.0 * x0) / Q) * at));
}
// PW92 fit G(r_s)
__device__ __forceinline__ T5 pw92_fit(const T5& rs, const T5& srs, double A, double a1, double b1, double b2, double b3, double b4) {
  const T5 q = (2.0 * A) * (srs * (b1 + b3 * rs) + rs * (b2 + b4 * rs));
  return (-2.0 * A) * (1.0 + a1 * rs) * tlog1p(1.0 / q);
}
// eps(r_s, zeta) = e0 + ac f/f''(0) (1 - z^4) + (e1 - e0) f z^4
__device__ __forceinline__ T5 spin_interp(const T5& e0, const T5& e1, const T5& ac, const T5& z) {
  const T5 f = spin_f(z), z2 = z * z, z4 = z2 * z2;
  return e0 + ac * f * (1.0 / kFpp0) * (1.0 - z4) + (e1 - e0) * f * z4;
}

__device__ __forceinline__ T5 lda_pol(const T5& ra, const T5& rb) {
  const T5 rho = ra + rb, z = (ra - rb) / rho;
  // Slater, spin-scaled: -C_x 2^(1/3) (ra^(4/3) + rb^(4/3))
  const T5 fx = (-kCx * 1.2599210498948731647672106072782) * (ra * tcbrt(ra) + rb * tcbrt(rb));
  const T5 x = tsqrt(kRs / tcbrt(rho));
  const T5 eP = vwn_fit(x, 0.0310907, -0.10498, 3.72744, 12.9352);
  const T5 eF = vwn_fit(x, 0.01554535, -0.32500, 7.06042, 18.0578);
  const T5 ac = vwn_fit(x, -1.0 / (6.0 * kPi * kPi), -0.0047584, 1.13107, 13.0045);
  return fx + rho * spin_interp(eP, eF, ac, z);
}

__device__ __forceinline__ T5 pbe_x_channel(const T5& r2, const T5& s4) {   // unpolarised PBE exchange at (2 rho_s, 4 s_ss)
  const double kappa = 0.804, mu = 0.2195149727645171, c_s2 = 38.283120002509214;   // 4 (3 pi^2)^(2/3)
  const T5 r13 = tcbrt(r2), r43 = r2 * r13;
  const T5 s2 = s4 / (c_s2 * r43 * r43);
  const T5 F = (1.0 + kappa) - (kappa * kappa) / (kappa + mu * s2);
  return (-kCx) * r43 * F;
}
// PBE correlation at (rho, zeta, sigma = |grad rho|^2), per unit volume
__device__ __forceinline__ T5 pbe_c_pol(const T5& rho, const T5& z, const T5& sigma) {
  const double gamma = 0.031090690869654895, beta = 0.06672455060314922;
  const T5 r13 = tcbrt(rho);
  const T5 rs = kRs / r13, srs = tsqrt(rs);
  const T5 e0 = pw92_fit(rs, srs, 0.0310907, 0.21370, 7.5957, 3.5876, 1.6382, 0.49294);
  const T5 e1 = pw92_fit(rs, srs, 0.01554535, 0.20548, 14.1189, 6.1977, 3.3662, 0.62517);
  const T5 mac = pw92_fit(rs, srs, 0.0168869, 0.11125, 10.357, 3.6231, 0.88026, 0.49671);   // -alpha_c
  const T5 eu = spin_interp(e0, e1, 0.0 - mac, z);
  const T5 phi = 0.5 * (tpow(1.0 + z, 2.0 / 3.0) + tpow(1.0 - z, 2.0 / 3.0));
  const T5 phi2 = phi * phi, phi3 = phi2 * phi;
  // t^2 = sigma / (4 phi^2 k_s^2 rho^2), k_s^2 = 4 (3 pi^2 rho)^(1/3) / pi:  t^2 = c_t2 sigma / (phi^2 rho^(7/3))
  const double c_t2 = 0.06346820609770369;     // pi / (16 (3 pi^2)^(1/3))
  const T5 t2 = c_t2 * sigma / (phi2 * rho * rho * r13);
  const T5 Ac = (beta / gamma) / texpm1((-1.0 / gamma) * eu / phi3);
  const T5 At = Ac * t2;
  const T5 H = gamma * phi3 * tlog1p((beta / gamma) * t2 * (1.0 + At) / (1.0 + At + At * At));
  return rho * (eu + H);
}
__device__ __forceinline__ T5 pbe_pol(const T5& ra, const T5& rb, const T5& saa, const T5& sab, const T5& sbb) {
  const T5 rho = ra + rb, z = (ra - rb) / rho, sigma = saa + 2.0 * sab + sbb;
  const T5 fx = 0.5 * (pbe_x_channel(2.0 * ra, 4.0 * saa) + pbe_x_channel(2.0 * rb, 4.0 * sbb));
  return fx + pbe_c_pol(rho, z, sigma);
}
// restricted meta-GGA of reading A23: MS0 exchange (Sun, Xiao, Ruzsinszky 2012) + PBE correlation; tangent slots 0 = rho,
// 1 = sigma, 2 = tau.  F_x = F1 + f(alpha) (F0 - F1), F_int(p; c) = 1 + kappa - kappa^2 / (kappa + mu_GE p + c)
__device__ __forceinline__ T5 mgga_ms0_pbe(const T5& rho, const T5& sigma, const T5& tau) {
  const double kappa = 0.29, c = 0.28771, muGE = 10.0 / 81.0;
  const double k23 = 9.5707800006273037;         // (3 pi^2)^(2/3)
  const T5 r13 = tcbrt(rho), r23 = r13 * r13;
  const T5 r43 = rho * r13, r53 = rho * r23;
  const T5 p = sigma / ((4.0 * k23) * r43 * r43);
  const T5 al = (tau - sigma / (8.0 * rho)) / ((0.3 * k23) * r53);
  const T5 F1 = (1.0 + kappa) - (kappa * kappa) / (kappa + muGE * p);
  const T5 F0 = (1.0 + kappa) - (kappa * kappa) / ((kappa + c) + muGE * p);
  const T5 a2 = al * al, a3 = a2 * al, om = 1.0 - a2;
  const T5 fa = om * om * om / (1.0 + a3 + a3 * a3);
  const T5 fx = (-kCx) * r43 * (F1 + fa * (F0 - F1));
  return fx + pbe_c_pol(rho, cst(0.0), sigma);
}

constexpr int kUksThreads = 256;

}  // namespace

// one thread per grid point; rho / grho hold [2][npts] and [2][npts][3] (spin-major); points with w = 0 were not
// visited by the density passes and contribute nothing
template <bool GGA>
__global__ void __launch_bounds__(kUksThreads) k_functional_uks(int64_t npts, const double* __restrict__ w, const double* __restrict__ rho,
                                                                const double* __restrict__ grho, double rho_tol, double* __restrict__ cA,
                                                                double* __restrict__ cG, double* __restrict__ part /* [nblocks][3] */) {
  __shared__ double sred[3][kUksThreads / 32];
  const int64_t i = (int64_t)blockIdx.x * kUksThreads + threadIdx.x;
  double e = 0.0, na = 0.0, nb = 0.0;
  if (i < npts) {
    const double wi = w[i];
    double aa = 0.0, ab = 0.0, ga[3] = {0.0, 0.0, 0.0}, gb[3] = {0.0, 0.0, 0.0};
    if (wi != 0.0) {
      const double ra = rho[i], rb = rho[npts + i];
      double xa[3] = {0.0, 0.0, 0.0}, xb[3] = {0.0, 0.0, 0.0};
      if (GGA) {
        for (int c = 0; c < 3; ++c) { xa[c] = grho[3 * i + c]; xb[c] = grho[3 * (npts + i) + c]; }
      }
      na = wi * ra; nb = wi * rb;
      if (!(ra + rb <= rho_tol)) {               // reading A20 (a NaN density is not skipped: it propagates)
        const double saa = xa[0] * xa[0] + xa[1] * xa[1] + xa[2] * xa[2];
        const double sab = xa[0] * xb[0] + xa[1] * xb[1] + xa[2] * xb[2];
        const double sbb = xb[0] * xb[0] + xb[1] * xb[1] + xb[2] * xb[2];
        const T5 Ra = seed(ra < rho_tol ? rho_tol : ra, 0), Rb = seed(rb < rho_tol ? rho_tol : rb, 1);
        const T5 f = GGA ? pbe_pol(Ra, Rb, seed(saa, 2), seed(sab, 3), seed(sbb, 4)) : lda_pol(Ra, Rb);
        e = wi * f.v;
        aa = (GGA ? 0.5 : 1.0) * wi * f.t[0];
        ab = (GGA ? 0.5 : 1.0) * wi * f.t[1];
        if (GGA) {
          for (int c = 0; c < 3; ++c) {
            ga[c] = wi * (2.0 * f.t[2] * xa[c] + f.t[3] * xb[c]);
            gb[c] = wi * (2.0 * f.t[4] * xb[c] + f.t[3] * xa[c]);
          }
        }
      }
    }
    cA[i] = aa; cA[npts + i] = ab;
    if (GGA) {
      for (int c = 0; c < 3; ++c) { cG[3 * i + c] = ga[c]; cG[3 * (npts + i) + c] = gb[c]; }
    }
  }
  // deterministic block sums: xor butterfly, then the warps in order
#pragma unroll
  for (int o = 16; o >= 1; o >>= 1) {
    e += __shfl_xor_sync(0xffffffffu, e, o);
    na += __shfl_xor_sync(0xffffffffu, na, o);
    nb += __shfl_xor_sync(0xffffffffu, nb, o);
  }
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  if (lane == 0) { sred[0][warp] = e; sred[1][warp] = na; sred[2][warp] = nb; }
  __syncthreads();
  if (threadIdx.x < 3) {
    double s = 0.0;
    for (int q = 0; q < kUksThreads / 32; ++q) s += sred[threadIdx.x][q];
    part[(size_t)blockIdx.x * 3 + threadIdx.x] = s;
  }
}

// fixed-order sum of the block partials: out[0..2] = E_xc, N_a, N_b
__global__ void __launch_bounds__(1024) k_reduce3(int64_t n, const double* __restrict__ part, double* __restrict__ out) {
  __shared__ double sm[3][1024];
  double v[3] = {0.0, 0.0, 0.0};
  for (int64_t i = threadIdx.x; i < n; i += 1024)
    for (int c = 0; c < 3; ++c) v[c] += part[3 * i + c];
  for (int c = 0; c < 3; ++c) sm[c][threadIdx.x] = v[c];
  __syncthreads();
  for (int s = 512; s >= 1; s >>= 1) {
    if ((int)threadIdx.x < s)
      for (int c = 0; c < 3; ++c) sm[c][threadIdx.x] += sm[c][threadIdx.x + s];
    __syncthreads();
  }
  if (threadIdx.x < 3) out[threadIdx.x] = sm[threadIdx.x][0];
}

int64_t uks_functional_blocks(int64_t npts) { return (npts + kUksThreads - 1) / kUksThreads; }

// restricted meta-GGA: per point f(rho, sigma, tau) and the coefficients of the potential: a = 1/2 w v_rho, g = 2 w v_sigma
// grad rho (Eq. (20)), t = 1/2 w v_tau (the tau term of V^j); w f and w rho per point for the per-batch sums
__global__ void __launch_bounds__(kUksThreads) k_functional_mgga(int64_t npts, const double* __restrict__ w, const double* __restrict__ rho,
                                                                 const double* __restrict__ grho, const double* __restrict__ tau, double rho_tol,
                                                                 double* __restrict__ cA, double* __restrict__ cG, double* __restrict__ cT,
                                                                 double* __restrict__ ef, double* __restrict__ en) {
  const int64_t i = (int64_t)blockIdx.x * kUksThreads + threadIdx.x;
  if (i >= npts) return;
  const double wi = w[i];
  double a = 0.0, t = 0.0, g[3] = {0.0, 0.0, 0.0}, e = 0.0, n = 0.0;
  if (wi != 0.0) {
    const double r = rho[i], x[3] = {grho[3 * i], grho[3 * i + 1], grho[3 * i + 2]};
    n = wi * r;
    if (!(r <= rho_tol)) {                       // a NaN density is not skipped: it propagates
      const double sigma = x[0] * x[0] + x[1] * x[1] + x[2] * x[2];
      const T5 f = mgga_ms0_pbe(seed(r, 0), seed(sigma, 1), seed(tau[i], 2));
      e = wi * f.v;
      a = 0.5 * wi * f.t[0];
      t = 0.5 * wi * f.t[2];
      const double gs = 2.0 * wi * f.t[1];
      for (int c = 0; c < 3; ++c) g[c] = gs * x[c];
    }
  }
  cA[i] = a; cT[i] = t;
  for (int c = 0; c < 3; ++c) cG[3 * i + c] = g[c];
  ef[i] = e; en[i] = n;
}
// per-batch sums of w f and w rho (Eq. (16)): one block per batch, fixed order
__global__ void __launch_bounds__(128) k_batch_sums(const BatchRec* __restrict__ batches, const double* __restrict__ ef,
                                                    const double* __restrict__ en, double* __restrict__ Epart, double* __restrict__ Npart) {
  __shared__ double se[128], sn[128];
  const BatchRec b = batches[blockIdx.x];
  double e = 0.0, n = 0.0;
  for (int k = threadIdx.x; k < b.nq; k += 128) { e += ef[(int64_t)b.pt_off + k]; n += en[(int64_t)b.pt_off + k]; }
  se[threadIdx.x] = e; sn[threadIdx.x] = n;
  __syncthreads();
  for (int s = 64; s >= 1; s >>= 1) {
    if ((int)threadIdx.x < s) { se[threadIdx.x] += se[threadIdx.x + s]; sn[threadIdx.x] += sn[threadIdx.x + s]; }
    __syncthreads();
  }
  if (threadIdx.x == 0) { Epart[blockIdx.x] = se[0]; Npart[blockIdx.x] = sn[0]; }
}

cudaError_t launch_functional_mgga(int64_t npts, int nbatches, const BatchRec* batches, const double* w, const double* rho, const double* grho,
                                   const double* tau, double rho_tol, double* cA, double* cG, double* cT, double* ef, double* en, double* Epart,
                                   double* Npart, cudaStream_t st) {
  if (npts <= 0 || nbatches <= 0) return cudaSuccess;
  k_functional_mgga<<<(unsigned)uks_functional_blocks(npts), kUksThreads, 0, st>>>(npts, w, rho, grho, tau, rho_tol, cA, cG, cT, ef, en);
  cudaError_t e = cudaGetLastError();
  if (e != cudaSuccess) return e;
  k_batch_sums<<<nbatches, 128, 0, st>>>(batches, ef, en, Epart, Npart);
  return cudaGetLastError();
}


// ------------------------------------------------------------------------------------------------
// The same step with NO allocation (xc_functional_uks_static; for callers that cannot call cudaMalloc: CUDA graph capture,
// serving loops): the block partials go to a file-scope array instead of a cudaMalloc'ed buffer.  The array exists once per
// GPU that loads the library (768 KB, held until exit), every call on that GPU shares it, and it keeps the last call's
// contents.  Nothing in it has to start at zero: a call writes the partials of its blocks [0, nblk) before k_reduce3 reads
// exactly those.  Two calls that overlap on one GPU (different streams, or two host threads) race on it.
// In host code the array's NAME is a host-side stand-in, not a device address: the address the kernels get comes from
// cudaGetSymbolAddress, asked once per device with that device current.
// ------------------------------------------------------------------------------------------------
constexpr int64_t kStaticMaxBlocks = kUksStaticMaxPoints / kUksThreads;
static_assert(kUksStaticMaxPoints % kUksThreads == 0, "kUksStaticMaxPoints is a whole number of blocks");
static __device__ __align__(256) double g_uks_static_part[3 * kStaticMaxBlocks];

namespace {
constexpr int kMaxDevices = 64;
std::mutex g_static_mu;
double* g_static_part_addr[kMaxDevices] = {};   // device address of g_uks_static_part on device d (null: not asked yet)
}  // namespace

cudaError_t functional_uks_static(bool gga, int64_t npts, const double* w, const double* rho, const double* grho, double rho_tol,
                                  double* cA, double* cG, double* out3, cudaStream_t st) {
  if (npts <= 0) return cudaSuccess;
  if (npts > kUksStaticMaxPoints) return cudaErrorInvalidValue;   // (the C entry point rejects it with its own message first)
  int dev = -1;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) return e;
  if (dev < 0 || dev >= kMaxDevices) return cudaErrorInvalidDevice;
  double* part = nullptr;
  {
    std::lock_guard<std::mutex> lock(g_static_mu);
    if (!g_static_part_addr[dev]) {
      void* ptr = nullptr;
      e = cudaGetSymbolAddress(&ptr, g_uks_static_part);   // the current device's copy of the array
      if (e != cudaSuccess) return e;
      g_static_part_addr[dev] = (double*)ptr;
    }
    part = g_static_part_addr[dev];
  }
  return launch_functional_uks(gga, npts, w, rho, grho, rho_tol, cA, cG, part, out3, st);
}

cudaError_t launch_functional_uks(bool gga, int64_t npts, const double* w, const double* rho, const double* grho, double rho_tol,
                                  double* cA, double* cG, double* part, double* out3, cudaStream_t st) {
  if (npts <= 0) return cudaSuccess;
  const int64_t nblk = uks_functional_blocks(npts);
  if (gga) k_functional_uks<true><<<(unsigned)nblk, kUksThreads, 0, st>>>(npts, w, rho, grho, rho_tol, cA, cG, part);
  else k_functional_uks<false><<<(unsigned)nblk, kUksThreads, 0, st>>>(npts, w, rho, grho, rho_tol, cA, cG, part);
  cudaError_t e = cudaGetLastError();
  if (e != cudaSuccess) return e;
  k_reduce3<<<1, 1024, 0, st>>>(nblk, part, out3);
  return cudaGetLastError();
}

}  // namespace xcb
