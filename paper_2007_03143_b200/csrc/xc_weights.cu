// xc_weights.cu -- step (a) of the hot path: partition weights w_i = w_i^q P_A(r_i) / sum_B P_B(r_i)
// (Eq. (9), Alg. 4 l.4.1 PAPER.md:L261), P_B = prod_{C != B} s(mu_BC), mu_BC = (r_B - r_C) / R_BC.
//
//   k_weights_ssf     SSF (reading A2: a = 0.64, 7th-order polynomial), the timed path
//   k_weights_becke   Becke-1988 (reading A1), no compact support
//
// (Product code; shares nothing with oracle/.)
#include <cuda_runtime.h>

#include <algorithm>
#include <cstdint>

#include "xc_internal.h"
#include "xc_kernels.h"

namespace xcb {

// ------------------------------------------------------------------------------------------------
// step (a), hot path for SSF: one CTA per batch, one WARP per non-trivial point, the lanes split the atoms.
// Exact pruning only.  The batch's atom list (planner) is sorted by dmin(atom, batch box) <= r_atom,
// so every scan stops as soon as dmin reaches its bound, and all control flow is warp-uniform.
//
// The kernel is written for a SMALL instruction footprint (plain loops, one inlined copy of every routine, no library
// square roots): its warps run decorrelated, each in another phase of another point, so the whole body has to stay in the
// SM's instruction cache.
//
// Per batch (once): the list atoms (x, y, z, id) and the dmin of every chunk of 32 in shared memory; a table
//   1 / (a R_BC) for the first TB (owner) x TC (partner) list positions -- it takes all the shared memory that is left.
// Per point (one warp, points handed out dynamically):
//   0. r_A < (1-a)/2 R_nn(A)  =>  w = w^q (decided by the planner; the other points are compacted in order).
//   1. nearest atom m, r_min (32 atoms per step, scan while dmin < r_min).  Every distance r_C computed on the way is
//      kept in a per-warp shared-memory row (the first 32 ROWCH list positions, filled lazily chunk by chunk) and reused
//      by all cell products.
//   2. P_A first: P_A = 0 => w = 0 and the point is done.
//   3. owner candidates B, 32 per step, one per lane (scan while dmin < kappa r_min): r_B < kappa r_min, and not
//      already zeroed by the nearest atom or one of the kPre atoms nearest to the batch box (mu_BC >= a <=>
//      r_B - r_C >= a R_BC); each survivor's cell product P_B is then evaluated by the whole warp.
//   Cell product: partners C in chunks of 32 while dmin < kappa r_B (beyond, s(mu_BC) = 1 exactly).  Chunks served by
//   row and table run branch-free, four at a time (independent dependency chains): mu_BC / a = (r_B - r_C) / (a R_BC)
//   clamped to [-1, 1], where the polynomial is exactly 1 and 0; then the product is abandoned if some lane holds 0
//   (P_B = 0) or if it has become negligible (below).  The factor s(0) = 1/2 of the pair (B, B) (table entry 0) is undone
//   by an exact factor 2.  Partners the table or the row do not reach take 1 / (a R_BC) and r_C from the coordinates.
//   Lane products are combined by an xor butterfly (same value in every lane) and the owners are summed in
//   list order, so w is bit-identical from run to run.
// ------------------------------------------------------------------------------------------------
constexpr int kMaxCh = 128;                 // chunk-start dmin values held in shared memory
constexpr int kPre = 8;                     // partners used by the lane-parallel owner pre-filter
constexpr int kTCmax = 512, kTBmax = 64;    // 1/(a R_BC) table: at most kTBmax owner rows x kTCmax partner columns
constexpr int kLcapMax = 4096;              // list atoms held in shared memory (28 B each); beyond: global memory (BIG)
constexpr size_t kSsfSmem = 226 * 1024;     // one CTA per SM
__host__ __device__ constexpr size_t ssf_fixed_bytes(int nwarps, int rowch) {
  return (size_t)kMaxCh * 8 + (size_t)nwarps * rowch * 32 * 8 + 512 * 2;
}

// BIG: the list may be longer than the shared-memory copies (lcap atoms, kMaxCh chunks); else every access is to shared memory
template <bool BIG>
struct SsfCtx {
  const double* sX; const double* sY; const double* sZ; const double* sTab; const double* sDm; double* row;
  const WeightArgs* a; const double* box; int64_t wa_off;
  int nC, nch, lane, lcap, TB, TC, rowch;
  double x, y, z;
  int filled;     // chunks of the row that hold r_C of this point
  int nfac;       // chunks of 32 factors evaluated for this point (reported when WeightArgs::paircnt is set)
};

__device__ __forceinline__ double ssf_poly(double zz) {   // s(mu) for zz = mu / a in [-1, 1]; exactly 1 at -1, 0 at +1
  const double z2 = zz * zz;
  return fma(-zz, fma(z2, fma(z2, fma(z2, -5.0 / 32.0, 21.0 / 32.0), -35.0 / 32.0), 35.0 / 32.0), 0.5);
}
// zz clamped to [-1, 1] with integer operations on the high word only (|zz| >= 1  <=>  exponent field >= 0x3ff): the
// FP64 pipe is left to the arithmetic.  A NaN (never produced here: R_BC > 0, finite coordinates) would come out as +-1.
__device__ __forceinline__ double ssf_clamp(double zz) {
  const int hi = __double2hiint(zz);
  const bool big = (hi & 0x7fffffff) >= 0x3ff00000;
  return __hiloint2double(big ? ((hi & 0x80000000) | 0x3ff00000) : hi, big ? 0 : __double2loint(zz));
}
__device__ __forceinline__ double ssf_factor(double zz) { return ssf_poly(ssf_clamp(zz)); }   // s(mu) for any zz = mu / a

// 1 / sqrt(x) and sqrt(x) for x > 0 over the whole normal range: MUFU.RSQ64H seed (about 20 bits) and two (three for the
// root) fused Newton / Goldschmidt steps -- no special-case branches, no call: 9 and 11 instructions, <= 1 ulp.
__device__ __forceinline__ double ssf_rsqrt(double x) {
  double y;
  asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(x));
  const double hx = 0.5 * x;
  y = fma(y, fma(-hx * y, y, 0.5), y);
  y = fma(y, fma(-hx * y, y, 0.5), y);
  return y;
}
__device__ __forceinline__ double ssf_sqrt(double x) {    // sqrt(0) = 0
  double y;
  asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(x));
  double g = x * y, h = 0.5 * y;
  double r = fma(-g, h, 0.5);
  g = fma(g, r, g); h = fma(h, r, h);
  r = fma(-g, h, 0.5);
  g = fma(g, r, g); h = fma(h, r, h);
  g = fma(fma(-g, g, x), h, g);
  return x > 0.0 ? g : 0.0;
}

__device__ __forceinline__ double ssf_dmin_box(double cx, double cy, double cz, const double* box) {
  const double tx = cx < box[0] ? box[0] - cx : (cx > box[3] ? cx - box[3] : 0.0);
  const double ty = cy < box[1] ? box[1] - cy : (cy > box[4] ? cy - box[4] : 0.0);
  const double tz = cz < box[2] ? box[2] - cz : (cz > box[5] ? cz - box[5] : 0.0);
  // a hair below the true distance: the early exits must never cut an atom that matters
  return sqrt(tx * tx + ty * ty + tz * tz) * (1.0 - 1e-12) - 1e-12;
}

// coordinates of list entry c: shared memory for c < lcap, global beyond (BIG: systems with more atoms than fit)
template <bool BIG>
__device__ __forceinline__ void ssf_atom(const SsfCtx<BIG>& s, int c, double& cx, double& cy, double& cz) {
  if (!BIG || c < s.lcap) { cx = s.sX[c]; cy = s.sY[c]; cz = s.sZ[c]; return; }
  const int at = s.a->watoms[s.wa_off + c];
  cx = s.a->atoms[3 * at]; cy = s.a->atoms[3 * at + 1]; cz = s.a->atoms[3 * at + 2];
}
template <bool BIG>
__device__ __forceinline__ double ssf_chunk_dmin(const SsfCtx<BIG>& s, int ch) {
  if (!BIG || ch < kMaxCh) return s.sDm[ch];
  double cx, cy, cz;
  ssf_atom(s, ch * 32, cx, cy, cz);
  return ssf_dmin_box(cx, cy, cz, s.box);
}
// number of leading chunks whose first (smallest) dmin is below `bound`
template <bool BIG>
__device__ __forceinline__ int ssf_nscan(const SsfCtx<BIG>& s, double bound) {
#pragma unroll 1
  for (int base = 0; base < s.nch; base += 32) {
    const int ch = base + s.lane;
    const double v = ch < s.nch ? ssf_chunk_dmin(s, ch) : 1e300;
    const unsigned m = __ballot_sync(0xffffffffu, v >= bound);
    if (m) return base + __ffs(m) - 1;
  }
  return s.nch;
}

// r_C of list position c (1e300 past the end of the list)
template <bool BIG>
__device__ __forceinline__ double ssf_dist(const SsfCtx<BIG>& s, int c) {
  double cx, cy, cz;
  ssf_atom(s, min(c, s.nC - 1), cx, cy, cz);
  const double dx = s.x - cx, dy = s.y - cy, dz = s.z - cz;
  const double r = ssf_sqrt(fma(dx, dx, fma(dy, dy, dz * dz)));
  return c < s.nC ? r : 1e300;
}
// make sure the row holds r_C of the chunks [0, n) (n <= rowch, warp-uniform)
template <bool BIG>
__device__ __forceinline__ void ssf_fill(SsfCtx<BIG>& s, int n) {
#pragma unroll 1
  for (int j = s.filled; j < n; ++j) s.row[(j << 5) + s.lane] = ssf_dist(s, (j << 5) + s.lane);
  s.filled = max(s.filled, n);
  __syncwarp();
}
// 1 / (a R_BC) from the coordinates
__device__ __forceinline__ double ssf_inv_aR(double ex, double ey, double ez) {
  return ssf_rsqrt(fma(ex, ex, fma(ey, ey, ez * ez))) * (1.0 / 0.64);
}

// P_B = prod_C s(mu_BC).  bb = list position of B (warp-uniform, -1: not in the list), rB = r_B.
// (Bx, By, Bz) is only read for bb < 0; a list atom's coordinates are fetched where the table does not reach.
// thresh: the product is abandoned (returns 0) as soon as the product over the partners visited so far -- an upper bound
// of P_B, every factor being <= 1 -- is below thresh.  For an owner other than the parent thresh = 2^-61 of the running
// sum of the owners before it: adding such a P_B would not change the fp64 sum, so w stays bit-identical.
template <bool BIG>
__device__ __forceinline__ double ssf_cell_product(SsfCtx<BIG>& s, int bb, double Bx, double By, double Bz, double rB, double thresh) {
  const unsigned FULL = 0xffffffffu;
  const double kappa = (1.0 + 0.64) / (1.0 - 0.64);
  const double krB = kappa * rB;
  const int nscan = ssf_nscan(s, krB);                     // every later C has r_C >= kappa r_B: factor 1
  const int nrow = min(nscan, s.rowch);                    // chunks whose r_C the row serves
  if (nrow > s.filled) ssf_fill(s, nrow);
  const bool tab = bb >= 0 && bb < s.TB;
  const int tch = tab ? min(nrow, s.TC >> 5) : 0;          // chunks served by row and table
  if (bb >= 0 && nscan > tch) ssf_atom(s, bb, Bx, By, Bz);
  double part = 1.0;
  // Abandon test, one integer warp reduction: log2 of the product over the 32 lanes, bounded from ABOVE in fixed point
  // with 10 fractional bits: for x = m 2^e, m in [1, 2):  e + (m - 1) <= log2 x <= e + (m - 1) + 0.0861.  The high word
  // >> 10 is (e + 1023) 2^10 + the top 10 mantissa bits (truncated: + 1).  The bound is within 2^2.8 of the product;
  // thresh is bounded from BELOW the same way, so `true` implies product < thresh rigorously.  A lane that holds exactly
  // 0 (some mu_BC >= a: P_B = 0) makes the bound fall below any thresh >= 2^-1000; for the parent thresh is 2^-1000: its
  // product is only abandoned when it is 0 or, were it kept, would give w < 2^-990 w^q.
  const int lt = (__double2hiint(thresh) >> 10) - (1023 << 10);
  auto negligible = [&]() {
    const int I = __double2hiint(part) >> 10;
    const int ub = __reduce_add_sync(FULL, I) - 32 * (1023 << 10) + 32 * (1 + 89);   // 89 = ceil(0.0861 * 1024)
    return ub < lt;                                        // same value in every lane
  };
  // ---- row x table, branch-free.  (B, B): entry 0, factor 1/2; c >= nC: r_C = 1e300, entry 1, factor 1.  A lane that
  //      meets mu_BC >= a holds exactly 0 from then on. ----
  const double* trow = s.sTab + (size_t)max(bb, 0) * s.TC + s.lane;
  const double* rrow = s.row + s.lane;
  int j = 0;
#pragma unroll 1
  for (; j + 4 <= tch; j += 4) {
    const double f0 = ssf_factor((rB - rrow[j << 5]) * trow[j << 5]);
    const double f1 = ssf_factor((rB - rrow[(j + 1) << 5]) * trow[(j + 1) << 5]);
    const double f2 = ssf_factor((rB - rrow[(j + 2) << 5]) * trow[(j + 2) << 5]);
    const double f3 = ssf_factor((rB - rrow[(j + 3) << 5]) * trow[(j + 3) << 5]);
    part *= (f0 * f1) * (f2 * f3);
    if (negligible()) { s.nfac += j + 4; return 0.0; }
  }
  if (j < tch) {
#pragma unroll 1
    for (; j < tch; ++j) part *= ssf_factor((rB - rrow[j << 5]) * trow[j << 5]);
    if (negligible()) { s.nfac += tch; return 0.0; }
  }
  s.nfac += tch;
  // ---- partners the table does not reach: R_BC (and, past the row, r_C) from the coordinates ----
#pragma unroll 1
  for (int ch = tch; ch < nscan; ++ch) {
    const int c = (ch << 5) + s.lane;
    double cx, cy, cz;
    ssf_atom(s, min(c, s.nC - 1), cx, cy, cz);
    double rC;
    if (ch < nrow) {
      rC = rrow[ch << 5];
    } else {
      const double dx = s.x - cx, dy = s.y - cy, dz = s.z - cz;
      rC = c < s.nC ? ssf_sqrt(fma(dx, dx, fma(dy, dy, dz * dz))) : 1e300;
    }
    if (!__any_sync(FULL, rC < krB)) continue;             // 32 factors exactly 1
    const double zz = (c < s.nC && c != bb) ? (rB - rC) * ssf_inv_aR(Bx - cx, By - cy, Bz - cz) : -1.0;   // mu_BC / a
    part *= ssf_factor(zz);
    ++s.nfac;
    if (negligible()) return 0.0;
  }
#pragma unroll
  for (int o = 16; o >= 1; o >>= 1) part *= __shfl_xor_sync(FULL, part, o);
  // table path: the chunk of B itself is always visited (dmin_B <= r_B < kappa r_B; bb < TB <= min(TC, 32 rowch)) and
  // contributed s(0) = 1/2
  if (tab) part *= 2.0;
  return part;
}

template <int NW, int ROWCH, bool BIG>
__global__ void __launch_bounds__(NW * 32, 1) k_weights_ssf(WeightArgs a, const int32_t* __restrict__ batch_ids, int lcap, int TB, int TC) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  __shared__ int sCnt[NW];
  __shared__ int sNext;
  constexpr int NT = NW * 32;
  const unsigned FULL = 0xffffffffu;
  const int bid = batch_ids[blockIdx.x];
  const BatchRec b = a.batches[bid];
  const int nC = b.wa_nC, nB = b.wa_nB;
  double* sX = (double*)smem_raw;                        // [lcap] x 3
  double* sY = sX + lcap;
  double* sZ = sY + lcap;
  double* sDm = sZ + lcap;                               // [kMaxCh]
  double* sRow = sDm + kMaxCh;                           // [NW][32 ROWCH]: r_C of the first list positions, per warp
  double* sTab = sRow + NW * ROWCH * 32;                 // [TB][TC]
  int* sId = (int*)(sTab + (size_t)TB * TC);             // [lcap]
  short* sList = (short*)(sId + lcap);                   // compacted non-trivial points of the batch (<= 512)
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const double aa = 0.64, kappa = (1.0 + aa) / (1.0 - aa);
  const double* box = a.wbox + (size_t)6 * bid;

  // ---- 0. the first ntriv points of the batch have r_A < (1-a)/2 R_nn(A): w = w^q, set once when the plan was made
  //         (planner); ordered compaction of the others (N_q^j <= 512) ----
  int total = 0;
  for (int p0 = 0; p0 < b.nq; p0 += NT) {
    const int p = p0 + (int)threadIdx.x;
    const bool live = p >= b.ntriv && p < b.nq;
    const unsigned lmask = __ballot_sync(FULL, live);
    if (lane == 0) sCnt[warp] = __popc(lmask);
    __syncthreads();
    int off = total;
#pragma unroll 1
    for (int k = 0; k < NW; ++k) {
      if (k < warp) off += sCnt[k];
      total += sCnt[k];
    }
    if (live) sList[off + __popc(lmask & ((1u << lane) - 1u))] = (short)p;
    __syncthreads();
  }
  if (threadIdx.x == 0) sNext = NW;
  if (total == 0) return;
  const int nS = min(nC, lcap), nch = (nC + 31) >> 5;
#pragma unroll 1
  for (int c = threadIdx.x; c < nS; c += NT) {
    const int at = a.watoms[b.wa_off + c];
    const double cx = a.atoms[3 * at], cy = a.atoms[3 * at + 1], cz = a.atoms[3 * at + 2];
    sX[c] = cx; sY[c] = cy; sZ[c] = cz;
    sId[c] = at;
    if ((c & 31) == 0 && (c >> 5) < kMaxCh) sDm[c >> 5] = ssf_dmin_box(cx, cy, cz, box);
  }
  if (BIG) {
    for (int ch = (lcap >> 5) + threadIdx.x; ch < min(nch, kMaxCh); ch += NT) {
      const int at = a.watoms[b.wa_off + ch * 32];
      sDm[ch] = ssf_dmin_box(a.atoms[3 * at], a.atoms[3 * at + 1], a.atoms[3 * at + 2], box);
    }
  }
  __syncthreads();
  // ---- the table 1 / (a R_BC): rows = the first TB list atoms, columns = the first TC ----
  if (total < 4) TB = 0;                                   // too few points to pay for the table
  TC = min(TC, (nC + 31) & ~31);
  TB = min(TB, min(nS, TC));
#pragma unroll 1
  for (int e = threadIdx.x; e < TB * TC; e += NT) {
    const int bb = e / TC, c = e - bb * TC;
    double v = 1.0;                                        // neutral entry for c >= nC (r_C = 1e300 there)
    if (c < nC && c != bb) v = ssf_inv_aR(sX[bb] - sX[c], sY[bb] - sY[c], sZ[bb] - sZ[c]);   // TC <= 512 <= lcap or nC <= lcap
    sTab[(size_t)bb * TC + c] = c == bb ? 0.0 : v;
  }
  __syncthreads();

  SsfCtx<BIG> s;
  s.sX = sX; s.sY = sY; s.sZ = sZ; s.sTab = sTab; s.sDm = sDm; s.row = sRow + warp * (ROWCH * 32); s.a = &a; s.box = box;
  s.wa_off = b.wa_off; s.nC = nC; s.nch = nch; s.lane = lane; s.lcap = lcap; s.TB = TB; s.TC = TC; s.rowch = ROWCH;
  const int npre = min(kPre, nC);
  for (int n = warp; n < total;) {
    const int64_t gi = (int64_t)b.pt_off + sList[n];
    s.x = a.px[gi]; s.y = a.py[gi]; s.z = a.pz[gi];
    s.filled = 0;
    s.nfac = 0;
    const int A = a.parent[gi];
    __syncwarp();                                          // the previous point's readers of the row are done
    // ---- 1. nearest atom: per-lane minimum while the chunks can still hold a nearer atom (the stop test uses the
    //         high word of the warp minimum: an upper bound of r_min, so it never stops early) ----
    double best = 1e300, rub = 1e300;
    int bj = 0;
#pragma unroll 1
    for (int j = 0; j < nch && (j == 0 || ssf_chunk_dmin(s, j) < rub); ++j) {
      const double rr = ssf_dist(s, (j << 5) + lane);
      if (j < ROWCH) { s.row[(j << 5) + lane] = rr; s.filled = j + 1; }
      if (rr < best) { best = rr; bj = j; }
      rub = __hiloint2double((int)__reduce_min_sync(FULL, (unsigned)__double2hiint(best)), -1);
    }
    __syncwarp();
    // exact argmin over the lanes: r >= 0, so the bit patterns order like the values
    double rmin;
    int im;
    {
      const unsigned hi = (unsigned)__double2hiint(best);
      const unsigned mhi = __reduce_min_sync(FULL, hi);
      const unsigned lo = hi == mhi ? (unsigned)__double2loint(best) : 0xffffffffu;
      const unsigned mlo = __reduce_min_sync(FULL, lo);
      rmin = __hiloint2double((int)mhi, (int)mlo);
      const int src = __ffs(__ballot_sync(FULL, hi == mhi && lo == mlo)) - 1;
      im = (__shfl_sync(FULL, bj, src) << 5) + src;
    }
    const double own_lim = kappa * rmin;
    // ---- 2. the parent's cell product first, 3. then the other owners: one loop, one inlined cell product ----
    const double Ax = a.atoms[3 * A], Ay = a.atoms[3 * A + 1], Az = a.atoms[3 * A + 2];
    double rA;
    { const double dx = s.x - Ax, dy = s.y - Ay, dz = s.z - Az; rA = ssf_sqrt(fma(dx, dx, fma(dy, dy, dz * dz))); }
    double result = 0.0;
    if (!(rA >= own_lim && rA > rmin)) {
      int ia = -1;                                         // list position of the parent
#pragma unroll 1
      for (int c0 = 0; c0 < nC && ia < 0; c0 += 32) {
        const int c = c0 + lane;
        const unsigned m = __ballot_sync(FULL, c < nC && ((!BIG || c < lcap) ? sId[c] : a.watoms[b.wa_off + c]) == A);
        if (m) ia = c0 + __ffs(m) - 1;
      }
      double mx, my, mz;
      ssf_atom(s, im, mx, my, mz);
      const int nown = min(ssf_nscan(s, own_lim) << 5, nB);
      double PA = 0.0, sum = 0.0, rB = 0.0;
      int b0 = -32;
      unsigned mask = 0;
      bool first = true;
      for (;;) {
        int bs;
        double rBs;
        if (first) {
          bs = ia; rBs = rA;
        } else {
          while (!mask) {                                  // next chunk of owner candidates, one per lane
            b0 += 32;
            if (b0 >= nown) break;
            const int bb = b0 + lane;
            if ((b0 >> 5) < ROWCH) {
              if ((b0 >> 5) >= s.filled) ssf_fill(s, (b0 >> 5) + 1);
              rB = s.row[bb];
            } else {
              rB = ssf_dist(s, bb);
            }
            bool cand = bb < nB && bb != ia && rB < own_lim;   // else r_B >= kappa r_min: P_B = 0 exactly
            if (!__any_sync(FULL, cand)) continue;
            // pre-filter: mu_BC >= a for the nearest atom or one of the first kPre list atoms  =>  P_B = 0
            {
              double bx, by, bz;
              ssf_atom(s, min(bb, nC - 1), bx, by, bz);
              const double u = rB - rmin;
              const double ex = bx - mx, ey = by - my, ez = bz - mz;
              if (im != bb && u > 0.0 && u * u >= (aa * aa) * fma(ex, ex, fma(ey, ey, ez * ez))) cand = false;
            }
            if (TB >= npre && b0 + 32 <= TC) {
              // 1 / (a R_Bk) = table entry (k, B): row k is warp-uniform, the lanes read consecutive columns;
              // the entry (B, B) is 0, so k = B never fires
              for (int k = 0; k < npre; ++k)
                if ((rB - s.row[k]) * sTab[(size_t)k * TC + bb] >= 1.0) cand = false;
            }
            mask = __ballot_sync(FULL, cand);
          }
          if (!mask) break;                                // no owner candidates left
          const int src = __ffs(mask) - 1;
          mask &= mask - 1;
          bs = b0 + src; rBs = __shfl_sync(FULL, rB, src);
        }
        // an owner other than the parent may be dropped once it is below 2^-61 of the sum so far; the parent below 2^-1000
        const double PB = ssf_cell_product(s, bs, Ax, Ay, Az, rBs, first ? 9.332636185032189e-302 : sum * 4.3368086899420177e-19);
        if (first) {
          if (PB == 0.0) break;                            // P_A = 0: w = 0
          PA = PB; first = false;
        }
        sum += PB;
      }
      if (PA != 0.0) result = a.wq[gi] * PA / sum;
    }
    if (lane == 0) {
      a.w[gi] = result;
      n = atomicAdd(&sNext, 1);
      if (a.paircnt) atomicAdd(a.paircnt, (unsigned long long)s.nfac * 32ull);   // profiling builds of bench.py only
    }
    n = __shfl_sync(FULL, n, 0);
  }
}

// ------------------------------------------------------------------------------------------------
// Becke-1988 (three iterations of p(t) = 1.5 t - 0.5 t^3, no size adjustment; reading A1/A2): one CTA per batch, one
// WARP per point.  The batch's atom list (every atom, nearest to the batch box first) sits in shared memory; the lanes
// split the partners and the products are combined with an xor butterfly (same value in every lane, fixed order).
// The parent first (always in full), then the owners nearest to the batch first.  An owner's product is abandoned as
// soon as an upper bound of it (every factor is <= 1) is below 2^-60 of the sum so far: adding such a term would not
// change the fp64 sum, so w is bit-identical to the full O(N_A^2) evaluation in this order.
// ------------------------------------------------------------------------------------------------
__device__ __forceinline__ double s_becke(double mu) {
  double p = mu;
#pragma unroll
  for (int k = 0; k < 3; ++k) p = 1.5 * p - 0.5 * p * p * p;
  return 0.5 * (1.0 - p);
}

__global__ void __launch_bounds__(kWeightThreads) k_weights_becke(WeightArgs a, const int32_t* __restrict__ batch_ids, int nwarps) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  const unsigned FULL = 0xffffffffu;
  const BatchRec b = a.batches[batch_ids ? batch_ids[blockIdx.x] : blockIdx.x];
  const int nC = b.wa_nC, nB = b.wa_nC;
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
  for (int p = warp; p < b.nq; p += nwarps) {
    const int64_t gi = (int64_t)b.pt_off + p;
    const double x = a.px[gi], y = a.py[gi], z = a.pz[gi], base = a.wq[gi];
    const int A = a.parent[gi];
    double result = base;
    if (a.natoms > 1) {
      for (int c = lane; c < nC; c += 32) {
        double dx = x - sXYZ[3 * c], dy = y - sXYZ[3 * c + 1], dz = z - sXYZ[3 * c + 2];
        sD[c] = sqrt(dx * dx + dy * dy + dz * dz);
      }
      __syncwarp();
      double sum = 0.0, PA = 0.0;
      const int nsteps = (nC + 31) >> 5;
      int ia = -1;                                   // list position of the parent
#pragma unroll 1
      for (int c0 = 0; c0 < nC && ia < 0; c0 += 32) {
        const unsigned m = __ballot_sync(FULL, c0 + lane < nC && sAt[c0 + lane] == A);
        if (m) ia = c0 + __ffs(m) - 1;
      }
      unsigned premask = 0xffffffffu;
      for (int ib = -1; ib < nB; ++ib) {
        if (ib >= 0 && (ib & 31) == 0) {
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
        if (bb < 0 || (ib >= 0 && bb == ia)) continue;
        if (ib >= 0 && !((premask >> (ib & 31)) & 1u)) continue;
        const double thresh = ib >= 0 ? sum * 8.673617379884035e-19 : 0.0;   // 2^-60
        const double rB = sD[bb];
        const int Bid = sAt[bb];
        const double* iR = a.invR + (size_t)Bid * a.natoms;
        double part = 1.0;
        for (int k = 0; k < nsteps; ++k) {
          const int c = (k << 5) + lane;
          if (c < nC && c != bb) part *= s_becke((rB - sD[c]) * __ldg(iR + sAt[c]));
          if (thresh > 0.0) {                                                    // negligible owner?
            // log2 of the product over the 32 lanes, bounded from ABOVE in fixed point with 10 fractional bits by one integer
            // warp reduction: for v = m 2^e, m in [1, 2):  e + (m - 1) <= log2 v <= e + (m - 1) + 0.0861.  The high word >> 10
            // is (e + 1023) 2^10 + the top 10 mantissa bits (truncated: + 1); 89 = ceil(0.0861 * 1024).  thresh is bounded
            // from BELOW the same way, so `ub < lt` implies product < thresh rigorously.
            const int ub = __reduce_add_sync(FULL, __double2hiint(part) >> 10) - 32 * (1023 << 10) + 32 * (1 + 89);
            if (ub < (__double2hiint(thresh) >> 10) - (1023 << 10)) { part = -1.0; break; }
          }
        }
        if (part < 0.0) continue;                                               // warp-uniform
#pragma unroll
        for (int o = 16; o >= 1; o >>= 1) part *= __shfl_xor_sync(FULL, part, o);
        sum += part;
        if (Bid == A) PA = part;
      }
      result = base * PA / sum;
      __syncwarp();
    }
    if (lane == 0) a.w[gi] = result;
  }
}

// ------------------------------------------------------------------------------------------------

// ------------------------------------------------------------------------------------------------
// launchers
// ------------------------------------------------------------------------------------------------
template <int NW, int ROWCH, bool BIG>
static cudaError_t launch_ssf_t(const WeightArgs& a, const int32_t* batch_ids, int nbatches, int max_list, cudaStream_t st) {
  // shared-memory split: the atom list (28 B per atom), the per-warp distance rows, the rest for rows of the 1/(a R_BC) table
  const int lcap = std::min((max_list + 31) / 32 * 32, kLcapMax);
  const int TC = std::min((max_list + 31) / 32 * 32, kTCmax);
  const long avail = (long)kSsfSmem - (long)ssf_fixed_bytes(NW, ROWCH) - (long)lcap * 28;
  const int TB = (int)std::max(0L, std::min<long>(std::min(kTBmax, TC), avail / ((long)TC * 8)));
  const size_t smem = ssf_fixed_bytes(NW, ROWCH) + (size_t)lcap * 28 + (size_t)TB * TC * 8;
  cudaError_t e = cudaFuncSetAttribute(k_weights_ssf<NW, ROWCH, BIG>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
  if (e != cudaSuccess) return e;
  k_weights_ssf<NW, ROWCH, BIG><<<nbatches, NW * 32, smem, st>>>(a, batch_ids, lcap, TB, TC);
  return cudaGetLastError();
}

cudaError_t launch_weights_ssf(const WeightArgs& a, const int32_t* batch_ids, int nbatches, int max_list, cudaStream_t st) {
  if (nbatches <= 0) return cudaSuccess;
  // 24 warps (80 registers) per SM; rows of 256 list positions for short lists, of 512 otherwise (measured on c2 / c4 / c5 / g1
  // against 16-32 warps and rows of 256-512: DESIGN.md 5a)
  if (max_list > kLcapMax) return launch_ssf_t<16, 16, true>(a, batch_ids, nbatches, max_list, st);
  if (max_list <= 256) return launch_ssf_t<24, 8, false>(a, batch_ids, nbatches, max_list, st);
  return launch_ssf_t<24, 16, false>(a, batch_ids, nbatches, max_list, st);
}

cudaError_t launch_weights_becke(const WeightArgs& a, const int32_t* batch_ids, int nbatches, int nwarps, int max_list, cudaStream_t st) {
  if (nbatches <= 0) return cudaSuccess;
  const size_t smem = weights_smem_bytes(max_list, nwarps);
  cudaError_t e = cudaFuncSetAttribute(k_weights_becke, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)std::max<size_t>(smem, 1024));
  if (e != cudaSuccess) return e;
  k_weights_becke<<<nbatches, kWeightThreads, smem, st>>>(a, batch_ids, nwarps);
  return cudaGetLastError();
}

}  // namespace xcb
