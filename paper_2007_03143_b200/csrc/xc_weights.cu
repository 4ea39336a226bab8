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
  int nfac;       // chunks of 32 factors evaluated for this point (only counted when WeightArgs::paircnt is set)
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
      ++s.nfac;
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
    ++s.nfac;
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
    ++s.nfac;
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

  // ---- 0. the first ntriv points of the batch have r_A < (1-a)/2 R_nn(A): w = w^q, set once when the plan was made
  //         (planner); ordered compaction of the others ----
  const bool live = (int)threadIdx.x >= b.ntriv && (int)threadIdx.x < b.nq;
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
    s.nfac = 0;
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
// launchers
// ------------------------------------------------------------------------------------------------
cudaError_t launch_weights_ssf(const WeightArgs& a, const int32_t* batch_ids, int nbatches, int max_list, cudaStream_t st) {
  if (nbatches <= 0) return cudaSuccess;
  // shared-memory split: the whole atom list if it fits (28 B per atom), the rest for rows of the 1/(a R_BC) table
  const int lcap = std::min((max_list + 31) / 32 * 32, kSsfMaxLcap);
  const int tabB = std::min(32, (int)((kSsfSmem - kSsfFixed - (size_t)lcap * 28) / ((size_t)kTabC * 8)));
  cudaError_t e = cudaFuncSetAttribute(k_weights_ssf, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kSsfSmem);
  if (e != cudaSuccess) return e;
  k_weights_ssf<<<nbatches, kSsfThreads, kSsfSmem, st>>>(a, batch_ids, lcap, tabB);
  return cudaGetLastError();
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
