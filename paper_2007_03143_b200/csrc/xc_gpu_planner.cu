// xc_gpu_planner.cu -- step (b) on the GPU ("could be implemented on GPU", L401 / L427:
// host batching is the paper's scaling bottleneck): the grid points (Eq. (9), O3 order) and the global
// recursive median bisection of the pooled point cloud into cuboids of <= max_batch_pts points (reading A8),
// level by level, every segment of a level at once.
//
// The result is IDENTICAL to the host planner's (xc_planner.cpp: same bounding boxes, same axis rule, same split sizes,
// the `half` smallest points by (coordinate, canonical index) go left), so a plan does not depend on where it was made
// (tested: device plan == host-only plan).  Per level: segment bounding boxes (warp-aggregated integer atomics on
// order-preserving keys), one tiny kernel for axis and split size, then three stable radix sorts (library primitive:
// cub::DeviceRadixSort) that order every segment by (coordinate along its axis, index): by index, by coordinate, by segment.
// (Product code; shares nothing with oracle/.)
#include <cuda_runtime.h>

#include <cub/cub.cuh>

#include <algorithm>
#include <cstdint>
#include <cstring>
#include <string>
#include <vector>

#include "xc_internal.h"

namespace xcb {

namespace {

#define GP_CU(call)                     \
  do {                                  \
    cudaError_t _e = (call);            \
    if (_e != cudaSuccess) return _e;   \
  } while (0)

// order-preserving map double -> uint64 (-0.0 counts as +0.0, as in the host's comparisons)
__device__ __forceinline__ unsigned long long okey(double v) {
  v = v + 0.0;
  const unsigned long long b = (unsigned long long)__double_as_longlong(v);
  return (b >> 63) ? ~b : (b | 0x8000000000000000ULL);
}

// O3: r = R_A + r_i u_k, canonical order (atom, radial, angular); product and sum rounded separately, like the host's
__global__ void k_grid(int64_t npts, int64_t per_atom, int n_ang, const double* __restrict__ atoms, const double* __restrict__ rr,
                       const double* __restrict__ au, double* __restrict__ cx, double* __restrict__ cy, double* __restrict__ cz) {
  const int64_t p = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (p >= npts) return;
  const int a = (int)(p / per_atom);
  const int64_t q = p % per_atom;
  const int i = (int)(q / n_ang), k = (int)(q % n_ang);
  cx[p] = __dadd_rn(atoms[3 * a], __dmul_rn(rr[i], au[3 * k]));
  cy[p] = __dadd_rn(atoms[3 * a + 1], __dmul_rn(rr[i], au[3 * k + 1]));
  cz[p] = __dadd_rn(atoms[3 * a + 2], __dmul_rn(rr[i], au[3 * k + 2]));
}

struct Seg {          // one cuboid of the current level
  int32_t begin, end; // positions [begin, end) of the ordered point array
  int32_t axis, half; // split axis and size of the left part; half = 0: leaf (not split any more)
};

__global__ void k_iota(int64_t n, int32_t* idx) {
  const int64_t p = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (p < n) idx[p] = (int32_t)p;
}

// bounding boxes of the segments that are still to be split: warp-aggregated atomic min / max on ordered keys
__global__ void k_bounds(int64_t n, const int32_t* __restrict__ idx, const int32_t* __restrict__ seg, const Seg* __restrict__ segs,
                         const double* __restrict__ cx, const double* __restrict__ cy, const double* __restrict__ cz,
                         unsigned long long* __restrict__ box /* [nseg][6]: min xyz, max xyz */, int maxp) {
  const int64_t p = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  const bool in = p < n;
  const int s = in ? seg[p] : -1;
  bool act = false;
  unsigned long long k[3] = {0, 0, 0};
  if (in) {
    const Seg sg = segs[s];
    act = sg.end - sg.begin > maxp;
    if (act) { const int32_t i = idx[p]; k[0] = okey(cx[i]); k[1] = okey(cy[i]); k[2] = okey(cz[i]); }
  }
  const unsigned FULL = 0xffffffffu;
  const int s0 = __shfl_sync(FULL, s, 0);
  const bool uniform = __all_sync(FULL, s == s0);
  if (uniform) {
    if (!__any_sync(FULL, act)) return;
#pragma unroll
    for (int c = 0; c < 3; ++c) {
      unsigned long long lo = k[c], hi = k[c];
#pragma unroll
      for (int o = 16; o >= 1; o >>= 1) {
        const unsigned long long l2 = __shfl_xor_sync(FULL, lo, o), h2 = __shfl_xor_sync(FULL, hi, o);
        lo = l2 < lo ? l2 : lo; hi = h2 > hi ? h2 : hi;
      }
      if ((threadIdx.x & 31) == 0) { atomicMin(box + (size_t)s0 * 6 + c, lo); atomicMax(box + (size_t)s0 * 6 + 3 + c, hi); }
    }
  } else if (act) {
#pragma unroll
    for (int c = 0; c < 3; ++c) { atomicMin(box + (size_t)s * 6 + c, k[c]); atomicMax(box + (size_t)s * 6 + 3 + c, k[c]); }
  }
}

__device__ __forceinline__ double unkey(unsigned long long k) {
  const unsigned long long b = (k >> 63) ? (k & 0x7fffffffffffffffULL) : ~k;
  return __longlong_as_double((long long)b);
}

// axis = first axis of strictly largest extent; half = n / 2, rounded down to a multiple of 64 (at least 64) when the batches
// are tiled by 64 points -- the host planner's rule
__global__ void k_decide(int nseg, Seg* segs, const unsigned long long* __restrict__ box, int maxp, int* n_active) {
  const int s = blockIdx.x * blockDim.x + threadIdx.x;
  if (s >= nseg) return;
  Seg sg = segs[s];
  const int64_t n = sg.end - sg.begin;
  sg.axis = 0; sg.half = 0;
  if (n > maxp) {
    double ext[3];
    for (int c = 0; c < 3; ++c) ext[c] = __dsub_rn(unkey(box[(size_t)s * 6 + 3 + c]), unkey(box[(size_t)s * 6 + c]));
    int ax = 0;
    for (int c = 1; c < 3; ++c) if (ext[c] > ext[ax]) ax = c;
    int64_t half = n / 2;
    if (maxp >= 64 && n >= 128) half = half / 64 * 64 > 64 ? half / 64 * 64 : 64;
    sg.axis = ax; sg.half = (int32_t)half;
    atomicAdd(n_active, 1);
  }
  segs[s] = sg;
}

// sort keys of the level: the coordinate along the segment's axis (0 for points of finished segments)
__global__ void k_keys(int64_t n, const int32_t* __restrict__ idx, const int32_t* __restrict__ seg, const Seg* __restrict__ segs,
                       const double* __restrict__ cx, const double* __restrict__ cy, const double* __restrict__ cz,
                       unsigned long long* __restrict__ key, unsigned long long* __restrict__ val) {
  const int64_t p = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (p >= n) return;
  const int s = seg[p];
  const int32_t i = idx[p];
  const Seg sg = segs[s];
  unsigned long long k = 0;
  if (sg.half > 0) k = okey(sg.axis == 0 ? cx[i] : (sg.axis == 1 ? cy[i] : cz[i]));
  key[p] = k;
  val[p] = ((unsigned long long)(unsigned)s << 32) | (unsigned)i;
}
__global__ void k_unpack(int64_t n, const unsigned long long* __restrict__ val, int32_t* __restrict__ seg, int32_t* __restrict__ idx) {
  const int64_t p = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (p >= n) return;
  seg[p] = (int32_t)(val[p] >> 32);
  idx[p] = (int32_t)(val[p] & 0xffffffffu);
}
// the segments of the next level (order kept: left part, right part), and the new segment of every position
__global__ void k_children(int nseg, const Seg* __restrict__ segs, const int32_t* __restrict__ newbase, Seg* __restrict__ out) {
  const int s = blockIdx.x * blockDim.x + threadIdx.x;
  if (s >= nseg) return;
  const Seg sg = segs[s];
  const int b = newbase[s];
  if (sg.half > 0) {
    out[b] = Seg{sg.begin, sg.begin + sg.half, 0, 0};
    out[b + 1] = Seg{sg.begin + sg.half, sg.end, 0, 0};
  } else {
    out[b] = Seg{sg.begin, sg.end, 0, 0};
  }
}
__global__ void k_reseg(int64_t n, int32_t* __restrict__ seg, const Seg* __restrict__ segs, const int32_t* __restrict__ newbase) {
  const int64_t p = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (p >= n) return;
  const int s = seg[p];
  const Seg sg = segs[s];
  seg[p] = newbase[s] + ((sg.half > 0 && p >= sg.begin + sg.half) ? 1 : 0);
}
__global__ void k_fill_box(int64_t n6, unsigned long long* box) {
  const int64_t p = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (p < n6) box[p] = (p % 6) < 3 ? ~0ULL : 0ULL;
}

template <class T>
struct DevBuf {
  T* p = nullptr;
  ~DevBuf() { if (p) cudaFree(p); }
  cudaError_t alloc(size_t n) { return cudaMalloc((void**)&p, std::max<size_t>(n, 1) * sizeof(T)); }
};

// ---- ordering inside the batches (xc_planner.cpp: Morton order, then the SSF-trivial points first) and the permuted arrays ----
__device__ __forceinline__ unsigned long long spread21(unsigned v) {
  unsigned long long x = v & 0x1fffff;
  x = (x | x << 32) & 0x1f00000000ffffULL; x = (x | x << 16) & 0x1f0000ff0000ffULL;
  x = (x | x << 8) & 0x100f00f00f00f00fULL; x = (x | x << 4) & 0x10c30c30c30c30c3ULL; x = (x | x << 2) & 0x1249249249249249ULL;
  return x;
}
// r_A < lim R_nn(A): w = w^q exactly under SSF; the host's arithmetic, operation by operation
__device__ __forceinline__ bool trivial_point(int32_t i, int64_t per_atom, int natoms, const double* atoms, const double* rnn, double lim,
                                              const double* cx, const double* cy, const double* cz) {
  if (natoms == 1) return true;
  const int a = (int)(i / per_atom);
  const double dx = __dsub_rn(cx[i], atoms[3 * a]), dy = __dsub_rn(cy[i], atoms[3 * a + 1]), dz = __dsub_rn(cz[i], atoms[3 * a + 2]);
  const double r2 = __dadd_rn(__dadd_rn(__dmul_rn(dx, dx), __dmul_rn(dy, dy)), __dmul_rn(dz, dz));
  return __dsqrt_rn(r2) < __dmul_rn(lim, rnn[a]);
}
__global__ void k_morton(int64_t n, const int32_t* __restrict__ idx, const int32_t* __restrict__ seg, const unsigned long long* __restrict__ box,
                         const double* __restrict__ cx, const double* __restrict__ cy, const double* __restrict__ cz,
                         unsigned long long* __restrict__ key, unsigned long long* __restrict__ val) {
  const int64_t p = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (p >= n) return;
  const int s = seg[p];
  const int32_t i = idx[p];
  double lo[3], ext = 1e-300;
  for (int c = 0; c < 3; ++c) {
    lo[c] = unkey(box[(size_t)s * 6 + c]);
    const double e = __dsub_rn(unkey(box[(size_t)s * 6 + 3 + c]), lo[c]);
    ext = e > ext ? e : ext;
  }
  const double v[3] = {cx[i], cy[i], cz[i]};
  unsigned long long k = 0;
  for (int c = 0; c < 3; ++c) {
    const double t = floor(__dmul_rn(__ddiv_rn(__dsub_rn(v[c], lo[c]), ext), 1048576.0));
    const unsigned q = (unsigned)(t < 1048575.0 ? t : 1048575.0);
    k |= spread21(q) << c;
  }
  key[p] = k;
  val[p] = ((unsigned long long)(unsigned)s << 32) | (unsigned)i;
}
__global__ void k_flagkey(int64_t n, const int32_t* __restrict__ idx, const int32_t* __restrict__ seg, int ssf, int64_t per_atom, int natoms,
                          const double* __restrict__ atoms, const double* __restrict__ rnn, double lim, const double* __restrict__ cx,
                          const double* __restrict__ cy, const double* __restrict__ cz, int32_t* __restrict__ key, int32_t* __restrict__ ntriv) {
  const int64_t p = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (p >= n) return;
  const int s = seg[p];
  const bool tr = ssf && trivial_point(idx[p], per_atom, natoms, atoms, rnn, lim, cx, cy, cz);
  key[p] = (s << 1) | (tr ? 0 : 1);
  if (tr) atomicAdd(ntriv + s, 1);
}
__global__ void k_gather(int64_t n, const int32_t* __restrict__ idx, int64_t per_atom, int n_ang, const double* __restrict__ rw,
                         const double* __restrict__ aw, const double* __restrict__ cx, const double* __restrict__ cy, const double* __restrict__ cz,
                         double* __restrict__ px, double* __restrict__ py, double* __restrict__ pz, double* __restrict__ wq,
                         int32_t* __restrict__ parent, long long* __restrict__ orig) {
  const int64_t k = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (k >= n) return;
  const int32_t i = idx[k];
  px[k] = cx[i]; py[k] = cy[i]; pz[k] = cz[i];
  const int64_t q = i % per_atom;
  wq[k] = __dmul_rn(rw[q / n_ang], aw[q % n_ang]);
  parent[k] = (int32_t)(i / per_atom);
  orig[k] = i;
}
double host_unkey(unsigned long long k) {
  const unsigned long long b = (k >> 63) ? (k & 0x7fffffffffffffffULL) : ~k;
  double v;
  memcpy(&v, &b, 8);
  return v;
}

}  // namespace

// The state of a plan being made on the GPU: the canonical points, the current order, the cuboids.
struct GpuPlanner {
  int device = 0, prev = -1;
  int64_t n = 0, per_atom = 0;
  int natoms = 0, n_ang = 0, nseg = 0;
  DevBuf<double> d_atoms, d_rr, d_au, d_cx, d_cy, d_cz;
  DevBuf<int32_t> d_idx, d_idx2, d_seg, d_seg2, d_newbase;
  DevBuf<unsigned long long> d_key, d_key2, d_val, d_val2, d_box;
  DevBuf<Seg> d_segs, d_segs2;
  DevBuf<int> d_nact;
  DevBuf<unsigned char> d_tmp;
  size_t tmp_bytes = 0;
  int64_t max_seg = 0;
  ~GpuPlanner() { if (prev >= 0) cudaSetDevice(prev); }

  cudaError_t begin(int dev, int natoms_, const double* atoms, int n_rad, int n_ang_, const double* rr, const double* au, int maxp,
                    std::vector<std::pair<int64_t, int64_t>>& leaves, std::vector<double>& boxes) {
    device = dev; natoms = natoms_; n_ang = n_ang_;
    cudaGetDevice(&prev);
    GP_CU(cudaSetDevice(device));
    per_atom = (int64_t)n_rad * n_ang; n = per_atom * natoms;
    const int TPB = 256;
    const unsigned nblk = (unsigned)((n + TPB - 1) / TPB);
    GP_CU(d_atoms.alloc(3 * (size_t)natoms)); GP_CU(d_rr.alloc(n_rad)); GP_CU(d_au.alloc(3 * (size_t)n_ang));
    GP_CU(d_cx.alloc(n)); GP_CU(d_cy.alloc(n)); GP_CU(d_cz.alloc(n));
    GP_CU(cudaMemcpy(d_atoms.p, atoms, 3 * (size_t)natoms * 8, cudaMemcpyHostToDevice));
    GP_CU(cudaMemcpy(d_rr.p, rr, (size_t)n_rad * 8, cudaMemcpyHostToDevice));
    GP_CU(cudaMemcpy(d_au.p, au, 3 * (size_t)n_ang * 8, cudaMemcpyHostToDevice));
    k_grid<<<nblk, TPB>>>(n, per_atom, n_ang, d_atoms.p, d_rr.p, d_au.p, d_cx.p, d_cy.p, d_cz.p);
    GP_CU(cudaGetLastError());
    // every part of a split holds at least min(64, max_batch_pts / 2) points: that bounds the number of cuboids
    max_seg = n / std::max(1, std::min(64, maxp / 2)) + 2;
    GP_CU(d_idx.alloc(n)); GP_CU(d_idx2.alloc(n)); GP_CU(d_seg.alloc(n)); GP_CU(d_seg2.alloc(n));
    GP_CU(d_key.alloc(n)); GP_CU(d_key2.alloc(n)); GP_CU(d_val.alloc(n)); GP_CU(d_val2.alloc(n));
    GP_CU(d_segs.alloc(max_seg)); GP_CU(d_segs2.alloc(max_seg)); GP_CU(d_newbase.alloc(max_seg + 1));
    GP_CU(d_box.alloc(6 * (size_t)max_seg)); GP_CU(d_nact.alloc(1));
    size_t t1 = 0, t2 = 0, t3 = 0;
    cub::DeviceRadixSort::SortPairs(nullptr, t1, d_idx.p, d_idx2.p, d_seg.p, d_seg2.p, (int)n, 0, 32);
    cub::DeviceRadixSort::SortPairs(nullptr, t2, d_key.p, d_key2.p, d_val.p, d_val2.p, (int)n, 0, 64);
    cub::DeviceRadixSort::SortPairs(nullptr, t3, d_seg.p, d_seg2.p, d_idx.p, d_idx2.p, (int)n, 0, 32);
    tmp_bytes = std::max(std::max(t1, t2), t3);
    GP_CU(d_tmp.alloc(tmp_bytes));
    k_iota<<<nblk, TPB>>>(n, d_idx.p);
    GP_CU(cudaMemset(d_seg.p, 0, (size_t)n * 4));
    Seg root{0, (int32_t)n, 0, 0};
    GP_CU(cudaMemcpy(d_segs.p, &root, sizeof(Seg), cudaMemcpyHostToDevice));
    nseg = 1;
    int idx_bits = 1;
    while (((int64_t)1 << idx_bits) < n) ++idx_bits;
    std::vector<Seg> hs;
    for (int level = 0; level < 64; ++level) {
      const unsigned sblk = (unsigned)((nseg + TPB - 1) / TPB);
      k_fill_box<<<(unsigned)((6 * (int64_t)nseg + TPB - 1) / TPB), TPB>>>(6 * (int64_t)nseg, d_box.p);
      GP_CU(cudaMemset(d_nact.p, 0, 4));
      k_bounds<<<nblk, TPB>>>(n, d_idx.p, d_seg.p, d_segs.p, d_cx.p, d_cy.p, d_cz.p, d_box.p, maxp);
      k_decide<<<sblk, TPB>>>(nseg, d_segs.p, d_box.p, maxp, d_nact.p);
      int nact = 0;
      GP_CU(cudaMemcpy(&nact, d_nact.p, 4, cudaMemcpyDeviceToHost));
      if (nact == 0) break;
      if (nseg + nact > max_seg) return cudaErrorMemoryAllocation;
      GP_CU(sort_segments(nblk, idx_bits, /*morton=*/false, nullptr));
      // first child of every segment (a split one has two): a short host pass over the level's segment records
      hs.resize(nseg);
      GP_CU(cudaMemcpy(hs.data(), d_segs.p, (size_t)nseg * sizeof(Seg), cudaMemcpyDeviceToHost));
      std::vector<int32_t> hb(nseg + 1);
      int32_t acc = 0;
      for (int s = 0; s < nseg; ++s) { hb[s] = acc; acc += hs[s].half > 0 ? 2 : 1; }
      hb[nseg] = acc;
      GP_CU(cudaMemcpy(d_newbase.p, hb.data(), (size_t)(nseg + 1) * 4, cudaMemcpyHostToDevice));
      k_reseg<<<nblk, TPB>>>(n, d_seg.p, d_segs.p, d_newbase.p);
      k_children<<<sblk, TPB>>>(nseg, d_segs.p, d_newbase.p, d_segs2.p);
      std::swap(d_segs.p, d_segs2.p);
      nseg = acc;
      GP_CU(cudaGetLastError());
    }
    // tight bounding boxes of the final cuboids (Alg. 1 screens against them; the Morton order is relative to them)
    k_fill_box<<<(unsigned)((6 * (int64_t)nseg + TPB - 1) / TPB), TPB>>>(6 * (int64_t)nseg, d_box.p);
    k_bounds<<<nblk, TPB>>>(n, d_idx.p, d_seg.p, d_segs.p, d_cx.p, d_cy.p, d_cz.p, d_box.p, 0);
    hs.resize(nseg);
    GP_CU(cudaMemcpy(hs.data(), d_segs.p, (size_t)nseg * sizeof(Seg), cudaMemcpyDeviceToHost));
    std::vector<unsigned long long> hbox(6 * (size_t)nseg);
    GP_CU(cudaMemcpy(hbox.data(), d_box.p, hbox.size() * 8, cudaMemcpyDeviceToHost));
    leaves.clear(); boxes.resize(hbox.size());
    for (const Seg& s : hs) leaves.push_back({s.begin, s.end});
    for (size_t k = 0; k < hbox.size(); ++k) boxes[k] = host_unkey(hbox[k]);
    return cudaSuccess;
  }

  // orders every segment by (sort key, canonical index): by index, by key, by segment (three stable radix sorts).
  // morton = false: key = coordinate along the segment's split axis; true: Morton key relative to the segment's box.
  cudaError_t sort_segments(unsigned nblk, int idx_bits, bool morton, const int32_t*) {
    const int TPB = 256;
    GP_CU(cub::DeviceRadixSort::SortPairs(d_tmp.p, tmp_bytes, d_idx.p, d_idx2.p, d_seg.p, d_seg2.p, (int)n, 0, idx_bits));
    if (morton) k_morton<<<nblk, TPB>>>(n, d_idx2.p, d_seg2.p, d_box.p, d_cx.p, d_cy.p, d_cz.p, d_key.p, d_val.p);
    else k_keys<<<nblk, TPB>>>(n, d_idx2.p, d_seg2.p, d_segs.p, d_cx.p, d_cy.p, d_cz.p, d_key.p, d_val.p);
    GP_CU(cub::DeviceRadixSort::SortPairs(d_tmp.p, tmp_bytes, d_key.p, d_key2.p, d_val.p, d_val2.p, (int)n, 0, 64));
    k_unpack<<<nblk, TPB>>>(n, d_val2.p, d_seg.p, d_idx.p);
    int seg_bits = 1;
    while ((1 << seg_bits) < nseg) ++seg_bits;
    GP_CU(cub::DeviceRadixSort::SortPairs(d_tmp.p, tmp_bytes, d_seg.p, d_seg2.p, d_idx.p, d_idx2.p, (int)n, 0, seg_bits));
    std::swap(d_seg.p, d_seg2.p); std::swap(d_idx.p, d_idx2.p);
    return cudaGetLastError();
  }

  // the host finishes the plan itself (a batch had to be split again): canonical points and the order so far
  cudaError_t download(std::vector<double>& cx, std::vector<double>& cy, std::vector<double>& cz, std::vector<int64_t>& idx) {
    cx.resize(n); cy.resize(n); cz.resize(n);
    GP_CU(cudaMemcpy(cx.data(), d_cx.p, (size_t)n * 8, cudaMemcpyDeviceToHost));
    GP_CU(cudaMemcpy(cy.data(), d_cy.p, (size_t)n * 8, cudaMemcpyDeviceToHost));
    GP_CU(cudaMemcpy(cz.data(), d_cz.p, (size_t)n * 8, cudaMemcpyDeviceToHost));
    std::vector<int32_t> h32(n);
    GP_CU(cudaMemcpy(h32.data(), d_idx.p, (size_t)n * 4, cudaMemcpyDeviceToHost));
    idx.resize(n);
    for (int64_t k = 0; k < n; ++k) idx[k] = h32[k];
    return cudaSuccess;
  }

  // Morton order inside every batch, SSF-trivial points first (stable); the permuted arrays stay on the device (the plan adopts
  // them: nothing per point crosses PCIe)
  cudaError_t order(bool ssf, const double* rnn, double lim, const double* rw, int n_rad, const double* aw, DevicePoints& out,
                    std::vector<int32_t>& ntriv) {
    const int TPB = 256;
    const unsigned nblk = (unsigned)((n + TPB - 1) / TPB);
    int idx_bits = 1;
    while (((int64_t)1 << idx_bits) < n) ++idx_bits;
    GP_CU(sort_segments(nblk, idx_bits, /*morton=*/true, nullptr));
    DevBuf<double> d_rnn, d_rw, d_aw;
    DevBuf<int32_t> d_ntriv;
    GP_CU(d_rnn.alloc(natoms)); GP_CU(d_rw.alloc(n_rad)); GP_CU(d_aw.alloc(n_ang)); GP_CU(d_ntriv.alloc(nseg));
    GP_CU(cudaMemcpy(d_rnn.p, rnn, (size_t)natoms * 8, cudaMemcpyHostToDevice));
    GP_CU(cudaMemcpy(d_rw.p, rw, (size_t)n_rad * 8, cudaMemcpyHostToDevice));
    GP_CU(cudaMemcpy(d_aw.p, aw, (size_t)n_ang * 8, cudaMemcpyHostToDevice));
    GP_CU(cudaMemset(d_ntriv.p, 0, (size_t)nseg * 4));
    // stable partition of every batch: key = (segment, non-trivial), values keep their Morton order
    k_flagkey<<<nblk, TPB>>>(n, d_idx.p, d_seg.p, ssf ? 1 : 0, per_atom, natoms, d_atoms.p, d_rnn.p, lim, d_cx.p, d_cy.p, d_cz.p, d_seg2.p, d_ntriv.p);
    int key_bits = 2;
    while ((1 << (key_bits - 1)) < nseg) ++key_bits;
    GP_CU(cub::DeviceRadixSort::SortPairs(d_tmp.p, tmp_bytes, d_seg2.p, d_seg.p, d_idx.p, d_idx2.p, (int)n, 0, key_bits));
    std::swap(d_idx.p, d_idx2.p);
    // the sort buffers are no longer needed: release them before the plan's arrays are allocated
    for (void** q : {(void**)&d_key.p, (void**)&d_key2.p, (void**)&d_val.p, (void**)&d_val2.p, (void**)&d_seg.p, (void**)&d_seg2.p,
                     (void**)&d_idx2.p, (void**)&d_tmp.p}) { cudaFree(*q); *q = nullptr; }
    const size_t m = std::max<size_t>((size_t)n, 1);
    GP_CU(cudaMalloc((void**)&out.px, m * 8)); GP_CU(cudaMalloc((void**)&out.py, m * 8)); GP_CU(cudaMalloc((void**)&out.pz, m * 8));
    GP_CU(cudaMalloc((void**)&out.wq, m * 8)); GP_CU(cudaMalloc((void**)&out.parent, m * 4)); GP_CU(cudaMalloc((void**)&out.orig, m * 8));
    k_gather<<<nblk, TPB>>>(n, d_idx.p, per_atom, n_ang, d_rw.p, d_aw.p, d_cx.p, d_cy.p, d_cz.p, out.px, out.py, out.pz, out.wq, out.parent,
                            (long long*)out.orig);
    GP_CU(cudaGetLastError());
    ntriv.resize(nseg);
    GP_CU(cudaMemcpy(ntriv.data(), d_ntriv.p, (size_t)nseg * 4, cudaMemcpyDeviceToHost));
    GP_CU(cudaDeviceSynchronize());
    return cudaSuccess;
  }
};

static int gp_fail(cudaError_t e, std::string& err) {
  cudaGetLastError();
  err = std::string("GPU planner: ") + cudaGetErrorString(e);
  return e == cudaErrorMemoryAllocation ? XC_ENOMEM : XC_ECUDA;
}
int gpu_planner_begin(int device, int natoms, const double* atoms, int n_rad, int n_ang, const double* rr, const double* au, int maxp,
                      GpuPlanner** out, std::vector<std::pair<int64_t, int64_t>>& leaves, std::vector<double>& boxes, std::string& err) {
  GpuPlanner* g = new GpuPlanner();
  const cudaError_t e = g->begin(device, natoms, atoms, n_rad, n_ang, rr, au, maxp, leaves, boxes);
  if (e != cudaSuccess) { delete g; *out = nullptr; return gp_fail(e, err); }
  *out = g;
  return XC_OK;
}
int gpu_planner_download(GpuPlanner* g, std::vector<double>& cx, std::vector<double>& cy, std::vector<double>& cz, std::vector<int64_t>& idx,
                         std::string& err) {
  const cudaError_t e = g->download(cx, cy, cz, idx);
  return e == cudaSuccess ? XC_OK : gp_fail(e, err);
}
int gpu_planner_order(GpuPlanner* g, bool ssf, const double* rnn, double lim, const double* rw, int n_rad, const double* aw,
                      DevicePoints& out, std::vector<int32_t>& ntriv, std::string& err) {
  const cudaError_t e = g->order(ssf, rnn, lim, rw, n_rad, aw, out, ntriv);
  return e == cudaSuccess ? XC_OK : gp_fail(e, err);
}
void gpu_planner_end(GpuPlanner* g) { delete g; }

}  // namespace xcb
