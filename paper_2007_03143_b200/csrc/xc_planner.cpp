// xc_planner.cpp -- host side of libxc_b200: atom-centred grid, spatial batching, shell screening,
// work lists (step (b) of the hot path; the analogue of Alg. 3 l.3.5-3.7, on one GPU).
//
// Batching (free by PAPER.md:L124 "the choice of batching scheme does not effect the methodological
// details"; reading A8): the WHOLE point cloud (all atoms pooled) is bisected recursively at the median
// of the longest bounding-box axis until a cuboid holds <= max_batch_pts points; split sizes are rounded
// to multiples of 64 so that almost every batch is a whole number of 64-point tiles.  Batches come out
// in depth-first order, i.e. spatially coherent.  Eq. (11) holds by construction.
// Screening: Alg. 1 (reading A7) on the tight bounding box of the batch's points with
// the cutoff radius of Eq. (10).
#include <algorithm>
#include <cmath>
#include <cstdlib>
#include <cstring>
#include <numeric>

#include "xc_internal.h"

namespace xcb {

namespace {

const double kPiH = 3.141592653589793238462643383279502884;

void radial_mura_knowles(int n, double alpha, std::vector<double>& r, std::vector<double>& w) {
  r.resize(n); w.resize(n);
  for (int i = 0; i < n; ++i) {
    double x = double(i + 1) / double(n + 1);
    double x3 = x * x * x;
    double om = 1.0 - x3;
    r[i] = -alpha * std::log(om);
    double drdx = 3.0 * alpha * x * x / om;
    w[i] = r[i] * r[i] * drdx / double(n + 1);
  }
}

bool angular_rule(int kind, int n, std::vector<double>& u, std::vector<double>& w) {
  u.resize(3 * (size_t)n); w.resize(n);
  if (kind == 0) {  // Fibonacci sphere
    const double ga = kPiH * (3.0 - std::sqrt(5.0));
    for (int k = 0; k < n; ++k) {
      double z = 1.0 - (2.0 * k + 1.0) / double(n);
      double s = std::sqrt(1.0 - z * z), ph = k * ga;
      u[3 * k] = s * std::cos(ph); u[3 * k + 1] = s * std::sin(ph); u[3 * k + 2] = z;
      w[k] = 4.0 * kPiH / double(n);
    }
    return true;
  }
  if (kind == 1) {  // Gauss-Legendre in cos(theta) x trapezoid in phi
    int nt = (int)std::lround(std::sqrt(n / 2.0));
    if (nt < 1 || 2 * nt * nt != n) return false;
    std::vector<double> xs(nt), ws(nt);
    for (int i = 0; i < nt; ++i) {
      double x = std::cos(kPiH * (i + 0.75) / (nt + 0.5)), dp = 1.0;
      for (int it = 0; it < 64; ++it) {
        double pm = 1.0, p = x;
        for (int k = 1; k < nt; ++k) { double pn = ((2 * k + 1) * x * p - k * pm) / (k + 1); pm = p; p = pn; }
        if (nt == 1) { pm = 1.0; p = x; }
        dp = nt * (pm - x * p) / (1.0 - x * x);
        double dx = p / dp;
        x -= dx;
        if (std::fabs(dx) < 1e-16) break;
      }
      double pm = 1.0, p = x;
      for (int k = 1; k < nt; ++k) { double pn = ((2 * k + 1) * x * p - k * pm) / (k + 1); pm = p; p = pn; }
      dp = nt * (pm - x * p) / (1.0 - x * x);
      xs[i] = x; ws[i] = 2.0 / ((1.0 - x * x) * dp * dp);
    }
    int k = 0;
    for (int i = 0; i < nt; ++i)
      for (int m = 0; m < 2 * nt; ++m, ++k) {
        double ph = (m + 0.5) * kPiH / nt, s = std::sqrt(1.0 - xs[i] * xs[i]);
        u[3 * k] = s * std::cos(ph); u[3 * k + 1] = s * std::sin(ph); u[3 * k + 2] = xs[i];
        w[k] = ws[i] * kPiH / nt;
      }
    return true;
  }
  return false;
}

struct Box { double lo[3], hi[3]; };

inline bool sphere_hits_box(const double* c, double r, const Box& b) {
  double d2 = 0.0;
  for (int p = 0; p < 3; ++p) {
    double t = c[p] < b.lo[p] ? b.lo[p] - c[p] : (c[p] > b.hi[p] ? c[p] - b.hi[p] : 0.0);
    d2 += t * t;
  }
  return d2 <= r * r;
}

struct Leaf { int64_t begin, end; };

}  // namespace

size_t batch_smem_bytes(int T, bool gga, int nb, int ns, int npr, int nthreads, int ring_g) {
  // must mirror the shared-memory carve of k_xc_batch (xc_kernels.cu)
  size_t nb16 = round_up(nb, 16);
  size_t b = 0;
  b += nb16 * (T + 4) * 8;                       // Phi tile
  if (gga) b += nb16 * (T + 4) * 8;              // Z tile
  if (gga) b += (size_t)ns * T * 2 * 8;          // R0/R1 panel
  b += (size_t)T * 8 * 16;                       // x,y,z,w of two tiles, scratch, a,g0,g1,g2
  b += (size_t)nthreads * 4 * 8;                 // cross-warp reduction buffer
  b += (size_t)kRingStages * ring_g * 256 * (round_up(nb, 8) / 8);   // P^j staging ring: kRingStages x ring_g k-steps x ntile fragments of 256 B
  b += 64 * 8;                                   // 2^(j/64) table of the collocation exp
  b += (size_t)npr * 16;                         // (exponent, coefficient) of the batch's primitives
  b += (size_t)ns * sizeof(ShellRec);            // shell records
  b += nb16 * 4;                                 // global function index
  b += (size_t)((ns + 3) & ~3) * 4;              // collocation order
  return b + 64;
}

// every batch CTA is launched with all of the SM's shared memory; what its tiles leave free goes to the ring
int batch_ring_g(size_t bytes_without_ring, int nb) {
  const size_t lim = kSmemLimit - kBatchStaticSmem;
  if (nb <= 0) return kRingGMax;
  if (bytes_without_ring >= lim) return 0;
  const size_t per_g = (size_t)kRingStages * 256 * (round_up(nb, 8) / 8);
  return (int)std::min<size_t>(kRingGMax, (lim - bytes_without_ring) / per_g);
}

size_t weights_smem_bytes(int nC, int warps) { return (size_t)nC * (24 + 4) + (size_t)warps * nC * 8 + 64; }

// Atom list of the weights kernels for a box of points (step (a)), exact SSF compact support, sorted by
// distance to the box.  U = min_C dmax(C, box) bounds r_min of every point of the box from above.  An atom B can own weight
// at some point only if r_B < kappa r_min <= kappa U, and a factor s(mu_BC) differs from 1 only if r_C < kappa r_B < kappa^2 U.
// With dmin(., box) <= r_. the lists {dmin < kappa U} (owners: the first nB) and {dmin < kappa^2 U} (partners: all) are
// supersets.  Becke-88 has no compact support: every atom is an owner and a partner; the order (nearest first) is what
// lets that kernel stop an owner's product once it is negligible.
void weight_atom_list(const double* atoms, int natoms, const double lo[3], const double hi[3], bool ssf, std::vector<int32_t>& out, int& nB) {
  const double a_ssf = 0.64, kappa = (1.0 + a_ssf) / (1.0 - a_ssf);
  double U = 1e300;
  for (int a = 0; a < natoms; ++a) {
    double d2 = 0.0;
    for (int p = 0; p < 3; ++p) { double t = std::max(std::fabs(atoms[3 * a + p] - lo[p]), std::fabs(atoms[3 * a + p] - hi[p])); d2 += t * t; }
    U = std::min(U, std::sqrt(d2));
  }
  const double rB = ssf ? kappa * U * (1.0 + 1e-12) + 1e-12 : 1e300, rC = ssf ? kappa * rB * (1.0 + 1e-12) + 1e-12 : 1e300;
  std::vector<std::pair<double, int32_t>> cand;
  for (int a = 0; a < natoms; ++a) {
    double d2 = 0.0;
    for (int p = 0; p < 3; ++p) {
      double c = atoms[3 * a + p];
      double t = c < lo[p] ? lo[p] - c : (c > hi[p] ? c - hi[p] : 0.0);
      d2 += t * t;
    }
    double d = std::sqrt(d2);
    if (d <= rC) cand.push_back({d, a});
  }
  std::sort(cand.begin(), cand.end());
  out.resize(cand.size());
  nB = 0;
  for (size_t k = 0; k < cand.size(); ++k) { out[k] = cand[k].second; if (cand[k].first <= rB) nB = (int)k + 1; }
}

int build_host_plan(const xc_atom* atoms, int natoms, const xc_shell* shells, int nshells, const double* exps,
                    const double* coefs, int nprim_total, const xc_grid_spec* spec, int device, HostPlan& hp, std::string& err) {
  if (!atoms || !shells || !exps || !coefs || !spec) { err = "null argument"; return XC_EINVAL; }
  if (natoms < 1 || nshells < 1 || nprim_total < 1) { err = "empty system"; return XC_EINVAL; }
  if (spec->n_rad < 1 || spec->n_ang < 1 || spec->max_batch_pts < 1 || spec->max_batch_pts > 512) {
    err = "bad grid_spec sizes (need n_rad,n_ang >= 1 and 1 <= max_batch_pts <= 512)"; return XC_EINVAL;
  }
  if (spec->radial != 0 || spec->angular < 0 || spec->angular > 1 || spec->partition < 0 || spec->partition > 1 ||
      spec->functional < 0 || spec->functional > 2) { err = "bad grid_spec enum"; return XC_EINVAL; }
  if (!(spec->eta > 0.0) || !(spec->mk_alpha > 0.0) || !(spec->rho_tol >= 0.0)) { err = "bad grid_spec reals"; return XC_EINVAL; }
  hp.natoms = natoms; hp.nshells = nshells; hp.nprim = nprim_total; hp.spec = *spec;
  hp.atoms.resize(3 * (size_t)natoms);
  for (int a = 0; a < natoms; ++a) { hp.atoms[3 * a] = atoms[a].x; hp.atoms[3 * a + 1] = atoms[a].y; hp.atoms[3 * a + 2] = atoms[a].z; }
  for (double v : hp.atoms)
    if (!std::isfinite(v)) { err = "non-finite atom coordinate"; return XC_EINVAL; }
  // nearest-neighbour distances (SSF "trivial point" rule); coincident centres make mu_BC undefined
  hp.rnn.assign(natoms, 1e300);
  {
    bool coincident = false;
#pragma omp parallel for schedule(static) reduction(|| : coincident)
    for (int a = 0; a < natoms; ++a) {
      double m = 1e300;
      for (int b = 0; b < natoms; ++b) {
        if (b == a) continue;
        const double dx = hp.atoms[3 * a] - hp.atoms[3 * b], dy = hp.atoms[3 * a + 1] - hp.atoms[3 * b + 1], dz = hp.atoms[3 * a + 2] - hp.atoms[3 * b + 2];
        m = std::min(m, std::sqrt(dx * dx + dy * dy + dz * dz));
      }
      hp.rnn[a] = m;
      if (!(m > 1e-8)) coincident = true;
    }
    if (coincident) { err = "two atoms coincide (R_AB < 1e-8 bohr)"; return XC_EINVAL; }
  }
  hp.exps.assign(exps, exps + nprim_total);
  hp.coefs.assign(coefs, coefs + nprim_total);
  for (int k = 0; k < nprim_total; ++k)
    if (!(exps[k] > 0.0) || !std::isfinite(exps[k]) || !std::isfinite(coefs[k])) { err = "non-positive or non-finite exponent/coefficient"; return XC_EINVAL; }
  hp.shells.resize(nshells); hp.rcut.resize(nshells);
  int foff = 0;
  for (int s = 0; s < nshells; ++s) {
    const xc_shell& sh = shells[s];
    if (sh.atom < 0 || sh.atom >= natoms || sh.nprim < 1 || sh.prim_off < 0 || sh.prim_off + sh.nprim > nprim_total || sh.L < 0) {
      err = "bad shell record"; return XC_EINVAL;
    }
    if ((sh.L & ~(0xff | XC_SHELL_PURE)) != 0) { err = "bad shell record (unknown bits in L)"; return XC_EINVAL; }
    const int Lq = sh.L & 0xff;
    if (Lq > kMaxL) { err = "angular momentum L > 2 is not supported"; return XC_EUNSUPPORTED; }
    const int type = ((sh.L & XC_SHELL_PURE) && Lq == 2) ? kPureD : Lq;   // a pure s or p shell is the Cartesian one
    if (sh.nprim > kMaxPrim) { err = "contraction depth > 16 is not supported"; return XC_EUNSUPPORTED; }
    ShellRec& r = hp.shells[s];
    r.x = atoms[sh.atom].x; r.y = atoms[sh.atom].y; r.z = atoms[sh.atom].z;
    r.L = type; r.nprim = sh.nprim; r.prim_off = sh.prim_off; r.func_off = foff; r.atom = sh.atom; r._pad = 0;
    foff += nfun(type);
    double m = 0.0;  // Eq. (10)
    for (int k = 0; k < sh.nprim; ++k) {
      double al = exps[sh.prim_off + k];
      double v = (0.5 * std::log(al) - std::log(spec->eta)) / al;
      if (v > 0.0) m = std::max(m, std::sqrt(v));
    }
    hp.rcut[s] = m;
  }
  hp.nbasis = foff;

  // ---- grid (canonical order: atom-major, radial, angular) ----
  std::vector<double> rr, rw, au, aw;
  radial_mura_knowles(spec->n_rad, spec->mk_alpha, rr, rw);
  if (!angular_rule(spec->angular, spec->n_ang, au, aw)) { err = "angular rule: n_ang must be 2*n_theta^2 for the product rule"; return XC_EINVAL; }
  const int64_t per_atom = (int64_t)spec->n_rad * spec->n_ang;
  const int64_t npts = per_atom * natoms;
  if (npts >= (int64_t)1 << 31) { err = "more than 2^31 grid points"; return XC_EUNSUPPORTED; }
  hp.npts = npts;
  std::vector<double> cx, cy, cz;
  std::vector<int64_t> idx;
  std::vector<Leaf> leaves;
  const int maxp = spec->max_batch_pts;
  GpuPlanner* gp = nullptr;                    // non-null while the plan is being made on the GPU
  struct GpGuard { GpuPlanner*& g; ~GpGuard() { if (g) gpu_planner_end(g); } } gp_guard{gp};
  std::vector<double> gboxes;                  // GPU path: tight bounding boxes of the cuboids
  if (device >= 0) {
    // grid and bisection on the GPU (xc_gpu_planner.cu): same points, same cuboids, same order
    std::vector<std::pair<int64_t, int64_t>> lv;
    const int rc = gpu_planner_begin(device, natoms, hp.atoms.data(), spec->n_rad, spec->n_ang, rr.data(), au.data(), maxp, &gp, lv, gboxes, err);
    if (rc != XC_OK) return rc;
    for (const auto& l : lv) leaves.push_back({l.first, l.second});
  } else {
  cx.resize(npts); cy.resize(npts); cz.resize(npts);
#pragma omp parallel for schedule(static)
  for (int64_t p = 0; p < npts; ++p) {
    int a = (int)(p / per_atom);
    int64_t q = p % per_atom;
    int i = (int)(q / spec->n_ang), k = (int)(q % spec->n_ang);
    cx[p] = hp.atoms[3 * a] + rr[i] * au[3 * k];
    cy[p] = hp.atoms[3 * a + 1] + rr[i] * au[3 * k + 1];
    cz[p] = hp.atoms[3 * a + 2] + rr[i] * au[3 * k + 2];
  }

  // ---- recursive median bisection ----
  idx.resize(npts);
  std::iota(idx.begin(), idx.end(), (int64_t)0);
  const double* coord[3] = {cx.data(), cy.data(), cz.data()};
  {
    // one bisection step: splits `cur` at the median of its longest axis (left part first => depth-first output order
    // is spatially coherent); returns false if the range is a leaf
    auto split = [&](const Leaf& cur, Leaf& left, Leaf& right) {
      int64_t n = cur.end - cur.begin;
      if (n <= maxp) return false;
      double lo[3] = {1e300, 1e300, 1e300}, hi[3] = {-1e300, -1e300, -1e300};
      for (int64_t k = cur.begin; k < cur.end; ++k)
        for (int p = 0; p < 3; ++p) { double v = coord[p][idx[k]]; lo[p] = std::min(lo[p], v); hi[p] = std::max(hi[p], v); }
      int ax = 0;
      for (int p = 1; p < 3; ++p) if (hi[p] - lo[p] > hi[ax] - lo[ax]) ax = p;
      int64_t half = n / 2;
      if (maxp >= 64 && n >= 128) half = std::max<int64_t>(64, half / 64 * 64);
      const double* c = coord[ax];
      std::nth_element(idx.begin() + cur.begin, idx.begin() + cur.begin + half, idx.begin() + cur.end,
                       [c](int64_t a, int64_t b) { return c[a] < c[b] || (c[a] == c[b] && a < b); });
      left = {cur.begin, cur.begin + half};
      right = {cur.begin + half, cur.end};
      return true;
    };
    auto subtree = [&](Leaf root, std::vector<Leaf>& out) {   // depth-first, left part first
      std::vector<Leaf> stack{root};
      while (!stack.empty()) {
        Leaf cur = stack.back(); stack.pop_back();
        Leaf l, r;
        if (!split(cur, l, r)) { out.push_back(cur); continue; }
        stack.push_back(r);
        stack.push_back(l);
      }
    };
    // the first levels breadth-first (kept in left-to-right order), then the subtrees in parallel; the ranges are
    // disjoint slices of idx, and the leaves are concatenated in subtree order: the plan does not depend on the
    // number of threads
    std::vector<Leaf> front{{0, npts}};
    for (int level = 0; level < 7; ++level) {
      std::vector<Leaf> next(2 * front.size());
      std::vector<char> isleaf(front.size(), 0);
#pragma omp parallel for schedule(dynamic, 1)
      for (int64_t k = 0; k < (int64_t)front.size(); ++k) {
        Leaf l, r;
        if (front[k].end - front[k].begin <= 16 * (int64_t)maxp || !split(front[k], l, r)) { isleaf[k] = 1; continue; }
        next[2 * k] = l; next[2 * k + 1] = r;
      }
      std::vector<Leaf> merged;
      bool any = false;
      for (size_t k = 0; k < front.size(); ++k) {
        if (isleaf[k]) merged.push_back(front[k]);
        else { merged.push_back(next[2 * k]); merged.push_back(next[2 * k + 1]); any = true; }
      }
      front.swap(merged);
      if (!any) break;
    }
    std::vector<std::vector<Leaf>> parts(front.size());
#pragma omp parallel for schedule(dynamic, 1)
    for (int64_t k = 0; k < (int64_t)front.size(); ++k) subtree(front[k], parts[k]);
    for (auto& v : parts) leaves.insert(leaves.end(), v.begin(), v.end());
  }
  }   // host grid + bisection
  const double* coord[3] = {cx.data(), cy.data(), cz.data()};   // (GPU path: null until a download)

  // ---- per-batch shell screening (Alg. 1 on the tight bounding box), with re-splitting of batches whose
  //      shell list exceeds the batch kernel's capacity (N_b^j <= kMaxNb, shared memory) ----
  std::vector<std::vector<int>> atom_shells(natoms);
  std::vector<double> atom_rmax(natoms, 0.0);
  for (int s = 0; s < nshells; ++s) {
    atom_shells[hp.shells[s].atom].push_back(s);
    atom_rmax[hp.shells[s].atom] = std::max(atom_rmax[hp.shells[s].atom], hp.rcut[s]);
  }
  const bool gga = spec->functional >= 1;       // 2 = meta-GGA (reading A23): the GGA footprint covers its passes
  auto screen = [&](const Leaf& lf, std::vector<int32_t>& out, int& nb, const double* known_box = nullptr) {
    Box b;
    if (known_box) {
      for (int p = 0; p < 3; ++p) { b.lo[p] = known_box[p]; b.hi[p] = known_box[3 + p]; }
    } else {
      for (int p = 0; p < 3; ++p) { b.lo[p] = 1e300; b.hi[p] = -1e300; }
      for (int64_t k = lf.begin; k < lf.end; ++k)
        for (int p = 0; p < 3; ++p) { double v = coord[p][idx[k]]; b.lo[p] = std::min(b.lo[p], v); b.hi[p] = std::max(b.hi[p], v); }
    }
    out.clear(); nb = 0;
    for (int a = 0; a < natoms; ++a) {
      if (!sphere_hits_box(&hp.atoms[3 * a], atom_rmax[a], b)) continue;
      for (int s : atom_shells[a])
        if (sphere_hits_box(&hp.atoms[3 * a], hp.rcut[s], b)) { out.push_back(s); nb += nfun(hp.shells[s].L); }
    }
    std::sort(out.begin(), out.end());
  };
  std::vector<std::vector<int32_t>> lists(leaves.size());
  std::vector<int> nbs(leaves.size());
#pragma omp parallel for schedule(dynamic, 64)
  for (int64_t j = 0; j < (int64_t)leaves.size(); ++j) screen(leaves[j], lists[j], nbs[j], gp ? &gboxes[6 * j] : nullptr);
  auto prim_sum = [&](const std::vector<int32_t>& sl) { int n = 0; for (int32_t sh : sl) n += hp.shells[sh].nprim; return n; };
  // re-split oversized batches (rare): sequential fix-up pass
  {
    std::vector<Leaf> L2; std::vector<std::vector<int32_t>> S2; std::vector<int> N2;
    bool any = false;
    for (size_t j = 0; j < leaves.size(); ++j)
      if (nbs[j] > kMaxNb || batch_ring_g(batch_smem_bytes(32, gga, nbs[j], (int)lists[j].size(), prim_sum(lists[j]), kBatchThreads, 0), nbs[j]) < 1) { any = true; break; }
    if (any) {
      if (gp) {   // the host finishes this plan: it needs the points and the order so far
        const int rc = gpu_planner_download(gp, cx, cy, cz, idx, err);
        gpu_planner_end(gp); gp = nullptr;
        if (rc != XC_OK) return rc;
        coord[0] = cx.data(); coord[1] = cy.data(); coord[2] = cz.data();
      }
      for (size_t j = 0; j < leaves.size(); ++j) {
        std::vector<Leaf> st{leaves[j]};
        bool first = true;
        while (!st.empty()) {
          Leaf cur = st.back(); st.pop_back();
          std::vector<int32_t> sl; int nb;
          if (first) { sl = lists[j]; nb = nbs[j]; first = false; } else screen(cur, sl, nb);
          int64_t n = cur.end - cur.begin;
          if (nb <= kMaxNb && batch_ring_g(batch_smem_bytes(32, gga, nb, (int)sl.size(), prim_sum(sl), kBatchThreads, 0), nb) >= 1) { L2.push_back(cur); S2.push_back(sl); N2.push_back(nb); continue; }
          if (n <= 1) { err = "a single grid point sees more basis functions than the batch kernel supports"; return XC_EUNSUPPORTED; }
          double lo[3] = {1e300, 1e300, 1e300}, hi[3] = {-1e300, -1e300, -1e300};
          for (int64_t k = cur.begin; k < cur.end; ++k)
            for (int p = 0; p < 3; ++p) { double v = coord[p][idx[k]]; lo[p] = std::min(lo[p], v); hi[p] = std::max(hi[p], v); }
          int ax = 0;
          for (int p = 1; p < 3; ++p) if (hi[p] - lo[p] > hi[ax] - lo[ax]) ax = p;
          int64_t half = n / 2;
          const double* c = coord[ax];
          std::nth_element(idx.begin() + cur.begin, idx.begin() + cur.begin + half, idx.begin() + cur.end,
                           [c](int64_t a, int64_t b) { return c[a] < c[b] || (c[a] == c[b] && a < b); });
          st.push_back({cur.begin + half, cur.end});
          st.push_back({cur.begin, cur.begin + half});
        }
      }
      leaves.swap(L2); lists.swap(S2); nbs.swap(N2);
    }
  }

  // ---- order the points inside each batch along a Morton curve: neighbouring threads of the weights kernel then
  //      see nearly the same atoms (warp-coherent loop bounds); the batch as a set is unchanged ----
  if (!gp) {
    auto spread = [](uint32_t v) { uint64_t x = v & 0x1fffff; x = (x | x << 32) & 0x1f00000000ffffULL; x = (x | x << 16) & 0x1f0000ff0000ffULL;
                                   x = (x | x << 8) & 0x100f00f00f00f00fULL; x = (x | x << 4) & 0x10c30c30c30c30c3ULL; x = (x | x << 2) & 0x1249249249249249ULL; return x; };
#pragma omp parallel
    {
      std::vector<std::pair<uint64_t, int64_t>> keyed;
#pragma omp for schedule(dynamic, 64)
      for (int64_t j = 0; j < (int64_t)leaves.size(); ++j) {
        double lo[3] = {1e300, 1e300, 1e300}, hi[3] = {-1e300, -1e300, -1e300};
        for (int64_t k = leaves[j].begin; k < leaves[j].end; ++k)
          for (int p = 0; p < 3; ++p) { double v = coord[p][idx[k]]; lo[p] = std::min(lo[p], v); hi[p] = std::max(hi[p], v); }
        double ext = std::max({hi[0] - lo[0], hi[1] - lo[1], hi[2] - lo[2], 1e-300});
        keyed.clear();
        for (int64_t k = leaves[j].begin; k < leaves[j].end; ++k) {
          uint64_t key = 0;
          for (int p = 0; p < 3; ++p) {
            uint32_t q = (uint32_t)std::min(1048575.0, std::floor((coord[p][idx[k]] - lo[p]) / ext * 1048576.0));
            key |= spread(q) << p;
          }
          keyed.push_back({key, idx[k]});
        }
        std::sort(keyed.begin(), keyed.end());
        for (size_t k = 0; k < keyed.size(); ++k) idx[leaves[j].begin + k] = keyed[k].second;
      }
    }
  }

  // ---- SSF: points with r_A < (1-a)/2 R_nn(A) have w = w^q exactly (every mu_AC <= -a).  They come first in their
  //      batch (each group keeps its Morton order); the weights kernel only visits the others ----
  std::vector<int32_t> ntriv(leaves.size(), 0);
  const double lim = 0.5 * (1.0 - 0.64);
  if (spec->partition == 0 && !gp) {
#pragma omp parallel for schedule(dynamic, 64)
    for (int64_t j = 0; j < (int64_t)leaves.size(); ++j) {
      auto trivial = [&](int64_t p) {
        if (natoms == 1) return true;
        const int a = (int)(p / per_atom);
        const double dx = cx[p] - hp.atoms[3 * a], dy = cy[p] - hp.atoms[3 * a + 1], dz = cz[p] - hp.atoms[3 * a + 2];
        return std::sqrt(dx * dx + dy * dy + dz * dz) < lim * hp.rnn[a];
      };
      auto mid = std::stable_partition(idx.begin() + leaves[j].begin, idx.begin() + leaves[j].end, trivial);
      ntriv[j] = (int32_t)(mid - (idx.begin() + leaves[j].begin));
    }
  }

  // ---- atom lists of the weights kernel (step (a)), exact SSF compact support ----
  // U = min_C dmax(C, box) bounds r_min of every point of the batch from above.  An atom B can own weight at some
  // point only if r_B < kappa r_min <= kappa U, and a factor s(mu_BC) differs from 1 only if r_C < kappa r_B < kappa^2 U.
  // With dmin(.,box) <= r_. the lists {dmin < kappa U} (owners) and {dmin < kappa^2 U} (partners) are supersets.
  hp.wbox.assign(6 * leaves.size(), 0.0);
  std::vector<std::vector<int32_t>> wlists(leaves.size());
  std::vector<int> wnB(leaves.size(), 0);
#pragma omp parallel for schedule(dynamic, 64)
  for (int64_t j = 0; j < (int64_t)leaves.size(); ++j) {
    double lo[3] = {1e300, 1e300, 1e300}, hi[3] = {-1e300, -1e300, -1e300};
    if (gp) {
      for (int p = 0; p < 3; ++p) { lo[p] = gboxes[6 * j + p]; hi[p] = gboxes[6 * j + 3 + p]; }
    } else {
      for (int64_t k = leaves[j].begin; k < leaves[j].end; ++k)
        for (int p = 0; p < 3; ++p) { double v = coord[p][idx[k]]; lo[p] = std::min(lo[p], v); hi[p] = std::max(hi[p], v); }
    }
    for (int p = 0; p < 3; ++p) { hp.wbox[6 * j + p] = lo[p]; hp.wbox[6 * j + 3 + p] = hi[p]; }
    weight_atom_list(hp.atoms.data(), natoms, lo, hi, spec->partition == 0, wlists[j], wnB[j]);
  }

  // ---- permuted point arrays ----
  if (gp) {
    // GPU path: Morton order, trivial points first and the permuted arrays in one go (identical to the host's stages above)
    const int rc = gpu_planner_order(gp, spec->partition == 0, hp.rnn.data(), lim, rw.data(), spec->n_rad, aw.data(), hp.dev, ntriv, err);
    gpu_planner_end(gp); gp = nullptr;
    if (rc != XC_OK) return rc;
  } else {
  hp.px.resize(npts); hp.py.resize(npts); hp.pz.resize(npts); hp.wq.resize(npts); hp.parent.resize(npts); hp.orig.resize(npts);
#pragma omp parallel for schedule(static)
  for (int64_t k = 0; k < npts; ++k) {
    int64_t p = idx[k];
    hp.px[k] = cx[p]; hp.py[k] = cy[p]; hp.pz[k] = cz[p];
    int a = (int)(p / per_atom);
    int64_t q = p % per_atom;
    hp.wq[k] = rw[q / spec->n_ang] * aw[q % spec->n_ang];
    hp.parent[k] = a; hp.orig[k] = p;
  }
  }

  // ---- batch records, function lists, work items ----
  const int64_t nbatch = (int64_t)leaves.size();
  hp.batches.resize(nbatch);
  int64_t sh_off = 0, f_off = 0, ppk = 0, wa_total = 0;
  hp.watoms.clear(); hp.wbatch_small.clear(); hp.wbatch_large.clear(); hp.w_max_small = hp.w_max_large = hp.w_max_list = 0;
  for (int64_t j = 0; j < nbatch; ++j) {
    BatchRec& b = hp.batches[j];
    b.pt_off = (int32_t)leaves[j].begin; b.nq = (int32_t)(leaves[j].end - leaves[j].begin);
    b.sh_off = (int32_t)sh_off; b.ns = (int32_t)lists[j].size();
    b.f_off = (int32_t)f_off; b.nb = nbs[j];
    b.ppk_off = ppk;
    ppk += round_up(b.nb, 4) * round_up(b.nb, 8);
    b.wa_off = wa_total; b.wa_nB = wnB[j]; b.wa_nC = (int32_t)wlists[j].size();
    wa_total += b.wa_nC;                                  // the lists themselves are copied in parallel below
    hp.w_max_list = std::max(hp.w_max_list, (int)b.wa_nC);
    b.ntriv = ntriv[j]; b.ring_g = 0;
    if (spec->partition == 0 && b.ntriv < b.nq) {          // SSF: batches whose points are all trivial need no kernel
      const int len = b.wa_nC;
      if (len <= kWeightSmallList) { hp.wbatch_small.push_back((int32_t)j); hp.w_max_small = std::max(hp.w_max_small, len); }
      else { hp.wbatch_large.push_back((int32_t)j); hp.w_max_large = std::max(hp.w_max_large, len); }
    }
    sh_off += b.ns; f_off += b.nb;
    if (sh_off >= ((int64_t)1 << 31) || f_off >= ((int64_t)1 << 31)) { err = "batch lists exceed 2^31 entries"; return XC_EUNSUPPORTED; }
  }
  hp.ppk_doubles = ppk;
  hp.watoms.resize(wa_total);
#pragma omp parallel for schedule(dynamic, 256)
  for (int64_t j = 0; j < nbatch; ++j) std::copy(wlists[j].begin(), wlists[j].end(), hp.watoms.begin() + hp.batches[j].wa_off);
  hp.bshells.resize(sh_off); hp.bsfoff.resize(sh_off); hp.bfidx.resize(f_off);
#pragma omp parallel for schedule(dynamic, 64)
  for (int64_t j = 0; j < nbatch; ++j) {
    const BatchRec& b = hp.batches[j];
    int f = b.f_off;
    for (int k = 0; k < b.ns; ++k) {
      int s = lists[j][k];
      hp.bshells[b.sh_off + k] = s;
      hp.bsfoff[b.sh_off + k] = f - b.f_off;
      for (int c = 0; c < nfun(hp.shells[s].L); ++c, ++f) hp.bfidx[f] = hp.shells[s].func_off + c;
    }
  }
  hp.sum_nbnq = hp.sum_nb2 = hp.flops = 0; hp.max_nb = hp.max_ns = 0; hp.smem_small = hp.smem_large = 0;
  hp.ids_small.clear(); hp.ids_large.clear();
  for (int64_t j = 0; j < nbatch; ++j) {
    const BatchRec& b = hp.batches[j];
    hp.sum_nbnq += (double)b.nb * b.nq; hp.sum_nb2 += (double)b.nb * b.nb; hp.flops += 4.0 * b.nb * (double)b.nb * b.nq;
    hp.max_nb = std::max(hp.max_nb, b.nb); hp.max_ns = std::max(hp.max_ns, b.ns);
    if (b.nb == 0) continue;  // nothing to integrate: rho = 0 on every point
    int npr = 0;
    for (int k = 0; k < b.ns; ++k) npr += hp.shells[hp.bshells[b.sh_off + k]].nprim;
    // class 0: 64-point tiles, 16 warps, one CTA per SM; class 1 (N_b^j > kSmallNb or a 64-point tile does not fit): 32-point tiles
    // the ring serves the GGA X GEMM only (LDA reads its lower-triangle fragments through L1, which needs the shared
    // memory it does not use)
    const size_t f64 = batch_smem_bytes(64, gga, b.nb, b.ns, npr, kBatchThreads, 0);
    const int g64 = batch_ring_g(f64, b.nb);
    BatchRec& bw = hp.batches[j];
    if (b.nb <= kSmallNb && g64 >= 2) {
      bw.ring_g = gga ? g64 : 0;
      hp.smem_small = std::max(hp.smem_small, batch_smem_bytes(64, gga, b.nb, b.ns, npr, kBatchThreads, bw.ring_g));
      hp.ids_small.push_back((int32_t)j);
    } else {
      const size_t f32 = batch_smem_bytes(32, gga, b.nb, b.ns, npr, kBatchThreads, 0);
      bw.ring_g = gga ? batch_ring_g(f32, b.nb) : 0;
      hp.smem_large = std::max(hp.smem_large, batch_smem_bytes(32, gga, b.nb, b.ns, npr, kBatchThreads, bw.ring_g));
      hp.ids_large.push_back((int32_t)j);
    }
  }
  // heaviest batches first: the tail of each launch is made of cheap CTAs
  auto cost = [&](int32_t j) { const BatchRec& b = hp.batches[j]; return (double)b.nb * b.nb * b.nq + 200.0 * b.ns * b.nq; };
  std::stable_sort(hp.ids_small.begin(), hp.ids_small.end(), [&](int32_t x, int32_t y) { return cost(x) > cost(y); });
  // (class 1: the batches with N_b^j > kMidNb first: they run as a launch of their own)
  std::stable_sort(hp.ids_large.begin(), hp.ids_large.end(), [&](int32_t x, int32_t y) {
    const bool hx = hp.batches[x].nb > kMidNb, hy = hp.batches[y].nb > kMidNb;
    return hx != hy ? hx : cost(x) > cost(y);
  });
  hp.n_heavy = 0;
  for (int32_t j : hp.ids_large) hp.n_heavy += hp.batches[j].nb > kMidNb ? 1 : 0;
  // a launch of its own costs the tail of one more kernel (about one CTA's time), the three-round kernel gains ~4 % on its
  // batches: with fewer than 4096 of them (28 waves) the whole class runs the five-round kernel, as one launch
  // (no batch beyond kMidNb at all: the whole class runs the three-round kernel, still as one launch)
  if (hp.n_heavy > 0 && (int)hp.ids_large.size() - hp.n_heavy < 4096 && !(spec->flags & XC_SPEC_SPLIT_CLASS1)) hp.n_heavy = (int)hp.ids_large.size();
  // Becke-88 weights launch: warps per CTA such that the per-warp distance rows fit in shared memory
  // (the SSF kernel has a fixed footprint and reads list entries beyond its cache from global memory)
  hp.w_warps = 8;
  while (spec->partition != 0 && hp.w_warps > 1 && weights_smem_bytes(hp.w_max_list, hp.w_warps) > kSmemLimit) hp.w_warps >>= 1;
  if (spec->partition != 0 && weights_smem_bytes(hp.w_max_list, hp.w_warps) > kSmemLimit) {
    err = "too many atoms for the Becke-88 weights kernel"; return XC_EUNSUPPORTED;
  }
  return XC_OK;
}

}  // namespace xcb
