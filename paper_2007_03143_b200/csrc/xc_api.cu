// xc_api.cu -- the C ABI of libxc_b200 (include/xc_b200.h): plan lifetime, uploads, the stream-ordered
// launch sequence of one E_xc / V_xc / N_el build (Alg. 2 l.2.2-2.9 on one GPU), diagnostics.
#include <cuda_runtime.h>

#include <algorithm>
#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <new>
#include <string>
#include <vector>

#include "xc_internal.h"
#include "xc_kernels.h"

using namespace xcb;

namespace {
thread_local std::string g_err;
int fail(int code, const std::string& msg) { g_err = msg; return code; }
int cuda_fail(cudaError_t e, const char* what) {
  g_err = std::string(what) + ": " + cudaGetErrorString(e);
  return e == cudaErrorMemoryAllocation ? XC_ENOMEM : XC_ECUDA;
}
#define CU(call)                                         \
  do {                                                   \
    cudaError_t _e = (call);                             \
    if (_e != cudaSuccess) return cuda_fail(_e, #call);  \
  } while (0)

// XC_DEBUG_SYNC=1 in the environment: synchronise after every kernel of xc_eval and name the one that failed
bool debug_sync() { static const bool on = std::getenv("XC_DEBUG_SYNC") != nullptr; return on; }
#define CUK(call, st)                                                  \
  do {                                                                 \
    cudaError_t _e = (call);                                           \
    if (_e == cudaSuccess && debug_sync()) _e = cudaStreamSynchronize(st); \
    if (_e != cudaSuccess) return cuda_fail(_e, #call);                \
  } while (0)

template <class T>
int upload(T** dptr, const std::vector<T>& h) {
  *dptr = nullptr;
  size_t bytes = std::max<size_t>(h.size(), 1) * sizeof(T);
  CU(cudaMalloc((void**)dptr, bytes));
  if (!h.empty()) CU(cudaMemcpy(*dptr, h.data(), h.size() * sizeof(T), cudaMemcpyHostToDevice));
  return XC_OK;
}
}  // namespace

struct xc_plan {
  int device = 0;
  HostPlan hp;
  // device copies
  double *d_px = nullptr, *d_py = nullptr, *d_pz = nullptr, *d_wq = nullptr, *d_w = nullptr;
  int32_t* d_parent = nullptr;
  int64_t* d_orig = nullptr;            // GPU-made plans only (xc_plan_export reads it back)
  double *d_atoms = nullptr, *d_invR = nullptr, *d_rnn = nullptr;
  ShellRec* d_shells = nullptr;
  double *d_exps = nullptr, *d_coefs = nullptr;
  BatchRec* d_batches = nullptr;
  int32_t *d_bshells = nullptr, *d_bsfoff = nullptr, *d_bfidx = nullptr;
  double* d_wbox = nullptr;
  int32_t *d_watoms = nullptr, *d_wsmall = nullptr, *d_wlarge = nullptr;
  int32_t *d_ids_small = nullptr, *d_ids_large = nullptr;
  double* d_ppk = nullptr;
  unsigned long long *d_vhi = nullptr, *d_vlo = nullptr;
  double *d_Epart = nullptr, *d_Npart = nullptr, *d_result = nullptr;   // d_result: E, N_el, then the two flag words of the accumulator
  double *d_rho = nullptr, *d_grho = nullptr;   // diagnostics, allocated on first use (XC_EVAL_DIAG)
  bool diag_valid = false;
  double* h_result = nullptr;  // pinned, 4 doubles
  unsigned long long* d_paircnt = nullptr;   // XC_EVAL_COUNT_PAIRS
  long long ssf_pairs = -1;    // pair factors evaluated by the last counted build (-1: none)
  int vexp = 0;                // exponent of the fixed-point V accumulator: resolution 2^(vexp - 64), range 2^(vexp + 31)
  double *d_Ptmp = nullptr, *d_Vtmp = nullptr;  // for xc_eval_host
  cudaStream_t copy_stream = nullptr;           // xc_eval_host: P crosses PCIe while step (a), which does not read P, runs
  cudaEvent_t ev_P = nullptr;                   // ... recorded behind that copy
  bool wait_P = false;                          // the next xc_eval waits for ev_P before its first read of P
  // spin-unrestricted build (xc_eval_uks), allocated on first use: rho_s [2][npts], grad rho_s [2][npts][3], the
  // coefficients of Z^s a_s [2][npts], g_s [2][npts][3], block partials of the functional kernel, (E, N_a, N_b)
  double *d_urho = nullptr, *d_ugrho = nullptr, *d_ucA = nullptr, *d_ucG = nullptr, *d_upart = nullptr, *d_ures = nullptr;
  bool weights_valid = false;
  std::vector<cudaEvent_t> ev;
  float ms[5] = {0, 0, 0, 0, 0};
  int launches = 0;
};

struct DeviceGuard {   // the entry points leave the caller's current device as they found it
  int prev = -1;
  explicit DeviceGuard(int dev) { if (cudaGetDevice(&prev) != cudaSuccess) prev = -1; if (prev != dev) cudaSetDevice(dev); else prev = -1; }
  ~DeviceGuard() { if (prev >= 0) cudaSetDevice(prev); }
};

static void free_plan(xc_plan* p) {
  if (!p) return;
  if (p->device < 0) { delete p; return; }
  DeviceGuard guard(p->device);
  void* ptrs[] = {p->d_px, p->d_py, p->d_pz, p->d_wq, p->d_w, p->d_parent, p->d_atoms, p->d_invR, p->d_rnn, p->d_shells,
                  p->d_exps, p->d_coefs, p->d_batches, p->d_bshells, p->d_bsfoff, p->d_bfidx, p->d_ids_small,
                  p->d_ids_large, p->d_ppk, p->d_vhi, p->d_vlo, p->d_Epart, p->d_Npart, p->d_result,
                  p->d_rho, p->d_grho, p->d_Ptmp, p->d_Vtmp, p->d_watoms, p->d_wsmall, p->d_wlarge, p->d_wbox, p->d_paircnt,
                  p->d_urho, p->d_ugrho, p->d_ucA, p->d_ucG, p->d_upart, p->d_ures, p->d_orig};
  for (void* q : ptrs) if (q) cudaFree(q);
  if (p->h_result) cudaFreeHost(p->h_result);
  for (cudaEvent_t e : p->ev) cudaEventDestroy(e);
  if (p->ev_P) cudaEventDestroy(p->ev_P);
  if (p->copy_stream) cudaStreamDestroy(p->copy_stream);
  delete p;
}

// [natoms][natoms] table 1 / R_BC, 0 on the diagonal (Becke-88 kernel)
static void pair_table(const std::vector<double>& atoms, int natoms, std::vector<double>& inv) {
  inv.assign((size_t)natoms * natoms, 0.0);
#pragma omp parallel for schedule(static)
  for (int a = 0; a < natoms; ++a)
    for (int b = 0; b < natoms; ++b) {
      if (a == b) continue;
      double dx = atoms[3 * a] - atoms[3 * b], dy = atoms[3 * a + 1] - atoms[3 * b + 1], dz = atoms[3 * a + 2] - atoms[3 * b + 2];
      inv[(size_t)a * natoms + b] = 1.0 / std::sqrt(dx * dx + dy * dy + dz * dz);
    }
}


// step (a) of a build (Alg. 4 l.4.1): the partition weights, unless the caller reuses those of the last build
static int run_weights(xc_plan* p, int32_t flags, cudaStream_t st, int& launches) {
  HostPlan& hp = p->hp;
  if (!(flags & XC_EVAL_REUSE_WEIGHTS) || !p->weights_valid) {
    WeightArgs wa;
    wa.batches = p->d_batches; wa.watoms = p->d_watoms; wa.atoms = p->d_atoms; wa.invR = p->d_invR;
    wa.paircnt = nullptr;
    if ((flags & XC_EVAL_COUNT_PAIRS) && hp.spec.partition == 0) {
      if (!p->d_paircnt) CU(cudaMalloc((void**)&p->d_paircnt, 8));
      CU(cudaMemsetAsync(p->d_paircnt, 0, 8, st));
      wa.paircnt = p->d_paircnt;
    }
    wa.wbox = p->d_wbox; wa.natoms = hp.natoms; wa.px = p->d_px; wa.py = p->d_py; wa.pz = p->d_pz; wa.wq = p->d_wq; wa.parent = p->d_parent; wa.w = p->d_w;
    if (hp.spec.partition == 0) {                          // long lists first: they are the long pole
      if (!hp.wbatch_large.empty()) { CUK(launch_weights_ssf(wa, p->d_wlarge, (int)hp.wbatch_large.size(), hp.w_max_large, st), st); ++launches; }
      if (!hp.wbatch_small.empty()) { CUK(launch_weights_ssf(wa, p->d_wsmall, (int)hp.wbatch_small.size(), hp.w_max_small, st), st); ++launches; }
    } else if (!hp.batches.empty()) {
      CUK(launch_weights_becke(wa, nullptr, (int)hp.batches.size(), hp.w_warps, hp.w_max_list, st), st);
      ++launches;
    }
    p->weights_valid = true;
    p->ssf_pairs = -1;
    if (wa.paircnt) {
      unsigned long long v = 0;
      CU(cudaMemcpyAsync(&v, p->d_paircnt, 8, cudaMemcpyDeviceToHost, st));
      CU(cudaStreamSynchronize(st));
      p->ssf_pairs = (long long)v;
    }
  }
  return XC_OK;
}

// Restricted meta-GGA build (grid_spec.functional = 2, reading A23): the stages of Alg. 4 as passes of the same
// kernels -- densities (MODE 1, full P^j), tau (MODE 3, lower triangle of P^j), the functional over the grid
// (k_functional_mgga) with the per-batch E / N sums, then the potential: Z Phi^T + Phi Z^T (MODE 2) and the tau term (MODE 4)
// into one fixed-point accumulator.
static int eval_mgga(xc_plan* p, const double* dP, int64_t ldp, double* dV, int64_t ldv, double* E_xc, double* N_el, int32_t flags,
                     cudaStream_t st) {
  HostPlan& hp = p->hp;
  const int64_t npts = hp.npts;
  const bool diag = (flags & XC_EVAL_DIAG) != 0;
  int launches = 0, nk = 0;
  if (!p->d_urho) {
    const size_t n = std::max<size_t>((size_t)npts, 1);
    CU(cudaMalloc((void**)&p->d_urho, 2 * n * 8));   // rho | tau
    CU(cudaMalloc((void**)&p->d_ugrho, 6 * n * 8));  // grad rho | w f, w rho (per point)
    CU(cudaMalloc((void**)&p->d_ucA, 2 * n * 8));    // a | t
    CU(cudaMalloc((void**)&p->d_ucG, 6 * n * 8));    // g
    CU(cudaMalloc((void**)&p->d_upart, std::max<size_t>((size_t)uks_functional_blocks(npts), 1) * 3 * 8));
    CU(cudaMalloc((void**)&p->d_ures, 4 * 8));
  }
  if (diag && !p->d_rho) {
    CU(cudaMalloc((void**)&p->d_rho, std::max<size_t>(npts * 8, 8)));
    CU(cudaMalloc((void**)&p->d_grho, std::max<size_t>(npts * 24, 8)));
  }
  CU(cudaEventRecord(p->ev[0], st));
  { const int rc = run_weights(p, flags, st, launches); if (rc != XC_OK) return rc; }
  CU(cudaEventRecord(p->ev[1], st));
  const size_t nb2 = (size_t)hp.nbasis * hp.nbasis;
  BatchArgs ba;
  ba.batches = p->d_batches; ba.bshells = p->d_bshells; ba.bsfoff = p->d_bsfoff; ba.bfidx = p->d_bfidx;
  ba.shells = p->d_shells; ba.exps = p->d_exps; ba.coefs = p->d_coefs;
  ba.px = p->d_px; ba.py = p->d_py; ba.pz = p->d_pz; ba.w = p->d_w;
  ba.P = dP; ba.ldp = ldp; ba.ppk = p->d_ppk;
  ba.Epart = p->d_Epart; ba.Npart = p->d_Npart; ba.vhi = p->d_vhi; ba.vlo = p->d_vlo; ba.nbasis = hp.nbasis;
  ba.rho_tol = hp.spec.rho_tol; ba.vexp = p->vexp;
  ba.vflags = (unsigned*)(p->d_result + 2);
  ba.cA = nullptr; ba.cG = nullptr;
  double* d_rho = p->d_urho; double* d_tau = p->d_urho + npts;
  double* d_gr = p->d_ugrho; double* d_ef = p->d_ugrho + 3 * npts; double* d_en = d_ef + npts;
  double* d_a = p->d_ucA; double* d_t = p->d_ucA + npts;
  const int nl = (int)hp.ids_large.size(), nsm = (int)hp.ids_small.size();
  // densities: full P^j
  ba.rho_out = d_rho; ba.grho_out = d_gr;
  if (nl) { CUK(launch_pack(ba, p->d_ids_large, nl, false, st), st); ++launches; }
  if (nsm) { CUK(launch_pack(ba, p->d_ids_small, nsm, false, st), st); ++launches; }
  if (nl) { CUK(launch_batch(1, true, 1, ba, p->d_ids_large, nl, hp.smem_large, st, hp.n_heavy, &nk), st); launches += nk; }
  if (nsm) { CUK(launch_batch(0, true, 1, ba, p->d_ids_small, nsm, hp.smem_small, st), st); ++launches; }
  // tau: lower triangle of P^j
  ba.rho_out = d_tau; ba.grho_out = nullptr;
  if (nl) { CUK(launch_pack(ba, p->d_ids_large, nl, true, st), st); ++launches; }
  if (nsm) { CUK(launch_pack(ba, p->d_ids_small, nsm, true, st), st); ++launches; }
  if (nl) { CUK(launch_batch(1, false, 3, ba, p->d_ids_large, nl, hp.smem_large, st, hp.n_heavy, &nk), st); launches += nk; }
  if (nsm) { CUK(launch_batch(0, false, 3, ba, p->d_ids_small, nsm, hp.smem_small, st), st); ++launches; }
  CU(cudaEventRecord(p->ev[2], st));
  // functional, per-batch partial sums
  CUK(launch_functional_mgga(npts, (int)hp.batches.size(), p->d_batches, p->d_w, d_rho, d_gr, d_tau, hp.spec.rho_tol, d_a, p->d_ucG, d_t, d_ef,
                             d_en, p->d_Epart, p->d_Npart, st), st);
  launches += 2;
  if (diag) {
    CU(cudaMemcpyAsync(p->d_rho, d_rho, (size_t)npts * 8, cudaMemcpyDeviceToDevice, st));
    CU(cudaMemcpyAsync(p->d_grho, d_gr, (size_t)npts * 24, cudaMemcpyDeviceToDevice, st));
  }
  p->diag_valid = diag;
  ba.rho_out = nullptr; ba.grho_out = nullptr;
  for (int attempt = 0;; ++attempt) {
    ba.vexp = p->vexp;
    CU(cudaMemsetAsync(p->d_vhi, 0, nb2 * 8, st));
    CU(cudaMemsetAsync(p->d_vlo, 0, nb2 * 8, st));
    CU(cudaMemsetAsync(p->d_result + 2, 0, 16, st));
    ba.cA = d_a; ba.cG = p->d_ucG;
    if (nl) { CUK(launch_batch(1, true, 2, ba, p->d_ids_large, nl, hp.smem_large, st, hp.n_heavy, &nk), st); launches += nk; }
    if (nsm) { CUK(launch_batch(0, true, 2, ba, p->d_ids_small, nsm, hp.smem_small, st), st); ++launches; }
    ba.cA = d_t; ba.cG = nullptr;
    if (nl) { CUK(launch_batch(1, false, 4, ba, p->d_ids_large, nl, hp.smem_large, st, hp.n_heavy, &nk), st); launches += nk; }
    if (nsm) { CUK(launch_batch(0, false, 4, ba, p->d_ids_small, nsm, hp.smem_small, st), st); ++launches; }
    CUK(launch_reduce((int64_t)hp.batches.size(), p->d_Epart, p->d_Npart, p->d_result, st), st);
    CUK(launch_finalize(hp.nbasis, p->d_vhi, p->d_vlo, dV, ldv, p->vexp, false, st), st);
    launches += 2;
    CU(cudaMemcpyAsync(p->h_result, p->d_result, 32, cudaMemcpyDeviceToHost, st));
    CU(cudaStreamSynchronize(st));
    unsigned vf[4];
    std::memcpy(vf, p->h_result + 2, 16);
    if (vf[1] != 0) {
      CUK(launch_finalize(hp.nbasis, p->d_vhi, p->d_vlo, dV, ldv, p->vexp, true, st), st);
      CU(cudaStreamSynchronize(st));
      *E_xc = *N_el = std::nan("");
      return fail(XC_EINVAL, "non-finite value met while accumulating V (NaN or Inf in P, or overflow); V is filled with NaN");
    }
    const int e = vf[0] ? (int)(vf[0] >> 20) - 1023 : p->vexp;
    const bool fits = p->vexp >= e - 10 && p->vexp <= e + 14;
    if (fits || attempt == 1) {
      if (!fits) return fail(XC_EUNSUPPORTED, "V increments span more than the fixed-point accumulator covers");
      break;
    }
    p->vexp = e - 8;
  }
  CU(cudaEventRecord(p->ev[3], st));
  CU(cudaEventRecord(p->ev[4], st));
  CU(cudaStreamSynchronize(st));
  *E_xc = p->h_result[0];
  *N_el = p->h_result[1];
  float t;
  CU(cudaEventElapsedTime(&t, p->ev[0], p->ev[1])); p->ms[0] = t;   // weights
  CU(cudaEventElapsedTime(&t, p->ev[1], p->ev[2])); p->ms[1] = t;   // packs, densities, tau
  CU(cudaEventElapsedTime(&t, p->ev[2], p->ev[3])); p->ms[2] = t;   // functional and potential passes
  p->ms[3] = 0.f;
  CU(cudaEventElapsedTime(&t, p->ev[0], p->ev[4])); p->ms[4] = t;
  p->launches = launches;
  return XC_OK;
}

extern "C" {

const char* xc_strerror(int code) {
  switch (code) {
    case XC_OK: return "ok";
    case XC_EINVAL: return "invalid argument";
    case XC_EUNSUPPORTED: return "unsupported input";
    case XC_ENOMEM: return "out of memory";
    case XC_ECUDA: return "CUDA error";
    default: return "unknown error";
  }
}
const char* xc_last_error(void) { return g_err.c_str(); }

int xc_plan_create(const xc_atom* atoms, int32_t natoms, const xc_shell* shells, int32_t nshells, const double* exps,
                   const double* coefs, int32_t nprim_total, const xc_grid_spec* spec, int32_t device, xc_plan** out) {
  if (!out) return fail(XC_EINVAL, "out is null");
  *out = nullptr;
  if (device != -1) {
    int ndev = 0;
    cudaError_t ce = cudaGetDeviceCount(&ndev);
    if (ce != cudaSuccess || ndev == 0) return fail(XC_ECUDA, std::string("no CUDA device: ") + cudaGetErrorString(ce));
    if (device < 0 || device >= ndev) return fail(XC_EINVAL, "bad device index");
  }
  xc_plan* p = new (std::nothrow) xc_plan();
  if (!p) return fail(XC_ENOMEM, "host allocation failed");
  p->device = device;
  std::string err;
  int rc;
  std::vector<double> ptab;   // 1 / R_BC (Becke-88 only: the SSF kernel forms its pair terms per tile)
  try {
    rc = build_host_plan(atoms, natoms, shells, nshells, exps, coefs, nprim_total, spec, device, p->hp, err);
    if (rc == XC_OK && device != -1 && p->hp.spec.partition == 1) pair_table(p->hp.atoms, p->hp.natoms, ptab);
  } catch (const std::bad_alloc&) {
    rc = XC_ENOMEM; err = "host allocation failed in planner";
  }
  // a GPU-made plan hands over its point arrays (adopted even on failure, so that free_plan releases them)
  p->d_px = p->hp.dev.px; p->d_py = p->hp.dev.py; p->d_pz = p->hp.dev.pz; p->d_wq = p->hp.dev.wq;
  p->d_parent = p->hp.dev.parent; p->d_orig = p->hp.dev.orig;
  const bool dev_points = p->hp.dev.px != nullptr;
  p->hp.dev = DevicePoints();
  if (rc != XC_OK) { free_plan(p); return fail(rc, err); }
  HostPlan& hp = p->hp;
  if (device == -1) { *out = p; return XC_OK; }   // host-only plan: info / stats / export only
  auto bail = [&](int code) { free_plan(p); return code; };
  DeviceGuard guard(device);
#define UP(d, h) do { int _r = upload(&p->d, h); if (_r != XC_OK) return bail(_r); } while (0)
  if (!dev_points) { UP(d_px, hp.px); UP(d_py, hp.py); UP(d_pz, hp.pz); UP(d_wq, hp.wq); UP(d_parent, hp.parent); }
  UP(d_atoms, hp.atoms);
  UP(d_invR, ptab);
  UP(d_shells, hp.shells); UP(d_exps, hp.exps); UP(d_coefs, hp.coefs);
  UP(d_batches, hp.batches); UP(d_bshells, hp.bshells); UP(d_bsfoff, hp.bsfoff); UP(d_bfidx, hp.bfidx);
  UP(d_wbox, hp.wbox);
  UP(d_watoms, hp.watoms); UP(d_wsmall, hp.wbatch_small); UP(d_wlarge, hp.wbatch_large);
  UP(d_ids_small, hp.ids_small); UP(d_ids_large, hp.ids_large);
#undef UP
  size_t nitems = hp.batches.size();
  size_t nb2 = (size_t)hp.nbasis * hp.nbasis;
#define AL(d, bytes) do { cudaError_t _e = cudaMalloc((void**)&p->d, std::max<size_t>((bytes), 8)); if (_e != cudaSuccess) return bail(cuda_fail(_e, "cudaMalloc " #d)); } while (0)
  AL(d_w, hp.npts * 8); AL(d_ppk, (size_t)hp.ppk_doubles * 8);
  AL(d_vhi, nb2 * 8); AL(d_vlo, nb2 * 8); AL(d_Epart, nitems * 8); AL(d_Npart, nitems * 8); AL(d_result, 32);
#undef AL
  // SSF: the points the weights kernel never visits (w = w^q exactly) get their weight once, here
  if (cudaMemcpy(p->d_w, p->d_wq, std::max<size_t>(hp.npts * 8, 8), cudaMemcpyDeviceToDevice) != cudaSuccess)
    return bail(fail(XC_ECUDA, "cudaMemcpy failed"));
  if (cudaMemset(p->d_Epart, 0, std::max<size_t>(nitems * 8, 8)) != cudaSuccess || cudaMemset(p->d_Npart, 0, std::max<size_t>(nitems * 8, 8)) != cudaSuccess)
    return bail(fail(XC_ECUDA, "cudaMemset failed"));   // batches without functions never write their partials
  if (cudaMallocHost((void**)&p->h_result, 32) != cudaSuccess) return bail(fail(XC_ENOMEM, "cudaMallocHost failed"));
  p->ev.resize(5);
  for (auto& e : p->ev)
    if (cudaEventCreate(&e) != cudaSuccess) return bail(fail(XC_ECUDA, "cudaEventCreate failed"));
  *out = p;
  return XC_OK;
}

int xc_plan_info(const xc_plan* p, int64_t* n_points, int64_t* n_batches, int32_t* n_basis, int64_t* n_shell_entries,
                 double* algorithmic_flops) {
  if (!p) return fail(XC_EINVAL, "plan is null");
  if (n_points) *n_points = p->hp.npts;
  if (n_batches) *n_batches = (int64_t)p->hp.batches.size();
  if (n_basis) *n_basis = p->hp.nbasis;
  if (n_shell_entries) *n_shell_entries = (int64_t)p->hp.bshells.size();
  if (algorithmic_flops) *algorithmic_flops = p->hp.flops;
  return XC_OK;
}

int xc_plan_stats(const xc_plan* p, double stats[12]) {
  if (!p || !stats) return fail(XC_EINVAL, "null argument");
  stats[0] = p->hp.sum_nbnq; stats[1] = p->hp.sum_nb2; stats[2] = p->hp.flops; stats[3] = p->hp.max_nb;
  stats[4] = p->hp.batches.empty() ? 0.0 : (double)p->hp.npts / (double)p->hp.batches.size();
  stats[5] = 8.0 * (double)p->hp.ppk_doubles;
  double snC = 0, snB = 0, mnC = 0, mnB = 0;
  for (const BatchRec& b : p->hp.batches) { snC += b.wa_nC; snB += b.wa_nB; mnC = std::max(mnC, (double)b.wa_nC); mnB = std::max(mnB, (double)b.wa_nB); }
  const double nbt = std::max<double>(1.0, (double)p->hp.batches.size());
  stats[6] = snC / nbt; stats[7] = mnC; stats[8] = snB / nbt; stats[9] = mnB; stats[10] = p->hp.max_ns; stats[11] = 0.0;
  return XC_OK;
}

int xc_plan_export(const xc_plan* p, double* pts, double* wq, int32_t* parent, int64_t* orig, int64_t* batch_off,
                   int64_t* shell_off, int32_t* shells) {
  if (!p) return fail(XC_EINVAL, "plan is null");
  const HostPlan& hp = p->hp;
  if (hp.px.empty() && hp.npts > 0) {
    // GPU-made plan: the point arrays live on the device
    if (p->device < 0 || !p->d_px) return fail(XC_EINVAL, "plan holds no point arrays");
    DeviceGuard guard(p->device);
    const size_t n = (size_t)hp.npts;
    if (pts) {
      std::vector<double> t(n);
      const double* src[3] = {p->d_px, p->d_py, p->d_pz};
      for (int c = 0; c < 3; ++c) {
        CU(cudaMemcpy(t.data(), src[c], n * 8, cudaMemcpyDeviceToHost));
        for (size_t i = 0; i < n; ++i) pts[3 * i + c] = t[i];
      }
    }
    if (wq) CU(cudaMemcpy(wq, p->d_wq, n * 8, cudaMemcpyDeviceToHost));
    if (parent) CU(cudaMemcpy(parent, p->d_parent, n * 4, cudaMemcpyDeviceToHost));
    if (orig) CU(cudaMemcpy(orig, p->d_orig, n * 8, cudaMemcpyDeviceToHost));
  } else {
    if (pts) for (int64_t i = 0; i < hp.npts; ++i) { pts[3 * i] = hp.px[i]; pts[3 * i + 1] = hp.py[i]; pts[3 * i + 2] = hp.pz[i]; }
    if (wq) std::copy(hp.wq.begin(), hp.wq.end(), wq);
    if (parent) std::copy(hp.parent.begin(), hp.parent.end(), parent);
    if (orig) std::copy(hp.orig.begin(), hp.orig.end(), orig);
  }
  size_t nb = hp.batches.size();
  if (batch_off) { for (size_t j = 0; j < nb; ++j) batch_off[j] = hp.batches[j].pt_off; batch_off[nb] = hp.npts; }
  if (shell_off) { for (size_t j = 0; j < nb; ++j) shell_off[j] = hp.batches[j].sh_off; shell_off[nb] = (int64_t)hp.bshells.size(); }
  if (shells) std::copy(hp.bshells.begin(), hp.bshells.end(), shells);
  return XC_OK;
}

int xc_eval(xc_plan* p, const double* dP, int64_t ldp, double* dV, int64_t ldv, double* E_xc, double* N_el,
            int32_t flags, void* cuda_stream) {
  if (!p || !dP || !dV || !E_xc || !N_el) return fail(XC_EINVAL, "null argument");
  if (p->device < 0) return fail(XC_ECUDA, "host-only plan (device = -1): no CUDA device bound, and there is no CPU fallback");
  HostPlan& hp = p->hp;
  if (ldp < hp.nbasis || ldv < hp.nbasis) return fail(XC_EINVAL, "leading dimension smaller than n_basis");
  cudaStream_t st = (cudaStream_t)cuda_stream;
  DeviceGuard guard(p->device);
  if (hp.spec.functional == 2) {
    if (p->wait_P) { p->wait_P = false; CU(cudaStreamWaitEvent(st, p->ev_P, 0)); }
    return eval_mgga(p, dP, ldp, dV, ldv, E_xc, N_el, flags, st);
  }
  const bool gga = hp.spec.functional == 1;
  const bool diag = (flags & XC_EVAL_DIAG) != 0;
  int launches = 0, nk = 0;
  size_t ie = 0;
  if (diag && !p->d_rho) {
    CU(cudaMalloc((void**)&p->d_rho, std::max<size_t>(hp.npts * 8, 8)));
    CU(cudaMalloc((void**)&p->d_grho, std::max<size_t>(hp.npts * 24, 8)));
  }
  CU(cudaEventRecord(p->ev[ie++], st));
  { const int rc = run_weights(p, flags, st, launches); if (rc != XC_OK) return rc; }
  if (p->wait_P) { p->wait_P = false; CU(cudaStreamWaitEvent(st, p->ev_P, 0)); }   // xc_eval_host: P is on its way on the copy stream
  CU(cudaEventRecord(p->ev[ie++], st));
  size_t nb2 = (size_t)hp.nbasis * hp.nbasis;
  BatchArgs ba;
  ba.batches = p->d_batches; ba.bshells = p->d_bshells; ba.bsfoff = p->d_bsfoff; ba.bfidx = p->d_bfidx;
  ba.shells = p->d_shells; ba.exps = p->d_exps; ba.coefs = p->d_coefs;
  ba.px = p->d_px; ba.py = p->d_py; ba.pz = p->d_pz; ba.w = p->d_w;
  ba.P = dP; ba.ldp = ldp; ba.ppk = p->d_ppk;
  ba.rho_out = diag ? p->d_rho : nullptr; ba.grho_out = (diag && gga) ? p->d_grho : nullptr;
  ba.Epart = p->d_Epart; ba.Npart = p->d_Npart; ba.vhi = p->d_vhi; ba.vlo = p->d_vlo; ba.nbasis = hp.nbasis;
  ba.rho_tol = hp.spec.rho_tol; ba.cA = nullptr; ba.cG = nullptr;
  ba.vflags = (unsigned*)(p->d_result + 2);
  if (diag) {
    CU(cudaMemsetAsync(p->d_rho, 0, hp.npts * 8, st));
    CU(cudaMemsetAsync(p->d_grho, 0, hp.npts * 24, st));
  }
  p->diag_valid = diag;
  // P^j pack (Alg. 4 l.4.2), then the fused batch kernel (l.4.3-4.10); large N_b^j first
  if (!hp.ids_large.empty()) { CUK(launch_pack(ba, p->d_ids_large, (int)hp.ids_large.size(), !gga, st), st); ++launches; }
  if (!hp.ids_small.empty()) { CUK(launch_pack(ba, p->d_ids_small, (int)hp.ids_small.size(), !gga, st), st); ++launches; }
  // The increments of V go to a fixed-point accumulator with resolution 2^(vexp - 64) and range 2^(vexp + 31).  The batch
  // kernel reports the largest |increment| and whether one was not finite; if the exponent the plan remembers from its last
  // build does not suit this P (first build with unusually scaled inputs), steps (c)-(g) are repeated once with the right one.
  for (int attempt = 0;; ++attempt) {
    ba.vexp = p->vexp;
    CU(cudaMemsetAsync(p->d_vhi, 0, nb2 * 8, st));
    CU(cudaMemsetAsync(p->d_vlo, 0, nb2 * 8, st));
    CU(cudaMemsetAsync(p->d_result + 2, 0, 16, st));
    if (attempt == 0) CU(cudaEventRecord(p->ev[ie++], st));
    if (!hp.ids_large.empty()) { CUK(launch_batch(1, gga, 0, ba, p->d_ids_large, (int)hp.ids_large.size(), hp.smem_large, st, hp.n_heavy, &nk), st); launches += nk; }
    if (!hp.ids_small.empty()) { CUK(launch_batch(0, gga, 0, ba, p->d_ids_small, (int)hp.ids_small.size(), hp.smem_small, st), st); ++launches; }
    if (attempt == 0) CU(cudaEventRecord(p->ev[ie++], st));
    CUK(launch_reduce((int64_t)hp.batches.size(), p->d_Epart, p->d_Npart, p->d_result, st), st);
    CUK(launch_finalize(hp.nbasis, p->d_vhi, p->d_vlo, dV, ldv, p->vexp, false, st), st);   // speculative: almost always the last word
    launches += 2;
    CU(cudaMemcpyAsync(p->h_result, p->d_result, 32, cudaMemcpyDeviceToHost, st));
    if (attempt == 0) CU(cudaEventRecord(p->ev[ie++], st));
    CU(cudaStreamSynchronize(st));
    unsigned vf[4];
    std::memcpy(vf, p->h_result + 2, 16);
    const bool poison = vf[1] != 0;
    if (poison) {
      CUK(launch_finalize(hp.nbasis, p->d_vhi, p->d_vlo, dV, ldv, p->vexp, true, st), st);
      CU(cudaStreamSynchronize(st));
      *E_xc = *N_el = std::nan("");
      return fail(XC_EINVAL, "non-finite value met while accumulating V (NaN or Inf in P, or overflow); V is filled with NaN");
    }
    // vf[0] = high word of the largest |increment| (0: every increment was 0); e = its binary exponent
    const int e = vf[0] ? (int)(vf[0] >> 20) - 1023 : p->vexp;
    const bool fits = p->vexp >= e - 10 && p->vexp <= e + 14;
    if (fits || attempt == 1) {
      if (!fits) return fail(XC_EUNSUPPORTED, "V increments span more than the fixed-point accumulator covers");
      break;
    }
    p->vexp = e - 8;
  }
  *E_xc = p->h_result[0];
  *N_el = p->h_result[1];
  // stage timings
  float t;
  p->ms[0] = p->ms[1] = p->ms[2] = p->ms[3] = p->ms[4] = 0.f;
  CU(cudaEventElapsedTime(&t, p->ev[0], p->ev[1])); p->ms[0] = t;
  CU(cudaEventElapsedTime(&t, p->ev[1], p->ev[2])); p->ms[1] = t;   // includes zeroing the accumulators
  CU(cudaEventElapsedTime(&t, p->ev[2], p->ev[3])); p->ms[2] = t;
  CU(cudaEventElapsedTime(&t, p->ev[3], p->ev[4])); p->ms[3] = t;
  CU(cudaEventElapsedTime(&t, p->ev[0], p->ev[4])); p->ms[4] = t;
  p->launches = launches;
  return XC_OK;
}

// Spin-unrestricted build (readings A20-A22): rho_s = sum P^s phi phi for s = a, b, the spin-polarised
// functional couples them, V^a and V^b come out.  Same plan, same kernels, run as passes: per spin {pack P^s, densities},
// the functional over the grid, per spin {Z^s, V^s,j, increment, finalise}.
int xc_eval_uks(xc_plan* p, const double* dPa, const double* dPb, int64_t ldp, double* dVa, double* dVb, int64_t ldv,
                double* E_xc, double* N_ab, int32_t flags, void* cuda_stream) {
  if (!p || !dPa || !dPb || !dVa || !dVb || !E_xc || !N_ab) return fail(XC_EINVAL, "null argument");
  if (p->device < 0) return fail(XC_ECUDA, "host-only plan (device = -1): no CUDA device bound, and there is no CPU fallback");
  HostPlan& hp = p->hp;
  if (ldp < hp.nbasis || ldv < hp.nbasis) return fail(XC_EINVAL, "leading dimension smaller than n_basis");
  if (!(hp.spec.rho_tol > 0.0)) return fail(XC_EINVAL, "the spin-unrestricted build needs rho_tol > 0 (reading A20)");
  if (hp.spec.functional > 1) return fail(XC_EUNSUPPORTED, "the spin-unrestricted build knows Slater+VWN5 and PBE only");
  cudaStream_t st = (cudaStream_t)cuda_stream;
  DeviceGuard guard(p->device);
  const bool gga = hp.spec.functional == 1;
  const int64_t npts = hp.npts;
  int launches = 0, nk = 0;
  if (!p->d_urho) {
    const size_t n = std::max<size_t>((size_t)npts, 1);
    CU(cudaMalloc((void**)&p->d_urho, 2 * n * 8));
    CU(cudaMalloc((void**)&p->d_ugrho, 6 * n * 8));
    CU(cudaMalloc((void**)&p->d_ucA, 2 * n * 8));
    CU(cudaMalloc((void**)&p->d_ucG, 6 * n * 8));
    CU(cudaMalloc((void**)&p->d_upart, std::max<size_t>((size_t)uks_functional_blocks(npts), 1) * 3 * 8));
    CU(cudaMalloc((void**)&p->d_ures, 4 * 8));
  }
  CU(cudaEventRecord(p->ev[0], st));
  { const int rc = run_weights(p, flags, st, launches); if (rc != XC_OK) return rc; }
  CU(cudaEventRecord(p->ev[1], st));
  const size_t nb2 = (size_t)hp.nbasis * hp.nbasis;
  BatchArgs ba;
  ba.batches = p->d_batches; ba.bshells = p->d_bshells; ba.bsfoff = p->d_bsfoff; ba.bfidx = p->d_bfidx;
  ba.shells = p->d_shells; ba.exps = p->d_exps; ba.coefs = p->d_coefs;
  ba.px = p->d_px; ba.py = p->d_py; ba.pz = p->d_pz; ba.w = p->d_w;
  ba.ldp = ldp; ba.ppk = p->d_ppk;
  ba.Epart = p->d_Epart; ba.Npart = p->d_Npart; ba.vhi = p->d_vhi; ba.vlo = p->d_vlo; ba.nbasis = hp.nbasis;
  ba.rho_tol = hp.spec.rho_tol; ba.vexp = p->vexp;
  ba.vflags = (unsigned*)(p->d_result + 2);
  ba.cA = nullptr; ba.cG = nullptr;
  // ---- densities of both spins (Alg. 4 l.4.2-4.5 per spin) ----
  for (int s = 0; s < 2; ++s) {
    ba.P = s == 0 ? dPa : dPb;
    ba.rho_out = p->d_urho + (size_t)s * npts; ba.grho_out = p->d_ugrho + (size_t)s * npts * 3;
    if (!hp.ids_large.empty()) { CUK(launch_pack(ba, p->d_ids_large, (int)hp.ids_large.size(), !gga, st), st); ++launches; }
    if (!hp.ids_small.empty()) { CUK(launch_pack(ba, p->d_ids_small, (int)hp.ids_small.size(), !gga, st), st); ++launches; }
    if (!hp.ids_large.empty()) { CUK(launch_batch(1, gga, 1, ba, p->d_ids_large, (int)hp.ids_large.size(), hp.smem_large, st, hp.n_heavy, &nk), st); launches += nk; }
    if (!hp.ids_small.empty()) { CUK(launch_batch(0, gga, 1, ba, p->d_ids_small, (int)hp.ids_small.size(), hp.smem_small, st), st); ++launches; }
  }
  CU(cudaEventRecord(p->ev[2], st));
  // ---- functional, E_xc, N_a, N_b (l.4.6-4.7) ----
  CUK(launch_functional_uks(gga, npts, p->d_w, p->d_urho, p->d_ugrho, hp.spec.rho_tol, p->d_ucA, p->d_ucG, p->d_upart, p->d_ures, st), st);
  launches += 2;
  // ---- Z^s, V^s,j, increment (l.4.8-4.10) per spin; the accumulator's exponent adapts as in xc_eval ----
  ba.rho_out = nullptr; ba.grho_out = nullptr; ba.P = nullptr;
  for (int s = 0; s < 2; ++s) {
    double* dV = s == 0 ? dVa : dVb;
    ba.cA = p->d_ucA + (size_t)s * npts; ba.cG = p->d_ucG + (size_t)s * npts * 3;
    for (int attempt = 0;; ++attempt) {
      ba.vexp = p->vexp;
      CU(cudaMemsetAsync(p->d_vhi, 0, nb2 * 8, st));
      CU(cudaMemsetAsync(p->d_vlo, 0, nb2 * 8, st));
      CU(cudaMemsetAsync(p->d_result + 2, 0, 16, st));
      if (!hp.ids_large.empty()) { CUK(launch_batch(1, gga, 2, ba, p->d_ids_large, (int)hp.ids_large.size(), hp.smem_large, st, hp.n_heavy, &nk), st); launches += nk; }
      if (!hp.ids_small.empty()) { CUK(launch_batch(0, gga, 2, ba, p->d_ids_small, (int)hp.ids_small.size(), hp.smem_small, st), st); ++launches; }
      CUK(launch_finalize(hp.nbasis, p->d_vhi, p->d_vlo, dV, ldv, p->vexp, false, st), st);
      ++launches;
      CU(cudaMemcpyAsync(p->h_result, p->d_result, 32, cudaMemcpyDeviceToHost, st));
      CU(cudaStreamSynchronize(st));
      unsigned vf[4];
      std::memcpy(vf, p->h_result + 2, 16);
      if (vf[1] != 0) {
        CUK(launch_finalize(hp.nbasis, p->d_vhi, p->d_vlo, dVa, ldv, p->vexp, true, st), st);
        CUK(launch_finalize(hp.nbasis, p->d_vhi, p->d_vlo, dVb, ldv, p->vexp, true, st), st);
        CU(cudaStreamSynchronize(st));
        *E_xc = N_ab[0] = N_ab[1] = std::nan("");
        return fail(XC_EINVAL, "non-finite value met while accumulating V (NaN or Inf in P, or overflow); V is filled with NaN");
      }
      const int e = vf[0] ? (int)(vf[0] >> 20) - 1023 : p->vexp;
      const bool fits = p->vexp >= e - 10 && p->vexp <= e + 14;
      if (fits || attempt == 1) {
        if (!fits) return fail(XC_EUNSUPPORTED, "V increments span more than the fixed-point accumulator covers");
        break;
      }
      p->vexp = e - 8;
    }
  }
  CU(cudaEventRecord(p->ev[3], st));
  double res[4];
  CU(cudaMemcpyAsync(res, p->d_ures, 24, cudaMemcpyDeviceToHost, st));
  CU(cudaEventRecord(p->ev[4], st));
  CU(cudaStreamSynchronize(st));
  *E_xc = res[0]; N_ab[0] = res[1]; N_ab[1] = res[2];
  float t;
  CU(cudaEventElapsedTime(&t, p->ev[0], p->ev[1])); p->ms[0] = t;   // weights
  CU(cudaEventElapsedTime(&t, p->ev[1], p->ev[2])); p->ms[1] = t;   // pack + densities of both spins
  CU(cudaEventElapsedTime(&t, p->ev[2], p->ev[3])); p->ms[2] = t;   // functional + potentials of both spins
  p->ms[3] = 0.f;
  CU(cudaEventElapsedTime(&t, p->ev[0], p->ev[4])); p->ms[4] = t;
  p->launches = launches;
  p->diag_valid = false;
  return XC_OK;
}

// rho_s [2][npts] and grad rho_s [2][npts][3] of the last xc_eval_uks, plan order (grad only for GGA plans); entries of
// points with w = 0 are not defined (they are never evaluated)
int xc_eval_uks_densities(const xc_plan* p, double* rho, double* grho) {
  if (!p) return fail(XC_EINVAL, "plan is null");
  if (p->device < 0 || !p->d_urho) return fail(XC_EINVAL, "no spin-unrestricted build has run on this plan");
  DeviceGuard guard(p->device);
  if (rho) CU(cudaMemcpy(rho, p->d_urho, (size_t)p->hp.npts * 16, cudaMemcpyDeviceToHost));
  if (grho) CU(cudaMemcpy(grho, p->d_ugrho, (size_t)p->hp.npts * 48, cudaMemcpyDeviceToHost));
  return XC_OK;
}

// The meta-GGA intermediate (reading A22): tau_i = 1/2 sum_mu grad Phi_mu,i . grad X_mu,i with
// X = P^j Phi^j, for the density matrix dP (one spin, or the total one), at every point with w != 0.
int xc_eval_tau(xc_plan* p, const double* dP, int64_t ldp, double* d_tau, int32_t flags, void* cuda_stream) {
  if (!p || !dP || !d_tau) return fail(XC_EINVAL, "null argument");
  if (p->device < 0) return fail(XC_ECUDA, "host-only plan (device = -1): no CUDA device bound, and there is no CPU fallback");
  HostPlan& hp = p->hp;
  if (ldp < hp.nbasis) return fail(XC_EINVAL, "leading dimension smaller than n_basis");
  cudaStream_t st = (cudaStream_t)cuda_stream;
  DeviceGuard guard(p->device);
  int launches = 0, nk = 0;
  { const int rc = run_weights(p, flags, st, launches); if (rc != XC_OK) return rc; }
  BatchArgs ba;
  ba.batches = p->d_batches; ba.bshells = p->d_bshells; ba.bsfoff = p->d_bsfoff; ba.bfidx = p->d_bfidx;
  ba.shells = p->d_shells; ba.exps = p->d_exps; ba.coefs = p->d_coefs;
  ba.px = p->d_px; ba.py = p->d_py; ba.pz = p->d_pz; ba.w = p->d_w;
  ba.P = dP; ba.ldp = ldp; ba.ppk = p->d_ppk;
  ba.rho_out = d_tau; ba.grho_out = nullptr; ba.cA = nullptr; ba.cG = nullptr;
  ba.Epart = p->d_Epart; ba.Npart = p->d_Npart; ba.vhi = p->d_vhi; ba.vlo = p->d_vlo; ba.nbasis = hp.nbasis;
  ba.rho_tol = hp.spec.rho_tol; ba.vexp = p->vexp; ba.vflags = (unsigned*)(p->d_result + 2);
  CU(cudaMemsetAsync(d_tau, 0, (size_t)hp.npts * 8, st));
  if (!hp.ids_large.empty()) { CUK(launch_pack(ba, p->d_ids_large, (int)hp.ids_large.size(), true, st), st); ++launches; }
  if (!hp.ids_small.empty()) { CUK(launch_pack(ba, p->d_ids_small, (int)hp.ids_small.size(), true, st), st); ++launches; }
  if (!hp.ids_large.empty()) { CUK(launch_batch(1, false, 3, ba, p->d_ids_large, (int)hp.ids_large.size(), hp.smem_large, st, hp.n_heavy, &nk), st); launches += nk; }
  if (!hp.ids_small.empty()) { CUK(launch_batch(0, false, 3, ba, p->d_ids_small, (int)hp.ids_small.size(), hp.smem_small, st), st); ++launches; }
  CU(cudaStreamSynchronize(st));
  p->launches = launches;
  p->diag_valid = false;
  return XC_OK;
}

int xc_eval_host(xc_plan* p, const double* hP, int64_t ldp, double* hV, int64_t ldv, double* E_xc, double* N_el, int32_t flags) {
  if (!p || !hP || !hV) return fail(XC_EINVAL, "null argument");
  if (p->device < 0) return fail(XC_ECUDA, "host-only plan (device = -1): no CUDA device bound, and there is no CPU fallback");
  const int n = p->hp.nbasis;
  if (ldp < n || ldv < n) return fail(XC_EINVAL, "leading dimension smaller than n_basis");
  DeviceGuard guard(p->device);
  size_t bytes = (size_t)n * n * 8;
  if (!p->d_Ptmp) CU(cudaMalloc((void**)&p->d_Ptmp, bytes));
  if (!p->d_Vtmp) CU(cudaMalloc((void**)&p->d_Vtmp, bytes));
  if (!p->copy_stream) {
    CU(cudaStreamCreateWithFlags(&p->copy_stream, cudaStreamNonBlocking));
    CU(cudaEventCreateWithFlags(&p->ev_P, cudaEventDisableTiming));
  }
  // the upload of P overlaps step (a) (Alg. 4 l.4.1 reads no P): xc_eval waits for it right before the P^j pack
  CU(cudaMemcpy2DAsync(p->d_Ptmp, (size_t)n * 8, hP, (size_t)ldp * 8, (size_t)n * 8, n, cudaMemcpyHostToDevice, p->copy_stream));
  CU(cudaEventRecord(p->ev_P, p->copy_stream));
  p->wait_P = true;
  int rc = xc_eval(p, p->d_Ptmp, n, p->d_Vtmp, n, E_xc, N_el, flags, nullptr);
  p->wait_P = false;
  if (rc != XC_OK) CU(cudaStreamSynchronize(p->copy_stream));   // hP must not be in flight when the caller gets it back
  if (rc != XC_OK) return rc;
  CU(cudaMemcpy2D(hV, (size_t)ldv * 8, p->d_Vtmp, (size_t)n * 8, (size_t)n * 8, n, cudaMemcpyDeviceToHost));
  return XC_OK;
}

int xc_eval_diagnostics(xc_plan* p, double* w, double* rho, double* grad_rho, double* E_batch, double* N_batch) {
  if (!p) return fail(XC_EINVAL, "plan is null");
  if (p->device < 0) return fail(XC_ECUDA, "host-only plan (device = -1)");
  const HostPlan& hp = p->hp;
  if ((rho || grad_rho) && !p->diag_valid) return fail(XC_EINVAL, "rho / grad_rho need the last xc_eval to have run with XC_EVAL_DIAG");
  DeviceGuard guard(p->device);
  CU(cudaDeviceSynchronize());
  if (w) CU(cudaMemcpy(w, p->d_w, hp.npts * 8, cudaMemcpyDeviceToHost));
  if (rho) CU(cudaMemcpy(rho, p->d_rho, hp.npts * 8, cudaMemcpyDeviceToHost));
  if (grad_rho) CU(cudaMemcpy(grad_rho, p->d_grho, hp.npts * 24, cudaMemcpyDeviceToHost));
  if (E_batch && !hp.batches.empty()) CU(cudaMemcpy(E_batch, p->d_Epart, hp.batches.size() * 8, cudaMemcpyDeviceToHost));
  if (N_batch && !hp.batches.empty()) CU(cudaMemcpy(N_batch, p->d_Npart, hp.batches.size() * 8, cudaMemcpyDeviceToHost));
  return XC_OK;
}

int xc_eval_timings(const xc_plan* p, float ms[5], int32_t* launches) {
  if (!p) return fail(XC_EINVAL, "plan is null");
  if (ms) std::copy(p->ms, p->ms + 5, ms);
  if (launches) *launches = p->launches;
  return XC_OK;
}

int xc_eval_counters(const xc_plan* p, int64_t* ssf_pairs, int64_t* nontrivial_points) {
  if (!p) return fail(XC_EINVAL, "plan is null");
  if (ssf_pairs) *ssf_pairs = p->ssf_pairs;
  if (nontrivial_points) {
    int64_t n = 0;
    for (const BatchRec& b : p->hp.batches) n += b.nq - b.ntriv;
    *nontrivial_points = n;
  }
  return XC_OK;
}

int xc_plan_destroy(xc_plan* p) {
  free_plan(p);
  return XC_OK;
}

int xc_integrate(const xc_atom* atoms, int32_t natoms, const xc_shell* shells, int32_t nshells, const double* exps,
                 const double* coefs, int32_t nprim_total, const xc_grid_spec* spec, int32_t device, const double* dP,
                 int64_t ldp, double* dV, int64_t ldv, double* E_xc, double* N_el, void* cuda_stream) {
  xc_plan* p = nullptr;
  int rc = xc_plan_create(atoms, natoms, shells, nshells, exps, coefs, nprim_total, spec, device, &p);
  if (rc != XC_OK) return rc;
  rc = xc_eval(p, dP, ldp, dV, ldv, E_xc, N_el, 0, cuda_stream);
  std::string keep = g_err;
  xc_plan_destroy(p);
  g_err = keep;
  return rc;
}

int xc_partition_weights(const xc_atom* atoms, int32_t natoms, int32_t partition, int64_t npts, const double* dx,
                         const double* dy, const double* dz, const double* dwq, const int32_t* dparent, double* dw_out,
                         void* cuda_stream) {
  if (!atoms || natoms < 1 || npts < 0 || (npts && (!dx || !dy || !dz || !dwq || !dparent || !dw_out)))
    return fail(XC_EINVAL, "bad argument");
  if (partition < 0 || partition > 1) return fail(XC_EINVAL, "bad partition enum");
  if (npts >= ((int64_t)1 << 31)) return fail(XC_EUNSUPPORTED, "more than 2^31 points");
  if (npts == 0) return XC_OK;
  // The kernels of xc_eval on an ad-hoc plan: pseudo-batches of 512 consecutive points, each with the bounding box of its
  // points and its own atom list (exact SSF support / every atom for Becke-88, sorted by distance to the box), no point
  // pre-classified as trivial.
  cudaStream_t st = (cudaStream_t)cuda_stream;
  const int64_t nbatch = (npts + 511) / 512;
  std::vector<double> a, ptab, box, hx, hy, hz;
  std::vector<int32_t> watoms, ids_small, ids_large;
  std::vector<BatchRec> recs;
  int nwarps = 8, max_small = 0, max_large = 0, max_list = 0;
  try {
    a.resize(3 * (size_t)natoms);
    for (int i = 0; i < natoms; ++i) {
      a[3 * i] = atoms[i].x; a[3 * i + 1] = atoms[i].y; a[3 * i + 2] = atoms[i].z;
      if (!std::isfinite(atoms[i].x) || !std::isfinite(atoms[i].y) || !std::isfinite(atoms[i].z)) return fail(XC_EINVAL, "non-finite atom coordinate");
    }
    for (int i = 0; i < natoms; ++i)
      for (int j = 0; j < i; ++j)
        if (a[3 * i] == a[3 * j] && a[3 * i + 1] == a[3 * j + 1] && a[3 * i + 2] == a[3 * j + 2]) return fail(XC_EINVAL, "two atoms coincide");
    if (partition == 1) pair_table(a, natoms, ptab);
    hx.resize(npts); hy.resize(npts); hz.resize(npts);
    CU(cudaStreamSynchronize(st));
    CU(cudaMemcpy(hx.data(), dx, npts * 8, cudaMemcpyDeviceToHost));
    CU(cudaMemcpy(hy.data(), dy, npts * 8, cudaMemcpyDeviceToHost));
    CU(cudaMemcpy(hz.data(), dz, npts * 8, cudaMemcpyDeviceToHost));
    recs.resize((size_t)nbatch);
    box.assign(6 * (size_t)nbatch, 0.0);
    std::vector<int32_t> lst;
    for (int64_t j = 0; j < nbatch; ++j) {
      BatchRec& b = recs[(size_t)j];
      std::memset(&b, 0, sizeof(b));
      b.pt_off = (int32_t)(j * 512); b.nq = (int32_t)std::min<int64_t>(512, npts - j * 512);
      double lo[3] = {1e300, 1e300, 1e300}, hi[3] = {-1e300, -1e300, -1e300};
      for (int64_t k = b.pt_off; k < (int64_t)b.pt_off + b.nq; ++k) {
        if (!std::isfinite(hx[k]) || !std::isfinite(hy[k]) || !std::isfinite(hz[k])) return fail(XC_EINVAL, "non-finite point coordinate");
        lo[0] = std::min(lo[0], hx[k]); hi[0] = std::max(hi[0], hx[k]);
        lo[1] = std::min(lo[1], hy[k]); hi[1] = std::max(hi[1], hy[k]);
        lo[2] = std::min(lo[2], hz[k]); hi[2] = std::max(hi[2], hz[k]);
      }
      for (int q = 0; q < 3; ++q) { box[6 * j + q] = lo[q]; box[6 * j + 3 + q] = hi[q]; }
      int nB = 0;
      weight_atom_list(a.data(), natoms, lo, hi, partition == 0, lst, nB);
      b.wa_off = (int64_t)watoms.size(); b.wa_nB = nB; b.wa_nC = (int32_t)lst.size();
      watoms.insert(watoms.end(), lst.begin(), lst.end());
      max_list = std::max(max_list, (int)lst.size());
      if ((int)lst.size() <= kWeightSmallList) { ids_small.push_back((int32_t)j); max_small = std::max(max_small, (int)lst.size()); }
      else { ids_large.push_back((int32_t)j); max_large = std::max(max_large, (int)lst.size()); }
    }
    if (partition == 1) {
      while (nwarps > 1 && weights_smem_bytes(max_list, nwarps) > kSmemLimit) nwarps >>= 1;
      if (weights_smem_bytes(max_list, nwarps) > kSmemLimit) return fail(XC_EUNSUPPORTED, "too many atoms for the Becke-88 weights kernel");
    }
  } catch (const std::bad_alloc&) {
    return fail(XC_ENOMEM, "host allocation failed");
  }
  double *da = nullptr, *dt = nullptr, *dbox = nullptr;
  int32_t *dl = nullptr, *dsm = nullptr, *dlg = nullptr;
  BatchRec* db = nullptr;
  int rc = upload(&da, a);
  if (rc == XC_OK) rc = upload(&dt, ptab);
  if (rc == XC_OK) rc = upload(&dbox, box);
  if (rc == XC_OK) rc = upload(&dl, watoms);
  if (rc == XC_OK) rc = upload(&db, recs);
  if (rc == XC_OK) rc = upload(&dsm, ids_small);
  if (rc == XC_OK) rc = upload(&dlg, ids_large);
  if (rc == XC_OK) {
    WeightArgs wa;
    wa.batches = db; wa.watoms = dl; wa.atoms = da; wa.invR = dt; wa.wbox = dbox; wa.natoms = natoms; wa.paircnt = nullptr;
    wa.px = dx; wa.py = dy; wa.pz = dz; wa.wq = dwq; wa.parent = dparent; wa.w = dw_out;
    cudaError_t e = cudaSuccess;
    if (partition == 0) {
      if (!ids_large.empty()) e = launch_weights_ssf(wa, dlg, (int)ids_large.size(), max_large, st);
      if (e == cudaSuccess && !ids_small.empty()) e = launch_weights_ssf(wa, dsm, (int)ids_small.size(), max_small, st);
    } else {
      e = launch_weights_becke(wa, nullptr, (int)nbatch, nwarps, max_list, st);
    }
    if (e == cudaSuccess) e = cudaStreamSynchronize(st);
    if (e != cudaSuccess) rc = cuda_fail(e, "xc_partition_weights");
  }
  cudaFree(da); cudaFree(dt); cudaFree(dbox); cudaFree(dl); cudaFree(db); cudaFree(dsm); cudaFree(dlg);
  return rc;
}

static_assert(kUksStaticMaxPoints == XC_STATIC_MAX_POINTS, "header and kernel agree on the static scratch size");
int xc_functional_uks_static(int32_t functional, int64_t npts, const double* d_w, const double* d_rho, const double* d_grho,
                             double rho_tol, double* d_cA, double* d_cG, double* d_out3, void* cuda_stream) {
  if (functional < 0 || functional > 1) return fail(XC_EINVAL, "xc_functional_uks_static: functional must be 0 (Slater+VWN5) or 1 (PBE)");
  if (npts < 0) return fail(XC_EINVAL, "xc_functional_uks_static: npts < 0");
  if (npts > kUksStaticMaxPoints)
    return fail(XC_EUNSUPPORTED, "xc_functional_uks_static: npts = " + std::to_string(npts) + " exceeds the static scratch (at most " +
                                     std::to_string(kUksStaticMaxPoints) + " points); use xc_eval_uks, which allocates");
  if (!(rho_tol > 0.0)) return fail(XC_EINVAL, "xc_functional_uks_static: rho_tol must be > 0 (reading A20)");
  if (!d_out3 || (npts && (!d_w || !d_rho || !d_cA || (functional == 1 && (!d_grho || !d_cG)))))
    return fail(XC_EINVAL, "xc_functional_uks_static: null argument");
  cudaStream_t st = (cudaStream_t)cuda_stream;
  if (npts == 0) { CU(cudaMemsetAsync(d_out3, 0, 24, st)); return XC_OK; }
  CU(functional_uks_static(functional == 1, npts, d_w, d_rho, d_grho, rho_tol, d_cA, d_cG, d_out3, st));
  return XC_OK;
}

int xc_functional(int32_t functional, int64_t n, const double* drho, const double* dsigma, double rho_tol, double* df,
                  double* dvrho, double* dvsigma, void* cuda_stream) {
  if (functional < 0 || functional > 1 || n < 0 || (n && (!drho || !df || !dvrho || !dvsigma)) || (functional == 1 && n && !dsigma))
    return fail(XC_EINVAL, "bad argument");
  CU(launch_functional(functional, n, drho, dsigma, rho_tol, df, dvrho, dvsigma, (cudaStream_t)cuda_stream));
  return XC_OK;
}

}  // extern "C"
