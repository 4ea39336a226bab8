// xc_api.cu -- the C ABI of libxc_b200 (include/xc_b200.h): plan lifetime, uploads, the stream-ordered
// launch sequence of one E_xc / V_xc / N_el build (Alg. 2 l.2.2-2.9 on one GPU), diagnostics.
#include <cuda_runtime.h>

#include <algorithm>
#include <cmath>
#include <cstdio>
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
  double *d_atoms = nullptr, *d_invR = nullptr, *d_rnn = nullptr;
  ShellRec* d_shells = nullptr;
  double *d_exps = nullptr, *d_coefs = nullptr;
  BatchRec* d_batches = nullptr;
  int32_t *d_bshells = nullptr, *d_bsfoff = nullptr, *d_bfidx = nullptr, *d_bfinfo = nullptr;
  double *d_wbox = nullptr;
  double2* d_pairtab = nullptr;
  int32_t *d_watoms = nullptr, *d_wsmall = nullptr, *d_wlarge = nullptr;
  int32_t *d_ids_small = nullptr, *d_ids_large = nullptr;
  double* d_ppk = nullptr;
  unsigned long long *d_vhi = nullptr, *d_vlo = nullptr;
  double *d_Epart = nullptr, *d_Npart = nullptr, *d_result = nullptr;
  double *d_rho = nullptr, *d_grho = nullptr;
  double* h_result = nullptr;  // pinned
  double *d_Ptmp = nullptr, *d_Vtmp = nullptr;  // for xc_eval_host
  bool weights_valid = false;
  std::vector<cudaEvent_t> ev;
  float ms[5] = {0, 0, 0, 0, 0};
  int launches = 0;
};

static void free_plan(xc_plan* p) {
  if (!p) return;
  if (p->device < 0) { delete p; return; }
  cudaSetDevice(p->device);
  void* ptrs[] = {p->d_px, p->d_py, p->d_pz, p->d_wq, p->d_w, p->d_parent, p->d_atoms, p->d_invR, p->d_rnn, p->d_shells,
                  p->d_exps, p->d_coefs, p->d_batches, p->d_bshells, p->d_bsfoff, p->d_bfidx, p->d_bfinfo, p->d_ids_small,
                  p->d_ids_large, p->d_ppk, p->d_vhi, p->d_vlo, p->d_Epart, p->d_Npart, p->d_result,
                  p->d_rho, p->d_grho, p->d_Ptmp, p->d_Vtmp, p->d_watoms, p->d_wsmall, p->d_wlarge, p->d_pairtab, p->d_wbox};
  for (void* q : ptrs) if (q) cudaFree(q);
  if (p->h_result) cudaFreeHost(p->h_result);
  for (cudaEvent_t e : p->ev) cudaEventDestroy(e);
  delete p;
}

static void atom_tables(const std::vector<double>& atoms, int natoms, std::vector<double>& invR, std::vector<double>& rnn) {
  invR.assign((size_t)natoms * natoms, 0.0);
  rnn.assign(natoms, 1e300);
  for (int a = 0; a < natoms; ++a)
    for (int b = 0; b < natoms; ++b) {
      if (a == b) continue;
      double dx = atoms[3 * a] - atoms[3 * b], dy = atoms[3 * a + 1] - atoms[3 * b + 1], dz = atoms[3 * a + 2] - atoms[3 * b + 2];
      double r = std::sqrt(dx * dx + dy * dy + dz * dz);
      invR[(size_t)a * natoms + b] = 1.0 / r;
      rnn[a] = std::min(rnn[a], r);
    }
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
  try {
    rc = build_host_plan(atoms, natoms, shells, nshells, exps, coefs, nprim_total, spec, p->hp, err);
  } catch (const std::bad_alloc&) {
    rc = XC_ENOMEM; err = "host allocation failed in planner";
  }
  if (rc != XC_OK) { free_plan(p); return fail(rc, err); }
  HostPlan& hp = p->hp;
  if (device == -1) { *out = p; return XC_OK; }   // host-only plan: info / stats / export only
  auto bail = [&](int code) { free_plan(p); return code; };
  if (cudaSetDevice(device) != cudaSuccess) return bail(fail(XC_ECUDA, "cudaSetDevice failed"));
  std::vector<double> invR, rnn;
  atom_tables(hp.atoms, hp.natoms, invR, rnn);
#define UP(d, h) do { int _r = upload(&p->d, h); if (_r != XC_OK) return bail(_r); } while (0)
  UP(d_px, hp.px); UP(d_py, hp.py); UP(d_pz, hp.pz); UP(d_wq, hp.wq); UP(d_parent, hp.parent);
  UP(d_atoms, hp.atoms); UP(d_invR, invR); UP(d_rnn, rnn);
  if (hp.spec.partition == 0) {   // SSF pair table: a R_BC, 1 / (a R_BC)
    std::vector<double2> tab(invR.size());
    for (size_t k = 0; k < invR.size(); ++k) tab[k] = invR[k] > 0.0 ? make_double2(0.64 / invR[k], invR[k] / 0.64) : make_double2(0.0, 0.0);
    UP(d_pairtab, tab);
  }
  UP(d_shells, hp.shells); UP(d_exps, hp.exps); UP(d_coefs, hp.coefs);
  UP(d_batches, hp.batches); UP(d_bshells, hp.bshells); UP(d_bsfoff, hp.bsfoff); UP(d_bfidx, hp.bfidx); UP(d_bfinfo, hp.bfinfo);
  UP(d_wbox, hp.wbox);
  UP(d_watoms, hp.watoms); UP(d_wsmall, hp.wbatch_small); UP(d_wlarge, hp.wbatch_large);
  UP(d_ids_small, hp.ids_small); UP(d_ids_large, hp.ids_large);
#undef UP
  size_t nitems = hp.batches.size();
  size_t nb2 = (size_t)hp.nbasis * hp.nbasis;
#define AL(d, bytes) do { cudaError_t _e = cudaMalloc((void**)&p->d, std::max<size_t>((bytes), 8)); if (_e != cudaSuccess) return bail(cuda_fail(_e, "cudaMalloc " #d)); } while (0)
  AL(d_w, hp.npts * 8); AL(d_ppk, (size_t)hp.ppk_doubles * 8);
  AL(d_vhi, nb2 * 8); AL(d_vlo, nb2 * 8); AL(d_Epart, nitems * 8); AL(d_Npart, nitems * 8); AL(d_result, 16);
  AL(d_rho, hp.npts * 8); AL(d_grho, hp.npts * 24);
#undef AL
  if (cudaMemset(p->d_Epart, 0, std::max<size_t>(nitems * 8, 8)) != cudaSuccess || cudaMemset(p->d_Npart, 0, std::max<size_t>(nitems * 8, 8)) != cudaSuccess)
    return bail(fail(XC_ECUDA, "cudaMemset failed"));   // batches without functions never write their partials
  if (cudaMallocHost((void**)&p->h_result, 16) != cudaSuccess) return bail(fail(XC_ENOMEM, "cudaMallocHost failed"));
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
  if (pts) for (int64_t i = 0; i < hp.npts; ++i) { pts[3 * i] = hp.px[i]; pts[3 * i + 1] = hp.py[i]; pts[3 * i + 2] = hp.pz[i]; }
  if (wq) std::copy(hp.wq.begin(), hp.wq.end(), wq);
  if (parent) std::copy(hp.parent.begin(), hp.parent.end(), parent);
  if (orig) std::copy(hp.orig.begin(), hp.orig.end(), orig);
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
  CU(cudaSetDevice(p->device));
  const bool gga = hp.spec.functional == 1;
  int launches = 0;
  size_t ie = 0;
  CU(cudaEventRecord(p->ev[ie++], st));
  if (!(flags & 1) || !p->weights_valid) {
    WeightArgs wa;
    wa.batches = p->d_batches; wa.watoms = p->d_watoms; wa.atoms = p->d_atoms; wa.invR = p->d_invR; wa.rnn = p->d_rnn;
    wa.pairtab = p->d_pairtab; wa.wbox = p->d_wbox; wa.natoms = hp.natoms; wa.px = p->d_px; wa.py = p->d_py; wa.pz = p->d_pz; wa.wq = p->d_wq; wa.parent = p->d_parent; wa.w = p->d_w;
    if (!hp.wbatch_large.empty()) {   // long lists first: they are the long pole
      CU(launch_weights_batched(hp.spec.partition, wa, p->d_wlarge, (int)hp.wbatch_large.size(), hp.w_warps_large, hp.w_max_large, st));
      ++launches;
    }
    if (!hp.wbatch_small.empty()) {
      CU(launch_weights_batched(hp.spec.partition, wa, p->d_wsmall, (int)hp.wbatch_small.size(), 8, hp.w_max_small, st));
      ++launches;
    }
    p->weights_valid = true;
  }
  CU(cudaEventRecord(p->ev[ie++], st));
  size_t nb2 = (size_t)hp.nbasis * hp.nbasis;
  CU(cudaMemsetAsync(p->d_vhi, 0, nb2 * 8, st));
  CU(cudaMemsetAsync(p->d_vlo, 0, nb2 * 8, st));
  CU(cudaMemsetAsync(p->d_rho, 0, hp.npts * 8, st));
  CU(cudaMemsetAsync(p->d_grho, 0, hp.npts * 24, st));
  BatchArgs ba;
  ba.batches = p->d_batches; ba.bshells = p->d_bshells; ba.bsfoff = p->d_bsfoff; ba.bfidx = p->d_bfidx; ba.bfinfo = p->d_bfinfo;
  ba.shells = p->d_shells; ba.exps = p->d_exps; ba.coefs = p->d_coefs;
  ba.px = p->d_px; ba.py = p->d_py; ba.pz = p->d_pz; ba.w = p->d_w;
  ba.P = dP; ba.ldp = ldp; ba.ppk = p->d_ppk;
  ba.rho_out = p->d_rho; ba.grho_out = gga ? p->d_grho : nullptr;
  ba.Epart = p->d_Epart; ba.Npart = p->d_Npart; ba.vhi = p->d_vhi; ba.vlo = p->d_vlo; ba.nbasis = hp.nbasis;
  ba.rho_tol = hp.spec.rho_tol;
  // P^j pack (Alg. 4 l.4.2), then the fused batch kernel (l.4.3-4.10); large N_b^j first
  if (!hp.ids_large.empty()) { CU(launch_pack(ba, p->d_ids_large, (int)hp.ids_large.size(), !gga, st)); ++launches; }
  if (!hp.ids_small.empty()) { CU(launch_pack(ba, p->d_ids_small, (int)hp.ids_small.size(), !gga, st)); ++launches; }
  CU(cudaEventRecord(p->ev[ie++], st));
  if (!hp.ids_large.empty()) { CU(launch_batch(1, gga, ba, p->d_ids_large, (int)hp.ids_large.size(), hp.smem_large, st)); ++launches; }
  if (!hp.ids_small.empty()) { CU(launch_batch(0, gga, ba, p->d_ids_small, (int)hp.ids_small.size(), hp.smem_small, st)); ++launches; }
  CU(cudaEventRecord(p->ev[ie++], st));
  CU(launch_finalize(hp.nbasis, p->d_vhi, p->d_vlo, dV, ldv, st));
  CU(launch_reduce((int64_t)hp.batches.size(), p->d_Epart, p->d_Npart, p->d_result, st));
  launches += 2;
  CU(cudaMemcpyAsync(p->h_result, p->d_result, 16, cudaMemcpyDeviceToHost, st));
  CU(cudaEventRecord(p->ev[ie++], st));
  CU(cudaStreamSynchronize(st));
  *E_xc = p->h_result[0];
  *N_el = p->h_result[1];
  // stage timings
  float t;
  p->ms[0] = p->ms[1] = p->ms[2] = p->ms[3] = p->ms[4] = 0.f;
  CU(cudaEventElapsedTime(&t, p->ev[0], p->ev[1])); p->ms[0] = t;
  CU(cudaEventElapsedTime(&t, p->ev[1], p->ev[2])); p->ms[1] = t;   // includes the memsets
  CU(cudaEventElapsedTime(&t, p->ev[2], p->ev[3])); p->ms[2] = t;
  CU(cudaEventElapsedTime(&t, p->ev[3], p->ev[4])); p->ms[3] = t;
  CU(cudaEventElapsedTime(&t, p->ev[0], p->ev[4])); p->ms[4] = t;
  p->launches = launches;
  return XC_OK;
}

int xc_eval_host(xc_plan* p, const double* hP, int64_t ldp, double* hV, int64_t ldv, double* E_xc, double* N_el, int32_t flags) {
  if (!p || !hP || !hV) return fail(XC_EINVAL, "null argument");
  if (p->device < 0) return fail(XC_ECUDA, "host-only plan (device = -1): no CUDA device bound, and there is no CPU fallback");
  const int n = p->hp.nbasis;
  if (ldp < n || ldv < n) return fail(XC_EINVAL, "leading dimension smaller than n_basis");
  CU(cudaSetDevice(p->device));
  size_t bytes = (size_t)n * n * 8;
  if (!p->d_Ptmp) CU(cudaMalloc((void**)&p->d_Ptmp, bytes));
  if (!p->d_Vtmp) CU(cudaMalloc((void**)&p->d_Vtmp, bytes));
  CU(cudaMemcpy2DAsync(p->d_Ptmp, (size_t)n * 8, hP, (size_t)ldp * 8, (size_t)n * 8, n, cudaMemcpyHostToDevice, 0));
  int rc = xc_eval(p, p->d_Ptmp, n, p->d_Vtmp, n, E_xc, N_el, flags, nullptr);
  if (rc != XC_OK) return rc;
  CU(cudaMemcpy2D(hV, (size_t)ldv * 8, p->d_Vtmp, (size_t)n * 8, (size_t)n * 8, n, cudaMemcpyDeviceToHost));
  return XC_OK;
}

int xc_eval_diagnostics(xc_plan* p, double* w, double* rho, double* grad_rho, double* E_batch, double* N_batch) {
  if (!p) return fail(XC_EINVAL, "plan is null");
  if (p->device < 0) return fail(XC_ECUDA, "host-only plan (device = -1)");
  const HostPlan& hp = p->hp;
  CU(cudaSetDevice(p->device));
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
  std::vector<double> a(3 * (size_t)natoms), invR, rnn;
  for (int i = 0; i < natoms; ++i) { a[3 * i] = atoms[i].x; a[3 * i + 1] = atoms[i].y; a[3 * i + 2] = atoms[i].z; }
  atom_tables(a, natoms, invR, rnn);
  double *da = nullptr, *di = nullptr, *dr = nullptr;
  int rc = upload(&da, a);
  if (rc == XC_OK) rc = upload(&di, invR);
  if (rc == XC_OK) rc = upload(&dr, rnn);
  cudaStream_t st = (cudaStream_t)cuda_stream;
  if (rc == XC_OK) {
    cudaError_t e = launch_weights(partition, natoms, da, di, dr, npts, dx, dy, dz, dwq, dparent, dw_out, st);
    if (e == cudaSuccess) e = cudaStreamSynchronize(st);
    if (e != cudaSuccess) rc = cuda_fail(e, "xc_partition_weights");
  }
  cudaFree(da); cudaFree(di); cudaFree(dr);
  return rc;
}

int xc_functional(int32_t functional, int64_t n, const double* drho, const double* dsigma, double rho_tol, double* df,
                  double* dvrho, double* dvsigma, void* cuda_stream) {
  if (functional < 0 || functional > 1 || n < 0 || (n && (!drho || !df || !dvrho || !dvsigma)) || (functional == 1 && n && !dsigma))
    return fail(XC_EINVAL, "bad argument");
  CU(launch_functional(functional, n, drho, dsigma, rho_tol, df, dvrho, dvsigma, (cudaStream_t)cuda_stream));
  return XC_OK;
}

}  // extern "C"
