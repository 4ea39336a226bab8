// xc_kernels.h -- launch interface between the C ABI (xc_api.cu) and the kernels (xc_kernels.cu).
#pragma once
#include <cuda_runtime.h>

#include "xc_internal.h"

namespace xcb {

struct BatchArgs {
  const BatchRec* batches;
  const int32_t* bshells;
  const int32_t* bsfoff;
  const int32_t* bfidx;
  const ShellRec* shells;
  const double* exps;
  const double* coefs;
  const double* px; const double* py; const double* pz; const double* w;
  const double* P; int64_t ldp;
  double* ppk;                         // packed P^j of every batch (DMMA B-fragment order)
  double* rho_out; double* grho_out;   // optional diagnostics (may be null); mode 1: rho_s / grad rho_s of one spin
  const double* cA; const double* cG;  // mode 2: per-point coefficients of Z^s, a [npts] and g [npts][3]
  double* Epart; double* Npart;        // one partial per batch
  unsigned long long* vhi; unsigned long long* vlo;   // fixed-point V accumulator (lower triangle), value = (hi 2^32 + lo) 2^(vexp - 64)
  int vexp;
  unsigned* vflags;                    // [0] high word of the largest |increment| of V, [1] != 0: a non-finite increment was met
  int nbasis;
  double rho_tol;
};

struct WeightArgs {
  const BatchRec* batches;
  const int32_t* watoms;
  const double* atoms;
  const double* invR;    // [natoms][natoms] 1 / R_BC (Becke-88), 0 on the diagonal
  const double* wbox;    // [nbatch][6] tight bounding boxes (lo xyz, hi xyz)
  int natoms;
  const double* px; const double* py; const double* pz; const double* wq; const int32_t* parent;
  double* w;
  unsigned long long* paircnt;   // null, or: counter of the pair factors s(mu_BC) the SSF kernel evaluated (XC_EVAL_COUNT_PAIRS)
};

// SSF: one CTA per batch, one warp per non-trivial point; max_list = longest atom list among the batches launched
cudaError_t launch_weights_ssf(const WeightArgs& a, const int32_t* batch_ids, int nbatches, int max_list, cudaStream_t st);
// Becke-88: one CTA per batch (batch_ids may be null: batch = block index)
cudaError_t launch_weights_becke(const WeightArgs& a, const int32_t* batch_ids, int nbatches, int nwarps, int max_list, cudaStream_t st);
cudaError_t launch_functional(int kind, int64_t n, const double* rho, const double* sigma, double rho_tol, double* f,
                              double* vr, double* vs, cudaStream_t st);
cudaError_t launch_pack(const BatchArgs& a, const int32_t* batch_ids, int nbatches, bool tri, cudaStream_t st);
// cls 1: the first n_heavy batches of the list have N_b^j > kMidNb (one launch of the five-round kernel), the others run the
// three-round kernel; *launched (may be null) receives the number of kernels launched (1 or 2)
cudaError_t launch_batch(int cls, bool gga, int mode, const BatchArgs& a, const int32_t* batch_ids, int nbatches, size_t smem,
                         cudaStream_t st, int n_heavy = 0, int* launched = nullptr);
// spin-unrestricted build: functional over the grid (xc_uks.cu); rho [2][npts], grho [2][npts][3] in, cA [2][npts], cG [2][npts][3]
// and out3 = (E_xc, N_a, N_b) out; part: scratch of 3 * uks_functional_blocks(npts) doubles
int64_t uks_functional_blocks(int64_t npts);
cudaError_t launch_functional_uks(bool gga, int64_t npts, const double* w, const double* rho, const double* grho, double rho_tol,
                                  double* cA, double* cG, double* part, double* out3, cudaStream_t st);
// the same without any allocation: block partials in a file-scope device array (xc_uks.cu); npts <= kUksStaticMaxPoints;
// works on the CURRENT device; calls that overlap on one GPU race on the array
constexpr int64_t kUksStaticMaxPoints = (int64_t)1 << 23;   // 32768 blocks of 256 points: 768 KB of partials per GPU
cudaError_t functional_uks_static(bool gga, int64_t npts, const double* w, const double* rho, const double* grho, double rho_tol,
                                  double* cA, double* cG, double* out3, cudaStream_t st);
// restricted meta-GGA (reading A23): functional over the grid and per-batch E / N partials (xc_uks.cu)
cudaError_t launch_functional_mgga(int64_t npts, int nbatches, const BatchRec* batches, const double* w, const double* rho, const double* grho,
                                   const double* tau, double rho_tol, double* cA, double* cG, double* cT, double* ef, double* en, double* Epart,
                                   double* Npart, cudaStream_t st);
cudaError_t launch_finalize(int nbasis, const unsigned long long* vhi, const unsigned long long* vlo, double* V,
                            int64_t ldv, int vexp, bool poison, cudaStream_t st);
cudaError_t launch_reduce(int64_t n, const double* ep, const double* np, double* out, cudaStream_t st);

}  // namespace xcb
