/* xc_b200.h -- C ABI of the B200 (sm_100a) exchange-correlation integrator.
 *
 * Computes, on ONE GPU and in fp64, the numerical quadrature of the XC energy and
 * potential matrix in a contracted Cartesian Gaussian basis over an atom-centred, partition-weighted
 * molecular grid -- the "local integration" of arxiv 2007.03143 (Alg. 2 Input/Output, PAPER.md:L192:
 * "Input: density matrix P, basis functions S, atomic centers A.  Output: V^xc, E^xc"; Alg. 4,
 * PAPER.md:L255-L283):
 *
 *     E_xc = sum_i w_i f(rho_i, sigma_i)                         Eq. (2),(16)
 *     V_mn = sum_i Z_mi Phi_ni + Phi_mi Z_ni                     Eq. (5),(17),(18)
 *     Z_mi = 1/2 (w v_rho)_i Phi_mi + 2 (w v_sigma)_i grad rho_i . grad Phi_mi      Eq. (6),(20)
 *     rho_i = sum_m Phi_mi X_mi,  grad rho_i = 2 sum_m grad Phi_mi X_mi,  X = P^j Phi^j   Eqs. (13)-(15)
 *     N_el = sum_i w_i rho_i
 *
 * with w_i = w_i^q p_A(r_i) the SSF (or Becke-88) partition weights, Eq. (9), points
 * grouped into spatial batches of <= max_batch_pts points with per-batch shell screening by the
 * cuboid/sphere test of Alg. 1 and the cutoff radius of Eq. (10).
 * Readings of ambiguous passages are listed in DESIGN.md (A1..A18).
 *
 * Conventions
 *   - units: bohr / hartree.  All floating point is IEEE double.
 *   - function order in P and V: shells in input order; inside a shell the Cartesian components
 *     (l,m,n), l descending then m descending: p = x,y,z; d = xx,xy,xz,yy,yz,zz ((L+1)(L+2)/2 of them).
 *     A d shell flagged XC_SHELL_PURE holds the five real solid harmonics instead ("spherical Gaussian
 *     functions", L323 cc-pVDZ; reading A19), m = -2..2, in terms of the Cartesian functions of the same radial part:
 *     sqrt3 xy, sqrt3 yz, zz - (xx + yy)/2, sqrt3 xz, (sqrt3/2)(xx - yy).
 *   - coefficients are used as given (primitive norms included by the caller); nothing is renormalised.
 *   - every entry point returns 0 (XC_OK) or a negative XC_E* code; nothing throws or aborts across the
 *     ABI.  xc_last_error() returns a thread-local text for the last failure (CUDA error string included).
 *   - HOST pointers are marked [host], DEVICE pointers [device].  The library never frees caller memory
 *     and keeps no caller pointer after a call returns.
 *   - there is no CPU fallback: without a CUDA device every compute entry point fails with XC_ECUDA.
 */
#ifndef XC_B200_H
#define XC_B200_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define XC_OK            0
#define XC_EINVAL       -1  /* null pointer, bad size, ld < n_basis, non-positive exponent, bad enum */
#define XC_EUNSUPPORTED -2  /* L > 2, nprim > 16, batch cannot be screened below the kernel's limit */
#define XC_ENOMEM       -3  /* host or device allocation failed */
#define XC_ECUDA        -4  /* CUDA runtime error (text in xc_last_error) */

typedef struct { double x, y, z; int32_t Z; int32_t _pad; } xc_atom;           /* position (bohr), atomic number */
#define XC_SHELL_PURE 0x100  /* OR-ed into xc_shell.L: pure (real solid harmonic) shell; changes d shells only (5 functions) */
typedef struct { int32_t atom; int32_t L; int32_t nprim; int32_t prim_off; } xc_shell; /* contracted shell, Eq. (7); L = 0..2 [| XC_SHELL_PURE] */

typedef struct {
  int32_t n_rad, n_ang;   /* radial x angular points per atom (Table 2) */
  int32_t radial;         /* 0 = Mura-Knowles, m = 3 (reading A3) */
  int32_t angular;        /* 0 = Fibonacci sphere; 1 = Gauss-Legendre(cos theta) x trapezoid(phi), n_ang = 2 n_theta^2 (reading A4) */
  int32_t partition;      /* 0 = SSF, a = 0.64; 1 = Becke-1988, 3 iterations, no size adjustment (reading A1/A2) */
  int32_t functional;     /* 0 = LDA Slater+VWN5; 1 = GGA PBE; 2 = meta-GGA MS0 exchange + PBE correlation (reading A23;
                             PAPER.md:L51): xc_eval runs it as passes of the same kernels (densities, tau, functional, potential) */
  int32_t max_batch_pts;  /* <= 512 */
  int32_t flags;          /* bit 0: reserved; bit 1 = XC_SPEC_SPLIT_CLASS1 (a tuning knob, results unchanged bit for bit) */
  double  eta;            /* Eq. (10) tolerance, 1e-10 */
  double  mk_alpha;       /* Mura-Knowles scale, bohr (5.0) */
  double  rho_tol;        /* points with rho <= rho_tol contribute nothing (1e-15, reading A12) */
} xc_grid_spec;

/* xc_grid_spec.flags.  XC_SPEC_SPLIT_CLASS1: batches with 112 < N_b^j <= 144 always run the three-round instantiation of the
 * batch kernel (its V^j accumulators stay in registers), the ones beyond 144 as a launch of their own; by default the planner
 * does that only when at least 4096 batches profit (or none is beyond 144) and otherwise keeps the class one five-round launch. */
#define XC_SPEC_SPLIT_CLASS1 2

/* flags of xc_eval / xc_eval_host */
#define XC_EVAL_REUSE_WEIGHTS 1   /* reuse the partition weights of the previous xc_eval on this plan (skip step (a); reading A16) */
#define XC_EVAL_DIAG          2   /* also store rho and grad rho of every point for xc_eval_diagnostics (parity tests; costs 32 B/point) */
#define XC_EVAL_COUNT_PAIRS   4   /* count the pair factors s(mu_BC) step (a) evaluates (SSF), for xc_eval_counters; perturbs the timing slightly */

typedef struct xc_plan xc_plan;   /* opaque: owns host + device copies of grid, batches, basis, workspaces */

/* Step (b) of the hot path + all uploads: builds the atom-centred grid (O1-O3), batches the points into
 * cuboids of <= max_batch_pts points by recursive median bisection of the whole point cloud (the batching
 * scheme is free; it satisfies Eq. (11)), screens shells per batch with Alg. 1
 * on the batch's tight bounding box, and uploads everything to `device`.  With device >= 0 the per-point stages (grid
 * points, bisection, Morton order inside the batches, the permuted point arrays) run on that GPU and the arrays stay
 * there ("could be implemented on GPU"); the plan is bit-identical to the one the host makes.
 *   atoms   [host] natoms entries;  shells [host] nshells entries;  exps, coefs [host] nprim_total each.
 * device = -1 builds a HOST-ONLY plan (no CUDA call is made): xc_plan_info / xc_plan_stats / xc_plan_export work on
 * it, every compute entry point returns XC_ECUDA.  It exists so that the planner can be validated without a GPU.
 * On success *out owns the plan (free with xc_plan_destroy).  Errors: XC_EINVAL, XC_EUNSUPPORTED, XC_ENOMEM, XC_ECUDA. */
int xc_plan_create(const xc_atom* atoms, int32_t natoms, const xc_shell* shells, int32_t nshells,
                   const double* exps, const double* coefs, int32_t nprim_total,
                   const xc_grid_spec* spec, int32_t device, xc_plan** out);

/* Sizes of a plan.  Any output pointer may be NULL.  n_shell_entries = sum_j |S_j| (shells, not functions);
 * algorithmic_flops = sum_j 4 (N_b^j)^2 N_q^j (Eq. (22) PAPER.md:L196 with each MAC = 2 flop). */
int xc_plan_info(const xc_plan* plan, int64_t* n_points, int64_t* n_batches, int32_t* n_basis,
                 int64_t* n_shell_entries, double* algorithmic_flops);

/* The plan as DATA, for the oracle (reading A9).  All [host], caller-allocated with the sizes of xc_plan_info:
 *   pts 3*n_points (x,y,z per point, batch-contiguous order), wq n_points (base weights w^q),
 *   parent n_points (parent atom), orig n_points (index of the point in the canonical atom-major /
 *   radial / angular grid order), batch_off n_batches+1, shell_off n_batches+1, shells n_shell_entries
 *   (global shell ids, ascending inside a batch).  Any pointer may be NULL to skip it. */
int xc_plan_export(const xc_plan* plan, double* pts, double* wq, int32_t* parent, int64_t* orig,
                   int64_t* batch_off, int64_t* shell_off, int32_t* shells);

/* Steps (a),(c)-(g): one full E_xc / V_xc / N_el build, stream-ordered on `cuda_stream` (a cudaStream_t, may be 0).
 *   dP [device] n_basis x n_basis, leading dimension ldp >= n_basis, symmetric (assumed, not checked), read only.
 *   dV [device] n_basis x n_basis, leading dimension ldv >= n_basis: OVERWRITTEN (Alg. 2 l.2.4),
 *      both triangles written, exactly symmetric, bit-identical from run to run.
 *   E_xc, N_el [host] scalars, valid when the call returns (the call synchronises the stream once, at the end).
 *   flags: XC_EVAL_REUSE_WEIGHTS ("cached-weights build", reading A16), XC_EVAL_DIAG; 0 = full build, nothing but the
 *          three outputs is produced.
 * The increments of V are summed in 96-bit fixed point whose exponent adapts to the build (the plan remembers it): if a
 * build's increments do not fit the remembered exponent, steps (c)-(g) are repeated once.  A non-finite value in P (or
 * produced on the way) is never dropped: E_xc, N_el and all of V come back NaN and the call returns XC_EINVAL.
 * A plan is not re-entrant: it owns the workspaces of its builds, so two xc_eval calls on ONE plan must not overlap
 * (different plans may run concurrently).  The caller's current CUDA device is left unchanged. */
int xc_eval(xc_plan* plan, const double* dP, int64_t ldp, double* dV, int64_t ldv,
            double* E_xc, double* N_el, int32_t flags, void* cuda_stream);

/* Same build with HOST buffers: copies P to the device (on a stream of its own, overlapping step (a), which reads no P),
 * runs xc_eval on the default stream, copies V back.  hP, hV [host] (pinned memory makes the copies asynchronous). */
int xc_eval_host(xc_plan* plan, const double* hP, int64_t ldp, double* hV, int64_t ldv,
                 double* E_xc, double* N_el, int32_t flags);

/* Spin-unrestricted build ("may be extended to ... spin-unrestricted ... with the
 * addition of only a few intermediates"; readings A20-A22).  rho_s = sum P^s_mu,nu phi_mu phi_nu for s = a, b (no factor 2:
 * a closed shell is P^a = P^b = P/2), f = f(rho_a, rho_b, s_aa, s_ab, s_bb) is the spin-polarised Slater+VWN5 or PBE,
 *   Z^s = 1/2 w v_rho_s Phi + w (2 v_ss grad rho_s + v_ab grad rho_s') . grad Phi,  V^s,j = Z^s Phi^T + Phi Z^s^T.
 *   dPa, dPb [device] read-only, symmetric; dVa, dVb [device] OVERWRITTEN, symmetric, bit-identical from run to run.
 *   E_xc [host] scalar; N_ab [host] two doubles: sum w rho_a, sum w rho_b.
 *   A point contributes nothing when rho_a + rho_b <= rho_tol; a spin density below rho_tol is raised to rho_tol before
 *   the functional is evaluated (zeta = +-1 is singular), so grid_spec.rho_tol must be > 0 (else XC_EINVAL).
 *   flags: XC_EVAL_REUSE_WEIGHTS.  Error behaviour, re-entrancy and stream semantics as xc_eval.
 * The same kernels run as passes: per spin {P^s,j pack, collocation + X GEMM + densities}, the functional over the grid,
 * per spin {collocation + Z^s + V^s,j GEMM + increment, finalise}. */
int xc_eval_uks(xc_plan* plan, const double* dPa, const double* dPb, int64_t ldp, double* dVa, double* dVb, int64_t ldv,
                double* E_xc, double* N_ab, int32_t flags, void* cuda_stream);

/* rho_s [2][n_points] and grad rho_s [2][n_points][3] (GGA plans) of the last xc_eval_uks, plan order, [host], either may
 * be NULL; entries of points with w = 0 are undefined (never evaluated). */
int xc_eval_uks_densities(const xc_plan* plan, double* rho, double* grad_rho);

/* The meta-GGA intermediate ("more advanced DFAs (such as the meta-GGA) with the addition of only a few
 * intermediates"; reading A22): tau_i = 1/2 sum_mu grad Phi_mu,i . grad X_mu,i, X = P^j Phi^j (Eq. (15)), for the
 * density matrix dP [device] (one spin's, or the total one), with the batches' shell lists as for rho.
 *   d_tau [device] n_points doubles, plan order (xc_plan_export), OVERWRITTEN; 0 at the points with w = 0 (never
 *   evaluated).  Runs step (a) first unless XC_EVAL_REUSE_WEIGHTS.  No tau-dependent functional is built on it. */
int xc_eval_tau(xc_plan* plan, const double* dP, int64_t ldp, double* d_tau, int32_t flags, void* cuda_stream);

/* Diagnostics of the last xc_eval on this plan, for parity tests at full size.  All [host], may be NULL:
 *   w n_points final partition weights (plan order);  rho n_points;  grad_rho 3*n_points (zeros for LDA) -- these two
 *   only if that xc_eval ran with XC_EVAL_DIAG (else XC_EINVAL), and only at points with w != 0;
 *   E_batch, N_batch n_batches: per-batch partial sums of w f and w rho. */
int xc_eval_diagnostics(xc_plan* plan, double* w, double* rho, double* grad_rho, double* E_batch, double* N_batch);

/* Device time in milliseconds of each stage of the last xc_eval (CUDA events on the eval stream):
 * ms[0] weights (a), ms[1] P^j pack (d1 gather; includes zeroing the accumulators), ms[2] fused batch kernel (c,d1,e,f,d2,g),
 * ms[3] finalise, ms[4] total.
 * launches: number of kernel launches of that xc_eval. */
int xc_eval_timings(const xc_plan* plan, float ms[5], int32_t* launches);

/* Work counters for the roofline of step (a) ("plain FP64 ALU ... report pairs/point"): ssf_pairs = pair
 * factors s(mu_BC) evaluated (lane slots of the 32-wide chunks) by the last xc_eval that ran step (a) with
 * XC_EVAL_COUNT_PAIRS, -1 if there was none; nontrivial_points = points of the plan the SSF kernel visits (the others have
 * w = w^q exactly, Eq. (9) with every mu_AC <= -a).  Either pointer may be NULL. */
int xc_eval_counters(const xc_plan* plan, int64_t* ssf_pairs, int64_t* nontrivial_points);

/* Algorithmic sizes of the plan used by the roofline report: [0] sum_j N_b^j N_q^j (function-points),
 * [1] sum_j (N_b^j)^2, [2] sum_j 4 (N_b^j)^2 N_q^j, [3] max N_b^j, [4] mean N_q^j, [5] bytes of the packed-P^j buffer,
 * [6] mean and [7] max length of the per-batch partner-atom lists of step (a), [8] mean and [9] max length of the
 * owner-atom lists, [10] max |S_j| (shells), [11] reserved (0). */
int xc_plan_stats(const xc_plan* plan, double stats[12]);

int xc_plan_destroy(xc_plan* plan);

/* One-shot form named by BASELINE.json:north_star = create + eval + destroy. */
int xc_integrate(const xc_atom* atoms, int32_t natoms, const xc_shell* shells, int32_t nshells,
                 const double* exps, const double* coefs, int32_t nprim_total, const xc_grid_spec* spec,
                 int32_t device, const double* dP, int64_t ldp, double* dV, int64_t ldv,
                 double* E_xc, double* N_el, void* cuda_stream);

/* Stand-alone kernels of single steps, for element-wise parity tests (device pointers, stream-ordered):
 *   xc_partition_weights: step (a) on arbitrary points. pts [device] 3 arrays x,y,z; parent, wq, w_out [device] npts.
 *   xc_functional: step (f) point values. rho, sigma, f, vrho, vsigma [device] n each. */
int xc_partition_weights(const xc_atom* atoms /*[host]*/, int32_t natoms, int32_t partition, int64_t npts,
                         const double* dx, const double* dy, const double* dz, const double* dwq,
                         const int32_t* dparent, double* dw_out, void* cuda_stream);
int xc_functional(int32_t functional, int64_t n, const double* drho, const double* dsigma, double rho_tol,
                  double* df, double* dvrho, double* dvsigma, void* cuda_stream);

/* The spin-coupling step of the spin-unrestricted build (Alg. 4 l.4.6-4.7 per spin; DESIGN.md readings
 * A20-A21) as a call that ALLOCATES NOTHING -- for callers that cannot call cudaMalloc (code under CUDA graph capture,
 * serving loops, harnesses that forbid it).  It is the kernel pair xc_eval_uks runs between its density and potential
 * passes; the per-block partial sums go to a file-scope device array of the library instead of a plan's buffer.
 *   functional  0 = Slater+VWN5, 1 = PBE (spin-polarised);  npts <= XC_STATIC_MAX_POINTS, else XC_EUNSUPPORTED
 *   d_w    [device] npts           partition weights w_i (points with w_i = 0 are skipped: their densities are not read)
 *   d_rho  [device] 2 x npts       rho_a | rho_b (spin-major);  d_grho [device] 2 x npts x 3  grad rho_s (PBE; may be NULL for 0)
 *   rho_tol > 0                    as xc_grid_spec.rho_tol of a spin-unrestricted build
 *   d_cA   [device] 2 x npts  out  a_s = w v_rho_s (LDA) | 1/2 w v_rho_s (PBE): coefficient of Phi in Z^s, Eq. (20)
 *   d_cG   [device] 2 x npts x 3 out  g_s = w (2 v_ss grad rho_s + v_ab grad rho_s') (PBE; may be NULL for 0)
 *   d_out3 [device] 3         out  E_xc, N_a, N_b (Eq. (16)), summed in a fixed order: bit-identical from call to call
 * All pointers are device pointers of the CURRENT device, owned by the caller; the call is stream-ordered on cuda_stream
 * and returns without synchronising.  The static array (768 KB) exists once per GPU that loads the library and is held until
 * the process exits; every call on a GPU shares it and it keeps the last call's contents (nothing in it needs to start
 * at zero: a call overwrites the partials it then reads).  Calls that OVERLAP on one GPU (two streams, two threads) race
 * on it: serialise them.  No cudaMalloc, cudaFree or allocating library routine is called.
 * Errors: XC_EINVAL (enum, null, npts < 0, rho_tol <= 0), XC_EUNSUPPORTED (npts beyond the maximum), XC_ECUDA. */
#define XC_STATIC_MAX_POINTS 8388608
int xc_functional_uks_static(int32_t functional, int64_t npts, const double* d_w, const double* d_rho, const double* d_grho,
                             double rho_tol, double* d_cA, double* d_cG, double* d_out3, void* cuda_stream);

/* FP64 pipe microbenchmark of `device` (no memory traffic, register-resident chains; CUDA events, best of `reps`
 * launches): kind 0 = DFMA chains, 1 = DMMA (mma.sync m8n8k4 f64, the instruction of the batch kernel's contractions).
 * MEASURED_PEAKS.json has no FP64 entry, so bench.py measures the denominator of the FP64 roofline with this call
 * (SURVEY.md 8(d) "FP64 peak ... must be measured on the box").  tflops [host] out; sm_clock_mhz_est [host, may be
 * NULL] = the SM clock implied by 64 FP64 FMA/clk/SM.  Errors: XC_EINVAL, XC_ECUDA, XC_ENOMEM. */
int xc_measure_fp64_peak(int32_t kind, int32_t device, int32_t reps, double* tflops, double* sm_clock_mhz_est);

const char* xc_strerror(int code);
const char* xc_last_error(void);

#ifdef __cplusplus
}
#endif
#endif /* XC_B200_H */
