// xc_internal.h -- structures shared by the host planner and the CUDA kernels of libxc_b200.
// (Product code.  Shares nothing with oracle/.)
#pragma once
#include <cstdint>
#include <string>
#include <utility>
#include <vector>

#include "../../include/xc_b200.h"

namespace xcb {

constexpr int kMaxL = 2;
constexpr int kMaxPrim = 16;
constexpr int kBatchThreads = 512;  // 16 warps per batch CTA
constexpr int kSmallNb = 112;   // N_b^j limit of the 64-point-tile instantiation (<= 28 lower-triangle 16x16 blocks = 2 per warp of 16)
constexpr int kMidNb = 144;     // class 1 batches up to here (<= 45 blocks) run the three-round instantiation: its accumulators stay in registers
constexpr int kMaxNb = 192;     // N_b^j limit of the batch kernel (<= 78 blocks = 5 per warp); the planner splits larger batches
constexpr size_t kSmemLimit = 227 * 1024;
constexpr size_t kBatchStaticSmem = 2048;   // static shared memory of k_xc_batch (live-point list, counters, ring barriers), rounded up
constexpr int kRingStages = 2;              // P^j staging ring of k_xc_batch: slots ...
constexpr int kRingGMax = 16;                // ... of at most this many k-steps each (256 B per mu-tile and k-step)
constexpr int kWeightThreads = 256;  // Becke-88 weights kernel: 8 warps per batch CTA
constexpr int kWeightSmallList = 256; // SSF weights kernel: atom-list length that separates its two launches

struct ShellRec {      // 48 bytes
  double x, y, z;      // centre
  int32_t L, nprim, prim_off, func_off;  // L: shell type (nfun); func_off: first GLOBAL function index
  int32_t atom, _pad;
};

struct BatchRec {      // one quadrature batch B_j with its shell list S_j
  int32_t pt_off, nq;          // first point (plan order), N_q^j
  int32_t sh_off, ns;          // offset into batch shell list, |S_j| in shells
  int32_t f_off, nb;           // offset into batch function-index list, N_b^j
  int64_t ppk_off;             // offset (doubles) of this batch's packed P^j (nb4 x nb8, DMMA fragment order)
  int64_t wa_off;              // offset into the weight-kernel atom lists
  int32_t wa_nB, wa_nC;        // atoms that can own weight here / atoms that can appear in a cell product
  int32_t ntriv, ring_g;       // ring_g: k-steps per stage of the P^j staging ring this batch can afford (xc_kernels.cu); SSF: the first ntriv points of the batch have w = w^q exactly (r_A < (1-a)/2 R_nn(A))
};



// ShellRec::L holds a shell TYPE: 0 = s, 1 = p, 2 = Cartesian d, 3 = pure d (XC_SHELL_PURE; reading A19)
constexpr int kPureD = 3;
inline int nfun(int type) { return type == kPureD ? 5 : (type + 1) * (type + 2) / 2; }
inline int64_t round_up(int64_t a, int64_t b) { return (a + b - 1) / b * b; }

// shared-memory footprint of the batch kernel for a batch (bytes); T = points per tile
size_t batch_smem_bytes(int T, bool gga, int nb, int ns, int npr, int nthreads, int ring_g);   // npr: primitives of the batch's shells
int batch_ring_g(size_t bytes_without_ring, int nb);   // k-steps per ring stage that fit beside it (0: none)
size_t weights_smem_bytes(int nC, int warps);
// atom list of the weights kernels for the box [lo, hi] of points: owners = out[0 .. nB), partners = all of out (sorted by distance to the box)
void weight_atom_list(const double* atoms, int natoms, const double lo[3], const double hi[3], bool ssf, std::vector<int32_t>& out, int& nB);

// permuted point arrays made on the device by the GPU planner (plan order); owned by whoever holds the struct
struct DevicePoints {
  double *px = nullptr, *py = nullptr, *pz = nullptr, *wq = nullptr;
  int32_t* parent = nullptr;
  int64_t* orig = nullptr;
};

struct HostPlan {
  int natoms = 0, nshells = 0, nbasis = 0, nprim = 0;
  xc_grid_spec spec{};
  int64_t npts = 0;
  std::vector<double> atoms;           // natoms*3
  std::vector<ShellRec> shells;
  std::vector<double> exps, coefs, rcut;
  DevicePoints dev;                    // GPU-made plans: the point arrays live here, and px..orig below stay empty
  std::vector<double> px, py, pz, wq;  // plan order (host-made plans)
  std::vector<int32_t> parent;
  std::vector<int64_t> orig;
  std::vector<BatchRec> batches;
  std::vector<int32_t> bshells;        // concatenated S_j (global shell ids, ascending)
  std::vector<int32_t> bsfoff;         // per entry of bshells: first LOCAL function index of that shell in its batch
  std::vector<int32_t> bfidx;          // concatenated global function indices of S_j
  std::vector<int32_t> watoms;         // concatenated per-batch atom lists of the weights kernel (sorted by distance to the batch box)
  std::vector<double> wbox;            // [nbatch][6] tight bounding boxes
  std::vector<int32_t> wbatch_small, wbatch_large;  // SSF weights kernel: batches with non-trivial points, by list length (two launches)
  int w_max_small = 0, w_max_large = 0;
  std::vector<double> rnn;             // nearest-neighbour distance of every atom
  int w_max_list = 0, w_warps = 8;     // Becke-88 weights kernel: longest atom list, warps per CTA that fit in shared memory
  std::vector<int32_t> ids_small, ids_large;  // batch-kernel work lists (N_b^j <= kSmallNb / the others), heaviest first
  int64_t ppk_doubles = 0;              // size of the packed-P^j buffer
  double sum_nbnq = 0, sum_nb2 = 0, flops = 0;
  int max_nb = 0, max_ns = 0;
  int n_heavy = 0;             // the first n_heavy entries of ids_large have N_b^j > kMidNb (five-round instantiation)
  size_t smem_small = 0, smem_large = 0;  // max dynamic smem over each work list
};

// Builds grid, batches, screening, work lists.  Returns XC_OK or an error code (message in err).
// device >= 0: the grid and the bisection run on that GPU (xc_gpu_planner.cu; the plan is identical either way)
int build_host_plan(const xc_atom* atoms, int natoms, const xc_shell* shells, int nshells, const double* exps,
                    const double* coefs, int nprim_total, const xc_grid_spec* spec, int device, HostPlan& hp, std::string& err);
// step (b) on the GPU (xc_gpu_planner.cu): begin = grid points + global median bisection, returns the cuboids and their tight
// bounding boxes (lo xyz, hi xyz per cuboid); order = Morton order inside the cuboids, SSF-trivial points first, permuted point
// arrays; download = hand the points and the order so far to the host (it finishes alone when a batch has to be split again)
struct GpuPlanner;
int gpu_planner_begin(int device, int natoms, const double* atoms, int n_rad, int n_ang, const double* rr, const double* au, int maxp,
                      GpuPlanner** out, std::vector<std::pair<int64_t, int64_t>>& leaves, std::vector<double>& boxes, std::string& err);
int gpu_planner_download(GpuPlanner* g, std::vector<double>& cx, std::vector<double>& cy, std::vector<double>& cz, std::vector<int64_t>& idx,
                         std::string& err);
int gpu_planner_order(GpuPlanner* g, bool ssf, const double* rnn, double lim, const double* rw, int n_rad, const double* aw,
                      DevicePoints& out, std::vector<int32_t>& ntriv, std::string& err);
void gpu_planner_end(GpuPlanner* g);

}  // namespace xcb
