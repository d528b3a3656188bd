// plan.hpp -- the opaque msm_plan: host mathematics + every device buffer of one MSM setup.
#pragma once
#include <cuda_runtime.h>

#include <string>
#include <vector>

#include "../../include/msm.h"
#include "anterp_tiled.cuh"
#include "conv.cuh"
#include "plan_math.hpp"

namespace msm {

constexpr int kMaxStages = 2 * MSM_MAX_LEVELS + 16;   // sort pair anterpolate restrict {filter,conv}_l* top ...

// one tap table of a level and, per stored value, what it is: (dx, dy, dz, kind) with kind
// 0 = padding zero, 1 = s_l, 2 = 2g, 3 = 2g dx, 4 = 2g dx^2 (g = k_l'(r)/r): msm_plan_set_box
// recomputes the values on the device from these descriptors
struct TapTable {
  void* values = nullptr;
  int4* desc = nullptr;
  int n = 0;
};

struct LevelDev {
  void *Q = nullptr, *E = nullptr, *pad = nullptr;   // grid charge, potential, haloed filtered charge
  void* scratch = nullptr;                           // slice partials of the convolution (nslices > 1)
  int taps = 0;
  TapTable tab[4];                                   // staps, taps2 (with its guard chunk), vtaps, vtaps2
  double hstruct[3] = {0, 0, 0};                     // spacings the table structure was sized for
};

// arguments of one msm_evaluate: a captured CUDA graph is replayed only for an identical call
struct GraphKey {
  int n = -1;
  const void *pos = nullptr, *q = nullptr;
  void *F = nullptr, *V = nullptr;
  bool virial = false, profiling = false;
  bool operator==(const GraphKey& o) const {
    return n == o.n && pos == o.pos && q == o.q && F == o.F && V == o.V && virial == o.virial && profiling == o.profiling;
  }
};

// makes the plan's device current for the duration of an entry point and restores the caller's
struct DeviceGuard {
  int prev = -1;
  bool ok = false;
  explicit DeviceGuard(int dev) {
    if (cudaGetDevice(&prev) != cudaSuccess) prev = -1;
    ok = cudaSetDevice(dev) == cudaSuccess;
  }
  ~DeviceGuard() { if (prev >= 0) cudaSetDevice(prev); }
};

}  // namespace msm

struct msm_plan {
  msm_params_t prm{};
  msm::Params mp{};
  msm::Hierarchy* H = nullptr;
  msm::Splitting* S = nullptr;
  int P = 4, n_t = 1, mu = 4, w = 0;
  bool fp32 = false;
  size_t esz = 8;
  std::vector<double> J, omega;
  msm::SplinePieces* pieces = nullptr;

  double reserve = 0.0;      // fraction by which msm_plan_set_box may shrink a periodic box edge
  std::vector<void*> allocs;
  size_t bytes = 0;
  int sm_count = 148;        // cudaDevAttrMultiProcessorCount of the plan's device (148 on B200)

  msm::LevelDev lev[MSM_MAX_LEVELS + 1];
  void *tmpA = nullptr, *tmpB = nullptr;
  msm::ConvTable conv{};                             // host copy; conv.lev[l - 1] is level l
  msm::ConvTable* d_conv = nullptr;
  size_t conv_smem = 0;
  int conv_ny_max = 0, conv_maxc = 0;   // largest row count 2 R_y + 1 and chunks per stencil row over the levels
  bool in_batch = false;                             // one of the plans of an msm_batch
  bool top_beside = true;                            // small jobs: the top-level operator runs beside the convolution (not in a batch)
  long long conv_tiles_total = 0;                    // output tiles of all tiled levels
  bool conv_rowsliced = false;                       // some level splits its plane slices by stencil rows (small jobs: no list kernels)
  bool conv_lists = true;                            // fp32: every level has the entry lists of k_conv_f2l
  size_t conv_dtables_smem = 0;                      // fp64: largest 4-tap chunk table of a level (bytes)
  size_t conv_vtables_smem = 0;                      // fp32: largest interleaved virial tap table of a level (bytes)
  size_t conv_tables_smem = 0;                       // fp32: largest row + tap table of a level (bytes)
  int conv_slices = 1, conv_vslices = 1;             // input-plane slices per output tile (potential, virial kernel)
  double* conv_wpart = nullptr;                      // total_vunits x 6

  // tiled anterpolation (anterp_tiled.cuh); false: gather kernel
  bool anterp_tiled = false;
  msm::AnterpTiles at{};
  void* anterp_scratch = nullptr;

  // top operator
  int G = 0;
  void *topT = nullptr, *topTD = nullptr;
  double* top_wrow = nullptr;

  // particles
  int cap = 0;
  msm::BinGeom bg{};
  int n_pcells = 0, n_gcells = 0, pair_rows = 0, pair_ymax = 1, pair_blocks = 0, pair_nsplit = 1;
  int* ibuf = nullptr;          // [phist(n_pcells) | ghist(n_gcells) | flag]: zeroed per call
  size_t ibuf_count = 0;
  int *phist = nullptr, *ghist = nullptr, *flag = nullptr;
  int *pstart = nullptr, *gstart = nullptr, *ptotals = nullptr, *gtotals = nullptr;
  int *pslot = nullptr, *gslot = nullptr;
  int *pcell = nullptr, *gcell = nullptr, *porder = nullptr, *gorder = nullptr, *pcellx = nullptr,
      *gcell_sorted = nullptr;
  void *prec = nullptr, *grec = nullptr, *Fsr = nullptr, *Vsr = nullptr;
  double *pair_wpart = nullptr, *epart = nullptr, *results = nullptr;
  int n_eblocks = 0;
  double* part = nullptr;       // block partials of the final reductions, part_blocks x 7
  int part_blocks = 0;
  double* h_results = nullptr;  // pinned: U, W[6], flag
  // staging for msm_evaluate_host
  void *in_pos = nullptr, *in_q = nullptr, *out_F = nullptr, *out_V = nullptr;

  // CUDA graph of the launch sequence (msm_evaluate.cu: run)
  bool graph_enabled = true;
  msm::GraphKey gkey{};
  cudaStream_t gstream = nullptr;
  cudaGraphExec_t gexec = nullptr;
  cudaEvent_t gev = nullptr;
  // completion of the last enqueued evaluation (msm_get_results waits on it)
  cudaEvent_t done_ev = nullptr;
  bool pending = false, pending_virial = false;

  // fine grids with at least this many points take the one-sweep restriction / prolongation
  // kernels of gridops_stream.cuh (the restriction only pays when the grid does not fit the L2;
  // the prolongation measured faster at every size); MSM_GRID_STREAM_MIN sets both
  long long stream_min_points = 1ll << 22, prolong_stream_min_points = 0, filter_stream_min_points = 1ll << 22;

  // second stream for the pair kernel (runs beside the grid pipeline)
  bool overlap = true;
  cudaStream_t pstream = nullptr, vstream = nullptr;
  cudaEvent_t fork_ev = nullptr, join_ev = nullptr, fork2_ev = nullptr, join2_ev = nullptr, top_ev = nullptr;

  // profiling
  bool profiling = false;
  cudaEvent_t ev[msm::kMaxStages + 1]{};
  float stage_ms[msm::kMaxStages]{};
  int n_stages = 0;                               // stages of the last evaluate
  std::vector<std::string> stage_name_store;      // fixed at plan creation (same order every call)
  std::vector<const char*> stage_names;
  int launches = 0;
};

namespace msm {
msm_status_t plan_create_opts(const msm_params_t* params, double reserve, bool in_batch, msm_plan_t** plan_out);
}
