// msm_evaluate.cu -- msm_evaluate: enqueues the whole hot path (S1..S9 of DESIGN.md) on one stream.
#include <algorithm>
#include <cstdlib>
#include <cstring>

#include "gridops.cuh"
#include "gridops_fused.cuh"
#include "gridops_stream.cuh"
#include "gridops_filter_stream.cuh"
#include "pair.cuh"
#include "particle_grid.cuh"
#include "plan.hpp"
#include "sort.cuh"

using namespace msm;

namespace {

struct Seg {
  const double* ptr;
  int count;      // rows of 6 doubles (width 6) or single doubles (width 1: energy partials)
  int width;
  int blk0;       // first block of this segment in k_partial_sums
  double scale[6];
};
constexpr int kMaxSegs = MSM_MAX_LEVELS + 4;
constexpr int kRowsPerBlock = 1024;
struct FinalizeArgs {
  int nseg, nblk;
  Seg seg[kMaxSegs];
};

// S9, stage 1: every block sums kRowsPerBlock rows of one segment (thread t takes rows t, t+256,
// ... then a fixed-order block reduction) into part[block][0..5] (scaled virial) / part[block][6]
// (energy). Stage 2 (k_finalize, one block) adds the block partials in block order. Both orders are
// fixed -> deterministic.
__global__ void __launch_bounds__(256) k_partial_sums(FinalizeArgs a, double* __restrict__ part) {
  __shared__ double red[8];
  int s = 0;
  for (int k = 1; k < a.nseg; ++k)
    if ((int)blockIdx.x >= a.seg[k].blk0) s = k;
  const Seg& sg = a.seg[s];
  const int r0 = ((int)blockIdx.x - sg.blk0) * kRowsPerBlock, r1 = min(r0 + kRowsPerBlock, sg.count);
  double v[6] = {0, 0, 0, 0, 0, 0};
  if (sg.width == 6) {
    for (int i = r0 + threadIdx.x; i < r1; i += 256)
#pragma unroll
      for (int k = 0; k < 6; ++k) v[k] += sg.ptr[(size_t)i * 6 + k];
  } else {
    for (int i = r0 + threadIdx.x; i < r1; i += 256) v[0] += sg.ptr[i];
  }
#pragma unroll
  for (int k = 0; k < 6; ++k) {
    const double r = block_reduce_sum<256>(v[k], red);
    if (threadIdx.x == 0) {
      if (sg.width == 6) part[(size_t)blockIdx.x * 7 + k] = sg.scale[k] * r;
      else if (k == 0) part[(size_t)blockIdx.x * 7 + 6] = r;
    }
  }
  if (threadIdx.x == 0) {
    if (sg.width == 6) part[(size_t)blockIdx.x * 7 + 6] = 0.0;
    else
      for (int k = 0; k < 6; ++k) part[(size_t)blockIdx.x * 7 + k] = 0.0;
  }
}

__global__ void __launch_bounds__(256) k_finalize(int nblk, const double* __restrict__ part,
                                                  const int* __restrict__ flag, double* __restrict__ results) {
  __shared__ double red[8];
  for (int k = 0; k < 7; ++k) {
    double w = 0.0;
    for (int i = threadIdx.x; i < nblk; i += 256) w += part[(size_t)i * 7 + k];
    w = block_reduce_sum<256>(w, red);
    if (threadIdx.x == 0) results[k == 6 ? 0 : 1 + k] = w;
  }
  if (threadIdx.x == 0) results[7] = (double)(*flag);
}

inline unsigned blocks_for(size_t n, int bs) { return (unsigned)std::max<size_t>(1, (n + bs - 1) / bs); }

template <typename T> AxisTaps<T> make_taps(const std::vector<double>& v) {
  AxisTaps<T> t;
  t.n = (int)v.size();
  for (int i = 0; i < t.n; ++i) t.c[i] = (T)v[i];
  return t;
}

template <typename T, int P> SplineTab<T, P> make_tab(const SplinePieces& sp) {
  SplineTab<T, P> t;
  for (int j = 0; j < P; ++j)
    for (int k = 0; k < P; ++k) { t.c[j][k] = (T)sp.coef[j][k]; t.d[j][k] = (T)sp.dcoef[j][k]; }
  return t;
}

#define MSM_LAUNCH(plan, ...) do { __VA_ARGS__; ++(plan)->launches; } while (0)

template <typename T, int P>
msm_status_t enqueue_t(msm_plan* p, int n, const void* d_pos, const void* d_q, void* d_F, void* d_V,
                       bool want_virial, cudaStream_t st, bool capturing) {
  using V4 = typename Vec4<T>::type;
  const Hierarchy& H = *p->H;
  const T* pos = (const T*)d_pos;
  const T* q = (const T*)d_q;
  int evi = 0;
  // stage events; inside a stream capture they become external event-record nodes of the graph
  auto mark = [&]() {
    if (p->profiling) {
      if (capturing) cudaEventRecordWithFlags(p->ev[evi], st, cudaEventRecordExternal);
      else cudaEventRecord(p->ev[evi], st);
    }
    ++evi;
  };
  p->launches = 0;
  mark();

  // ---------------- S1 sort
  cudaMemsetAsync(p->ibuf, 0, p->ibuf_count * sizeof(int), st);
  MSM_LAUNCH(p, (k_bin<T><<<blocks_for(n, 256), 256, 0, st>>>(n, pos, p->bg, p->pcell, p->gcell, p->phist,
                                                               p->ghist, p->pslot, p->gslot, p->flag)));
  if (p->n_pcells <= kScanSerialMax && p->n_gcells <= kScanSerialMax) {
    MSM_LAUNCH(p, (k_scan_serial2<<<2, kScanThreads, 0, st>>>(p->n_pcells, p->phist, p->pstart, p->n_gcells, p->ghist,
                                                                p->gstart, n)));
  } else {
    const int tp = (p->n_pcells + kScanTile - 1) / kScanTile, tg = (p->n_gcells + kScanTile - 1) / kScanTile;
    MSM_LAUNCH(p, (k_scan_tiles<<<tp, kScanThreads, 0, st>>>(p->n_pcells, p->phist, p->pstart, p->ptotals)));
    MSM_LAUNCH(p, (k_scan_tiles<<<tg, kScanThreads, 0, st>>>(p->n_gcells, p->ghist, p->gstart, p->gtotals)));
    MSM_LAUNCH(p, (k_scan_totals<<<1, kScanThreads, 0, st>>>(tp, p->ptotals)));
    MSM_LAUNCH(p, (k_scan_totals<<<1, kScanThreads, 0, st>>>(tg, p->gtotals)));
    MSM_LAUNCH(p, (k_scan_add<<<blocks_for(p->n_pcells, 256), 256, 0, st>>>(p->n_pcells, p->pstart, p->ptotals, n)));
    MSM_LAUNCH(p, (k_scan_add<<<blocks_for(p->n_gcells, 256), 256, 0, st>>>(p->n_gcells, p->gstart, p->gtotals, n)));
  }
  MSM_LAUNCH(p, (k_scatter<<<blocks_for(n, 256), 256, 0, st>>>(n, p->pcell, p->gcell, p->pstart, p->gstart,
                                                                 p->pslot, p->gslot, p->porder, p->gorder)));
  MSM_LAUNCH(p, (k_sort_cells<<<dim3(blocks_for(std::max(p->n_pcells, p->n_gcells), 128), 2), 128, 0, st>>>(
                    p->n_pcells, p->pstart, p->porder, p->pslot, p->n_gcells, p->gstart, p->gorder, p->gslot)));
  MSM_LAUNCH(p, (k_build_records<T><<<blocks_for(n, 256), 256, 0, st>>>(
                    n, pos, q, p->bg, p->porder, p->pcell, p->gorder, p->gcell, (V4*)p->prec, (V4*)p->grec,
                    p->gcell_sorted, p->pcellx)));
  mark();

  // ---------------- S2 pair
  bool forked = false, forked_v = false;
  {
    PairParams<T> pp;
    bool any_minimg = false;
    for (int ax = 0; ax < 3; ++ax) {
      pp.nc[ax] = p->bg.nc[ax];
      pp.periodic[ax] = p->bg.periodic[ax];
      pp.minimg[ax] = (p->bg.periodic[ax] && p->bg.nc[ax] < 5) ? 1 : 0;
      pp.omin[ax] = -2;
      pp.omax[ax] = pp.minimg[ax] ? std::min(2, p->bg.nc[ax] - 3) : 2;   // nc distinct cells
      if (pp.minimg[ax]) { pp.omin[ax] = -std::min(2, p->bg.nc[ax] - 1 - pp.omax[ax]); }
      any_minimg |= pp.minimg[ax] != 0;
      pp.edge[ax] = (T)p->bg.cell_edge[ax];
      pp.box[ax] = (T)p->bg.box[ax];
      pp.inv_box[ax] = (T)(1.0 / p->bg.box[ax]);
    }
    (void)any_minimg;
    const double a = p->mp.a;
    // x windows per row class: a row |dy| cells away starts max(|dy| - 1, 0) cell edges away, so the
    // cutoff sphere reaches sqrt(a^2 - gy^2 - gz^2) along x there (rounded up to whole sub-bins)
    pp.sxs = p->bg.sxs;
    for (int ax = 0; ax < 3; ++ax) pp.edge_d[ax] = p->bg.cell_edge[ax];
    for (int iy = 0; iy < 3; ++iy)
      for (int iz = 0; iz < 3; ++iz) {
        const double gy = std::max(iy - 1, 0) * p->bg.cell_edge[1], gz = std::max(iz - 1, 0) * p->bg.cell_edge[2];
        const double rem = a * a - gy * gy - gz * gz;
        const double sub = p->bg.cell_edge[0] / (double)(1 << p->bg.sxs);
        pp.wb[iy][iz] = rem > 0.0 ? (int)std::ceil(std::sqrt(rem) * (1.0 + 1e-9) / sub) : -1;
      }
    // fp32 scan: exact cutoff in fp32 mode (the drain repeats the same arithmetic); in fp64 mode a
    // slack of 1e-4 relative covers the rounding of cell-relative coordinates (< 2^-24 * 8 edges)
    pp.a2_scan = sizeof(T) == 4 ? (float)(a * a) : (float)(a * a * (1.0 + 1e-4));
    pp.a = (T)a; pp.a2 = (T)(a * a); pp.inv_a = (T)(1.0 / a); pp.inv_a2 = (T)(1.0 / (a * a)); pp.two_inv_a3 = (T)(2.0 / (a * a * a));
    for (int k = 0; k < 8; ++k) pp.c[k] = (T)p->S->c[k];
    pp.p = P;
    // clusters of kPairCluster particles per cell row, spread over gridDim.y blocks of kPairWarps warps
    constexpr int kPairWarps = PairWarps<T>::value;
    const int per_row = (n / kPairCluster + p->pair_rows) / p->pair_rows;
    // few tiles (small systems): deal the dz planes of the neighbourhood to separate blocks
    const int nplanes = pp.omax[2] - pp.omin[2] + 1;
    // fewer clusters than ~16 warps per SM: deal the dz planes to separate blocks
    pp.nsplit = n / kPairCluster < p->sm_count * 16 ? std::min(nplanes, kPairMaxSplit) : 1;
    pp.part_stride = (size_t)p->cap;
    p->pair_nsplit = pp.nsplit;
    const dim3 pgrid(p->pair_rows, std::max(1, std::min(p->pair_ymax, (per_row + kPairWarps - 1) / kPairWarps)),
                     pp.nsplit);
    p->pair_blocks = (int)(pgrid.x * pgrid.y * pgrid.z);
    const bool mi = pp.minimg[0] || pp.minimg[1] || pp.minimg[2];
    // The pair sum does not depend on the grid pipeline (S3..S7): it runs on the plan's second
    // stream beside it and joins before the interpolation, so that the two latency-bound halves of
    // the evaluation fill each other's idle issue slots. With per-stage profiling on, everything
    // stays on one stream (the stage times would otherwise overlap).
    cudaStream_t ps = st;
    if (p->overlap && !p->profiling && p->pstream) {
      cudaEventRecord(p->fork_ev, st);
      cudaStreamWaitEvent(p->pstream, p->fork_ev, 0);
      ps = p->pstream;
    }
#define MSM_PAIR(V, M) MSM_LAUNCH(p, (k_pair<T, P, V, M><<<pgrid, kPairWarps * 32, 0, ps>>>(           \
    pp, p->pstart, (const V4*)p->prec, p->pcellx, p->porder, (T*)p->Fsr, (T*)p->Vsr, p->pair_wpart)))
    if (want_virial) { if (mi) MSM_PAIR(true, true); else MSM_PAIR(true, false); }
    else { if (mi) MSM_PAIR(false, true); else MSM_PAIR(false, false); }
#undef MSM_PAIR
    if (ps != st) cudaEventRecord(p->join_ev, ps);
    forked = ps != st;
  }
  mark();

  // ---------------- S3 anterpolation
  GridGeom gg;
  for (int ax = 0; ax < 3; ++ax) {
    gg.M[ax] = H.lev[1].M[ax]; gg.lo[ax] = H.lev[1].lo[ax]; gg.ng[ax] = p->bg.ng[ax];
    gg.periodic[ax] = p->bg.periodic[ax];
  }
  const SplineTab<T, P> tab = make_tab<T, P>(*p->pieces);
  if (p->anterp_tiled) {
    const int D3 = p->at.D[0] * p->at.D[1] * p->at.D[2];
    const size_t sm = anterp_smem_bytes<T, P>(D3);
    const int ntiles = p->at.nt[0] * p->at.nt[1] * p->at.nt[2] * p->at.split;
    MSM_LAUNCH(p, (k_anterp_tiles<T, P><<<ntiles, 32, sm, st>>>(gg, p->at, tab, p->gstart, (const V4*)p->grec,
                                                                 p->gcell_sorted, (T*)p->anterp_scratch)));
    const dim3 cgrid((H.lev[1].M[0] + 31) / 32, (H.lev[1].M[1] + 3) / 4, H.lev[1].M[2]), cblock(32, 4);
    if (p->at.split > 1)
      MSM_LAUNCH(p, (k_anterp_combine<T, P, true><<<cgrid, cblock, 0, st>>>(gg, p->at, (const T*)p->anterp_scratch, (T*)p->lev[1].Q)));
    else
      MSM_LAUNCH(p, (k_anterp_combine<T, P, false><<<cgrid, cblock, 0, st>>>(gg, p->at, (const T*)p->anterp_scratch, (T*)p->lev[1].Q)));
  } else {
    // lanes per node: 16; 1 in a batch (64 x 512 particles: 0.91 against 1.00 ms per batch with 16)
    const int lg = p->in_batch ? 0 : 4;
    MSM_LAUNCH(p, (k_anterpolate<T, P><<<blocks_for(H.lev[1].points() << lg, 128), 128, 0, st>>>(
                      gg, tab, p->gstart, (const V4*)p->grec, (T*)p->lev[1].Q, lg)));
  }
  mark();

  // ---------------- S4 restriction
  const AxisTaps<T> Jt = make_taps<T>(p->J), Wt = make_taps<T>(p->omega);
  auto grid3 = [](const Level& lv) {
    Grid3 g;
    for (int ax = 0; ax < 3; ++ax) { g.M[ax] = lv.M[ax]; g.lo[ax] = lv.lo[ax]; }
    return g;
  };
  const int per3[3] = {p->bg.periodic[0], p->bg.periodic[1], p->bg.periodic[2]};
  // one-sweep kernels: x periodic (lo = 0, whole 16-byte chunks), grid too large for the L2
  auto stream_ok = [&](const Level& f, const Level& c, long long min_points) {
    constexpr int VE = VecT<T>::VE;
    return per3[0] && f.lo[0] == 0 && c.lo[0] == 0 && f.M[0] % (2 * VE) == 0 && c.M[0] * 2 == f.M[0] &&
           (long long)f.points() >= min_points;
  };
  auto stream_geom = [&](const Level& f, const Level& c) {
    StreamGeom sg;
    sg.f = grid3(f); sg.c = grid3(c);
    sg.per_y = per3[1]; sg.per_z = per3[2];
    sg.ntx = 1; sg.zseg = 1;
    return sg;
  };
  // planes per block along the marching axis: enough blocks for ~8 per SM, at least min_planes each
  auto stream_zseg = [&](int columns, int nplanes, int min_planes) {
    const int want = std::max(1, (p->sm_count * 8 + columns - 1) / columns);
    return std::max(std::min(min_planes, nplanes), (nplanes + want - 1) / want);
  };
  for (int l = 1; l < p->n_t; ++l) {
    const Level &f = H.lev[l], &c = H.lev[l + 1];
    const T* src = (const T*)p->lev[l].Q;
    if (stream_ok(f, c, p->stream_min_points)) {
      // large grid: one sweep over the fine grid (gridops_stream.cuh)
      constexpr int CY = 8;
      StreamGeom sg = stream_geom(f, c);
      const int cx = restrict_stream_cx<T, P + 1>();
      sg.ntx = (c.M[0] + cx - 1) / cx;
      const int nty = (c.M[1] + CY - 1) / CY;
      sg.zseg = stream_zseg(sg.ntx * nty, c.M[2], 8);
      const dim3 grid(sg.ntx * nty, (c.M[2] + sg.zseg - 1) / sg.zseg);
      MSM_LAUNCH(p, (k_restrict_stream<T, P + 1, CY><<<grid, kStreamThreads, 0, st>>>(sg, Jt, src, (T*)p->lev[l + 1].Q)));
      continue;
    }
    int din[3] = {f.M[0], f.M[1], f.M[2]};
    for (int ax = 0; ax < 3; ++ax) {
      AxisDims d;
      for (int k = 0; k < 3; ++k) { d.in[k] = din[k]; d.out[k] = din[k]; }
      d.out[ax] = c.M[ax];
      d.axis = ax; d.periodic = p->bg.periodic[ax];
      T* dst = ax == 2 ? (T*)p->lev[l + 1].Q : (T*)(ax == 0 ? p->tmpA : p->tmpB);
      // (a periodic axis that is already down to one point is copied: only the generic kernel does that)
      if (d.periodic && f.M[ax] == 1) {
        if (ax == 0) MSM_LAUNCH(p, (k_restrict_axis<T, 0><<<axis_grid(d), axis_block(), 0, st>>>(d, f.lo[ax], c.lo[ax], Jt, src, dst)));
        else if (ax == 1) MSM_LAUNCH(p, (k_restrict_axis<T, 1><<<axis_grid(d), axis_block(), 0, st>>>(d, f.lo[ax], c.lo[ax], Jt, src, dst)));
        else MSM_LAUNCH(p, (k_restrict_axis<T, 2><<<axis_grid(d), axis_block(), 0, st>>>(d, f.lo[ax], c.lo[ax], Jt, src, dst)));
      } else {
        const unsigned rg = filter_run_grid(d);
        if (ax == 0) MSM_LAUNCH(p, (k_restrict_axis_run<T, 0, P + 1><<<rg, axis_block(), 0, st>>>(d, f.lo[ax], c.lo[ax], Jt, src, dst)));
        else if (ax == 1) MSM_LAUNCH(p, (k_restrict_axis_run<T, 1, P + 1><<<rg, axis_block(), 0, st>>>(d, f.lo[ax], c.lo[ax], Jt, src, dst)));
        else MSM_LAUNCH(p, (k_restrict_axis_run<T, 2, P + 1><<<rg, axis_block(), 0, st>>>(d, f.lo[ax], c.lo[ax], Jt, src, dst)));
      }
      src = dst;
      din[ax] = c.M[ax];
    }
  }
  mark();

  // ---------------- S5 convolution on the tiled levels
  int nseg = 0;
  FinalizeArgs fa;
  for (int l = 1; l < p->n_t; ++l) {
    LevelDev& d = p->lev[l];
    const ConvLevel& g = p->conv.lev[l - 1];
    const Level& lv = H.lev[l];
    // omega' filter + halo, x then y then z
    const T* src = (const T*)d.Q;
    int din[3] = {lv.M[0], lv.M[1], lv.M[2]};
    const int halo[3] = {g.X0, g.R[1], g.R[2]};
    {
      // large grid: one sweep (gridops_filter_stream.cuh)
      constexpr int VE = VecT<T>::VE;
      const bool shape_ok = lv.M[0] % VE == 0 && g.P[0] % VE == 0 && g.X0 % VE == 0 &&
                            (Wt.n == 11 || Wt.n == 13 || Wt.n == 15);
      if (shape_ok && (long long)lv.points() >= p->filter_stream_min_points) {
        FilterGeom fg;
        for (int k = 0; k < 3; ++k) { fg.M[k] = lv.M[k]; fg.P[k] = g.P[k]; fg.H[k] = halo[k]; fg.per[k] = p->bg.periodic[k]; }
        fg.ntx = (g.P[0] / VE + kFilterTXC - 1) / kFilterTXC;
        FilterTaps2 w2;
        auto tap = [&](int k) { return k >= 0 && k < Wt.n ? (float)Wt.c[k] : 0.f; };
        for (int k = 0; k < 15; ++k) w2.c[k] = make_float2(tap(k), tap(k));
        for (int k = 0; k < 16; ++k) w2.x[k] = make_float2(tap(k - 1), tap(k));
        // segments of planes: full waves of resident blocks against the 2 HW extra planes per segment
        auto launch = [&](auto kern, int minb, int ty, size_t sm) {
          const int ncols = fg.ntx * ((g.P[1] + ty - 1) / ty);
          const int resident = p->sm_count * minb, extra = Wt.n - 1;
          int best = 1; double best_eff = 0.0;
          for (int ns = 1; ns <= std::max(1, g.P[2] / 16); ++ns) {
            const long long nb = (long long)ncols * ns;
            const int zs = (g.P[2] + ns - 1) / ns;
            const double eff = (double)nb / (double)((nb + resident - 1) / resident * resident) * zs / (zs + extra);
            if (eff > best_eff + 1e-9) { best_eff = eff; best = ns; }
          }
          fg.zseg = (g.P[2] + best - 1) / best;
          const dim3 grid(ncols, (g.P[2] + fg.zseg - 1) / fg.zseg);
          cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sm);
          MSM_LAUNCH(p, (kern<<<grid, kStreamThreads, sm, st>>>(fg, Wt, w2, src, (T*)d.pad)));
        };
        constexpr int MINB = sizeof(T) == 4 ? 2 : 1;
        switch (Wt.n) {
          case 11: launch(k_pad_filter_stream<T, 11, MINB, 32>, MINB, 32, filter_stream_smem<T, 11, 32>()); break;
          case 13: launch(k_pad_filter_stream<T, 13, 1, 32>, 1, 32, filter_stream_smem<T, 13, 32>()); break;
          default: launch(k_pad_filter_stream<T, 15, 1, 32>, 1, 32, filter_stream_smem<T, 15, 32>()); break;
        }
        continue;
      }
    }
    for (int ax = 0; ax < 3; ++ax) {
      AxisDims ad;
      for (int k = 0; k < 3; ++k) { ad.in[k] = din[k]; ad.out[k] = din[k]; }
      ad.out[ax] = g.P[ax];
      ad.axis = ax; ad.periodic = p->bg.periodic[ax];
      T* dst = ax == 2 ? (T*)d.pad : (T*)(ax == 0 ? p->tmpA : p->tmpB);
      // along the filtered axis the logical size is the grid's, not the (already padded) array's
      ad.in[ax] = lv.M[ax];
#define MSM_FILTER_RUN(AX, NT) MSM_LAUNCH(p, (k_pad_filter_run<T, AX, NT><<<filter_run_grid(ad), axis_block(), 0, st>>>( \
    ad, halo[ax], Wt, src, dst)))
#define MSM_FILTER_AX(AX)                                                                                  \
      switch (Wt.n) {                                                                                      \
        case 11: MSM_FILTER_RUN(AX, 11); break;                                                            \
        case 13: MSM_FILTER_RUN(AX, 13); break;                                                            \
        case 15: MSM_FILTER_RUN(AX, 15); break;                                                            \
        default: MSM_LAUNCH(p, (k_pad_filter<T, AX><<<axis_grid(ad), axis_block(), 0, st>>>(ad, halo[ax], Wt, src, dst))); \
      }
      if (ax == 0) { MSM_FILTER_AX(0) } else if (ax == 1) { MSM_FILTER_AX(1) } else { MSM_FILTER_AX(2) }
#undef MSM_FILTER_AX
#undef MSM_FILTER_RUN
      src = dst;
      din[ax] = g.P[ax];
    }
  }
  mark();
  bool top_early = false;
  auto launch_top = [&](cudaStream_t ts) {
    LevelDev& d = p->lev[p->n_t];
    const unsigned nb = blocks_for((size_t)p->G * 32, 128);
    if (want_virial)
      MSM_LAUNCH(p, (k_top_dense<T, true><<<nb, 128, 0, ts>>>(p->G, (const T*)p->topT, (const T*)p->topTD, (const T*)d.Q,
                                                             (T*)d.E, p->top_wrow)));
    else
      MSM_LAUNCH(p, (k_top_dense<T, false><<<nb, 128, 0, ts>>>(p->G, (const T*)p->topT, (const T*)p->topTD, (const T*)d.Q,
                                                              (T*)d.E, p->top_wrow)));
  };
  if (p->conv.nlev > 0) {
    constexpr int XT = sizeof(T) == 4 ? 16 : 8, ZT = 4;
    // shared memory of a generic (fp64) unit: plane | row entries of ZT layers | two row-tap buffers
    auto conv_layout = [&](int elems_per_chunk, int layers, size_t& total) {
      ConvSmemLayout sl;
      sl.rows_off = (int)((p->conv_smem + 15) / 16 * 16);
      sl.taps_off = sl.rows_off + layers * p->conv_ny_max * 16;
      sl.tapk = p->conv_maxc * elems_per_chunk;
      sl.tapbuf = layers * sl.tapk;
      total = (size_t)sl.taps_off + 2 * (size_t)sl.tapbuf * sizeof(T);
      return sl;
    };
    auto launch_virial = [&](cudaStream_t vs) {
      if constexpr (sizeof(T) == 4) {
        // list-driven kernel, one block of kConvVW warps per SM with the tap tables in shared memory
        // (not for small jobs: the table copy does not pay)
        const size_t plane_b = (p->conv_smem + 15) / 16 * 16;
        const size_t sm_l = p->conv_vtables_smem + kConvVW * plane_b + kConvVW * 8;   // + one mbarrier per warp
        static const bool no_l = std::getenv("MSM_CONV_NO_LISTS") != nullptr;
        if (!no_l && !p->conv_rowsliced && sm_l <= 226 * 1024 && p->conv.total_vunits >= 2048) {
          auto kern = k_conv_virial_f2l<XT>;
          cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sm_l);
          MSM_LAUNCH(p, (kern<<<p->conv.total_vsunits / kConvVW, 32 * kConvVW, sm_l, vs>>>(p->d_conv, (int)plane_b)));
          return;
        }
        auto kern = k_conv_virial_f2<XT>;             // packed FMAs (FFMA2)
        size_t sm;
        const ConvSmemLayout sl = conv_layout(24, 2, sm);
        if (sm > 48 * 1024) cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sm);
        MSM_LAUNCH(p, (kern<<<p->conv.total_vunits, 32, sm, vs>>>(p->d_conv, sl)));
      } else {
        auto kern = k_conv_virial<T, XT, ZT>;
        size_t sm;
        const ConvSmemLayout sl = conv_layout(12, ZT, sm);
        if (sm > 48 * 1024) cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sm);
        MSM_LAUNCH(p, (kern<<<p->conv.total_vunits, 32, sm, vs>>>(p->d_conv, sl)));
      }
    };
    // the virial correlation only needs the filtered grid charge: it runs on a third stream beside
    // the potential convolution (not with per-stage profiling on) and joins before the reductions
    // So does the dense top-level operator (it needs only the restricted charge): it goes first on
    // that stream and the prolongation waits for it (a small system's critical path is its chain of
    // dependent kernels: 0.025 ms of 0.13 at N = 3000).
    // Only where that stream is forked anyway (virial requested: a fork for the top operator alone
    // costs more than it gives) and only for small jobs outside a batch: at N = 10^6 it costs 0.06 ms (the virial kernel then starts
    // behind the potential kernel instead of in front of it), and the extra graph nodes of 64 batched
    // systems cost more than the overlap gives (0.94 -> 1.09 ms per batch).
    const bool beside = p->overlap && !p->profiling && p->vstream;
    const bool top_beside = beside && want_virial && p->top_beside && p->conv.total_units < 4096;
    if (beside && want_virial) {
      cudaEventRecord(p->fork2_ev, st);
      cudaStreamWaitEvent(p->vstream, p->fork2_ev, 0);
      if (top_beside) {
        launch_top(p->vstream);
        cudaEventRecord(p->top_ev, p->vstream);
        top_early = true;
      }
      if (want_virial) launch_virial(p->vstream);
      cudaEventRecord(p->join2_ev, p->vstream);
      forked_v = true;
    }
    {
      if constexpr (sizeof(T) == 4) {
        // packed FMAs (FFMA2); the stencil tables go to shared memory when two blocks of kConvSW
        // warps with their planes and tables fit on an SM
        const size_t plane_b = (p->conv_smem + 15) / 16 * 16;
        const size_t sm_s = p->conv_tables_smem + kConvSW * plane_b;
        static const bool no_s = std::getenv("MSM_CONV_GLOBAL_TAPS") != nullptr;
        static const bool no_l = std::getenv("MSM_CONV_NO_LISTS") != nullptr;
        if (!no_s && !p->conv_rowsliced && sm_s <= 110 * 1024 && p->conv.total_units >= 4096) {   // small jobs: the table copy does not pay
          // list-driven inner loops when every level has its entry lists (msm_create.cu)
          auto kern = p->conv_lists && !no_l ? k_conv_f2l<XT> : k_conv_f2s<XT>;
          const size_t sm_k = sm_s + kConvSW * 8;       // + one mbarrier per warp (k_conv_f2l)
          cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sm_k);
          MSM_LAUNCH(p, (kern<<<p->conv.total_sunits / kConvSW, 32 * kConvSW, sm_k, st>>>(p->d_conv, (int)plane_b)));
        } else {
          auto kern = k_conv_f2<XT>;
          size_t sm;
          const ConvSmemLayout sl = conv_layout(8, 2, sm);
          if (sm > 48 * 1024) cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sm);
          MSM_LAUNCH(p, (kern<<<p->conv.total_units, 32, sm, st>>>(p->d_conv, sl)));
        }
      } else {
        // fp64: list-driven kernel, one block of kConvDW warps per SM with the tap table in shared
        // memory (large jobs)
        const size_t plane_b = (p->conv_smem + 15) / 16 * 16;
        const size_t sm_d = p->conv_dtables_smem + kConvDW * plane_b + kConvDW * 8;
        static const bool no_l = std::getenv("MSM_CONV_NO_LISTS") != nullptr;
        if (!no_l && !p->conv_rowsliced && sm_d <= 226 * 1024 && p->conv.total_units >= 4096) {
          auto kern = k_conv_dl<8>;
          cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sm_d);
          MSM_LAUNCH(p, (kern<<<p->conv.total_dsunits / kConvDW, 32 * kConvDW, sm_d, st>>>(p->d_conv, (int)plane_b)));
        } else {
        auto kern = k_conv<T, XT, ZT>;
        size_t sm;
        const ConvSmemLayout sl = conv_layout(4, ZT, sm);
        if (sm > 48 * 1024) cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sm);
        MSM_LAUNCH(p, (kern<<<p->conv.total_units, 32, sm, st>>>(p->d_conv, sl)));
        }
      }
      for (int l = 1; l < p->n_t; ++l) {
        const ConvLevel& g = p->conv.lev[l - 1];
        if (g.nslices > 1) {
          const size_t pts = H.lev[l].points();
          MSM_LAUNCH(p, (k_sum_slices<T><<<blocks_for(pts, 256), 256, 0, st>>>(pts, g.nslices, (const T*)p->lev[l].scratch,
                                                                               (T*)p->lev[l].E)));
        }
      }
    }
    mark();
    if (want_virial) {
      if (!forked_v) launch_virial(st);
      for (int l = 1; l < p->n_t; ++l) {
        const ConvLevel& g = p->conv.lev[l - 1];
        const Level& lv = H.lev[l];
        Seg& s = fa.seg[nseg++];
        s.ptr = g.wpart; s.width = 6;
        s.count = g.tiles[0] * g.tiles[1] * g.tiles[2] * g.vslices;
        const double hx = lv.h[0], hy = lv.h[1], hz = lv.h[2];
        const double sc[6] = {hx * hx, hy * hy, hz * hz, hx * hy, hx * hz, hy * hz};
        for (int k = 0; k < 6; ++k) s.scale[k] = -0.5 * sc[k];
      }
    }
    mark();
  } else {
    mark(); mark();
  }

  // ---------------- S6 top level
  if (top_early) cudaStreamWaitEvent(st, p->top_ev, 0);
  else launch_top(st);
  if (want_virial) {
    Seg& s = fa.seg[nseg++];
    s.ptr = p->top_wrow; s.count = p->G; s.width = 6;
    for (int k = 0; k < 6; ++k) s.scale[k] = 1.0;
  }
  mark();

  // ---------------- S7 prolongation + accumulate, z then y then x
  for (int l = p->n_t - 1; l >= 1; --l) {
    const Level &f = H.lev[l], &c = H.lev[l + 1];
    if (stream_ok(f, c, p->prolong_stream_min_points)) {
      StreamGeom sg = stream_geom(f, c);
      constexpr int FXP = 64 * VecT<T>::VE, BY = 4;
      sg.ntx = (f.M[0] + FXP - 1) / FXP;
      auto pairs = [](int lo, int M) { return ((lo + M - 1) >> 1) - (lo >> 1) + 1; };   // node pairs (2b, 2b + 1) covering the axis
      const int nty = (pairs(f.lo[1], f.M[1]) + BY - 1) / BY, npz = pairs(f.lo[2], f.M[2]);
      sg.zseg = stream_zseg(sg.ntx * nty, npz, 2);     // small grids: short marches, more blocks
      const dim3 grid(sg.ntx * nty, (npz + sg.zseg - 1) / sg.zseg);
      MSM_LAUNCH(p, (k_prolong_stream<T, P + 1><<<grid, kStreamThreads, 0, st>>>(sg, Jt, (const T*)p->lev[l + 1].E,
                                                                                  (T*)p->lev[l].E)));
      continue;
    }
    const size_t sm = prolong3_smem_elems(P) * sizeof(T);
    auto kern = k_prolong3<T>;
    if (sm > 48 * 1024) cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sm);
    const dim3 grid((f.M[0] + kPTX - 1) / kPTX, (f.M[1] + kPTY - 1) / kPTY, (f.M[2] + kPTZ - 1) / kPTZ);
    MSM_LAUNCH(p, (kern<<<grid, 256, sm, st>>>(grid3(f), grid3(c), per3[0], per3[1], per3[2], Jt,
                                               (const T*)p->lev[l + 1].E, (T*)p->lev[l].E)));
  }
  mark();

  // ---------------- S8 interpolation + outputs
  if (forked) cudaStreamWaitEvent(st, p->join_ev, 0);
  const int neb = (int)blocks_for(n, 128);
  MSM_LAUNCH(p, (k_interpolate<T, P><<<neb, 128, 0, st>>>(
                    n, p->pair_nsplit, (size_t)p->cap, gg, tab, (T)(1.0 / H.lev[1].h[0]), (T)(1.0 / H.lev[1].h[1]), (T)(1.0 / H.lev[1].h[2]),
                    (T)(p->S->gamma0() / p->mp.a), (const V4*)p->grec, p->gcell_sorted, p->gorder,
                    (const T*)p->lev[1].E, (const T*)p->Fsr, (const T*)p->Vsr, (T*)d_F, (T*)d_V, p->epart)));
  mark();

  // ---------------- S9 reductions
  if (want_virial) {
    Seg& s = fa.seg[nseg++];
    s.ptr = p->pair_wpart; s.count = p->pair_blocks * PairWarps<T>::value; s.width = 6;
    for (int k = 0; k < 6; ++k) s.scale[k] = 1.0;
  }
  {
    Seg& s = fa.seg[nseg++];
    s.ptr = p->epart; s.count = neb; s.width = 1;
    for (int k = 0; k < 6; ++k) s.scale[k] = 0.0;
  }
  fa.nseg = nseg;
  int nblk = 0;
  for (int k = 0; k < nseg; ++k) {
    fa.seg[k].blk0 = nblk;
    nblk += (fa.seg[k].count + kRowsPerBlock - 1) / kRowsPerBlock;
  }
  fa.nblk = nblk;
  if (nblk > p->part_blocks) return MSM_ERR_CUDA;   // sized at plan creation; cannot happen
  if (forked_v) cudaStreamWaitEvent(st, p->join2_ev, 0);
  if (nblk > 0) MSM_LAUNCH(p, (k_partial_sums<<<nblk, 256, 0, st>>>(fa, p->part)));
  MSM_LAUNCH(p, (k_finalize<<<1, 256, 0, st>>>(nblk, p->part, p->flag, p->results)));
  mark();
  cudaMemcpyAsync(p->h_results, p->results, 8 * sizeof(double), cudaMemcpyDeviceToHost, st);
  return MSM_OK;
}

msm_status_t enqueue(msm_plan* p, int n, const void* pos, const void* q, void* F, void* V, bool wv, cudaStream_t st,
                     bool capturing) {
#define MSM_CASE(TT, PP) return enqueue_t<TT, PP>(p, n, pos, q, F, V, wv, st, capturing)
  if (p->fp32) {
    switch (p->P) { case 4: MSM_CASE(float, 4); case 6: MSM_CASE(float, 6); case 8: MSM_CASE(float, 8); }
  } else {
    switch (p->P) { case 4: MSM_CASE(double, 4); case 6: MSM_CASE(double, 6); case 8: MSM_CASE(double, 8); }
  }
#undef MSM_CASE
  return MSM_ERR_UNSUPPORTED;
}

// wait for the last enqueued evaluation, then read the stage times
msm_status_t finish(msm_plan* p) {
  if (!p->pending) return MSM_OK;
  p->pending = false;
  if (cudaEventSynchronize(p->done_ev) != cudaSuccess) { cudaGetLastError(); return MSM_ERR_CUDA; }
  if (cudaGetLastError() != cudaSuccess) return MSM_ERR_CUDA;
  if (p->profiling)
    for (int i = 0; i < p->n_stages; ++i) cudaEventElapsedTime(&p->stage_ms[i], p->ev[i], p->ev[i + 1]);
  return MSM_OK;
}

void drop_graph(msm_plan* p) {
  if (p->gexec) { cudaGraphExecDestroy(p->gexec); p->gexec = nullptr; }
}

// One evaluation, stream-ordered on st: returns as soon as the work is enqueued. The ~40-60 dependent
// launches of a small system cost more than their work, so the second consecutive call with the
// same arguments captures the launch sequence into a CUDA graph (on a plan-owned stream) and later
// calls replay it, ordered after everything already enqueued on st and joined back into st (work
// enqueued on st afterwards sees the outputs). Any change of arguments, or any failure of the
// capture, falls back to direct launches on the caller's stream.
msm_status_t run(msm_plan* p, int n, const void* pos, const void* q, void* F, void* V, bool wv, cudaStream_t st) {
  // the plan's scratch buffers are single: an evaluation still running (possibly on another stream)
  // is ordered in front of this one on the device; the host does not wait
  if (p->pending && cudaStreamWaitEvent(st, p->done_ev, 0) != cudaSuccess) { cudaGetLastError(); return MSM_ERR_CUDA; }
  const msm::GraphKey key{n, pos, q, F, V, wv, p->profiling};
  p->pending_virial = wv;
  if (p->graph_enabled && p->gstream && key == p->gkey) {
    if (!p->gexec) {
      cudaGraph_t g = nullptr;
      if (cudaStreamBeginCapture(p->gstream, cudaStreamCaptureModeThreadLocal) == cudaSuccess) {
        const msm_status_t es = enqueue(p, n, pos, q, F, V, wv, p->gstream, true);
        const cudaError_t ce = cudaStreamEndCapture(p->gstream, &g);
        if (es == MSM_OK && ce == cudaSuccess && g && cudaGraphInstantiate(&p->gexec, g, 0) != cudaSuccess)
          p->gexec = nullptr;
        if (g) cudaGraphDestroy(g);
      }
      if (!p->gexec) { cudaGetLastError(); p->graph_enabled = false; }   // never try again on this plan
    }
    if (p->gexec) {
      if (cudaEventRecord(p->gev, st) == cudaSuccess && cudaStreamWaitEvent(p->gstream, p->gev, 0) == cudaSuccess &&
          cudaGraphLaunch(p->gexec, p->gstream) == cudaSuccess && cudaEventRecord(p->done_ev, p->gstream) == cudaSuccess &&
          cudaStreamWaitEvent(st, p->done_ev, 0) == cudaSuccess) {
        p->pending = true;
        return MSM_OK;
      }
      cudaGetLastError();
      drop_graph(p);
      p->graph_enabled = false;
    }
  } else if (!(key == p->gkey)) {
    p->gkey = key;
    drop_graph(p);
  }
  const msm_status_t es = enqueue(p, n, pos, q, F, V, wv, st, false);
  if (es != MSM_OK) return es;
  if (cudaEventRecord(p->done_ev, st) != cudaSuccess) { cudaGetLastError(); return MSM_ERR_CUDA; }
  p->pending = true;
  return MSM_OK;
}

msm_status_t check_args(msm_plan* p, int n, const void* pos, const void* q) {
  if (!p || n < 0 || (n > 0 && (!pos || !q))) return MSM_ERR_INVALID_ARG;
  if (n > p->cap) return MSM_ERR_TOO_MANY_PARTICLES;
  return MSM_OK;
}

}  // namespace

extern "C" {

msm_status_t msm_evaluate_async(msm_plan_t* p, int n, const void* d_positions, const void* d_charges, void* d_forces,
                                void* d_potentials, int want_virial, void* cuda_stream) {
  const msm_status_t a = check_args(p, n, d_positions, d_charges);
  if (a != MSM_OK) return a;
  DeviceGuard dg(p->prm.device);
  if (!dg.ok) return MSM_ERR_CUDA;
  return run(p, n, d_positions, d_charges, d_forces, d_potentials, want_virial != 0, (cudaStream_t)cuda_stream);
}

msm_status_t msm_get_results(msm_plan_t* p, double* h_energy, double* h_virial) {
  if (!p) return MSM_ERR_INVALID_ARG;
  DeviceGuard dg(p->prm.device);
  if (!dg.ok) return MSM_ERR_CUDA;
  const msm_status_t s = finish(p);
  if (s != MSM_OK) return s;
  if (h_energy) *h_energy = p->h_results[0];
  if (h_virial) {
    if (p->pending_virial) std::memcpy(h_virial, p->h_results + 1, 6 * sizeof(double));
    else std::memset(h_virial, 0, 6 * sizeof(double));
  }
  if (p->h_results[7] != 0.0) return MSM_ERR_OUT_OF_BOX;
  return MSM_OK;
}

msm_status_t msm_evaluate(msm_plan_t* p, int n, const void* d_positions, const void* d_charges, void* d_forces,
                          void* d_potentials, double* h_energy, double* h_virial, void* cuda_stream) {
  const msm_status_t s = msm_evaluate_async(p, n, d_positions, d_charges, d_forces, d_potentials, h_virial != nullptr,
                                            cuda_stream);
  if (s != MSM_OK) return s;
  if (!h_energy && !h_virial) return MSM_OK;       // stream-ordered: no host output, no synchronisation
  return msm_get_results(p, h_energy, h_virial);
}

msm_status_t msm_evaluate_host(msm_plan_t* p, int n, const void* h_positions, const void* h_charges, void* h_forces,
                               void* h_potentials, double* h_energy, double* h_virial, void* cuda_stream) {
  const msm_status_t a = check_args(p, n, h_positions, h_charges);
  if (a != MSM_OK) return a;
  DeviceGuard dg(p->prm.device);
  if (!dg.ok) return MSM_ERR_CUDA;
  cudaStream_t st = (cudaStream_t)cuda_stream;
  const size_t e = p->esz;
  msm_status_t fs = finish(p);                      // the staging buffers may still be in use
  if (fs != MSM_OK) return fs;
  if (cudaMemcpyAsync(p->in_pos, h_positions, (size_t)n * 3 * e, cudaMemcpyHostToDevice, st) != cudaSuccess ||
      cudaMemcpyAsync(p->in_q, h_charges, (size_t)n * e, cudaMemcpyHostToDevice, st) != cudaSuccess) {
    cudaGetLastError();
    return MSM_ERR_CUDA;
  }
  msm_status_t s = msm_evaluate_async(p, n, p->in_pos, p->in_q, h_forces ? p->out_F : nullptr,
                                      h_potentials ? p->out_V : nullptr, h_virial != nullptr, cuda_stream);
  if (s != MSM_OK) return s;
  if (h_forces) cudaMemcpyAsync(h_forces, p->out_F, (size_t)n * 3 * e, cudaMemcpyDeviceToHost, st);
  if (h_potentials) cudaMemcpyAsync(h_potentials, p->out_V, (size_t)n * e, cudaMemcpyDeviceToHost, st);
  s = msm_get_results(p, h_energy, h_virial);
  if (cudaStreamSynchronize(st) != cudaSuccess) { cudaGetLastError(); return MSM_ERR_CUDA; }
  return s;
}

msm_status_t msm_set_profiling(msm_plan_t* p, int enabled) {
  if (!p) return MSM_ERR_INVALID_ARG;
  p->profiling = enabled != 0;
  return MSM_OK;
}

msm_status_t msm_get_stage_times(const msm_plan_t* p, int* n_stages, const char* const** names,
                                 const float** milliseconds) {
  if (!p || !n_stages || !names || !milliseconds) return MSM_ERR_INVALID_ARG;
  *n_stages = p->n_stages;
  *names = p->stage_names.data();
  *milliseconds = p->stage_ms;
  return MSM_OK;
}

msm_status_t msm_get_launch_count(const msm_plan_t* p, int* count) {
  if (!p || !count) return MSM_ERR_INVALID_ARG;
  *count = p->launches;
  return MSM_OK;
}

msm_status_t msm_debug_copy_grid(const msm_plan_t* p, int level, int kind, double* h_out, size_t capacity) {
  if (!p || !h_out || level < 1 || level > p->n_t || (kind != 0 && kind != 1)) return MSM_ERR_INVALID_ARG;
  const size_t pts = p->H->lev[level].points();
  if (capacity < pts) return MSM_ERR_INVALID_ARG;
  DeviceGuard dg(p->prm.device);
  if (!dg.ok) return MSM_ERR_CUDA;
  if (p->pending && cudaEventSynchronize(p->done_ev) != cudaSuccess) { cudaGetLastError(); return MSM_ERR_CUDA; }
  const void* src = kind == 0 ? p->lev[level].Q : p->lev[level].E;
  if (p->fp32) {
    // fp32 values are exact in fp64: copy into the upper half of the caller's buffer, widen in place
    float* tmp = reinterpret_cast<float*>(h_out) + pts;
    if (cudaMemcpy(tmp, src, pts * 4, cudaMemcpyDeviceToHost) != cudaSuccess) return MSM_ERR_CUDA;
    for (size_t i = 0; i < pts; ++i) h_out[i] = tmp[i];
  } else if (cudaMemcpy(h_out, src, pts * 8, cudaMemcpyDeviceToHost) != cudaSuccess) {
    return MSM_ERR_CUDA;
  }
  return MSM_OK;
}

}  // extern "C"

// ------------------------------------------------------------------------------------------------
// Batched evaluation of many small systems of one geometry (msmJAX batches structures
// with vmap, fixed grid counts and zero-charge padding; a small system is dominated by a
// constant overhead). One evaluation of a 512-particle system is a chain of ~40 dependent kernel
// launches that leaves the GPU almost empty; a batch is B such chains captured as parallel branches
// of ONE CUDA graph: every system has its own scratch (a plan of the shared geometry), the
// branches are spread over a pool of streams, and one graph launch runs them side by side.
struct msm_batch {
  int B = 0, device = 0, cap = 0, nstreams = 0;
  size_t esz = 8;
  std::vector<msm_plan*> plans;
  std::vector<cudaStream_t> streams;
  std::vector<cudaEvent_t> join_ev;
  cudaStream_t origin = nullptr;
  cudaEvent_t fork_ev = nullptr, in_ev = nullptr, done_ev = nullptr;
  cudaGraphExec_t gexec = nullptr;
  // arguments of the captured graph
  std::vector<int> n;
  const void *pos = nullptr, *q = nullptr;
  void *F = nullptr, *V = nullptr;
  bool virial = false;
};

namespace {
constexpr int kBatchStreams = 32;

void batch_drop_graph(msm_batch* b) {
  if (b->gexec) { cudaGraphExecDestroy(b->gexec); b->gexec = nullptr; }
}
}  // namespace

extern "C" {

void msm_batch_destroy(msm_batch_t* b) {
  if (!b) return;
  DeviceGuard dg(b->device);
  if (b->origin) cudaStreamSynchronize(b->origin);
  batch_drop_graph(b);
  for (msm_plan* p : b->plans) msm_plan_destroy(p);
  for (cudaStream_t s : b->streams) cudaStreamDestroy(s);
  for (cudaEvent_t e : b->join_ev) cudaEventDestroy(e);
  if (b->fork_ev) cudaEventDestroy(b->fork_ev);
  if (b->in_ev) cudaEventDestroy(b->in_ev);
  if (b->done_ev) cudaEventDestroy(b->done_ev);
  if (b->origin) cudaStreamDestroy(b->origin);
  delete b;
}

msm_status_t msm_batch_create(const msm_params_t* params, int batch, msm_batch_t** batch_out) {
  if (!batch_out) return MSM_ERR_INVALID_ARG;
  *batch_out = nullptr;
  if (!params || batch < 1 || batch > 65536) return MSM_ERR_INVALID_ARG;
  msm_batch* b = new (std::nothrow) msm_batch();
  if (!b) return MSM_ERR_NOMEM;
  b->B = batch; b->device = params->device; b->cap = params->max_particles;
  b->esz = params->precision == MSM_FP32 ? 4 : 8;
  try {
    b->plans.reserve(batch);
    for (int i = 0; i < batch; ++i) {
      msm_plan_t* p = nullptr;
      const msm_status_t s = msm::plan_create_opts(params, 0.0, true, &p);
      if (s != MSM_OK) { msm_batch_destroy(b); return s; }
      p->graph_enabled = false;                     // the batch owns the graph
      b->plans.push_back(p);
    }
  } catch (...) { msm_batch_destroy(b); return MSM_ERR_NOMEM; }
  DeviceGuard dg(b->device);
  if (!dg.ok) { msm_batch_destroy(b); return MSM_ERR_CUDA; }
  b->nstreams = std::min(batch, kBatchStreams);
  bool ok = cudaStreamCreateWithFlags(&b->origin, cudaStreamNonBlocking) == cudaSuccess &&
            cudaEventCreateWithFlags(&b->fork_ev, cudaEventDisableTiming) == cudaSuccess &&
            cudaEventCreateWithFlags(&b->in_ev, cudaEventDisableTiming) == cudaSuccess &&
            cudaEventCreateWithFlags(&b->done_ev, cudaEventDisableTiming) == cudaSuccess;
  for (int i = 0; ok && i < b->nstreams; ++i) {
    cudaStream_t s = nullptr;
    cudaEvent_t e = nullptr;
    ok = cudaStreamCreateWithFlags(&s, cudaStreamNonBlocking) == cudaSuccess &&
         cudaEventCreateWithFlags(&e, cudaEventDisableTiming) == cudaSuccess;
    if (s) b->streams.push_back(s);
    if (e) b->join_ev.push_back(e);
  }
  if (!ok) { cudaGetLastError(); msm_batch_destroy(b); return MSM_ERR_CUDA; }
  *batch_out = b;
  return MSM_OK;
}

msm_status_t msm_evaluate_batch(msm_batch_t* b, const int* h_n, const void* d_positions, const void* d_charges,
                                void* d_forces, void* d_potentials, double* h_energy, double* h_virial,
                                void* cuda_stream) {
  if (!b || !h_n || !d_positions || !d_charges) return MSM_ERR_INVALID_ARG;
  for (int i = 0; i < b->B; ++i) {
    if (h_n[i] < 0) return MSM_ERR_INVALID_ARG;
    if (h_n[i] > b->cap) return MSM_ERR_TOO_MANY_PARTICLES;
  }
  DeviceGuard dg(b->device);
  if (!dg.ok) return MSM_ERR_CUDA;
  cudaStream_t st = (cudaStream_t)cuda_stream;
  const bool wv = h_virial != nullptr;
  bool same = b->gexec && b->pos == d_positions && b->q == d_charges && b->F == d_forces && b->V == d_potentials &&
              b->virial == wv && (int)b->n.size() == b->B;
  for (int i = 0; same && i < b->B; ++i) same = b->n[i] == h_n[i];
  if (!same) {
    if (cudaStreamSynchronize(b->origin) != cudaSuccess) { cudaGetLastError(); return MSM_ERR_CUDA; }
    batch_drop_graph(b);
    const size_t cap = (size_t)b->cap, e = b->esz;
    cudaGraph_t g = nullptr;
    msm_status_t es = MSM_OK;
    if (cudaStreamBeginCapture(b->origin, cudaStreamCaptureModeThreadLocal) != cudaSuccess) { cudaGetLastError(); return MSM_ERR_CUDA; }
    cudaEventRecord(b->fork_ev, b->origin);
    for (int s = 0; s < b->nstreams; ++s) cudaStreamWaitEvent(b->streams[s], b->fork_ev, 0);
    for (int i = 0; i < b->B && es == MSM_OK; ++i) {
      const char* pp = (const char*)d_positions + (size_t)i * cap * 3 * e;
      const char* qq = (const char*)d_charges + (size_t)i * cap * e;
      char* ff = d_forces ? (char*)d_forces + (size_t)i * cap * 3 * e : nullptr;
      char* vv = d_potentials ? (char*)d_potentials + (size_t)i * cap * e : nullptr;
      es = enqueue(b->plans[i], h_n[i], pp, qq, ff, vv, wv, b->streams[i % b->nstreams], true);
    }
    for (int s = 0; s < b->nstreams; ++s) {
      cudaEventRecord(b->join_ev[s], b->streams[s]);
      cudaStreamWaitEvent(b->origin, b->join_ev[s], 0);
    }
    const cudaError_t ce = cudaStreamEndCapture(b->origin, &g);
    if (es != MSM_OK || ce != cudaSuccess || !g || cudaGraphInstantiate(&b->gexec, g, 0) != cudaSuccess) {
      if (g) cudaGraphDestroy(g);
      b->gexec = nullptr;
      cudaGetLastError();
      return es != MSM_OK ? es : MSM_ERR_CUDA;
    }
    cudaGraphDestroy(g);
    b->n.assign(h_n, h_n + b->B);
    b->pos = d_positions; b->q = d_charges; b->F = d_forces; b->V = d_potentials; b->virial = wv;
  }
  // ordered after the caller's stream, joined back into it
  if (cudaEventRecord(b->in_ev, st) != cudaSuccess || cudaStreamWaitEvent(b->origin, b->in_ev, 0) != cudaSuccess ||
      cudaGraphLaunch(b->gexec, b->origin) != cudaSuccess || cudaEventRecord(b->done_ev, b->origin) != cudaSuccess ||
      cudaStreamWaitEvent(st, b->done_ev, 0) != cudaSuccess) {
    cudaGetLastError();
    return MSM_ERR_CUDA;
  }
  if (!h_energy && !h_virial) return MSM_OK;        // stream-ordered, as msm_evaluate
  if (cudaEventSynchronize(b->done_ev) != cudaSuccess) { cudaGetLastError(); return MSM_ERR_CUDA; }
  msm_status_t rs = MSM_OK;
  for (int i = 0; i < b->B; ++i) {
    const double* r = b->plans[i]->h_results;
    if (h_energy) h_energy[i] = r[0];
    if (h_virial) std::memcpy(h_virial + 6 * (size_t)i, r + 1, 6 * sizeof(double));
    if (r[7] != 0.0) rs = MSM_ERR_OUT_OF_BOX;
  }
  return rs;
}

}  // extern "C"
