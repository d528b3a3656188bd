// msm_create.cu -- msm_plan_create / msm_plan_destroy / msm_plan_info: host mathematics (fp64)
// and every device buffer of a plan. See include/msm.h.
#include <algorithm>
#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <map>
#include <new>

#include "pair.cuh"
#include "plan.hpp"

using namespace msm;

namespace {

struct CudaFail {};

void* dev_alloc(msm_plan* p, size_t bytes) {
  void* d = nullptr;
  if (bytes == 0) bytes = 16;
  if (cudaMalloc(&d, bytes) != cudaSuccess) throw std::bad_alloc();
  if (cudaMemset(d, 0, bytes) != cudaSuccess) throw CudaFail();
  p->allocs.push_back(d);
  p->bytes += bytes;
  return d;
}

template <typename T> void* upload_as(msm_plan* p, const std::vector<double>& v) {
  std::vector<T> t(v.size());
  for (size_t i = 0; i < v.size(); ++i) t[i] = (T)v[i];
  void* d = dev_alloc(p, std::max<size_t>(t.size(), 4) * sizeof(T));
  if (!t.empty() && cudaMemcpy(d, t.data(), t.size() * sizeof(T), cudaMemcpyHostToDevice) != cudaSuccess)
    throw CudaFail();
  return d;
}

void* upload(msm_plan* p, const std::vector<double>& v) {
  return p->fp32 ? upload_as<float>(p, v) : upload_as<double>(p, v);
}

int round_up(int v, int m) { return (v + m - 1) / m * m; }

// balanced partition of n weighted items into S contiguous slices: bounds b[0..S]
void balanced_bounds(const std::vector<double>& w, int S, unsigned char* b) {
  const int n = (int)w.size();
  double tot = 0;
  for (double v : w) tot += v;
  b[0] = 0;
  int i = 0;
  double run = 0;
  for (int s = 1; s < S; ++s) {
    const double target = tot * s / S;
    while (i < n && run + 0.5 * w[i] < target && n - (i + 1) >= S - s) { run += w[i]; ++i; }
    if (i < s) { while (i < s) { run += w[i]; ++i; } }   // at least one plane per slice
    b[s] = (unsigned char)i;
  }
  b[S] = (unsigned char)n;
}

// stencil row tables + chunked taps of one tiled level (see conv.cuh)
int4* upload_desc(msm_plan* p, const std::vector<int4>& v) {
  int4* d = (int4*)dev_alloc(p, std::max<size_t>(v.size(), 1) * sizeof(int4));
  if (!v.empty() && cudaMemcpy(d, v.data(), v.size() * sizeof(int4), cudaMemcpyHostToDevice) != cudaSuccess) throw CudaFail();
  return d;
}

void build_conv_tables(msm_plan* p, int l, int XT, int ZT) {
  const Level& lv = p->H->lev[l];
  LevelDev& d = p->lev[l];
  // the table STRUCTURE (which taps exist, halo widths) is sized for the smallest spacings the plan
  // reserves room for; the VALUES are sampled at the actual spacings (zero outside the ellipsoid)
  double hs[3];
  for (int ax = 0; ax < 3; ++ax) hs[ax] = p->mp.periodic[ax] ? lv.h[ax] * (1.0 - p->reserve) : lv.h[ax];
  for (int ax = 0; ax < 3; ++ax) d.hstruct[ax] = hs[ax];
  const SampledStencil st = sample_level_stencil(*p->H, *p->S, l, hs);
  std::vector<int4> tsd, tvd, t2d(8, make_int4(0, 0, 0, 0)), tv2d;
  d.taps = st.taps;
  ConvLevel& g = p->conv.lev[l - 1];
  for (int ax = 0; ax < 3; ++ax) { g.M[ax] = lv.M[ax]; g.R[ax] = st.R[ax]; }
  g.X0 = round_up(st.R[0], 4);
  g.tiles[0] = (lv.M[0] + XT - 1) / XT;
  g.tiles[1] = (lv.M[1] + 31) / 32;
  g.tiles[2] = (lv.M[2] + ZT - 1) / ZT;
  g.P[0] = g.tiles[0] * XT + 2 * g.X0 + 4;
  g.P[1] = g.tiles[1] * 32 + 2 * st.R[1];
  g.P[2] = g.tiles[2] * ZT + 2 * st.R[2];
  const int WX = XT + 2 * g.X0 + 4;
  int pitch = WX;
  if (p->fp32) { pitch = round_up(pitch, 4); if (((pitch / 4) & 1) == 0) pitch += 4; }
  else { pitch = round_up(pitch, 2); if (((pitch / 2) & 1) == 0) pitch += 2; }
  g.pitch = pitch;
  g.ny = 2 * st.R[1] + 1;
  p->conv_ny_max = std::max(p->conv_ny_max, g.ny);
  p->conv_smem = std::max(p->conv_smem, (size_t)(32 + 2 * st.R[1]) * pitch * p->esz);

  const double A = std::ldexp(p->mp.a, l);
  const int ny = g.ny, nz = 2 * st.R[2] + 1, Rz = st.R[2];
  std::vector<int4> rows((size_t)ny * nz), vrows((size_t)ny * (Rz + 1));
  std::vector<double> ts, tv;
  std::vector<double> wz(nz, 0.0), wzv(Rz + 1, 0.0);     // chunks per tap plane (work weights)
  std::map<std::pair<int, int>, int> seen_rows, seen_vrows;
  for (int dz = -Rz; dz <= Rz; ++dz)
    for (int dy = -st.R[1]; dy <= st.R[1]; ++dy) {
      int4& r = rows[(size_t)(dz + Rz) * ny + (dy + st.R[1])];
      const double y = dy * hs[1], z = dz * hs[2];
      const double rem = A * A - y * y - z * z;
      int Rx = -1;
      if (rem > 0) {
        Rx = std::min(st.R[0], (int)std::floor(std::sqrt(rem) / hs[0]));
        while (Rx >= 0 && (Rx * hs[0]) * (Rx * hs[0]) >= rem) --Rx;
      }
      if (Rx < 0) { r = make_int4(0, 1, 0, 0); }
      else {
        const int clo = (-Rx + g.X0) / 4, chi = (Rx + g.X0) / 4;
        p->conv_maxc = std::max(p->conv_maxc, chi - clo + 1);
        wz[dz + Rz] += chi - clo + 1 + 0.5;
        // s is even in every coordinate (for any spacings): the rows (+-dz, +-dy) share one copy
        const std::pair<int, int> key(std::abs(dz), std::abs(dy));
        auto it = seen_rows.find(key);
        if (it == seen_rows.end()) {
          it = seen_rows.emplace(key, (int)(ts.size() / 4)).first;
          for (int c = clo; c <= chi; ++c)
            for (int t = 0; t < 4; ++t) {
              const int dx = 4 * c - g.X0 + t;
              const bool in = dx >= -Rx && dx <= Rx;
              ts.push_back(in ? st.at(st.s, dx, dy, dz) : 0.0);
              tsd.push_back(make_int4(dx, dy, dz, in ? 1 : 0));
            }
        }
        r = make_int4(it->second, clo, chi, 0);
      }
      // virial: half space n > 0 (z, then y, then x), weight 2 (C(n) is even, reading V)
      if (dz < 0) continue;
      int4& v = vrows[(size_t)dz * ny + (dy + st.R[1])];
      const bool whole = dz > 0 || dy > 0, centre = dz == 0 && dy == 0;
      if (Rx < 0 || !(whole || centre) || (centre && Rx < 1)) { v = make_int4(0, 1, 0, 0); continue; }
      const int xlo = centre ? 1 : -Rx;
      const int clo = (xlo + g.X0) / 4, chi = (Rx + g.X0) / 4;
      wzv[dz] += chi - clo + 1 + 0.5;
      // g is even in every coordinate: the whole rows (dz > 0, +-dy) share one copy
      const std::pair<int, int> vkey(dz, dz > 0 ? std::abs(dy) : dy);
      auto vit = seen_vrows.find(vkey);
      if (vit == seen_vrows.end()) {
        vit = seen_vrows.emplace(vkey, (int)(tv.size() / 12)).first;
        for (int c = clo; c <= chi; ++c)
          for (int m = 0; m < 3; ++m)
            for (int t = 0; t < 4; ++t) {
              const int dx = 4 * c - g.X0 + t;
              const bool in = dx >= xlo && dx <= Rx;
              const double gv = in ? 2.0 * st.at(st.g, dx, dy, dz) : 0.0;
              tv.push_back(m == 0 ? gv : m == 1 ? gv * dx : gv * dx * dx);
              tvd.push_back(make_int4(dx, dy, dz, in ? 2 + m : 0));
            }
      }
      v = make_int4(vit->second, clo, chi, 0);
    }
  auto up_rows = [&](const std::vector<int4>& r) {
    int4* dptr = (int4*)dev_alloc(p, r.size() * sizeof(int4));
    if (cudaMemcpy(dptr, r.data(), r.size() * sizeof(int4), cudaMemcpyHostToDevice) != cudaSuccess) throw CudaFail();
    return dptr;
  };
  g.rows = up_rows(rows);
  g.vrows = up_rows(vrows);
  g.staps = upload(p, ts);
  g.vtaps = upload(p, tv);
  d.tab[0] = TapTable{const_cast<void*>(g.staps), upload_desc(p, tsd), (int)ts.size()};
  g.dlist = nullptr;
  g.dhead = nullptr;
  g.n_stapsq = (int)((ts.size() * p->esz + 15) / 16);
  if (!p->fp32) {
    // entry lists of the fp64 list-driven potential kernel (k_conv_dl): input plane offset zr feeds
    // output plane k through stencil layer dz = zr - k; lists: all four planes / planes (0, 1) /
    // planes (2, 3) / one plane alone
    auto on = [&](int dz, int j, int c, int& chunk) {
      if (dz < -Rz || dz > Rz) return false;
      const int4& r = rows[(size_t)(dz + Rz) * ny + j];
      if (c < r.y || c > r.z) return false;
      chunk = r.x + (c - r.y);
      return true;
    };
    std::vector<int4> el;
    std::vector<int> eh;
    const int cmax = (2 * g.X0) / 4 + 1;
    for (int zr = -Rz; zr <= Rz + 3; ++zr) {
      std::vector<int4> lists[kConvListTypes];
      for (int j = 0; j < ny; ++j)
        for (int c = 0; c <= cmax; ++c) {
          int ch[4] = {0, 0, 0, 0};
          bool a[4];
          for (int k = 0; k < 4; ++k) a[k] = on(zr - k, j, c, ch[k]);
          if (!(a[0] || a[1] || a[2] || a[3])) continue;
          const int4 e0 = make_int4((j * g.pitch + 4 * c) * 8, ch[0] * 32, ch[1] * 32, ch[2] * 32), e1 = make_int4(ch[3] * 32, 0, 0, 0);
          auto put = [&](int t) { lists[t].push_back(e0); lists[t].push_back(e1); };
          if (a[0] && a[1] && a[2] && a[3]) { put(0); continue; }
          if (a[0] && a[1]) put(1); else { if (a[0]) put(3); if (a[1]) put(4); }
          if (a[2] && a[3]) put(2); else { if (a[2]) put(5); if (a[3]) put(6); }
        }
      for (int t = 0; t < kConvListTypes; ++t) {
        eh.push_back((int)(el.size() / 2));
        el.insert(el.end(), lists[t].begin(), lists[t].end());
      }
      eh.push_back((int)(el.size() / 2));
    }
    el.push_back(make_int4(0, 0, 0, 0));
    el.push_back(make_int4(0, 0, 0, 0));
    int4* eld = (int4*)dev_alloc(p, el.size() * sizeof(int4));
    int* ehd = (int*)dev_alloc(p, eh.size() * sizeof(int));
    if (cudaMemcpy(eld, el.data(), el.size() * sizeof(int4), cudaMemcpyHostToDevice) != cudaSuccess ||
        cudaMemcpy(ehd, eh.data(), eh.size() * sizeof(int), cudaMemcpyHostToDevice) != cudaSuccess)
      throw CudaFail();
    g.dlist = eld;
    g.dhead = ehd;
  }
  d.tab[2] = TapTable{const_cast<void*>(g.vtaps), upload_desc(p, tvd), (int)tv.size()};
  g.rows2 = nullptr;
  g.elist = nullptr;
  g.ehead = nullptr;
  g.vlist = nullptr;
  g.vhead = nullptr;
  g.n_vtaps2q = 0;
  g.taps2 = nullptr;
  g.vrows2 = nullptr;
  g.vtaps2 = nullptr;
  if (p->fp32) {
    // packed path (k_conv_f2): stencil rows d and d - 1 merged, taps interleaved per tap
    auto row_rx = [&](int dz, int dy) {               // x half-width of row (dz, dy), -1 if empty
      if (dz < -Rz || dz > Rz) return -1;
      const int4& r = rows[(size_t)(dz + Rz) * ny + (dy + st.R[1])];
      if (r.y > r.z) return -1;
      const double y = dy * hs[1], z = dz * hs[2];
      const double rem = A * A - y * y - z * z;
      int Rx = std::min(st.R[0], (int)std::floor(std::sqrt(rem) / hs[0]));
      while (Rx >= 0 && (Rx * hs[0]) * (Rx * hs[0]) >= rem) --Rx;
      return Rx;
    };
    std::vector<int4> r2((size_t)ny * (nz + 1));
    std::vector<double> t2(8, 0.0);                  // guard chunk in front of the table (index -1)
    std::map<std::vector<double>, int> seen2, seenv2;
    for (int d = -Rz; d <= Rz + 1; ++d)
      for (int dy = -st.R[1]; dy <= st.R[1]; ++dy) {
        const int ra = row_rx(d, dy), rb = row_rx(d - 1, dy), Rx = std::max(ra, rb);
        int4& r = r2[(size_t)(d + Rz) * ny + (dy + st.R[1])];
        if (Rx < 0) { r = make_int4(0, 0, -1, 0); continue; }   // empty: clamps to chunk -1
        const int clo = (-Rx + g.X0) / 4, chi = (Rx + g.X0) / 4;
        // first and last 2-tap half-chunk that holds a tap: the kernel skips the empty half of the
        // first and of the last chunk of a row
        const int halves = ((-Rx + g.X0) / 2) | (((Rx + g.X0) / 2) << 16);
        std::vector<double> rowv;
        std::vector<int4> rowd;
        for (int c = clo; c <= chi; ++c)
          for (int t = 0; t < 4; ++t) {
            const int dx = 4 * c - g.X0 + t;
            const bool ia = ra >= 0 && dx >= -ra && dx <= ra, ib = rb >= 0 && dx >= -rb && dx <= rb;
            rowv.push_back(ia ? st.at(st.s, dx, dy, d) : 0.0);
            rowv.push_back(ib ? st.at(st.s, dx, dy, d - 1) : 0.0);
            rowd.push_back(make_int4(dx, dy, d, ia ? 1 : 0));
            rowd.push_back(make_int4(dx, dy, d - 1, ib ? 1 : 0));
          }
        // rows (d, dy) and (d, -dy) hold the same taps (for any spacings): stored once (half the
        // table, better L1 reuse)
        auto it = seen2.find(rowv);
        if (it == seen2.end()) {
          it = seen2.emplace(rowv, (int)(t2.size() / 8) - 1).first;
          t2.insert(t2.end(), rowv.begin(), rowv.end());
          t2d.insert(t2d.end(), rowd.begin(), rowd.end());
        }
        r = make_int4(it->second, clo, chi, halves);
      }
    // virial, packed: half-space rows d and d - 1 merged, per chunk 24 floats (2g, 2g dx, 2g dx^2)
    // x 4 taps x (row d, row d - 1)
    auto vrange = [&](int dz, int dy, int& xlo, int& xhi) {          // taps of half-space row (dz, dy)
      if (dz < 0 || dz > Rz) return false;
      const int Rx = row_rx(dz, dy);
      const bool whole = dz > 0 || dy > 0, centre = dz == 0 && dy == 0;
      if (Rx < 0 || !(whole || centre) || (centre && Rx < 1)) return false;
      xlo = centre ? 1 : -Rx; xhi = Rx;
      return true;
    };
    std::vector<int4> vr2((size_t)ny * (Rz + 2));
    std::vector<double> tv2;
    for (int d = 0; d <= Rz + 1; ++d)
      for (int dy = -st.R[1]; dy <= st.R[1]; ++dy) {
        int alo = 0, ahi = -1, blo = 0, bhi = -1;
        const bool ha = vrange(d, dy, alo, ahi), hb = vrange(d - 1, dy, blo, bhi);
        int4& r = vr2[(size_t)d * ny + (dy + st.R[1])];
        if (!ha && !hb) { r = make_int4(0, 1, 0, 0); continue; }
        const int xlo = ha && hb ? std::min(alo, blo) : (ha ? alo : blo);
        const int xhi = ha && hb ? std::max(ahi, bhi) : (ha ? ahi : bhi);
        const int clo = (xlo + g.X0) / 4, chi = (xhi + g.X0) / 4;
        const int halves = ((xlo + g.X0) / 2) | (((xhi + g.X0) / 2) << 16);
        p->conv_maxc = std::max(p->conv_maxc, chi - clo + 1);
        std::vector<double> rowv;
        std::vector<int4> rowd;
        for (int c = clo; c <= chi; ++c)
          for (int m = 0; m < 3; ++m)
            for (int t = 0; t < 4; ++t) {
              const int dx = 4 * c - g.X0 + t;
              const bool ia = ha && dx >= alo && dx <= ahi, ib = hb && dx >= blo && dx <= bhi;
              const double ga = ia ? 2.0 * st.at(st.g, dx, dy, d) : 0.0;
              const double gb = ib ? 2.0 * st.at(st.g, dx, dy, d - 1) : 0.0;
              const double f = m == 0 ? 1.0 : m == 1 ? (double)dx : (double)dx * dx;
              rowv.push_back(ga * f);
              rowv.push_back(gb * f);
              rowd.push_back(make_int4(dx, dy, d, ia ? 2 + m : 0));
              rowd.push_back(make_int4(dx, dy, d - 1, ib ? 2 + m : 0));
            }
        auto it = seenv2.find(rowv);
        if (it == seenv2.end()) {
          it = seenv2.emplace(rowv, (int)(tv2.size() / 24)).first;
          tv2.insert(tv2.end(), rowv.begin(), rowv.end());
          tv2d.insert(tv2d.end(), rowd.begin(), rowd.end());
        }
        r = make_int4(it->second, clo, chi, halves);
      }
    g.vrows2 = up_rows(vr2);
    g.vtaps2 = upload(p, tv2);
    g.n_vtaps2q = (int)(tv2.size() / 4);
    // entry lists of the list-driven virial kernel (as for the potential, see below): input plane zr
    // (dz >= 0 only) feeds the plane pairs k = 0, 1 through the merged half-space layers zr and zr - 2
    {
      auto vstate = [&](int d, int j, int c, int& chunk) {     // 0 off, 1 full, 2 lower half, 3 upper half
        if (d < 0 || d > Rz + 1) return 0;
        const int4& r = vr2[(size_t)d * ny + j];
        if (c < r.y || c > r.z) return 0;
        chunk = r.x + (c - r.y);
        const bool lo = 2 * c >= (r.w & 0xffff), hi = 2 * c + 1 <= (r.w >> 16);
        return lo && hi ? 1 : lo ? 2 : hi ? 3 : 0;
      };
      std::vector<int4> el;
      std::vector<int> eh;
      const int cmax = (2 * g.X0) / 4 + 1;
      for (int zr = 0; zr <= Rz + 3; ++zr) {
        std::vector<int4> lists[kConvListTypes];
        for (int j = 0; j < ny; ++j) {
          const float fy = (float)(j - st.R[1]);
          int fyb;
          std::memcpy(&fyb, &fy, 4);
          for (int c = 0; c <= cmax; ++c) {
            int c0 = 0, c1 = 0;
            const int s0 = vstate(zr, j, c, c0), s1 = vstate(zr - 2, j, c, c1);
            const int4 e = make_int4((j * g.pitch + 4 * c) * 4, c0 * 96, c1 * 96, fyb);   // bytes
            if (s0 == 1 && s1 == 1) { lists[0].push_back(e); continue; }
            if (s0 == 1) lists[1].push_back(e);
            if (s1 == 1) lists[2].push_back(e);
            if (s0 == 2) lists[3].push_back(e);
            if (s0 == 3) lists[4].push_back(e);
            if (s1 == 2) lists[5].push_back(e);
            if (s1 == 3) lists[6].push_back(e);
          }
        }
        for (int t = 0; t < kConvListTypes; ++t) {
          eh.push_back((int)el.size());
          el.insert(el.end(), lists[t].begin(), lists[t].end());
        }
        eh.push_back((int)el.size());
      }
      el.push_back(make_int4(0, 0, 0, 0));
      int4* eld = (int4*)dev_alloc(p, el.size() * sizeof(int4));
      int* ehd = (int*)dev_alloc(p, eh.size() * sizeof(int));
      if (cudaMemcpy(eld, el.data(), el.size() * sizeof(int4), cudaMemcpyHostToDevice) != cudaSuccess ||
          cudaMemcpy(ehd, eh.data(), eh.size() * sizeof(int), cudaMemcpyHostToDevice) != cudaSuccess)
        throw CudaFail();
      g.vlist = eld;
      g.vhead = ehd;
    }
    d.tab[3] = TapTable{const_cast<void*>(g.vtaps2), upload_desc(p, tv2d), (int)tv2.size()};
    g.rows2 = up_rows(r2);
    void* t2dev = upload(p, t2);
    d.tab[1] = TapTable{t2dev, upload_desc(p, t2d), (int)t2.size()};
    g.taps2 = (const char*)t2dev + 8 * p->esz;   // chunk 0 of the table follows the guard chunk
    g.n_rows2 = (int)r2.size();
    g.n_taps2q = (int)(t2.size() / 4);
    // Entry lists of the list-driven kernel (k_conv_f2l): input plane zr feeds the output plane pairs
    // k = 0, 1 through the merged layers d0 = zr and d0 - 2. Per d0, the chunks of all stencil rows
    // are sorted by what they need -- both pairs in full / one pair in full / the lower or upper 2-tap
    // half of one pair -- so that each list runs through a loop body without any branch.
    g.elist = nullptr;
    g.ehead = nullptr;
    {
      auto state = [&](int d, int j, int c, int& chunk) {      // 0 off, 1 full, 2 lower half, 3 upper half
        if (d < -Rz || d > Rz + 1) return 0;
        const int4& r = r2[(size_t)(d + Rz) * ny + j];
        if (c < r.y || c > r.z) return 0;
        chunk = r.x + (c - r.y);
        const bool lo = 2 * c >= (r.w & 0xffff), hi = 2 * c + 1 <= (r.w >> 16);
        return lo && hi ? 1 : lo ? 2 : hi ? 3 : 0;
      };
      std::vector<int4> el;
      std::vector<int> eh;
      const int cmax = (2 * g.X0) / 4 + 1;
      for (int d0 = -Rz; d0 <= Rz + 3; ++d0) {
        std::vector<int4> lists[kConvListTypes];
        for (int j = 0; j < ny; ++j)
          for (int c = 0; c <= cmax; ++c) {
            int c0 = 0, c1 = 0;
            const int s0 = state(d0, j, c, c0), s1 = state(d0 - 2, j, c, c1);
            const int4 e = make_int4((j * g.pitch + 4 * c) * 4, c0 * 32, c1 * 32, 0);   // bytes
            if (s0 == 1 && s1 == 1) { lists[0].push_back(e); continue; }
            if (s0 == 1) lists[1].push_back(e);
            if (s1 == 1) lists[2].push_back(e);
            if (s0 == 2) lists[3].push_back(e);
            if (s0 == 3) lists[4].push_back(e);
            if (s1 == 2) lists[5].push_back(e);
            if (s1 == 3) lists[6].push_back(e);
          }
        for (int t = 0; t < kConvListTypes; ++t) {
          eh.push_back((int)el.size());
          el.insert(el.end(), lists[t].begin(), lists[t].end());
        }
        eh.push_back((int)el.size());
      }
      el.push_back(make_int4(0, 0, 0, 0));                           // the loops prefetch one entry ahead
      int4* eld = (int4*)dev_alloc(p, el.size() * sizeof(int4));
      int* ehd = (int*)dev_alloc(p, eh.size() * sizeof(int));
      if (cudaMemcpy(eld, el.data(), el.size() * sizeof(int4), cudaMemcpyHostToDevice) != cudaSuccess ||
          cudaMemcpy(ehd, eh.data(), eh.size() * sizeof(int), cudaMemcpyHostToDevice) != cudaSuccess)
        throw CudaFail();
      g.elist = eld;
      g.ehead = ehd;
    }
  }
  d.pad = dev_alloc(p, (size_t)g.P[0] * g.P[1] * g.P[2] * p->esz);
  g.pad = d.pad;
  g.Q = d.Q;

  // slices of the input planes, balanced by the taps each plane feeds into the ZT output planes
  const int nplanes = 2 * Rz + ZT, vplanes = Rz + ZT;
  std::vector<double> wp(nplanes, 0.0), wv(vplanes, 0.0);
  for (int pz = 0; pz < nplanes; ++pz)
    for (int k = 0; k < ZT; ++k) {
      const int dz = pz - Rz - k;
      if (dz >= -Rz && dz <= Rz) wp[pz] += wz[dz + Rz];
      wp[pz] += 0.3;   // staging
    }
  for (int pz = 0; pz < vplanes; ++pz)
    for (int k = 0; k < ZT; ++k) {
      const int dz = pz - k;
      if (dz >= 0 && dz <= Rz) wv[pz] += wzv[dz];
      wv[pz] += 0.3;
    }
  const int tiles = g.tiles[0] * g.tiles[1] * g.tiles[2];
  // units per tile: slices of the input planes; a PLAN with fewer plane-slice units than SMs over all
  // its levels (16^3 grids: 96) deals each plane slice to several units by stencil rows, at least three rows each.
  // Measured: N = 3000 (16^3) 0.147 -> 0.135 ms per evaluation; applied to 32^3 grids (432 units)
  // it made config 2 slower (0.26 -> 0.32 ms: the units crowd out the pair kernel beside them)
  const int pslices = std::max(1, std::min({p->conv_slices, nplanes, kMaxConvSlices}));
  const int pvslices = std::max(1, std::min({p->conv_vslices, vplanes, kMaxConvSlices}));
  const int ymax = std::max(1, std::min(kMaxRowSlices, ny / 3));
  auto row_slices = [&](int units) {
    return units < p->sm_count && !p->in_batch ? std::max(1, std::min(ymax, (2 * p->sm_count + units - 1) / units)) : 1;
  };
  g.ysl = row_slices((int)std::min<long long>(p->conv_tiles_total * pslices, 1 << 30));
  g.vysl = row_slices((int)std::min<long long>(p->conv_tiles_total * pvslices, 1 << 30));
  if (g.ysl > 1 || g.vysl > 1) p->conv_rowsliced = true;
  g.nslices = pslices * g.ysl;
  g.vslices = pvslices * g.vysl;
  balanced_bounds(wp, pslices, g.pb);
  balanced_bounds(wv, pvslices, g.vb);
  g.unit0 = p->conv.total_units;
  g.vunit0 = p->conv.total_vunits;
  g.sunit0 = p->conv.total_sunits;                       // blocks of kConvSW units never straddle two levels
  p->conv.total_sunits += (tiles * g.nslices + kConvSW - 1) / kConvSW * kConvSW;
  g.dsunit0 = p->conv.total_dsunits;
  p->conv.total_dsunits += (tiles * g.nslices + kConvDW - 1) / kConvDW * kConvDW;
  if (!p->fp32) p->conv_dtables_smem = std::max(p->conv_dtables_smem, (size_t)g.n_stapsq * 16);
  g.vsunit0 = p->conv.total_vsunits;
  p->conv.total_vsunits += (tiles * g.vslices + kConvVW - 1) / kConvVW * kConvVW;
  if (p->fp32) {
    p->conv_tables_smem = std::max(p->conv_tables_smem, (size_t)g.n_taps2q * 16 + (size_t)g.n_rows2 * 16);
    p->conv_vtables_smem = std::max(p->conv_vtables_smem, (size_t)g.n_vtaps2q * 16);
  }
  p->conv.total_units += tiles * g.nslices;
  p->conv.total_vunits += tiles * g.vslices;
  if (g.nslices > 1) {
    d.scratch = dev_alloc(p, (size_t)g.nslices * lv.points() * p->esz);
    g.out = d.scratch;
  } else {
    g.out = d.E;
  }
}

msm_status_t create_impl(const msm_params_t* prm, msm_plan* p) {
  p->prm = *prm;
  p->fp32 = prm->precision == MSM_FP32;
  p->esz = p->fp32 ? 4 : 8;
  p->mu = prm->mu < 0 ? 4 : prm->mu;
  Params& mp = p->mp;
  for (int ax = 0; ax < 3; ++ax) { mp.box[ax] = prm->box[ax]; mp.periodic[ax] = prm->periodic[ax] ? 1 : 0; }
  mp.h = prm->h; mp.a = prm->a; mp.p = prm->p; mp.levels = prm->levels; mp.mu = p->mu;
  if (prm->max_particles < 1 || (prm->precision != MSM_FP32 && prm->precision != MSM_FP64) || p->mu > 28)
    return MSM_ERR_INVALID_ARG;
  if (prm->p != 4 && prm->p != 6 && prm->p != 8) return prm->p > 0 && (prm->p & 1) == 0 && prm->p <= 8
                                                             ? MSM_ERR_UNSUPPORTED : MSM_ERR_INVALID_ARG;
  p->H = new Hierarchy(mp);
  if (p->H->status == 2) return MSM_ERR_UNSUPPORTED;
  if (p->H->status == 3) return MSM_ERR_INVALID_ARG;
  if (p->H->status == 4) return MSM_ERR_CUTOFF_TOO_LARGE;
  const Hierarchy& H = *p->H;
  p->P = prm->p;
  p->w = H.w;
  p->n_t = std::min(prm->levels, H.L);
  if (H.lev[p->n_t].points() > MSM_MAX_TOP_POINTS) return MSM_ERR_UNSUPPORTED;
  p->S = new Splitting(prm->p, prm->a, H.L);
  p->J = two_scale_mask(prm->p);
  p->omega = quasi_interp_sequence(prm->p, p->mu);
  p->pieces = new SplinePieces(prm->p);

  if (cudaSetDevice(prm->device) != cudaSuccess) return MSM_ERR_CUDA;
  if (cudaDeviceGetAttribute(&p->sm_count, cudaDevAttrMultiProcessorCount, prm->device) != cudaSuccess || p->sm_count < 1)
    return MSM_ERR_CUDA;

  // ---- grids
  // slices per output tile of the convolution. fp32: one-warp units for about two resident waves of
  // the potential kernel and one of the virial kernel (16 warps per SM). Measured at 128^3 + 64^3 +
  // 32^3 (1168 tiles, 148 SMs): 4 / 2 slices 0.630 / 0.555 ms; 7 / 4 (3.45 / 1.97 waves) 0.663 / 0.609 ms
  {
    const int XTc = p->fp32 ? 16 : 8;
    long long tiles = 0;
    for (int l = 1; l < p->n_t; ++l)
      tiles += (long long)((H.lev[l].M[0] + XTc - 1) / XTc) * ((H.lev[l].M[1] + 31) / 32) * ((H.lev[l].M[2] + 3) / 4);
    p->conv_tiles_total = tiles;
    const long long slots = (long long)p->sm_count * 16;
    if (p->fp32) {
      auto per_tile = [&](long long units) {
        return tiles > 0 ? (int)std::max<long long>(1, std::min<long long>(kMaxConvSlices, (units + tiles / 2) / tiles)) : 1;
      };
      p->conv_slices = per_tile(2 * slots);
      p->conv_vslices = per_tile(slots);
    } else {
      // fp64 (12 / 9 resident warps per SM, units twice as long): more, smaller units measured faster
      // (N = 10^6: 4 / 2 slices 1.736 / 1.545 ms, 2 / 1 slices 1.812 / 1.567 ms)
      p->conv_slices = tiles > 0 ? (int)std::max<long long>(1, std::min<long long>(kMaxConvSlices, (3 * slots + tiles - 1) / tiles)) : 1;
      p->conv_vslices = p->conv_slices;             // (virial 1.55 -> 1.48 ms at N = 10^6 against half as many)
      // large jobs run the list-driven potential kernel, ONE block of kConvDW warps per SM: few slices
      // whose blocks fill whole waves of SMs (N = 10^6, 2336 tiles: 3 slices = 3.95 waves 1.22 ms,
      // 4 slices = 5.26 waves 1.40 ms, 6 slices = 7.9 waves 1.38 ms)
      if (tiles * p->conv_slices >= 4096) {
        double best = -1.0;
        for (int sl = 2; sl <= 8; ++sl) {
          const double waves = (double)((tiles * sl + kConvDW - 1) / kConvDW) / (double)p->sm_count;
          const double score = waves / std::ceil(waves) - 0.01 * sl;
          if (tiles * sl >= 4096 && score > best) { best = score; p->conv_slices = sl; }
        }
      }
    }
    if (const char* e = std::getenv("MSM_CONV_SLICES")) p->conv_slices = std::max(1, std::atoi(e));
    if (const char* e = std::getenv("MSM_CONV_VSLICES")) p->conv_vslices = std::max(1, std::atoi(e));
  }
  size_t tmp_elems = 16;
  const int XT = p->fp32 ? 16 : 8, ZT = 4;
  for (int l = 1; l <= p->n_t; ++l) {
    const size_t pts = H.lev[l].points();
    p->lev[l].Q = dev_alloc(p, pts * p->esz);
    p->lev[l].E = dev_alloc(p, pts * p->esz);
    tmp_elems = std::max(tmp_elems, pts);
    if (l < p->n_t) {
      if (l > kMaxConvLevels) return MSM_ERR_UNSUPPORTED;
      build_conv_tables(p, l, XT, ZT);
      const ConvLevel& g = p->conv.lev[l - 1];
      tmp_elems = std::max(tmp_elems, (size_t)g.P[0] * g.P[1] * g.P[2]);
      if (p->conv_smem > 227 * 1024) return MSM_ERR_UNSUPPORTED;
    }
  }
  p->conv.nlev = p->n_t - 1;
  if (p->conv.nlev > 0) {
    // the exact dynamic shared memory of the convolution launches (conv_layout in msm_evaluate.cu:
    // plane | row entries | two row-tap buffers) has to fit an SM; refuse here, not at the launch
    auto total = [&](int elems_per_chunk, int layers) {
      const size_t rows_off = (p->conv_smem + 15) / 16 * 16;
      return rows_off + (size_t)layers * p->conv_ny_max * 16 + 2 * (size_t)layers * p->conv_maxc * elems_per_chunk * p->esz;
    };
    const size_t need = p->fp32 ? std::max(total(24, 2), total(8, 2)) : std::max(total(12, 4), total(4, 4));
    if (need > 227 * 1024) return MSM_ERR_UNSUPPORTED;
    for (int l = 1; l < p->n_t; ++l)
      if (2 * p->conv.lev[l - 1].R[2] + 4 > 255) return MSM_ERR_UNSUPPORTED;   // plane indices are bytes
    p->conv_wpart =(double*)dev_alloc(p, (size_t)p->conv.total_vunits * 6 * sizeof(double));
    for (int l = 1; l < p->n_t; ++l) {
      ConvLevel& g = p->conv.lev[l - 1];
      g.wpart = p->conv_wpart + (size_t)g.vunit0 * 6;
    }
    p->d_conv = (ConvTable*)dev_alloc(p, sizeof(ConvTable));
    if (cudaMemcpy(p->d_conv, &p->conv, sizeof(ConvTable), cudaMemcpyHostToDevice) != cudaSuccess) throw CudaFail();
  }
  p->tmpA = dev_alloc(p, tmp_elems * p->esz);
  p->tmpB = dev_alloc(p, tmp_elems * p->esz);

  // ---- top operator (always built with its strain derivatives: plan-time cost only)
  {
    const TopOperator top = build_top_operator(H, *p->S, p->omega, p->J, p->n_t, true);
    p->G = top.G;
    p->topT = upload(p, top.T);
    std::vector<double> td;
    td.reserve((size_t)6 * top.G * top.G);
    for (int k = 0; k < 6; ++k) td.insert(td.end(), top.TD[k].begin(), top.TD[k].end());
    p->topTD = upload(p, td);
    p->top_wrow = (double*)dev_alloc(p, (size_t)top.G * 6 * sizeof(double));
  }

  // ---- particle side
  BinGeom& bg = p->bg;
  for (int ax = 0; ax < 3; ++ax) {
    bg.box[ax] = prm->box[ax];
    bg.periodic[ax] = mp.periodic[ax];
    // (cells stay >= a/2 wide down to the smallest box the plan reserves room for)
    bg.nc[ax] = std::max(1, (int)std::floor(prm->box[ax] * (mp.periodic[ax] ? 1.0 - p->reserve : 1.0) / (0.5 * prm->a)));
    bg.cell_edge[ax] = prm->box[ax] / bg.nc[ax];
    bg.h1[ax] = H.lev[1].h[ax];
    bg.ng[ax] = mp.periodic[ax] ? H.lev[1].M[ax] : (int)std::floor(prm->box[ax] / prm->h) + 1;
  }
  // tiled anterpolation when each tile grid fits once into every periodic axis and there are enough
  // tiles (one warp each) to fill the GPU; otherwise the gather kernel
  {
    const int tdim[3] = {8, 8, 4};
    p->anterp_tiled = true;
    long long ntiles = 1;
    for (int ax = 0; ax < 3; ++ax) {
      p->at.T[ax] = prm->p - 1 <= tdim[ax] ? tdim[ax] : 8;   // power of two >= p - 1: divides periodic M, <= 2 tiles per node and axis
      p->at.tshift[ax] = p->at.T[ax] == 8 ? 3 : 2;
      p->at.D[ax] = p->at.T[ax] + prm->p - 1;
      p->at.nt[ax] = (bg.ng[ax] + p->at.T[ax] - 1) / p->at.T[ax];
      ntiles *= p->at.nt[ax];
      if (mp.periodic[ax] && H.lev[1].M[ax] < p->at.D[ax]) p->anterp_tiled = false;
    }
    {
      const char* e = std::getenv("MSM_ANTERP_MIN_TILES");
      if (ntiles < (e ? std::atoi(e) : 128)) p->anterp_tiled = false;
    }
    if (const char* e = std::getenv("MSM_ANTERP_TILED")) p->anterp_tiled = p->anterp_tiled && std::atoi(e) != 0;
    // few tiles: several warps per tile (each its own scratch grid) so that ~2000 warps run
    p->at.split = (int)std::max<long long>(1, std::min<long long>(8, 2048 / std::max<long long>(ntiles, 1)));
    if (p->anterp_tiled)
      p->anterp_scratch = dev_alloc(p, (size_t)ntiles * p->at.split * p->at.D[0] * p->at.D[1] * p->at.D[2] * p->esz);
  }
  // x sub-bins per pair cell: 8, fewer when the bins would far outnumber the particles
  bg.sxs = 3;
  while (bg.sxs > 0 && (((long long)bg.nc[0] * bg.nc[1] * bg.nc[2]) << bg.sxs) > 8LL * prm->max_particles + (1 << 16)) --bg.sxs;
  if (const char* e = std::getenv("MSM_PAIR_SUBBINS_LOG2")) bg.sxs = std::max(0, std::min(3, std::atoi(e)));
  const long long npc = ((long long)bg.nc[0] * bg.nc[1] * bg.nc[2]) << bg.sxs;
  const long long ngc = (long long)bg.ng[0] * bg.ng[1] * bg.ng[2];
  if (npc > (1ll << 28) || ngc > (1ll << 28)) return MSM_ERR_UNSUPPORTED;
  p->n_pcells = (int)npc; p->n_gcells = (int)ngc;
  p->pair_rows = bg.nc[1] * bg.nc[2];
  p->cap = prm->max_particles;
  const size_t cap = (size_t)p->cap;
  p->ibuf_count = (size_t)p->n_pcells + p->n_gcells + 8;
  p->ibuf = (int*)dev_alloc(p, p->ibuf_count * sizeof(int));
  p->phist = p->ibuf;
  p->ghist = p->phist + p->n_pcells;
  p->flag = p->ghist + p->n_gcells;
  p->pstart = (int*)dev_alloc(p, ((size_t)p->n_pcells + 1) * sizeof(int));
  p->gstart = (int*)dev_alloc(p, ((size_t)p->n_gcells + 1) * sizeof(int));
  p->ptotals = (int*)dev_alloc(p, ((size_t)p->n_pcells / 4096 + 2) * sizeof(int));
  p->gtotals = (int*)dev_alloc(p, ((size_t)p->n_gcells / 4096 + 2) * sizeof(int));
  p->pslot = (int*)dev_alloc(p, cap * sizeof(int));
  p->gslot = (int*)dev_alloc(p, cap * sizeof(int));
  p->pcell = (int*)dev_alloc(p, cap * sizeof(int));
  p->gcell = (int*)dev_alloc(p, cap * sizeof(int));
  p->porder = (int*)dev_alloc(p, cap * sizeof(int));
  p->gorder = (int*)dev_alloc(p, cap * sizeof(int));
  p->pcellx = (int*)dev_alloc(p, cap * sizeof(int));
  p->gcell_sorted = (int*)dev_alloc(p, cap * sizeof(int));
  p->prec = dev_alloc(p, cap * 4 * p->esz);
  p->grec = dev_alloc(p, cap * 4 * p->esz);
  p->Fsr = dev_alloc(p, (size_t)kPairMaxSplit * cap * 3 * p->esz);   // per-split partials of the pair kernel
  p->Vsr = dev_alloc(p, (size_t)kPairMaxSplit * cap * p->esz);
  const int pw = p->fp32 ? PairWarps<float>::value : PairWarps<double>::value;
  p->pair_ymax = (int)((cap / kPairCluster + p->pair_rows) / p->pair_rows + pw - 1) / pw + 1;
  p->pair_wpart = (double*)dev_alloc(p, (size_t)p->pair_rows * p->pair_ymax * kPairMaxSplit * pw * 6 * sizeof(double));
  p->n_eblocks = (int)((cap + 127) / 128);
  p->epart = (double*)dev_alloc(p, (size_t)p->n_eblocks * sizeof(double));
  {
    const size_t rows = (size_t)p->pair_rows * p->pair_ymax * kPairMaxSplit * pw + p->conv.total_vunits + p->G + p->n_eblocks;
    p->part_blocks = (int)(rows / 1024 + MSM_MAX_LEVELS + 8);
    p->part = (double*)dev_alloc(p, (size_t)p->part_blocks * 7 * sizeof(double));
  }
  p->results = (double*)dev_alloc(p, 8 * sizeof(double));
  p->in_pos = dev_alloc(p, cap * 3 * p->esz);
  p->in_q = dev_alloc(p, cap * p->esz);
  p->out_F = dev_alloc(p, cap * 3 * p->esz);
  p->out_V = dev_alloc(p, cap * p->esz);
  if (cudaMallocHost((void**)&p->h_results, 8 * sizeof(double)) != cudaSuccess) return MSM_ERR_NOMEM;
  for (int i = 0; i <= kMaxStages; ++i)
    if (cudaEventCreate(&p->ev[i]) != cudaSuccess) return MSM_ERR_CUDA;
  // stream priorities: the grid pipeline first, the pair kernel last, so that the convolution blocks
  // take the slots the pair kernel leaves free instead of queueing behind its whole grid
  int prio_lo = 0, prio_hi = 0;
  cudaDeviceGetStreamPriorityRange(&prio_lo, &prio_hi);
  if (cudaStreamCreateWithPriority(&p->gstream, cudaStreamNonBlocking, prio_hi) != cudaSuccess ||
      cudaEventCreateWithFlags(&p->gev, cudaEventDisableTiming) != cudaSuccess ||
      cudaEventCreateWithFlags(&p->done_ev, cudaEventDisableTiming) != cudaSuccess)
    return MSM_ERR_CUDA;
  if (const char* e = std::getenv("MSM_NO_GRAPH")) p->graph_enabled = std::atoi(e) == 0;
  if (cudaStreamCreateWithPriority(&p->pstream, cudaStreamNonBlocking, prio_lo) != cudaSuccess ||
      cudaEventCreateWithFlags(&p->fork_ev, cudaEventDisableTiming) != cudaSuccess ||
      cudaEventCreateWithFlags(&p->join_ev, cudaEventDisableTiming) != cudaSuccess ||
      cudaStreamCreateWithPriority(&p->vstream, cudaStreamNonBlocking, prio_hi) != cudaSuccess ||
      cudaEventCreateWithFlags(&p->fork2_ev, cudaEventDisableTiming) != cudaSuccess ||
      cudaEventCreateWithFlags(&p->join2_ev, cudaEventDisableTiming) != cudaSuccess ||
      cudaEventCreateWithFlags(&p->top_ev, cudaEventDisableTiming) != cudaSuccess)
    return MSM_ERR_CUDA;
  if (const char* e = std::getenv("MSM_NO_OVERLAP")) p->overlap = std::atoi(e) == 0;
  if (const char* e = std::getenv("MSM_GRID_STREAM_MIN")) p->stream_min_points = p->prolong_stream_min_points = p->filter_stream_min_points = std::atoll(e);
  if (const char* e = std::getenv("MSM_FILTER_STREAM_MIN")) p->filter_stream_min_points = std::atoll(e);
  // stage list of msm_evaluate, in launch order
  for (const char* s : {"sort", "pair", "anterpolate", "restrict"}) p->stage_name_store.push_back(s);
  for (const char* s : {"filter", "conv", "conv_virial"}) p->stage_name_store.push_back(s);
  for (const char* s : {"top", "prolongate", "interpolate", "reduce"}) p->stage_name_store.push_back(s);
  for (const std::string& s : p->stage_name_store) p->stage_names.push_back(s.c_str());
  p->n_stages = (int)p->stage_names.size();
  return MSM_OK;
}

// ---- dynamic cell: tap values recomputed on the device (with a dynamic cell the
// stencils are rebuilt from the current cell at every call; every intermediate level has
// the same functional form, so one kernel serves all levels)
struct TapGeom {
  double h[3];
  double A0, A1;      // 2^(l-1) a, 2^l a
  int p;
  double c[8];        // binom(-1/2, k)
};

__device__ double dev_gamma(const TapGeom& g, double rho) {
  if (rho >= 1.0) return 1.0 / rho;
  const double s = rho * rho - 1.0;
  double acc = g.c[g.p - 1];
  for (int k = g.p - 2; k >= 0; --k) acc = acc * s + g.c[k];
  return acc;
}
__device__ double dev_dgamma(const TapGeom& g, double rho) {
  if (rho >= 1.0) return -1.0 / (rho * rho);
  const double s = rho * rho - 1.0;
  double acc = (g.p - 1) * g.c[g.p - 1];
  for (int k = g.p - 2; k >= 1; --k) acc = acc * s + k * g.c[k];
  return 2.0 * rho * acc;
}

// values[i] from desc[i] = (dx, dy, dz, kind): s_l = k_l(|h o n|) (Eq. 21 middle case, reading
// K1) or 2 k_l'(r)/r times 1, dx, dx^2; zero outside the cutoff ellipsoid r < 2^l a (Eq. 3)
template <typename T>
__global__ void k_rebuild_taps(int n, const int4* __restrict__ desc, TapGeom g, T* __restrict__ values) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  const int4 d = desc[i];
  double v = 0.0;
  if (d.w != 0) {
    const double x = d.x * g.h[0], y = d.y * g.h[1], z = d.z * g.h[2];
    const double r = sqrt(x * x + y * y + z * z);
    if (r < g.A1) {
      if (d.w == 1) {
        v = dev_gamma(g, r / g.A0) / g.A0 - dev_gamma(g, r / g.A1) / g.A1;
      } else if (r > 0.0) {
        const double dk = dev_dgamma(g, r / g.A0) / (g.A0 * g.A0) - dev_dgamma(g, r / g.A1) / (g.A1 * g.A1);
        const double gv = 2.0 * dk / r;
        v = d.w == 2 ? gv : (d.w == 3 ? gv * d.x : gv * d.x * d.x);
      }
    }
  }
  values[i] = (T)v;
}

msm_status_t set_box_impl(msm_plan* p, const double* box) {
  const Hierarchy& H0 = *p->H;
  for (int ax = 0; ax < 3; ++ax) {
    if (!(box[ax] > 0.0)) return MSM_ERR_INVALID_ARG;
    if (!p->mp.periodic[ax]) {
      // an open axis has no spacing of its own: its node set follows box / h (reading G2)
      if (std::fabs(box[ax] - p->mp.box[ax]) > 1e-12 * p->mp.box[ax]) return MSM_ERR_UNSUPPORTED;
      continue;
    }
    if (p->mp.a > 0.5 * box[ax]) return MSM_ERR_CUTOFF_TOO_LARGE;           // minimum image
    if (box[ax] / p->bg.nc[ax] < 0.5 * p->mp.a * (1.0 - 1e-12)) return MSM_ERR_UNSUPPORTED;   // below the reserve
    for (int l = 1; l < p->n_t; ++l)
      if (box[ax] / H0.lev[l].M[ax] < p->lev[l].hstruct[ax] * (1.0 - 1e-12)) return MSM_ERR_UNSUPPORTED;
  }
  if (p->pending && cudaEventSynchronize(p->done_ev) != cudaSuccess) { cudaGetLastError(); return MSM_ERR_CUDA; }
  p->pending = false;
  if (p->gexec) { cudaGraphExecDestroy(p->gexec); p->gexec = nullptr; }     // geometry is baked into the graph
  p->gkey = msm::GraphKey{};
  // host copies of the geometry: the number of grid points is what stays fixed
  Hierarchy& H = *p->H;
  for (int ax = 0; ax < 3; ++ax) {
    p->prm.box[ax] = p->mp.box[ax] = H.prm.box[ax] = p->bg.box[ax] = box[ax];
    p->bg.cell_edge[ax] = box[ax] / p->bg.nc[ax];
    if (!p->mp.periodic[ax]) continue;
    for (int l = 1; l <= H.L; ++l) H.lev[l].h[ax] = box[ax] / H.lev[l].M[ax];
    p->bg.h1[ax] = H.lev[1].h[ax];
  }
  // sampled stencils of every tiled level, on the device
  for (int l = 1; l < p->n_t; ++l) {
    TapGeom g;
    for (int ax = 0; ax < 3; ++ax) g.h[ax] = H.lev[l].h[ax];
    g.A0 = std::ldexp(p->mp.a, l - 1); g.A1 = std::ldexp(p->mp.a, l);
    g.p = p->P;
    for (int k = 0; k < 8; ++k) g.c[k] = p->S->c[k];
    for (int t = 0; t < 4; ++t) {
      const TapTable& tb = p->lev[l].tab[t];
      if (!tb.values || tb.n == 0) continue;
      const unsigned nb = (unsigned)((tb.n + 255) / 256);
      if (p->fp32) k_rebuild_taps<float><<<nb, 256>>>(tb.n, tb.desc, g, (float*)tb.values);
      else k_rebuild_taps<double><<<nb, 256>>>(tb.n, tb.desc, g, (double*)tb.values);
    }
  }
  // the dense operator of the top grid (<= 4096 points): rebuilt on the host and uploaded
  {
    const TopOperator top = build_top_operator(H, *p->S, p->omega, p->J, p->n_t, true);
    std::vector<double> td;
    td.reserve((size_t)6 * top.G * top.G);
    for (int k = 0; k < 6; ++k) td.insert(td.end(), top.TD[k].begin(), top.TD[k].end());
    auto put = [&](void* dst, const std::vector<double>& v) {
      if (p->fp32) {
        std::vector<float> t(v.begin(), v.end());
        return cudaMemcpy(dst, t.data(), t.size() * 4, cudaMemcpyHostToDevice) == cudaSuccess;
      }
      return cudaMemcpy(dst, v.data(), v.size() * 8, cudaMemcpyHostToDevice) == cudaSuccess;
    };
    if (!put(p->topT, top.T) || !put(p->topTD, td)) { cudaGetLastError(); return MSM_ERR_CUDA; }
  }
  if (cudaDeviceSynchronize() != cudaSuccess || cudaGetLastError() != cudaSuccess) return MSM_ERR_CUDA;
  return MSM_OK;
}

}  // namespace

extern "C" {

msm_status_t msm_plan_set_box(msm_plan_t* p, const double* box) {
  if (!p || !box) return MSM_ERR_INVALID_ARG;
  DeviceGuard dg(p->prm.device);
  if (!dg.ok) return MSM_ERR_CUDA;
  try {
    return set_box_impl(p, box);
  } catch (const std::bad_alloc&) {
    return MSM_ERR_NOMEM;
  } catch (...) {
    return MSM_ERR_CUDA;
  }
}

void msm_plan_destroy(msm_plan_t* p) {
  if (!p) return;
  DeviceGuard dg(p->prm.device);
  if (p->pending) cudaEventSynchronize(p->done_ev);
  for (void* d : p->allocs) cudaFree(d);
  if (p->pstream) cudaStreamDestroy(p->pstream);
  if (p->vstream) cudaStreamDestroy(p->vstream);
  if (p->fork2_ev) cudaEventDestroy(p->fork2_ev);
  if (p->join2_ev) cudaEventDestroy(p->join2_ev);
  if (p->top_ev) cudaEventDestroy(p->top_ev);
  if (p->fork_ev) cudaEventDestroy(p->fork_ev);
  if (p->join_ev) cudaEventDestroy(p->join_ev);
  if (p->gexec) cudaGraphExecDestroy(p->gexec);
  if (p->gstream) cudaStreamDestroy(p->gstream);
  if (p->gev) cudaEventDestroy(p->gev);
  if (p->done_ev) cudaEventDestroy(p->done_ev);
  if (p->h_results) cudaFreeHost(p->h_results);
  for (int i = 0; i <= kMaxStages; ++i)
    if (p->ev[i]) cudaEventDestroy(p->ev[i]);
  delete p->H; delete p->S; delete p->pieces;
  delete p;
}

msm_status_t msm_plan_create(const msm_params_t* params, msm_plan_t** plan_out) {
  return msm_plan_create_dynamic(params, 0.0, plan_out);
}

msm_status_t msm_plan_create_dynamic(const msm_params_t* params, double reserve, msm_plan_t** plan_out) {
  return msm::plan_create_opts(params, reserve, false, plan_out);
}

}  // extern "C"

// (internal) in_batch: the plan is one of many that run side by side in one graph (msm_batch_create):
// no extra units or streams for latency's sake, the batch fills the GPU
msm_status_t msm::plan_create_opts(const msm_params_t* params, double reserve, bool in_batch, msm_plan_t** plan_out) {
  if (!plan_out) return MSM_ERR_INVALID_ARG;
  *plan_out = nullptr;
  if (!params || !(reserve >= 0.0) || reserve > 0.5) return MSM_ERR_INVALID_ARG;
  msm_plan* p = new (std::nothrow) msm_plan();
  if (!p) return MSM_ERR_NOMEM;
  p->reserve = reserve;
  p->in_batch = in_batch;
  p->top_beside = !in_batch;
  if (const char* e = std::getenv("MSM_TOP_BESIDE")) p->top_beside = p->top_beside && std::atoi(e) != 0;
  msm_status_t st;
  int prev_dev = -1;
  if (cudaGetDevice(&prev_dev) != cudaSuccess) { prev_dev = -1; cudaGetLastError(); }
  try {
    st = create_impl(params, p);
  } catch (const std::bad_alloc&) {
    st = MSM_ERR_NOMEM;
  } catch (const CudaFail&) {
    st = MSM_ERR_CUDA;
  } catch (...) {
    st = MSM_ERR_CUDA;
  }
  if (st != MSM_OK) {
    cudaGetLastError();
    msm_plan_destroy(p);
    if (prev_dev >= 0) cudaSetDevice(prev_dev);
    return st;
  }
  if (prev_dev >= 0) cudaSetDevice(prev_dev);      // the caller's current device is left as it was
  *plan_out = p;
  return MSM_OK;
}

extern "C" {

msm_status_t msm_plan_info(const msm_plan_t* p, msm_plan_info_t* info) {
  if (!p || !info) return MSM_ERR_INVALID_ARG;
  std::memset(info, 0, sizeof(*info));
  info->L_full = p->H->L;
  info->n_tiled = p->n_t;
  info->mu = p->mu;
  info->omega_halfwidth = p->w;
  for (int l = 1; l <= p->H->L && l <= MSM_MAX_LEVELS; ++l)
    for (int ax = 0; ax < 3; ++ax) {
      info->grid_dims[l - 1][ax] = p->H->lev[l].M[ax];
      info->grid_lo[l - 1][ax] = p->H->lev[l].lo[ax];
      info->grid_h[l - 1][ax] = p->H->lev[l].h[ax];
    }
  for (int l = 1; l < p->n_t; ++l) info->stencil_taps[l - 1] = p->lev[l].taps;
  for (int ax = 0; ax < 3; ++ax) info->pair_cells[ax] = p->bg.nc[ax];
  info->top_points = p->G;
  info->device_bytes = p->bytes;
  return MSM_OK;
}

const char* msm_status_string(msm_status_t s) {
  switch (s) {
    case MSM_OK: return "ok";
    case MSM_ERR_INVALID_ARG: return "invalid argument";
    case MSM_ERR_UNSUPPORTED: return "unsupported configuration";
    case MSM_ERR_CUTOFF_TOO_LARGE: return "cutoff larger than half a periodic box edge";
    case MSM_ERR_TOO_MANY_PARTICLES: return "more particles than the plan's capacity";
    case MSM_ERR_OUT_OF_BOX: return "coordinate outside an open box axis, or non-finite input";
    case MSM_ERR_NOMEM: return "out of memory";
    case MSM_ERR_CUDA: return "CUDA error";
    case MSM_ERR_SCRATCH_LIMIT: return "grids need more than the static scratch array (MSM_NOALLOC_SCRATCH_BYTES)";
  }
  return "unknown status";
}

}  // extern "C"
