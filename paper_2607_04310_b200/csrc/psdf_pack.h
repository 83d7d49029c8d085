// Host-side scene packing (H0; EncodeEdges of Alg.1 l.1-4; eq.(10),
// eq.(17)): padded (A,B,S) -> packed valid-edge records, in
// double, validated against Assumption 1.
#pragma once
#include <cmath>
#include <cstdint>
#include <cstring>
#include <vector>

#include "psdf_device.cuh"

namespace psdf {

struct PackedScene {
  std::vector<EdgeRec> edges;     // grouped by obstacle
  std::vector<int> row_begin;     // [Mv+1]
  std::vector<PairRec> pairs;     // tile-scan records: two edges each, grouped by obstacle
  std::vector<int> pair_begin;    // [Mv+1]
  std::vector<int> empty_rows;
};

// returns 0 ok, -2 degenerate
inline int pack_scene(const float* A, const float* B, const uint8_t* S, int M, int E, PackedScene& out) {
  out.edges.clear();
  out.row_begin.assign(1, 0);
  out.empty_rows.clear();
  std::vector<int> idx;
  for (int i = 0; i < M; ++i) {
    idx.clear();
    for (int j = 0; j < E; ++j)
      if (S[(size_t)i * E + j]) idx.push_back(j);
    const int e = (int)idx.size();
    if (e == 0) { out.empty_rows.push_back(i); continue; }
    if (e < 3) return -2;
    const float* Ai = A + (size_t)i * E * 2;
    const float* Bi = B + (size_t)i * E * 2;
    double area2 = 0.0;
    for (int k = 0; k < e; ++k) {
      const int j = idx[k], jn = idx[(k + 1) % e];
      if (std::memcmp(Bi + 2 * j, Ai + 2 * jn, 2 * sizeof(float)) != 0) return -2;   // not closed
      area2 += (double)Ai[2 * j] * Ai[2 * jn + 1] - (double)Ai[2 * jn] * Ai[2 * j + 1];
    }
    if (!(std::fabs(area2) > 0.0) || !std::isfinite(area2)) return -2;
    const bool ccw = area2 > 0.0;
    const int slot = (int)out.row_begin.size() - 1;
    double ptx = 0, pty = 0;
    for (int k = 0; k <= e; ++k) {     // one extra turn closes the convexity check
      const int j = idx[k % e];
      // CCW-normalised edge: for a clockwise row the edge is traversed backwards (origin B_j).
      const double ox = ccw ? Ai[2 * j] : Bi[2 * j], oy = ccw ? Ai[2 * j + 1] : Bi[2 * j + 1];
      const double qx = ccw ? Bi[2 * j] : Ai[2 * j], qy = ccw ? Bi[2 * j + 1] : Ai[2 * j + 1];
      const double dx = qx - ox, dy = qy - oy;
      const double L2 = dx * dx + dy * dy;
      if (!(L2 >= 1e-12) || !std::isfinite(L2)) return -2;
      const double L = std::sqrt(L2), tx = dx / L, ty = dy / L;
      if (k > 0) {
        // consecutive tangents must turn left (CCW order) or right (CW order, walked backwards)
        const double cr = ccw ? (ptx * ty - pty * tx) : (tx * pty - ty * ptx);
        if (cr < -1e-6) return -2;                                                    // not convex
      }
      ptx = tx; pty = ty;
      if (k == e) break;
      EdgeRec r;
      r.ax = (float)ox; r.ay = (float)oy;
      r.tx = (float)tx; r.ty = (float)ty;
      r.h = (float)(0.5 * L);
      r.last = (k == e - 1) ? i : -1;
      r.slot = slot;
      r.pad = 0.f;
      out.edges.push_back(r);
    }
    out.row_begin.push_back((int)out.edges.size());
  }
  // pair records for the tile-scan kernel
  out.pairs.clear();
  out.pair_begin.assign(1, 0);
  const int Mv = (int)out.row_begin.size() - 1;
  for (int s = 0; s < Mv; ++s) {
    const int b = out.row_begin[s], e = out.row_begin[s + 1];
    for (int k = b; k < e; k += 2) {
      const EdgeRec& r0 = out.edges[k];
      const EdgeRec& r1 = out.edges[k + 1 < e ? k + 1 : k];      // odd count: repeat the last edge
      PairRec pr;
      pr.q0 = make_float4(r0.ax, r0.ay, r0.tx, r0.ty);
      pr.q1 = make_float4(r1.ax, r1.ay, r1.tx, r1.ty);
      const int last = (k + 2 >= e) ? out.edges[e - 1].last : -1;
      float lf, sf;
      std::memcpy(&lf, &last, 4);
      std::memcpy(&sf, &s, 4);
      pr.q2 = make_float4(r0.h, r1.h, lf, sf);
      out.pairs.push_back(pr);
    }
    out.pair_begin.push_back((int)out.pairs.size());
  }
  return 0;
}

// Supported compile-time vertex counts (even: the scan kernel packs vertices in pairs); other V are padded with collinear midpoints
// (splitting an edge changes neither the polygon nor any min/max of eqs.(14)-(22)).
inline int padded_vertex_count(int V) {
  static const int sizes[] = {4, 6, 8, 10, 12, 16};
  for (int s : sizes)
    if (V <= s) return s;
  return -1;
}

// returns 0 ok, -1 invalid, -2 degenerate
inline int pack_footprint(const float* fpv, int V, Footprint& fp, int& Vp) {
  if (V < 3 || V > kMaxV) return -1;
  std::vector<double> x(V), y(V);
  for (int l = 0; l < V; ++l) { x[l] = fpv[2 * l]; y[l] = fpv[2 * l + 1]; if (!std::isfinite(x[l]) || !std::isfinite(y[l])) return -2; }
  double area2 = 0;
  for (int l = 0; l < V; ++l) area2 += x[l] * y[(l + 1) % V] - x[(l + 1) % V] * y[l];
  if (!(area2 > 0.0)) return -2;                                   // CW or empty interior
  for (int l = 0; l < V; ++l) {
    const int a = l, b = (l + 1) % V, c = (l + 2) % V;
    const double e1x = x[b] - x[a], e1y = y[b] - y[a], e2x = x[c] - x[b], e2y = y[c] - y[b];
    const double l1 = std::hypot(e1x, e1y), l2 = std::hypot(e2x, e2y);
    if (!(l1 * l1 >= 1e-12)) return -2;
    if ((e1x * e2y - e1y * e2x) < -1e-6 * l1 * l2) return -2;      // not convex
  }
  Vp = padded_vertex_count(V);
  while ((int)x.size() < Vp) {                                     // split the longest edge
    int best = 0; double bl = -1;
    const int n = (int)x.size();
    for (int l = 0; l < n; ++l) {
      const double d = std::hypot(x[(l + 1) % n] - x[l], y[(l + 1) % n] - y[l]);
      if (d > bl) { bl = d; best = l; }
    }
    const double mx = 0.5 * (x[best] + x[(best + 1) % n]), my = 0.5 * (y[best] + y[(best + 1) % n]);
    x.insert(x.begin() + best + 1, mx);
    y.insert(y.begin() + best + 1, my);
  }
  std::memset(&fp, 0, sizeof(fp));
  double rmax = 0;
  for (int l = 0; l < Vp; ++l) {
    const int b = (l + 1) % Vp;
    const double dx = x[b] - x[l], dy = y[b] - y[l], L = std::hypot(dx, dy);
    const double tx = dx / L, ty = dy / L;
    fp.vx[l] = (float)x[l]; fp.vy[l] = (float)y[l];
    fp.tx[l] = (float)tx; fp.ty[l] = (float)ty;
    fp.h[l] = (float)(0.5 * L);
    fp.cN[l] = (float)(x[l] * (-ty) + y[l] * tx);
    fp.cT[l] = (float)(x[l] * tx + y[l] * ty + 0.5 * L);
    fp.ncN[l] = -fp.cN[l]; fp.ncT[l] = -fp.cT[l]; fp.nh[l] = -fp.h[l];
  }
  for (int l = 0; l < V; ++l) rmax = std::fmax(rmax, std::hypot((double)fpv[2 * l], (double)fpv[2 * l + 1]));
  fp.rmax = (float)rmax;
  return 0;
}

}  // namespace psdf
