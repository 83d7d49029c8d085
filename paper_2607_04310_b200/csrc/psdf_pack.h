// Host-side scene packing (H0; EncodeEdges of Alg.1 l.1-4; eq.(10),
// eq.(17)): padded (A,B,S) -> packed valid-edge records, in
// double, validated against Assumption 1.
#pragma once
#include <algorithm>
#include <atomic>
#include <cmath>
#include <cstdint>
#include <cstring>
#include <thread>
#include <vector>

#include "psdf_device.cuh"

namespace psdf {

struct PackedScene {
  std::vector<EdgeRec> edges;     // grouped by obstacle
  std::vector<int> row_begin;     // [Mv+1]
  std::vector<PairRec> pairs;     // tile-scan records: two edges each, grouped by obstacle
  std::vector<int> pair_begin;    // [Mv+1]
  std::vector<int> empty_rows;
  std::vector<float4> bounds;     // [2 Mv] per obstacle: bounding circle + first pair record, oriented box
  std::vector<int> row_slot;      // [M+1] non-empty rows before each row
};

// Double-precision helpers that round identically on host and device: nvcc contracts a*b+c
// into FMA in device code, the host compiler does not, so the device side uses the
// never-contracted intrinsics.  This makes the device pack kernel (psdf_pack_kernels.cuh)
// bit-identical to the host packer.
#ifdef __CUDA_ARCH__
#define PSDF_HD __host__ __device__ __forceinline__
__device__ __forceinline__ double pk_mul(double a, double b) { return __dmul_rn(a, b); }
__device__ __forceinline__ double pk_add(double a, double b) { return __dadd_rn(a, b); }
__device__ __forceinline__ double pk_sub(double a, double b) { return __dsub_rn(a, b); }
__device__ __forceinline__ double pk_div(double a, double b) { return __ddiv_rn(a, b); }
__device__ __forceinline__ double pk_sqrt(double a) { return __dsqrt_rn(a); }
#else
#ifdef __CUDACC__
#define PSDF_HD __host__ __device__ inline
#else
#define PSDF_HD inline
#endif
inline double pk_mul(double a, double b) { return a * b; }
inline double pk_add(double a, double b) { return a + b; }
inline double pk_sub(double a, double b) { return a - b; }
inline double pk_div(double a, double b) { return a / b; }
inline double pk_sqrt(double a) { return std::sqrt(a); }
#endif

PSDF_HD bool pk_same_point(const float* p, const float* q) {      // bitwise, like memcmp
  const uint32_t* a = reinterpret_cast<const uint32_t*>(p);
  const uint32_t* b = reinterpret_cast<const uint32_t*>(q);
  return a[0] == b[0] && a[1] == b[1];
}
PSDF_HD bool pk_finite(double x) { return x - x == 0.0; }

// One obstacle row of (A,B,S): validates Assumption 1 (closed, convex, non-degenerate) and,
// if `out` is non-null, writes its `*e_out` EdgeRec records (CCW-normalised) to out[0..e).
// returns 0 ok (e may be 0: absent obstacle), -2 degenerate.
PSDF_HD int pack_row(const float* Ai, const float* Bi, const uint8_t* Si, int E, int row, int slot,
                     EdgeRec* out, int* e_out) {
  int e = 0, first = -1;
  for (int j = 0; j < E; ++j)
    if (Si[j]) { if (first < 0) first = j; ++e; }
  *e_out = e;
  if (e == 0) return 0;
  if (e < 3) return -2;
  auto next_valid = [&](int j) {
    for (int q = j + 1; q < E; ++q) if (Si[q]) return q;
    return first;
  };
  double area2 = 0.0;
  for (int k = 0, j = first; k < e; ++k) {
    const int jn = next_valid(j);
    if (!pk_same_point(Bi + 2 * j, Ai + 2 * jn)) return -2;                              // not closed
    area2 = pk_add(area2, pk_sub(pk_mul((double)Ai[2 * j], (double)Ai[2 * jn + 1]),
                                 pk_mul((double)Ai[2 * jn], (double)Ai[2 * j + 1])));
    j = jn;
  }
  if (!(area2 > 0.0 || area2 < 0.0) || !pk_finite(area2)) return -2;
  const bool ccw = area2 > 0.0;
  double ptx = 0, pty = 0;
  for (int k = 0, j = first; k <= e; ++k) {   // one extra turn closes the convexity check
    // CCW-normalised edge: for a clockwise row the edge is traversed backwards (origin B_j).
    const double ox = ccw ? Ai[2 * j] : Bi[2 * j], oy = ccw ? Ai[2 * j + 1] : Bi[2 * j + 1];
    const double qx = ccw ? Bi[2 * j] : Ai[2 * j], qy = ccw ? Bi[2 * j + 1] : Ai[2 * j + 1];
    const double dx = pk_sub(qx, ox), dy = pk_sub(qy, oy);
    const double L2 = pk_add(pk_mul(dx, dx), pk_mul(dy, dy));
    if (!(L2 >= 1e-12) || !pk_finite(L2)) return -2;
    const double L = pk_sqrt(L2), tx = pk_div(dx, L), ty = pk_div(dy, L);
    if (k > 0) {
      // consecutive tangents must turn left (CCW order) or right (CW order, walked backwards)
      const double cr = ccw ? pk_sub(pk_mul(ptx, ty), pk_mul(pty, tx)) : pk_sub(pk_mul(tx, pty), pk_mul(ty, ptx));
      if (cr < -1e-6) return -2;                                                         // not convex
    }
    ptx = tx; pty = ty;
    if (k == e) break;
    if (out) {
      EdgeRec r;
      r.ax = (float)ox; r.ay = (float)oy;
      r.tx = (float)tx; r.ty = (float)ty;
      r.h = (float)pk_mul(0.5, L);
      r.last = (k == e - 1) ? row : -1;
      r.slot = slot;
      r.pad = 0.f;
      out[k] = r;
    }
    j = next_valid(j);
  }
  return 0;
}

// Pair record k2 (edges 2*k2, 2*k2+1) of an obstacle with e edge records `er`.
PSDF_HD PairRec make_pair_rec(const EdgeRec* er, int e, int k2, int slot) {
  const int k = 2 * k2;
  const EdgeRec r0 = er[k];
  const EdgeRec r1 = er[k + 1 < e ? k + 1 : k];                    // odd count: second half unused
  PairRec pr;
  pr.q0 = make_float4(r0.ax, r0.ay, r0.tx, r0.ty);
  pr.q1 = make_float4(r1.ax, r1.ay, r1.tx, r1.ty);
  const int last = (k + 2 >= e) ? er[e - 1].last : -1;
  pr.q2 = make_float4(r0.h, k + 1 < e ? r1.h : -1.f, __builtin_bit_cast(float, last),
                      __builtin_bit_cast(float, slot));            // h1 < 0: no second edge
  return pr;
}

// Bounds of an obstacle for the culled path (psdf_cull_kernels.cuh), two float4:
//   obb  = (ux, uy, hx, hy): the smallest-area box among those aligned with one of the
//          obstacle's own edges: axis u (unit), half extents along u and rot90(u);
//   circ = (cx, cy, R, first pair record): box centre and the radius of the circle around it
//          that holds every vertex.
// Extents and radius are measured from the float-rounded centre/axis and rounded up.
struct ObstacleBound { float4 circ, obb; };
PSDF_HD ObstacleBound obstacle_bound(const EdgeRec* er, int e, int pair_begin) {
  double best_area = 0.0, b_lt = 0, b_ht = 0, b_ln = 0, b_hn = 0;
  int best = -1;
  for (int k = 0; k < e; ++k) {
    const double tx = er[k].tx, ty = er[k].ty;
    double lt = 0, ht = 0, ln = 0, hn = 0;
    for (int m = 0; m < e; ++m) {
      const double x = er[m].ax, y = er[m].ay;
      const double pt = pk_add(pk_mul(x, tx), pk_mul(y, ty)), pn = pk_sub(pk_mul(y, tx), pk_mul(x, ty));
      if (m == 0) { lt = ht = pt; ln = hn = pn; }
      lt = pt < lt ? pt : lt; ht = pt > ht ? pt : ht;
      ln = pn < ln ? pn : ln; hn = pn > hn ? pn : hn;
    }
    const double area = pk_mul(pk_sub(ht, lt), pk_sub(hn, ln));
    if (best < 0 || area < best_area) { best = k; best_area = area; b_lt = lt; b_ht = ht; b_ln = ln; b_hn = hn; }
  }
  const float ux = er[best].tx, uy = er[best].ty;
  const double mt = pk_mul(0.5, pk_add(b_lt, b_ht)), mn = pk_mul(0.5, pk_add(b_ln, b_hn));
  const float cx = (float)pk_sub(pk_mul(mt, (double)ux), pk_mul(mn, (double)uy));
  const float cy = (float)pk_add(pk_mul(mt, (double)uy), pk_mul(mn, (double)ux));
  double hx = 0.0, hy = 0.0, r2 = 0.0;
  for (int k = 0; k < e; ++k) {
    const double dx = pk_sub((double)er[k].ax, (double)cx), dy = pk_sub((double)er[k].ay, (double)cy);
    double a = pk_add(pk_mul(dx, (double)ux), pk_mul(dy, (double)uy));
    double b = pk_sub(pk_mul(dy, (double)ux), pk_mul(dx, (double)uy));
    a = a < 0 ? -a : a; b = b < 0 ? -b : b;
    hx = a > hx ? a : hx; hy = b > hy ? b : hy;
    const double d2 = pk_add(pk_mul(dx, dx), pk_mul(dy, dy));
    r2 = d2 > r2 ? d2 : r2;
  }
  ObstacleBound ob;
  ob.circ = make_float4(cx, cy, (float)pk_add(pk_mul(pk_sqrt(r2), 1.000001), 1e-6), __builtin_bit_cast(float, pair_begin));
  ob.obb = make_float4(ux, uy, (float)pk_add(pk_mul(hx, 1.000001), 1e-6), (float)pk_add(pk_mul(hy, 1.000001), 1e-6));
  return ob;
}

// Host packer.  returns 0 ok, -2 degenerate
inline int pack_scene(const float* A, const float* B, const uint8_t* S, int M, int E, PackedScene& out) {
  // pass 1: valid-edge counts -> offsets (what the device packer's scan kernel does)
  out.row_slot.assign((size_t)M + 1, 0);
  out.row_begin.assign(1, 0);
  out.pair_begin.assign(1, 0);
  out.empty_rows.clear();
  std::vector<int> cnt((size_t)M);
  for (int i = 0; i < M; ++i) {
    int e = 0;
    for (int j = 0; j < E; ++j) e += S[(size_t)i * E + j] ? 1 : 0;
    cnt[i] = e;
    out.row_slot[i] = (int)out.row_begin.size() - 1;
    if (e == 0) { out.empty_rows.push_back(i); continue; }
    out.row_begin.push_back(out.row_begin.back() + e);
    out.pair_begin.push_back(out.pair_begin.back() + (e + 1) / 2);
  }
  const int Mv = (int)out.row_begin.size() - 1;
  out.row_slot[M] = Mv;
  out.edges.assign((size_t)out.row_begin.back(), EdgeRec{});
  out.pairs.assign((size_t)out.pair_begin.back(), PairRec{});
  out.bounds.assign(2 * (size_t)Mv, float4{});
  // pass 2: rows are independent; large scenes are split over a few threads
  std::atomic<int> status{0};
  auto work = [&](int i0, int i1) {
    for (int i = i0; i < i1 && status.load(std::memory_order_relaxed) == 0; ++i) {
      const int slot = out.row_slot[i];
      EdgeRec* er = cnt[i] ? out.edges.data() + out.row_begin[slot] : nullptr;
      int e = 0;
      if (pack_row(A + (size_t)i * E * 2, B + (size_t)i * E * 2, S + (size_t)i * E, E, i, slot, er, &e) != 0) {
        status.store(-2);
        return;
      }
      if (e == 0) continue;
      const int pb = out.pair_begin[slot];
      const ObstacleBound ob = obstacle_bound(er, e, pb);
      out.bounds[2 * (size_t)slot] = ob.circ;
      out.bounds[2 * (size_t)slot + 1] = ob.obb;
      for (int k2 = 0; k2 < (e + 1) / 2; ++k2) out.pairs[(size_t)pb + k2] = make_pair_rec(er, e, k2, slot);
    }
  };
  const int n_thr = M >= 512 ? (int)std::min<unsigned>(8u, std::max(1u, std::thread::hardware_concurrency())) : 1;
  if (n_thr == 1) {
    work(0, M);
  } else {
    std::vector<std::thread> pool;
    for (int t = 0; t < n_thr; ++t) pool.emplace_back(work, (int)((long long)M * t / n_thr), (int)((long long)M * (t + 1) / n_thr));
    for (auto& th : pool) th.join();
  }
  return status.load();
}

// Supported compile-time vertex counts (even: the kernels pack vertices in pairs); other V are
// padded with copies of the last vertex (pack_footprint; changes neither the polygon nor any
// min/max of eqs.(14)-(22)).
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
  std::memset(&fp, 0, sizeof(fp));
  double rmax = 0;
  // The Vp - V padding vertices repeat the LAST vertex: the edges between the copies have zero
  // length and borrow the tangent of the last-but-one real edge, so they add only duplicates of
  // candidates and axes that exist already (a vertex distance, a face depth) and no new
  // vertex-region / edge-region boundary.  (Splitting an edge at its midpoint would: at long range
  // fp32 cannot tell the two collinear halves apart and the witness snaps to the artificial vertex.)
  for (int l = 0; l < Vp; ++l) {
    const int a = l < V ? l : V - 1;                                  // start vertex of edge l
    const bool closing = l == Vp - 1, zero = l >= V - 1 && !closing;
    const int ea = zero ? V - 2 : (closing ? V - 1 : l);              // the real edge that lends its tangent
    const int eb = (ea + 1) % V;
    const double dx = x[eb] - x[ea], dy = y[eb] - y[ea], L = std::hypot(dx, dy);
    const double tx = dx / L, ty = dy / L, h = zero ? 0.0 : 0.5 * L;
    fp.vx[l] = (float)x[a]; fp.vy[l] = (float)y[a];
    fp.tx[l] = (float)tx; fp.ty[l] = (float)ty;
    fp.h[l] = (float)h;
    fp.cN[l] = (float)(x[a] * (-ty) + y[a] * tx);
    fp.cT[l] = (float)(x[a] * tx + y[a] * ty + h);
    fp.ncN[l] = -fp.cN[l]; fp.ncT[l] = -fp.cT[l]; fp.nh[l] = -fp.h[l];
  }
  // centrally symmetric about the reference point (v_{l+V/2} == -v_l bitwise; no padding vertices; V a
  // multiple of 4 so that mirrored vertices sit in mirrored f32x2 pairs): the kernels take edge_step2_sym
  fp.sym = (V == Vp && V % 4 == 0) ? 1 : 0;
  for (int l = 0; fp.sym && l < V / 2; ++l)
    if (fpv[2 * (l + V / 2)] != -fpv[2 * l] || fpv[2 * (l + V / 2) + 1] != -fpv[2 * l + 1]) fp.sym = 0;
  for (int l = 0; fp.sym && l < V / 2; ++l)      // (the derived constants mirror exactly; checked, not assumed)
    if (fp.tx[l + V / 2] != -fp.tx[l] || fp.ty[l + V / 2] != -fp.ty[l] || fp.h[l + V / 2] != fp.h[l] ||
        fp.cN[l + V / 2] != fp.cN[l] || fp.cT[l + V / 2] != fp.cT[l]) fp.sym = 0;
  for (int l = 0; l < V; ++l) rmax = std::fmax(rmax, std::hypot((double)fpv[2 * l], (double)fpv[2 * l + 1]));
  fp.rmax = (float)rmax;
  // robot-frame bounding box and the circle around its centre (culled path), rounded up
  double x0 = x[0], x1 = x[0], y0 = y[0], y1 = y[0];
  for (int l = 1; l < V; ++l) { x0 = std::fmin(x0, x[l]); x1 = std::fmax(x1, x[l]); y0 = std::fmin(y0, y[l]); y1 = std::fmax(y1, y[l]); }
  fp.bcx = (float)(0.5 * (x0 + x1)); fp.bcy = (float)(0.5 * (y0 + y1));
  double hx = 0, hy = 0, rb = 0;
  for (int l = 0; l < V; ++l) {
    hx = std::fmax(hx, std::fabs(x[l] - (double)fp.bcx)); hy = std::fmax(hy, std::fabs(y[l] - (double)fp.bcy));
    rb = std::fmax(rb, std::hypot(x[l] - (double)fp.bcx, y[l] - (double)fp.bcy));
  }
  fp.bhx = (float)(hx * 1.000001 + 1e-6); fp.bhy = (float)(hy * 1.000001 + 1e-6); fp.rbox = (float)(rb * 1.000001 + 1e-6);
  return 0;
}

}  // namespace psdf
