// Exact broad-phase culling (beyond the paper).  phi is a minimum
// over obstacles (eq.(6)), so an obstacle whose lower bound
//     sd^i >= |p - c_i| - R_i - r_max          (bounding circles of obstacle and footprint)
// exceeds an upper bound of phi already in hand cannot be the arg-min and cannot change the
// value: skipping it is exact.  The culled path evaluates every surviving (pose, obstacle)
// pair with the same arithmetic as the dense tile-scan kernel (edge_step2), so its outputs
// are bit-identical to the dense path.
//
//   * poses are bucketed into a uniform grid (counting sort: bbox -> histogram -> scan ->
//     scatter) so that the 32 poses of a warp are spatially close;
//   * one warp owns 32 sorted poses and walks the obstacle bounds 32 at a time: lane j tests
//     obstacle j against the warp's pose box and its largest running upper bound (one test per
//     obstacle per WARP), the ballot gives the survivors, each survivor is re-tested per lane
//     and evaluated only if some lane still needs it; records are read straight from L2/L1
//     with warp-uniform 128-bit loads (no shared memory, no block barriers);
//   * the running upper bound is the exact value over the obstacles evaluated so far.
#pragma once
#include "psdf_kernels.cuh"

namespace psdf {

constexpr int kSortGridMax = 64;      // pose grid is G x G cells, G <= 64

__device__ __forceinline__ float warp_min_f(float v) { return fkey_inv(__reduce_min_sync(0xffffffffu, fkey(v))); }
__device__ __forceinline__ float warp_max_f(float v) { return fkey_inv(__reduce_max_sync(0xffffffffu, fkey(v))); }

struct SortParams {
  const float* poses;
  int N, G;
  unsigned int* bbox;      // [4] ordered keys: min x, min y, ~max x, ~max y  (all atomicMin; clean = 0xff..)
  int* cell;               // [G*G + 1] histogram -> offsets -> cursors
  int* perm;               // [N] sorted position -> pose index
};

__device__ __forceinline__ bool pose_finite(float x, float y) { return isfinite(x) && isfinite(y); }

__global__ void __launch_bounds__(256) pose_bbox_kernel(const SortParams s) {
  __shared__ float red[4][8];
  float x0 = kInf, y0 = kInf, x1 = -kInf, y1 = -kInf;
  for (int n = blockIdx.x * blockDim.x + threadIdx.x; n < s.N; n += gridDim.x * blockDim.x) {
    const float x = __ldg(s.poses + 3 * n), y = __ldg(s.poses + 3 * n + 1);
    if (pose_finite(x, y)) { x0 = fminf(x0, x); y0 = fminf(y0, y); x1 = fmaxf(x1, x); y1 = fmaxf(y1, y); }
  }
  x0 = warp_min_f(x0); y0 = warp_min_f(y0); x1 = warp_max_f(x1); y1 = warp_max_f(y1);
  const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
  if (lane == 0) { red[0][wid] = x0; red[1][wid] = y0; red[2][wid] = x1; red[3][wid] = y1; }
  __syncthreads();
  if (wid == 0) {                                         // one atomic per quantity per block
    const int nw = blockDim.x >> 5;
    x0 = warp_min_f(lane < nw ? red[0][lane] : kInf); y0 = warp_min_f(lane < nw ? red[1][lane] : kInf);
    x1 = warp_max_f(lane < nw ? red[2][lane] : -kInf); y1 = warp_max_f(lane < nw ? red[3][lane] : -kInf);
    if (lane == 0) {
      atomicMin(s.bbox + 0, fkey(x0)); atomicMin(s.bbox + 1, fkey(y0));
      atomicMin(s.bbox + 2, ~fkey(x1)); atomicMin(s.bbox + 3, ~fkey(y1));
    }
  }
}

__device__ __forceinline__ int pose_cell(const SortParams& s, int n) {
  const float x = __ldg(s.poses + 3 * n), y = __ldg(s.poses + 3 * n + 1);
  if (!pose_finite(x, y)) return 0;
  const float x0 = fkey_inv(s.bbox[0]), y0 = fkey_inv(s.bbox[1]);
  const float x1 = fkey_inv(~s.bbox[2]), y1 = fkey_inv(~s.bbox[3]);
  const float sx = (float)s.G / fmaxf(x1 - x0, 1e-6f), sy = (float)s.G / fmaxf(y1 - y0, 1e-6f);
  const int gx = min(max((int)((x - x0) * sx), 0), s.G - 1);
  int gy = min(max((int)((y - y0) * sy), 0), s.G - 1);
  if (gx & 1) gy = s.G - 1 - gy;                          // snake order: neighbours stay neighbours
  return gx * s.G + gy;
}

// exclusive scan of the (<= 4096) cell counts, in place, by one CTA of 1024 threads
__device__ __forceinline__ void scan_cells(int* cell, int cells) {
  __shared__ int wsum[32];
  const int tid = threadIdx.x, lane = tid & 31, wid = tid >> 5;
  int v[4], sum = 0;
#pragma unroll
  for (int k = 0; k < 4; ++k) { const int c = 4 * tid + k; v[k] = c < cells ? __ldcg(cell + c) : 0; sum += v[k]; }
  int inc = sum;
#pragma unroll
  for (int o = 1; o < 32; o <<= 1) { const int t = __shfl_up_sync(0xffffffffu, inc, o); if (lane >= o) inc += t; }
  if (lane == 31) wsum[wid] = inc;
  __syncthreads();
  if (wid == 0) {
    const int w = wsum[lane];
    int winc = w;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) { const int t = __shfl_up_sync(0xffffffffu, winc, o); if (lane >= o) winc += t; }
    wsum[lane] = winc - w;
  }
  __syncthreads();
  int run = wsum[wid] + inc - sum;
#pragma unroll
  for (int k = 0; k < 4; ++k) { const int c = 4 * tid + k; if (c < cells) cell[c] = run; run += v[k]; }
}

// histogram of the pose cells; the last block to arrive turns the counts into offsets
// (cell[G*G] is the arrival counter).  block = 1024 threads.
__global__ void __launch_bounds__(1024) pose_hist_kernel(const SortParams s) {
  __shared__ int is_last;
  const int n = blockIdx.x * blockDim.x + threadIdx.x;
  {  // warp-aggregated: neighbouring poses (same trajectory) share a cell, one atomic per distinct cell
    const int c = n < s.N ? pose_cell(s, n) : -1;
    const unsigned peers = __match_any_sync(0xffffffffu, c);
    if (c >= 0 && (int)(__ffs(peers) - 1) == (int)(threadIdx.x & 31)) atomicAdd(s.cell + c, __popc(peers));
  }
  __threadfence();
  __syncthreads();
  if (threadIdx.x == 0) is_last = atomicAdd(s.cell + s.G * s.G, 1) == (int)gridDim.x - 1;
  __syncthreads();
  if (!is_last) return;
  __threadfence();
  scan_cells(s.cell, s.G * s.G);
}

__global__ void pose_scatter_kernel(const SortParams s) {
  const int n = blockIdx.x * blockDim.x + threadIdx.x;
  const int lane = threadIdx.x & 31;
  const int c = n < s.N ? pose_cell(s, n) : -1;
  const unsigned peers = __match_any_sync(0xffffffffu, c);          // warp-aggregated cursor bump
  const int leader = __ffs(peers) - 1;
  int base = 0;
  if (c >= 0 && leader == lane) base = atomicAdd(s.cell + c, __popc(peers));
  base = __shfl_sync(0xffffffffu, base, leader);
  if (c >= 0) s.perm[base + __popc(peers & ((1u << lane) - 1u))] = n;
}

// Per-obstacle bound, one float4 per packed obstacle: bounding circle (cx, cy, R) of its
// vertices and the index of its first pair record (int bits).
//
// Culled evaluation: one warp (= one CTA) per 32 sorted poses, lane = pose.  MODE in
// {0, kGrad, kCoeff}.  The workspace left dirty by the pose sort is cleaned here for the next
// call.  (Several warps per pose group sharing the running bound were measured: never faster.)
template <int V, int MODE>
__global__ void __launch_bounds__(32) psdf_cull_kernel(const __grid_constant__ Footprint fp,
                                                        const __grid_constant__ EvalParams p) {
  const int lane = threadIdx.x & 31;
#ifdef PSDF_CULL_LOG
  const long long t_start = clock64();
#endif
  {  // clean the sort workspace (its last reader, pose_scatter_kernel, has completed)
    const int t = blockIdx.x * blockDim.x + threadIdx.x;
    if (t <= p.sort_cells) p.sort_cell[t] = 0;
    if (t < 4) p.sort_bbox[t] = 0xffffffffu;
  }
  const int k = blockIdx.x * 32 + lane;
  const int n = __ldg(p.perm + min(k, p.N - 1));           // tail lanes recompute the last pose
  const float x = __ldg(p.poses + 3 * n), y = __ldg(p.poses + 3 * n + 1), th = __ldg(p.poses + 3 * n + 2);
  const bool finite = isfinite(x) && isfinite(y) && isfinite(th);
  Posed2<V> P;
  pose_setup2<V>(fp, x, y, th, P);
  // pose box of the 32 poses (non-finite poses take no part; they are finalised to NaN)
  const float xmin = warp_min_f(finite ? x : kInf), xmax = warp_max_f(finite ? x : -kInf);
  const float ymin = warp_min_f(finite ? y : kInf), ymax = warp_max_f(finite ? y : -kInf);
  const float rpad = fp.rmax * 1.0001f + 1e-4f;            // footprint radius + safety for fp32 rounding

  ObstacleAcc<V> acc;
  float minD2 = kInf, prevD2 = kInf, maxDepth = -kInf;
  float ub = finite ? kInf : -kInf;                        // running upper bound of phi for this lane
  int idD2 = -1, idDepth = -1;
  unsigned n_visit = 0, n_edge = 0;                        // statistics (psdf_cull_stats)
  const float4* __restrict__ bounds = p.bounds;
  const float4* __restrict__ recs = reinterpret_cast<const float4*>(p.pairs);

  // evaluates one obstacle for the whole warp if some lane still needs it (exact per-lane test)
  auto visit = [&](const float cx, const float cy, const float R, const int rec) {
    const float dx = cx - x, dy = cy - y;
    const float t = (ub + R) * 1.0001f + rpad;
    const bool need = !((t < 0.f) || (fmaf(dx, dx, dy * dy) > t * t));
    if (!__any_sync(0xffffffffu, need)) return;
    acc.reset();
    const float4* src = recs + 3 * (size_t)rec;
    float4 q0 = __ldg(src), q1 = __ldg(src + 1), q2 = __ldg(src + 2);
    int last, slot;
    while (true) {
      last = __float_as_int(q2.z);
      slot = __float_as_int(q2.w);
      const float4 c0 = q0, c1 = q1;
      const float h0 = q2.x, h1 = q2.y;
      if (last < 0) {                                      // prefetch the next record of this obstacle
        src += 3;
        q0 = __ldg(src); q1 = __ldg(src + 1); q2 = __ldg(src + 2);
      }
      edge_step2<V>(fp, P, c0, h0, acc, minD2);
      if (h1 >= 0.f) edge_step2<V>(fp, P, c1, h1, acc, minD2);
      n_edge += h1 >= 0.f ? 2u : 1u;
      if (last >= 0) break;
    }
    ++n_visit;
    const float depth = acc.depth();
    if (MODE & (kGrad | kCoeff)) {
      if (minD2 < prevD2) { prevD2 = minD2; idD2 = slot; }
    }
    if (depth > maxDepth) { maxDepth = depth; idDepth = slot; }
    if (finite) {
      const float nub = fminf(ub, maxDepth >= 0.f ? -maxDepth : sqrtf(minD2));
      ub = nub;
    }
  };
  // squared distance from an obstacle centre to the pose box of the warp
  auto box_d2 = [&](const float4 b) {
    const float ddx = fmaxf(fmaxf(xmin - b.x, b.x - xmax), 0.f), ddy = fmaxf(fmaxf(ymin - b.y, b.y - ymax), 0.f);
    return fmaf(ddx, ddx, ddy * ddy);
  };

  // Phase A: the two obstacles nearest to the pose box go first, so that the running upper
  // bound is tight before the memory-order walk (evaluated obstacles per warp drop ~2x).
  int first0 = -1, first1 = -1;
  {
    unsigned k0 = 0xffffffffu, k1 = 0xffffffffu;           // this lane's two smallest keys
    int i0 = -1, i1 = -1;
    // (ordering heuristic only: squared box distance minus squared radius, no sqrt)
#pragma unroll 4
    for (int i = lane; i < p.Mv; i += 32) {
      const float4 b = __ldg(bounds + i);
      const unsigned key = fkey(box_d2(b) - b.z * b.z);
      if (key < k0) { k1 = k0; i1 = i0; k0 = key; i0 = i; }
      else if (key < k1) { k1 = key; i1 = i; }
    }
#pragma unroll
    for (int r = 0; r < 2; ++r) {
      const unsigned m = __reduce_min_sync(0xffffffffu, k0);
      const int owner = __ffs(__ballot_sync(0xffffffffu, k0 == m && i0 >= 0)) - 1;
      if (owner < 0) break;
      const int idx = __shfl_sync(0xffffffffu, i0, owner);
      if (lane == owner) { k0 = k1; i0 = i1; k1 = 0xffffffffu; i1 = -1; }
      if (r == 0) first0 = idx; else first1 = idx;
      const float4 b = __ldg(bounds + idx);
      visit(b.x, b.y, b.z, __float_as_int(b.w));
    }
  }

#ifdef PSDF_CULL_LOG
  const long long t_phaseA = clock64();
#endif
  // Phase B: memory-order walk, 4 x 32 obstacles per step (four independent loads, tests and
  // ballots in flight: the walk is latency bound): one box test per obstacle per warp.  A
  // survivor of a stale warp-level bound is still re-tested per lane inside visit().
  for (int base = 0; base < p.Mv; base += 128) {
    float4 b[4];
    unsigned mask[4];
#pragma unroll
    for (int u = 0; u < 4; ++u) {
      const int i = base + 32 * u + lane;
      b[u] = i < p.Mv ? __ldg(bounds + i) : make_float4(0.f, 0.f, 0.f, 0.f);
    }
    const float ubmax = warp_max_f(ub);
#pragma unroll
    for (int u = 0; u < 4; ++u) {
      const int i = base + 32 * u + lane;
      const float thr = (ubmax + b[u].z) * 1.0001f + rpad;
      const bool skip = (i >= p.Mv) || (i == first0) || (i == first1) || (thr < 0.f) || (box_d2(b[u]) > thr * thr);
      mask[u] = __ballot_sync(0xffffffffu, !skip);
    }
    if ((mask[0] | mask[1] | mask[2] | mask[3]) == 0u) continue;
#pragma unroll 1
    for (int u = 0; u < 4; ++u) {
      const float4 bu = u == 0 ? b[0] : (u == 1 ? b[1] : (u == 2 ? b[2] : b[3]));
      unsigned m = u == 0 ? mask[0] : (u == 1 ? mask[1] : (u == 2 ? mask[2] : mask[3]));
      while (m) {
        const int j = __ffs(m) - 1;
        m &= m - 1;
        visit(__shfl_sync(0xffffffffu, bu.x, j), __shfl_sync(0xffffffffu, bu.y, j), __shfl_sync(0xffffffffu, bu.z, j),
              __shfl_sync(0xffffffffu, __float_as_int(bu.w), j));
      }
    }
  }
#ifdef PSDF_CULL_LOG
  if (p.stats && lane == 0) {   // per-warp log after the two counters: (cycles, visits, tA, tB)
    unsigned long long* lg = p.stats + 2 + 4 * (size_t)blockIdx.x;
    lg[0] = clock64() - t_start; lg[1] = n_visit; lg[2] = t_phaseA - t_start; lg[3] = clock64() - t_phaseA;
  }
#endif
  if (p.stats && lane == 0) {
    atomicAdd(p.stats, (unsigned long long)n_visit);
    atomicAdd(p.stats + 1, (unsigned long long)n_edge);
  }
  if (!(MODE & (kGrad | kCoeff))) idD2 = minD2 < kInf ? 0 : -1;
  if (k >= p.N) return;
  const bool separated = !(maxDepth >= 0.f);
  const float value = separated ? sqrtf(minD2) : -maxDepth;
  Posed<V> Ps;
  unpack_pose<V>(P, Ps);
  finalize_pose<V, MODE>(fp, p, Ps, n, th, value, separated ? idD2 : idDepth, separated);
}

}  // namespace psdf
