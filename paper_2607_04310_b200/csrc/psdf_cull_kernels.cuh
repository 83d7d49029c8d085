// Exact broad-phase culling (beyond the paper).  phi is a minimum
// over obstacles (eq.(6)), so an obstacle whose lower bound on sd^i exceeds an
// upper bound of phi already in hand cannot be the arg-min and cannot change the value:
// skipping it is exact.  Two lower bounds are used, cheapest first:
//     sd^i >= |c_R - c_i| - R_i - r_R            (bounding circles of obstacle and footprint)
//     sd^i >= sd(box_R, box_i)                   (oriented bounding boxes, separating axes)
// Every surviving (pose, obstacle) pair is evaluated with the same arithmetic as the dense
// tile-scan kernel (edge_step2) and reduced with the same keys, so the outputs are
// bit-identical to the dense path.
#pragma once
#include "psdf_kernels.cuh"

namespace psdf {

__device__ __forceinline__ float warp_min_f(float v) { return fkey_inv(__reduce_min_sync(0xffffffffu, fkey(v))); }
__device__ __forceinline__ float warp_max_f(float v) { return fkey_inv(__reduce_max_sync(0xffffffffu, fkey(v))); }

// ------------------------------------------------------------------------------------------
// Obstacle grid: the bounds re-ordered by cell of a G x G grid over the obstacle centres
// (row-major: a rectangle of cells is one contiguous range of `gbounds` per grid row), built on
// the device by one CTA when culling is switched on and after every pack while it is on.
struct GridHdr {
  float x0, y0, sx, sy;    // cell(x) = clamp((int)((x - x0) * sx), 0, G-1)
  float rmax;              // largest bounding-circle radius
  float cell;              // larger cell edge [m]
  int G, Mv;
};
constexpr int kObsGridMax = 64;

__device__ __forceinline__ int grid_coord(float v, float v0, float s, int G) {
  return min(max((int)((v - v0) * s), 0), G - 1);      // monotone non-decreasing in v
}

// totals2 = {status, Mv} written by the device packer (or null: Mv_host is used)
__global__ void __launch_bounds__(1024) obstacle_grid_kernel(const float4* __restrict__ bounds, int Mv_host,
                                                             const int* __restrict__ totals2,
                                                             float4* __restrict__ gbounds, int* __restrict__ gcell,
                                                             GridHdr* __restrict__ hdr) {
  __shared__ int cnt[kObsGridMax * kObsGridMax + 1];
  __shared__ float red[5][32];
  __shared__ int wsum[32];
  const int tid = threadIdx.x, lane = tid & 31, wid = tid >> 5;
  const int Mv = totals2 ? (totals2[0] == 0 ? totals2[1] : 0) : Mv_host;
  float x0 = kInf, y0 = kInf, x1 = -kInf, y1 = -kInf, rm = 0.f;
  for (int i = tid; i < Mv; i += 1024) {
    const float4 b = bounds[2 * i];
    x0 = fminf(x0, b.x); y0 = fminf(y0, b.y); x1 = fmaxf(x1, b.x); y1 = fmaxf(y1, b.y); rm = fmaxf(rm, b.z);
  }
  x0 = warp_min_f(x0); y0 = warp_min_f(y0); x1 = warp_max_f(x1); y1 = warp_max_f(y1); rm = warp_max_f(rm);
  if (lane == 0) { red[0][wid] = x0; red[1][wid] = y0; red[2][wid] = x1; red[3][wid] = y1; red[4][wid] = rm; }
  __syncthreads();
  x0 = warp_min_f(red[0][lane]); y0 = warp_min_f(red[1][lane]);
  x1 = warp_max_f(red[2][lane]); y1 = warp_max_f(red[3][lane]); rm = warp_max_f(red[4][lane]);
  int G = (int)sqrtf(0.5f * (float)Mv);
  G = G < 1 ? 1 : (G > kObsGridMax ? kObsGridMax : G);
  const float wx = fmaxf(x1 - x0, 1e-6f), wy = fmaxf(y1 - y0, 1e-6f);
  const float sx = (float)G / wx, sy = (float)G / wy;
  const int cells = G * G;
  for (int c = tid; c <= cells; c += 1024) cnt[c] = 0;
  __syncthreads();
  for (int i = tid; i < Mv; i += 1024) {
    const float4 b = bounds[2 * i];
    atomicAdd(&cnt[grid_coord(b.y, y0, sy, G) * G + grid_coord(b.x, x0, sx, G)], 1);
  }
  __syncthreads();
  {  // exclusive scan of cnt[0..cells) in place, four cells per thread
    int v[4], sum = 0;
#pragma unroll
    for (int k = 0; k < 4; ++k) { const int c = 4 * tid + k; v[k] = c < cells ? cnt[c] : 0; sum += v[k]; }
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
    for (int k = 0; k < 4; ++k) {
      const int c = 4 * tid + k;
      if (c < cells) { cnt[c] = run; gcell[c] = run; }
      run += v[k];
    }
    if (tid == 0) gcell[cells] = Mv;
  }
  __syncthreads();
  // scatter of the bounds themselves (cnt = cursors).  The order inside a cell is whatever the
  // atomics give: the culled kernel's results do not depend on it (its reductions are arg-min /
  // arg-max keys with the packed slot as tie-break), and a rank pass to make it deterministic would
  // be quadratic in the cell size (every obstacle in one cell: Mv^2 / 1024 steps per thread).
  for (int i = tid; i < Mv; i += 1024) {
    const float4 b = bounds[2 * i];
    const int at = atomicAdd(&cnt[grid_coord(b.y, y0, sy, G) * G + grid_coord(b.x, x0, sx, G)], 1);
    gbounds[at] = b;
    gbounds[Mv + at] = bounds[2 * i + 1];
  }
  if (tid == 0) {
    GridHdr h;
    h.x0 = x0; h.y0 = y0; h.sx = sx; h.sy = sy; h.rmax = rm;
    h.cell = fmaxf(wx, wy) / (float)G;
    h.G = G; h.Mv = Mv;
    *hdr = h;
  }
}


// ------------------------------------------------------------------------------------------
// Culled evaluation over the obstacle grid, pair-queue formulation.  CTA = NP poses, one per
// thread.  Every thread walks the grid cells around ITS pose and pushes the
// obstacles that pass the bounding-circle test as (pose, obstacle) pairs into a shared-memory
// queue; the CTA then evaluates the queued pairs one per lane, whatever pose they belong to
// (the posed footprints sit in shared memory), with the dense kernel's arithmetic (edge_step2),
// and folds each result into its pose's 64-bit arg-max / arg-min keys with shared-memory
// atomics (same keys as the dense kernel: lowest slot on ties).  Two rounds: a seed round (one
// near obstacle per pose) gives every pose a finite upper bound, the main round queues whatever
// that bound cannot exclude.  The last step is the dense kernel's tail (finalize_pose).
template <int V>
struct __align__(16) PosedSlot {      // one posed footprint in shared memory
  float2 rx[V / 2], ry[V / 2], Tx[V / 2], Ty[V / 2];
  float px, py, ub, pad;
};

// NP = poses (= threads) per CTA; NP = 32 makes every warp an independent unit (no block barriers)
template <int V, int MODE, int NP>
__global__ void __launch_bounds__(NP) psdf_cull_kernel(const __grid_constant__ Footprint fp,
                                                        const __grid_constant__ EvalParams p) {
  constexpr int kCullQueue = (NP * 16 * (int)sizeof(int2) + NP * (int)sizeof(PosedSlot<V>) > 44 * 1024) ? NP * 8 : NP * 16;
  __shared__ PosedSlot<V> s_pose[NP];
  __shared__ unsigned long long s_kd[NP], s_k2[NP];
  __shared__ int2 s_queue[kCullQueue];
  __shared__ int s_count;
  __shared__ unsigned int s_stat[2];
  const int tid = threadIdx.x;
  const int k = blockIdx.x * NP + tid;
  const int n = min(k, p.N - 1);                           // tail threads recompute the last pose
  const float x = __ldg(p.poses + 3 * n), y = __ldg(p.poses + 3 * n + 1), th = __ldg(p.poses + 3 * n + 2);
  const bool active = k < p.N && isfinite(x) && isfinite(y) && isfinite(th);
  float sn, cs;
  sincosf(th, &sn, &cs);
  {
    Posed2<V> P;
    pose_setup2_sc<V>(fp, x, y, sn, cs, P);
    PosedSlot<V>& d = s_pose[tid];
#pragma unroll
    for (int l = 0; l < V / 2; ++l) { d.rx[l] = P.rx[l]; d.ry[l] = P.ry[l]; d.Tx[l] = P.Tx[l]; d.Ty[l] = P.Ty[l]; }
    d.px = x; d.py = y;
  }
  s_kd[tid] = 0ull;
  s_k2[tid] = ~0ull;
  if (tid == 0) { s_count = 0; s_stat[0] = 0u; s_stat[1] = 0u; }
  __syncthreads();
  // broad-phase proxies of the posed footprint: its bounding box (centre bx,by; axes (cs,sn),
  // (-sn,cs); half extents fp.bhx, fp.bhy) and the circle of radius fp.rbox around the box centre
  const float bx = fmaf(cs, fp.bcx, fmaf(-sn, fp.bcy, x)), by = fmaf(sn, fp.bcx, fmaf(cs, fp.bcy, y));
  // safety for fp32 rounding: relative 1e-4 on every bound, 1e-4 m absolute, and 4 ulp of the
  // coordinates themselves (the posed box centre is a rounded sum: 1 mm at 2e4 m from the origin)
  const float cpad = 4.8e-7f * fmaxf(fabsf(bx), fabsf(by));
  const float rpad = fp.rbox * 1.0001f + 1e-4f + cpad;    // footprint radius + safety
  const GridHdr gh = *p.ghdr;
  const int G = gh.G;
  const float4* __restrict__ gcirc = p.gbounds;            // (cx, cy, R, first pair record), grid order
  const float4* __restrict__ gobb = p.gbounds + gh.Mv;     // (ux, uy, hx, hy), grid order
  const int* __restrict__ gcell = p.gcell;
  const float4* __restrict__ recs = reinterpret_cast<const float4*>(p.pairs);
  unsigned n_pair = 0, n_edge = 0;

  // evaluates the first nq queued pairs, one per lane
  auto drain = [&](int nq) {
    for (int j = tid; j < nq; j += NP) {
      const int2 pr = s_queue[j];
      const PosedSlot<V>& sp = s_pose[pr.x];
      Posed2<V> P;
#pragma unroll
      for (int l = 0; l < V / 2; ++l) { P.rx[l] = sp.rx[l]; P.ry[l] = sp.ry[l]; P.Tx[l] = sp.Tx[l]; P.Ty[l] = sp.Ty[l]; }
      P.px = sp.px; P.py = sp.py;
      ObstacleAcc<V> acc;
      acc.reset();
      float minD2 = kInf;
      const float4* src = recs + 3 * (size_t)pr.y;
      float4 q0 = __ldg(src), q1 = __ldg(src + 1), q2 = __ldg(src + 2);
      int last, slot;
      while (true) {
        last = __float_as_int(q2.z);
        slot = __float_as_int(q2.w);
        const float4 c0 = q0, c1 = q1;
        const float h0 = q2.x, h1 = q2.y;
        if (last < 0) {                                    // prefetch the next record of this obstacle
          src += 3;
          q0 = __ldg(src); q1 = __ldg(src + 1); q2 = __ldg(src + 2);
        }
        edge_step2<V>(fp, P, c0, h0, acc, minD2);
        if (h1 >= 0.f) edge_step2<V>(fp, P, c1, h1, acc, minD2);
        n_edge += h1 >= 0.f ? 2u : 1u;
        if (last >= 0) break;
      }
      ++n_pair;
      const float depth = acc.depth();
      atomicMax(&s_kd[pr.x], ((unsigned long long)fkey(depth) << 32) | (0xffffffffu - (unsigned)slot));
      atomicMin(&s_k2[pr.x], ((unsigned long long)__float_as_uint(minD2) << 32) | (unsigned)slot);
    }
  };
  // this pose's upper bound of phi from its keys
  auto bound_now = [&]() {
    const unsigned long long kd = s_kd[tid], k2 = s_k2[tid];
    const float depth = kd ? fkey_inv((uint32_t)(kd >> 32)) : -kInf;
    const float d2 = (k2 != ~0ull) ? __uint_as_float((uint32_t)(k2 >> 32)) : kInf;
    return depth >= 0.f ? -depth : sqrtf(d2);
  };

  // ---- seed round: the entry with the smallest (d^2 - R^2) in a growing rectangle of cells
  int seed_rec = -1;
  if (active) {
    float ext = rpad + 0.5f * gh.cell;
    int px0 = 0, px1 = -1, py0 = 0, py1 = -1;
    float best = kInf;
    auto scan = [&](int s, int e) {                        // four independent loads in flight
      for (int i = s; i < e; i += 4) {
        float4 b[4];
#pragma unroll
        for (int u = 0; u < 4; ++u) b[u] = __ldg(gcirc + min(i + u, e - 1));
#pragma unroll
        for (int u = 0; u < 4; ++u) {
          const float dx = b[u].x - bx, dy = b[u].y - by;
          const float key = fmaf(dx, dx, fmaf(dy, dy, -b[u].z * b[u].z));
          if (key < best) { best = key; seed_rec = __float_as_int(b[u].w); }   // (a repeated last entry is harmless)
        }
      }
    };
    while (true) {
      const int cx0 = grid_coord(bx - ext, gh.x0, gh.sx, G), cx1 = grid_coord(bx + ext, gh.x0, gh.sx, G);
      const int cy0 = grid_coord(by - ext, gh.y0, gh.sy, G), cy1 = grid_coord(by + ext, gh.y0, gh.sy, G);
      for (int row = cy0; row <= cy1; ++row) {
        const int s = __ldg(gcell + row * G + cx0), e = __ldg(gcell + row * G + cx1 + 1);
        if (row >= py0 && row <= py1) {                    // skip what the previous rectangle covered
          scan(s, __ldg(gcell + row * G + px0));
          scan(__ldg(gcell + row * G + px1 + 1), e);
        } else {
          scan(s, e);
        }
      }
      if (seed_rec >= 0 || (cx0 == 0 && cy0 == 0 && cx1 == G - 1 && cy1 == G - 1)) break;
      px0 = cx0; px1 = cx1; py0 = cy0; py1 = cy1;
      ext *= 2.f;
    }
  }
  if (seed_rec >= 0) s_queue[atomicAdd(&s_count, 1)] = make_int2(tid, seed_rec);
  __syncthreads();
  drain(s_count);
  __syncthreads();
  if (tid == 0) s_count = 0;
  __syncthreads();

  // ---- main round: everything the seed bound cannot exclude, resumable when the queue fills
  const float ub = active ? bound_now() : -kInf;
  const float need = (ub + gh.rmax) * 1.0001f + rpad;
  const float ub_pad = fmaf(fabsf(ub), 1e-4f, ub) + 2e-4f + cpad;
  bool done = !active || !(need >= 0.f);
  int cx0 = 0, cx1 = 0, cy1 = -1, row = 0, i = 0, e = 0;
  if (!done) {
    cx0 = grid_coord(bx - need, gh.x0, gh.sx, G); cx1 = grid_coord(bx + need, gh.x0, gh.sx, G);
    row = grid_coord(by - need, gh.y0, gh.sy, G) - 1; cy1 = grid_coord(by + need, gh.y0, gh.sy, G);
  }
  while (true) {
    while (!done) {
      if (i >= e) {
        if (++row > cy1) { done = true; break; }
        i = __ldg(gcell + row * G + cx0);
        e = __ldg(gcell + row * G + cx1 + 1);
        continue;
      }
      float4 b[4];
#pragma unroll
      for (int u = 0; u < 4; ++u) b[u] = __ldg(gcirc + min(i + u, e - 1));   // four independent loads in flight
      bool full = false;
#pragma unroll
      for (int u = 0; u < 4; ++u) {
        if (full || i + u >= e) continue;
        const float dx = b[u].x - bx, dy = b[u].y - by;
        const float t = (ub + b[u].z) * 1.0001f + rpad;
        if ((t < 0.f) || (fmaf(dx, dx, dy * dy) > t * t) || __float_as_int(b[u].w) == seed_rec) continue;
        // box-box separating-axis bound: sd(boxes) = max over the four box axes of the gap of the
        // projections (exact when they overlap, a lower bound of the distance otherwise), and
        // sd(footprint, obstacle) >= sd(boxes) because each polygon lies inside its box
        const float4 o = __ldg(gobb + i + u);              // (ux, uy, hx, hy)
        const float a1 = fabsf(fmaf(o.x, cs, o.y * sn)), a2 = fabsf(fmaf(o.y, cs, -o.x * sn));
        const float g0 = fabsf(fmaf(dx, o.x, dy * o.y)) - (o.z + fmaf(fp.bhx, a1, fp.bhy * a2));
        const float g1 = fabsf(fmaf(dy, o.x, -dx * o.y)) - (o.w + fmaf(fp.bhx, a2, fp.bhy * a1));
        const float g2 = fabsf(fmaf(dx, cs, dy * sn)) - (fp.bhx + fmaf(o.z, a1, o.w * a2));
        const float g3 = fabsf(fmaf(dy, cs, -dx * sn)) - (fp.bhy + fmaf(o.z, a2, o.w * a1));
        if (fmaxf(fmaxf(g0, g1), fmaxf(g2, g3)) > ub_pad) continue;
        const int at = atomicAdd(&s_count, 1);
        if (at >= kCullQueue) { full = true; i += u; continue; }   // queue full: retry this entry next round
        s_queue[at] = make_int2(tid, __float_as_int(b[u].w));
      }
      if (full) break;
      i += 4;
    }
    __syncthreads();
    const int nq = min(s_count, kCullQueue);
    drain(nq);
    __syncthreads();
    if (tid == 0) s_count = 0;
    if (__syncthreads_and(done)) break;
  }

  if (p.stats) {
    atomicAdd(&s_stat[0], n_pair);
    atomicAdd(&s_stat[1], n_edge);
    __syncthreads();
    if (tid == 0) {
      atomicAdd(p.stats, (unsigned long long)s_stat[0]);
      atomicAdd(p.stats + 1, (unsigned long long)s_stat[1]);
    }
  }
  if (k >= p.N) return;
  const unsigned long long kd = s_kd[tid], k2 = s_k2[tid];
  const float maxDepth = kd ? fkey_inv((uint32_t)(kd >> 32)) : -kInf;
  const int idDepth = kd ? (int)(0xffffffffu - (uint32_t)kd) : -1;
  const float minD2 = (k2 != ~0ull) ? __uint_as_float((uint32_t)(k2 >> 32)) : kInf;
  const int idD2 = (k2 != ~0ull) ? (int)(uint32_t)k2 : -1;
  const bool separated = !(maxDepth >= 0.f);
  const float value = separated ? sqrtf(minD2) : -maxDepth;
  Posed<V> Ps;
  {
    const PosedSlot<V>& sp = s_pose[tid];
    Ps.px = x; Ps.py = y;
#pragma unroll
    for (int l = 0; l < V / 2; ++l) {
      Ps.rx[2 * l] = sp.rx[l].x; Ps.rx[2 * l + 1] = sp.rx[l].y; Ps.ry[2 * l] = sp.ry[l].x; Ps.ry[2 * l + 1] = sp.ry[l].y;
      Ps.Tx[2 * l] = sp.Tx[l].x; Ps.Tx[2 * l + 1] = sp.Tx[l].y; Ps.Ty[2 * l] = sp.Ty[l].x; Ps.Ty[2 * l + 1] = sp.Ty[l].y;
    }
  }
  finalize_pose<V, MODE>(fp, p, Ps, n, th, value, separated ? idD2 : idDepth, separated);
}

}  // namespace psdf
