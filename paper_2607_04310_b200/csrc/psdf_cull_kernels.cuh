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
// Culled evaluation over the obstacle grid.  CTA = NP poses.  The work of a pose is irregular (its
// upper bound decides how many grid cells it has to look at, its neighbourhood how many obstacles
// survive), so every stage hands its output to the WHOLE CTA through shared memory and the next
// stage runs one item per lane, whatever pose it belongs to:
//   seed     thread per pose: the nearest bounding circle in a small rectangle of cells -> pair queue
//   drain    lane per queued (pose, obstacle) pair: the dense kernel's arithmetic (edge_step2), result
//            folded into the pose's 64-bit arg-max / arg-min keys with shared-memory atomics (the
//            dense kernel's keys: lowest slot on ties); every pose now has a finite upper bound ub
//   rows     thread per pose: the grid rows within ub + R_max + r_R of the pose go into a segment
//            list, one (pose, row) per entry: a row of the cell rectangle is one contiguous range of
//            the grid-ordered bounds
//   circles  lane per segment: bounding-circle test of its entries against the segment's pose ->
//            queue 1 of (pose, entry)
//   boxes    lane per queue-1 item: oriented-box separating-axis bound -> pair queue
//   drain    as above
//   tail     value; separated poses take their witness gradient in place, the few penetrating ones are
//            compacted into the first lanes (their branch would otherwise run in every warp for two or
//            three lanes); stores as in the dense kernel (finalize_store).
// Queues and the segment list have fixed sizes: a stage that finds its output full stops, the
// stages behind it run, and it resumes where it stopped.
template <int V>
struct __align__(16) PosedSlot {      // one posed footprint in shared memory
  float2 rx[V / 2], ry[V / 2], Tx[V / 2], Ty[V / 2];
  float px, py, pad0, pad1;
};

struct __align__(16) WalkPose {       // what the shared stages need to know about a pose
  float bx, by, cs, sn;               // posed bounding-box centre, rotation
  float ub, ub_pad, rpad;             // upper bound of phi, padded copies for the two tests
  int seed_rec;                       // the seed obstacle (already evaluated)
  int cx0, cx1, pad0, pad1;           // columns of the cell rectangle
};

template <int V, int NP>
struct CullShape {
  // queue entries: as many as fit next to the posed footprints in 48 KB of static shared memory
  static constexpr int kFixed = NP * ((int)sizeof(PosedSlot<V>) + (int)sizeof(WalkPose) + 16 + 12 + 2) + NP * 8 * 2 + 64;
  static constexpr int kQueue = (kFixed + NP * 8 * 16 <= 48 * 1024 - 256) ? NP * 8 : NP * 4;
  static constexpr int kSeg = NP * 8;
  static_assert(kFixed + kQueue * 16 <= 48 * 1024 - 256, "culled kernel: static shared memory budget");
};

// NP = poses (= threads) per CTA; NP = 32 makes every warp an independent unit
template <int V, int MODE, int NP>
__global__ void __launch_bounds__(NP) psdf_cull_kernel(const __grid_constant__ Footprint fp,
                                                        const __grid_constant__ EvalParams p) {
  constexpr int kQueue = CullShape<V, NP>::kQueue, kSeg = CullShape<V, NP>::kSeg;
  __shared__ PosedSlot<V> s_pose[NP];
  __shared__ WalkPose s_walk[NP];
  __shared__ unsigned long long s_kd[NP], s_k2[NP];
  __shared__ int2 s_q1[kQueue];          // circle survivors: (pose, grid entry)
  __shared__ int2 s_q2[kQueue];          // pairs to evaluate: (pose, first pair record)
  __shared__ unsigned short s_seg[kSeg]; // (pose << 6) | grid row
  __shared__ float s_g[NP][3];           // gradients of the compacted penetrating poses
  __shared__ unsigned short s_pen[NP];
  __shared__ int s_n1, s_n2, s_nseg, s_npen;
  __shared__ unsigned int s_stat[2];
  const int tid = threadIdx.x;
  const int k = blockIdx.x * NP + tid;
  const int n = min(k, p.N - 1);                           // tail threads recompute the last pose
  const float x = __ldg(p.poses + 3 * n), y = __ldg(p.poses + 3 * n + 1), th = __ldg(p.poses + 3 * n + 2);
  const bool finite = isfinite(x) && isfinite(y) && isfinite(th);
  const bool active = k < p.N && finite;
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
  if (tid == 0) { s_n1 = 0; s_n2 = 0; s_nseg = 0; s_npen = 0; s_stat[0] = 0u; s_stat[1] = 0u; }
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
      const int2 pr = s_q2[j];
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

  // ---- seed: the entry with the smallest (d^2 - R^2) in a growing rectangle of cells
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
  if (seed_rec >= 0) s_q2[atomicAdd(&s_n2, 1)] = make_int2(tid, seed_rec);
  __syncthreads();
  drain(s_n2);
  __syncthreads();

  // ---- rows: the cell rectangle the seed bound cannot exclude
  int row_next = 0, n_rows = 0;
  {
    float ub = -kInf;
    if (active) {
      const unsigned long long kd = s_kd[tid], k2 = s_k2[tid];
      const float depth = kd ? fkey_inv((uint32_t)(kd >> 32)) : -kInf;
      const float d2 = (k2 != ~0ull) ? __uint_as_float((uint32_t)(k2 >> 32)) : kInf;
      ub = depth >= 0.f ? -depth : sqrtf(d2);
    }
    const float need = (ub + gh.rmax) * 1.0001f + rpad;
    WalkPose wp;
    wp.bx = bx; wp.by = by; wp.cs = cs; wp.sn = sn;
    wp.ub = ub; wp.ub_pad = fmaf(fabsf(ub), 1e-4f, ub) + 2e-4f + cpad; wp.rpad = rpad;
    wp.seed_rec = seed_rec;
    wp.cx0 = wp.cx1 = wp.pad0 = wp.pad1 = 0;
    if (active && need >= 0.f) {
      wp.cx0 = grid_coord(bx - need, gh.x0, gh.sx, G); wp.cx1 = grid_coord(bx + need, gh.x0, gh.sx, G);
      row_next = grid_coord(by - need, gh.y0, gh.sy, G);
      n_rows = grid_coord(by + need, gh.y0, gh.sy, G) - row_next + 1;
    }
    s_walk[tid] = wp;
  }
  if (tid == 0) s_n2 = 0;

  while (true) {
    __syncthreads();                                       // (s_nseg = 0 and the previous round's reads are done)
    // every pose appends as many of its remaining rows as fit into the segment list
    if (n_rows > 0) {
      const int base = atomicAdd(&s_nseg, n_rows);
      const int take = min(n_rows, max(kSeg - base, 0));
      for (int r = 0; r < take; ++r) s_seg[base + r] = (unsigned short)((tid << 6) | (row_next + r));
      row_next += take;
      n_rows -= take;
    }
    __syncthreads();
    const int n_seg = min(s_nseg, kSeg);
    // ---- circles: lane per segment, resumable when queue 1 fills
    int seg = tid, i = 0, e = 0, pose = 0;
    float wbx = 0.f, wby = 0.f, wub = 0.f, wrpad = 0.f;
    int wseed = -1;
    bool cdone = false;
    while (true) {
      while (!cdone) {
        if (i >= e) {
          if (seg >= n_seg) { cdone = true; break; }
          const int sv = s_seg[seg];
          seg += NP;
          pose = sv >> 6;
          const WalkPose& wp = s_walk[pose];
          const int row = sv & 63;
          i = __ldg(gcell + row * G + wp.cx0);
          e = __ldg(gcell + row * G + wp.cx1 + 1);
          wbx = wp.bx; wby = wp.by; wub = wp.ub; wrpad = wp.rpad; wseed = wp.seed_rec;
          continue;
        }
        float4 b[4];
#pragma unroll
        for (int u = 0; u < 4; ++u) b[u] = __ldg(gcirc + min(i + u, e - 1));   // four independent loads in flight
        unsigned hit = 0u;
#pragma unroll
        for (int u = 0; u < 4; ++u) {
          const float dx = b[u].x - wbx, dy = b[u].y - wby;
          const float t = (wub + b[u].z) * 1.0001f + wrpad;
          const bool ok = (i + u < e) && !(t < 0.f) && !(fmaf(dx, dx, dy * dy) > t * t) && (__float_as_int(b[u].w) != wseed);
          hit |= ok ? (1u << u) : 0u;
        }
        if (hit) {
          const int cnt = __popc(hit);
          const int at = atomicAdd(&s_n1, cnt);
          if (at + cnt > kQueue) {                         // queue 1 full: these four entries again next round
            for (int w = at; w < kQueue; ++w) s_q1[w] = make_int2(0, -1);   // reserved, not filled
            break;
          }
          int w = at;
#pragma unroll
          for (int u = 0; u < 4; ++u)
            if (hit & (1u << u)) s_q1[w++] = make_int2(pose, i + u);
        }
        i += 4;
      }
      __syncthreads();
      // (after the first failed reservation the counter is past the end, so every later one fails
      // too: valid entries, then the failed reservation's blanked slots up to the end)
      const int n1 = min(s_n1, kQueue);
      // ---- boxes: lane per circle survivor
      for (int j = tid; j < n1; j += NP) {
        const int2 it = s_q1[j];
        if (it.y < 0) continue;                            // slot reserved by a failed push
        const WalkPose& wp = s_walk[it.x];
        const float4 c = __ldg(gcirc + it.y);
        const float4 o = __ldg(gobb + it.y);               // (ux, uy, hx, hy)
        const float dx = c.x - wp.bx, dy = c.y - wp.by, pcs = wp.cs, psn = wp.sn;
        // box-box separating-axis bound: sd(boxes) = max over the four box axes of the gap of the
        // projections (exact when they overlap, a lower bound of the distance otherwise), and
        // sd(footprint, obstacle) >= sd(boxes) because each polygon lies inside its box
        const float a1 = fabsf(fmaf(o.x, pcs, o.y * psn)), a2 = fabsf(fmaf(o.y, pcs, -o.x * psn));
        const float g0 = fabsf(fmaf(dx, o.x, dy * o.y)) - (o.z + fmaf(fp.bhx, a1, fp.bhy * a2));
        const float g1 = fabsf(fmaf(dy, o.x, -dx * o.y)) - (o.w + fmaf(fp.bhx, a2, fp.bhy * a1));
        const float g2 = fabsf(fmaf(dx, pcs, dy * psn)) - (fp.bhx + fmaf(o.z, a1, o.w * a2));
        const float g3 = fabsf(fmaf(dy, pcs, -dx * psn)) - (fp.bhy + fmaf(o.z, a2, o.w * a1));
        if (fmaxf(fmaxf(g0, g1), fmaxf(g2, g3)) > wp.ub_pad) continue;
        s_q2[atomicAdd(&s_n2, 1)] = make_int2(it.x, __float_as_int(c.w));   // (never more than n1 <= kQueue)
      }
      __syncthreads();
      drain(s_n2);
      __syncthreads();
      if (tid == 0) { s_n1 = 0; s_n2 = 0; }
      if (__syncthreads_and(cdone)) break;
    }
    if (tid == 0) s_nseg = 0;
    if (__syncthreads_and(n_rows == 0)) break;
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
  // ---- tail: value, witness gradient (penetrating poses compacted into the first lanes), stores
  const unsigned long long kd = s_kd[tid], k2 = s_k2[tid];
  const float maxDepth = kd ? fkey_inv((uint32_t)(kd >> 32)) : -kInf;
  const int idDepth = kd ? (int)(0xffffffffu - (uint32_t)kd) : -1;
  const float minD2 = (k2 != ~0ull) ? __uint_as_float((uint32_t)(k2 >> 32)) : kInf;
  const int idD2 = (k2 != ~0ull) ? (int)(uint32_t)k2 : -1;
  const bool separated = !(maxDepth >= 0.f);
  const float value = separated ? sqrtf(minD2) : -maxDepth;
  const int slot = separated ? idD2 : idDepth;
  auto posed_of = [&](int q, Posed<V>& Ps) {
    const PosedSlot<V>& sp = s_pose[q];
    Ps.px = sp.px; Ps.py = sp.py;
#pragma unroll
    for (int l = 0; l < V / 2; ++l) {
      Ps.rx[2 * l] = sp.rx[l].x; Ps.rx[2 * l + 1] = sp.rx[l].y; Ps.ry[2 * l] = sp.ry[l].x; Ps.ry[2 * l + 1] = sp.ry[l].y;
      Ps.Tx[2 * l] = sp.Tx[l].x; Ps.Tx[2 * l + 1] = sp.Tx[l].y; Ps.Ty[2 * l] = sp.Ty[l].x; Ps.Ty[2 * l + 1] = sp.Ty[l].y;
    }
  };
  float g[3] = {0.f, 0.f, 0.f};
  if (MODE & (kGrad | kCoeff)) {
    const bool want = active && slot >= 0;
    if (want && !separated) {                              // queue this pose for the compacted pass
      s_pen[atomicAdd(&s_npen, 1)] = (unsigned short)tid;
      s_walk[tid].seed_rec = __float_as_int(__ldg(&p.bounds[2 * slot].w));   // (the walk is over: reuse the field)
    }
    if (want && separated) {
      Posed<V> Ps;
      posed_of(tid, Ps);
      witness_separated<V>(fp, Ps, recs, __float_as_int(__ldg(&p.bounds[2 * slot].w)), g);
    }
    __syncthreads();
    if (tid < s_npen) {
      const int q = s_pen[tid];
      Posed<V> Ps;
      posed_of(q, Ps);
      float gp[3];
      witness_penetrating<V>(fp, Ps, recs, s_walk[q].seed_rec, gp);
      s_g[q][0] = gp[0]; s_g[q][1] = gp[1]; s_g[q][2] = gp[2];
    }
    __syncthreads();
    if (want && !separated) { g[0] = s_g[tid][0]; g[1] = s_g[tid][1]; g[2] = s_g[tid][2]; }
  }
  if (k >= p.N) return;
  finalize_store<MODE>(fp, p, n, finite, value, slot, g);
}

}  // namespace psdf
