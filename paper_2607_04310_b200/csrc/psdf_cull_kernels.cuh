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
constexpr int kObsGridMax = 64;
constexpr int kShortRecords = 3;       // culled kernel: obstacles of up to this many pair records count as short

__device__ __forceinline__ int grid_coord(float v, float v0, float s, int G) {
  return min(max((int)((v - v0) * s), 0), G - 1);      // monotone non-decreasing in v
}

// totals2 = {status, Mv, n_edges, n_pairs} written by the device packer (or null: the host values are used)
__global__ void __launch_bounds__(1024) obstacle_grid_kernel(const float4* __restrict__ bounds, int Mv_host,
                                                             int n_pairs_host, const int* __restrict__ totals2,
                                                             float4* __restrict__ gbounds, int* __restrict__ gcell,
                                                             GridHdr* __restrict__ hdr, float per_cell) {
  __shared__ int cnt[kObsGridMax * kObsGridMax + 1];
  __shared__ float red[5][32];
  __shared__ int wsum[32];
  const int tid = threadIdx.x, lane = tid & 31, wid = tid >> 5;
  const int Mv = totals2 ? (totals2[0] == 0 ? totals2[1] : 0) : Mv_host;
  const int n_pairs = totals2 ? totals2[3] : n_pairs_host;
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
  int G = (int)sqrtf((float)Mv / per_cell);                // ~per_cell obstacles in a cell
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
    float4 b = bounds[2 * i];
    const int at = atomicAdd(&cnt[grid_coord(b.y, y0, sy, G) * G + grid_coord(b.x, x0, sx, G)], 1);
    // grid-ordered copy: w = first pair record (24 bits) | min(number of pair records, 127) << 24
    const int rec = __float_as_int(b.w);
    const int rec_end = i + 1 < Mv ? __float_as_int(bounds[2 * (i + 1)].w) : n_pairs;
    b.w = __int_as_float(rec | (min(rec_end - rec, 127) << 24));
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
//   pieces   thread per pose: the grid rows within ub + R_max + r_R of the pose (a row of the cell
//            rectangle is one contiguous range of the grid-ordered bounds) are cut into pieces of at
//            most eight entries: (pose, first entry, count)
//   circles  lane per piece: bounding-circle test against the piece's pose -> queue 1 of (pose, entry)
//   boxes    lane per queue-1 item: oriented-box separating-axis bound -> pair queue
//   drain    as above
//   tail     value; separated poses take their witness gradient in place, the few penetrating ones are
//            compacted into the first lanes (their branch would otherwise run in every warp for two or
//            three lanes); stores as in the dense kernel (finalize_store).
// Piece list and queues have fixed sizes: a stage that finds its output full stops, the stages
// behind it run, and it resumes where it stopped.
template <int V>
struct __align__(16) PosedSlot {      // one posed footprint in shared memory
  float2 rx[V / 2], ry[V / 2], Tx[V / 2], Ty[V / 2];
  float px, py, pad0, pad1;
};

struct __align__(16) WalkPose {       // what the shared stages need to know about a pose
  float bx, by, cs, sn;               // posed bounding-box centre, rotation
  float ub, ub_pad, rpad;             // upper bound of phi, padded copies for the two tests
  int seed_rec;                       // the seed obstacle (already evaluated)
};

// Dynamic shared memory of one CTA: 440 bytes per pose (four CTAs of 128 poses per SM), what the
// posed footprints leave goes to the piece list and the two queues.
template <int V, int NP>
struct CullShape {
  static constexpr int kPerPose = (int)sizeof(PosedSlot<V>) + (int)sizeof(WalkPose) + 16 + 12 + 4;
  static constexpr int kRest = 440 - kPerPose;
  static constexpr int kPieceMul = kRest >= 192 ? 12 : (kRest >= 96 ? 6 : 4);
  static constexpr int kQ1Mul = kRest >= 192 ? 16 : 8;
  static constexpr int kQ2Mul = kRest >= 192 ? 8 : 4;
  static_assert(kPieceMul * 8 + kQ1Mul * 4 + kQ2Mul * 4 <= kRest, "culled kernel: shared memory budget");
  static constexpr int kPiece = NP * kPieceMul, kQ1 = NP * kQ1Mul, kQ2 = NP * kQ2Mul;
  static constexpr int oPose = 0;
  static constexpr int oWalk = oPose + NP * (int)sizeof(PosedSlot<V>);
  static constexpr int oKd = oWalk + NP * (int)sizeof(WalkPose);
  static constexpr int oK2 = oKd + NP * 8;
  static constexpr int oPiece = oK2 + NP * 8;
  static constexpr int oQ1 = oPiece + kPiece * 8;
  static constexpr int oQ2 = oQ1 + kQ1 * 4;
  static constexpr int oG = oQ2 + kQ2 * 4;
  static constexpr int oPen = oG + NP * 12;
  static constexpr int kBytes = oPen + NP * 4;
};

// NP = poses (= threads) per CTA; NP = 32 makes every warp an independent unit
template <int V, int MODE, int NP>
__global__ void __launch_bounds__(NP) psdf_cull_kernel(const __grid_constant__ Footprint fp,
                                                        const __grid_constant__ EvalParams p) {
  using Sh = CullShape<V, NP>;
  constexpr int kPiece = Sh::kPiece, kQ1 = Sh::kQ1, kQ2 = Sh::kQ2;
  extern __shared__ __align__(16) unsigned char smem[];
  PosedSlot<V>* s_pose = reinterpret_cast<PosedSlot<V>*>(smem + Sh::oPose);
  WalkPose* s_walk = reinterpret_cast<WalkPose*>(smem + Sh::oWalk);
  unsigned long long* s_kd = reinterpret_cast<unsigned long long*>(smem + Sh::oKd);
  unsigned long long* s_k2 = reinterpret_cast<unsigned long long*>(smem + Sh::oK2);
  int2* s_piece = reinterpret_cast<int2*>(smem + Sh::oPiece);   // (first grid entry, pose << 8 | count)
  int* s_q1 = reinterpret_cast<int*>(smem + Sh::oQ1);          // circle survivors: (pose << 24) | grid entry
  int* s_q2 = reinterpret_cast<int*>(smem + Sh::oQ2);          // pairs to evaluate: (pose << 24) | first pair record
  float* s_g = reinterpret_cast<float*>(smem + Sh::oG);        // [NP][3] gradients of the compacted penetrating poses
  int* s_pen = reinterpret_cast<int*>(smem + Sh::oPen);
  __shared__ int s_n1, s_n2[2], s_nl[2], s_npiece, s_npen;  // (two sets of pair-queue counters, used alternately)
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
  if (tid == 0) { s_n1 = 0; s_n2[0] = 0; s_n2[1] = 0; s_nl[0] = 0; s_nl[1] = 0; s_npiece = 0; s_npen = 0; s_stat[0] = 0u; s_stat[1] = 0u; }
  __syncthreads();
  // broad-phase proxies of the posed footprint: its bounding box (centre bx,by; axes (cs,sn),
  // (-sn,cs); half extents fp.bhx, fp.bhy) and the circle of radius fp.rbox around the box centre
  const float bx = fmaf(cs, fp.bcx, fmaf(-sn, fp.bcy, x)), by = fmaf(sn, fp.bcx, fmaf(cs, fp.bcy, y));
  // safety for fp32 rounding: relative 1e-4 on every bound, 1e-4 m absolute, and 4 ulp of the
  // coordinates themselves (the posed box centre is a rounded sum: 1 mm at 2e4 m from the origin)
  const float cpad = 4.8e-7f * fmaxf(fabsf(bx), fabsf(by));
  const float rpad = fp.rbox * 1.0001f + 1e-4f + cpad;    // footprint radius + safety
  const GridHdr& gh = p.grid;                              // by value in the launch parameters (read back at pack time)
  const int G = gh.G;
  const float4* __restrict__ gcirc = p.gbounds;            // (cx, cy, R, first pair record), grid order
  const float4* __restrict__ gobb = p.gbounds + gh.Mv;     // (ux, uy, hx, hy), grid order
  const int* __restrict__ gcell = p.gcell;
  const float4* __restrict__ recs = reinterpret_cast<const float4*>(p.pairs);
  unsigned n_pair = 0, n_edge = 0;

  // evaluates the queued pairs, one per lane: `ns` obstacles of few pair records queued from the front
  // of the pair queue, `nl` longer ones from its back, so that the lanes of a warp mostly run loops of
  // similar length
  auto drain = [&](int ns, int nl) {
    for (int j = tid; j < ns + nl; j += NP) {
      const int pr = s_q2[j < ns ? j : kQ2 - 1 - (j - ns)];
      const int q = (int)((unsigned)pr >> 24);
      const PosedSlot<V>& sp = s_pose[q];
      Posed2<V> P;
#pragma unroll
      for (int l = 0; l < V / 2; ++l) { P.rx[l] = sp.rx[l]; P.ry[l] = sp.ry[l]; P.Tx[l] = sp.Tx[l]; P.Ty[l] = sp.Ty[l]; }
      P.px = sp.px; P.py = sp.py;
      ObstacleAcc<V> acc;
      acc.reset();
      float minD2 = kInf;
      const float4* src = recs + 3 * (size_t)(pr & 0xffffff);
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
        if (V % 4 == 0 && fp.sym) {                        // (uniform)
          edge_step_any<V, true, true>(fp, P, c0, h0, acc, minD2);
          if (h1 >= 0.f) edge_step_any<V, true, true>(fp, P, c1, h1, acc, minD2);
        } else {
          edge_step2<V>(fp, P, c0, h0, acc, minD2);
          if (h1 >= 0.f) edge_step2<V>(fp, P, c1, h1, acc, minD2);
        }
        n_edge += h1 >= 0.f ? 2u : 1u;
        if (last >= 0) break;
      }
      ++n_pair;
      const float depth = acc.depth();
      atomicMax(&s_kd[q], ((unsigned long long)fkey(depth) << 32) | (0xffffffffu - (unsigned)slot));
      atomicMin(&s_k2[q], ((unsigned long long)__float_as_uint(minD2) << 32) | (unsigned)slot);
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
    {
      // first rectangle (it almost always holds an obstacle): the cell ranges of up to four rows are
      // loaded together, then the first four entries of each, so that one pose costs two dependent
      // round trips to L2 here instead of two per row
      const int cx0 = grid_coord(bx - ext, gh.x0, gh.sx, G), cx1 = grid_coord(bx + ext, gh.x0, gh.sx, G);
      const int cy0 = grid_coord(by - ext, gh.y0, gh.sy, G), cy1 = grid_coord(by + ext, gh.y0, gh.sy, G);
      int rs[4], re[4];
#pragma unroll
      for (int u = 0; u < 4; ++u) {
        const int r = min(cy0 + u, cy1);
        rs[u] = __ldg(gcell + r * G + cx0);
        re[u] = (cy0 + u <= cy1) ? __ldg(gcell + r * G + cx1 + 1) : rs[u];
      }
      float4 b[4][4];
#pragma unroll
      for (int u = 0; u < 4; ++u)
#pragma unroll
        for (int v = 0; v < 4; ++v) b[u][v] = __ldg(gcirc + max(min(rs[u] + v, re[u] - 1), 0));
#pragma unroll
      for (int u = 0; u < 4; ++u) {
#pragma unroll
        for (int v = 0; v < 4; ++v) {
          const float dx = b[u][v].x - bx, dy = b[u][v].y - by;
          const float key = fmaf(dx, dx, fmaf(dy, dy, -b[u][v].z * b[u][v].z));
          if (rs[u] + v < re[u] && key < best) { best = key; seed_rec = __float_as_int(b[u][v].w); }   // (record | count << 24)
        }
        scan(rs[u] + 4, re[u]);                            // (rows with more than four entries)
      }
      for (int row = cy0 + 4; row <= cy1; ++row) scan(__ldg(gcell + row * G + cx0), __ldg(gcell + row * G + cx1 + 1));
      px0 = cx0; px1 = cx1; py0 = cy0; py1 = cy1;
      ext *= 2.f;
      if (cx0 == 0 && cy0 == 0 && cx1 == G - 1 && cy1 == G - 1) ext = -1.f;    // the whole grid already
    }
    while (seed_rec < 0 && ext > 0.f) {                    // rare: nothing near, the rectangle doubles
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
      if (cx0 == 0 && cy0 == 0 && cx1 == G - 1 && cy1 == G - 1) break;
      px0 = cx0; px1 = cx1; py0 = cy0; py1 = cy1;
      ext *= 2.f;
    }
  }
  auto push_pair = [&](int q, int w, int set) {            // w = first pair record | count << 24
    const int at = (w >> 24) <= kShortRecords ? atomicAdd(&s_n2[set], 1) : kQ2 - 1 - atomicAdd(&s_nl[set], 1);
    s_q2[at] = (q << 24) | (w & 0xffffff);
  };
  if (seed_rec >= 0) push_pair(tid, seed_rec, 0);
  seed_rec &= seed_rec >= 0 ? 0xffffff : -1;               // from here on: the record index alone
  __syncthreads();
  drain(s_n2[0], s_nl[0]);
  __syncthreads();
  // the pair-queue counter of one round is reset after its drain and used again two rounds later, with
  // barriers in between: no barrier is spent on the reset itself
  if (tid == 0) { s_n2[0] = 0; s_nl[0] = 0; }
  int par = 1;

  // ---- the cell rectangle the seed bound cannot exclude: rows [row, row_end), columns [cx0, cx1]
  int row = 0, row_end = 0, cx0 = 0, cx1 = 0;
  int pi = 0, pe = 0;                                      // entries of the current row not yet cut into pieces
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
    if (active && need >= 0.f) {
      cx0 = grid_coord(bx - need, gh.x0, gh.sx, G); cx1 = grid_coord(bx + need, gh.x0, gh.sx, G);
      row = grid_coord(by - need, gh.y0, gh.sy, G);
      row_end = grid_coord(by + need, gh.y0, gh.sy, G) + 1;
    }
    s_walk[tid] = wp;
  }

  while (true) {
    __syncthreads();                                       // (counters reset, the previous round's reads done)
    // ---- pieces: every pose cuts its remaining rows into pieces of <= 8 entries until the list is full
    bool room = true;
    auto cut = [&]() {                                     // cuts [pi, pe) into pieces; false when the list is full
      if (pi >= pe) return true;
      const int np_ = (pe - pi + 7) >> 3;
      const int base = atomicAdd(&s_npiece, np_);
      const int take = min(np_, max(kPiece - base, 0));
      for (int r = 0; r < take; ++r) s_piece[base + r] = make_int2(pi + 8 * r, (tid << 8) | min(8, pe - pi - 8 * r));
      pi += 8 * take;
      return take == np_;
    };
    room = cut();                                          // (the remainder of a row that did not fit last round)
    while (room && row < row_end) {
      int rs[4], re[4];                                    // the cell ranges of four rows, loaded together
#pragma unroll
      for (int u = 0; u < 4; ++u) {
        const int r = min(row + u, row_end - 1);
        rs[u] = __ldg(gcell + r * G + cx0);
        re[u] = __ldg(gcell + r * G + cx1 + 1);
      }
#pragma unroll
      for (int u = 0; u < 4; ++u) {
        if (room && row < row_end) {
          pi = rs[u]; pe = re[u];
          ++row;
          room = cut();
        }
      }
    }
    const bool pdone = !(row < row_end || pi < pe);
    __syncthreads();
    const int n_piece = min(s_npiece, kPiece);
    // ---- circles: lane per piece (two steps of four entries, loads issued together); resumable when
    // queue 1 fills
    int pc = tid;
    bool cdone = false;
    while (true) {
      for (; pc < n_piece; pc += NP) {
        const int2 pcx = s_piece[pc];
        const int i0 = pcx.x, cnt = pcx.y & 0xff, pose = pcx.y >> 8;
        const WalkPose& wp = s_walk[pose];
        const float wbx = wp.bx, wby = wp.by, wub = wp.ub, wrpad = wp.rpad;
        const int wseed = wp.seed_rec;
        float4 b[8];
#pragma unroll
        for (int u = 0; u < 8; ++u) b[u] = __ldg(gcirc + i0 + min(u, cnt - 1));
        unsigned hit = 0u;
#pragma unroll
        for (int u = 0; u < 8; ++u) {
          const float dx = b[u].x - wbx, dy = b[u].y - wby;
          const float t = (wub + b[u].z) * 1.0001f + wrpad;
          const bool ok = (u < cnt) && !(t < 0.f) && !(fmaf(dx, dx, dy * dy) > t * t) && ((__float_as_int(b[u].w) & 0xffffff) != wseed);
          hit |= ok ? (1u << u) : 0u;
        }
        if (hit) {
          const int c = __popc(hit);
          const int at = atomicAdd(&s_n1, c);
          if (at + c > kQ1) {                              // queue 1 full: this piece again next round
            for (int w = at; w < kQ1; ++w) s_q1[w] = -1;   // reserved, not filled
            break;
          }
          int w = at;
          while (hit) {
            const int u = __ffs(hit) - 1;
            hit &= hit - 1;
            s_q1[w++] = (pose << 24) | (i0 + u);
          }
        }
      }
      cdone = pc >= n_piece;
      __syncthreads();
      // (after the first failed reservation the counter is past the end, so every later one fails
      // too: valid entries, then the failed reservation's blanked slots up to the end)
      const int n1 = min(s_n1, kQ1);
      // ---- boxes: lane per circle survivor, a slice of at most kQ2 survivors at a time -> pair queue
      for (int base = 0; base < n1; base += kQ2) {
        for (int j = base + tid; j < min(base + kQ2, n1); j += NP) {
          const int it = s_q1[j];
          if (it < 0) continue;                            // slot reserved by a failed push
          const int q = (int)((unsigned)it >> 24), entry = it & 0xffffff;
          const WalkPose& wp = s_walk[q];
          const float4 c = __ldg(gcirc + entry);
          const float4 o = __ldg(gobb + entry);            // (ux, uy, hx, hy)
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
          push_pair(q, __float_as_int(c.w), par);
        }
        __syncthreads();
        drain(s_n2[par], s_nl[par]);
        __syncthreads();                                   // (every lane has read the counters and its pairs)
        if (tid == 0) { s_n2[par] = 0; s_nl[par] = 0; }
        par ^= 1;
      }
      if (tid == 0) s_n1 = 0;
      if (__syncthreads_and(cdone)) break;
    }
    if (tid == 0) s_npiece = 0;
    if (__syncthreads_and(pdone)) break;
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
      s_pen[atomicAdd(&s_npen, 1)] = tid;
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
      s_g[3 * q] = gp[0]; s_g[3 * q + 1] = gp[1]; s_g[3 * q + 2] = gp[2];
    }
    __syncthreads();
    if (want && !separated) { g[0] = s_g[3 * tid]; g[1] = s_g[3 * tid + 1]; g[2] = s_g[3 * tid + 2]; }
  }
  if (k < p.N) finalize_store<MODE>(fp, p, n, finite, value, slot, g);
  if (!(MODE & kCoeff)) trajectory_epilogue(p.traj, p.value, blockIdx.x * NP, min(NP, p.N - (int)blockIdx.x * NP));
}

}  // namespace psdf
