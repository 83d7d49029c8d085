// Reductions on top of the PSDF outputs:
//   * components: non-convex obstacles are given as several convex components (Assumption 1,
//     PAPER.md:62; eq.(6) PAPER.md:93-97 minimises over all components); per-component values sd^i
//     fold into per-obstacle values through a component -> obstacle id map.  Fused form: the
//     per-obstacle epilogue of the evaluation kernels (ComponentFold, psdf_set_components) writes
//     [N, n_obstacles] directly, no [N, M] array in between; stand-alone form: component_min_kernel
//     over a materialised [N, M] array and an arbitrary map;
//   * trajectories: sampled-trajectory batches (N = T trajectories x H stages, pose index =
//     traj * H + stage): clearance min_s phi_s with its first arg-min stage and the soft penalty
//     sum_s max(0, d_safe - phi_s)^2, one warp per trajectory, fixed reduction order
//     (deterministic).  Fused form: trajectory_epilogue at the end of the evaluation kernels (the
//     CTA that completes a trajectory reduces it, same routine, same bits); stand-alone form:
//     trajectory_reduce_kernel.
#pragma once
#include "psdf_device.cuh"

namespace psdf {

// ---- components ------------------------------------------------------------------------------
// Stand-alone: one CTA per pose; keys (order-preserving uint32 of the float) are min-reduced in place
// in the output row, then turned back into floats: O(M + n_obstacles) per pose for any map.  Ids
// outside [0, n_obstacles) are ignored.
__global__ void __launch_bounds__(128) component_min_kernel(const float* __restrict__ per_component, int N, int M,
                                                            const int* __restrict__ comp_to_obstacle, int n_obstacles,
                                                            float* __restrict__ out) {
  const int n = blockIdx.x;
  unsigned int* row = reinterpret_cast<unsigned int*>(out + (size_t)n * n_obstacles);
  const float* src = per_component + (size_t)n * M;
  for (int o = threadIdx.x; o < n_obstacles; o += blockDim.x) row[o] = fkey(kInf);
  __syncthreads();
  for (int i = threadIdx.x; i < M; i += blockDim.x) {
    const int o = __ldg(comp_to_obstacle + i);
    if (o >= 0 && o < n_obstacles) atomicMin(row + o, fkey(__ldg(src + i)));
  }
  __syncthreads();
  for (int o = threadIdx.x; o < n_obstacles; o += blockDim.x) out[(size_t)n * n_obstacles + o] = fkey_inv(row[o]);
}

// Fused: running minimum over the components of one obstacle while the scan walks the packed
// obstacles in row order (the components of an obstacle are consecutive rows: psdf_set_components).
// Every (pose, obstacle) entry of [first_group, end_group) is written exactly once: the minimum when
// the next obstacle begins, +INF for obstacles without a valid component in between.
struct ComponentFold {
  float* row;        // out + n * n_obstacles (or null: this thread writes nothing)
  int first;         // first obstacle of this CTA's range
  int cur;           // obstacle whose components are being folded (first - 1 before the first)
  float m;
  __device__ __forceinline__ void begin(float* out_row, int first_group) { row = out_row; first = first_group; cur = first_group - 1; m = kInf; }
  __device__ __forceinline__ void add(int group, float sd) {
    if (group != cur) {
      if (row) {
        if (cur >= first) row[cur] = m;
        for (int g = cur + 1; g < group; ++g) row[g] = kInf;
      }
      cur = group;
      m = kInf;
    }
    m = fminf(m, sd);
  }
  __device__ __forceinline__ void end(int end_group) {
    if (!row) return;
    if (cur >= first) row[cur] = m;
    for (int g = cur + 1; g < end_group; ++g) row[g] = kInf;
  }
};

// ---- trajectories ----------------------------------------------------------------------------
// One warp reduces trajectory t of `value` [T*H]; all 32 lanes call it.  COHERENT: the values were
// written by other CTAs of the same launch (read past L1).
template <bool COHERENT>
__device__ __forceinline__ void trajectory_reduce_warp(const float* __restrict__ value, int t, int H, float d_safe,
                                                       float* __restrict__ min_value, int* __restrict__ argmin_stage,
                                                       float* __restrict__ penalty) {
  const int lane = threadIdx.x & 31;
  const float* v = value + (size_t)t * H;
  unsigned long long best = ~0ull;          // (ordered key of phi) << 32 | stage: min = first arg-min
  float pen = 0.f;
  for (int s = lane; s < H; s += 32) {
    const float phi = COHERENT ? __ldcg(v + s) : __ldg(v + s);
    const unsigned long long key = ((unsigned long long)fkey(phi) << 32) | (unsigned)s;
    best = key < best ? key : best;
    const float d = fmaxf(d_safe - phi, 0.f);
    pen = fmaf(d, d, pen);
  }
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) {
    const unsigned long long other = __shfl_xor_sync(0xffffffffu, best, o);
    best = other < best ? other : best;
    pen += __shfl_xor_sync(0xffffffffu, pen, o);
  }
  if (lane == 0) {
    if (min_value) min_value[t] = H > 0 ? fkey_inv((uint32_t)(best >> 32)) : kInf;
    if (argmin_stage) argmin_stage[t] = H > 0 ? (int)(uint32_t)best : -1;
    if (penalty) penalty[t] = pen;
  }
}

__global__ void trajectory_reduce_kernel(const float* __restrict__ value, int T, int H, float d_safe,
                                         float* __restrict__ min_value, int* __restrict__ argmin_stage,
                                         float* __restrict__ penalty) {
  const int t = (blockIdx.x * blockDim.x + threadIdx.x) >> 5;
  if (t >= T) return;
  trajectory_reduce_warp<false>(value, t, H, d_safe, min_value, argmin_stage, penalty);
}

struct TrajParams {
  int H;                       // stages per trajectory (0 = no trajectory epilogue)
  float d_safe;
  float* min_value;            // [T] or null
  int* argmin_stage;           // [T] or null
  float* penalty;              // [T] or null
  unsigned int* count;         // [T] arrival counters (clean = 0, left clean)
};

// Tail of an evaluation kernel, called by ALL threads of a CTA (blockDim a multiple of 32) that has
// just stored value[n0 .. n0 + cnt): the poses are counted into their trajectories' arrival
// counters, and the warp that completes a trajectory reduces it (values of other CTAs are visible:
// their fence precedes their count).  Same routine as the stand-alone kernel: same bits.
__device__ __forceinline__ void trajectory_epilogue(const TrajParams& tp, const float* __restrict__ value, int n0, int cnt) {
  if (tp.H <= 0 || cnt <= 0) return;
  __threadfence();
  __syncthreads();
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, n_warps = blockDim.x >> 5;
  const int t0 = n0 / tp.H, t1 = (n0 + cnt - 1) / tp.H;
  for (int t = t0 + warp; t <= t1; t += n_warps) {
    int done = 0;
    if (lane == 0) {
      const int lo = max(n0, t * tp.H), hi = min(n0 + cnt, (t + 1) * tp.H);
      const unsigned here = (unsigned)(hi - lo);
      done = atomicAdd(tp.count + t, here) + here == (unsigned)tp.H;
      if (done) { tp.count[t] = 0u; __threadfence(); }
    }
    done = __shfl_sync(0xffffffffu, done, 0);
    if (done) trajectory_reduce_warp<true>(value, t, tp.H, tp.d_safe, tp.min_value, tp.argmin_stage, tp.penalty);
  }
}

}  // namespace psdf
