// On-device EncodeEdges (Alg.1 l.1-4; eq.(10)): padded
// (A,B,S) already resident in HBM -> packed EdgeRec / PairRec records, without a host
// round trip.  Three small kernels:
//   pack_count_kernel   one thread per obstacle row: validates Assumption 1
//                       with the same double arithmetic as the host packer (pack_row) and
//                       writes the row's valid-edge count; any violation lowers *status;
//   pack_scan_kernel    one CTA: exclusive scans of (slot, edge, pair, empty) offsets;
//   pack_write_kernel   one thread per row: writes the records, row_begin, pair_begin and
//                       the empty-row list at the scanned offsets.
// The records go to the scene's INACTIVE buffer set and the host flips the sets only if *status
// is still 0 after its single synchronisation, so a rejected update leaves the old scene in force.
#pragma once
#include "psdf_pack.h"

namespace psdf {

struct PackTotals {
  int status;      // 0 ok, -2 degenerate
  int Mv;          // rows with >= 1 valid edge
  int n_edges;
  int n_pairs;
  int n_empty;
  int pad[3];
};

__global__ void pack_count_kernel(const float* __restrict__ A, const float* __restrict__ B,
                                  const uint8_t* __restrict__ S, int M, int E, int* __restrict__ count,
                                  PackTotals* __restrict__ totals) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= M) return;
  int e = 0;
  const int rc = pack_row(A + (size_t)i * E * 2, B + (size_t)i * E * 2, S + (size_t)i * E, E, i, 0, nullptr, &e);
  count[i] = e;
  if (rc != 0) atomicMin(&totals->status, rc);
}

// Exclusive scan over the rows by a single CTA of 1024 threads (M is small: <= a few 1e5).
// offs[i] = (slot, first edge, first pair, index among the empty rows).
__global__ void __launch_bounds__(1024) pack_scan_kernel(const int* __restrict__ count, int M,
                                                         int4* __restrict__ offs, PackTotals* __restrict__ totals) {
  __shared__ int4 warp_sum[32];
  __shared__ int4 carry;
  const int tid = threadIdx.x, lane = tid & 31, wid = tid >> 5;
  if (tid == 0) carry = make_int4(0, 0, 0, 0);
  __syncthreads();
  for (int base = 0; base < M; base += 1024) {
    const int i = base + tid;
    const int e = i < M ? count[i] : 0;
    int4 v = make_int4(e > 0 ? 1 : 0, e, (e + 1) >> 1, (i < M && e == 0) ? 1 : 0);
    int4 inc = v;                                         // inclusive warp scan
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
      const int a = __shfl_up_sync(0xffffffffu, inc.x, o), b = __shfl_up_sync(0xffffffffu, inc.y, o);
      const int c = __shfl_up_sync(0xffffffffu, inc.z, o), d = __shfl_up_sync(0xffffffffu, inc.w, o);
      if (lane >= o) { inc.x += a; inc.y += b; inc.z += c; inc.w += d; }
    }
    if (lane == 31) warp_sum[wid] = inc;
    __syncthreads();
    if (wid == 0) {
      int4 w = warp_sum[lane];
      int4 winc = w;
#pragma unroll
      for (int o = 1; o < 32; o <<= 1) {
        const int a = __shfl_up_sync(0xffffffffu, winc.x, o), b = __shfl_up_sync(0xffffffffu, winc.y, o);
        const int c = __shfl_up_sync(0xffffffffu, winc.z, o), d = __shfl_up_sync(0xffffffffu, winc.w, o);
        if (lane >= o) { winc.x += a; winc.y += b; winc.z += c; winc.w += d; }
      }
      warp_sum[lane] = make_int4(winc.x - w.x, winc.y - w.y, winc.z - w.z, winc.w - w.w);   // exclusive
    }
    __syncthreads();
    const int4 wb = warp_sum[wid], cb = carry;
    if (i < M)
      offs[i] = make_int4(cb.x + wb.x + inc.x - v.x, cb.y + wb.y + inc.y - v.y, cb.z + wb.z + inc.z - v.z,
                          cb.w + wb.w + inc.w - v.w);
    __syncthreads();
    if (tid == 1023) carry = make_int4(cb.x + wb.x + inc.x, cb.y + wb.y + inc.y, cb.z + wb.z + inc.z, cb.w + wb.w + inc.w);
    __syncthreads();
  }
  if (tid == 0) {
    totals->Mv = carry.x;
    totals->n_edges = carry.y;
    totals->n_pairs = carry.z;
    totals->n_empty = carry.w;
  }
}

__global__ void pack_write_kernel(const float* __restrict__ A, const float* __restrict__ B,
                                  const uint8_t* __restrict__ S, int M, int E, const int* __restrict__ count,
                                  const int4* __restrict__ offs, const PackTotals* __restrict__ totals,
                                  EdgeRec* __restrict__ edges, PairRec* __restrict__ pairs,
                                  int* __restrict__ row_begin, int* __restrict__ pair_begin,
                                  int* __restrict__ empty_rows, float4* __restrict__ bounds,
                                  int* __restrict__ row_slot) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (totals->status != 0) return;                    // rejected: the host will not flip the buffers
  if (i == 0) {
    row_begin[totals->Mv] = totals->n_edges;
    pair_begin[totals->Mv] = totals->n_pairs;
    row_slot[M] = totals->Mv;
  }
  if (i >= M) return;
  const int4 o = offs[i];
  row_slot[i] = o.x;
  int e = count[i];
  if (e == 0) { empty_rows[o.w] = i; return; }
  EdgeRec* er = edges + o.y;
  pack_row(A + (size_t)i * E * 2, B + (size_t)i * E * 2, S + (size_t)i * E, E, i, o.x, er, &e);
  for (int k2 = 0; k2 < (e + 1) >> 1; ++k2) pairs[o.z + k2] = make_pair_rec(er, e, k2, o.x);
  { const ObstacleBound ob = obstacle_bound(er, e, o.z); bounds[2 * o.x] = ob.circ; bounds[2 * o.x + 1] = ob.obb; }
  row_begin[o.x] = o.y;
  pair_begin[o.x] = o.z;
}

// Small scenes (the MPC case; used for M <= 256, valid up to 1024): count + scan + write fused into ONE single-CTA
// launch (1024 threads, one per row), so a perception update costs one kernel and one copy.
__global__ void __launch_bounds__(1024) pack_fused_kernel(const float* __restrict__ A, const float* __restrict__ B,
                                                          const uint8_t* __restrict__ S, int M, int E,
                                                          PackTotals* __restrict__ totals, EdgeRec* __restrict__ edges,
                                                          PairRec* __restrict__ pairs, int* __restrict__ row_begin,
                                                          int* __restrict__ pair_begin, int* __restrict__ empty_rows,
                                                          float4* __restrict__ bounds, int* __restrict__ row_slot) {
  __shared__ int4 warp_sum[32];
  const int i = threadIdx.x, lane = i & 31, wid = i >> 5;
  int e = 0, rc = 0;
  if (i < M) rc = pack_row(A + (size_t)i * E * 2, B + (size_t)i * E * 2, S + (size_t)i * E, E, i, 0, nullptr, &e);
  const int bad = __syncthreads_or(rc != 0);
  const int4 v = make_int4(e > 0 ? 1 : 0, e, (e + 1) >> 1, (i < M && e == 0) ? 1 : 0);
  int4 inc = v;
#pragma unroll
  for (int o = 1; o < 32; o <<= 1) {
    const int a = __shfl_up_sync(0xffffffffu, inc.x, o), b = __shfl_up_sync(0xffffffffu, inc.y, o);
    const int c = __shfl_up_sync(0xffffffffu, inc.z, o), d = __shfl_up_sync(0xffffffffu, inc.w, o);
    if (lane >= o) { inc.x += a; inc.y += b; inc.z += c; inc.w += d; }
  }
  if (lane == 31) warp_sum[wid] = inc;
  __syncthreads();
  if (wid == 0) {
    const int4 w = warp_sum[lane];
    int4 winc = w;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
      const int a = __shfl_up_sync(0xffffffffu, winc.x, o), b = __shfl_up_sync(0xffffffffu, winc.y, o);
      const int c = __shfl_up_sync(0xffffffffu, winc.z, o), d = __shfl_up_sync(0xffffffffu, winc.w, o);
      if (lane >= o) { winc.x += a; winc.y += b; winc.z += c; winc.w += d; }
    }
    warp_sum[lane] = make_int4(winc.x - w.x, winc.y - w.y, winc.z - w.z, winc.w - w.w);
    if (lane == 31) {
      totals->status = bad ? -2 : 0;
      totals->Mv = winc.x; totals->n_edges = winc.y; totals->n_pairs = winc.z; totals->n_empty = winc.w;
      if (!bad) { row_begin[winc.x] = winc.y; pair_begin[winc.x] = winc.z; row_slot[M] = winc.x; }
    }
  }
  __syncthreads();
  if (bad || i >= M) return;
  const int4 wb = warp_sum[wid];
  const int4 o = make_int4(wb.x + inc.x - v.x, wb.y + inc.y - v.y, wb.z + inc.z - v.z, wb.w + inc.w - v.w);
  row_slot[i] = o.x;
  if (e == 0) { empty_rows[o.w] = i; return; }
  EdgeRec* er = edges + o.y;
  pack_row(A + (size_t)i * E * 2, B + (size_t)i * E * 2, S + (size_t)i * E, E, i, o.x, er, &e);
  for (int k2 = 0; k2 < (e + 1) >> 1; ++k2) pairs[o.z + k2] = make_pair_rec(er, e, k2, o.x);
  { const ObstacleBound ob = obstacle_bound(er, e, o.z); bounds[2 * o.x] = ob.circ; bounds[2 * o.x + 1] = ob.obb; }
  row_begin[o.x] = o.y;
  pair_begin[o.x] = o.z;
}

}  // namespace psdf
