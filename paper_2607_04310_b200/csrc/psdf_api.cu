// C-ABI implementation of include/psdf.h: scene handle, dispatch, CUDA-graph host path.
#include <atomic>
#include <cstdio>
#include <cstdlib>
#include <new>

#include "../../include/psdf.h"
#include "psdf_kernels.cuh"
#include "psdf_cull_kernels.cuh"
#include "psdf_pack.h"
#include "psdf_pack_kernels.cuh"
#include "psdf_reduce_kernels.cuh"

using namespace psdf;

namespace {

std::atomic<int> g_last_cuda_error{0};
std::atomic<long long> g_launches{0};

#define CU_TRY(expr)                                   \
  do {                                                 \
    cudaError_t _e = (expr);                           \
    if (_e != cudaSuccess) {                           \
      g_last_cuda_error.store((int)_e);                \
      (void)cudaGetLastError();                        \
      return PSDF_ERR_CUDA;                            \
    }                                                  \
  } while (0)

struct GraphEntry {
  int N = -1, mode = 0;
  float d_min = 0, rho_p = 0, rho_theta = 0;
  cudaGraphExec_t exec = nullptr;
  unsigned long long stamp = 0;
};
constexpr int kGraphCache = 8;
constexpr int kCullMinPoses = 2048;     // the culled path serves larger batches only

}  // namespace

struct psdf_scene {
  int V = 0, Vp = 0, M = 0, E = 0, max_poses = 0;
  Footprint fp;
  int n_edges = 0, Mv = 0, n_empty = 0;
  int edge_cap = 0;
  int sm_count = 148;
  std::vector<int> h_pair_begin;      // host copy for chunk planning
  int n_pairs = 0;
  // packed scene, double buffered: an update writes the inactive set and flips `cur` only
  // after validation has passed (a rejected update leaves the old scene in force)
  struct Packed {
    EdgeRec* edges = nullptr;         // device packer scratch (one record per valid edge)
    PairRec* pairs = nullptr;
    int* row_begin = nullptr;
    int* row_slot = nullptr;          // [M+1]
    int* empty = nullptr;
    float4* bounds = nullptr;         // [2 M] circle, box per obstacle
    float4* gbounds = nullptr;        // [2 M] bounds in obstacle-grid order
    int* gcell = nullptr;             // [kObsGridMax^2 + 1]
    GridHdr* ghdr = nullptr;
  } pk[2];
  int cur = 0;
  int* h_win = nullptr;               // pinned [max_poses,2]  (psdf_eval_windows_host)
  int* d_win = nullptr;
  unsigned long long* d_ws_depth = nullptr;
  unsigned long long* d_ws_d2 = nullptr;
  unsigned int* d_ws_count = nullptr;
  // device packer scratch (psdf_pack_kernels.cuh)
  int* d_cnt = nullptr;               // [M] valid edges per row
  int4* d_offs = nullptr;             // [M] scanned offsets
  int* d_pair_begin = nullptr;        // [M+1]
  PackTotals* d_totals = nullptr;
  PackTotals* h_totals = nullptr;     // pinned
  int* h_pair_begin_pinned = nullptr; // pinned [M+1]
  // culled path (psdf_cull_kernels.cuh)
  int tune_bd = 0, tune_chunks = 0;   // PSDF_BD / PSDF_CHUNKS, read once at create
  int culling = 0;                    // psdf_set_culling
  unsigned long long* d_stats = nullptr;   // [2] psdf_cull_stats
  // host (graph) path
  cudaStream_t gstream = nullptr;
  float* h_in = nullptr;              // pinned [max_poses,3]
  float* h_out = nullptr;             // pinned [max_poses,4]   value | grad  (or coeff)
  float* h_per = nullptr;             // pinned [max_poses,M]   lazily
  float* d_in = nullptr;
  float* d_out = nullptr;
  float* d_per = nullptr;
  int zero_copy = 1;                  // pinned staging is device-accessible (UVA): see run_zero_copy
  const PoseArgs* arg_poses = nullptr;   // set around a launch whose poses travel as a kernel parameter
  PoseArgs h_args;                    // the MPC host path's poses (N <= kArgPoses)
  GraphEntry graphs[kGraphCache];
  unsigned long long stamp = 0;
};

namespace {

template <int V, int MODE>
cudaError_t launch_one(const psdf_scene* sc, const EvalParams& p, bool lanes, dim3 grid, int bd, cudaStream_t st) {
  if (lanes && sc->arg_poses)
    psdf_lanes_args_kernel<V, MODE><<<grid, bd, 0, st>>>(sc->fp, p, *sc->arg_poses);
  else if (lanes)
    psdf_lanes_kernel<V, MODE><<<grid, bd, 0, st>>>(sc->fp, p);
  else
    psdf_scan_kernel<V, MODE><<<grid, bd, 0, st>>>(sc->fp, p);
  g_launches.fetch_add(1);
  return cudaGetLastError();
}

template <int V>
cudaError_t launch_mode(const psdf_scene* sc, const EvalParams& p, int mode, bool lanes, dim3 grid, int bd,
                        cudaStream_t st) {
  switch (mode) {
    case 0: return launch_one<V, 0>(sc, p, lanes, grid, bd, st);
    case kGrad: return launch_one<V, kGrad>(sc, p, lanes, grid, bd, st);
    case kPerObs: return launch_one<V, kPerObs>(sc, p, lanes, grid, bd, st);
    case kGrad | kPerObs: return launch_one<V, kGrad | kPerObs>(sc, p, lanes, grid, bd, st);
    case kCoeff: return launch_one<V, kCoeff>(sc, p, lanes, grid, bd, st);
    default: return cudaErrorInvalidValue;
  }
}

template <int V, int NP>
cudaError_t launch_cull_mode(const psdf_scene* sc, const EvalParams& p, int mode, cudaStream_t st) {
  const dim3 grid((unsigned)((p.N + NP - 1) / NP));
  switch (mode) {
    case 0: psdf_cull_kernel<V, 0, NP><<<grid, NP, 0, st>>>(sc->fp, p); break;
    case kGrad: psdf_cull_kernel<V, kGrad, NP><<<grid, NP, 0, st>>>(sc->fp, p); break;
    case kCoeff: psdf_cull_kernel<V, kCoeff, NP><<<grid, NP, 0, st>>>(sc->fp, p); break;
    default: return cudaErrorInvalidValue;
  }
  g_launches.fetch_add(1);
  return cudaGetLastError();
}

template <int NP>
cudaError_t launch_cull_v(const psdf_scene* sc, const EvalParams& p, int mode, cudaStream_t st) {
  switch (sc->Vp) {
    case 4: return launch_cull_mode<4, NP>(sc, p, mode, st);
    case 6: return launch_cull_mode<6, NP>(sc, p, mode, st);
    case 8: return launch_cull_mode<8, NP>(sc, p, mode, st);
    case 10: return launch_cull_mode<10, NP>(sc, p, mode, st);
    case 12: return launch_cull_mode<12, NP>(sc, p, mode, st);
    case 16: return launch_cull_mode<16, NP>(sc, p, mode, st);
    default: return cudaErrorInvalidValue;
  }
}

// Culled path: one launch.  Small batches take one warp per CTA so that they
// still spread over all SMs; large ones 128 poses per CTA (measured: cfg4 133 vs 146 us).
cudaError_t enqueue_culled(const psdf_scene* sc, EvalParams& p, int mode, cudaStream_t st) {
  p.gbounds = sc->pk[sc->cur].gbounds;
  p.gcell = sc->pk[sc->cur].gcell;
  p.ghdr = sc->pk[sc->cur].ghdr;
  p.stats = sc->d_stats;
  p.n_chunks = 1;
  if (p.N <= 32768) return launch_cull_v<32>(sc, p, mode, st);
  return launch_cull_v<128>(sc, p, mode, st);
}

cudaError_t launch_v(const psdf_scene* sc, const EvalParams& p, int mode, bool lanes, dim3 grid, int bd,
                     cudaStream_t st) {
  switch (sc->Vp) {
    case 4: return launch_mode<4>(sc, p, mode, lanes, grid, bd, st);
    case 6: return launch_mode<6>(sc, p, mode, lanes, grid, bd, st);
    case 8: return launch_mode<8>(sc, p, mode, lanes, grid, bd, st);
    case 10: return launch_mode<10>(sc, p, mode, lanes, grid, bd, st);
    case 12: return launch_mode<12>(sc, p, mode, lanes, grid, bd, st);
    case 16: return launch_mode<16>(sc, p, mode, lanes, grid, bd, st);
    default: return cudaErrorInvalidValue;
  }
}

// lane-split kernel: few poses or little work (measured crossover against the tile-scan kernel)
inline bool lanes_plan(const psdf_scene* sc, int N) {
  return N <= 128 || (long long)N * (sc->Mv > 0 ? sc->Mv : 1) <= (1 << 17);
}

// Launch plan: lane-split kernel for MPC-sized batches; otherwise the
// tile-scan kernel, with the obstacle range cut into chunks when the pose tiles alone
// would not fill 148 SMs several times over.
psdf_status enqueue_eval(const psdf_scene* sc, const float* poses, int N, float* value, float* grad,
                         float* per_obs, float* coeff, float d_min, float rho_p, float rho_theta,
                         cudaStream_t st, float* packed = nullptr, const int* window = nullptr) {
  if (N == 0) return PSDF_OK;
  EvalParams p{};
  p.pairs = sc->pk[sc->cur].pairs;
  p.row_slot = sc->pk[sc->cur].row_slot;
  p.bounds = sc->pk[sc->cur].bounds;
  p.window = window;
  p.empty_rows = sc->pk[sc->cur].empty;
  p.poses = poses;
  p.value = value;
  p.grad = grad;
  p.per_obs = per_obs;
  p.coeff = coeff;
  p.packed = packed;
  p.ws_depth = sc->d_ws_depth;
  p.ws_d2 = sc->d_ws_d2;
  p.ws_count = sc->d_ws_count;
  p.n_edges = sc->n_edges;
  p.Mv = sc->Mv;
  p.M_rows = sc->M;
  p.n_empty = sc->n_empty;
  p.N = N;
  p.d_min = d_min;
  p.rho_p = rho_p;
  p.rho_theta = rho_theta;
  const int mode = coeff ? kCoeff : ((grad ? kGrad : 0) | (per_obs ? kPerObs : 0));

  const bool lanes = lanes_plan(sc, N) || window != nullptr;
  dim3 grid;
  int bd;
  if (sc->culling && !lanes && N > kCullMinPoses && !per_obs && sc->Mv >= 64) {
    cudaError_t e = enqueue_culled(sc, p, mode, st);
    if (e != cudaSuccess) {
      g_last_cuda_error.store((int)e);
      return PSDF_ERR_CUDA;
    }
    return PSDF_OK;
  }
  if (lanes) {
    // lanes per pose: enough to put ~148 x 1024 lanes in flight, at most one lane per obstacle;
    // K of them inside a CTA (<= 256), the rest as C CTAs per pose group (<= 16)
    long long want = (long long)sc->sm_count * 1024 / N;
    int L = 1;
    while (L < 4096 && L < sc->Mv && L * 2 <= want) L <<= 1;
    const int K = L < 256 ? L : 256;
    int C = L / K;
    if (C > 16) C = 16;
    p.lanes = K;
    p.n_chunks = C;
    bd = K <= 64 ? 64 : K;
    const int ppc = bd / K;
    grid = dim3((unsigned)((N + ppc - 1) / ppc), (unsigned)C);
  } else {
    // One thread per pose leaves only N/32 warps; the loop is issue/operand-bound and wants many
    // resident warps, and many small CTAs balance the tail: the obstacle range is cut into C
    // chunks (C CTAs of 64 poses per pose tile, combined by atomics) so that ~256 warps per SM are
    // launched in total (measured sweep: cfg5 64x19, cfg4 64x12, cfg3 64x6).
    bd = 64;
    int C = 1;
    const double warps_per_sm = (double)N / 32.0 / sc->sm_count;
    if (warps_per_sm < 256.0) C = (int)std::ceil(256.0 / warps_per_sm);
    const int maxC = sc->Mv / 16 > 0 ? sc->Mv / 16 : 1;
    if (sc->tune_bd > 0) bd = sc->tune_bd;                                   // tuning overrides
    if (sc->tune_chunks > 0) C = sc->tune_chunks;
    if (bd != 32 && bd != 64 && bd != 128 && bd != 256) bd = 64;
    if (C < 1) C = 1;
    if (C > maxC) C = maxC;
    if (C > kMaxChunks) C = kMaxChunks;
    const int tiles = (N + bd - 1) / bd;
    // chunk boundaries on obstacle boundaries, balanced by edge count
    p.chunk_begin[0] = 0;
    int o = 0;
    for (int c = 1; c < C; ++c) {
      const long long target = (long long)sc->n_pairs * c / C;
      while (o < sc->Mv && sc->h_pair_begin[o] < target) ++o;
      p.chunk_begin[c] = sc->h_pair_begin[o];
    }
    p.chunk_begin[C] = sc->n_pairs;
    p.n_chunks = C;
    grid = dim3((unsigned)tiles, (unsigned)C);
  }
  cudaError_t e = launch_v(sc, p, mode, lanes, grid, bd, st);
  if (e != cudaSuccess) {
    g_last_cuda_error.store((int)e);
    return PSDF_ERR_CUDA;
  }
  return PSDF_OK;
}

// Device-resident (A,B,S): pack on the GPU (count+validate -> scan -> write); only the
// totals and the per-obstacle pair offsets (for the host launch plan) come back.
psdf_status pack_on_device(psdf_scene* sc, const float* A, const float* B, const uint8_t* S, cudaStream_t st) {
  const int M = sc->M, E = sc->E;
  const int bd = 128, gd = (M + bd - 1) / bd;
  const psdf_scene::Packed& dst = sc->pk[sc->cur ^ 1];      // the inactive set
  // d_totals and d_pair_begin are one allocation [PackTotals | pair_begin[M+1]]: one copy back
  if (M <= 256) {                                            // measured: fused wins below ~256 rows
    pack_fused_kernel<<<1, 1024, 0, st>>>(A, B, S, M, E, sc->d_totals, dst.edges, dst.pairs, dst.row_begin,
                                          sc->d_pair_begin, dst.empty, dst.bounds, dst.row_slot);
    g_launches.fetch_add(1);
  } else {
    CU_TRY(cudaMemsetAsync(sc->d_totals, 0, sizeof(PackTotals), st));
    pack_count_kernel<<<gd, bd, 0, st>>>(A, B, S, M, E, sc->d_cnt, sc->d_totals);
    pack_scan_kernel<<<1, 1024, 0, st>>>(sc->d_cnt, M, sc->d_offs, sc->d_totals);
    pack_write_kernel<<<gd, bd, 0, st>>>(A, B, S, M, E, sc->d_cnt, sc->d_offs, sc->d_totals, dst.edges, dst.pairs,
                                         dst.row_begin, sc->d_pair_begin, dst.empty, dst.bounds, dst.row_slot);
    g_launches.fetch_add(3);
  }
  if (sc->max_poses > kCullMinPoses) {                       // the culled path's grid (never used by small scenes)
    obstacle_grid_kernel<<<1, 1024, 0, st>>>(dst.bounds, 0, reinterpret_cast<const int*>(sc->d_totals), dst.gbounds,
                                             dst.gcell, sc->d_cnt, dst.ghdr);
    g_launches.fetch_add(1);
  }
  CU_TRY(cudaMemcpyAsync(sc->h_totals, sc->d_totals, sizeof(PackTotals) + sizeof(int) * ((size_t)M + 1),
                         cudaMemcpyDeviceToHost, st));
  CU_TRY(cudaStreamSynchronize(st));                         // the only synchronisation of an update
  CU_TRY(cudaGetLastError());
  const PackTotals t = *sc->h_totals;
  if (t.status != 0) return PSDF_ERR_DEGENERATE;             // the live set has not been touched
  sc->h_pair_begin.assign(sc->h_pair_begin_pinned, sc->h_pair_begin_pinned + t.Mv + 1);
  sc->n_edges = t.n_edges;
  sc->Mv = t.Mv;
  sc->n_empty = t.n_empty;
  sc->n_pairs = t.n_pairs;
  sc->cur ^= 1;
  return PSDF_OK;
}

psdf_status upload_scene(psdf_scene* sc, const float* A, const float* B, const uint8_t* S, psdf_mem where,
                         cudaStream_t st) {
  if (where == PSDF_MEM_DEVICE) return pack_on_device(sc, A, B, S, st);
  PackedScene ps;
  if (pack_scene(A, B, S, sc->M, sc->E, ps) != 0) return PSDF_ERR_DEGENERATE;
  const psdf_scene::Packed& dst = sc->pk[sc->cur ^ 1];
  const int n_edges = (int)ps.edges.size(), Mv = (int)ps.row_begin.size() - 1, n_empty = (int)ps.empty_rows.size();
  const int n_pairs = (int)ps.pairs.size();
  // (dst.edges / dst.row_begin are the device packer's scratch: the kernels read pair records only)
  if (n_edges) CU_TRY(cudaMemcpyAsync(dst.pairs, ps.pairs.data(), sizeof(PairRec) * n_pairs, cudaMemcpyHostToDevice, st));
  CU_TRY(cudaMemcpyAsync(dst.row_slot, ps.row_slot.data(), sizeof(int) * (size_t)(sc->M + 1), cudaMemcpyHostToDevice, st));
  if (Mv) CU_TRY(cudaMemcpyAsync(dst.bounds, ps.bounds.data(), sizeof(float4) * 2 * Mv, cudaMemcpyHostToDevice, st));
  if (n_empty) CU_TRY(cudaMemcpyAsync(dst.empty, ps.empty_rows.data(), sizeof(int) * n_empty, cudaMemcpyHostToDevice, st));
  if (sc->max_poses > kCullMinPoses) {                       // the culled path's grid (never used by small scenes)
    obstacle_grid_kernel<<<1, 1024, 0, st>>>(dst.bounds, Mv, nullptr, dst.gbounds, dst.gcell, sc->d_cnt, dst.ghdr);
    g_launches.fetch_add(1);
  }
  CU_TRY(cudaStreamSynchronize(st));       // the staging vectors die here
  sc->n_edges = n_edges;
  sc->Mv = Mv;
  sc->n_empty = n_empty;
  sc->n_pairs = n_pairs;
  sc->h_pair_begin.swap(ps.pair_begin);
  sc->cur ^= 1;
  return PSDF_OK;
}

}  // namespace

// =============================================================================== C ABI
extern "C" {

void psdf_destroy_scene(psdf_scene* sc) {
  if (!sc) return;
  for (auto& g : sc->graphs)
    if (g.exec) cudaGraphExecDestroy(g.exec);
  if (sc->gstream) cudaStreamDestroy(sc->gstream);
  for (auto& b : sc->pk) {
    cudaFree(b.edges); cudaFree(b.pairs); cudaFree(b.row_begin); cudaFree(b.row_slot); cudaFree(b.empty); cudaFree(b.bounds);
    cudaFree(b.gbounds); cudaFree(b.gcell); cudaFree(b.ghdr);
  }
  cudaFree(sc->d_win);
  if (sc->h_totals) cudaFreeHost(sc->h_totals);
  if (sc->h_win) cudaFreeHost(sc->h_win);
  cudaFree(sc->d_ws_depth); cudaFree(sc->d_ws_d2); cudaFree(sc->d_ws_count);
  cudaFree(sc->d_stats);
  cudaFree(sc->d_cnt); cudaFree(sc->d_offs); cudaFree(sc->d_totals);   // d_pair_begin lives inside d_totals' block
  cudaFree(sc->d_in); cudaFree(sc->d_out); cudaFree(sc->d_per);
  if (sc->h_in) cudaFreeHost(sc->h_in);
  if (sc->h_out) cudaFreeHost(sc->h_out);
  if (sc->h_per) cudaFreeHost(sc->h_per);
  delete sc;
}

psdf_status psdf_create_scene(const float* footprint, int V, const float* A, const float* B,
                              const uint8_t* S, int M, int E, psdf_mem where, int max_poses,
                              void* cuda_stream, psdf_scene** out) {
  if (!footprint || !A || !B || !S || !out || M < 1 || E < 3 || max_poses < 1 || V < 3 || V > kMaxV ||
      (where != PSDF_MEM_HOST && where != PSDF_MEM_DEVICE))
    return PSDF_ERR_INVALID_ARG;
  psdf_scene* sc = new (std::nothrow) psdf_scene();
  if (!sc) return PSDF_ERR_ALLOC;
  sc->V = V; sc->M = M; sc->E = E; sc->max_poses = max_poses;
  if (const char* e = std::getenv("PSDF_BD")) sc->tune_bd = std::atoi(e);             // measurement sweeps only
  if (const char* e = std::getenv("PSDF_CHUNKS")) sc->tune_chunks = std::atoi(e);
  const int rc = pack_footprint(footprint, V, sc->fp, sc->Vp);
  if (rc != 0) { delete sc; return rc == -1 ? PSDF_ERR_INVALID_ARG : PSDF_ERR_DEGENERATE; }
  if (where == PSDF_MEM_HOST) {   // validate before touching CUDA (Assumption 1)
    PackedScene probe;
    if (pack_scene(A, B, S, M, E, probe) != 0) { delete sc; return PSDF_ERR_DEGENERATE; }
  }
  cudaStream_t st = (cudaStream_t)cuda_stream;
  sc->edge_cap = M * E;
  int dev = 0;
  psdf_status status = PSDF_OK;
  auto body = [&]() -> psdf_status {
    CU_TRY(cudaGetDevice(&dev));
    CU_TRY(cudaDeviceGetAttribute(&sc->sm_count, cudaDevAttrMultiProcessorCount, dev));
    for (auto& b : sc->pk) {
      CU_TRY(cudaMalloc(&b.edges, sizeof(EdgeRec) * (size_t)sc->edge_cap));
      CU_TRY(cudaMalloc(&b.pairs, sizeof(PairRec) * (size_t)(sc->edge_cap / 2 + M)));
      CU_TRY(cudaMalloc(&b.row_begin, sizeof(int) * (size_t)(M + 1)));
      CU_TRY(cudaMalloc(&b.row_slot, sizeof(int) * (size_t)(M + 1)));
      CU_TRY(cudaMalloc(&b.empty, sizeof(int) * (size_t)M));
      CU_TRY(cudaMalloc(&b.bounds, sizeof(float4) * 2 * (size_t)M));
      CU_TRY(cudaMalloc(&b.gbounds, sizeof(float4) * 2 * (size_t)M));
      CU_TRY(cudaMalloc(&b.gcell, sizeof(int) * (size_t)(kObsGridMax * kObsGridMax + 1)));
      CU_TRY(cudaMalloc(&b.ghdr, sizeof(GridHdr)));
    }
    CU_TRY(cudaMallocHost(&sc->h_totals, sizeof(PackTotals) + sizeof(int) * (size_t)(M + 1)));
    sc->h_pair_begin_pinned = reinterpret_cast<int*>(sc->h_totals + 1);
    CU_TRY(cudaMalloc(&sc->d_cnt, sizeof(int) * (size_t)M));
    CU_TRY(cudaMalloc(&sc->d_offs, sizeof(int4) * (size_t)M));
    CU_TRY(cudaMalloc(&sc->d_totals, sizeof(PackTotals) + sizeof(int) * (size_t)(M + 1)));
    sc->d_pair_begin = reinterpret_cast<int*>(sc->d_totals + 1);
    CU_TRY(cudaMalloc(&sc->d_stats, sizeof(unsigned long long) * 2));
    CU_TRY(cudaMemsetAsync(sc->d_stats, 0, sizeof(unsigned long long) * 2, st));
    CU_TRY(cudaMalloc(&sc->d_ws_depth, sizeof(unsigned long long) * (size_t)max_poses));
    CU_TRY(cudaMalloc(&sc->d_ws_d2, sizeof(unsigned long long) * (size_t)max_poses));
    const size_t n_cnt = (size_t)max_poses + 1;          // scan: one per pose tile; lanes: one per pose group
    CU_TRY(cudaMalloc(&sc->d_ws_count, sizeof(unsigned int) * n_cnt));
    CU_TRY(cudaMemsetAsync(sc->d_ws_depth, 0x00, sizeof(unsigned long long) * (size_t)max_poses, st));
    CU_TRY(cudaMemsetAsync(sc->d_ws_d2, 0xff, sizeof(unsigned long long) * (size_t)max_poses, st));
    CU_TRY(cudaMemsetAsync(sc->d_ws_count, 0x00, sizeof(unsigned int) * n_cnt, st));
    return upload_scene(sc, A, B, S, where, st);
  };
  status = body();
  if (status != PSDF_OK) { psdf_destroy_scene(sc); return status; }
  *out = sc;
  return PSDF_OK;
}

psdf_status psdf_update_scene(psdf_scene* sc, const float* A, const float* B, const uint8_t* S,
                              psdf_mem where, void* cuda_stream) {
  if (!sc || !A || !B || !S) return PSDF_ERR_INVALID_ARG;
  // both paths validate before anything live changes (host: pack_scene; device: status word
  // checked before the buffer flip), so a bad update leaves the old scene in force
  cudaStream_t st = (cudaStream_t)cuda_stream;
  if (sc->gstream) CU_TRY(cudaStreamSynchronize(sc->gstream));
  psdf_status s = upload_scene(sc, A, B, S, where, st);
  if (s != PSDF_OK) return s;
  for (auto& g : sc->graphs) {           // launch plans are baked into the captured graphs
    if (g.exec) cudaGraphExecDestroy(g.exec);
    g = GraphEntry();
  }
  return PSDF_OK;
}

psdf_status psdf_eval(psdf_scene* sc, const float* poses, int N, float* value, float* grad,
                      float* per_obstacle, void* cuda_stream) {
  if (!sc || N < 0 || (N > 0 && (!poses || !value))) return PSDF_ERR_INVALID_ARG;
  if (N > sc->max_poses) return PSDF_ERR_CAPACITY;
  return enqueue_eval(sc, poses, N, value, grad, per_obstacle, nullptr, 0.f, 0.f, 0.f, (cudaStream_t)cuda_stream);
}

static psdf_status ensure_host_path(psdf_scene* sc, bool per_obs) {
  if (!sc->gstream) {
    CU_TRY(cudaStreamCreateWithFlags(&sc->gstream, cudaStreamNonBlocking));
    CU_TRY(cudaHostAlloc(&sc->h_in, sizeof(float) * 4 * (size_t)sc->max_poses, cudaHostAllocMapped));
    CU_TRY(cudaHostAlloc(&sc->h_out, sizeof(float) * 4 * (size_t)sc->max_poses, cudaHostAllocMapped));
    int dev = 0, uva = 0;
    CU_TRY(cudaGetDevice(&dev));
    CU_TRY(cudaDeviceGetAttribute(&uva, cudaDevAttrUnifiedAddressing, dev));
    if (const char* e = std::getenv("PSDF_NO_ZERO_COPY")) uva = (e[0] == '1') ? 0 : uva;
    sc->zero_copy = uva;
    CU_TRY(cudaMalloc(&sc->d_in, sizeof(float) * 3 * (size_t)sc->max_poses));
    CU_TRY(cudaMalloc(&sc->d_out, sizeof(float) * 4 * (size_t)sc->max_poses));
  }
  if (per_obs && !sc->d_per) {
    CU_TRY(cudaHostAlloc(&sc->h_per, sizeof(float) * (size_t)sc->max_poses * sc->M, cudaHostAllocMapped));
    CU_TRY(cudaMalloc(&sc->d_per, sizeof(float) * (size_t)sc->max_poses * sc->M));
  }
  return PSDF_OK;
}

// MPC-sized batches: ONE kernel launch that reads the poses from, and writes the results to,
// the pinned (mapped) staging buffers directly: a few hundred bytes cross PCIe inside the
// kernel instead of through two copy-engine operations, which removes two graph nodes'
// worth of latency.  Same output layout as the graph path.
constexpr int kZeroCopyMaxPoses = 512;
constexpr int kZeroCopyMaxObstaclesPerObs = 64;

// Measured on B200 (bench.py mpc_latency, Table-I shapes up to 1000 obstacles): the single launch
// beats the 3-node graph by 4-7 us whenever the batch is MPC sized; only the [N,M] per-obstacle
// output of a large scene stays on the copy engine (scattered 4-byte stores over PCIe otherwise).
static inline bool use_zero_copy(const psdf_scene* sc, int N, bool per_obs) {
  return sc->zero_copy && N <= kZeroCopyMaxPoses && lanes_plan(sc, N) &&      // (the lane-split kernel reads the staging layout)
         (!per_obs || sc->Mv <= kZeroCopyMaxObstaclesPerObs);
}

static psdf_status run_zero_copy(psdf_scene* sc, int N, int mode, float d_min, float rho_p, float rho_theta) {
  // staging layout: h_in [N,4] poses (padded), h_out [N,4] = (value, grad) or coefficients;
  // up to kArgPoses poses go into the launch itself (kernel parameter) instead
  sc->arg_poses = N <= kArgPoses ? &sc->h_args : nullptr;
  psdf_status s = enqueue_eval(sc, sc->h_in, N, sc->d_in /*unused*/, (mode & kGrad) ? sc->d_out : nullptr,
                               (mode & kPerObs) ? sc->h_per : nullptr, (mode & kCoeff) ? sc->h_out : nullptr, d_min,
                               rho_p, rho_theta, sc->gstream, sc->h_out);
  sc->arg_poses = nullptr;
  if (s != PSDF_OK) return s;
  CU_TRY(cudaStreamSynchronize(sc->gstream));
  return PSDF_OK;
}

// Graph replay {H2D poses, kernel, D2H results}; captured once per (N, outputs, MPC constants).
static psdf_status run_graph(psdf_scene* sc, int N, int mode, float d_min, float rho_p, float rho_theta) {
  if (use_zero_copy(sc, N, (mode & kPerObs) != 0)) return run_zero_copy(sc, N, mode, d_min, rho_p, rho_theta);
  GraphEntry* hit = nullptr;
  GraphEntry* victim = &sc->graphs[0];
  for (auto& g : sc->graphs) {
    if (g.exec && g.N == N && g.mode == mode && g.d_min == d_min && g.rho_p == rho_p && g.rho_theta == rho_theta) {
      hit = &g;
      break;
    }
    if (g.stamp < victim->stamp) victim = &g;
  }
  if (!hit) {
    if (victim->exec) { cudaGraphExecDestroy(victim->exec); *victim = GraphEntry(); }
    cudaGraph_t graph = nullptr;
    CU_TRY(cudaStreamBeginCapture(sc->gstream, cudaStreamCaptureModeThreadLocal));
    cudaError_t e = cudaMemcpyAsync(sc->d_in, sc->h_in, sizeof(float) * 3 * (size_t)N, cudaMemcpyHostToDevice, sc->gstream);
    psdf_status s = PSDF_OK;
    if (e == cudaSuccess) {
      float* value = sc->d_out;                       // [N] value | [N,3] grad, or [N,4] coeff + value after
      if (mode & kCoeff)
        s = enqueue_eval(sc, sc->d_in, N, sc->d_in /*scratch: value not returned*/, nullptr, nullptr, sc->d_out,
                         d_min, rho_p, rho_theta, sc->gstream);
      else
        s = enqueue_eval(sc, sc->d_in, N, value, (mode & kGrad) ? sc->d_out + N : nullptr,
                         (mode & kPerObs) ? sc->d_per : nullptr, nullptr, 0.f, 0.f, 0.f, sc->gstream);
    }
    if (e == cudaSuccess && s == PSDF_OK) {
      const size_t nout = (mode & (kGrad | kCoeff)) ? 4 * (size_t)N : (size_t)N;
      e = cudaMemcpyAsync(sc->h_out, sc->d_out, sizeof(float) * nout, cudaMemcpyDeviceToHost, sc->gstream);
      if (e == cudaSuccess && (mode & kPerObs))
        e = cudaMemcpyAsync(sc->h_per, sc->d_per, sizeof(float) * (size_t)N * sc->M, cudaMemcpyDeviceToHost, sc->gstream);
    }
    cudaError_t e2 = cudaStreamEndCapture(sc->gstream, &graph);
    if (e != cudaSuccess || e2 != cudaSuccess || s != PSDF_OK || !graph) {
      if (graph) cudaGraphDestroy(graph);
      g_last_cuda_error.store((int)(e != cudaSuccess ? e : e2));
      (void)cudaGetLastError();
      return s != PSDF_OK ? s : PSDF_ERR_CUDA;
    }
    cudaGraphExec_t exec = nullptr;
    e = cudaGraphInstantiate(&exec, graph, 0);
    cudaGraphDestroy(graph);
    CU_TRY(e);
    victim->exec = exec; victim->N = N; victim->mode = mode;
    victim->d_min = d_min; victim->rho_p = rho_p; victim->rho_theta = rho_theta;
    hit = victim;
  }
  hit->stamp = ++sc->stamp;
  CU_TRY(cudaGraphLaunch(hit->exec, sc->gstream));
  g_launches.fetch_add(1);   // the replayed graph holds one kernel node
  CU_TRY(cudaStreamSynchronize(sc->gstream));
  return PSDF_OK;
}

static void stage_poses(psdf_scene* sc, const float* poses, int N, bool per_obs) {
  if (!use_zero_copy(sc, N, per_obs)) { std::memcpy(sc->h_in, poses, sizeof(float) * 3 * (size_t)N); return; }
  if (N <= kArgPoses) {
    for (int n = 0; n < N; ++n) sc->h_args.q[n] = make_float4(poses[3 * n], poses[3 * n + 1], poses[3 * n + 2], 0.f);
    return;
  }
  for (int n = 0; n < N; ++n) {
    sc->h_in[4 * n] = poses[3 * n]; sc->h_in[4 * n + 1] = poses[3 * n + 1];
    sc->h_in[4 * n + 2] = poses[3 * n + 2]; sc->h_in[4 * n + 3] = 0.f;
  }
}

psdf_status psdf_eval_host(psdf_scene* sc, const float* poses, int N, float* value, float* grad,
                           float* per_obstacle) {
  if (!sc || N < 0 || (N > 0 && (!poses || !value))) return PSDF_ERR_INVALID_ARG;
  if (N > sc->max_poses) return PSDF_ERR_CAPACITY;
  if (N == 0) return PSDF_OK;
  psdf_status s = ensure_host_path(sc, per_obstacle != nullptr);
  if (s != PSDF_OK) return s;
  stage_poses(sc, poses, N, per_obstacle != nullptr);
  const int mode = (grad ? kGrad : 0) | (per_obstacle ? kPerObs : 0);
  s = run_graph(sc, N, mode, 0.f, 0.f, 0.f);
  if (s != PSDF_OK) return s;
  if (use_zero_copy(sc, N, per_obstacle != nullptr)) {
    for (int n = 0; n < N; ++n) {
      value[n] = sc->h_out[4 * n];
      if (grad) { grad[3 * n] = sc->h_out[4 * n + 1]; grad[3 * n + 1] = sc->h_out[4 * n + 2]; grad[3 * n + 2] = sc->h_out[4 * n + 3]; }
    }
  } else {
    std::memcpy(value, sc->h_out, sizeof(float) * (size_t)N);
    if (grad) std::memcpy(grad, sc->h_out + N, sizeof(float) * 3 * (size_t)N);
  }
  if (per_obstacle) std::memcpy(per_obstacle, sc->h_per, sizeof(float) * (size_t)N * sc->M);
  return PSDF_OK;
}

psdf_status psdf_eval_windows(psdf_scene* sc, const float* poses, int N, const int* row_window, float* value,
                              float* grad, void* cuda_stream) {
  if (!sc || N < 0 || (N > 0 && (!poses || !value || !row_window))) return PSDF_ERR_INVALID_ARG;
  if (N > sc->max_poses) return PSDF_ERR_CAPACITY;
  return enqueue_eval(sc, poses, N, value, grad, nullptr, nullptr, 0.f, 0.f, 0.f, (cudaStream_t)cuda_stream, nullptr,
                      row_window);
}

psdf_status psdf_eval_windows_host(psdf_scene* sc, const float* poses, int N, const int* row_window, float* value,
                                   float* grad) {
  if (!sc || N < 0 || (N > 0 && (!poses || !value || !row_window))) return PSDF_ERR_INVALID_ARG;
  if (N > sc->max_poses) return PSDF_ERR_CAPACITY;
  if (N == 0) return PSDF_OK;
  psdf_status s = ensure_host_path(sc, false);
  if (s != PSDF_OK) return s;
  if (!sc->h_win) {
    CU_TRY(cudaMallocHost(&sc->h_win, sizeof(int) * 2 * (size_t)sc->max_poses));
    CU_TRY(cudaMalloc(&sc->d_win, sizeof(int) * 2 * (size_t)sc->max_poses));
  }
  std::memcpy(sc->h_in, poses, sizeof(float) * 3 * (size_t)N);
  std::memcpy(sc->h_win, row_window, sizeof(int) * 2 * (size_t)N);
  cudaStream_t st = sc->gstream;
  CU_TRY(cudaMemcpyAsync(sc->d_in, sc->h_in, sizeof(float) * 3 * (size_t)N, cudaMemcpyHostToDevice, st));
  CU_TRY(cudaMemcpyAsync(sc->d_win, sc->h_win, sizeof(int) * 2 * (size_t)N, cudaMemcpyHostToDevice, st));
  s = enqueue_eval(sc, sc->d_in, N, sc->d_out, grad ? sc->d_out + N : nullptr, nullptr, nullptr, 0.f, 0.f, 0.f, st,
                   nullptr, sc->d_win);
  if (s != PSDF_OK) return s;
  CU_TRY(cudaMemcpyAsync(sc->h_out, sc->d_out, sizeof(float) * (grad ? 4 : 1) * (size_t)N, cudaMemcpyDeviceToHost, st));
  CU_TRY(cudaStreamSynchronize(st));
  std::memcpy(value, sc->h_out, sizeof(float) * (size_t)N);
  if (grad) std::memcpy(grad, sc->h_out + N, sizeof(float) * 3 * (size_t)N);
  return PSDF_OK;
}

psdf_status psdf_mpc_coeffs_host(psdf_scene* sc, const float* poses, int N, float d_min, float rho_p,
                                 float rho_theta, float* coeff) {
  if (!sc || N < 0 || (N > 0 && (!poses || !coeff))) return PSDF_ERR_INVALID_ARG;
  if (N > sc->max_poses) return PSDF_ERR_CAPACITY;
  if (N == 0) return PSDF_OK;
  psdf_status s = ensure_host_path(sc, false);
  if (s != PSDF_OK) return s;
  stage_poses(sc, poses, N, false);
  s = run_graph(sc, N, kCoeff, d_min, rho_p, rho_theta);
  if (s != PSDF_OK) return s;
  std::memcpy(coeff, sc->h_out, sizeof(float) * 4 * (size_t)N);
  return PSDF_OK;
}

psdf_status psdf_set_culling(psdf_scene* sc, int enable) {
  if (!sc) return PSDF_ERR_INVALID_ARG;
  if (sc->gstream) CU_TRY(cudaStreamSynchronize(sc->gstream));
  sc->culling = enable ? 1 : 0;
  for (auto& g : sc->graphs) {           // launch plans are baked into the captured graphs
    if (g.exec) cudaGraphExecDestroy(g.exec);
    g = GraphEntry();
  }
  return PSDF_OK;
}

psdf_status psdf_component_min(const float* per_component, int N, int M, const int* comp_to_obstacle,
                               int n_obstacles, float* out, void* cuda_stream) {
  if (N < 0 || M < 1 || n_obstacles < 1 || (N > 0 && (!per_component || !comp_to_obstacle || !out)))
    return PSDF_ERR_INVALID_ARG;
  if (N == 0) return PSDF_OK;
  const long long total = (long long)N * n_obstacles;
  component_min_kernel<<<(unsigned)((total + 255) / 256), 256, 0, (cudaStream_t)cuda_stream>>>(
      per_component, N, M, comp_to_obstacle, n_obstacles, out);
  g_launches.fetch_add(1);
  CU_TRY(cudaGetLastError());
  return PSDF_OK;
}

psdf_status psdf_trajectory_reduce(const float* value, int T, int H, float d_safe, float* min_value,
                                   int* argmin_stage, float* penalty, void* cuda_stream) {
  if (T < 0 || H < 1 || (T > 0 && !value)) return PSDF_ERR_INVALID_ARG;
  if (T == 0) return PSDF_OK;
  trajectory_reduce_kernel<<<(unsigned)((T + 3) / 4), 128, 0, (cudaStream_t)cuda_stream>>>(value, T, H, d_safe, min_value,
                                                                                          argmin_stage, penalty);
  g_launches.fetch_add(1);
  CU_TRY(cudaGetLastError());
  return PSDF_OK;
}

psdf_status psdf_cull_stats(psdf_scene* sc, void* cuda_stream, unsigned long long* out2) {
  if (!sc || !out2) return PSDF_ERR_INVALID_ARG;
  cudaStream_t st = (cudaStream_t)cuda_stream;
  CU_TRY(cudaMemcpyAsync(out2, sc->d_stats, sizeof(unsigned long long) * 2, cudaMemcpyDeviceToHost, st));
  CU_TRY(cudaMemsetAsync(sc->d_stats, 0, sizeof(unsigned long long) * 2, st));
  CU_TRY(cudaStreamSynchronize(st));
  return PSDF_OK;
}

int psdf_scene_num_obstacles(const psdf_scene* sc) { return sc ? sc->Mv : 0; }
int psdf_scene_num_edges(const psdf_scene* sc) { return sc ? sc->n_edges : 0; }
int psdf_last_cuda_error(void) { return g_last_cuda_error.load(); }
long long psdf_kernel_launches(void) { return g_launches.load(); }
const char* psdf_version(void) { return "psdf-b200 0.1 (sm_100a)"; }

const char* psdf_status_string(psdf_status s) {
  switch (s) {
    case PSDF_OK: return "ok";
    case PSDF_ERR_INVALID_ARG: return "invalid argument";
    case PSDF_ERR_DEGENERATE: return "degenerate geometry (Assumption 1 violated)";
    case PSDF_ERR_CAPACITY: return "N exceeds max_poses";
    case PSDF_ERR_CUDA: return "CUDA error";
    case PSDF_ERR_ALLOC: return "allocation failed";
  }
  return "unknown status";
}

psdf_status psdf_measure_fp32_peak(int iters, void* cuda_stream, double* tflops_out) {
  if (!tflops_out || iters < 1) return PSDF_ERR_INVALID_ARG;
  cudaStream_t st = (cudaStream_t)cuda_stream;
  int dev = 0, sms = 0;
  CU_TRY(cudaGetDevice(&dev));
  CU_TRY(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
  float* d = nullptr;
  CU_TRY(cudaMalloc(&d, sizeof(float)));
  cudaEvent_t a, b;
  CU_TRY(cudaEventCreate(&a));
  CU_TRY(cudaEventCreate(&b));
  const int blocks = sms * 8, threads = 256;
  fp32_peak_kernel<<<blocks, threads, 0, st>>>(d, iters, 0.999f, 0.001f);   // warm-up
  float best = 1e30f;
  for (int r = 0; r < 5; ++r) {
    cudaEventRecord(a, st);
    fp32_peak_kernel<<<blocks, threads, 0, st>>>(d, iters, 0.999f, 0.001f);
    cudaEventRecord(b, st);
    CU_TRY(cudaEventSynchronize(b));
    float ms = 0;
    cudaEventElapsedTime(&ms, a, b);
    if (ms < best) best = ms;
  }
  g_launches.fetch_add(6);
  cudaEventDestroy(a); cudaEventDestroy(b); cudaFree(d);
  CU_TRY(cudaGetLastError());
  *tflops_out = 2.0 * 16.0 * (double)iters * blocks * threads / (best * 1e-3) / 1e12;
  return PSDF_OK;
}

}  // extern "C"
