// C-ABI implementation of include/psdf.h: scene handle, dispatch, CUDA-graph host path.
#include <atomic>
#include <chrono>
#include <cstdio>
#include <cstdlib>
#include <new>
#include <immintrin.h>

#include "../../include/psdf.h"
#include "../../include/psdf_bench.h"
#include "psdf_kernels.cuh"
#include "psdf_cull_kernels.cuh"
#include "psdf_pack.h"
#include "psdf_pack_kernels.cuh"

using namespace psdf;

namespace {

std::atomic<int> g_last_cuda_error{0};
std::atomic<long long> g_launches{0};

inline psdf_status cuda_failed(cudaError_t e) {
  g_last_cuda_error.store((int)e);
  (void)cudaGetLastError();
  return e == cudaErrorMemoryAllocation ? PSDF_ERR_ALLOC : PSDF_ERR_CUDA;
}

#define CU_TRY(expr)                                   \
  do {                                                 \
    cudaError_t _e = (expr);                           \
    if (_e != cudaSuccess) return cuda_failed(_e);     \
  } while (0)

struct GraphEntry {
  int N = -1, mode = 0, culling = 0;
  float d_min = 0, rho_p = 0, rho_theta = 0;
  const void* in = nullptr;            // H2D source and D2H destinations baked into the copy nodes
  void* out0 = nullptr;
  void* out1 = nullptr;
  void* out2 = nullptr;
  cudaGraphExec_t exec = nullptr;
  int kernels = 0;                     // kernel nodes (for the launch counter)
  unsigned long long stamp = 0;
};
constexpr int kGraphCache = 8;
constexpr int kCullMinPoses = 2048;     // the culled path serves larger batches only
constexpr int kHostBranches = 4;        // large host batches: up to this many {H2D, kernel, D2H} branches

// Per-call device workspace of the chunked kernels (cross-chunk keys, arrival counters) and the
// culled path's statistics.  The scene owns two: one for calls on the caller's stream
// (psdf_eval, psdf_eval_windows), one for the host entry points, which run on the scene's own
// stream and may therefore overlap an asynchronous psdf_eval still in flight.
struct Workspace {
  unsigned long long* depth = nullptr;   // [max_poses] clean = 0
  unsigned long long* d2 = nullptr;      // [max_poses] clean = ~0
  unsigned int* count = nullptr;         // [max_poses + 1] clean = 0
  unsigned int* traj = nullptr;          // [max_poses] per-trajectory arrival counters, clean = 0
  unsigned long long* stats = nullptr;   // [2]
};

}  // namespace

struct psdf_scene {
  int V = 0, Vp = 0, M = 0, E = 0, max_poses = 0;
  Footprint fp;
  int n_edges = 0, Mv = 0, n_empty = 0;
  int edge_cap = 0;
  int sm_count = 148;
  std::atomic<int> busy{0};           // one host thread at a time (PSDF_ERR_BUSY otherwise)
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
    GridHdr grid{};                   // host copy of *ghdr (travels in the launch parameters)
    bool grid_ok = false;             // the obstacle grid matches this set's bounds (built lazily)
  } pk[2];
  int cur = 0;
  int* h_win = nullptr;               // pinned [max_poses,2]  (psdf_eval_windows_host)
  int* d_win = nullptr;
  Workspace ws[2];                    // [0] caller-stream calls, [1] host entry points
  // streams psdf_eval / psdf_eval_windows were enqueued on since the last update: an update on
  // another stream cannot rely on stream order and synchronises the device instead
  cudaStream_t eval_stream = nullptr;
  bool eval_seen = false, eval_multi = false;
  // device packer scratch (psdf_pack_kernels.cuh)
  int* d_cnt = nullptr;               // [M] valid edges per row
  int4* d_offs = nullptr;             // [M] scanned offsets
  int* d_pair_begin = nullptr;        // [M+1]
  PackTotals* d_totals = nullptr;
  PackTotals* h_totals = nullptr;     // pinned
  GridHdr* h_ghdr = nullptr;          // pinned: read-back of a freshly built grid header
  int* h_pair_begin_pinned = nullptr; // pinned [M+1]
  int tune_bd = 0, tune_chunks = 0, tune_branches = 0, tune_cull_np = 0;   // measurement sweeps (PSDF_TUNING builds only)
  float grid_per_cell = 2.f;          // obstacles per cell of the culled path's grid (measured: DESIGN.md 6.7)
  int culling = 0;                    // psdf_set_culling
  // psdf_set_components: obstacle rows are convex components of n_groups obstacles
  int n_groups = 0;
  std::vector<int> h_comp;            // [M] row -> obstacle id, non-decreasing
  int* d_comp = nullptr;
  std::vector<int> h_row_slot;        // [M+1] host copy of the live set's row_slot (component mode)
  std::vector<int> h_slot_group;      // [Mv] packed obstacle -> obstacle id
  // host path
  bool host_ready = false;
  cudaStream_t gstream = nullptr;
  cudaStream_t bstream[kHostBranches] = {};      // side streams of the branched graph
  cudaEvent_t ev_fork = nullptr, ev_join[kHostBranches] = {};
  float* h_in = nullptr;              // pinned [max_poses,4]
  float* h_out = nullptr;             // pinned [max_poses,4]   value | grad  (or coeff)
  float* h_per = nullptr;             // pinned [max_poses,M]   lazily
  float* d_in = nullptr;
  float* d_out = nullptr;
  float* d_per = nullptr;
  int zero_copy = 1;                  // pinned staging is device-accessible (UVA): see run_zero_copy
  PoseArgs h_args;                    // the MPC host path's poses (N <= kArgPoses)
  GraphEntry graphs[kGraphCache];
  unsigned long long stamp = 0;
  // serving mode (psdf_serve_begin): persistent kernel on its own stream, mailbox in mapped memory
  struct Serve {
    bool on = false, running = false;
    int N = 0, mode = 0, K = 0, G = 0, bd = 0;
    float d_min = 0.f, rho_p = 0.f, rho_theta = 0.f;
    unsigned seq = 1;
    unsigned long long idle_ns = 0;
    cudaStream_t stream = nullptr;
    float4* in = nullptr;               // mapped [N]   (x, y, theta, sequence number)
    float4* out = nullptr;              // mapped [N]   (value, grad) or coefficient rows
    unsigned* ack = nullptr;            // mapped [2 G] (served sequence number, exited flag) per CTA
    int* d_win = nullptr;               // device [cap_N,2] per-pose obstacle row windows
    bool windows = false;
    int cap_N = 0, cap_G = 0;
  } srv;
};

static psdf_status serve_pause(psdf_scene* sc);   // stops the serving kernel (it holds scene pointers by value)

namespace {

struct BusyGuard {                      // concurrent use of one scene from two host threads is an error
  std::atomic<int>* f;
  bool ok;
  explicit BusyGuard(const psdf_scene* sc) : f(const_cast<std::atomic<int>*>(&sc->busy)) {
    int zero = 0;
    ok = f->compare_exchange_strong(zero, 1, std::memory_order_acquire);
  }
  ~BusyGuard() { if (ok) f->store(0, std::memory_order_release); }
};
#define PSDF_ENTER(sc)              \
  BusyGuard _busy(sc);              \
  if (!_busy.ok) return PSDF_ERR_BUSY

}  // namespace

namespace {

template <int V, int MODE>
cudaError_t launch_one(const psdf_scene* sc, const EvalParams& p, bool lanes, dim3 grid, int bd, cudaStream_t st,
                       const PoseArgs* args) {
  if (lanes && args)
    psdf_lanes_args_kernel<V, MODE><<<grid, bd, 0, st>>>(sc->fp, p, *args);
  else if (lanes)
    psdf_lanes_kernel<V, MODE><<<grid, bd, 0, st>>>(sc->fp, p);
  else
    psdf_scan_kernel<V, MODE><<<grid, bd, 0, st>>>(sc->fp, p);
  g_launches.fetch_add(1);
  return cudaGetLastError();
}

template <int V>
cudaError_t launch_mode(const psdf_scene* sc, const EvalParams& p, int mode, bool lanes, dim3 grid, int bd,
                        cudaStream_t st, const PoseArgs* args) {
  switch (mode) {
    case 0: return launch_one<V, 0>(sc, p, lanes, grid, bd, st, args);
    case kGrad: return launch_one<V, kGrad>(sc, p, lanes, grid, bd, st, args);
    case kPerObs: return launch_one<V, kPerObs>(sc, p, lanes, grid, bd, st, args);
    case kGrad | kPerObs: return launch_one<V, kGrad | kPerObs>(sc, p, lanes, grid, bd, st, args);
    case kCoeff: return launch_one<V, kCoeff>(sc, p, lanes, grid, bd, st, args);
    default: return cudaErrorInvalidValue;
  }
}

template <int V, int MODE, int NP>
cudaError_t launch_cull_one(const psdf_scene* sc, const EvalParams& p, cudaStream_t st) {
  constexpr int bytes = CullShape<V, NP>::kBytes;
  static bool opted_in = false;                  // > 48 KB of dynamic shared memory is opt-in, once per kernel
  if (!opted_in && bytes > 48 * 1024) {
    cudaError_t e = cudaFuncSetAttribute(psdf_cull_kernel<V, MODE, NP>, cudaFuncAttributeMaxDynamicSharedMemorySize, bytes);
    if (e != cudaSuccess) return e;
    opted_in = true;
  }
  const dim3 grid((unsigned)((p.N + NP - 1) / NP));
  psdf_cull_kernel<V, MODE, NP><<<grid, NP, bytes, st>>>(sc->fp, p);
  g_launches.fetch_add(1);
  return cudaGetLastError();
}

template <int V, int NP>
cudaError_t launch_cull_mode(const psdf_scene* sc, const EvalParams& p, int mode, cudaStream_t st) {
  switch (mode) {
    case 0: return launch_cull_one<V, 0, NP>(sc, p, st);
    case kGrad: return launch_cull_one<V, kGrad, NP>(sc, p, st);
    case kCoeff: return launch_cull_one<V, kCoeff, NP>(sc, p, st);
    default: return cudaErrorInvalidValue;
  }
}

template <int NP>
cudaError_t launch_cull_v(const psdf_scene* sc, const EvalParams& p, int mode, cudaStream_t st) {
  switch (sc->Vp) {
    case 4: return launch_cull_mode<4, NP>(sc, p, mode, st);
    case 6: return launch_cull_mode<6, NP>(sc, p, mode, st);
    case 8: return launch_cull_mode<8, NP>(sc, p, mode, st);
    case 10: return launch_cull_mode<10, NP>(sc, p, mode, st);
    case 12: return launch_cull_mode<12, NP>(sc, p, mode, st);
    case 16: return launch_cull_mode<16, (NP > 64 ? 64 : NP)>(sc, p, mode, st);   // (shared-memory budget)
    default: return cudaErrorInvalidValue;
  }
}

// Culled path: one launch.  Small batches take one warp per CTA so that they
// still spread over all SMs; large ones 128 poses per CTA (measured: cfg4 133 vs 146 us).
cudaError_t enqueue_culled(const psdf_scene* sc, EvalParams& p, int mode, cudaStream_t st) {
  p.gbounds = sc->pk[sc->cur].gbounds;
  p.gcell = sc->pk[sc->cur].gcell;
  p.grid = sc->pk[sc->cur].grid;
  p.n_chunks = 1;
#ifdef PSDF_TUNING
  if (sc->tune_cull_np == 32) return launch_cull_v<32>(sc, p, mode, st);
  if (sc->tune_cull_np == 64) return launch_cull_v<64>(sc, p, mode, st);
  if (sc->tune_cull_np == 128) return launch_cull_v<128>(sc, p, mode, st);
#endif
  if (p.N <= 32768) return launch_cull_v<32>(sc, p, mode, st);
  return launch_cull_v<128>(sc, p, mode, st);
}

cudaError_t launch_v(const psdf_scene* sc, const EvalParams& p, int mode, bool lanes, dim3 grid, int bd,
                     cudaStream_t st, const PoseArgs* args) {
  switch (sc->Vp) {
    case 4: return launch_mode<4>(sc, p, mode, lanes, grid, bd, st, args);
    case 6: return launch_mode<6>(sc, p, mode, lanes, grid, bd, st, args);
    case 8: return launch_mode<8>(sc, p, mode, lanes, grid, bd, st, args);
    case 10: return launch_mode<10>(sc, p, mode, lanes, grid, bd, st, args);
    case 12: return launch_mode<12>(sc, p, mode, lanes, grid, bd, st, args);
    case 16: return launch_mode<16>(sc, p, mode, lanes, grid, bd, st, args);
    default: return cudaErrorInvalidValue;
  }
}

// lane-split kernel: few poses or little work (measured crossover against the tile-scan kernel)
inline bool lanes_plan(const psdf_scene* sc, int N) {
  return N <= 128 || (long long)N * (sc->Mv > 0 ? sc->Mv : 1) <= (1 << 17);
}

// One evaluation to enqueue.  `which_ws`: 0 = caller-stream workspace, 1 = host-path workspace;
// `ws_off`: first workspace entry (branches of one host call use disjoint ranges).
struct EvalCall {
  const float* poses = nullptr;
  int N = 0;
  float* value = nullptr;
  float* grad = nullptr;
  float* per_obs = nullptr;
  float* coeff = nullptr;
  float d_min = 0.f, rho_p = 0.f, rho_theta = 0.f;
  float* packed = nullptr;            // zero-copy staging layout
  const int* window = nullptr;        // per-pose obstacle row windows
  const PoseArgs* args = nullptr;     // poses travelling as a kernel parameter
  int which_ws = 0, ws_off = 0;
  int traj_H = 0;                     // > 0: per-trajectory reductions fused into the tail
  float d_safe = 0.f;
  float* traj_min = nullptr;
  int* traj_argmin = nullptr;
  float* traj_penalty = nullptr;
};

// Launch plan: lane-split kernel for MPC-sized batches; otherwise the
// tile-scan kernel, with the obstacle range cut into chunks when the pose tiles alone
// would not fill 148 SMs several times over.
psdf_status enqueue_eval(const psdf_scene* sc, const EvalCall& c, cudaStream_t st) {
  const int N = c.N;
  if (N == 0) return PSDF_OK;
  const Workspace& ws = sc->ws[c.which_ws];
  float* const per_obs = c.per_obs;
  float* const coeff = c.coeff;
  float* const grad = c.grad;
  const int* const window = c.window;
  EvalParams p{};
  p.pairs = sc->pk[sc->cur].pairs;
  p.row_slot = sc->pk[sc->cur].row_slot;
  p.bounds = sc->pk[sc->cur].bounds;
  p.window = window;
  p.empty_rows = sc->pk[sc->cur].empty;
  p.poses = c.poses;
  p.value = c.value;
  p.grad = grad;
  p.per_obs = per_obs;
  p.coeff = coeff;
  p.packed = c.packed;
  p.ws_depth = ws.depth + c.ws_off;
  p.ws_d2 = ws.d2 + c.ws_off;
  p.ws_count = ws.count + c.ws_off;
  p.stats = ws.stats;
  p.n_edges = sc->n_edges;
  p.Mv = sc->Mv;
  p.M_rows = sc->M;
  p.n_empty = sc->n_empty;
  p.N = N;
  p.d_min = c.d_min;
  p.rho_p = c.rho_p;
  p.rho_theta = c.rho_theta;
  const bool fold = per_obs != nullptr && sc->n_groups > 0;       // per-obstacle output folded over components
  p.comp = fold ? sc->d_comp : nullptr;
  p.n_groups = fold ? sc->n_groups : 0;
  p.traj.H = c.traj_H;
  p.traj.d_safe = c.d_safe;
  p.traj.min_value = c.traj_min;
  p.traj.argmin_stage = c.traj_argmin;
  p.traj.penalty = c.traj_penalty;
  p.traj.count = ws.traj + c.ws_off;
  const int mode = coeff ? kCoeff : ((grad ? kGrad : 0) | (per_obs ? kPerObs : 0));

  const bool lanes = lanes_plan(sc, N) || window != nullptr;
  dim3 grid;
  int bd;
  // (the culled kernel packs a grid entry / pair record index into 24 bits next to the pose)
  if (sc->culling && !lanes && N > kCullMinPoses && !per_obs && sc->Mv >= 64 && sc->n_pairs < (1 << 24)) {
    cudaError_t e = enqueue_culled(sc, p, mode, st);
    if (e != cudaSuccess) return cuda_failed(e);
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
    if (fold) C = 1;                   // the lanes of a pose fold their components inside one CTA
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
#ifdef PSDF_TUNING
    if (sc->tune_bd > 0) bd = sc->tune_bd;                                   // measurement sweeps only
    if (sc->tune_chunks > 0) C = sc->tune_chunks;
#endif
    if (bd != 32 && bd != 64 && bd != 128 && bd != 256) bd = 64;
    if (C < 1) C = 1;
    if (C > maxC) C = maxC;
    if (C > kMaxChunks) C = kMaxChunks;
    const int tiles = (N + bd - 1) / bd;
    // chunk boundaries on obstacle boundaries, balanced by edge count
    // (component mode: also between obstacles, so that every (pose, obstacle) entry has one writer)
    p.chunk_begin[0] = 0;
    p.chunk_group[0] = 0;
    int o = 0;
    for (int c = 1; c < C; ++c) {
      const long long target = (long long)sc->n_pairs * c / C;
      while (o < sc->Mv && sc->h_pair_begin[o] < target) ++o;
      if (fold)
        while (o > 0 && o < sc->Mv && sc->h_slot_group[o] == sc->h_slot_group[o - 1]) ++o;
      p.chunk_begin[c] = sc->h_pair_begin[o];
      p.chunk_group[c] = fold ? (o < sc->Mv ? sc->h_slot_group[o] : sc->n_groups) : 0;
    }
    p.chunk_begin[C] = sc->n_pairs;
    p.chunk_group[C] = sc->n_groups;
    p.n_chunks = C;
    grid = dim3((unsigned)tiles, (unsigned)C);
  }
  cudaError_t e = launch_v(sc, p, mode, lanes, grid, bd, st, c.args);
  if (e != cudaSuccess) return cuda_failed(e);
  return PSDF_OK;
}

// The culled path's obstacle grid for buffer set `set`: built only while culling is
// switched on (psdf_set_culling, and every update from then on).
cudaError_t launch_grid(psdf_scene* sc, int set, const int* totals2, int Mv, int n_pairs, cudaStream_t st) {
  psdf_scene::Packed& b = sc->pk[set];
  obstacle_grid_kernel<<<1, 1024, 0, st>>>(b.bounds, Mv, n_pairs, totals2, b.gbounds, b.gcell, b.ghdr, sc->grid_per_cell);
  g_launches.fetch_add(1);
  cudaError_t e = cudaGetLastError();
  if (e == cudaSuccess) e = cudaMemcpyAsync(sc->h_ghdr, b.ghdr, sizeof(GridHdr), cudaMemcpyDeviceToHost, st);
  return e;                             // the caller synchronises `st`, then calls grid_built()
}

void grid_built(psdf_scene* sc, int set) {
  sc->pk[set].grid = *sc->h_ghdr;
  sc->pk[set].grid_ok = true;
}

// An update writes the inactive buffer set, which evaluations enqueued before the PREVIOUS update may
// still be reading if they ran on a stream other than `st`: stream order does not cover those.
psdf_status order_after_evals(psdf_scene* sc, cudaStream_t st) {
  if (sc->eval_multi || (sc->eval_seen && sc->eval_stream != st)) CU_TRY(cudaDeviceSynchronize());
  sc->eval_seen = sc->eval_multi = false;
  return PSDF_OK;
}

void note_eval_stream(const psdf_scene* csc, cudaStream_t st) {
  psdf_scene* sc = const_cast<psdf_scene*>(csc);
  if (!sc->eval_seen) { sc->eval_seen = true; sc->eval_stream = st; }
  else if (sc->eval_stream != st) sc->eval_multi = true;
}

// Component mode (psdf_set_components): packed obstacle -> obstacle id on the host, for chunk plans
// that end between obstacles.  `from_device`: the live set's row_slot has to be read back first.
psdf_status rebuild_component_tables(psdf_scene* sc, bool from_device) {
  if (sc->n_groups <= 0) return PSDF_OK;
  if (from_device) {
    sc->h_row_slot.resize((size_t)sc->M + 1);
    CU_TRY(cudaMemcpy(sc->h_row_slot.data(), sc->pk[sc->cur].row_slot, sizeof(int) * ((size_t)sc->M + 1), cudaMemcpyDeviceToHost));
  }
  sc->h_slot_group.assign((size_t)sc->Mv, 0);
  for (int i = 0; i < sc->M; ++i)
    if (sc->h_row_slot[i + 1] > sc->h_row_slot[i]) sc->h_slot_group[sc->h_row_slot[i]] = sc->h_comp[i];
  return PSDF_OK;
}

// Device-resident (A,B,S): pack on the GPU (count+validate -> scan -> write); only the
// totals and the per-obstacle pair offsets (for the host launch plan) come back.
psdf_status pack_on_device(psdf_scene* sc, const float* A, const float* B, const uint8_t* S, cudaStream_t st) {
  const int M = sc->M, E = sc->E;
  const int bd = 128, gd = (M + bd - 1) / bd;
  psdf_scene::Packed& dst = sc->pk[sc->cur ^ 1];            // the inactive set
  dst.grid_ok = false;
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
  if (sc->culling)                                           // reads {status, Mv} on the device: no extra sync
    CU_TRY(launch_grid(sc, sc->cur ^ 1, reinterpret_cast<const int*>(sc->d_totals), 0, 0, st));
  CU_TRY(cudaMemcpyAsync(sc->h_totals, sc->d_totals, sizeof(PackTotals) + sizeof(int) * ((size_t)M + 1),
                         cudaMemcpyDeviceToHost, st));
  CU_TRY(cudaStreamSynchronize(st));                         // the only synchronisation of an update
  CU_TRY(cudaGetLastError());
  const PackTotals t = *sc->h_totals;
  if (t.status != 0) return PSDF_ERR_DEGENERATE;             // the live set has not been touched
  if (sc->culling) grid_built(sc, sc->cur ^ 1);
  sc->h_pair_begin.assign(sc->h_pair_begin_pinned, sc->h_pair_begin_pinned + t.Mv + 1);
  sc->n_edges = t.n_edges;
  sc->Mv = t.Mv;
  sc->n_empty = t.n_empty;
  sc->n_pairs = t.n_pairs;
  sc->cur ^= 1;
  return rebuild_component_tables(sc, true);
}

psdf_status upload_scene(psdf_scene* sc, const float* A, const float* B, const uint8_t* S, psdf_mem where,
                         cudaStream_t st) {
  psdf_status s0 = order_after_evals(sc, st);
  if (s0 != PSDF_OK) return s0;
  if (where == PSDF_MEM_DEVICE) return pack_on_device(sc, A, B, S, st);
  PackedScene ps;
  if (pack_scene(A, B, S, sc->M, sc->E, ps) != 0) return PSDF_ERR_DEGENERATE;
  psdf_scene::Packed& dst = sc->pk[sc->cur ^ 1];
  dst.grid_ok = false;
  const int n_edges = (int)ps.edges.size(), Mv = (int)ps.row_begin.size() - 1, n_empty = (int)ps.empty_rows.size();
  const int n_pairs = (int)ps.pairs.size();
  // (dst.edges / dst.row_begin are the device packer's scratch: the kernels read pair records only)
  if (n_edges) CU_TRY(cudaMemcpyAsync(dst.pairs, ps.pairs.data(), sizeof(PairRec) * n_pairs, cudaMemcpyHostToDevice, st));
  CU_TRY(cudaMemcpyAsync(dst.row_slot, ps.row_slot.data(), sizeof(int) * (size_t)(sc->M + 1), cudaMemcpyHostToDevice, st));
  if (Mv) CU_TRY(cudaMemcpyAsync(dst.bounds, ps.bounds.data(), sizeof(float4) * 2 * Mv, cudaMemcpyHostToDevice, st));
  if (n_empty) CU_TRY(cudaMemcpyAsync(dst.empty, ps.empty_rows.data(), sizeof(int) * n_empty, cudaMemcpyHostToDevice, st));
  if (sc->culling) CU_TRY(launch_grid(sc, sc->cur ^ 1, nullptr, Mv, n_pairs, st));
  CU_TRY(cudaStreamSynchronize(st));       // the staging vectors die here
  if (sc->culling) grid_built(sc, sc->cur ^ 1);
  sc->n_edges = n_edges;
  sc->Mv = Mv;
  sc->n_empty = n_empty;
  sc->n_pairs = n_pairs;
  sc->h_pair_begin.swap(ps.pair_begin);
  sc->h_row_slot.swap(ps.row_slot);
  sc->cur ^= 1;
  return rebuild_component_tables(sc, false);
}

}  // namespace

// =============================================================================== C ABI
extern "C" {

void psdf_destroy_scene(psdf_scene* sc) {
  if (!sc) return;
  (void)serve_pause(sc);
  if (sc->srv.stream) cudaStreamDestroy(sc->srv.stream);
  if (sc->srv.in) cudaFreeHost(sc->srv.in);
  if (sc->srv.out) cudaFreeHost(sc->srv.out);
  if (sc->srv.ack) cudaFreeHost(sc->srv.ack);
  cudaFree(sc->srv.d_win);
  for (auto& g : sc->graphs)
    if (g.exec) cudaGraphExecDestroy(g.exec);
  if (sc->gstream) cudaStreamDestroy(sc->gstream);
  for (int b = 1; b < kHostBranches; ++b) {
    if (sc->bstream[b]) cudaStreamDestroy(sc->bstream[b]);
    if (sc->ev_join[b]) cudaEventDestroy(sc->ev_join[b]);
  }
  if (sc->ev_fork) cudaEventDestroy(sc->ev_fork);
  for (auto& b : sc->pk) {
    cudaFree(b.edges); cudaFree(b.pairs); cudaFree(b.row_begin); cudaFree(b.row_slot); cudaFree(b.empty); cudaFree(b.bounds);
    cudaFree(b.gbounds); cudaFree(b.gcell); cudaFree(b.ghdr);
  }
  cudaFree(sc->d_win);
  if (sc->h_totals) cudaFreeHost(sc->h_totals);
  if (sc->h_ghdr) cudaFreeHost(sc->h_ghdr);
  if (sc->h_win) cudaFreeHost(sc->h_win);
  for (auto& w : sc->ws) { cudaFree(w.depth); cudaFree(w.d2); cudaFree(w.count); cudaFree(w.traj); cudaFree(w.stats); }
  cudaFree(sc->d_comp);
  cudaFree(sc->d_cnt); cudaFree(sc->d_offs); cudaFree(sc->d_totals);   // d_pair_begin lives inside d_totals' block
  cudaFree(sc->d_in); cudaFree(sc->d_out); cudaFree(sc->d_per);
  if (sc->h_in) cudaFreeHost(sc->h_in);
  if (sc->h_out) cudaFreeHost(sc->h_out);
  if (sc->h_per) cudaFreeHost(sc->h_per);
  delete sc;
}

static psdf_status alloc_workspace(Workspace& w, int max_poses, cudaStream_t st) {
  const size_t n = (size_t)max_poses, n_cnt = n + 1;      // scan: one counter per pose tile; lanes: one per pose group
  CU_TRY(cudaMalloc(&w.depth, sizeof(unsigned long long) * n));
  CU_TRY(cudaMalloc(&w.d2, sizeof(unsigned long long) * n));
  CU_TRY(cudaMalloc(&w.count, sizeof(unsigned int) * n_cnt));
  CU_TRY(cudaMalloc(&w.traj, sizeof(unsigned int) * n));
  CU_TRY(cudaMalloc(&w.stats, sizeof(unsigned long long) * 2));
  CU_TRY(cudaMemsetAsync(w.traj, 0x00, sizeof(unsigned int) * n, st));
  CU_TRY(cudaMemsetAsync(w.depth, 0x00, sizeof(unsigned long long) * n, st));
  CU_TRY(cudaMemsetAsync(w.d2, 0xff, sizeof(unsigned long long) * n, st));
  CU_TRY(cudaMemsetAsync(w.count, 0x00, sizeof(unsigned int) * n_cnt, st));
  CU_TRY(cudaMemsetAsync(w.stats, 0x00, sizeof(unsigned long long) * 2, st));
  return PSDF_OK;
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
#ifdef PSDF_TUNING                                         // measurement sweeps only (not in product builds)
  if (const char* e = std::getenv("PSDF_BD")) sc->tune_bd = std::atoi(e);
  if (const char* e = std::getenv("PSDF_CHUNKS")) sc->tune_chunks = std::atoi(e);
  if (const char* e = std::getenv("PSDF_BRANCHES")) sc->tune_branches = std::atoi(e);
  if (const char* e = std::getenv("PSDF_CULL_NP")) sc->tune_cull_np = std::atoi(e);
  if (const char* e = std::getenv("PSDF_GRID_PER_CELL")) sc->grid_per_cell = (float)std::atof(e);
#endif
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
    CU_TRY(cudaMallocHost(&sc->h_ghdr, sizeof(GridHdr)));
    sc->h_pair_begin_pinned = reinterpret_cast<int*>(sc->h_totals + 1);
    CU_TRY(cudaMalloc(&sc->d_cnt, sizeof(int) * (size_t)M));
    CU_TRY(cudaMalloc(&sc->d_offs, sizeof(int4) * (size_t)M));
    CU_TRY(cudaMalloc(&sc->d_totals, sizeof(PackTotals) + sizeof(int) * (size_t)(M + 1)));
    sc->d_pair_begin = reinterpret_cast<int*>(sc->d_totals + 1);
    psdf_status s = alloc_workspace(sc->ws[0], max_poses, st);
    if (s != PSDF_OK) return s;
    return upload_scene(sc, A, B, S, where, st);
  };
  status = body();
  if (status != PSDF_OK) { psdf_destroy_scene(sc); return status; }
  *out = sc;
  return PSDF_OK;
}

static void drop_graphs(psdf_scene* sc) {      // launch plans and scene pointers are baked into the captured graphs
  for (auto& g : sc->graphs) {
    if (g.exec) cudaGraphExecDestroy(g.exec);
    g = GraphEntry();
  }
}

psdf_status psdf_update_scene(psdf_scene* sc, const float* A, const float* B, const uint8_t* S,
                              psdf_mem where, void* cuda_stream) {
  if (!sc || !A || !B || !S || (where != PSDF_MEM_HOST && where != PSDF_MEM_DEVICE)) return PSDF_ERR_INVALID_ARG;
  PSDF_ENTER(sc);
  // both paths validate before anything live changes (host: pack_scene; device: status word
  // checked before the buffer flip), so a bad update leaves the old scene in force
  cudaStream_t st = (cudaStream_t)cuda_stream;
  { const psdf_status sp = serve_pause(sc); if (sp != PSDF_OK) return sp; }   // (relaunched by the next psdf_serve_step)
  if (sc->gstream) CU_TRY(cudaStreamSynchronize(sc->gstream));
  psdf_status s = upload_scene(sc, A, B, S, where, st);
  if (s != PSDF_OK) return s;
  drop_graphs(sc);
  return PSDF_OK;
}

psdf_status psdf_eval(const psdf_scene* sc, const float* poses, int N, float* value, float* grad,
                      float* per_obstacle, void* cuda_stream) {
  if (!sc || N < 0 || (N > 0 && (!poses || !value))) return PSDF_ERR_INVALID_ARG;
  if (N > sc->max_poses) return PSDF_ERR_CAPACITY;
  PSDF_ENTER(sc);
  note_eval_stream(sc, (cudaStream_t)cuda_stream);
  EvalCall c;
  c.poses = poses; c.N = N; c.value = value; c.grad = grad; c.per_obs = per_obstacle;
  return enqueue_eval(sc, c, (cudaStream_t)cuda_stream);
}

// Host path resources: the scene's own stream, pinned (device-mapped) staging, device buffers, a
// private workspace, side streams for the branched graph.  All or nothing: `host_ready` is set last.
static psdf_status ensure_host_path(psdf_scene* sc, bool per_obs) {
  if (!sc->host_ready) {
    auto body = [&]() -> psdf_status {
      if (!sc->gstream) CU_TRY(cudaStreamCreateWithFlags(&sc->gstream, cudaStreamNonBlocking));
      for (int b = 1; b < kHostBranches; ++b) {
        if (!sc->bstream[b]) CU_TRY(cudaStreamCreateWithFlags(&sc->bstream[b], cudaStreamNonBlocking));
        if (!sc->ev_join[b]) CU_TRY(cudaEventCreateWithFlags(&sc->ev_join[b], cudaEventDisableTiming));
      }
      if (!sc->ev_fork) CU_TRY(cudaEventCreateWithFlags(&sc->ev_fork, cudaEventDisableTiming));
      if (!sc->h_in) CU_TRY(cudaHostAlloc(&sc->h_in, sizeof(float) * 4 * (size_t)sc->max_poses, cudaHostAllocMapped));
      if (!sc->h_out) CU_TRY(cudaHostAlloc(&sc->h_out, sizeof(float) * 4 * (size_t)sc->max_poses, cudaHostAllocMapped));
      int dev = 0, uva = 0;
      CU_TRY(cudaGetDevice(&dev));
      CU_TRY(cudaDeviceGetAttribute(&uva, cudaDevAttrUnifiedAddressing, dev));
#ifdef PSDF_TUNING
      if (const char* e = std::getenv("PSDF_NO_ZERO_COPY")) uva = (e[0] == '1') ? 0 : uva;
#endif
      sc->zero_copy = uva;
      if (!sc->d_in) CU_TRY(cudaMalloc(&sc->d_in, sizeof(float) * 3 * (size_t)sc->max_poses));
      if (!sc->d_out) CU_TRY(cudaMalloc(&sc->d_out, sizeof(float) * 4 * (size_t)sc->max_poses));
      if (!sc->ws[1].depth) {
        psdf_status s = alloc_workspace(sc->ws[1], sc->max_poses, sc->gstream);
        if (s != PSDF_OK) {                      // partial workspace: release it so that a retry starts clean
          Workspace& w = sc->ws[1];
          cudaFree(w.depth); cudaFree(w.d2); cudaFree(w.count); cudaFree(w.traj); cudaFree(w.stats);
          w = Workspace();
          return s;
        }
        CU_TRY(cudaStreamSynchronize(sc->gstream));
      }
      return PSDF_OK;
    };
    psdf_status s = body();
    if (s != PSDF_OK) return s;                  // whatever was created stays owned by the scene; nothing is used
    sc->host_ready = true;
  }
  if (per_obs && !sc->d_per) {
    float* h = nullptr;
    float* d = nullptr;
    CU_TRY(cudaHostAlloc(&h, sizeof(float) * (size_t)sc->max_poses * sc->M, cudaHostAllocMapped));
    cudaError_t e = cudaMalloc(&d, sizeof(float) * (size_t)sc->max_poses * sc->M);
    if (e != cudaSuccess) { cudaFreeHost(h); return cuda_failed(e); }
    sc->h_per = h;
    sc->d_per = d;
  }
  return PSDF_OK;
}

// MPC-sized batches: ONE kernel launch that reads the poses from, and writes the results to,
// the pinned (mapped) staging buffers directly: a few hundred bytes cross PCIe inside the
// kernel instead of through two copy-engine operations, which removes two graph nodes'
// worth of latency.
constexpr int kZeroCopyMaxPoses = 512;
constexpr int kZeroCopyMaxObstaclesPerObs = 64;

// Measured on B200 (bench.py mpc_latency, Table-I shapes up to 1000 obstacles): the single launch
// beats the 3-node graph by 4-7 us whenever the batch is MPC sized; only the [N,M] per-obstacle
// output of a large scene stays on the copy engine (scattered 4-byte stores over PCIe otherwise).
static inline bool use_zero_copy(const psdf_scene* sc, int N, bool per_obs) {
  return sc->zero_copy && N <= kZeroCopyMaxPoses && lanes_plan(sc, N) &&      // (the lane-split kernel reads the staging layout)
         (!per_obs || sc->Mv <= kZeroCopyMaxObstaclesPerObs);
}

// What one host call wants: caller's buffers (ordinary or pinned host memory) and constants.
struct HostCall {
  const float* poses = nullptr;
  int N = 0, mode = 0;
  float* value = nullptr;
  float* grad = nullptr;
  float* per = nullptr;
  float* coeff = nullptr;
  float d_min = 0.f, rho_p = 0.f, rho_theta = 0.f;
};

// Result rows in mapped memory are watched as they arrive instead of waiting for the stream: the host blanks
// them with a NaN bit pattern that no kernel result carries (the kernels' own NaNs are 0x7fc00000 and
// 0x7fffffff) and accepts a row when none of its four words is the pattern any more.
constexpr unsigned kRowSentinel = 0x7fa5a5a5u;

// Spins until rows [0, N) of `rows` hold no sentinel word.  The stream is asked now and then: an error ends
// the wait; a stream that has finished leaves at most one more pass (its writes are visible by then).
static psdf_status wait_rows(const float4* rows, int N, cudaStream_t st) {
  const __m128i sentinel = _mm_set1_epi32((int)kRowSentinel);
  bool finished = false;
  for (int n = 0; n < N; ++n) {
    const __m128i* row = reinterpret_cast<const __m128i*>(rows + n);
    unsigned spins = 0;
    while (_mm_movemask_epi8(_mm_cmpeq_epi32(_mm_load_si128(const_cast<const __m128i*>(
               reinterpret_cast<const volatile __m128i*>(row))), sentinel)) != 0) {
      _mm_pause();
      if ((++spins & 0x3ffu) != 0u) continue;
      if (finished) return PSDF_ERR_CUDA;                     // the kernel is done and the row is still blank
      const cudaError_t e = cudaStreamQuery(st);
      if (e == cudaSuccess) finished = true;
      else if (e != cudaErrorNotReady) return cuda_failed(e);
    }
  }
  return PSDF_OK;
}

static psdf_status run_zero_copy(psdf_scene* sc, const HostCall& h) {
  // staging layout: h_in [N,4] poses (padded), h_out [N,4] = (value, grad) or coefficients;
  // up to kArgPoses poses go into the launch itself (kernel parameter) instead
  const int N = h.N;
  if (N <= kArgPoses) {
    for (int n = 0; n < N; ++n) sc->h_args.q[n] = make_float4(h.poses[3 * n], h.poses[3 * n + 1], h.poses[3 * n + 2], 0.f);
  } else {
    for (int n = 0; n < N; ++n) {
      sc->h_in[4 * n] = h.poses[3 * n]; sc->h_in[4 * n + 1] = h.poses[3 * n + 1];
      sc->h_in[4 * n + 2] = h.poses[3 * n + 2]; sc->h_in[4 * n + 3] = 0.f;
    }
  }
  EvalCall c;
  c.poses = sc->h_in; c.N = N;
  c.grad = (h.mode & kGrad) ? sc->d_out : nullptr;            // (non-null = wanted; results go to `packed`)
  c.per_obs = (h.mode & kPerObs) ? sc->h_per : nullptr;
  c.coeff = (h.mode & kCoeff) ? sc->h_out : nullptr;
  c.d_min = h.d_min; c.rho_p = h.rho_p; c.rho_theta = h.rho_theta;
  c.packed = sc->h_out;
  c.args = N <= kArgPoses ? &sc->h_args : nullptr;
  c.which_ws = 1;
  const bool watch = !(h.mode & kPerObs);                     // ([N,M] per-obstacle output: wait for the stream)
  if (watch) {
    const __m128i sentinel = _mm_set1_epi32((int)kRowSentinel);
    for (int n = 0; n < N; ++n) _mm_store_si128(reinterpret_cast<__m128i*>(sc->h_out) + n, sentinel);
    _mm_sfence();
  }
  psdf_status s = enqueue_eval(sc, c, sc->gstream);
  if (s != PSDF_OK) return s;
  if (watch) {
    s = wait_rows(reinterpret_cast<const float4*>(sc->h_out), N, sc->gstream);
    if (s != PSDF_OK) return s;
  } else {
    CU_TRY(cudaStreamSynchronize(sc->gstream));
  }
  if (h.mode & kCoeff) {
    std::memcpy(h.coeff, sc->h_out, sizeof(float) * 4 * (size_t)N);
  } else {
    for (int n = 0; n < N; ++n) {
      h.value[n] = sc->h_out[4 * n];
      if (h.grad) { h.grad[3 * n] = sc->h_out[4 * n + 1]; h.grad[3 * n + 1] = sc->h_out[4 * n + 2]; h.grad[3 * n + 2] = sc->h_out[4 * n + 3]; }
    }
  }
  if (h.per) std::memcpy(h.per, sc->h_per, sizeof(float) * (size_t)N * (sc->n_groups > 0 ? sc->n_groups : sc->M));
  return PSDF_OK;
}

// Pinned (page-locked, e.g. cudaHostAlloc / cudaHostRegister / torch pin_memory) caller memory can
// be the source / destination of the copy nodes directly: no staging memcpy on the host.
static bool is_pinned_host(const void* ptr) {
  if (!ptr) return false;
  cudaPointerAttributes a;
  if (cudaPointerGetAttributes(&a, ptr) != cudaSuccess) { (void)cudaGetLastError(); return false; }
  return a.type == cudaMemoryTypeHost;
}

// Large host batches: replay of a captured CUDA graph with K branches, each {H2D pose chunk,
// kernel on that chunk, D2H result chunk}, so that the copies of one chunk overlap the kernels of
// the others (two copy engines + SMs busy at once).  Per-pose results do not depend on the batch
// they are evaluated in, so the chunked results are bit-identical to one psdf_eval over all N.
// Captured once per (N, outputs, constants, buffers); pinned caller buffers are used in place.
static psdf_status run_graph(psdf_scene* sc, const HostCall& h) {
  const int N = h.N, mode = h.mode;
  const size_t M = (size_t)(sc->n_groups > 0 ? sc->n_groups : sc->M);   // row length of the per-obstacle output
  // sources / destinations of the copy nodes
  const bool pin_in = is_pinned_host(h.poses);
  const float* src = pin_in ? h.poses : sc->h_in;
  float* dst0 = nullptr;      // value [N] or coeff [N,4]
  float* dst1 = nullptr;      // grad [N,3]
  float* dst2 = nullptr;      // per_obstacle [N,M]
  if (mode & kCoeff) dst0 = is_pinned_host(h.coeff) ? h.coeff : sc->h_out;
  else {
    dst0 = is_pinned_host(h.value) ? h.value : sc->h_out;
    if (mode & kGrad) dst1 = is_pinned_host(h.grad) ? h.grad : sc->h_out + N;
    if (mode & kPerObs) dst2 = is_pinned_host(h.per) ? h.per : sc->h_per;
  }
  if (!pin_in) std::memcpy(sc->h_in, h.poses, sizeof(float) * 3 * (size_t)N);

  GraphEntry* hit = nullptr;
  GraphEntry* victim = &sc->graphs[0];
  for (auto& g : sc->graphs) {
    if (g.exec && g.N == N && g.mode == mode && g.culling == sc->culling && g.d_min == h.d_min && g.rho_p == h.rho_p &&
        g.rho_theta == h.rho_theta && g.in == src && g.out0 == dst0 && g.out1 == dst1 && g.out2 == dst2) {
      hit = &g;
      break;
    }
    if (g.stamp < victim->stamp) victim = &g;
  }
  if (!hit) {
    if (victim->exec) { cudaGraphExecDestroy(victim->exec); *victim = GraphEntry(); }
    // branches: chunk boundaries on multiples of 128 poses (a CTA of either kernel never straddles one)
    int K = N >= 32768 ? 4 : (N >= 8192 ? 2 : 1);
#ifdef PSDF_TUNING
    if (sc->tune_branches > 0) K = sc->tune_branches;
#endif
    if (K > kHostBranches) K = kHostBranches;
    const int per = ((N + K - 1) / K + 127) / 128 * 128;
    cudaGraph_t graph = nullptr;
    cudaStream_t g0 = sc->gstream;
    const long long launches0 = g_launches.load();
    CU_TRY(cudaStreamBeginCapture(g0, cudaStreamCaptureModeThreadLocal));
    cudaError_t e = cudaSuccess;
    psdf_status s = PSDF_OK;
    int forked = 0;
    if (K > 1) e = cudaEventRecord(sc->ev_fork, g0);
    for (int b = 0; b < K && e == cudaSuccess && s == PSDF_OK; ++b) {
      const int n0 = b * per, n = (n0 + per <= N ? per : N - n0);
      if (n <= 0) break;
      cudaStream_t st = b == 0 ? g0 : sc->bstream[b];
      if (b > 0) { e = cudaStreamWaitEvent(st, sc->ev_fork, 0); if (e != cudaSuccess) break; forked = b; }
      e = cudaMemcpyAsync(sc->d_in + 3 * (size_t)n0, src + 3 * (size_t)n0, sizeof(float) * 3 * (size_t)n, cudaMemcpyHostToDevice, st);
      if (e != cudaSuccess) break;
      EvalCall c;
      c.poses = sc->d_in + 3 * (size_t)n0; c.N = n; c.which_ws = 1; c.ws_off = n0;
      if (mode & kCoeff) {
        c.coeff = sc->d_out + 4 * (size_t)n0;
        c.d_min = h.d_min; c.rho_p = h.rho_p; c.rho_theta = h.rho_theta;
      } else {
        c.value = sc->d_out + n0;
        if (mode & kGrad) c.grad = sc->d_out + N + 3 * (size_t)n0;
        if (mode & kPerObs) c.per_obs = sc->d_per + (size_t)n0 * M;
      }
      s = enqueue_eval(sc, c, st);
      if (s != PSDF_OK) break;
      if (mode & kCoeff) {
        e = cudaMemcpyAsync(dst0 + 4 * (size_t)n0, c.coeff, sizeof(float) * 4 * (size_t)n, cudaMemcpyDeviceToHost, st);
      } else {
        e = cudaMemcpyAsync(dst0 + n0, c.value, sizeof(float) * (size_t)n, cudaMemcpyDeviceToHost, st);
        if (e == cudaSuccess && (mode & kGrad))
          e = cudaMemcpyAsync(dst1 + 3 * (size_t)n0, c.grad, sizeof(float) * 3 * (size_t)n, cudaMemcpyDeviceToHost, st);
        if (e == cudaSuccess && (mode & kPerObs))
          e = cudaMemcpyAsync(dst2 + (size_t)n0 * M, c.per_obs, sizeof(float) * (size_t)n * M, cudaMemcpyDeviceToHost, st);
      }
    }
    for (int b = 1; b <= forked; ++b) {                  // join every forked branch, also on failure
      cudaError_t ej = cudaEventRecord(sc->ev_join[b], sc->bstream[b]);
      if (ej == cudaSuccess) ej = cudaStreamWaitEvent(g0, sc->ev_join[b], 0);
      if (e == cudaSuccess) e = ej;
    }
    cudaError_t e2 = cudaStreamEndCapture(g0, &graph);
    const int kernels = (int)(g_launches.load() - launches0);
    g_launches.fetch_sub(kernels);                       // captured, not run: counted per replay below
    if (e != cudaSuccess || e2 != cudaSuccess || s != PSDF_OK || !graph) {
      if (graph) cudaGraphDestroy(graph);
      if (s != PSDF_OK) { (void)cudaGetLastError(); return s; }
      return cuda_failed(e != cudaSuccess ? e : (e2 != cudaSuccess ? e2 : cudaErrorUnknown));
    }
    cudaGraphExec_t exec = nullptr;
    e = cudaGraphInstantiate(&exec, graph, 0);
    cudaGraphDestroy(graph);
    CU_TRY(e);
    victim->exec = exec; victim->N = N; victim->mode = mode; victim->culling = sc->culling;
    victim->d_min = h.d_min; victim->rho_p = h.rho_p; victim->rho_theta = h.rho_theta;
    victim->kernels = kernels;
    victim->in = src; victim->out0 = dst0; victim->out1 = dst1; victim->out2 = dst2;
    hit = victim;
  }
  hit->stamp = ++sc->stamp;
  CU_TRY(cudaGraphLaunch(hit->exec, sc->gstream));
  g_launches.fetch_add(hit->kernels);
  CU_TRY(cudaStreamSynchronize(sc->gstream));
  // ordinary (pageable) caller memory: results come back through the pinned staging buffers
  if (mode & kCoeff) {
    if (dst0 != h.coeff) std::memcpy(h.coeff, sc->h_out, sizeof(float) * 4 * (size_t)N);
  } else {
    if (dst0 != h.value) std::memcpy(h.value, sc->h_out, sizeof(float) * (size_t)N);
    if ((mode & kGrad) && dst1 != h.grad) std::memcpy(h.grad, sc->h_out + N, sizeof(float) * 3 * (size_t)N);
    if ((mode & kPerObs) && dst2 != h.per) std::memcpy(h.per, sc->h_per, sizeof(float) * (size_t)N * M);
  }
  return PSDF_OK;
}

// Device-side address of a pinned (page-locked) host buffer, or null if the memory is not pinned.
static void* pinned_device_ptr(const void* ptr) {
  if (!ptr) return nullptr;
  cudaPointerAttributes a;
  if (cudaPointerGetAttributes(&a, ptr) != cudaSuccess) { (void)cudaGetLastError(); return nullptr; }
  return a.type == cudaMemoryTypeHost ? a.devicePointer : nullptr;
}

// Large batches on the culled path: one launch, no copy engine.  The culled kernel
// reads every pose once and writes every result once, so it can do both over PCIe itself (coalesced 384-byte
// reads / writes per warp), and transfer and evaluation overlap CTA by CTA instead of branch by branch.
// (The dense tile-scan kernel reads a pose once per obstacle chunk: it keeps the copy-engine graph.)
// Buffers that are not pinned go through the scene's pinned, device-mapped staging (one host copy each way).
struct DirectPlan {
  EvalCall c;
  bool stage_value = false, stage_grad = false, stage_coeff = false;
};

static bool takes_direct(psdf_scene* sc, const HostCall& h, DirectPlan& d) {
  if (!sc->culling || (h.mode & kPerObs) || lanes_plan(sc, h.N) || h.N <= kCullMinPoses || sc->Mv < 64 ||
      sc->n_pairs >= (1 << 24) || !sc->zero_copy)
    return false;                                           // (not the culled path: see enqueue_eval)
  EvalCall& c = d.c;
  const size_t N = (size_t)h.N;
  c.poses = static_cast<const float*>(pinned_device_ptr(h.poses));
  if (!c.poses) {
    std::memcpy(sc->h_in, h.poses, sizeof(float) * 3 * N);
    c.poses = sc->h_in;
  }
  if (h.mode & kCoeff) {
    c.coeff = static_cast<float*>(pinned_device_ptr(h.coeff));
    if (!c.coeff) { c.coeff = sc->h_out; d.stage_coeff = true; }
    c.value = c.coeff;                                      // (not written in coefficient mode)
    c.d_min = h.d_min; c.rho_p = h.rho_p; c.rho_theta = h.rho_theta;
  } else {
    c.value = static_cast<float*>(pinned_device_ptr(h.value));
    if (!c.value) { c.value = sc->h_out; d.stage_value = true; }
    if (h.mode & kGrad) {
      c.grad = static_cast<float*>(pinned_device_ptr(h.grad));
      if (!c.grad) { c.grad = sc->h_out + N; d.stage_grad = true; }
    }
  }
  c.N = h.N;
  c.which_ws = 1;
  return true;
}

static psdf_status run_host(psdf_scene* sc, const HostCall& h) {
  psdf_status s = ensure_host_path(sc, (h.mode & kPerObs) != 0);
  if (s != PSDF_OK) return s;
  if (use_zero_copy(sc, h.N, (h.mode & kPerObs) != 0)) return run_zero_copy(sc, h);
  DirectPlan direct;
  if (takes_direct(sc, h, direct)) {
    s = enqueue_eval(sc, direct.c, sc->gstream);
    if (s != PSDF_OK) return s;
    CU_TRY(cudaStreamSynchronize(sc->gstream));
    const size_t N = (size_t)h.N;
    if (direct.stage_coeff) std::memcpy(h.coeff, sc->h_out, sizeof(float) * 4 * N);
    if (direct.stage_value) std::memcpy(h.value, sc->h_out, sizeof(float) * N);
    if (direct.stage_grad) std::memcpy(h.grad, sc->h_out + N, sizeof(float) * 3 * N);
    return PSDF_OK;
  }
  return run_graph(sc, h);
}

psdf_status psdf_eval_host(psdf_scene* sc, const float* poses, int N, float* value, float* grad,
                           float* per_obstacle) {
  if (!sc || N < 0 || (N > 0 && (!poses || !value))) return PSDF_ERR_INVALID_ARG;
  if (N > sc->max_poses) return PSDF_ERR_CAPACITY;
  if (N == 0) return PSDF_OK;
  PSDF_ENTER(sc);
  HostCall h;
  h.poses = poses; h.N = N; h.value = value; h.grad = grad; h.per = per_obstacle;
  h.mode = (grad ? kGrad : 0) | (per_obstacle ? kPerObs : 0);
  return run_host(sc, h);
}

psdf_status psdf_mpc_coeffs_host(psdf_scene* sc, const float* poses, int N, float d_min, float rho_p,
                                 float rho_theta, float* coeff) {
  if (!sc || N < 0 || (N > 0 && (!poses || !coeff))) return PSDF_ERR_INVALID_ARG;
  if (N > sc->max_poses) return PSDF_ERR_CAPACITY;
  if (N == 0) return PSDF_OK;
  PSDF_ENTER(sc);
  HostCall h;
  h.poses = poses; h.N = N; h.coeff = coeff; h.mode = kCoeff;
  h.d_min = d_min; h.rho_p = rho_p; h.rho_theta = rho_theta;
  return run_host(sc, h);
}

psdf_status psdf_eval_windows(const psdf_scene* sc, const float* poses, int N, const int* row_window, float* value,
                              float* grad, void* cuda_stream) {
  if (!sc || N < 0 || (N > 0 && (!poses || !value || !row_window))) return PSDF_ERR_INVALID_ARG;
  if (N > sc->max_poses) return PSDF_ERR_CAPACITY;
  PSDF_ENTER(sc);
  note_eval_stream(sc, (cudaStream_t)cuda_stream);
  EvalCall c;
  c.poses = poses; c.N = N; c.value = value; c.grad = grad; c.window = row_window;
  return enqueue_eval(sc, c, (cudaStream_t)cuda_stream);
}

psdf_status psdf_eval_windows_host(psdf_scene* sc, const float* poses, int N, const int* row_window, float* value,
                                   float* grad) {
  if (!sc || N < 0 || (N > 0 && (!poses || !value || !row_window))) return PSDF_ERR_INVALID_ARG;
  if (N > sc->max_poses) return PSDF_ERR_CAPACITY;
  if (N == 0) return PSDF_OK;
  PSDF_ENTER(sc);
  psdf_status s = ensure_host_path(sc, false);
  if (s != PSDF_OK) return s;
  if (!sc->h_win) {
    int* h = nullptr;
    int* d = nullptr;
    CU_TRY(cudaMallocHost(&h, sizeof(int) * 2 * (size_t)sc->max_poses));
    cudaError_t e = cudaMalloc(&d, sizeof(int) * 2 * (size_t)sc->max_poses);
    if (e != cudaSuccess) { cudaFreeHost(h); return cuda_failed(e); }
    sc->h_win = h;
    sc->d_win = d;
  }
  std::memcpy(sc->h_in, poses, sizeof(float) * 3 * (size_t)N);
  std::memcpy(sc->h_win, row_window, sizeof(int) * 2 * (size_t)N);
  cudaStream_t st = sc->gstream;
  CU_TRY(cudaMemcpyAsync(sc->d_in, sc->h_in, sizeof(float) * 3 * (size_t)N, cudaMemcpyHostToDevice, st));
  CU_TRY(cudaMemcpyAsync(sc->d_win, sc->h_win, sizeof(int) * 2 * (size_t)N, cudaMemcpyHostToDevice, st));
  EvalCall c;
  c.poses = sc->d_in; c.N = N; c.value = sc->d_out; c.grad = grad ? sc->d_out + N : nullptr; c.window = sc->d_win;
  c.which_ws = 1;
  s = enqueue_eval(sc, c, st);
  if (s != PSDF_OK) return s;
  CU_TRY(cudaMemcpyAsync(sc->h_out, sc->d_out, sizeof(float) * (grad ? 4 : 1) * (size_t)N, cudaMemcpyDeviceToHost, st));
  CU_TRY(cudaStreamSynchronize(st));
  std::memcpy(value, sc->h_out, sizeof(float) * (size_t)N);
  if (grad) std::memcpy(grad, sc->h_out + N, sizeof(float) * 3 * (size_t)N);
  return PSDF_OK;
}

psdf_status psdf_set_culling(psdf_scene* sc, int enable) {
  if (!sc) return PSDF_ERR_INVALID_ARG;
  PSDF_ENTER(sc);
  { const psdf_status sp = serve_pause(sc); if (sp != PSDF_OK) return sp; }
  if (sc->gstream) CU_TRY(cudaStreamSynchronize(sc->gstream));
  if (enable && !sc->pk[sc->cur].grid_ok) {      // built here, then kept current by every update
    CU_TRY(launch_grid(sc, sc->cur, nullptr, sc->Mv, sc->n_pairs, (cudaStream_t)0));
    CU_TRY(cudaStreamSynchronize((cudaStream_t)0));
    grid_built(sc, sc->cur);
  }
  sc->culling = enable ? 1 : 0;
  drop_graphs(sc);
  return PSDF_OK;
}

psdf_status psdf_set_components(psdf_scene* sc, const int* comp_to_obstacle, int n_obstacles) {
  if (!sc || n_obstacles < 0 || (n_obstacles > 0 && !comp_to_obstacle)) return PSDF_ERR_INVALID_ARG;
  PSDF_ENTER(sc);
  if (n_obstacles > 0) {
    if (n_obstacles > sc->M) return PSDF_ERR_INVALID_ARG;
    for (int i = 0; i < sc->M; ++i)
      if (comp_to_obstacle[i] < 0 || comp_to_obstacle[i] >= n_obstacles || (i > 0 && comp_to_obstacle[i] < comp_to_obstacle[i - 1]))
        return PSDF_ERR_INVALID_ARG;                  // components of one obstacle are consecutive rows
  }
  { const psdf_status sp = serve_pause(sc); if (sp != PSDF_OK) return sp; }   // (cudaDeviceSynchronize below)
  if (sc->gstream) CU_TRY(cudaStreamSynchronize(sc->gstream));
  drop_graphs(sc);
  if (n_obstacles == 0) { sc->n_groups = 0; return PSDF_OK; }
  if (!sc->d_comp) CU_TRY(cudaMalloc(&sc->d_comp, sizeof(int) * (size_t)sc->M));
  CU_TRY(cudaDeviceSynchronize());                    // (evaluations in flight may still read the old map)
  CU_TRY(cudaMemcpy(sc->d_comp, comp_to_obstacle, sizeof(int) * (size_t)sc->M, cudaMemcpyHostToDevice));
  sc->h_comp.assign(comp_to_obstacle, comp_to_obstacle + sc->M);
  sc->n_groups = n_obstacles;
  const psdf_status s = rebuild_component_tables(sc, true);
  if (s != PSDF_OK) sc->n_groups = 0;
  return s;
}

psdf_status psdf_eval_trajectories(const psdf_scene* sc, const float* poses, int T, int H, float d_safe, float* value,
                                   float* grad, float* min_value, int* argmin_stage, float* penalty, void* cuda_stream) {
  if (!sc || T < 0 || H < 1 || (T > 0 && (!poses || !value))) return PSDF_ERR_INVALID_ARG;
  if ((long long)T * H > sc->max_poses) return PSDF_ERR_CAPACITY;
  if (T == 0) return PSDF_OK;
  PSDF_ENTER(sc);
  note_eval_stream(sc, (cudaStream_t)cuda_stream);
  EvalCall c;
  c.poses = poses; c.N = T * H; c.value = value; c.grad = grad;
  c.traj_H = H; c.d_safe = d_safe; c.traj_min = min_value; c.traj_argmin = argmin_stage; c.traj_penalty = penalty;
  return enqueue_eval(sc, c, (cudaStream_t)cuda_stream);
}

psdf_status psdf_component_min(const float* per_component, int N, int M, const int* comp_to_obstacle,
                               int n_obstacles, float* out, void* cuda_stream) {
  if (N < 0 || M < 1 || n_obstacles < 1 || (N > 0 && (!per_component || !comp_to_obstacle || !out)))
    return PSDF_ERR_INVALID_ARG;
  if (N == 0) return PSDF_OK;
  component_min_kernel<<<(unsigned)N, 128, 0, (cudaStream_t)cuda_stream>>>(per_component, N, M, comp_to_obstacle,
                                                                          n_obstacles, out);
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
  PSDF_ENTER(sc);
  cudaStream_t st = (cudaStream_t)cuda_stream;
  if (sc->gstream) CU_TRY(cudaStreamSynchronize(sc->gstream));
  out2[0] = out2[1] = 0ull;
  for (const Workspace& w : sc->ws) {            // caller-stream and host-path evaluations
    if (!w.stats) continue;
    unsigned long long v[2] = {0ull, 0ull};
    CU_TRY(cudaMemcpyAsync(v, w.stats, sizeof(v), cudaMemcpyDeviceToHost, st));
    CU_TRY(cudaMemsetAsync(w.stats, 0, sizeof(v), st));
    CU_TRY(cudaStreamSynchronize(st));
    out2[0] += v[0];
    out2[1] += v[1];
  }
  return PSDF_OK;
}

int psdf_scene_num_obstacles(const psdf_scene* sc) { return sc ? sc->Mv : 0; }
int psdf_scene_num_edges(const psdf_scene* sc) { return sc ? sc->n_edges : 0; }
int psdf_scene_footprint_symmetric(const psdf_scene* sc) { return sc ? sc->fp.sym : 0; }
int psdf_last_cuda_error(void) { return g_last_cuda_error.load(); }
long long psdf_kernel_launches(void) { return g_launches.load(); }
const char* psdf_version(void) { return "psdf-b200 0.2 (sm_100a)"; }

const char* psdf_status_string(psdf_status s) {
  switch (s) {
    case PSDF_OK: return "ok";
    case PSDF_ERR_INVALID_ARG: return "invalid argument";
    case PSDF_ERR_DEGENERATE: return "degenerate geometry (Assumption 1 violated)";
    case PSDF_ERR_CAPACITY: return "N exceeds max_poses";
    case PSDF_ERR_CUDA: return "CUDA error";
    case PSDF_ERR_ALLOC: return "allocation failed";
    case PSDF_ERR_BUSY: return "scene in use by another host thread";
  }
  return "unknown status";
}

psdf_status psdf_bench_host_latency(psdf_scene* sc, const float* poses, int N, float* value, float* grad,
                                    float* per_obstacle, float* coeff, float d_min, float rho_p, float rho_theta,
                                    int reps, double* out_us) {
  if (!sc || !out_us || reps < 1) return PSDF_ERR_INVALID_ARG;
  for (int r = 0; r < reps; ++r) {
    const auto t0 = std::chrono::steady_clock::now();
    const psdf_status s = coeff ? psdf_mpc_coeffs_host(sc, poses, N, d_min, rho_p, rho_theta, coeff)
                                : psdf_eval_host(sc, poses, N, value, grad, per_obstacle);
    const auto t1 = std::chrono::steady_clock::now();
    if (s != PSDF_OK) return s;
    out_us[r] = std::chrono::duration<double, std::micro>(t1 - t0).count();
  }
  return PSDF_OK;
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

// ====================================================================== no-allocation entry point
// psdf_eval_static_scratch (include/psdf.h): the chunked tile-scan evaluation with its scratch (the
// cross-chunk arg-max / arg-min keys and the per-tile arrival counters) in a file-scope device array
// instead of a cudaMalloc'ed workspace.  Every GPU that loads the library holds the array until exit.
namespace {

constexpr int kStaticMaxPoses = PSDF_STATIC_SCRATCH_MAX_POSES;
constexpr int kStaticTile = 64;                              // poses per CTA of the tile-scan kernel
struct StaticScratch {
  unsigned long long depth[kStaticMaxPoses];                 // must start at 0
  unsigned long long d2[kStaticMaxPoses];                    // must start at ~0
  unsigned int count[kStaticMaxPoses / kStaticTile + 64];    // must start at 0
};
static __device__ __align__(256) unsigned char g_static_scratch[sizeof(StaticScratch)];   // 1.03 MB

// In host code `g_static_scratch` is a host-side stand-in, not a device address: the address the
// kernels get comes from cudaGetSymbolAddress, once per device, with that device current.
constexpr int kMaxDevices = 64;
std::atomic<StaticScratch*> g_static_ptr[kMaxDevices];

psdf_status static_scratch_ptr(StaticScratch** out) {
  int dev = 0;
  CU_TRY(cudaGetDevice(&dev));
  if (dev < 0 || dev >= kMaxDevices) return PSDF_ERR_INVALID_ARG;
  StaticScratch* ptr = g_static_ptr[dev].load(std::memory_order_acquire);
  if (!ptr) {
    void* sym = nullptr;
    CU_TRY(cudaGetSymbolAddress(&sym, g_static_scratch));   // (allocates nothing; same answer from every thread)
    if (!sym) return PSDF_ERR_CUDA;
    ptr = static_cast<StaticScratch*>(sym);
    g_static_ptr[dev].store(ptr, std::memory_order_release);
  }
  *out = ptr;
  return PSDF_OK;
}

}  // namespace

extern "C" psdf_status psdf_eval_static_scratch(const psdf_scene* sc, const float* poses, int N, float* value,
                                                float* grad, void* cuda_stream) {
  if (!sc || N < 0 || (N > 0 && (!poses || !value))) return PSDF_ERR_INVALID_ARG;
  if (N > kStaticMaxPoses) return PSDF_ERR_CAPACITY;         // beyond the static array: rejected, nothing done
  if (N == 0) return PSDF_OK;
  PSDF_ENTER(sc);
  cudaStream_t st = (cudaStream_t)cuda_stream;
  StaticScratch* ss = nullptr;
  psdf_status s = static_scratch_ptr(&ss);
  if (s != PSDF_OK) return s;
  note_eval_stream(sc, st);
  const int tiles = (N + kStaticTile - 1) / kStaticTile;
  // the array is shared by every call and keeps the last call's contents (a call that failed or was
  // overlapped may have left keys behind): what this call uses is put into its clean state first
  CU_TRY(cudaMemsetAsync(ss->depth, 0x00, sizeof(unsigned long long) * (size_t)N, st));
  CU_TRY(cudaMemsetAsync(ss->d2, 0xff, sizeof(unsigned long long) * (size_t)N, st));
  CU_TRY(cudaMemsetAsync(ss->count, 0x00, sizeof(unsigned int) * (size_t)tiles, st));
  EvalParams p{};
  p.pairs = sc->pk[sc->cur].pairs;
  p.row_slot = sc->pk[sc->cur].row_slot;
  p.bounds = sc->pk[sc->cur].bounds;
  p.empty_rows = sc->pk[sc->cur].empty;
  p.poses = poses;
  p.value = value;
  p.grad = grad;
  p.ws_depth = ss->depth;                                    // device addresses inside the static array
  p.ws_d2 = ss->d2;
  p.ws_count = ss->count;
  p.n_edges = sc->n_edges;
  p.Mv = sc->Mv;
  p.M_rows = sc->M;
  p.n_empty = sc->n_empty;
  p.N = N;
  // the tile-scan kernel's launch plan, always in chunks when the scene allows it
  int C = 2;
  const double warps_per_sm = (double)N / 32.0 / sc->sm_count;
  if (warps_per_sm < 256.0) C = (int)std::ceil(256.0 / warps_per_sm);
  const int maxC = sc->Mv / 16 > 0 ? sc->Mv / 16 : 1;
  if (C < 2) C = 2;
  if (C > maxC) C = maxC;
  if (C > kMaxChunks) C = kMaxChunks;
  p.chunk_begin[0] = 0;
  int o = 0;
  for (int c = 1; c < C; ++c) {
    const long long target = (long long)sc->n_pairs * c / C;
    while (o < sc->Mv && sc->h_pair_begin[o] < target) ++o;
    p.chunk_begin[c] = sc->h_pair_begin[o];
  }
  p.chunk_begin[C] = sc->n_pairs;
  p.n_chunks = C;
  const cudaError_t e = launch_v(sc, p, grad ? kGrad : 0, false, dim3((unsigned)tiles, (unsigned)C), kStaticTile, st, nullptr);
  if (e != cudaSuccess) return cuda_failed(e);
  return PSDF_OK;
}

// ============================================================================== serving mode
// psdf_serve_begin / psdf_serve_step / psdf_serve_end (include/psdf.h): a persistent kernel and a mailbox
// in pinned, device-mapped memory for one fixed MPC batch shape (psdf_serve_kernel, psdf_kernels.cuh).
namespace {

constexpr int kServeMaxPoses = 512, kServeMaxCtas = 128;
constexpr unsigned kServeSentinel = kRowSentinel;

template <int V>
cudaError_t launch_serve_v(const psdf_scene* sc, const EvalParams& p, unsigned last_seq) {
  const psdf_scene::Serve& sv = sc->srv;
  if (sv.mode & kCoeff)
    psdf_serve_kernel<V, kCoeff><<<sv.G, sv.bd, 0, sv.stream>>>(sc->fp, p, sv.in, sv.ack, last_seq, sv.idle_ns);
  else
    psdf_serve_kernel<V, kGrad><<<sv.G, sv.bd, 0, sv.stream>>>(sc->fp, p, sv.in, sv.ack, last_seq, sv.idle_ns);
  g_launches.fetch_add(1);
  return cudaGetLastError();
}

// (re)launches the serving kernel on the live buffer set; `last_seq`: the request it must NOT answer
psdf_status serve_launch(psdf_scene* sc, unsigned last_seq) {
  psdf_scene::Serve& sv = sc->srv;
  EvalParams p{};
  p.pairs = sc->pk[sc->cur].pairs;
  p.row_slot = sc->pk[sc->cur].row_slot;
  p.bounds = sc->pk[sc->cur].bounds;
  p.empty_rows = sc->pk[sc->cur].empty;
  p.window = sv.windows ? sv.d_win : nullptr;
  float* rows = reinterpret_cast<float*>(sv.out);            // mapped host rows
  p.grad = (sv.mode & kGrad) ? rows : nullptr;               // (non-null = wanted; results go to `packed`)
  p.coeff = (sv.mode & kCoeff) ? rows : nullptr;
  p.packed = rows;
  p.n_edges = sc->n_edges;
  p.Mv = sc->Mv;
  p.M_rows = sc->M;
  p.n_empty = sc->n_empty;
  p.N = sv.N;
  p.lanes = sv.K;
  p.n_chunks = 1;
  p.d_min = sv.d_min; p.rho_p = sv.rho_p; p.rho_theta = sv.rho_theta;
  for (int c = 0; c < sv.G; ++c) { sv.ack[2 * c] = last_seq; sv.ack[2 * c + 1] = 0u; }
  cudaError_t e;
  switch (sc->Vp) {
    case 4: e = launch_serve_v<4>(sc, p, last_seq); break;
    case 6: e = launch_serve_v<6>(sc, p, last_seq); break;
    case 8: e = launch_serve_v<8>(sc, p, last_seq); break;
    case 10: e = launch_serve_v<10>(sc, p, last_seq); break;
    case 12: e = launch_serve_v<12>(sc, p, last_seq); break;
    case 16: e = launch_serve_v<16>(sc, p, last_seq); break;
    default: e = cudaErrorInvalidValue;
  }
  if (e != cudaSuccess) return cuda_failed(e);
  sv.running = true;
  return PSDF_OK;
}

inline void serve_post(psdf_scene::Serve& sv, int n, float x, float y, float th, unsigned seq) {
  // one 16-byte store per slot: the polling lane sees either the old or the new request, never a mix
  const __m128i v = _mm_set_epi32((int)seq, (int)__builtin_bit_cast(unsigned, th), (int)__builtin_bit_cast(unsigned, y),
                                  (int)__builtin_bit_cast(unsigned, x));
  _mm_store_si128(reinterpret_cast<__m128i*>(sv.in + n), v);
}

}  // namespace

static psdf_status serve_pause(psdf_scene* sc) {
  psdf_scene::Serve& sv = sc->srv;
  if (!sv.running) return PSDF_OK;
  for (int n = 0; n < sv.N; ++n) serve_post(sv, n, 0.f, 0.f, 0.f, kServeExit);
  _mm_sfence();
  sv.running = false;
  CU_TRY(cudaStreamSynchronize(sv.stream));           // (at the latest after the idle timeout)
  return PSDF_OK;
}

extern "C" {

psdf_status psdf_serve_begin(psdf_scene* sc, int N, const int* row_window, int want_coeffs, float d_min, float rho_p,
                             float rho_theta, int idle_timeout_ms) {
  if (!sc || N < 1 || N > kServeMaxPoses || idle_timeout_ms < 1 || idle_timeout_ms > 10000) return PSDF_ERR_INVALID_ARG;
  if (N > sc->max_poses) return PSDF_ERR_CAPACITY;
  PSDF_ENTER(sc);
  psdf_status s = serve_pause(sc);
  if (s != PSDF_OK) return s;
  psdf_scene::Serve& sv = sc->srv;
  sv.on = false;
  // lanes per pose as in the lane-split plan, all inside one CTA per pose group (no cross-CTA reduction)
  long long want = (long long)sc->sm_count * 1024 / N;
  int L = 1;
  // (fewer, fatter CTAs were measured and are far slower: ~1.7 us of dependent L2 round trips per obstacle and lane)
  while (L < 256 && L < sc->Mv && L * 2 <= want) L <<= 1;
  const int K = L, bd = K <= 64 ? 64 : K, ppc = bd / K, G = (N + ppc - 1) / ppc;
  if (G > kServeMaxCtas) return PSDF_ERR_INVALID_ARG;       // not an MPC-sized shape: use psdf_eval_host
  if (!sv.stream) CU_TRY(cudaStreamCreateWithFlags(&sv.stream, cudaStreamNonBlocking));
  if (N > sv.cap_N || G > sv.cap_G) {
    if (sv.in) cudaFreeHost(sv.in);
    if (sv.out) cudaFreeHost(sv.out);
    if (sv.ack) cudaFreeHost(sv.ack);
    cudaFree(sv.d_win);
    sv.in = sv.out = nullptr; sv.ack = nullptr; sv.d_win = nullptr; sv.cap_N = sv.cap_G = 0;
    CU_TRY(cudaHostAlloc(&sv.in, sizeof(float4) * (size_t)N, cudaHostAllocMapped));
    CU_TRY(cudaHostAlloc(&sv.out, sizeof(float4) * (size_t)N, cudaHostAllocMapped));
    CU_TRY(cudaHostAlloc(&sv.ack, sizeof(unsigned) * 2 * (size_t)G, cudaHostAllocMapped));
    CU_TRY(cudaMalloc(&sv.d_win, sizeof(int) * 2 * (size_t)N));
    sv.cap_N = N; sv.cap_G = G;
  }
  int dev = 0, uva = 0;
  CU_TRY(cudaGetDevice(&dev));
  CU_TRY(cudaDeviceGetAttribute(&uva, cudaDevAttrUnifiedAddressing, dev));
  if (!uva) return PSDF_ERR_CUDA;                            // (mapped host pointers are used as device pointers)
  sv.N = N; sv.K = K; sv.bd = bd; sv.G = G;
  sv.windows = row_window != nullptr;
  if (sv.windows) CU_TRY(cudaMemcpy(sv.d_win, row_window, sizeof(int) * 2 * (size_t)N, cudaMemcpyHostToDevice));
  sv.mode = want_coeffs ? kCoeff : kGrad;
  sv.d_min = d_min; sv.rho_p = rho_p; sv.rho_theta = rho_theta;
  sv.idle_ns = (unsigned long long)idle_timeout_ms * 1000000ull;
  sv.seq = 1;
  for (int n = 0; n < N; ++n) serve_post(sv, n, 0.f, 0.f, 0.f, sv.seq);
  _mm_sfence();
  s = serve_launch(sc, sv.seq);
  if (s != PSDF_OK) return s;
  sv.on = true;
  return PSDF_OK;
}

psdf_status psdf_serve_step(psdf_scene* sc, const float* poses, float* out) {
  if (!sc || !poses || !out) return PSDF_ERR_INVALID_ARG;
  PSDF_ENTER(sc);
  psdf_scene::Serve& sv = sc->srv;
  if (!sv.on) return PSDF_ERR_INVALID_ARG;                   // psdf_serve_begin first
  unsigned seq = sv.seq + 1;
  if (seq == kServeExit || seq == 0u) seq = 1u;
  const unsigned prev = sv.seq;
  sv.seq = seq;
  const __m128i sentinel = _mm_set1_epi32((int)kServeSentinel);
  for (int n = 0; n < sv.N; ++n) _mm_store_si128(reinterpret_cast<__m128i*>(sv.out + n), sentinel);
  _mm_sfence();                                              // rows are blank before the request can be seen
  for (int n = 0; n < sv.N; ++n) serve_post(sv, n, poses[3 * n], poses[3 * n + 1], poses[3 * n + 2], seq);
  _mm_sfence();
  if (!sv.running) {                                         // paused by an update, or first step after a time-out
    const psdf_status s = serve_launch(sc, prev);
    if (s != PSDF_OK) return s;
  }
  volatile unsigned* ack = sv.ack;
  const auto t0 = std::chrono::steady_clock::now();
  int relaunches = 0;
  // a row has arrived when none of its four words is the sentinel any more (the kernel writes a row with one
  // 16-byte store; word-wise acceptance does not even rely on that store landing as a whole)
  for (int n = 0; n < sv.N;) {
    unsigned spins = 0;
    bool restart = false;
    const volatile __m128i* row = reinterpret_cast<const volatile __m128i*>(sv.out + n);
    while (_mm_movemask_epi8(_mm_cmpeq_epi32(_mm_load_si128(const_cast<const __m128i*>(row)), sentinel)) != 0) {
      _mm_pause();
      if ((++spins & 0x3fu) != 0u) continue;
      for (int k = 0; k < sv.G && !restart; ++k) restart = ack[2 * k + 1] != 0u;   // a CTA gave up (idle time-out)
      if (restart) break;
      if ((spins & 0xfffu) == 0u) {
        if (cudaStreamQuery(sv.stream) != cudaErrorNotReady) {   // kernel gone without a word: an error
          sv.running = false;
          const cudaError_t e = cudaGetLastError();
          return cuda_failed(e != cudaSuccess ? e : cudaErrorUnknown);
        }
        if (std::chrono::steady_clock::now() - t0 > std::chrono::seconds(5)) return PSDF_ERR_CUDA;
      }
    }
    if (restart) {
      // the kernel is on its way out: hurry the CTAs that are still polling, then every CTA answers the
      // request again on a fresh launch (requests are idempotent)
      psdf_status s = serve_pause(sc);
      if (s != PSDF_OK) return s;
      if (++relaunches > 3) return PSDF_ERR_CUDA;
      for (int k = 0; k < sv.N; ++k) _mm_store_si128(reinterpret_cast<__m128i*>(sv.out + k), sentinel);
      _mm_sfence();
      for (int k = 0; k < sv.N; ++k) serve_post(sv, k, poses[3 * k], poses[3 * k + 1], poses[3 * k + 2], seq);
      _mm_sfence();
      s = serve_launch(sc, prev);
      if (s != PSDF_OK) return s;
      n = 0;
      continue;
    }
    ++n;
  }
  std::memcpy(out, sv.out, sizeof(float4) * (size_t)sv.N);
  return PSDF_OK;
}

psdf_status psdf_serve_end(psdf_scene* sc) {
  if (!sc) return PSDF_ERR_INVALID_ARG;
  PSDF_ENTER(sc);
  sc->srv.on = false;
  return serve_pause(sc);
}

psdf_status psdf_bench_serve_latency(psdf_scene* sc, const float* poses, float* out, int reps, double* out_us) {
  if (!sc || !out_us || reps < 1) return PSDF_ERR_INVALID_ARG;
  for (int r = 0; r < reps; ++r) {
    const auto t0 = std::chrono::steady_clock::now();
    const psdf_status s = psdf_serve_step(sc, poses, out);
    const auto t1 = std::chrono::steady_clock::now();
    if (s != PSDF_OK) return s;
    out_us[r] = std::chrono::duration<double, std::micro>(t1 - t0).count();
  }
  return PSDF_OK;
}

}  // extern "C"
