// Pipe micro-benchmarks behind DESIGN.md section 6.4 (measurement helper, not on the product path).
// Build + run:  python -m paper_2607_04310_b200.build ubench && paper_2607_04310_b200/csrc/ubench/pipes
// Section 1: instruction mixes (FFMA2 / FFMA / FMNMX / FMNMX3 / IADD), independent chains, 8 warps/SMSP.
// Section 2: FFMA2 / FMUL2 / FADD2 / FMNMX operand forms (which register-operand patterns cost an extra cycle).
// Section 3: the tile-scan kernel's inner step (edge_step2 from psdf_device.cuh) in isolation,
//            cycles per edge step per SMSP for 2..12 resident warps.
// All numbers are cycles at the SM clock passed as argv[1] in MHz (default 1965).
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <cuda_runtime.h>
#include "../psdf_device.cuh"
static double g_mhz = 1965.0;

// ------------------------------------------------------------------ section 1: instruction mixes
namespace mixes {
constexpr int kIter = 2048;
__device__ __forceinline__ float2 ffma2(float2 a, float2 b, float2 c) {
  unsigned long long ra = *reinterpret_cast<unsigned long long*>(&a), rb = *reinterpret_cast<unsigned long long*>(&b),
                     rc = *reinterpret_cast<unsigned long long*>(&c), rd;
  asm volatile("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(rd) : "l"(ra), "l"(rb), "l"(rc));
  return *reinterpret_cast<float2*>(&rd);
}
__device__ __forceinline__ float fmx(float a, float b) { float d; asm volatile("max.f32 %0, %1, %2;" : "=f"(d) : "f"(a), "f"(b)); return d; }
__device__ __forceinline__ float fmn(float a, float b) { float d; asm volatile("min.f32 %0, %1, %2;" : "=f"(d) : "f"(a), "f"(b)); return d; }
__device__ __forceinline__ float fmx3(float a, float b, float c) { float d; asm volatile("max.f32 %0, %1, %2, %3;" : "=f"(d) : "f"(a), "f"(b), "f"(c)); return d; }
__device__ __forceinline__ float ffma(float a, float b, float c) { float d; asm volatile("fma.rn.f32 %0, %1, %2, %3;" : "=f"(d) : "f"(a), "f"(b), "f"(c)); return d; }
__device__ __forceinline__ int iadd(int a, int b) { int d; asm volatile("add.s32 %0, %1, %2;" : "=r"(d) : "r"(a), "r"(b)); return d; }

// per loop trip: NF2 FFMA2, NF FFMA, NM FMNMX (min/max alternating so that ptxas cannot fuse them into
// FMNMX3), NM3 FMNMX3, NI IADD3, each on its own dependency chain, four trips unrolled
template <int NF2, int NF, int NM, int NM3, int NI>
__global__ void k(float* out, float a, float b) {
  float2 x[NF2 > 0 ? NF2 : 1];
  float y[NF > 0 ? NF : 1], m[NM > 0 ? NM : 1], m3[NM3 > 0 ? NM3 : 1];
  int iv[NI > 0 ? NI : 1];
  for (int i = 0; i < NF2; i++) x[i] = make_float2(threadIdx.x * 1e-3f + i, i);
  for (int i = 0; i < NF; i++) y[i] = threadIdx.x * 1e-3f + i;
  for (int i = 0; i < NM; i++) m[i] = threadIdx.x * 1e-3f + i;
  for (int i = 0; i < NM3; i++) m3[i] = threadIdx.x * 1e-3f + i;
  for (int i = 0; i < NI; i++) iv[i] = threadIdx.x + i;
  const float2 a2 = make_float2(a, a), b2 = make_float2(b, b);
#pragma unroll 1
  for (int it = 0; it < kIter; it++) {
#pragma unroll
    for (int r = 0; r < 4; r++) {
#pragma unroll
      for (int i = 0; i < 16; i++) {
        if (i < NF2) x[i] = ffma2(x[i], a2, b2);
        if (i < NF) y[i] = ffma(y[i], a, b);
        if (i < NM) m[i] = (r & 1) ? fmn(m[i], b) : fmx(m[i], a);
        if (i < NM3) m3[i] = fmx3(m3[i], a, b);
        if (i < NI) iv[i] = iadd(iv[i], it);
      }
    }
  }
  float s = 0;
  for (int i = 0; i < NF2; i++) s += x[i].x + x[i].y;
  for (int i = 0; i < NF; i++) s += y[i];
  for (int i = 0; i < NM; i++) s += m[i];
  for (int i = 0; i < NM3; i++) s += m3[i];
  for (int i = 0; i < NI; i++) s += iv[i];
  if (s == 123.456f) out[0] = s;
}
template <int NF2, int NF, int NM, int NM3, int NI>
void run(const char* name) {
  float* d;
  cudaMalloc(&d, 4);
  const int blocks = 148 * 2, threads = 512;               // 8 warps per SMSP
  k<NF2, NF, NM, NM3, NI><<<blocks, threads>>>(d, 0.999f, 0.001f);
  cudaEvent_t e0, e1;
  cudaEventCreate(&e0); cudaEventCreate(&e1);
  float best = 1e9f;
  for (int r = 0; r < 3; r++) {
    cudaEventRecord(e0); k<NF2, NF, NM, NM3, NI><<<blocks, threads>>>(d, 0.999f, 0.001f); cudaEventRecord(e1);
    cudaEventSynchronize(e1);
    float ms; cudaEventElapsedTime(&ms, e0, e1); best = fminf(best, ms);
  }
  const int ninst = NF2 + NF + NM + NM3 + NI;
  const double cyc = best * 1e-3 * g_mhz * 1e6 / (kIter * 4.0 * 8.0);   // SMSP cycles per trip of ninst instructions
  printf("mix   %-30s %2d inst  %6.2f clk/trip  %5.3f inst/clk/SMSP\n", name, ninst, cyc, ninst / cyc);
  cudaFree(d);
}
void all() {
  run<8, 0, 0, 0, 0>("8 FFMA2");
  run<8, 0, 2, 0, 0>("8 FFMA2 + 2 FMNMX");
  run<8, 0, 4, 0, 0>("8 FFMA2 + 4 FMNMX");
  run<8, 0, 8, 0, 0>("8 FFMA2 + 8 FMNMX");
  run<8, 0, 0, 4, 0>("8 FFMA2 + 4 FMNMX3");
  run<8, 0, 0, 8, 0>("8 FFMA2 + 8 FMNMX3");
  run<8, 0, 0, 0, 8>("8 FFMA2 + 8 IADD3");
  run<0, 16, 0, 0, 0>("16 FFMA");
  run<0, 16, 4, 0, 0>("16 FFMA + 4 FMNMX");
  run<0, 16, 8, 0, 0>("16 FFMA + 8 FMNMX");
  run<0, 0, 16, 0, 0>("16 FMNMX");
  run<0, 0, 0, 16, 0>("16 FMNMX3");
  run<4, 8, 4, 0, 0>("4 FFMA2 + 8 FFMA + 4 FMNMX");
  run<8, 4, 4, 0, 0>("8 FFMA2 + 4 FFMA + 4 FMNMX");
}
}  // namespace mixes

// ------------------------------------------------------------------ section 2: operand forms
namespace forms {
constexpr int kIter = 4096;
struct C { float2 c[8]; };
template <int F>
__global__ void k(float* out, const float* in, const __grid_constant__ C cc) {
  float2 x[8], y[8];
  float s[8], t[8];
  for (int i = 0; i < 8; i++) {
    x[i] = make_float2(in[threadIdx.x + i], in[threadIdx.x + 8 + i]);
    s[i] = in[16 + i + threadIdx.x];
    t[i] = in[32 + i + threadIdx.x];
    y[i] = make_float2(in[48 + i + threadIdx.x], in[64 + i + threadIdx.x]);
  }
#pragma unroll 1
  for (int it = 0; it < kIter; it++) {
#pragma unroll
    for (int r = 0; r < 4; r++) {
#pragma unroll
      for (int i = 0; i < 8; i++) {
        if (F == 1) x[i] = __ffma2_rn(x[i], y[i], y[(i + 1) & 7]);                           // R64 * R64 + R64
        if (F == 2) x[i] = __ffma2_rn(x[i], make_float2(s[i], s[i]), y[i]);                  // R64 * R32 + R64
        if (F == 3) x[i] = __ffma2_rn(x[i], make_float2(s[i], s[i]), make_float2(t[i], t[i]));  // R64 * R32 + R32
        if (F == 4) x[i] = __ffma2_rn(make_float2(s[i], s[i]), x[i], cc.c[i]);               // R32 * R64 + UR64
        if (F == 5) x[i] = __fmul2_rn(x[i], x[i]);
        if (F == 6) x[i] = __fadd2_rn(x[i], cc.c[i]);
        if (F == 7) x[i] = __ffma2_rn(y[i], make_float2(s[i], s[i]), x[i]);                  // R64 * R32 + acc64
        if (F == 8) x[i] = __ffma2_rn(x[i], x[i], y[i]);                                     // R64 * same + R64
        if (F == 9) x[i] = __fadd2_rn(x[i], make_float2(-s[i], -s[i]));
        if (F == 10) { x[i].x = fmaxf(fabsf(x[i].x), s[i]); x[i].y = fminf(fabsf(x[i].y), t[i]); }
        if (F == 11) { x[i].x = fmaxf(fabsf(x[i].x), cc.c[i].x); x[i].y = fminf(fabsf(x[i].y), cc.c[i].y); }
      }
    }
  }
  float a = 0;
  for (int i = 0; i < 8; i++) a += x[i].x + x[i].y + t[i];
  out[blockIdx.x * blockDim.x + threadIdx.x] = a;
}
template <int F>
void run(const char* name) {
  float *d, *in;
  cudaMalloc(&d, 148 * 2 * 512 * 4);
  cudaMalloc(&in, 4096);
  cudaMemset(in, 0, 4096);
  C cc;
  for (int i = 0; i < 8; i++) cc.c[i] = make_float2(0.f, 0.f);
  k<F><<<296, 512>>>(d, in, cc);
  cudaEvent_t e0, e1;
  cudaEventCreate(&e0); cudaEventCreate(&e1);
  float best = 1e9f;
  for (int r = 0; r < 3; r++) {
    cudaEventRecord(e0); k<F><<<296, 512>>>(d, in, cc); cudaEventRecord(e1);
    cudaEventSynchronize(e1);
    float ms; cudaEventElapsedTime(&ms, e0, e1); best = fminf(best, ms);
  }
  const double inst_per_smsp = 8.0 * kIter * 4 * 8 * (F >= 10 ? 2 : 1);
  printf("form  %-44s %5.2f clk/inst\n", name, best * 1e-3 * g_mhz * 1e6 / inst_per_smsp);
  cudaFree(d); cudaFree(in);
}
void all() {
  run<1>("FFMA2 R64 * R64 + R64 (3 distinct pairs)");
  run<2>("FFMA2 R64 * R32 + R64");
  run<7>("FFMA2 R64 * R32 + acc64");
  run<3>("FFMA2 R64 * R32 + R32");
  run<4>("FFMA2 R32 * R64 + UR64");
  run<8>("FFMA2 R64 * same + R64");
  run<5>("FMUL2 R64 * same");
  run<6>("FADD2 R64 + UR64");
  run<9>("FADD2 R64 + -R32");
  run<10>("FMNMX |R|, R   (two per count)");
  run<11>("FMNMX |R|, UR  (two per count)");
}
}  // namespace forms

// ------------------------------------------------------------------ section 3: the inner step
namespace step {
using namespace psdf;
// VAR 0: edge_step2 as shipped.  VAR 1: without the SAT max accumulations.  VAR 2: without the
// |tau| clamps (FMNMX with |.|).  Removing ALU-pipe instructions shows what they cost in situ.
template <int V, int VAR>
__device__ __forceinline__ void step_var(const Footprint& fp, const Posed2<V>& P, const float4 q, const float h,
                                         ObstacleAcc<V>& acc, float& minD2) {
  if (VAR == 0) { edge_step2<V>(fp, P, q, h, acc, minD2); return; }
  const float sax = q.x - P.px, say = q.y - P.py;
  const float sncn = fmaf(sax, q.w, -say * q.z);
  const float snct = -fmaf(sax, q.z, fmaf(say, q.w, h));
  const float2 ax = bc2(sax), ay = bc2(say), nax = bc2(-sax);
  const float2 tx = bc2(q.z), ty = bc2(q.w), nty = bc2(-q.w);
  const float2 ncn = bc2(sncn), nct = bc2(snct), nh = bc2(-h);
  float gj = -kInf, m = minD2;
#pragma unroll
  for (int l = 0; l < V / 2; ++l) {
    const float2 s = __ffma2_rn(P.ry[l], tx, __ffma2_rn(P.rx[l], nty, ncn));
    const float2 u = __ffma2_rn(P.rx[l], tx, __ffma2_rn(P.ry[l], ty, nct));
    const float2 e = VAR == 2 ? __fadd2_rn(u, nh)
                              : __fadd2_rn(make_float2(fmaxf(fabsf(u.x), h), fmaxf(fabsf(u.y), h)), nh);
    const float2 d = __ffma2_rn(e, e, __fmul2_rn(s, s));
    if (VAR != 1) gj = fmax3(gj, s.x, s.y);
    const float2 ncN = *reinterpret_cast<const float2*>(&fp.ncN[2 * l]);
    const float2 ncT = *reinterpret_cast<const float2*>(&fp.ncT[2 * l]);
    const float2 hR = *reinterpret_cast<const float2*>(&fp.h[2 * l]);
    const float2 nhR = *reinterpret_cast<const float2*>(&fp.nh[2 * l]);
    const float2 pp = __ffma2_rn(ay, P.Tx[l], __ffma2_rn(nax, P.Ty[l], ncN));
    const float2 w = __ffma2_rn(ax, P.Tx[l], __ffma2_rn(ay, P.Ty[l], ncT));
    const float2 f = VAR == 2 ? __fadd2_rn(w, nhR)
                              : __fadd2_rn(make_float2(fmaxf(fabsf(w.x), hR.x), fmaxf(fabsf(w.y), hR.y)), nhR);
    const float2 g = __ffma2_rn(f, f, __fmul2_rn(pp, pp));
    if (VAR != 1) {
      acc.gR[2 * l] = fmaxf(acc.gR[2 * l], pp.x);
      acc.gR[2 * l + 1] = fmaxf(acc.gR[2 * l + 1], pp.y);
    }
    m = fmin3(m, d.x, d.y);
    m = fmin3(m, g.x, g.y);
  }
  acc.gO = fminf(acc.gO, gj);
  minD2 = m;
}

template <int V, int VAR>
__global__ void __launch_bounds__(128) k(const __grid_constant__ Footprint fp, const float4* __restrict__ g, int iters,
                                         float* out, const float* poses) {
  __shared__ float4 tile[256];
  for (int i = threadIdx.x; i < 256; i += blockDim.x) tile[i] = g[i];
  __syncthreads();
  const int t = blockIdx.x * blockDim.x + threadIdx.x;
  Posed2<V> P;
  pose_setup2<V>(fp, poses[3 * t], poses[3 * t + 1], poses[3 * t + 2], P);
  ObstacleAcc<V> acc;
  acc.reset();
  float m = kInf, best = -kInf;
#pragma unroll 1
  for (int it = 0; it < iters; ++it) {
#pragma unroll 1
    for (int k2 = 0; k2 < 128; ++k2) {
      const float4 q0 = tile[2 * k2], q1 = tile[2 * k2 + 1];
      step_var<V, VAR>(fp, P, q0, q1.x, acc, m);
      if (__float_as_int(q1.z) >= 0) { best = fmaxf(best, acc.depth()); acc.reset(); }
    }
  }
  out[t] = m + best;
}

template <int V, int VAR>
void run(const char* name) {
  Footprint fp;
  memset(&fp, 0, sizeof(fp));
  for (int l = 0; l < 16; ++l) {
    fp.vx[l] = cosf(l); fp.vy[l] = sinf(l); fp.tx[l] = cosf(l + .5f); fp.ty[l] = sinf(l + .5f);
    fp.h[l] = .3f; fp.nh[l] = -.3f; fp.ncN[l] = .1f * l; fp.ncT[l] = .2f * l;
  }
  float4 h[256];
  for (int i = 0; i < 128; ++i) {
    h[2 * i] = make_float4(i * .37f, i * .11f, cosf(i), sinf(i));
    const int last = (i % 8 == 7) ? i : -1;
    float lf;
    memcpy(&lf, &last, 4);
    h[2 * i + 1] = make_float4(.4f, 0, lf, 0);
  }
  float4* dg;
  cudaMalloc(&dg, sizeof(h));
  cudaMemcpy(dg, h, sizeof(h), cudaMemcpyHostToDevice);
  for (int wps = 2; wps <= 12; wps += 2) {                  // resident warps per SMSP
    const int blocks = 148 * wps, threads = 128, iters = 40;
    float *out, *poses;
    cudaMalloc(&out, blocks * threads * 4);
    cudaMalloc(&poses, blocks * threads * 12);
    cudaMemset(poses, 0, blocks * threads * 12);
    k<V, VAR><<<blocks, threads>>>(fp, dg, 2, out, poses);
    cudaEvent_t e0, e1;
    cudaEventCreate(&e0); cudaEventCreate(&e1);
    float best = 1e9f;
    for (int r = 0; r < 3; ++r) {
      cudaEventRecord(e0); k<V, VAR><<<blocks, threads>>>(fp, dg, iters, out, poses); cudaEventRecord(e1);
      cudaEventSynchronize(e1);
      float ms; cudaEventElapsedTime(&ms, e0, e1); best = fminf(best, ms);
    }
    printf("step  %-28s V=%d warps/SMSP=%2d  %6.1f clk/edge-step\n", name, V, wps,
           best * 1e-3 * g_mhz * 1e6 / ((double)wps * iters * 128));
    cudaFree(out); cudaFree(poses);
  }
  cudaFree(dg);
}
void all() {
  run<6, 0>("edge_step2 (shipped)");
  run<6, 1>("without SAT max ops");
  run<6, 2>("without |tau| clamps");
  run<4, 0>("edge_step2 (shipped)");
  run<8, 0>("edge_step2 (shipped)");
}
}  // namespace step

int main(int argc, char** argv) {
  if (argc > 1) g_mhz = atof(argv[1]);
  cudaDeviceProp prop;
  if (cudaGetDeviceProperties(&prop, 0) != cudaSuccess) { printf("no CUDA device\n"); return 1; }
  printf("# %s, %d SMs, cycles at %.0f MHz\n", prop.name, prop.multiProcessorCount, g_mhz);
  mixes::all();
  forms::all();
  step::all();
  return cudaDeviceSynchronize() == cudaSuccess ? 0 : 2;
}
