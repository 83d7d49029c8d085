// Device-side PSDF arithmetic for sm_100a (no code shared with oracle/).
//
// Formulation (equivalent to PAPER.md eqs.(11)-(23) by rigid-motion
// invariance and one-sided SAT):
//   * pose-relative world frame: r_l = R(theta) v_l (posed robot vertex minus p) and
//     a_j = A_j - p; rotation is applied to the footprint once per pose instead of to
//     every obstacle endpoint (eq.(11) PAPER.md:141-145 moved onto eq.(9));
//   * obstacle edge j has unit tangent t_j, inward unit normal n_j = rot90(t_j) (CCW),
//     half length h_j; robot edge l has rotated tangent T_l, inward normal N_l;
//   * per (l, j):  sigma = (r_l - a_j).n_j, tau_m = (r_l - a_j).t_j - h_j   (pool 1,
//     eqs.(12)-(14) PAPER.md:153-167) and sigma' = (a_j - r_l).N_l,
//     tau'_m = (a_j - r_l).T_l - h_l (pool 2, eq.(15));
//     point-to-segment d^2 = sigma^2 + max(|tau_m| - h, 0)^2  (eq.(13) with the clamp
//     of eq.(12) written around the edge midpoint; as FADD2 with |.| + two FMNMX against zero:
//     64 operand bits per vertex pair fewer than max(|tau_m|, h) - h, same bits out);
//   * SAT (eqs.(17)-(22) PAPER.md:181-217), one-sided: face depth G_j = max_l sigma,
//     G'_l = max_j sigma'; depth^i = min over the faces of both polygons; separated^i
//     <=> depth^i < 0 (eq.21); pen = depth^i otherwise (eq.22) — the "other side" term of
//     eq.(20) can never be the minimum;
//   * phi = -max_i depth^i if any depth^i >= 0 else sqrt(min over everything of d^2)
//     (eqs.(23),(6) PAPER.md:221-225, 93-95).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace psdf {

constexpr int kMaxV = 16;
constexpr float kInf = __builtin_huge_valf();

// One packed valid edge, 32 bytes (two float4): built in double at scene creation (H0).
struct __align__(16) EdgeRec {
  float ax, ay;   // edge start A_j, world frame (the obstacle vertex of eq.(15))
  float tx, ty;   // unit tangent; inward normal is (-ty, tx)
  float h;        // half length |B-A|/2
  int last;       // -1, or the obstacle row index if this is the row's last valid edge
  int slot;       // packed obstacle index (0..Mv-1)
  float pad;
};

// Footprint constants (pose independent), passed by value as a kernel parameter so that
// the unrolled loops read them as constant-bank operands.
struct __align__(16) Footprint {
  float vx[kMaxV], vy[kMaxV];   // vertices v_l (robot-local)
  float tx[kMaxV], ty[kMaxV];   // unit edge tangents t~_l of E_l = [v_l, v_{l+1}]
  float h[kMaxV];               // half lengths
  float cN[kMaxV];              // v_l . n~_l      (n~_l = rot90(t~_l), inward)
  float cT[kMaxV];              // v_l . t~_l + h_l
  float ncN[kMaxV], ncT[kMaxV], nh[kMaxV];   // negated copies (f32x2 constant operands)
  float rmax;                   // max_l |v_l|  (Prop.1)
  float bcx, bcy, bhx, bhy;     // robot-frame bounding box: centre, half extents (culled path)
  float rbox;                   // max_l |v_l - box centre|
  int sym;                      // 1: centrally symmetric about the reference point, v_{l+V/2} == -v_l (edge_step2_sym)
};

// Per-pose state: posed footprint in registers (H1).
template <int V>
struct Posed {
  float px, py;
  float rx[V], ry[V];   // r_l = R v_l
  float Tx[V], Ty[V];   // T_l = R t~_l
};

template <int V>
__device__ __forceinline__ void pose_setup(const Footprint& fp, float x, float y, float th, Posed<V>& P) {
  float s, c;
  sincosf(th, &s, &c);                       // full-accuracy (not __sincosf): reading G13
  P.px = x;
  P.py = y;
#pragma unroll
  for (int l = 0; l < V; ++l) {
    P.rx[l] = c * fp.vx[l] - s * fp.vy[l];
    P.ry[l] = s * fp.vx[l] + c * fp.vy[l];
    P.Tx[l] = c * fp.tx[l] - s * fp.ty[l];
    P.Ty[l] = s * fp.tx[l] + c * fp.ty[l];
  }
}

__device__ __forceinline__ float fmax3(float a, float b, float c) { return fmaxf(fmaxf(a, b), c); }
__device__ __forceinline__ float fmin3(float a, float b, float c) { return fminf(fminf(a, b), c); }

// Scan accumulators for the obstacle currently being traversed.
template <int V>
struct ObstacleAcc {
  float gR[V];   // G'_l = max_j sigma'   (robot faces)
  float gO;      // min_j G_j             (obstacle faces)
  __device__ __forceinline__ void reset() {
#pragma unroll
    for (int l = 0; l < V; ++l) gR[l] = -kInf;
    gO = kInf;
  }
  __device__ __forceinline__ float depth() const {
    float d = gO;
#pragma unroll
    for (int l = 0; l + 1 < V; l += 2) d = fmin3(d, gR[l], gR[l + 1]);
    if (V & 1) d = fminf(d, gR[V - 1]);
    return d;
  }
};

// Two packed edges of the same obstacle, 48 bytes (three float4): the tile-scan kernel's
// record.  q2 = (h0, h1, last, slot): h1 < 0 marks a record whose second half is unused
// (obstacle with an odd edge count; skipped by a uniform branch); `last` = obstacle row if this pair ends the
// obstacle, else -1 (int bits); slot = packed obstacle index (int bits).
struct __align__(16) PairRec {
  float4 q0, q1, q2;
};


// ---- packed (FFMA2) formulation used by the tile-scan kernel -------------------------------
// Robot vertices/edges are held two per 64-bit register pair so that the eight dot products,
// the squares and the excess subtraction of two (l, l+1) candidates issue as one f32x2
// instruction each (fma.rn.f32x2 -> FFMA2; the per-edge scalars enter as broadcast operands).
// V must be even (odd footprints are padded with a collinear midpoint at pack time).
template <int V>
struct Posed2 {
  float px, py;
  float2 rx[V / 2], ry[V / 2], Tx[V / 2], Ty[V / 2];
};

template <int V>
__device__ __forceinline__ void pose_setup2_sc(const Footprint& fp, float x, float y, float s, float c, Posed2<V>& P) {
  P.px = x;
  P.py = y;
#pragma unroll
  for (int l = 0; l < V / 2; ++l) {
    P.rx[l] = make_float2(c * fp.vx[2 * l] - s * fp.vy[2 * l], c * fp.vx[2 * l + 1] - s * fp.vy[2 * l + 1]);
    P.ry[l] = make_float2(s * fp.vx[2 * l] + c * fp.vy[2 * l], s * fp.vx[2 * l + 1] + c * fp.vy[2 * l + 1]);
    P.Tx[l] = make_float2(c * fp.tx[2 * l] - s * fp.ty[2 * l], c * fp.tx[2 * l + 1] - s * fp.ty[2 * l + 1]);
    P.Ty[l] = make_float2(s * fp.tx[2 * l] + c * fp.ty[2 * l], s * fp.tx[2 * l + 1] + c * fp.ty[2 * l + 1]);
  }
}

template <int V>
__device__ __forceinline__ void pose_setup2(const Footprint& fp, float x, float y, float th, Posed2<V>& P) {
  float s, c;
  sincosf(th, &s, &c);
  pose_setup2_sc<V>(fp, x, y, s, c, P);
}

template <int V>
__device__ __forceinline__ void unpack_pose(const Posed2<V>& P2, Posed<V>& P) {
  P.px = P2.px;
  P.py = P2.py;
#pragma unroll
  for (int l = 0; l < V / 2; ++l) {
    P.rx[2 * l] = P2.rx[l].x; P.rx[2 * l + 1] = P2.rx[l].y;
    P.ry[2 * l] = P2.ry[l].x; P.ry[2 * l + 1] = P2.ry[l].y;
    P.Tx[2 * l] = P2.Tx[l].x; P.Tx[2 * l + 1] = P2.Tx[l].y;
    P.Ty[2 * l] = P2.Ty[l].x; P.Ty[2 * l + 1] = P2.Ty[l].y;
  }
}

__device__ __forceinline__ float2 bc2(float a) { return make_float2(a, a); }

// Hot inner step (H2-H5) for one edge against all V robot vertices/edges, two at a time.
// SUB_FIRST picks between two forms of the clamp that give the same bits: max(|tau| - h, 0) reads 64
// register-operand bits per vertex pair less (throughput kernels: DESIGN.md 6.4); max(|tau|, h) - h lets
// the compiler keep more of the latency-bound lane-split kernel in flight (MPC p50 0.4 us lower).
template <int V, bool SUB_FIRST = true>
__device__ __forceinline__ void edge_step2(const Footprint& fp, const Posed2<V>& P, const float4 q,
                                           const float h, ObstacleAcc<V>& acc, float& minD2) {
  const float sax = q.x - P.px, say = q.y - P.py;                 // H2: a_j = A_j - p
  const float sncn = fmaf(sax, q.w, -say * q.z);                  // -(a_j . n_j)
  const float snct = -fmaf(sax, q.z, fmaf(say, q.w, h));          // -(a_j . t_j + h_j)
  const float2 ax = bc2(sax), ay = bc2(say), nax = bc2(-sax);
  const float2 tx = bc2(q.z), ty = bc2(q.w), nty = bc2(-q.w);
  const float2 ncn = bc2(sncn), nct = bc2(snct), nh = bc2(-h);
  float gj = -kInf;
  float m = minD2;
#pragma unroll
  for (int l = 0; l < V / 2; ++l) {
    // pool 1 + obstacle axis j
    const float2 s = __ffma2_rn(P.ry[l], tx, __ffma2_rn(P.rx[l], nty, ncn));
    const float2 u = __ffma2_rn(P.rx[l], tx, __ffma2_rn(P.ry[l], ty, nct));
    float2 e;
    if (SUB_FIRST) {
      const float2 et = __fadd2_rn(make_float2(fabsf(u.x), fabsf(u.y)), nh);
      e = make_float2(fmaxf(et.x, 0.f), fmaxf(et.y, 0.f));
    } else {
      e = __fadd2_rn(make_float2(fmaxf(fabsf(u.x), h), fmaxf(fabsf(u.y), h)), nh);
    }
    const float2 d = __ffma2_rn(e, e, __fmul2_rn(s, s));
    gj = fmax3(gj, s.x, s.y);
    // pool 2 + robot axes l, l+1
    const float2 ncN = *reinterpret_cast<const float2*>(&fp.ncN[2 * l]);
    const float2 ncT = *reinterpret_cast<const float2*>(&fp.ncT[2 * l]);
    const float2 hR = *reinterpret_cast<const float2*>(&fp.h[2 * l]);
    const float2 nhR = *reinterpret_cast<const float2*>(&fp.nh[2 * l]);
    const float2 pp = __ffma2_rn(ay, P.Tx[l], __ffma2_rn(nax, P.Ty[l], ncN));
    const float2 w = __ffma2_rn(ax, P.Tx[l], __ffma2_rn(ay, P.Ty[l], ncT));
    float2 f;
    if (SUB_FIRST) {
      const float2 ft = __fadd2_rn(make_float2(fabsf(w.x), fabsf(w.y)), nhR);
      f = make_float2(fmaxf(ft.x, 0.f), fmaxf(ft.y, 0.f));
    } else {
      f = __fadd2_rn(make_float2(fmaxf(fabsf(w.x), hR.x), fmaxf(fabsf(w.y), hR.y)), nhR);
    }
    const float2 g = __ffma2_rn(f, f, __fmul2_rn(pp, pp));
    acc.gR[2 * l] = fmaxf(acc.gR[2 * l], pp.x);
    acc.gR[2 * l + 1] = fmaxf(acc.gR[2 * l + 1], pp.y);
    m = fmin3(m, d.x, d.y);
    m = fmin3(m, g.x, g.y);
  }
  acc.gO = fminf(acc.gO, gj);
  minD2 = m;
}

// Two edges of one pair record at once (tile-scan kernel, full records): the same arithmetic as two
// edge_step2 calls, written vertex pair by vertex pair for both edges, so that consecutive instructions read the
// same posed-vertex register pairs (operand reuse) and the two robot-face updates fold into one three-input
// maximum.  min / max are exact, so the order of the updates does not change a bit.
template <int V>
__device__ __forceinline__ void edge_step2_two(const Footprint& fp, const Posed2<V>& P, const float4 qa, const float4 qb,
                                               const float ha, const float hb, ObstacleAcc<V>& acc, float& minD2) {
  const float saxa = qa.x - P.px, saya = qa.y - P.py, saxb = qb.x - P.px, sayb = qb.y - P.py;
  const float sncna = fmaf(saxa, qa.w, -saya * qa.z), sncnb = fmaf(saxb, qb.w, -sayb * qb.z);
  const float sncta = -fmaf(saxa, qa.z, fmaf(saya, qa.w, ha)), snctb = -fmaf(saxb, qb.z, fmaf(sayb, qb.w, hb));
  const float2 axa = bc2(saxa), aya = bc2(saya), naxa = bc2(-saxa), axb = bc2(saxb), ayb = bc2(sayb), naxb = bc2(-saxb);
  const float2 txa = bc2(qa.z), tya = bc2(qa.w), ntya = bc2(-qa.w), txb = bc2(qb.z), tyb = bc2(qb.w), ntyb = bc2(-qb.w);
  const float2 ncna = bc2(sncna), ncta = bc2(sncta), nha = bc2(-ha), ncnb = bc2(sncnb), nctb = bc2(snctb), nhb = bc2(-hb);
  float gja = -kInf, gjb = -kInf;
  float m = minD2;
#pragma unroll
  for (int l = 0; l < V / 2; ++l) {
    // pool 1 + obstacle axes a, b
    const float2 sa = __ffma2_rn(P.ry[l], txa, __ffma2_rn(P.rx[l], ntya, ncna));
    const float2 sb = __ffma2_rn(P.ry[l], txb, __ffma2_rn(P.rx[l], ntyb, ncnb));
    const float2 ua = __ffma2_rn(P.rx[l], txa, __ffma2_rn(P.ry[l], tya, ncta));
    const float2 ub = __ffma2_rn(P.rx[l], txb, __ffma2_rn(P.ry[l], tyb, nctb));
    const float2 eta = __fadd2_rn(make_float2(fabsf(ua.x), fabsf(ua.y)), nha);
    const float2 etb = __fadd2_rn(make_float2(fabsf(ub.x), fabsf(ub.y)), nhb);
    const float2 ea = make_float2(fmaxf(eta.x, 0.f), fmaxf(eta.y, 0.f)), eb = make_float2(fmaxf(etb.x, 0.f), fmaxf(etb.y, 0.f));
    const float2 da = __ffma2_rn(ea, ea, __fmul2_rn(sa, sa)), db = __ffma2_rn(eb, eb, __fmul2_rn(sb, sb));
    gja = fmax3(gja, sa.x, sa.y);
    gjb = fmax3(gjb, sb.x, sb.y);
    // pool 2 + robot axes l, l+1
    const float2 ncN = *reinterpret_cast<const float2*>(&fp.ncN[2 * l]);
    const float2 ncT = *reinterpret_cast<const float2*>(&fp.ncT[2 * l]);
    const float2 nhR = *reinterpret_cast<const float2*>(&fp.nh[2 * l]);
    const float2 ppa = __ffma2_rn(aya, P.Tx[l], __ffma2_rn(naxa, P.Ty[l], ncN));
    const float2 ppb = __ffma2_rn(ayb, P.Tx[l], __ffma2_rn(naxb, P.Ty[l], ncN));
    const float2 wa = __ffma2_rn(axa, P.Tx[l], __ffma2_rn(aya, P.Ty[l], ncT));
    const float2 wb = __ffma2_rn(axb, P.Tx[l], __ffma2_rn(ayb, P.Ty[l], ncT));
    const float2 fta = __fadd2_rn(make_float2(fabsf(wa.x), fabsf(wa.y)), nhR);
    const float2 ftb = __fadd2_rn(make_float2(fabsf(wb.x), fabsf(wb.y)), nhR);
    const float2 fa = make_float2(fmaxf(fta.x, 0.f), fmaxf(fta.y, 0.f)), fb = make_float2(fmaxf(ftb.x, 0.f), fmaxf(ftb.y, 0.f));
    const float2 ga = __ffma2_rn(fa, fa, __fmul2_rn(ppa, ppa)), gb = __ffma2_rn(fb, fb, __fmul2_rn(ppb, ppb));
    acc.gR[2 * l] = fmax3(acc.gR[2 * l], ppa.x, ppb.x);
    acc.gR[2 * l + 1] = fmax3(acc.gR[2 * l + 1], ppa.y, ppb.y);
    m = fmin3(m, da.x, da.y);
    m = fmin3(m, db.x, db.y);
    m = fmin3(m, ga.x, ga.y);
    m = fmin3(m, gb.x, gb.y);
  }
  acc.gO = fmin3(acc.gO, gja, gjb);
  minD2 = m;
}

// The same step for a footprint that is centrally symmetric about its reference point, v_{l+V/2} = -v_l
// (rectangles, car outlines; V a multiple of 4; Footprint::sym, set at pack time when it holds bitwise).
// Then r_{l+V/2} = -r_l, T_{l+V/2} = -T_l, and the constants c_N, c_T, h of edge l+V/2 equal those of edge
// l, so the dot products of the far half follow from the near half by a sign:
//     sigma_l  =  r_l.n_j - a_j.n_j        sigma_{l+V/2}  = -r_l.n_j - a_j.n_j        (same for tau)
//     sigma'_l =  a_j.N_l - c_N,l          sigma'_{l+V/2} = -a_j.N_l - c_N,l          (same for tau')
// i.e. per two vertex pairs eight FMUL2/FFMA2 and eight FADD2 instead of sixteen FFMA2: the same number
// of instructions on the same pipe, 512 register-operand bits fewer (that is what bounds
// the loop).  Every kernel of a scene takes the same variant, so they stay bit-identical to each other.
template <int V, bool SUB_FIRST = true>
__device__ __forceinline__ void edge_step2_sym(const Footprint& fp, const Posed2<V>& P, const float4 q,
                                               const float h, ObstacleAcc<V>& acc, float& minD2) {
  static_assert(V % 4 == 0, "symmetric variant: V must be a multiple of 4");
  const float sax = q.x - P.px, say = q.y - P.py;                 // H2: a_j = A_j - p
  const float sncn = fmaf(sax, q.w, -say * q.z);                  // -(a_j . n_j)
  const float snct = -fmaf(sax, q.z, fmaf(say, q.w, h));          // -(a_j . t_j + h_j)
  const float2 ax = bc2(sax), ay = bc2(say), nax = bc2(-sax);
  const float2 tx = bc2(q.z), ty = bc2(q.w), nty = bc2(-q.w);
  const float2 ncn = bc2(sncn), nct = bc2(snct), nh = bc2(-h);
  float gj = -kInf;
  float m = minD2;
  auto neg2 = [](float2 a) { return make_float2(-a.x, -a.y); };
  // H3-H5 for one vertex pair whose four dot products are known
  auto tail = [&](const float2 s, const float2 u, const float2 pp, const float2 w, const float2 hR, const float2 nhR,
                  float& gR0, float& gR1) {
    float2 e, f;
    if (SUB_FIRST) {
      const float2 et = __fadd2_rn(make_float2(fabsf(u.x), fabsf(u.y)), nh);
      e = make_float2(fmaxf(et.x, 0.f), fmaxf(et.y, 0.f));
      const float2 ft = __fadd2_rn(make_float2(fabsf(w.x), fabsf(w.y)), nhR);
      f = make_float2(fmaxf(ft.x, 0.f), fmaxf(ft.y, 0.f));
    } else {
      e = __fadd2_rn(make_float2(fmaxf(fabsf(u.x), h), fmaxf(fabsf(u.y), h)), nh);
      f = __fadd2_rn(make_float2(fmaxf(fabsf(w.x), hR.x), fmaxf(fabsf(w.y), hR.y)), nhR);
    }
    const float2 d = __ffma2_rn(e, e, __fmul2_rn(s, s));
    const float2 g = __ffma2_rn(f, f, __fmul2_rn(pp, pp));
    gj = fmax3(gj, s.x, s.y);
    gR0 = fmaxf(gR0, pp.x);
    gR1 = fmaxf(gR1, pp.y);
    m = fmin3(m, d.x, d.y);
    m = fmin3(m, g.x, g.y);
  };
#pragma unroll
  for (int b = 0; b < V / 4; ++b) {
    const float2 pn = __ffma2_rn(P.ry[b], tx, __fmul2_rn(P.rx[b], nty));       // r_l . n_j,  l = 2b, 2b+1
    const float2 pt = __ffma2_rn(P.rx[b], tx, __fmul2_rn(P.ry[b], ty));        // r_l . t_j
    const float2 an = __ffma2_rn(ay, P.Tx[b], __fmul2_rn(nax, P.Ty[b]));       // a_j . N_l
    const float2 at = __ffma2_rn(ax, P.Tx[b], __fmul2_rn(ay, P.Ty[b]));        // a_j . T_l
    const float2 ncN = *reinterpret_cast<const float2*>(&fp.ncN[2 * b]);
    const float2 ncT = *reinterpret_cast<const float2*>(&fp.ncT[2 * b]);
    const float2 hR = *reinterpret_cast<const float2*>(&fp.h[2 * b]);
    const float2 nhR = *reinterpret_cast<const float2*>(&fp.nh[2 * b]);
    tail(__fadd2_rn(pn, ncn), __fadd2_rn(pt, nct), __fadd2_rn(an, ncN), __fadd2_rn(at, ncT), hR, nhR,
         acc.gR[2 * b], acc.gR[2 * b + 1]);
    tail(__fadd2_rn(neg2(pn), ncn), __fadd2_rn(neg2(pt), nct), __fadd2_rn(neg2(an), ncN), __fadd2_rn(neg2(at), ncT), hR, nhR,
         acc.gR[2 * b + V / 2], acc.gR[2 * b + 1 + V / 2]);
  }
  acc.gO = fminf(acc.gO, gj);
  minD2 = m;
}

// Compile-time / run-time choice of the variant: SYM instantiations exist for V % 4 == 0 only.
template <int V, bool SUB_FIRST, bool SYM>
__device__ __forceinline__ void edge_step_any(const Footprint& fp, const Posed2<V>& P, const float4 q, const float h,
                                          ObstacleAcc<V>& acc, float& minD2) {
  if constexpr (SYM && V % 4 == 0) edge_step2_sym<V, SUB_FIRST>(fp, P, q, h, acc, minD2);
  else edge_step2<V, SUB_FIRST>(fp, P, q, h, acc, minD2);
}

// Order-preserving float -> uint32 key (works for negatives and +-inf).
__device__ __forceinline__ uint32_t fkey(float f) {
  uint32_t u = __float_as_uint(f);
  return (u & 0x80000000u) ? ~u : (u | 0x80000000u);
}
__device__ __forceinline__ float fkey_inv(uint32_t k) {
  return __uint_as_float((k & 0x80000000u) ? (k & 0x7fffffffu) : ~k);
}

// H8: analytic gradient at the arg-min witness of obstacle [e_begin, e_end), re-evaluated
// with witness tracking (only the winning obstacle: 1/M of the scan work).
//   separated:   n = unit vector from the obstacle witness to the robot witness, c = robot
//                witness (pose-relative);   not separated: n = push-out normal of the
//                minimum-overlap face, c = deepest vertex.   grad = (n_x, n_y, c x n).
// Two passes, because every kernel ends with this serial chain: pass 1 only finds WHICH
// candidate wins (value + index through predicated selects: branch-free, independent
// candidates overlap in the pipe; loads run one edge ahead), pass 2 recomputes that one
// candidate with its witness points.  Ties go to the first candidate in (edge, vertex, pool)
// order.
// The winner's pair records (two edges each: q0, q1 = (A, t), q2 = (h0, h1, last, slot)) are read
// again: the evaluation pass of this CTA has just pulled them into L1.
template <int V>
__device__ __forceinline__ void witness_separated(const Footprint& fp, const Posed<V>& P,
                                                  const float4* __restrict__ recs, int rec_begin, float* g) {
  float nx = 0.f, ny = 0.f, cx = 0.f, cy = 0.f;
  const float4* __restrict__ src = recs + 3 * (size_t)rec_begin;
  // edge `j` of the obstacle (j = 2 * record + half), whichever half it is
  auto edge_at = [&](int j, float4& e0, float& h) {
    const float4* r = src + 3 * (j >> 1);
    e0 = __ldg(r + (j & 1));
    const float4 q2 = __ldg(r + 2);
    h = (j & 1) ? q2.y : q2.x;
  };
  float best = kInf;
  int idx = 0;                                           // (j * V + l) * 2 + pool
  int base = 0;
  for (const float4* r = src;; r += 3) {
    const float4 c0 = __ldg(r), c1 = __ldg(r + 1), q2 = __ldg(r + 2);
    const float h0 = q2.x, h1 = q2.y;
    const bool more = __float_as_int(q2.z) < 0;
#pragma unroll
    for (int half = 0; half < 2; ++half) {
      const float4 e0 = half ? c1 : c0;
      const float h = half ? h1 : h0;
      if (half && !(h1 >= 0.f)) break;                   // odd edge count: second half unused
      const float ax = e0.x - P.px, ay = e0.y - P.py, tx = e0.z, ty = e0.w;
#pragma unroll
      for (int l = 0; l < V; ++l) {
        const float dx = P.rx[l] - ax, dy = P.ry[l] - ay;
        // pool 1: robot vertex l -> obstacle edge j
        const float sig = dy * tx - dx * ty;
        const float tm = fmaf(dx, tx, dy * ty) - h;
        const float ex = fmaxf(fabsf(tm), h) - h;
        const float d1 = fmaf(ex, ex, sig * sig);
        // pool 2: obstacle vertex a_j -> robot edge l
        const float Tx = P.Tx[l], Ty = P.Ty[l];
        const float sigp = -(dy * Tx - dx * Ty);
        const float tmp = -fmaf(dx, Tx, dy * Ty) - fp.h[l];
        const float exp_ = fmaxf(fabsf(tmp), fp.h[l]) - fp.h[l];
        const float d2 = fmaf(exp_, exp_, sigp * sigp);
        const bool p1 = d1 < best;
        best = p1 ? d1 : best;
        idx = p1 ? base + 2 * l : idx;
        const bool p2 = d2 < best;
        best = p2 ? d2 : best;
        idx = p2 ? base + 2 * l + 1 : idx;
      }
      base += 2 * V;
    }
    if (!more) break;
  }
  // pass 2: the winning candidate again, with its witness
  const int j = idx / (2 * V), l = (idx / 2) % V;
  float4 e0;
  float h;
  edge_at(j, e0, h);
  const float ax = e0.x - P.px, ay = e0.y - P.py;
  float rx = 0.f, ry = 0.f, Tx = 0.f, Ty = 0.f, hl = 0.f;
#pragma unroll
  for (int q = 0; q < V; ++q)
    if (q == l) { rx = P.rx[q]; ry = P.ry[q]; Tx = P.Tx[q]; Ty = P.Ty[q]; hl = fp.h[q]; }
  const float dx = rx - ax, dy = ry - ay;
  if (!(idx & 1)) {                                      // (w - Q) = sig n + ex t
    const float tx = e0.z, ty = e0.w;
    const float sig = dy * tx - dx * ty;
    const float tm = fmaf(dx, tx, dy * ty) - h;
    const float ex = copysignf(fmaxf(fabsf(tm), h) - h, tm);
    const float inv = rsqrtf(fmaxf(fmaf(ex, ex, sig * sig), 1e-30f));
    nx = (ex * tx - sig * ty) * inv;
    ny = (ex * ty + sig * tx) * inv;
    cx = rx;
    cy = ry;
  } else {                                               // (a - Q) = sig' N + ex' T
    const float sig = -(dy * Tx - dx * Ty);
    const float tm = -fmaf(dx, Tx, dy * Ty) - hl;
    const float ex = copysignf(fmaxf(fabsf(tm), hl) - hl, tm);
    const float inv = rsqrtf(fmaxf(fmaf(ex, ex, sig * sig), 1e-30f));
    const float ux = (ex * Tx - sig * Ty), uy = (ex * Ty + sig * Tx);      // a - Q
    nx = -ux * inv;
    ny = -uy * inv;
    cx = ax - ux;
    cy = ay - uy;
  }
  g[0] = nx;
  g[1] = ny;
  g[2] = cx * ny - cy * nx;
}

template <int V>
__device__ __forceinline__ void witness_penetrating(const Footprint& fp, const Posed<V>& P,
                                                    const float4* __restrict__ recs, int rec_begin, float* g) {
  float nx = 0.f, ny = 0.f, cx = 0.f, cy = 0.f;
  const float4* __restrict__ src = recs + 3 * (size_t)rec_begin;
  // edge `j` of the obstacle (j = 2 * record + half), whichever half it is
  auto edge_at = [&](int j, float4& e0, float& h) {
    const float4* r = src + 3 * (j >> 1);
    e0 = __ldg(r + (j & 1));
    const float4 q2 = __ldg(r + 2);
    h = (j & 1) ? q2.y : q2.x;
  };
  float bestO = kInf;                                    // minimum obstacle-face depth and its edge
  int jO = 0;
  float gR[V];                                           // robot-face depths and the edge whose start is deepest
  int jR[V];
#pragma unroll
  for (int l = 0; l < V; ++l) { gR[l] = -kInf; jR[l] = 0; }
  int j = 0;
  for (const float4* r = src;; r += 3) {
    const float4 c0 = __ldg(r), c1 = __ldg(r + 1), q2 = __ldg(r + 2);
    const float h1 = q2.y;
    const bool more = __float_as_int(q2.z) < 0;
#pragma unroll
    for (int half = 0; half < 2; ++half) {
      if (half && !(h1 >= 0.f)) break;
      const float4 e0 = half ? c1 : c0;
      const float ax = e0.x - P.px, ay = e0.y - P.py, tx = e0.z, ty = e0.w;
      float gj = -kInf;
#pragma unroll
      for (int l = 0; l < V; ++l) {
        const float dx = P.rx[l] - ax, dy = P.ry[l] - ay;
        gj = fmaxf(gj, dy * tx - dx * ty);
        const float sigp = -(dy * P.Tx[l] - dx * P.Ty[l]);
        const bool pr = sigp > gR[l];
        gR[l] = pr ? sigp : gR[l];
        jR[l] = pr ? j : jR[l];
      }
      const bool po = gj < bestO;
      bestO = po ? gj : bestO;
      jO = po ? j : jO;
      ++j;
    }
    if (!more) break;
  }
  float best = bestO;
  int face = -1, jF = jO;                                // -1: obstacle face jO, else robot face
#pragma unroll
  for (int l = 0; l < V; ++l)
    if (gR[l] < best) { best = gR[l]; face = l; jF = jR[l]; nx = -P.Ty[l]; ny = P.Tx[l]; }
  float4 e0;
  float h;
  edge_at(jF, e0, h);
  const float ax = e0.x - P.px, ay = e0.y - P.py;
  if (face < 0) {                                        // n = -n_in of edge jO, c = its deepest robot vertex
    const float tx = e0.z, ty = e0.w;
    float gj = -kInf;
#pragma unroll
    for (int l = 0; l < V; ++l) {
      const float sig = (P.ry[l] - ay) * tx - (P.rx[l] - ax) * ty;
      if (sig > gj) { gj = sig; cx = P.rx[l]; cy = P.ry[l]; }
    }
    nx = ty;
    ny = -tx;
  } else {                                               // c = the obstacle vertex deepest behind robot face `face`
    cx = ax;
    cy = ay;
  }
  g[0] = nx;
  g[1] = ny;
  g[2] = cx * ny - cy * nx;
}

template <int V>
__device__ __forceinline__ void witness_gradient(const Footprint& fp, const Posed<V>& P,
                                                 const float4* __restrict__ recs, int rec_begin,
                                                 bool separated, float* g) {
  if (separated) witness_separated<V>(fp, P, recs, rec_begin, g);
  else witness_penetrating<V>(fp, P, recs, rec_begin, g);
}


}  // namespace psdf
