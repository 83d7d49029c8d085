// PSDF oracle — TEST INFRASTRUCTURE, NOT THE PRODUCT.
//
// A plain, slow, double-precision CPU restatement of the polygonal signed distance
// function of arxiv/paper_2607_04310 (§IV, eqs.(9)-(23), (6)), written from the
// paper step by step in the paper's own robot-local frame and notation.  Only tests/,
// __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may call
// it.  It shares no code, header, table or constant with the CUDA path
// (paper_2607_04310_b200/csrc) and neither side includes the other.
//
// What it computes, per pose x=(p,theta) and obstacle i (PAPER.md line numbers):
//   O1  A~ = R(theta)^T (A - p), B~ likewise                      eq.(11)
//   O2  d(P,[A,B]): v=B-A, u=(P-A).v/|v|^2, t=ReLU(u)-ReLU(u-1),
//       Q=A+t v, d=|P-Q|                                           eqs.(12)-(13) PAPER.md:153-163
//   O3  d_v (14), d_e (15), d_sep=min (16)
//   O4  axes (17)-(18), intervals (19), overlap (20),
//       separated (21), depth delta (22)
//   O5  sd^i (23), phi = min_i sd^i (6), first index on ties
//   O6  gradient d phi / d(x,y,theta): forward-mode dual numbers through O1-O5
//       literally ("automatic differentiation" of the graph); min / max /
//       select propagate the tangent of the selected operand (first index on ties),
//       ReLU'(u)=0 for u<=0.
//   O7  margin: along the selected path, the smallest value gap to any competing
//       operand of a min/max whose tangent differs by more than 1e-6 (DESIGN.md reading
//       G9).  ReLU kinks are exempt (the point-to-segment distance is C^1 across them).
//
// Masking (reading G6): entries with S=0 are skipped in every
// reduction and contribute no axis and no vertex; a row with no valid entry has sd=+inf.
// No epsilon anywhere; Assumption 1 is asserted by the caller.
//
// Parity pins (tests/test_oracle_*.py): closed forms P1-P11, Minkowski-difference
// definition of (5a-c), dense-sampling brute force, invariances, finite differences.
// "parity unpinned": only the paper-literal treatment of OPEN polylines (vertex set =
// valid A_j only, reading G7) — generators never emit them.
//
// Build: g++ -O2 -fopenmp -shared -fPIC (no -ffast-math); see oracle/build.py.
#include <cmath>
#include <cstdint>
#include <limits>
#include <vector>
#ifdef _OPENMP
#include <omp.h>
#endif

namespace {

const double INF = std::numeric_limits<double>::infinity();
const double TANGENT_TOL = 1e-6;   // "gradient differs" threshold of reading G9

// ---------------------------------------------------------------- dual number (x,y,theta)
struct Dual {
  double v;      // value
  double g[3];   // tangent w.r.t. (x, y, theta)
  double m;      // margin accumulated along the selected path (metres)
};

inline Dual mk(double v) { return Dual{v, {0, 0, 0}, INF}; }
inline double val(const Dual& a) { return a.v; }
inline double val(double a) { return a; }

inline Dual operator+(const Dual& a, const Dual& b) {
  return Dual{a.v + b.v, {a.g[0] + b.g[0], a.g[1] + b.g[1], a.g[2] + b.g[2]}, std::fmin(a.m, b.m)};
}
inline Dual operator-(const Dual& a, const Dual& b) {
  return Dual{a.v - b.v, {a.g[0] - b.g[0], a.g[1] - b.g[1], a.g[2] - b.g[2]}, std::fmin(a.m, b.m)};
}
inline Dual operator-(const Dual& a) { return Dual{-a.v, {-a.g[0], -a.g[1], -a.g[2]}, a.m}; }
inline Dual operator*(const Dual& a, const Dual& b) {
  return Dual{a.v * b.v,
              {a.g[0] * b.v + a.v * b.g[0], a.g[1] * b.v + a.v * b.g[1], a.g[2] * b.v + a.v * b.g[2]},
              std::fmin(a.m, b.m)};
}
inline Dual operator/(const Dual& a, const Dual& b) {
  double q = a.v / b.v;
  return Dual{q,
              {(a.g[0] - q * b.g[0]) / b.v, (a.g[1] - q * b.g[1]) / b.v, (a.g[2] - q * b.g[2]) / b.v},
              std::fmin(a.m, b.m)};
}
inline Dual operator+(const Dual& a, double b) { return Dual{a.v + b, {a.g[0], a.g[1], a.g[2]}, a.m}; }
inline Dual operator-(const Dual& a, double b) { return Dual{a.v - b, {a.g[0], a.g[1], a.g[2]}, a.m}; }
inline Dual operator-(double a, const Dual& b) { return Dual{a - b.v, {-b.g[0], -b.g[1], -b.g[2]}, b.m}; }
inline Dual operator*(const Dual& a, double b) { return Dual{a.v * b, {a.g[0] * b, a.g[1] * b, a.g[2] * b}, a.m}; }
inline Dual operator*(double a, const Dual& b) { return b * a; }

inline Dual Sqrt(const Dual& a) {
  double r = std::sqrt(a.v);
  if (r == 0.0) return Dual{0.0, {0, 0, 0}, a.m};     // |.| at 0: subgradient 0
  double k = 0.5 / r;
  return Dual{r, {a.g[0] * k, a.g[1] * k, a.g[2] * k}, a.m};
}
inline double Sqrt(double a) { return std::sqrt(a); }

// ReLU(u) = max(u,0) with ReLU'(0)=0; exempt from the margin (O7).
inline Dual Relu(const Dual& u) { return u.v > 0.0 ? u : Dual{0.0, {0, 0, 0}, u.m}; }
inline double Relu(double u) { return u > 0.0 ? u : 0.0; }

inline bool tangent_differs(const Dual& a, const Dual& b) {
  return std::fabs(a.g[0] - b.g[0]) > TANGENT_TOL || std::fabs(a.g[1] - b.g[1]) > TANGENT_TOL ||
         std::fabs(a.g[2] - b.g[2]) > TANGENT_TOL;
}

// Reductions over an explicit candidate list.  sign=+1: min, sign=-1: max.  First index
// wins exact ties.  Margin of the result (O7): min over the losers of
//   gap                    if the loser's tangent differs from the winner's,
//   gap + loser's margin   otherwise (same witness: its own runner-ups are that far away).
inline Dual reduce(const std::vector<Dual>& c, int sign, int* arg = nullptr) {
  size_t best = 0;
  for (size_t k = 1; k < c.size(); ++k)
    if (sign > 0 ? (c[k].v < c[best].v) : (c[k].v > c[best].v)) best = k;
  Dual r = c[best];
  for (size_t k = 0; k < c.size(); ++k) {
    if (k == best) continue;
    double gap = std::fabs(c[k].v - r.v);
    double mk_ = tangent_differs(c[k], r) ? gap : gap + c[k].m;
    if (mk_ < r.m) r.m = mk_;
  }
  if (arg) *arg = (int)best;
  return r;
}
inline double reduce(const std::vector<double>& c, int sign, int* arg = nullptr) {
  size_t best = 0;
  for (size_t k = 1; k < c.size(); ++k)
    if (sign > 0 ? (c[k] < c[best]) : (c[k] > c[best])) best = k;
  if (arg) *arg = (int)best;
  return c[best];
}
template <class T> inline T Min2(const T& a, const T& b) { return reduce(std::vector<T>{a, b}, +1); }
template <class T> inline T Max2(const T& a, const T& b) { return reduce(std::vector<T>{a, b}, -1); }

template <class T> struct Vec2 { T x, y; };

// ---------------------------------------------------------------- O2: eqs.(12)-(13)
template <class T>
T point_segment(const Vec2<T>& P, const Vec2<T>& A, const Vec2<T>& B) {
  T vx = B.x - A.x, vy = B.y - A.y;                       // v = B - A
  T u = ((P.x - A.x) * vx + (P.y - A.y) * vy) / (vx * vx + vy * vy);
  T t = Relu(u) - Relu(u - 1.0);                          // eq.(12)
  T Qx = A.x + t * vx, Qy = A.y + t * vy;                 // eq.(13)
  T ex = P.x - Qx, ey = P.y - Qy;
  return Sqrt(ex * ex + ey * ey);
}

template <class T> inline T cst(double c);
template <> inline double cst<double>(double c) { return c; }
template <> inline Dual cst<Dual>(double c) { return mk(c); }

struct Scene {
  int V, M, E;
  const double* fp;   // [V,2]
  const double* A;    // [M,E,2]
  const double* B;    // [M,E,2]
  const uint8_t* S;   // [M,E]
};

// ---------------------------------------------------------------- sd^i: O1-O5 for one obstacle
// Returns false for a row with no valid edge (sd = +inf).
template <class T>
bool sd_obstacle(const Scene& sc, int i, const T& px, const T& py, const T& c, const T& s, T* out,
                 bool* separated_out) {
  const int V = sc.V, E = sc.E;
  // O1, eq.(11): localise valid endpoints.  R^T = [[c, s], [-s, c]].
  std::vector<Vec2<T>> At, Bt;
  for (int j = 0; j < E; ++j) {
    if (!sc.S[(size_t)i * E + j]) continue;               // masked: excluded everywhere
    const double* a = sc.A + ((size_t)i * E + j) * 2;
    const double* b = sc.B + ((size_t)i * E + j) * 2;
    T ax = a[0] - px, ay = a[1] - py, bx = b[0] - px, by = b[1] - py;
    At.push_back(Vec2<T>{c * ax + s * ay, c * ay - s * ax});
    Bt.push_back(Vec2<T>{c * bx + s * by, c * by - s * bx});
  }
  const int e = (int)At.size();
  if (e == 0) return false;
  std::vector<Vec2<T>> v0(V);                             // robot vertices in L (constants)
  for (int l = 0; l < V; ++l) v0[l] = Vec2<T>{cst<T>(sc.fp[2 * l]), cst<T>(sc.fp[2 * l + 1])};

  // O3, eq.(14): robot vertices x obstacle edges.
  std::vector<T> pool1;
  for (int l = 0; l < V; ++l)
    for (int j = 0; j < e; ++j) pool1.push_back(point_segment(v0[l], At[j], Bt[j]));
  T d_v = reduce(pool1, +1);
  // eq.(15): obstacle vertices (valid A~_j) x robot edges E_l = [v_l, v_{l+1}].
  std::vector<T> pool2;
  for (int j = 0; j < e; ++j)
    for (int l = 0; l < V; ++l) pool2.push_back(point_segment(At[j], v0[l], v0[(l + 1) % V]));
  T d_e = reduce(pool2, +1);
  T d_sep = Min2(d_v, d_e);                               // eq.(16)

  // O4, eqs.(17)-(18): candidate axes = robot edge normals, then valid obstacle edge normals.
  std::vector<Vec2<T>> axes;
  for (int l = 0; l < V; ++l) {
    T ux = v0[(l + 1) % V].x - v0[l].x, uy = v0[(l + 1) % V].y - v0[l].y;
    T nrm = Sqrt(ux * ux + uy * uy);
    axes.push_back(Vec2<T>{-uy / nrm, ux / nrm});          // rot90(x,y) = (-y,x)
  }
  for (int j = 0; j < e; ++j) {
    T ux = Bt[j].x - At[j].x, uy = Bt[j].y - At[j].y;
    T nrm = Sqrt(ux * ux + uy * uy);
    axes.push_back(Vec2<T>{-uy / nrm, ux / nrm});
  }
  bool separated = false;
  std::vector<T> clipped;
  for (const Vec2<T>& n : axes) {
    std::vector<T> pr0, pri;                              // eq.(19)
    for (int l = 0; l < V; ++l) pr0.push_back(v0[l].x * n.x + v0[l].y * n.y);
    for (int j = 0; j < e; ++j) pri.push_back(At[j].x * n.x + At[j].y * n.y);
    T a0 = reduce(pr0, +1), b0 = reduce(pr0, -1);
    T ai = reduce(pri, +1), bi = reduce(pri, -1);
    T delta = Min2(bi - a0, b0 - ai);                     // eq.(20)
    if (val(delta) < 0.0) separated = true;               // eq.(21)
    clipped.push_back(Max2(delta, cst<T>(0.0)));          // eq.(22) operand
  }
  T depth = reduce(clipped, +1);                          // eq.(22)
  *out = separated ? d_sep : -depth;                      // eq.(23)
  if (separated_out) *separated_out = separated;
  return true;
}

}  // namespace

extern "C" {

// All arrays host, row-major, double (the Python wrapper widens float32 exactly).
//   footprint [V,2]   A,B [M,E,2]   S [M,E] (0/1)   poses [N,3] = x,y,theta
// Outputs (any may be NULL except value):
//   value [N]; grad [N,3]; per_obstacle [N,M] (+inf for empty rows); margin [N];
//   winner [N] (obstacle row, -1 if none); branch [N] (1 separated, 0 penetrating/contact).
// window >= 0: forward-mode duals are evaluated only for obstacles whose plain-double
//   sd^i lies within `window` of phi (the reported margin is then capped at `window`);
//   window < 0: duals for every obstacle (used by tests to check the two agree).
// nthreads <= 0: OpenMP default.  Returns 0, or -1 on bad arguments.
int psdf_oracle_eval(const double* footprint, int V, const double* A, const double* B,
                     const uint8_t* S, int M, int E, const double* poses, int N, double* value,
                     double* grad, double* per_obstacle, double* margin, int* winner, int* branch,
                     double window, int nthreads) {
  if (!footprint || !A || !B || !S || !poses || !value || V < 3 || M < 1 || E < 1 || N < 0) return -1;
  Scene sc{V, M, E, footprint, A, B, S};
#ifdef _OPENMP
  if (nthreads > 0) omp_set_num_threads(nthreads);
#endif
#pragma omp parallel for schedule(dynamic, 16)
  for (int n = 0; n < N; ++n) {
    const double px = poses[3 * n], py = poses[3 * n + 1], th = poses[3 * n + 2];
    const double c = std::cos(th), s = std::sin(th);
    // plain-double pass: sd^i for every obstacle, phi = min_i (eq.6)
    std::vector<double> sd(M, INF);
    std::vector<char> sepf(M, 0);
    for (int i = 0; i < M; ++i) {
      double v; bool sp = false;
      if (sd_obstacle<double>(sc, i, px, py, c, s, &v, &sp)) { sd[i] = v; sepf[i] = sp; }
      if (per_obstacle) per_obstacle[(size_t)n * M + i] = sd[i];
    }
    int win = 0;
    double phi = reduce(sd, +1, &win);
    if (phi == INF) win = -1;
    value[n] = phi;
    if (winner) winner[n] = win;
    if (branch) branch[n] = win >= 0 ? (int)sepf[win] : 1;
    if (!grad && !margin) continue;
    if (win < 0) {
      if (grad) grad[3 * n] = grad[3 * n + 1] = grad[3 * n + 2] = 0.0;
      if (margin) margin[n] = INF;
      continue;
    }
    // forward-mode pass (O6): seeds dx=(1,0,0), dy=(0,1,0), dtheta=(0,0,1)
    Dual Px{px, {1, 0, 0}, INF}, Py{py, {0, 1, 0}, INF};
    Dual C{c, {0, 0, -s}, INF}, Sn{s, {0, 0, c}, INF};
    std::vector<Dual> cand;
    for (int i = 0; i < M; ++i) {
      if (sd[i] == INF) continue;
      if (window >= 0.0 && sd[i] > phi + window) continue;
      Dual v;
      sd_obstacle<Dual>(sc, i, Px, Py, C, Sn, &v, nullptr);
      cand.push_back(v);
    }
    Dual r = reduce(cand, +1);                            // eq.(6), first index on ties
    if (grad) { grad[3 * n] = r.g[0]; grad[3 * n + 1] = r.g[1]; grad[3 * n + 2] = r.g[2]; }
    if (margin) margin[n] = (window >= 0.0 && r.m > window) ? window : r.m;
  }
  return 0;
}

int psdf_oracle_max_threads(void) {
#ifdef _OPENMP
  return omp_get_max_threads();
#else
  return 1;
#endif
}

}  // extern "C"
