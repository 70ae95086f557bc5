// fk_oracle.cpp -- CPU oracle of the Feynman-Kac exit-time scheme (arXiv 2104.14561).
//
// TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only tests/, __graft_entry__.smoke() and
// bench.py's cpu_baseline / --impl reference legs may build, load or call this file.
// It shares no code, header, table or helper with paper_2104_14561_b200/csrc (the CUDA path).
//
// Plain, slow and meant to be checked against the paper by eye: one quadrature point at a
// time, no merged weights, no tiling, no operator matrix.  Arithmetic is fp64; the weighted
// sum over quadrature points is accumulated in long double so that what is left between this
// file and the CUDA path is the CUDA path's own rounding.  Compile with -ffp-contract=off.
//
// What follows what (PAPER.md line, equation):
//   ofk_gauss_hermite   PAPER.md:197       Gauss-Hermite rule for the density pi^{-1/2} e^{-xi^2}
//   ofk_chi             PAPER.md:266-269   Eq. 28 terminal vector chi
//   ofk_pchip_slopes    PAPER.md:150-160   Eq. 15 nodal slopes (incl. the end-node rule)
//   ofk_interp          PAPER.md:138-148   Eq. 13-14, multi-D by tensor product (reading R4/A)
//   ofk_apply           PAPER.md:224-229   Scheme 1 steps 1-3 = Eq. 21, 20, 22 for one field
//   ofk_column          PAPER.md:271-273   Eq. 29: p^m = A_0 (A_1 ... (A_{m-1} chi))
//   ofk_algorithm1      PAPER.md:277-291   Algorithm 1 (all columns, one pass)
//   ofk_reduce          PAPER.md:62-66, 453  sum_j w_j P(t_m, x_j): the quadrature of
//                                          int P(t,x) P_init(x) dx and of the moment of Eq. 42
// Readings of silent / garbled points (R1..R20) are listed in DESIGN.md; the ones used here:
//   R1 weights normalised to sum 1; R2 sigma*sqrt(2 dt)*a_q; R4 values + nodal gradient, no
//   mixed derivatives; R5 unweighted harmonic mean; R6 end nodes use the first/last two
//   divided differences with the same sign test; R7 a zero difference gives slope 0;
//   R8 a point strictly outside an ABSORB face takes that face's value g; R9 CLAMP faces
//   project the point onto the box first, then the lowest ABSORB dimension left outside
//   decides g; R10 column 0 is chi; R11 coefficients at the left end t_nu; R15 Dirichlet
//   nodes (on an ABSORB face) keep their value; R19 cell = the one with x[c] <= z < x[c+1];
//   R21 PERIODIC dimension ("periodic in x1"): the last node is the image of the
//   first, a point is wrapped into [alpha, beta) before it is located, slopes use the cell across
//   the seam; R22 slope_rule = 1: Fritsch-Carlson weighted harmonic mean (ref [17], PAPER.md:134,
//   152-160) -- interior nodes w1 = 2 h_j + h_{j-1}, w2 = h_j + 2 h_{j-1}; the end nodes apply the
//   same weights to their first / last two cells.
//
// Pins (tests/test_oracle_*.py, none of them re-types these formulas): closed-form GH rules
// and moments; the hand-derived 5-node micro-example in tests/golden/; affine exactness;
// pure shift at sigma=0; the textbook series for Brownian exit from an interval with the
// first-order-in-dt convergence the paper claims; invariants; Monte-Carlo exit counts;
// Algorithm 1 == per-column Scheme 1; the autonomous chain property.
// Parity unpinned against truth: the multi-D configs 3-5 have no analytic solution and the
// paper's figure data is not available; they are pinned only through the operator-level
// identities above, the reduction to 1-D along lines, and loose Monte-Carlo.

#include <algorithm>
#include <cmath>
#include <cstdlib>
#include <cstring>
#include <vector>
#ifdef _OPENMP
#include <omp.h>
#endif

extern "C" {

enum { OFK_ABSORB = 0, OFK_CLAMP = 1, OFK_PERIODIC = 2 };

typedef struct {
  int d;                    // 1..3
  int n[3];                 // nodes per dimension
  const double* x[3];       // node coordinates, strictly increasing
  double dt;                // time step
  int Q[3];                 // Gauss-Hermite points per dimension
  int face_kind[3][2];      // [dim][lo/hi]
  double face_value[3][2];  // g for ABSORB faces
  int slope_rule;           // 0: Eq. 15 as printed (unweighted harmonic mean); 1: weighted (R22)
} ofk_problem;

// ---------------------------------------------------------------------------------------
// Gauss-Hermite rule for weight e^{-x^2}, weights divided by sqrt(pi).
// Roots of the physicists' Hermite polynomial H_Q by interlacing: the roots of H_m separate
// those of H_{m+1}, so each root is bracketed by bisection, then polished by Newton.
// w_q = 2^{Q-1} Q! sqrt(pi) / (Q^2 H_{Q-1}(a_q)^2), divided by sqrt(pi).
// ---------------------------------------------------------------------------------------
static long double hermite_H(int m, long double x) {
  long double h0 = 1.0L, h1 = 2.0L * x;
  if (m == 0) return h0;
  for (int k = 1; k < m; ++k) {
    long double h2 = 2.0L * x * h1 - 2.0L * k * h0;
    h0 = h1;
    h1 = h2;
  }
  return h1;
}

int ofk_gauss_hermite(int Q, double* a, double* w) {
  if (Q < 1 || Q > 64) return 1;
  std::vector<long double> prev, cur;
  for (int m = 1; m <= Q; ++m) {
    cur.assign(m, 0.0L);
    const long double B = std::sqrt((long double)(2 * m + 1)) + 1.0L;  // all roots lie inside
    for (int i = 0; i < m; ++i) {
      long double lo = (i == 0) ? -B : prev[i - 1];
      long double hi = (i == m - 1) ? B : prev[i];
      long double flo = hermite_H(m, lo);
      for (int it = 0; it < 200; ++it) {
        long double mid = 0.5L * (lo + hi);
        long double fm = hermite_H(m, mid);
        if ((fm < 0) == (flo < 0)) { lo = mid; flo = fm; } else { hi = mid; }
      }
      long double r = 0.5L * (lo + hi);
      for (int it = 0; it < 4; ++it) {               // H_m' = 2 m H_{m-1}
        long double dH = 2.0L * m * hermite_H(m - 1, r);
        r -= hermite_H(m, r) / dH;
      }
      cur[i] = r;
    }
    prev = cur;
  }
  long double fact = 1.0L;
  for (int k = 2; k <= Q; ++k) fact *= k;
  long double pow2 = std::pow(2.0L, Q - 1);
  for (int i = 0; i < Q; ++i) {
    long double r = cur[i];
    if (Q % 2 == 1 && i == Q / 2) r = 0.0L;          // exact middle root
    long double h = hermite_H(Q - 1, r);
    a[i] = (double)r;
    w[i] = (double)(pow2 * fact / ((long double)Q * Q * h * h));
  }
  return 0;
}

// ---------------------------------------------------------------------------------------
// helpers on the tensor grid; node index j = ((i0*n1)+i1)*n2+i2 (last dimension fastest)
// ---------------------------------------------------------------------------------------
static long total_nodes(const ofk_problem* p) {
  long J = 1;
  for (int k = 0; k < p->d; ++k) J *= p->n[k];
  return J;
}

static void strides(const ofk_problem* p, long st[3]) {
  st[0] = st[1] = st[2] = 0;
  long s = 1;
  for (int k = p->d - 1; k >= 0; --k) { st[k] = s; s *= p->n[k]; }
}

static void unravel(const ofk_problem* p, long j, int idx[3]) {
  for (int k = p->d - 1; k >= 0; --k) { idx[k] = (int)(j % p->n[k]); j /= p->n[k]; }
}

// Is node idx on an ABSORB face?  If so *g is the face value; lowest dimension wins (R9).
static bool dirichlet(const ofk_problem* p, const int idx[3], double* g) {
  for (int k = 0; k < p->d; ++k) {
    if (idx[k] == 0 && p->face_kind[k][0] == OFK_ABSORB) { *g = p->face_value[k][0]; return true; }
    if (idx[k] == p->n[k] - 1 && p->face_kind[k][1] == OFK_ABSORB) { *g = p->face_value[k][1]; return true; }
  }
  return false;
}

// Eq. 28: chi = g on the ABSORB faces, 0 elsewhere.
int ofk_chi(const ofk_problem* p, double* chi) {
  long J = total_nodes(p);
  for (long j = 0; j < J; ++j) {
    int idx[3];
    unravel(p, j, idx);
    double g;
    chi[j] = dirichlet(p, idx, &g) ? g : 0.0;
  }
  return 0;
}

// ---------------------------------------------------------------------------------------
// Eq. 15: PCHIP slopes on one grid line.
// delta_j = (u_{j+1}-u_j)/(x_{j+1}-x_j), j = 0..n-2.
// interior j: 0 if delta_{j-1}, delta_j differ in sign (or one is 0), else 2/(1/d_{j-1}+1/d_j)
// node 0 uses (delta_0, delta_1); node n-1 uses (delta_{n-2}, delta_{n-3}).
// ---------------------------------------------------------------------------------------
static double harmonic(double da, double db) {
  bool same = (da > 0.0 && db > 0.0) || (da < 0.0 && db < 0.0);
  if (!same) return 0.0;
  return 2.0 / (1.0 / da + 1.0 / db);
}

// R22: weighted harmonic mean of the divided differences da (cell of width ha) and db (cell of
// width hb) that meet at a node: (w1 + w2) / (w1 / da + w2 / db), w1 = 2 hb + ha, w2 = hb + 2 ha.
static double harmonic_weighted(double da, double db, double ha, double hb) {
  bool same = (da > 0.0 && db > 0.0) || (da < 0.0 && db < 0.0);
  if (!same) return 0.0;
  double w1 = 2.0 * hb + ha, w2 = hb + 2.0 * ha;
  return (w1 + w2) / (w1 / da + w2 / db);
}

static double node_slope(double da, double db, double ha, double hb, int weighted) {
  return weighted ? harmonic_weighted(da, db, ha, hb) : harmonic(da, db);
}

// periodic != 0 (R21): node n-1 is the image of node 0, so both take the slope of the two cells
// that meet there, the last cell (n-2) and the first (0).
int ofk_pchip_slopes_ex(int n, const double* x, const double* u, long stride, double* du,
                        int periodic, int weighted) {
  if (n < 3) return 1;
  std::vector<double> delta(n - 1), h(n - 1);
  for (int j = 0; j < n - 1; ++j) {
    h[j] = x[j + 1] - x[j];
    delta[j] = (u[(long)(j + 1) * stride] - u[(long)j * stride]) / h[j];
  }
  for (int j = 1; j < n - 1; ++j)
    du[(long)j * stride] = node_slope(delta[j - 1], delta[j], h[j - 1], h[j], weighted);
  if (periodic) {
    double s = node_slope(delta[n - 2], delta[0], h[n - 2], h[0], weighted);
    du[0] = s;
    du[(long)(n - 1) * stride] = s;
  } else {
    du[0] = node_slope(delta[0], delta[1], h[0], h[1], weighted);
    du[(long)(n - 1) * stride] = node_slope(delta[n - 2], delta[n - 3], h[n - 2], h[n - 3], weighted);
  }
  return 0;
}

int ofk_pchip_slopes(int n, const double* x, const double* u, long stride, double* du) {
  return ofk_pchip_slopes_ex(n, x, u, stride, du, 0, 0);
}

// All d partial-derivative fields of u: du[k][j], slopes along the grid lines of axis k.
static void gradient_fields(const ofk_problem* p, const double* u, double* du /*[d][J]*/) {
  long J = total_nodes(p);
  long st[3];
  strides(p, st);
  for (int k = 0; k < p->d; ++k) {
    double* dk = du + (long)k * J;
#pragma omp parallel for schedule(static)
    for (long j = 0; j < J; ++j) {
      int idx[3];
      unravel(p, j, idx);
      if (idx[k] != 0) continue;                     // j is the first node of a line along k
      ofk_pchip_slopes_ex(p->n[k], p->x[k], u + j, st[k], dk + j,
                          p->face_kind[k][0] == OFK_PERIODIC, p->slope_rule);
    }
  }
}

// Eq. 14 basis on a cell of width h at s = x - x_j:
//   value-right (3 h s^2 - 2 s^3)/h^3, value-left (h^3 - 3 h s^2 + 2 s^3)/h^3,
//   slope-right s^2 (s-h)/h^2,         slope-left s (s-h)^2/h^2.
static void hermite_basis(double s, double h, double* vl, double* vr, double* sl, double* sr) {
  double h2 = h * h, h3 = h2 * h, s2 = s * s, s3 = s2 * s;
  *vr = (3.0 * h * s2 - 2.0 * s3) / h3;
  *vl = (h3 - 3.0 * h * s2 + 2.0 * s3) / h3;
  *sr = s2 * (s - h) / h2;
  *sl = s * (s - h) * (s - h) / h2;
}

// cell c with x[c] <= z < x[c+1], clamped to 0..n-2 (so z = x[n-1] falls in the last cell)
static int locate(int n, const double* x, double z) {
  int c = (int)(std::upper_bound(x, x + n, z) - x) - 1;   // last node with x[c] <= z
  if (c < 0) c = 0;
  if (c > n - 2) c = n - 2;
  return c;
}

// Eq. 13 in d dimensions, reading R4/A: on the cell containing z,
//   u(z) = sum_{corner c} [ u_c prod_k V_{c_k}(z_k)
//                          + sum_k (d_k u)_c S_{c_k}(z_k) prod_{l != k} V_{c_l}(z_l) ].
static long double interp_point(const ofk_problem* p, const double* u, const double* du,
                                const double z[3]) {
  long J = total_nodes(p);
  long st[3];
  strides(p, st);
  int cell[3];
  double V[3][2], S[3][2];
  for (int k = 0; k < p->d; ++k) {
    cell[k] = locate(p->n[k], p->x[k], z[k]);
    double h = p->x[k][cell[k] + 1] - p->x[k][cell[k]];
    double s = z[k] - p->x[k][cell[k]];
    hermite_basis(s, h, &V[k][0], &V[k][1], &S[k][0], &S[k][1]);
  }
  long double val = 0.0L;
  for (int corner = 0; corner < (1 << p->d); ++corner) {
    int c[3];
    long node = 0;
    for (int k = 0; k < p->d; ++k) {
      c[k] = (corner >> k) & 1;
      node += (long)(cell[k] + c[k]) * st[k];
    }
    long double pv = 1.0L;
    for (int k = 0; k < p->d; ++k) pv *= V[k][c[k]];
    val += pv * (long double)u[node];
    for (int k = 0; k < p->d; ++k) {
      long double ps = S[k][c[k]];
      for (int l = 0; l < p->d; ++l)
        if (l != k) ps *= V[l][c[l]];
      val += ps * (long double)du[(long)k * J + node];
    }
  }
  return val;
}

// Interpolate a field at npts points (row-major pts[npts][d]); points must lie in the box.
int ofk_interp(const ofk_problem* p, const double* u, long npts, const double* pts, double* out) {
  long J = total_nodes(p);
  std::vector<double> du((size_t)p->d * J);
  gradient_fields(p, u, du.data());
  for (long i = 0; i < npts; ++i) {
    double z[3] = {0, 0, 0};
    for (int k = 0; k < p->d; ++k) z[k] = pts[i * p->d + k];
    out[i] = (double)interp_point(p, u, du.data(), z);
  }
  return 0;
}

// ---------------------------------------------------------------------------------------
// One application of the step operator to one field (Scheme 1 steps 1-3):
//   u_out(j) = sum_q w_q u_in^J(z_jq),  z_jq = x_j + b dt + sigma sqrt(2 dt) a_q  (Eq. 20-22)
// with the face rules R8/R9 for points outside the box.  Dirichlet nodes keep their value.
// b, sigma: [d][J].  a[k], w[k]: the per-dimension Gauss-Hermite rule.
// ---------------------------------------------------------------------------------------
static void apply_with_rule(const ofk_problem* p, const double* b, const double* sigma,
                            const double* const a[3], const double* const w[3],
                            const double* u_in, double* u_out, double* du_scratch) {
  const int d = p->d;
  long J = total_nodes(p);
  gradient_fields(p, u_in, du_scratch);
  const double sq = std::sqrt(2.0 * p->dt);
  long nq = 1;
  for (int k = 0; k < d; ++k) nq *= p->Q[k];
#pragma omp parallel for schedule(static)
  for (long j = 0; j < J; ++j) {
    int idx[3];
    unravel(p, j, idx);
    double g;
    if (dirichlet(p, idx, &g)) { u_out[j] = u_in[j]; continue; }
    long double acc = 0.0L;
    for (long qq = 0; qq < nq; ++qq) {
      int q[3];
      long r = qq;
      for (int k = d - 1; k >= 0; --k) { q[k] = (int)(r % p->Q[k]); r /= p->Q[k]; }
      long double wq = 1.0L;
      double z[3] = {0, 0, 0};
      for (int k = 0; k < d; ++k) {
        wq *= w[k][q[k]];
        double xk = p->x[k][idx[k]];
        double drift = b[(long)k * J + j] * p->dt;
        double spread = sigma[(long)k * J + j] * sq;
        z[k] = (xk + drift) + spread * a[k][q[k]];                  // Eq. 21
      }
      for (int k = 0; k < d; ++k) {                                 // R9: CLAMP faces first
        double lo = p->x[k][0], hi = p->x[k][p->n[k] - 1];
        if (p->face_kind[k][0] == OFK_PERIODIC) {                   // R21: wrap into [lo, hi)
          if (z[k] < lo || z[k] >= hi) {
            double L = hi - lo;
            double r = std::fmod(z[k] - lo, L);
            if (r < 0.0) r += L;
            z[k] = lo + r;
          }
          continue;
        }
        if (z[k] < lo && p->face_kind[k][0] == OFK_CLAMP) z[k] = lo;
        if (z[k] > hi && p->face_kind[k][1] == OFK_CLAMP) z[k] = hi;
      }
      bool outside = false;
      long double val = 0.0L;
      for (int k = 0; k < d && !outside; ++k) {                     // R8: lowest dimension decides
        double lo = p->x[k][0], hi = p->x[k][p->n[k] - 1];
        if (z[k] < lo) { outside = true; val = p->face_value[k][0]; }
        else if (z[k] > hi) { outside = true; val = p->face_value[k][1]; }
      }
      if (!outside) val = interp_point(p, u_in, du_scratch, z);
      acc += wq * val;
    }
    u_out[j] = (double)acc;
  }
}

struct Rule {
  std::vector<double> a[3], w[3];
  const double* ap[3];
  const double* wp[3];
  explicit Rule(const ofk_problem* p) {
    for (int k = 0; k < 3; ++k) { ap[k] = wp[k] = nullptr; }
    for (int k = 0; k < p->d; ++k) {
      a[k].resize(p->Q[k]);
      w[k].resize(p->Q[k]);
      ofk_gauss_hermite(p->Q[k], a[k].data(), w[k].data());
      ap[k] = a[k].data();
      wp[k] = w[k].data();
    }
  }
};

int ofk_apply(const ofk_problem* p, const double* b, const double* sigma, const double* u_in,
              double* u_out) {
  long J = total_nodes(p);
  Rule rule(p);
  std::vector<double> du((size_t)p->d * J);
  apply_with_rule(p, b, sigma, rule.ap, rule.wp, u_in, u_out, du.data());
  return 0;
}

// Eq. 29: column m = A_0 A_1 ... A_{m-1} chi.  b_tab, s_tab: [>=m][d][J]
// (operator nu uses slice nu; with `autonomous` != 0 slice 0 is used for every nu).
int ofk_column(const ofk_problem* p, const double* b_tab, const double* s_tab, int autonomous,
               int m, double* out) {
  long J = total_nodes(p);
  Rule rule(p);
  std::vector<double> u(J), v(J), du((size_t)p->d * J);
  ofk_chi(p, u.data());
  for (int nu = m - 1; nu >= 0; --nu) {
    long off = autonomous ? 0 : (long)nu * p->d * J;
    apply_with_rule(p, b_tab + off, s_tab + off, rule.ap, rule.wp, u.data(), v.data(), du.data());
    u.swap(v);
  }
  std::memcpy(out, u.data(), sizeof(double) * J);
  return 0;
}

// Algorithm 1.  P is [N+1][J] (column m = row m here), column 0 = chi.
//   P = repmat(chi); for n = N..1: P(:, n:N) = Q Psi^{n-1} F^{n-1} P(:, n:N).
int ofk_algorithm1(const ofk_problem* p, const double* b_tab, const double* s_tab, int autonomous,
                   int N, double* P) {
  long J = total_nodes(p);
  Rule rule(p);
  for (int m = 0; m <= N; ++m) ofk_chi(p, P + (long)m * J);
  for (int n = N; n >= 1; --n) {
    long off = autonomous ? 0 : (long)(n - 1) * p->d * J;
    // the columns n..N are independent: one thread per column when there are
    // several (the node loop inside then runs serially), node-parallel otherwise
#pragma omp parallel for schedule(dynamic, 1) if (N - n + 1 >= 4)
    for (int m = n; m <= N; ++m) {
      std::vector<double> v(J), du((size_t)p->d * J);
      double* col = P + (long)m * J;
      apply_with_rule(p, b_tab + off, s_tab + off, rule.ap, rule.wp, col, v.data(), du.data());
      std::memcpy(col, v.data(), sizeof(double) * J);
    }
  }
  return 0;
}

// sum_j w_j P(t_m, x_j) for M columns stored as P[M][J] (the exit probability
// for initial conditions distributed as P_init is int P(t,x) P_init(x) dx -- w_j = quadrature
// weight times P_init(x_j); Eq. 42: the same with w_j = 2 pi n_0 f_M(p_j) times the
// (xi, p) quadrature weights on the slice r = r_0).  Plain definition, long-double sum.
int ofk_reduce(long J, int M, const double* P, const double* w, double* out) {
  for (int m = 0; m < M; ++m) {
    long double s = 0.0L;
    for (long j = 0; j < J; ++j) s += (long double)w[j] * (long double)P[(long)m * J + j];
    out[m] = (double)s;
  }
  return 0;
}

void ofk_set_num_threads(int t) {
#ifdef _OPENMP
  if (t >= 1) omp_set_num_threads(t);
#else
  (void)t;
#endif
}

int ofk_num_threads(void) {
#ifdef _OPENMP
  return omp_get_max_threads();
#else
  return 1;
#endif
}

}  // extern "C"
