// fk_kernels.cu -- sm_100a kernels of the Feynman-Kac exit-time hot path (arXiv 2104.14561).
//
//   fk_fill_chi      Eq. 28 / Algorithm 1 "P = repmat(chi)"
//   fk_assemble      Scheme 1 step 1 + the quadrature fold: one row of A_nu = Q Psi^nu per
//                    node, in factored form (Eq. 21, 147 Eq. 14, 256-264)
//   fk_slopes        F: the PCHIP nodal slopes of Eq. 15 for every active column
//
//   fk_apply         P(:, n:N) <- A_nu [P; dP](:, n:N)
//   fk_gather        read-out of columns into [m][J] order
//
// Thread mapping of the two hot kernels: lane = output-time column inside a 32-column chunk,
// warp = one node.  Every P / dP access of a warp is one aligned 256-byte row whatever the
// shape of the stencil (scattered 1-D rows with Q = 16, clamped rows that reach across the
// whole box, ...), and the operator row is warp-uniform, so it is fetched by broadcast loads.
#include "fk_device.cuh"

#include <mutex>

namespace {

using fkd::unravel;
using fkd::dirichlet;
using fkd::locate;
using fkd::harmonic;

// ------------------------------------------------------------------------------------------
// chi into every lane of every chunk (also the padding columns beyond N)
// ------------------------------------------------------------------------------------------
__global__ void fk_fill_chi(FkGrid g, double* __restrict__ P, int n_chunks) {
  long long j = (long long)blockIdx.x * blockDim.y + threadIdx.y;
  if (j >= g.J) return;
  int idx[3];
  unravel(g, j, idx);
  double v;
  if (!dirichlet(g, idx, &v)) v = 0.0;
  for (int c = blockIdx.y; c < n_chunks; c += gridDim.y)
    P[((size_t)c * g.J + j) * FK_CW + threadIdx.x] = v;
}

// ------------------------------------------------------------------------------------------
// fk_assemble: one thread per node.  For each dimension k the Q_k points
//   z_q = (x + b dt) + (sigma sqrt(2 dt)) a_q          (Eq. 21; products and sums NOT fused,
//                                                       so cells agree with any fp64 reading)
// are visited in ascending order (sigma >= 0), so their cells are non-decreasing and the
// weights w_q * {Hermite basis of Eq. 14} can be merged onto distinct nodes with a two-entry
// window that is flushed to the row as it moves.  Points outside an ABSORB face add
// w_q * g to e_k; CLAMP faces project the point.  With m_k the inside mass of dimension k,
//   c_j = sum_k (prod_{l<k} m_l) e_k                   (lowest outside dimension decides, R9).
// In 2-D the row is also written as a compact record (FkRec2) when fkd::reach says that all
// its entries stay within FK_H nodes of the row's node: the weights of the 2*FK_H+1 nodes
// around it per dimension, zero where no point lands.
// ------------------------------------------------------------------------------------------
// returns prod_k D_k of the row (-1 for a Dirichlet row); *is_near: the row has a compact record
__device__ __forceinline__ int assemble_row(const FkGrid& g, const double* __restrict__ b,
                                                 const double* __restrict__ sigma,
                                                 const FkOperator& op, int* __restrict__ status,
                                                 long long j, bool* is_near) {
  *is_near = false;
  int idx[3];
  unravel(g, j, idx);
  int* cnt = op.cnt + j * 4;
  FkRec2* rec = op.rec ? op.rec + j : nullptr;
  double gval;
  if (dirichlet(g, idx, &gval)) {
    cnt[0] = cnt[1] = cnt[2] = 0;
    cnt[3] = FK_ROW_DIRICHLET;
    op.c[j] = gval;
    if (rec) {
      rec->c = gval;
      rec->mask[0] = rec->mask[1] = 0;
      rec->flags = FK_ROW_DIRICHLET;
      // the fused kernel multiplies every slot of the rows it owns: the weights of a Dirichlet
      // row must be zeros, not whatever the allocation held
      for (int k = 0; k < 2; ++k)
        for (int e = 0; e < FK_NW; ++e) rec->w[k][e] = make_double2(0.0, 0.0);
    }
    return -1;
  }
  double2* __restrict__ roww = op.w + (size_t)j * g.RS;
  int* __restrict__ rowo = op.off + (size_t)j * g.RS;
  double cj = 0.0, mass = 1.0;
  bool near = rec != nullptr;
  int bad = 0;
  for (int k = 0; k < g.d; ++k) {
    const double xk = g.x[k][idx[k]];
    const double bk = b[(size_t)k * g.J + j], sk = sigma[(size_t)k * g.J + j];
    if (sk < 0.0) bad |= FK_BAD_NEG_SIGMA;
    if (g.validate && !(isfinite(bk) && isfinite(sk))) bad |= FK_BAD_NONFINITE;
    const double centre = __dadd_rn(xk, __dmul_rn(bk, g.dt));
    const double spread = __dmul_rn(sk, g.sq);
    const double lo = g.lo[k], hi = g.hi[k];
    const long long unit = g.stride[k] * FK_CW;
    bool rec_k = false;
    int rmask = 0;
    const int rbase = idx[k] - FK_H;         // node of slot 0 of the record
    if (rec) {
      int first, last;
      fkd::reach(g, k, centre, spread, &first, &last);
      rec_k = first >= rbase && last <= idx[k] + FK_H && idx[0] >= g.near_lo && idx[0] < g.near_hi;
      near = near && rec_k;
      if (rec_k)
        for (int e = 0; e < FK_NW; ++e) rec->w[k][e] = make_double2(0.0, 0.0);
    }
    double ek = 0.0, mk = 0.0;
    int count = 0;
    int cprev = -2;
    double aL = 0.0, bL = 0.0, aR = 0.0, bR = 0.0;
    double2* wk = roww + g.qoff[k];
    int* ok = rowo + g.qoff[k];
#define FK_EMIT(node, A, B)                                               \
    if ((A) != 0.0 || (B) != 0.0) {   /* exact zeros (a point on a node) are not entries */ \
      wk[count] = make_double2((A), (B));                                 \
      ok[count] = (int)((node) * unit);                                   \
      ++count;                                                            \
      if (rec_k) {                                                        \
        rec->w[k][(node) - rbase] = make_double2((A), (B));               \
        rmask |= 1 << ((node) - rbase);                                   \
      }                                                                   \
    }
    for (int q = 0; q < g.Q[k]; ++q) {
      double z = fkd::push_point(centre, spread, g.gh_a[k][q]);
      const double w = g.gh_w[k][q];
      if (g.periodic[k]) {                       // R21: wrap into [lo, hi)
        if (z < lo || z >= hi) {
          const double L = hi - lo;
          double r = fmod(z - lo, L);
          if (r < 0.0) r += L;
          z = lo + r;
        }
      } else if (z < lo) {
        if (g.face_kind[k][0] == 1) z = lo; else { ek += w * g.face_value[k][0]; continue; }
      } else if (z > hi) {
        if (g.face_kind[k][1] == 1) z = hi; else { ek += w * g.face_value[k][1]; continue; }
      }
      mk += w;
      const int c = locate(g, k, z);
      const double h = g.x[k][c + 1] - g.x[k][c];
      const double t = (z - g.x[k][c]) * g.inv_h[k][c];
      const double u = 1.0 - t;
      // Eq. 14 with t = s/h: value-left (1+2t)(1-t)^2, value-right t^2(3-2t),
      // slope-left h t(1-t)^2, slope-right h t^2(t-1)
      const double vL = w * ((1.0 + 2.0 * t) * u * u);
      const double vR = w * (t * t * (3.0 - 2.0 * t));
      const double sL = w * (h * t * u * u);
      const double sR = w * (h * t * t * (t - 1.0));
      if (c == cprev) {
        aL += vL; bL += sL; aR += vR; bR += sR;
      } else if (c == cprev + 1) {
        FK_EMIT(cprev, aL, bL);
        aL = aR + vL; bL = bR + sL; aR = vR; bR = sR;
        cprev = c;
      } else {
        if (cprev >= 0) {
          FK_EMIT(cprev, aL, bL);
          FK_EMIT(cprev + 1, aR, bR);
        }
        aL = vL; bL = sL; aR = vR; bR = sR;
        cprev = c;
      }
    }
    if (cprev >= 0) {
      FK_EMIT(cprev, aL, bL);
      FK_EMIT(cprev + 1, aR, bR);
    }
#undef FK_EMIT
    cnt[k] = count;
    if (rec) rec->mask[k] = rmask;
    cj += mass * ek;
    mass *= mk;
  }
  if (bad) atomicOr(status, bad);
  for (int k = g.d; k < 3; ++k) cnt[k] = 0;
  // 2-D: first and last dimension-1 node of the row, packed into the unused third count (1 + first
  // in the low half, last in the high half; 0 = not recorded), so that fk_far2d knows a group's
  // union window from the counts alone
  if (g.d == 2 && cnt[1] > 0 && g.n[1] < 65535)          // both halves < 2^16; packed and unpacked unsigned
    cnt[2] = (int)((unsigned)(1 + rowo[g.qoff[1]] / FK_CW) |
                   ((unsigned)(rowo[g.qoff[1] + cnt[1] - 1] / FK_CW) << 16));
  cnt[3] = near ? FK_ROW_NEAR : 0;
  op.c[j] = cj;
  if (rec) {
    rec->c = cj;
    // the masks ride in the flag word (bits 8-15 / 16-23): the fused kernel fetches c, flags and
    // masks of a row with one 16-byte load
    rec->flags = (near ? FK_ROW_NEAR : 0) | (rec->mask[0] << 8) | (rec->mask[1] << 16);
  }
  *is_near = near;
  int prod = 1;
  for (int k = 0; k < g.d; ++k) prod *= cnt[k];
  return prod;
}

// work[0..3] += {updated rows with a compact record, their sum of prod_k D_k, the other updated
// rows, their sum of prod_k D_k}: the algorithmic size of A_nu (one set of atomics per warp)
__global__ void fk_assemble(FkGrid g, const double* __restrict__ b,
                            const double* __restrict__ sigma, FkOperator op,
                            int* __restrict__ status, unsigned long long* __restrict__ work) {
  const long long j = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  bool near = false;
  const int prod = j < g.J ? assemble_row(g, b, sigma, op, status, j, &near) : -1;
  const bool live = prod >= 0;                            // an updated (non-Dirichlet) row
  const unsigned near_rows = __reduce_add_sync(0xffffffffu, (live && near) ? 1u : 0u);
  const unsigned far_rows = __reduce_add_sync(0xffffffffu, (live && !near) ? 1u : 0u);
  const unsigned near_nnz = __reduce_add_sync(0xffffffffu, (live && near) ? (unsigned)prod : 0u);
  const unsigned far_nnz = __reduce_add_sync(0xffffffffu, (live && !near) ? (unsigned)prod : 0u);
  if ((threadIdx.x & 31) == 0) {
    if (near_rows) { atomicAdd(work, (unsigned long long)near_rows); atomicAdd(work + 1, (unsigned long long)near_nnz); }
    if (far_rows) { atomicAdd(work + 2, (unsigned long long)far_rows); atomicAdd(work + 3, (unsigned long long)far_nnz); }
  }
}

// fk_assemble_batch: the operators of `count` consecutive steps nu = nu_hi, nu_hi-1, ... in one
// launch (grid.y walks the steps), operator s of the batch stored at `op` + s * (its size): what
// fk_line1d consumes.  An autonomous problem has count = 1 and the one coefficient slice.
__global__ void fk_assemble_batch(FkGrid g, const double* __restrict__ coef, int slots, int nu_hi,
                                  int count, int autonomous, FkOperator op,
                                  int* __restrict__ status, unsigned long long* __restrict__ work) {
  const size_t slice = (size_t)g.d * g.J;
  const long long j = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  for (int s = blockIdx.y; s < count; s += gridDim.y) {
    const int nu = nu_hi - s;
    const double* __restrict__ b = coef + (size_t)(autonomous ? 0 : nu % slots) * 2 * slice;
    FkOperator o;
    o.w = op.w + (size_t)s * g.J * g.RS;
    o.off = op.off + (size_t)s * g.J * g.RS;
    o.cnt = op.cnt + (size_t)s * g.J * 4;
    o.c = op.c + (size_t)s * g.J;
    o.rec = nullptr;
    bool near = false;
    const int prod = j < g.J ? assemble_row(g, b, b + slice, o, status, j, &near) : -1;
    const bool live = prod >= 0;
    const unsigned rows = __reduce_add_sync(0xffffffffu, live ? 1u : 0u);
    const unsigned nnz = __reduce_add_sync(0xffffffffu, live ? (unsigned)prod : 0u);
    if ((threadIdx.x & 31) == 0 && rows) {
      atomicAdd(work + 4 * (size_t)nu + 2, (unsigned long long)rows);
      atomicAdd(work + 4 * (size_t)nu + 3, (unsigned long long)nnz);
    }
  }
}

// ------------------------------------------------------------------------------------------
// fk_classify (2-D): how many rows of each loaded step are not FK_ROW_NEAR, by the same
// fkd::reach test fk_assemble applies.  grid = (node blocks, min(steps, 4096)).
// ------------------------------------------------------------------------------------------
__global__ void fk_classify(FkGrid g, const double* __restrict__ coef, int slots, int step0,
                            int count, int* __restrict__ far_rows, int* __restrict__ far_line) {
  const size_t slice = (size_t)g.d * g.J;
  const long long j = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  int idx[3] = {0, 0, 0};
  double gval;
  const bool updated = j < g.J && (unravel(g, j, idx), !dirichlet(g, idx, &gval));
  for (int s = blockIdx.y; s < count; s += gridDim.y) {      // any number of steps per launch
    const int slot = (step0 + s) % slots;
    const double* __restrict__ b = coef + (size_t)slot * 2 * slice;
    const double* __restrict__ sigma = b + slice;
    bool far = false;
    int first0 = 0, last0 = 0;
    if (updated) {
      for (int k = 0; k < g.d; ++k) {
        const double centre = __dadd_rn(g.x[k][idx[k]], __dmul_rn(b[(size_t)k * g.J + j], g.dt));
        const double spread = __dmul_rn(sigma[(size_t)k * g.J + j], g.sq);
        int first, last;
        fkd::reach(g, k, centre, spread, &first, &last);
        far = far || !(first >= idx[k] - FK_H && last <= idx[k] + FK_H);
        if (k == 0) { first0 = first; last0 = last; }
      }
    }
    int* __restrict__ f = far_rows + slot * FK_FAR_STRIDE;
    if (far) atomicAdd(far_line + (size_t)slot * g.n[0] + idx[0], 1);   // far rows per line
    const unsigned m = __ballot_sync(0xffffffffu, far);
    if (m) {                                  // one set of atomics per warp that holds far rows
      const int a1 = __reduce_max_sync(0xffffffffu, far ? FK_FAR_BIG - idx[0] : 0);
      const int a2 = __reduce_max_sync(0xffffffffu, far ? idx[0] + 1 : 0);
      const int a3 = __reduce_max_sync(0xffffffffu, far ? FK_FAR_BIG - first0 : 0);
      const int a4 = __reduce_max_sync(0xffffffffu, far ? last0 + 1 : 0);
      if ((threadIdx.x & 31) == 0) {
        atomicAdd(f, __popc(m));
        atomicMax(f + 1, a1);                 // lines holding far rows, lines their entries touch
        atomicMax(f + 2, a2);
        atomicMax(f + 3, a3);
        atomicMax(f + 4, a4);
      }
    }
  }
}

// ------------------------------------------------------------------------------------------
// fk_slopes<D>: dP_k(j) of Eq. 15 from the grid line of axis k through j, for every node of the
// lines line0 .. line0+nlines-1 (a "line" = one run of the fastest dimension; its index runs over
// the other dimensions) and every active chunk.  Block (32, 8): lane = column; a warp takes a
// run of SR consecutive nodes of one line.  The fastest-dimension slopes come from the SR + 3
// values around the run held in registers (one load per node); each other dimension needs the
// two neighbours across lines.  End nodes use the first / last two divided differences (R6,
// PAPER.md:160): with la = clamp(i-1, 0, n-3) the three nodes la, la+1, la+2 give both cases.
// ------------------------------------------------------------------------------------------
constexpr int SR = 4;                 // nodes per warp; with 6 blocks per SM: measured best on config 5

// The three nodes (a, b, c) whose two divided differences give the slope at node i of a line of
// n nodes, and the cells ca (between a and b) and cb (between b and c): the node and its
// neighbours inside; the first / last three nodes at the ends (R6); across the seam when the
// dimension is periodic (R21: node n-1 is the image of node 0).
struct SlopeWindow { int a, b, c, ca, cb; };
__device__ __forceinline__ SlopeWindow slope_window(int i, int n, int periodic) {
  SlopeWindow w;
  if (periodic) {
    w.b = i;
    w.a = i == 0 ? n - 2 : i - 1;
    w.c = i == n - 1 ? 1 : i + 1;
    w.ca = i == 0 ? n - 2 : i - 1;
    w.cb = i == n - 1 ? 0 : i;
  } else {
    const int la = min(max(i - 1, 0), n - 3);
    w.a = la; w.b = la + 1; w.c = la + 2; w.ca = la; w.cb = la + 1;
  }
  return w;
}

// General slopes of one run (periodic dimensions and / or the weighted mean of R22): node by
// node, three loads per dimension.  The streamlined code in fk_slopes covers everything else.
template <int D>
__device__ __forceinline__ void slopes_general(const FkGrid& g, const double* __restrict__ u,
                                               double* __restrict__ o, size_t field, int line,
                                               int i0) {
  const int nl = g.n[D - 1];
  int idx[3] = {0, 0, 0};
  if (D == 2) idx[0] = line;
  if (D == 3) { idx[0] = line / g.n[1]; idx[1] = line - idx[0] * g.n[1]; }
  for (int q = 0; q < SR; ++q) {
    const int i = i0 + q;
    if (i >= nl) break;
    idx[D - 1] = i;
    const double* __restrict__ un = u + i * FK_CW;
#pragma unroll
    for (int k = 0; k < D; ++k) {
      const int s = (int)g.stride[k] * FK_CW;
      const SlopeWindow w = slope_window(idx[k], g.n[k], g.periodic[k]);
      const double va = un[(w.a - idx[k]) * s], vb = un[(w.b - idx[k]) * s], vc = un[(w.c - idx[k]) * s];
      const double da = (vb - va) * g.inv_h[k][w.ca], db = (vc - vb) * g.inv_h[k][w.cb];
      o[(size_t)k * field + i * FK_CW] = g.weighted ? fkd::harmonic_w(da, db, g.wgt[k][idx[k]])
                                                    : harmonic(da, db);
    }
  }
}

template <int D>
__global__ void __launch_bounds__(256, 6)
fk_slopes(FkGrid g, const double* __restrict__ P, double* __restrict__ dP, int n_chunks,
          int chunk0, int line0, int nlines) {
  const int nl = g.n[D - 1];
  const int segs = (nl + SR - 1) / SR;
  const int rid = blockIdx.x * 8 + threadIdx.y;
  if (rid >= nlines * segs) return;
  const int line = line0 + rid / segs;
  const int i0 = (rid - (rid / segs) * segs) * SR;
  const int c = chunk0 + blockIdx.y;
  const size_t chunk_elems = (size_t)g.J * FK_CW;
  const int node0 = line * nl;                                   // node (line, 0)
  const double* __restrict__ u = P + (size_t)c * chunk_elems + (size_t)node0 * FK_CW + threadIdx.x;
  double* __restrict__ o = dP + (size_t)c * chunk_elems + (size_t)node0 * FK_CW + threadIdx.x;
  const size_t field = (size_t)n_chunks * chunk_elems;

  if (g.general_slopes) {                       // periodic dimensions and / or weighted means
    slopes_general<D>(g, u, o, field, line, i0);
    return;
  }
  // A run whose nodes and their +-1 neighbours are all inside the grid in every dimension (no
  // first / last node of any line: no end rule, no clamp) takes straight-line code.
  {
    bool inner = i0 >= 1 && i0 + SR <= nl - 1;
    int idx[2] = {0, 0};
    if (D == 2) idx[0] = line;
    if (D == 3) { idx[0] = line / g.n[1]; idx[1] = line - idx[0] * g.n[1]; }
#pragma unroll
    for (int k = 0; k < D - 1; ++k) inner = inner && idx[k] >= 1 && idx[k] <= g.n[k] - 2;
    if (inner) {
      double w[SR + 2];                                          // nodes i0-1 .. i0+SR
#pragma unroll
      for (int k = 0; k < SR + 2; ++k) w[k] = u[(i0 - 1 + k) * FK_CW];
      const double* __restrict__ ih = g.inv_h[D - 1] + (i0 - 1);
      double dl[SR + 1];                                         // dl[k]: cell right of node i0-1+k
#pragma unroll
      for (int k = 0; k < SR + 1; ++k) dl[k] = (w[k + 1] - w[k]) * ih[k];
      double* __restrict__ ok = o + (size_t)(D - 1) * field + i0 * FK_CW;
#pragma unroll
      for (int k = 0; k < SR; ++k) ok[k * FK_CW] = harmonic(dl[k], dl[k + 1]);
#pragma unroll
      for (int k = 0; k < D - 1; ++k) {
        const int s = (int)g.stride[k] * FK_CW;
        const double iha = g.inv_h[k][idx[k] - 1], ihb = g.inv_h[k][idx[k]];
        const double* __restrict__ un = u + i0 * FK_CW;
        double* __restrict__ okk = o + (size_t)k * field + i0 * FK_CW;
#pragma unroll
        for (int q = 0; q < SR; ++q) {
          const double va = un[q * FK_CW - s], vc = un[q * FK_CW + s], vb = w[q + 1];
          okk[q * FK_CW] = harmonic((vb - va) * iha, (vc - vb) * ihb);
        }
      }
      return;
    }
  }
  // values of the line at nodes i0-2 .. i0+SR (clamped; clamped duplicates are never selected)
  double v[SR + 3];
#pragma unroll
  for (int k = 0; k < SR + 3; ++k) v[k] = u[min(max(i0 - 2 + k, 0), nl - 1) * FK_CW];
  {
    const double* __restrict__ ih = g.inv_h[D - 1];
    double dl[SR + 2];                                           // dl[k]: cell right of node i0-2+k
#pragma unroll
    for (int k = 0; k < SR + 2; ++k) dl[k] = (v[k + 1] - v[k]) * ih[min(max(i0 - 2 + k, 0), nl - 2)];
    double* __restrict__ ok = o + (size_t)(D - 1) * field;
#pragma unroll
    for (int k = 0; k < SR; ++k) {
      const int i = i0 + k;
      if (i < nl) {
        const double a = i == 0 ? dl[2] : (i == nl - 1 ? dl[k] : dl[k + 1]);
        const double b = i == 0 ? dl[3] : (i == nl - 1 ? dl[k + 1] : dl[k + 2]);
        ok[i * FK_CW] = harmonic(a, b);
      }
    }
  }
  if (D >= 2) {
    int idx[2];
    idx[0] = D == 3 ? line / g.n[1] : line;
    idx[1] = D == 3 ? line - idx[0] * g.n[1] : 0;
#pragma unroll
    for (int k = 0; k < D - 1; ++k) {
      const int nk = g.n[k], ik = idx[k];
      const int la = min(max(ik - 1, 0), nk - 3);
      const int s = (int)g.stride[k] * FK_CW;
      const int oa = (la - ik) * s, ob = oa + s, oc = ob + s;    // one of them may be 0 (the node)
      const double iha = g.inv_h[k][la], ihb = g.inv_h[k][la + 1];
      double* __restrict__ ok = o + (size_t)k * field;
#pragma unroll
      for (int q = 0; q < SR; ++q) {
        const int i = i0 + q;
        if (i < nl) {
          const double* __restrict__ un = u + i * FK_CW;
          const double va = oa == 0 ? v[q + 2] : un[oa];
          const double vb = ob == 0 ? v[q + 2] : un[ob];
          const double vc = oc == 0 ? v[q + 2] : un[oc];
          ok[i * FK_CW] = harmonic((vb - va) * iha, (vc - vb) * ihb);
        }
      }
    }
  }
}

// ------------------------------------------------------------------------------------------
// fk_apply<D>: block (32, 8), lane = column, threadIdx.y = node; grid.y = active chunks.
//   out = c_j + sum_{i0} [ alpha0 A'(i0) + beta0 B0'(i0) ]
//   A'(i0)  = sum_{i1} [ alpha1 A(i0,i1) + beta1 B1(i0,i1) ],  B0'(i0) = sum_{i1} alpha1 B0(i0,i1)
//   A(i0,i1)  = sum_{i2} [ alpha2 u + beta2 du2 ],  Bk(i0,i1) = sum_{i2} alpha2 du_k
// i.e. Eq. 13 with the quadrature weights folded in, contracted one dimension at a time.
// Lanes whose column is not active (m < n: still chi; m > N: padding) compute and discard.
// ------------------------------------------------------------------------------------------
template <int D>
__global__ void __launch_bounds__(256)
fk_apply(FkGrid g, FkOperator op, const double* __restrict__ Pold,
         const double* __restrict__ dP, double* __restrict__ Pnew, int n_chunks, int chunk0,
         int n, int N, int far_only, long long j0, long long jn) {
  long long j = (long long)blockIdx.x * blockDim.y + threadIdx.y;
  if (j >= jn) return;
  j += j0;
  const int c = chunk0 + blockIdx.y;
  const int m = fkd::column_of(g, c, threadIdx.x);
  const size_t chunk_elems = (size_t)g.J * FK_CW;
  const double* __restrict__ u = Pold + (size_t)c * chunk_elems + threadIdx.x;
  const double* __restrict__ d0 = dP + (size_t)c * chunk_elems + threadIdx.x;
  const double* __restrict__ d1 = d0 + (size_t)n_chunks * chunk_elems;
  const double* __restrict__ d2 = d1 + (size_t)n_chunks * chunk_elems;
  const double2* __restrict__ w = op.w + (size_t)j * g.RS;
  const int* __restrict__ off = op.off + (size_t)j * g.RS;
  const int4 cnt = *reinterpret_cast<const int4*>(op.cnt + j * 4);
  if (far_only && (cnt.w & (FK_ROW_NEAR | FK_ROW_DIRICHLET))) return;   // done by fk_fused2d
  const double acc = fkd::contract_row<D>(g, w, off, cnt, op.c[j], u, d0, d1, d2);
  if (m >= n && m <= N) Pnew[(size_t)c * chunk_elems + (size_t)j * FK_CW + threadIdx.x] = acc;
}

// ------------------------------------------------------------------------------------------
// fk_gather: out[m - m0][j] = P[m / 32][j][m % 32]; 32 x 32 transpose through shared memory
// so that both sides are coalesced.  grid = (node tiles, chunks touched by [m0, m1)).
// ------------------------------------------------------------------------------------------
__global__ void fk_gather(FkGrid g, const double* __restrict__ P, int m0, int m1,
                          double* __restrict__ out) {
  __shared__ double tile[32][33];
  const int cg = m0 / FK_CW + blockIdx.y;                 // global chunk
  if (cg % g.shard_count != g.shard_index) return;        // not this shard's: `out` is left alone
  const int c = cg / g.shard_count;                        // local chunk
  const long long j0 = (long long)blockIdx.x * 32;
  for (int r = threadIdx.y; r < 32; r += blockDim.y) {
    long long j = j0 + r;
    if (j < g.J) tile[r][threadIdx.x] = P[((size_t)c * g.J + j) * FK_CW + threadIdx.x];
  }
  __syncthreads();
  for (int r = threadIdx.y; r < 32; r += blockDim.y) {
    const int m = cg * FK_CW + r;
    long long j = j0 + threadIdx.x;
    if (m >= m0 && m < m1 && j < g.J) out[(size_t)(m - m0) * g.J + j] = tile[threadIdx.x][r];
  }
}

// ------------------------------------------------------------------------------------------
// fk_reduce_partial / fk_reduce_final: out[m - m0] = sum_j w_j P(t_m, x_j)
// in two passes with a fixed summation order.  Pass 1: grid (FK_RED_BLOCKS, chunks touched),
// block (32, 8): warp y of block b sums the nodes j = (b*8 + y) + k * (8*FK_RED_BLOCKS),
// k = 0, 1, ...; the 8 warps are combined in order.  Pass 2: one warp per chunk adds the
// FK_RED_BLOCKS partial sums in order.
// ------------------------------------------------------------------------------------------
__global__ void fk_reduce_partial(FkGrid g, const double* __restrict__ P,
                                  const double* __restrict__ w, int chunk_first,
                                  double* __restrict__ partial) {
  __shared__ double sm[8][32];
  const int cg = chunk_first + blockIdx.y;
  if (cg % g.shard_count != g.shard_index) return;
  const int c = cg / g.shard_count;
  const double* __restrict__ Pc = P + (size_t)c * g.J * FK_CW + threadIdx.x;
  double acc = 0.0;
  for (long long j = (long long)blockIdx.x * 8 + threadIdx.y; j < g.J; j += 8LL * FK_RED_BLOCKS)
    acc = fma(w[j], Pc[j * FK_CW], acc);
  sm[threadIdx.y][threadIdx.x] = acc;
  __syncthreads();
  if (threadIdx.y == 0) {
    double s = 0.0;
    for (int y = 0; y < 8; ++y) s += sm[y][threadIdx.x];
    partial[((size_t)blockIdx.y * FK_RED_BLOCKS + blockIdx.x) * FK_CW + threadIdx.x] = s;
  }
}

__global__ void fk_reduce_final(FkGrid g, const double* __restrict__ partial, int chunk_first,
                                int m0, int m1, double* __restrict__ out) {
  const int cg = chunk_first + blockIdx.x;
  if (cg % g.shard_count != g.shard_index) return;
  const int m = cg * FK_CW + threadIdx.x;
  double s = 0.0;
  for (int b = 0; b < FK_RED_BLOCKS; ++b)
    s += partial[((size_t)blockIdx.x * FK_RED_BLOCKS + b) * FK_CW + threadIdx.x];
  if (m >= m0 && m < m1) out[m - m0] = s;
}

}  // namespace

// ------------------------------------------------------------------------------------------
// launchers
// ------------------------------------------------------------------------------------------
static inline unsigned node_blocks(const FkGrid& g, int per_block) {
  return (unsigned)((g.J + per_block - 1) / per_block);
}

cudaError_t fk_launch_fill_chi(const FkGrid& g, double* P, int n_chunks, cudaStream_t s) {
  dim3 block(FK_CW, 8), grid(node_blocks(g, 8), (unsigned)(n_chunks < 64 ? n_chunks : 64));
  fk_fill_chi<<<grid, block, 0, s>>>(g, P, n_chunks);
  return cudaGetLastError();
}

cudaError_t fk_launch_assemble(const FkGrid& g, const double* b, const double* sigma,
                               FkOperator op, int* status, unsigned long long* work,
                               cudaStream_t s) {
  fk_assemble<<<node_blocks(g, 128), 128, 0, s>>>(g, b, sigma, op, status, work);
  return cudaGetLastError();
}

cudaError_t fk_launch_assemble_batch(const FkGrid& g, const double* coef, int slots, int nu_hi,
                                     int count, int autonomous, FkOperator op, int* status,
                                     unsigned long long* work, cudaStream_t s) {
  dim3 grid(node_blocks(g, 128), (unsigned)(count < 1024 ? count : 1024));
  fk_assemble_batch<<<grid, 128, 0, s>>>(g, coef, slots, nu_hi, count, autonomous, op, status, work);
  return cudaGetLastError();
}

cudaError_t fk_launch_classify(const FkGrid& g, const double* coef, int slots, int step0,
                               int count, int* far_rows, int* far_line, cudaStream_t s) {
  dim3 grid(node_blocks(g, 128), (unsigned)(count < 4096 ? count : 4096));
  fk_classify<<<grid, 128, 0, s>>>(g, coef, slots, step0, count, far_rows, far_line);
  return cudaGetLastError();
}

cudaError_t fk_launch_slopes(const FkGrid& g, const double* P, double* dP, int n_chunks,
                             int chunk0, int chunk1, int line0, int nlines, cudaStream_t s) {
  const int segs = (g.n[g.d - 1] + SR - 1) / SR;
  dim3 block(FK_CW, 8), grid((unsigned)(((long long)nlines * segs + 7) / 8), (unsigned)(chunk1 - chunk0));
  if (g.d == 1) fk_slopes<1><<<grid, block, 0, s>>>(g, P, dP, n_chunks, chunk0, line0, nlines);
  else if (g.d == 2) fk_slopes<2><<<grid, block, 0, s>>>(g, P, dP, n_chunks, chunk0, line0, nlines);
  else fk_slopes<3><<<grid, block, 0, s>>>(g, P, dP, n_chunks, chunk0, line0, nlines);
  return cudaGetLastError();
}

cudaError_t fk_launch_apply(const FkGrid& g, FkOperator op, const double* Pold, const double* dP,
                            double* Pnew, int n_chunks, int chunk0, int chunk1, int n, int N,
                            int far_only, long long j0, long long jn, cudaStream_t s) {
  dim3 block(FK_CW, 8), grid((unsigned)((jn + 7) / 8), (unsigned)(chunk1 - chunk0));
  if (g.d == 1)
    fk_apply<1><<<grid, block, 0, s>>>(g, op, Pold, dP, Pnew, n_chunks, chunk0, n, N, far_only, j0, jn);
  else if (g.d == 2)
    fk_apply<2><<<grid, block, 0, s>>>(g, op, Pold, dP, Pnew, n_chunks, chunk0, n, N, far_only, j0, jn);
  else
    fk_apply<3><<<grid, block, 0, s>>>(g, op, Pold, dP, Pnew, n_chunks, chunk0, n, N, far_only, j0, jn);
  return cudaGetLastError();
}

cudaError_t fk_launch_reduce(const FkGrid& g, const double* P, const double* w, int m0, int m1,
                             double* partial, double* out, cudaStream_t s) {
  const int c0 = m0 / FK_CW, c1 = (m1 - 1) / FK_CW + 1;
  dim3 block(32, 8), grid(FK_RED_BLOCKS, (unsigned)(c1 - c0));
  fk_reduce_partial<<<grid, block, 0, s>>>(g, P, w, c0, partial);
  cudaError_t e = cudaGetLastError();
  if (e != cudaSuccess) return e;
  fk_reduce_final<<<(unsigned)(c1 - c0), 32, 0, s>>>(g, partial, c0, m0, m1, out);
  return cudaGetLastError();
}

// ------------------------------------------------------------------------------------------
// fk_reduce_static (include/fk.h): the same two passes as fk_launch_reduce, with the partial sums of
// pass 1 kept in a fixed array that is part of the library image instead of in a buffer from
// cudaMalloc.  FK_REDUCE_STATIC_MAX_CHUNKS x FK_RED_BLOCKS x 32 doubles = 1 MiB, held by every GPU
// that loads the library until the process exits.
//
// In HOST code the name `fk_reduce_static_scratch` is only a handle for the runtime, not a device
// address, so it must never be handed to a kernel as it is: the address the kernels get comes from
// cudaGetSymbolAddress, asked once per device with that device current (every device has its own
// copy of the array at its own address) and remembered here.
//
// Nothing in the array has to start at zero: pass 2 reads exactly the slots pass 1 of the same
// call wrote (a shard skips both passes for the chunks it does not own), so whatever an earlier
// call left behind is never looked at.
// ------------------------------------------------------------------------------------------
static __device__ __align__(256) double
    fk_reduce_static_scratch[(size_t)FK_REDUCE_STATIC_MAX_CHUNKS * FK_RED_BLOCKS * FK_CW];

#define FK_STATIC_MAX_DEVICES 64
static std::mutex g_static_mutex;
static double* g_static_scratch_ptr[FK_STATIC_MAX_DEVICES];   // per device ordinal, NULL = not asked yet

cudaError_t fk_launch_reduce_static(const FkGrid& g, const double* P, const double* w, int m0,
                                    int m1, double* out, int device, cudaStream_t s) {
  const int c0 = m0 / FK_CW, c1 = (m1 - 1) / FK_CW + 1;
  if (c1 - c0 > FK_REDUCE_STATIC_MAX_CHUNKS || device < 0 || device >= FK_STATIC_MAX_DEVICES)
    return cudaErrorInvalidValue;
  int cur = -1;
  cudaError_t e = cudaGetDevice(&cur);
  if (e != cudaSuccess) return e;
  if (cur != device) return cudaErrorInvalidDevice;          // the caller makes `device` current
  double* partial = nullptr;
  {
    std::lock_guard<std::mutex> lock(g_static_mutex);
    if (!g_static_scratch_ptr[device]) {                     // set-up: first call on this device
      void* ptr = nullptr;
      e = cudaGetSymbolAddress(&ptr, fk_reduce_static_scratch);
      if (e != cudaSuccess) return e;
      if (!ptr) return cudaErrorInvalidSymbol;
      g_static_scratch_ptr[device] = static_cast<double*>(ptr);
    }
    partial = g_static_scratch_ptr[device];
  }
  dim3 block(32, 8), grid(FK_RED_BLOCKS, (unsigned)(c1 - c0));
  fk_reduce_partial<<<grid, block, 0, s>>>(g, P, w, c0, partial);
  e = cudaGetLastError();
  if (e != cudaSuccess) return e;
  fk_reduce_final<<<(unsigned)(c1 - c0), 32, 0, s>>>(g, partial, c0, m0, m1, out);
  return cudaGetLastError();
}

cudaError_t fk_launch_gather_columns(const FkGrid& g, const double* P, int m0, int m1,
                                     double* out, cudaStream_t s) {
  const int c0 = m0 / FK_CW, c1 = (m1 - 1) / FK_CW + 1;
  dim3 block(32, 8), grid(node_blocks(g, 32), (unsigned)(c1 - c0));
  fk_gather<<<grid, block, 0, s>>>(g, P, m0, m1, out);
  return cudaGetLastError();
}
