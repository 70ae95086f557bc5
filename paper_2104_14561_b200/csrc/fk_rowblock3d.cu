// fk_rowblock3d.cu -- the 3-D apply kernel: P(:, n:N) <- A_nu [P; dP](:, n:N) with
// the rows of A_nu taken FOUR AT A TIME.
//
// Lane = output-time column of a 32-column chunk, as everywhere in this library; a warp owns a
// group of RB = 4 rows that are adjacent along the fastest dimension (dimension 2).  In the
// factored row (fk_internal.h) the weights of dimension 0 and 1 multiply whole dimension-2 runs,
//     out_r = c_r + sum_{e0, e1} [ a0 a1 (A_r + A2_r) + a0 b1 B1_r + b0 a1 B0_r ],
//     A_r = sum_t alpha2_r(t) u(e0, e1, i2_r + t), ...  (fkd::contract_row),
// so when the four rows put their dimension-0 and dimension-1 entries on the SAME nodes (drift and
// diffusion vary slowly along dimension 2: the usual case) the four inner sums read the same
// run of RB + 2H nodes: every u / dP value is loaded once per group and feeds up to RB rows,
// with the dimension-2 weights in registers at static indices (slot t of row r is union node
// q = r + t, as in the fused 2-D kernel).  The kernel body is instantiated for the slot ranges
// that occur (own node only -- where the dimension-2 motion vanishes a group reads 4 nodes --,
// +-1, ..., all 2H+1), chosen per group by a warp-uniform test.
// Groups whose rows disagree (a quadrature point of one row falls into the next cell) are
// contracted on the union of the rows' entry lists (zero weights where a row has no entry);
// groups that reach beyond H nodes along dimension 2 or need more than EMAX entries in
// dimension 0 or 1 take the row-at-a-time path (fkd::contract_row) inside the same kernel.
//
// What bounds it (profiles/r2_cfg5_kernels_ncu_full.md): a node is 1 KB here (4 fields x 32
// columns), so the L1 holds ~190 nodes and about half of the loads miss it; the L2 -> SM traffic
// that results (~8 GB per chunk launch at ~4.5 TB/s) is the limiter, not DRAM, fp64 or issue.
// One staging serves CPB = 2 chunks, and each group pulls its own rows of the plane L2PF steps
// ahead into L2 with a bulk prefetch, so the misses are at least L2 hits.
//
// u and dP come from global memory through L1: a block is 4 warps = the same dimension-2 group of
// 4 consecutive dimension-1 lines, whose dimension-0 / dimension-1 nodes largely coincide.
#include <climits>

#include "fk_device.cuh"

namespace {

constexpr int RB = 4;                      // rows per warp
constexpr int H2 = FK_H;                   // dimension-2 halo of the blocked path
constexpr int NS = 2 * H2 + 1;             // slots per row along dimension 2
constexpr int EMAX = 16;                   // entries per row in dimension 0 / 1 (blocked path)
constexpr int WARPS = 4;                   // a block = the same dimension-2 group of 4 dimension-1 lines
constexpr int MINB = 3;                    // blocks per SM the register budget is set for
constexpr int CPB = 2;                     // chunks served by one staging of a group's rows
constexpr int L2PF = 3;                    // planes ahead whose rows a group pulls into L2
constexpr int WMAX2 = 32;                  // widest dimension-2 union window of the banded path (nodes)

struct GroupStage {                        // per warp, shared memory
  double2 w0[RB][EMAX];
  double2 w1[RB][EMAX];
  double2 w2[RB][NS];
  int off0[EMAX], off1[EMAX];
  double c[RB];
  union {
    struct {                               // the rows' own lists, when they have to be merged
      int roff[2][RB][EMAX];
      double2 rw[2][RB][EMAX];
    };
    double2 W2[WMAX2][RB];                 // dense dimension-2 weights of a wide union window (after the merge)
  };
  int ucnt[2];
};

// The contraction of a group whose rows use only the dimension-2 slots TLO..THI: union nodes
// q = TLO .. RB-1+THI of the run starting at ub / d0b / ... (node i2b - H2).  Every load has a
// compile-time offset and no predicate; a union node outside the line (first / last group) is a
// node of the neighbouring line, chunk or guard row -- finite values that only ever meet zero
// weights (fk_api.cu allocates P and dP with guard rows at both ends).
// All loads of a pair (4 fields x up to RB + 2H nodes) are issued before its arithmetic.
template <int NQ>
struct PairVals {
  double U[NQ], D0[NQ], D1[NQ], D2[NQ];
};

template <int TLO, int THI>
__device__ __forceinline__ void contract_group(const GroupStage& st, int4 cref,
                                               const double* __restrict__ ub,
                                               const double* __restrict__ d0b,
                                               const double* __restrict__ d1b,
                                               const double* __restrict__ d2b, double acc[RB]) {
  constexpr int Q0 = TLO, Q1 = RB - 1 + THI, NQ = Q1 - Q0 + 1;   // union nodes Q0..Q1
  double2 w2[RB][THI - TLO + 1];
  double Ap[RB], B0p[RB];
#pragma unroll
  for (int r = 0; r < RB; ++r) {
    acc[r] = st.c[r];
    Ap[r] = B0p[r] = 0.0;
#pragma unroll
    for (int t = TLO; t <= THI; ++t) w2[r][t - TLO] = st.w2[r][t];
  }
  const int n0e = cref.x, n1e = cref.y;
  auto load = [&](PairVals<NQ>& v, int e0, int e1) {
    const int o = st.off0[e0] + st.off1[e1] + Q0 * FK_CW;
    const double* __restrict__ pu = ub + o;
    const double* __restrict__ p0 = d0b + o;
    const double* __restrict__ p1 = d1b + o;
    const double* __restrict__ p2 = d2b + o;
#pragma unroll
    for (int q = 0; q < NQ; ++q) {
      v.U[q] = pu[q * FK_CW];
      v.D0[q] = p0[q * FK_CW];
      v.D1[q] = p1[q * FK_CW];
      v.D2[q] = p2[q * FK_CW];
    }
  };
  auto compute = [&](const PairVals<NQ>& v, int e0, int e1) {
    double A[RB], B0[RB], B1[RB];
#pragma unroll
    for (int r = 0; r < RB; ++r) A[r] = B0[r] = B1[r] = 0.0;
#pragma unroll
    for (int q = Q0; q <= Q1; ++q) {
#pragma unroll
      for (int r = 0; r < RB; ++r) {
        const int t = q - r;
        if (t >= TLO && t <= THI) {
          const double2 w = w2[r][t - TLO];
          A[r] = fma(w.x, v.U[q - Q0], A[r]);
          A[r] = fma(w.y, v.D2[q - Q0], A[r]);
          B0[r] = fma(w.x, v.D0[q - Q0], B0[r]);
          B1[r] = fma(w.x, v.D1[q - Q0], B1[r]);
        }
      }
    }
#pragma unroll
    for (int r = 0; r < RB; ++r) {
      const double2 w1 = st.w1[r][e1];
      Ap[r] = fma(w1.x, A[r], Ap[r]);
      Ap[r] = fma(w1.y, B1[r], Ap[r]);
      B0p[r] = fma(w1.x, B0[r], B0p[r]);
    }
    if (e1 == n1e - 1) {                                 // last pair of this e0: fold it in
#pragma unroll
      for (int r = 0; r < RB; ++r) {
        const double2 w0 = st.w0[r][e0];
        acc[r] = fma(w0.x, Ap[r], acc[r]);
        acc[r] = fma(w0.y, B0p[r], acc[r]);
        Ap[r] = B0p[r] = 0.0;
      }
    }
  };
  const int pairs = n0e * n1e;
  if (pairs == 0) return;
  PairVals<NQ> v;
  for (int e0 = 0; e0 < n0e; ++e0)
    for (int e1 = 0; e1 < n1e; ++e1) {
      load(v, e0, e1);
      compute(v, e0, e1);
    }
}

// The contraction of a group whose dimension-2 weights were spread densely over the union window
// wlo .. wlo+wwidth-1 (GroupStage::W2): weights broadcast from shared memory, every u / dP value of
// the window loaded once for the four rows.  Not inlined: its registers stay out of the budget of
// the static-slot paths.
__device__ __noinline__ void contract_wide(const GroupStage& st, int n0e, int n1e,
                                           const double* __restrict__ u,
                                           const double* __restrict__ d0,
                                           const double* __restrict__ d1,
                                           const double* __restrict__ d2, int wlo, int wwidth,
                                           double* __restrict__ acc) {
#pragma unroll
      for (int r = 0; r < RB; ++r) acc[r] = st.c[r];
      for (int e0 = 0; e0 < n0e; ++e0) {
        double Ap[RB], B0p[RB];
#pragma unroll
        for (int r = 0; r < RB; ++r) Ap[r] = B0p[r] = 0.0;
        for (int e1 = 0; e1 < n1e; ++e1) {
          const int o = st.off0[e0] + st.off1[e1] + wlo * FK_CW;
          const double* pu = u + o;
          const double* p0 = d0 + o;
          const double* p1 = d1 + o;
          const double* p2 = d2 + o;
          asm volatile("" : "+l"(pu), "+l"(p0), "+l"(p1), "+l"(p2));
          double A[RB], B0[RB], B1[RB];
#pragma unroll
          for (int r = 0; r < RB; ++r) A[r] = B0[r] = B1[r] = 0.0;
          // two window nodes per iteration; an odd window reads one node past its end with the zero
          // weights W2 was cleared to (a node of the next line, chunk or a guard row)
          for (int q = 0; q < wwidth; q += 2) {
            double U[2], D0[2], D1[2], D2[2];
#pragma unroll
            for (int h = 0; h < 2; ++h) {
              U[h] = pu[h * FK_CW]; D0[h] = p0[h * FK_CW]; D1[h] = p1[h * FK_CW]; D2[h] = p2[h * FK_CW];
            }
#pragma unroll
            for (int h = 0; h < 2; ++h)
#pragma unroll
              for (int r = 0; r < RB; ++r) {
                const double2 w = st.W2[q + h][r];
                A[r] = fma(w.x, U[h], A[r]);
                A[r] = fma(w.y, D2[h], A[r]);
                B0[r] = fma(w.x, D0[h], B0[r]);
                B1[r] = fma(w.x, D1[h], B1[r]);
              }
            pu += 2 * FK_CW; p0 += 2 * FK_CW; p1 += 2 * FK_CW; p2 += 2 * FK_CW;
          }
#pragma unroll
          for (int r = 0; r < RB; ++r) {
            const double2 w1 = st.w1[r][e1];
            Ap[r] = fma(w1.x, A[r], Ap[r]);
            Ap[r] = fma(w1.y, B1[r], Ap[r]);
            B0p[r] = fma(w1.x, B0[r], B0p[r]);
          }
        }
#pragma unroll
        for (int r = 0; r < RB; ++r) {
          const double2 w0 = st.w0[r][e0];
          acc[r] = fma(w0.x, Ap[r], acc[r]);
          acc[r] = fma(w0.y, B0p[r], acc[r]);
        }
      }
}

// WIDE: with the banded dimension-2 path (instantiated for grids whose last dimension is non-uniform;
// on uniform grids the few rows that reach beyond H2 nodes take the row-at-a-time path and the
// kernel keeps the register budget of the static-slot paths)
template <bool WIDE>
__global__ void __launch_bounds__(WARPS * 32, MINB)
fk_rowblock3d(FkGrid g, FkOperator op, const double* __restrict__ Pold,
              const double* __restrict__ dP, double* __restrict__ Pnew, int n_chunks, int chunk0,
              int chunk1, int n, int N, int G2, int NT1) {
  __shared__ GroupStage stage_all[WARPS];
  GroupStage& st = stage_all[threadIdx.y];
  const int lane = threadIdx.x;
  const int n1 = g.n[1], n2 = g.n[2];
  const int g2 = blockIdx.x % G2;
  const int t01 = blockIdx.x / G2;
  const int i1 = (t01 % NT1) * WARPS + threadIdx.y;
  const int i0 = t01 / NT1;
  if (i1 >= n1) return;
  const int i2b = g2 * RB;
  const int rows = min(RB, n2 - i2b);
  const int jb = (i0 * n1 + i1) * n2 + i2b;
  // the staged rows serve CPB consecutive chunks: blockIdx.y counts chunk groups
  const int cfirst = chunk0 + blockIdx.y * CPB, clast = min(chunk1, cfirst + CPB);
  const size_t chunk_elems = (size_t)g.J * FK_CW;
  const size_t field = (size_t)n_chunks * chunk_elems;

  // ---- stage the group's rows; decide whether they can be contracted together
  int4 cnt[RB];
  int4 cref = make_int4(0, 0, 0, 0);
  int ref = -1;                                         // first row that is not a Dirichlet row
#pragma unroll
  for (int r = 0; r < RB; ++r) {
    cnt[r] = r < rows ? *reinterpret_cast<const int4*>(op.cnt + (size_t)(jb + r) * 4)
                      : make_int4(0, 0, 0, FK_ROW_DIRICHLET);
    if (ref < 0 && !(cnt[r].w & FK_ROW_DIRICHLET)) { ref = r; cref = cnt[r]; }
  }
  if (ref < 0) {                                        // only Dirichlet rows: the constants
    for (int chunk = cfirst; chunk < clast; ++chunk) {
      const int m = fkd::column_of(g, chunk, lane);
      double* __restrict__ out = Pnew + (size_t)chunk * chunk_elems + (size_t)jb * FK_CW + lane;
      for (int r = 0; r < rows; ++r)
        if (m >= n && m <= N) out[r * FK_CW] = op.c[jb + r];
    }
    return;
  }
  // every load of the stage is issued before anything is compared (one round of latency)
  bool ok = true;                                       // dimension-0 / 1 lists fit the blocked paths
  bool ok2 = !g.periodic[2];                            // dimension 2 fits the static slots (a wrapped run has none)
  bool same = true;                                     // rows put their dimension-0 / 1 entries on the same nodes
  {
    const int dim = lane >> 4, e = lane & (EMAX - 1);   // lanes 0..15: dimension 0, 16..31: 1
    const int q = g.qoff[dim] + e;
    const int q2 = g.qoff[2] + lane;
    int off01[RB], off2[RB];
    double2 w01[RB], w2[RB];
    double cr = 0.0;
#pragma unroll
    for (int r = 0; r < RB; ++r) {
      const bool dir = (cnt[r].w & FK_ROW_DIRICHLET) != 0;
      const size_t row = (size_t)(jb + r) * g.RS;
      const int ne = dim ? cnt[r].y : cnt[r].x;
      off01[r] = INT_MAX;                               // "no entry": sorts last in the merge
      off2[r] = 0;
      w01[r] = w2[r] = make_double2(0.0, 0.0);
      ok = ok && cnt[r].x <= EMAX && cnt[r].y <= EMAX;
      ok2 = ok2 && cnt[r].z <= NS;
      if (!dir && ne <= EMAX && e < ne) { off01[r] = op.off[row + q]; w01[r] = op.w[row + q]; }
      if (!dir && lane < cnt[r].z && lane < NS) { off2[r] = op.off[row + q2]; w2[r] = op.w[row + q2]; }
      if (lane == r && r < rows) cr = op.c[jb + r];
    }
    int oref = INT_MAX;
#pragma unroll
    for (int r = 0; r < RB; ++r) if (r == ref) oref = off01[r];
    if (lane < RB * NS) st.w2[lane / NS][lane % NS] = make_double2(0.0, 0.0);
    if (lane < RB) st.c[lane] = cr;
#pragma unroll
    for (int r = 0; r < RB; ++r)
      if (!(cnt[r].w & FK_ROW_DIRICHLET)) same = same && off01[r] == oref;
    same = __all_sync(0xffffffffu, same);
    ok = __all_sync(0xffffffffu, ok);
    ok2 = __all_sync(0xffffffffu, ok2);
    if (!WIDE) ok = ok && ok2;          // no banded path: such a group goes row by row, skip the merge
    __syncwarp();
    if (same) {
      if (dim) st.off1[e] = oref; else st.off0[e] = oref;
#pragma unroll
      for (int r = 0; r < RB; ++r)
        if (dim) st.w1[r][e] = w01[r]; else st.w0[r][e] = w01[r];
    } else if (ok) {
      // the rows disagree somewhere (a quadrature point of one row fell into the next cell):
      // contract them together on the UNION of their entry lists, zero weights where a row has no
      // entry.  One lane per dimension merges the four ascending lists (rare path, <= 64 steps).
#pragma unroll
      for (int r = 0; r < RB; ++r) { st.roff[dim][r][e] = off01[r]; st.rw[dim][r][e] = w01[r]; }
      __syncwarp();
      if (e == 0) {
        int head[RB] = {0, 0, 0, 0};
        int k = 0;
        for (;;) {
          int lo = INT_MAX;
#pragma unroll
          for (int r = 0; r < RB; ++r)
            if (head[r] < EMAX) lo = min(lo, st.roff[dim][r][head[r]]);
          if (lo == INT_MAX) break;
          if (k == EMAX) { k = EMAX + 1; break; }           // more than EMAX distinct nodes
          if (dim) st.off1[k] = lo; else st.off0[k] = lo;
#pragma unroll
          for (int r = 0; r < RB; ++r) {
            double2 w = make_double2(0.0, 0.0);
            if (head[r] < EMAX && st.roff[dim][r][head[r]] == lo) w = st.rw[dim][r][head[r]++];
            if (dim) st.w1[r][k] = w; else st.w0[r][k] = w;
          }
          ++k;
        }
        st.ucnt[dim] = k;
      }
      __syncwarp();
      cref.x = st.ucnt[0];
      cref.y = st.ucnt[1];
      ok = cref.x <= EMAX && cref.y <= EMAX;
    }
#pragma unroll
    for (int r = 0; r < RB; ++r) {
      if (cnt[r].w & FK_ROW_DIRICHLET) continue;
      if (ok && ok2 && lane < cnt[r].z && lane < NS) {
        // dimension 2: entries -> slots around the row's own node (its stride is 1 node)
        const int t = off2[r] / FK_CW - (i2b + r) + H2;
        if (t >= 0 && t < NS) st.w2[r][t] = w2[r];
        else ok2 = false;
      }
    }
  }
  ok = __all_sync(0xffffffffu, ok);
  ok2 = __all_sync(0xffffffffu, ok2);
  __syncwarp();

  // ---- rows that reach beyond H2 nodes along dimension 2 (a fine non-uniform grid: the paper's radial
  // grid): if their union window is a band of at most WMAX2 nodes, spread the
  // dimension-2 weights densely over it in shared memory (zero where a row has no entry) and contract
  // the four rows together on the window -- every u / dP value still loaded once per group
  int wlo = INT_MAX, whi = -1;
  bool wide = WIDE && ok && !ok2 && !g.periodic[2];
  if (wide) {
#pragma unroll
    for (int r = 0; r < RB; ++r) {
      if ((cnt[r].w & FK_ROW_DIRICHLET) || cnt[r].z == 0) continue;
      const int* __restrict__ o = op.off + (size_t)(jb + r) * g.RS + g.qoff[2];
      wlo = min(wlo, o[0] / FK_CW);
      whi = max(whi, o[cnt[r].z - 1] / FK_CW);
    }
    wide = whi >= wlo && whi - wlo + 1 <= WMAX2;
  }
  const int wwidth = whi - wlo + 1;
  if (wide) {
    for (int k = lane; k < WMAX2 * RB; k += 32) (&st.W2[0][0])[k] = make_double2(0.0, 0.0);
    __syncwarp();
#pragma unroll
    for (int r = 0; r < RB; ++r) {
      if (cnt[r].w & FK_ROW_DIRICHLET) continue;
      const size_t row = (size_t)(jb + r) * g.RS + g.qoff[2];
      for (int e = lane; e < cnt[r].z; e += 32) st.W2[op.off[row + e] / FK_CW - wlo][r] = op.w[row + e];
    }
    __syncwarp();
  }
  ok = ok && ok2;                                        // the static-slot blocked path
  if (g.paths && lane == 0 && blockIdx.y == 0)           // FK_FLAG_COUNT_PATHS: which path this group takes
    atomicAdd(g.paths + (wide ? (same ? FK_PATH_3D_WIDE : FK_PATH_3D_WIDE_MERGED)
                              : ok ? (same ? FK_PATH_3D_SAME : FK_PATH_3D_MERGED) : FK_PATH_3D_ROWWISE), 1ULL);

  // ---- which dimension-2 slots carry a weight in any row decides the variant of the blocked path
  unsigned tmask = 0;
#pragma unroll
  for (int r = 0; r < RB; ++r)
#pragma unroll
    for (int t = 0; t < NS; ++t) {
      const double2 w = st.w2[r][t];
      if (w.x != 0.0 || w.y != 0.0) tmask |= 1u << t;
    }
  tmask = __reduce_or_sync(0xffffffffu, tmask);          // uniform
  const int base2 = (i2b - H2) * FK_CW;                  // union node 0

  // pull this group's own rows of the plane L2PF steps ahead into L2 (one bulk prefetch
  // per field): the blocks that will read them find them there instead of in DRAM
  if (lane < 4 && i0 + L2PF < g.n[0]) {
    const size_t ahead = (size_t)(jb + L2PF * n1 * n2) * FK_CW;
    for (int chunk = cfirst; chunk < clast; ++chunk) {
      const double* src = (lane == 0 ? Pold : dP + (size_t)(lane - 1) * field) + (size_t)chunk * chunk_elems + ahead;
      asm volatile("cp.async.bulk.prefetch.L2.global [%0], %1;" ::"l"(src), "r"(rows * FK_CW * 8) : "memory");
    }
  }
  if (lane >= 4 && lane < 7 && blockIdx.y == 0 && i0 + L2PF < g.n[0]) {   // and the operator rows
    const size_t ja = (size_t)jb + (size_t)L2PF * n1 * n2;
    const void* src = lane == 4 ? (const void*)(op.w + ja * g.RS)
                    : lane == 5 ? (const void*)(op.off + ja * g.RS) : (const void*)(op.cnt + ja * 4);
    const int bytes = rows * (lane == 4 ? g.RS * 16 : lane == 5 ? g.RS * 4 : 16);
    // the bulk prefetch wants a 16-byte aligned start and a size that is a multiple of 16; a row of
    // op.off is RS*4 = 8*sum(Q_k) bytes, so with an odd sum(Q_k) every other row starts 8 bytes off:
    // start rounded down, end rounded down (both stay inside the allocation; a hint may lose a tail)
    const unsigned long long a0 = (unsigned long long)src & ~15ull;
    const unsigned long long a1 = ((unsigned long long)src + (unsigned long long)bytes) & ~15ull;
    if (a1 > a0)
      asm volatile("cp.async.bulk.prefetch.L2.global [%0], %1;" ::"l"(a0), "r"((int)(a1 - a0)) : "memory");
  }
  for (int chunk = cfirst; chunk < clast; ++chunk) {
    const int m = fkd::column_of(g, chunk, lane);
    const bool active = m >= n && m <= N;
    const double* __restrict__ u = Pold + (size_t)chunk * chunk_elems + lane;
    const double* __restrict__ d0 = dP + (size_t)chunk * chunk_elems + lane;
    const double* __restrict__ d1 = d0 + field;
    const double* __restrict__ d2 = d1 + field;
    double* __restrict__ out = Pnew + (size_t)chunk * chunk_elems + (size_t)jb * FK_CW + lane;
    if (wide) {
      // ---- banded along dimension 2: dense window, weights broadcast from shared memory
      double acc[RB];
      contract_wide(st, cref.x, cref.y, u, d0, d1, d2, wlo, wwidth, acc);
#pragma unroll
      for (int r = 0; r < RB; ++r)
        if (r < rows && active) out[r * FK_CW] = (cnt[r].w & FK_ROW_DIRICHLET) ? st.c[r] : acc[r];
      continue;
    }
    if (!ok) {
      // ---- row-at-a-time path
#pragma unroll
      for (int r = 0; r < RB; ++r) {
        if (r < rows) {
          const size_t j = (size_t)(jb + r);
          const double acc = fkd::contract_row<3>(g, op.w + j * g.RS, op.off + j * g.RS, cnt[r],
                                                  op.c[j], u, d0, d1, d2);
          if (active) out[r * FK_CW] = acc;
        }
      }
      continue;
    }
    // ---- blocked path
    double acc[RB];
    const double* __restrict__ ub = u + base2;
    const double* __restrict__ d0b = d0 + base2;
    const double* __restrict__ d1b = d1 + base2;
    const double* __restrict__ d2b = d2 + base2;
    if ((tmask & ~0x04u) == 0) contract_group<2, 2>(st, cref, ub, d0b, d1b, d2b, acc);
    else if ((tmask & ~0x06u) == 0) contract_group<1, 2>(st, cref, ub, d0b, d1b, d2b, acc);
    else if ((tmask & ~0x0cu) == 0) contract_group<2, 3>(st, cref, ub, d0b, d1b, d2b, acc);
    else if ((tmask & ~0x0eu) == 0) contract_group<1, 3>(st, cref, ub, d0b, d1b, d2b, acc);
    else contract_group<0, 4>(st, cref, ub, d0b, d1b, d2b, acc);
#pragma unroll
    for (int r = 0; r < RB; ++r)
      if (r < rows && active) out[r * FK_CW] = acc[r];
  }
}

}  // namespace

cudaError_t fk_launch_rowblock3d(const FkGrid& g, FkOperator op, const double* Pold,
                                 const double* dP, double* Pnew, int n_chunks, int chunk0,
                                 int chunk1, int n, int N, cudaStream_t s) {
  const int G2 = (g.n[2] + RB - 1) / RB;
  const int NT1 = (g.n[1] + WARPS - 1) / WARPS;
  dim3 block(FK_CW, WARPS), grid((unsigned)((long long)g.n[0] * NT1 * G2), (unsigned)((chunk1 - chunk0 + CPB - 1) / CPB));
  if (g.uniform[2]) fk_rowblock3d<false><<<grid, block, 0, s>>>(g, op, Pold, dP, Pnew, n_chunks, chunk0, chunk1, n, N, G2, NT1);
  else fk_rowblock3d<true><<<grid, block, 0, s>>>(g, op, Pold, dP, Pnew, n_chunks, chunk0, chunk1, n, N, G2, NT1);
  return cudaGetLastError();
}
