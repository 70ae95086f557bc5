// fk_far2d.cu -- the 2-D apply kernel for the rows the fused kernel leaves out (not FK_ROW_NEAR):
// P(:, n:N) <- A_nu [P; dP](:, n:N) on the rows whose quadrature points travel more
// than FK_H nodes (config 4: small momenta, where pitch-angle scattering carries a point across
// tens of nodes in one step).  dP comes from fk_slopes (HBM / L2).
//
// Lane = output-time column of a 32-column chunk; a warp owns a group of RB = 4 rows adjacent
// along dimension 1 (the fast one) and serves CPB chunks with one reading of the rows' weights.
// Two shapes of row occur, and the warp picks per group (warp-uniform test):
//
//   banded    the points of a row land in a run of nodes a few cells wide and the four runs
//             overlap: the rows' dimension-1 weights are spread out DENSELY over the union window
//             [qlo, qhi] (shared memory, zero where a row has no entry) and every u / d0 / d1 value
//             of the window is loaded ONCE for the four rows: per union node 3 loads per chunk +
//             4 broadcast weight loads feed 12 multiply-adds per chunk.  Needs the four rows to put
//             their dimension-0 entries on the same lines (the usual case).
//   scattered each of the Q points lands in a cell of its own, many cells apart (2Q isolated entries
//             in a window of up to n1 nodes): no two rows share a node, every multiply-add needs
//             its own operand; the row is contracted entry by entry (fkd::contract_row's order) and
//             only the weight / offset loads are shared by the CPB chunks.  This shape is bound by
//             the L1 data path: one 256-byte operand row (2 wavefronts) per multiply-add.
#include <climits>

#include "fk_device.cuh"

namespace {

constexpr int RB = 4;                      // rows per warp
constexpr int WARPS = 4;                   // warps per block: consecutive groups of one line
constexpr int CPB = 2;                     // chunks served by one staging of a group's rows
constexpr int WMAX = 32;                   // widest union window of the banded path (nodes)
constexpr int E0MAX = 16;                  // dimension-0 entries per row in the banded path

struct FarStage {                          // per warp, shared memory
  double2 W1[WMAX][RB];                    // dense dimension-1 weights of the union window
  double2 w0[E0MAX][RB];
  int off0[E0MAX];
};

__global__ void __launch_bounds__(WARPS * 32, 4)
fk_far2d(FkGrid g, FkOperator op, const double* __restrict__ Pold, const double* __restrict__ dP,
         double* __restrict__ Pnew, int n_chunks, int chunk0, int chunk1, int n, int N, int line0,
         int nlines, int G1) {
  __shared__ FarStage stage_all[WARPS];
  FarStage& st = stage_all[threadIdx.y];
  const int lane = threadIdx.x;
  const int gid = blockIdx.x * WARPS + threadIdx.y;
  if (gid >= nlines * G1) return;
  const int n1 = g.n[1];
  const int i0 = line0 + gid / G1;
  const int i1b = (gid - (gid / G1) * G1) * RB;
  const int rows = min(RB, n1 - i1b);
  const int jb = i0 * n1 + i1b;

  int4 cnt[RB];
  bool mine[RB];
  bool any = false;
#pragma unroll
  for (int r = 0; r < RB; ++r) {
    cnt[r] = r < rows ? *reinterpret_cast<const int4*>(op.cnt + (size_t)(jb + r) * 4)
                      : make_int4(0, 0, 0, FK_ROW_DIRICHLET);
    mine[r] = !(cnt[r].w & (FK_ROW_NEAR | FK_ROW_DIRICHLET));   // the others: fk_fused2d
    any = any || mine[r];
  }
  if (!any) return;

  const size_t chunk_elems = (size_t)g.J * FK_CW;
  const size_t field = (size_t)n_chunks * chunk_elems;
  const int cfirst = chunk0 + blockIdx.y * CPB;
  const double* __restrict__ u[CPB];
  const double* __restrict__ d0[CPB];
  const double* __restrict__ d1[CPB];
  double* __restrict__ out[CPB];
  bool store[CPB];
#pragma unroll
  for (int c = 0; c < CPB; ++c) {
    const int chunk = min(cfirst + c, chunk1 - 1);       // a missing last chunk: computed twice, stored once
    const int m = fkd::column_of(g, chunk, lane);
    store[c] = cfirst + c < chunk1 && m >= n && m <= N;
    u[c] = Pold + (size_t)chunk * chunk_elems + lane;
    d0[c] = dP + (size_t)chunk * chunk_elems + lane;
    d1[c] = d0[c] + field;
    out[c] = Pnew + (size_t)chunk * chunk_elems + (size_t)jb * FK_CW + lane;
  }
  const int q1 = g.qoff[1];

  // ---- shape of the group: union window along dimension 1, dimension-0 lists equal?
  int qlo = INT_MAX, qhi = -1, sum_d1 = 0, n0e = 0, ref = -1;
#pragma unroll
  for (int r = 0; r < RB; ++r) {
    if (mine[r]) {
      if (ref < 0) { ref = r; n0e = cnt[r].x; }
      if (cnt[r].y > 0) {
        if (cnt[r].z) {                        // packed by fk_assemble: 1 + first node | last node << 16
          qlo = min(qlo, (cnt[r].z & 0xffff) - 1);
          qhi = max(qhi, (int)((unsigned)cnt[r].z >> 16));   // logical shift: last node up to 65534
        } else {
          const int* __restrict__ o = op.off + (size_t)(jb + r) * g.RS + q1;
          qlo = min(qlo, o[0] / FK_CW);
          qhi = max(qhi, o[cnt[r].y - 1] / FK_CW);
        }
        sum_d1 += cnt[r].y;
      }
    }
  }
  const int width = qhi - qlo + 1;
  bool dense = sum_d1 > 0 && width > 0 && width <= WMAX && n0e <= E0MAX &&
               width * (6 * CPB + 4) < sum_d1 * (6 * CPB + 2);   // L1 wavefronts of the two paths
  if (dense) {                                   // the rows' dimension-0 entries on the same lines?
    int oref = INT_MAX;
    bool same = true;
#pragma unroll
    for (int r = 0; r < RB; ++r) {
      if (mine[r]) {
        const int o = lane < cnt[r].x ? op.off[(size_t)(jb + r) * g.RS + lane] : INT_MAX;
        if (r == ref) oref = o;
        same = same && cnt[r].x == n0e && o == oref;
      }
    }
    dense = __all_sync(0xffffffffu, same);
    if (dense && lane < n0e) st.off0[lane] = oref;
  }

  if (g.paths && lane == 0 && blockIdx.y == 0)           // FK_FLAG_COUNT_PATHS
    atomicAdd(g.paths + (dense ? FK_PATH_2D_BANDED : FK_PATH_2D_SCATTERED), 1ULL);
  if (dense) {
    // ---- banded path
    for (int k = lane; k < WMAX * RB; k += 32) (&st.W1[0][0])[k] = make_double2(0.0, 0.0);
    __syncwarp();
    double acc[RB][CPB];
#pragma unroll
    for (int r = 0; r < RB; ++r) {
      const size_t row = (size_t)(jb + r) * g.RS;
      if (mine[r])
        for (int e = lane; e < cnt[r].y; e += 32)
          st.W1[op.off[row + q1 + e] / FK_CW - qlo][r] = op.w[row + q1 + e];
      if (lane < n0e) st.w0[lane][r] = mine[r] ? op.w[row + lane] : make_double2(0.0, 0.0);
      const double cr = mine[r] ? op.c[jb + r] : 0.0;
#pragma unroll
      for (int c = 0; c < CPB; ++c) acc[r][c] = cr;
    }
    __syncwarp();
    for (int e0 = 0; e0 < n0e; ++e0) {
      const int base = st.off0[e0] + qlo * FK_CW;
      // one pointer per chunk and field, advanced two nodes per iteration (kept opaque: otherwise
      // every load re-derives its 64-bit address from the chunk index)
      const double* pu[CPB];
      const double* p0[CPB];
      const double* p1[CPB];
#pragma unroll
      for (int c = 0; c < CPB; ++c) {
        pu[c] = u[c] + base; p0[c] = d0[c] + base; p1[c] = d1[c] + base;
        asm volatile("" : "+l"(pu[c]), "+l"(p0[c]), "+l"(p1[c]));
      }
      double A[RB][CPB], B0[RB][CPB];
#pragma unroll
      for (int r = 0; r < RB; ++r)
#pragma unroll
        for (int c = 0; c < CPB; ++c) A[r][c] = B0[r][c] = 0.0;
      // two union nodes per iteration; an odd window reads one node past its end with the zero
      // weights W1 was cleared to (a node of the same line, the next line or a guard row)
      for (int q = 0; q < width; q += 2) {
        double U[2][CPB], D0[2][CPB], D1[2][CPB];
#pragma unroll
        for (int h = 0; h < 2; ++h)
#pragma unroll
          for (int c = 0; c < CPB; ++c) {
            U[h][c] = pu[c][h * FK_CW]; D0[h][c] = p0[c][h * FK_CW]; D1[h][c] = p1[c][h * FK_CW];
          }
#pragma unroll
        for (int h = 0; h < 2; ++h) {
          double2 w[RB];
#pragma unroll
          for (int r = 0; r < RB; ++r) w[r] = st.W1[q + h][r];
#pragma unroll
          for (int c = 0; c < CPB; ++c)
#pragma unroll
            for (int r = 0; r < RB; ++r) {
              A[r][c] = fma(w[r].x, U[h][c], A[r][c]);
              A[r][c] = fma(w[r].y, D1[h][c], A[r][c]);
              B0[r][c] = fma(w[r].x, D0[h][c], B0[r][c]);
            }
        }
#pragma unroll
        for (int c = 0; c < CPB; ++c) { pu[c] += 2 * FK_CW; p0[c] += 2 * FK_CW; p1[c] += 2 * FK_CW; }
      }
#pragma unroll
      for (int r = 0; r < RB; ++r) {
        const double2 w0 = st.w0[e0][r];
#pragma unroll
        for (int c = 0; c < CPB; ++c) {
          acc[r][c] = fma(w0.x, A[r][c], acc[r][c]);
          acc[r][c] = fma(w0.y, B0[r][c], acc[r][c]);
        }
      }
    }
#pragma unroll
    for (int r = 0; r < RB; ++r)
#pragma unroll
      for (int c = 0; c < CPB; ++c)
        if (mine[r] && store[c]) out[c][r * FK_CW] = acc[r][c];
    return;
  }

  // ---- scattered path: row by row, entry by entry
#pragma unroll
  for (int c = 0; c < CPB; ++c) asm volatile("" : "+l"(u[c]), "+l"(d0[c]), "+l"(d1[c]));
#pragma unroll
  for (int r = 0; r < RB; ++r) {
    if (!mine[r]) continue;
    const size_t row = (size_t)(jb + r) * g.RS;
    const double2* __restrict__ w0p = op.w + row;
    const int* __restrict__ o0p = op.off + row;
    const double2* __restrict__ w1p = w0p + q1;
    const int* __restrict__ o1p = o0p + q1;
    const int n0r = cnt[r].x, n1r = cnt[r].y;
    double acc[CPB];
    const double cr = op.c[jb + r];
#pragma unroll
    for (int c = 0; c < CPB; ++c) acc[c] = cr;
    for (int e0 = 0; e0 < n0r; ++e0) {
      const double2 w0 = w0p[e0];
      const int o0 = o0p[e0];
      double A[CPB], B0[CPB];
#pragma unroll
      for (int c = 0; c < CPB; ++c) A[c] = B0[c] = 0.0;
#pragma unroll 4
      for (int e1 = 0; e1 < n1r; ++e1) {
        const double2 w1 = w1p[e1];
        const int o = o0 + o1p[e1];
#pragma unroll
        for (int c = 0; c < CPB; ++c) {
          A[c] = fma(w1.x, u[c][o], A[c]);
          A[c] = fma(w1.y, d1[c][o], A[c]);
          B0[c] = fma(w1.x, d0[c][o], B0[c]);
        }
      }
#pragma unroll
      for (int c = 0; c < CPB; ++c) {
        acc[c] = fma(w0.x, A[c], acc[c]);
        acc[c] = fma(w0.y, B0[c], acc[c]);
      }
    }
#pragma unroll
    for (int c = 0; c < CPB; ++c)
      if (store[c]) out[c][r * FK_CW] = acc[c];
  }
}

}  // namespace

cudaError_t fk_launch_far2d(const FkGrid& g, FkOperator op, const double* Pold, const double* dP,
                            double* Pnew, int n_chunks, int chunk0, int chunk1, int n, int N,
                            int line0, int nlines, cudaStream_t s) {
  const int G1 = (g.n[1] + RB - 1) / RB;
  dim3 block(FK_CW, WARPS),
      grid((unsigned)(((long long)nlines * G1 + WARPS - 1) / WARPS), (unsigned)((chunk1 - chunk0 + CPB - 1) / CPB));
  fk_far2d<<<grid, block, 0, s>>>(g, op, Pold, dP, Pnew, n_chunks, chunk0, chunk1, n, N, line0,
                                  nlines, G1);
  return cudaGetLastError();
}
