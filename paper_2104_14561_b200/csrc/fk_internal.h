// fk_internal.h -- types shared by the host side (fk_api.cu) and the kernels (fk_kernels.cu)
// of the CUDA path.  Nothing here is shared with oracle/.
//
// HBM layout:
//   P      two buffers, each [n_chunks][J][FK_CW] fp64: output-time columns are grouped in
//          chunks of FK_CW = 32; inside a chunk the node index is slow and the column fast,
//          so one warp (lane = column) reads or writes one 256-byte row per node.
//          Column m lives in chunk m / 32, lane m % 32.
//   dP     [d][n_chunks][J][FK_CW] fp64: the nodal slopes of Eq. 15 of the buffer being read.
//   A_nu   the step operator in FACTORED ELL form, one row per node:
//          per dimension k up to 2*Q_k entries (offset, alpha, beta) = the quadrature-folded
//          value and slope weights on the distinct nodes the Q_k points touch, plus the
//          absorbed constant c_j.  The full row is the sum of (d+1) rank-1 tensor products
//          of these lists and is never expanded.
#ifndef FK_INTERNAL_H
#define FK_INTERNAL_H

#include <cuda_runtime.h>

#define FK_CW 32          // columns per chunk = lanes per warp
#define FK_QMAX 32        // == FK_MAX_Q of include/fk.h

struct FkGrid {
  int d;
  int n[3];               // nodes per dimension
  int Q[3];               // Gauss-Hermite points per dimension
  int qoff[3];            // first entry of dimension k inside a row
  int RS;                 // row stride in entries = sum_k 2*Q[k]
  int uniform[3];         // 1: x[k] is uniform to rounding -> O(1) cell guess
  int face_kind[3][2];
  long long J;            // prod n[k]
  long long stride[3];    // node-index stride of dimension k (last dimension fastest)
  double face_value[3][2];
  double lo[3], hi[3];    // box faces = x[k][0], x[k][n-1]
  double inv_h0[3];       // (n-1)/(hi-lo)
  double dt, sq;          // sq = sqrt(2 dt)
  const double* x[3];     // device: node coordinates
  const double* inv_h[3]; // device: 1/(x[i+1]-x[i]), n-1 values
  double gh_a[3][FK_QMAX];
  double gh_w[3][FK_QMAX];
};

struct FkOperator {       // device pointers of one assembled A_nu
  double2* w;             // [J][RS] (alpha, beta)
  int* off;               // [J][RS] element offset i_k*stride_k*FK_CW inside a chunk
  int* cnt;               // [J][4]  entries used per dimension
  double* c;              // [J]     absorbed constant (= g on Dirichlet nodes)
};

// launchers (fk_kernels.cu); all asynchronous on `s`, return the launch's cudaError_t
cudaError_t fk_launch_fill_chi(const FkGrid& g, double* P, int n_chunks, cudaStream_t s);
cudaError_t fk_launch_assemble(const FkGrid& g, const double* b, const double* sigma,
                               FkOperator op, cudaStream_t s);
cudaError_t fk_launch_slopes(const FkGrid& g, const double* P, double* dP, int n_chunks,
                             int chunk0, int chunk1, cudaStream_t s);
cudaError_t fk_launch_apply(const FkGrid& g, FkOperator op, const double* Pold, const double* dP,
                            double* Pnew, int n_chunks, int chunk0, int chunk1, int n, int N,
                            cudaStream_t s);
cudaError_t fk_launch_gather_columns(const FkGrid& g, const double* P, int m0, int m1,
                                     double* out, cudaStream_t s);

#endif
