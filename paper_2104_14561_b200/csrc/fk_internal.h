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

#include "../../include/fk.h"   // FK_PATH_* (the only part of the ABI the kernels see)

#define FK_CW 32          // columns per chunk = lanes per warp
#define FK_QMAX 32        // == FK_MAX_Q of include/fk.h
#define FK_GUARD_ROWS 8   // zeroed node rows before and after the P and dP allocations

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
  int validate;           // FK_FLAG_VALIDATE: report NaN / Inf coefficients of updated nodes
  int periodic[3];        // dimension k is FK_FACE_PERIODIC (R21)
  int weighted;           // FK_FLAG_WEIGHTED_SLOPES (R22)
  int general_slopes;     // any periodic dimension or weighted slopes: fk_slopes takes its general path
  int shard_index, shard_count;   // this context owns the chunks c with c % count == index
  int near_lo, near_hi;           // 2-D: only rows on the lines near_lo .. near_hi-1 may be FK_ROW_NEAR (set per
                                  // step by fk_evolve: lines where most rows are far go to fk_far2d whole)
  unsigned long long* paths;      // device, FK_FLAG_COUNT_PATHS only (else NULL): FK_PATH_COUNT counters, one
                                  // per group of four rows and step, of the path the group was contracted on
  const double2* wgt[3];  // device, weighted only: per node the normalised weights (omega_a, omega_b)
                          // attached to the two divided differences its slope is the mean of
  const double* x[3];     // device: node coordinates
  const double* inv_h[3]; // device: 1/(x[i+1]-x[i]), n-1 values
  double gh_a[3][FK_QMAX];
  double gh_w[3][FK_QMAX];
};

// bits of the device status word (coefficient errors found by fk_assemble)
#define FK_BAD_NEG_SIGMA 1
#define FK_BAD_NONFINITE 2

// Row flags kept in cnt[j][3]
#define FK_ROW_DIRICHLET 1   // node on an ABSORB face: the row is the constant c_j = g
#define FK_ROW_NEAR 2        // every entry lies within FK_H nodes of the row's node in each
                             // dimension: the row has a compact record for the fused kernel

#define FK_H 2               // halo of the fused 2-D kernel (nodes per side and dimension)
#define FK_NW (2 * FK_H + 1) // entries per dimension of a compact record

// Per coefficient slot, what fk_classify finds about the rows that leave the fused halo (2-D):
// [0] their number, [1] FK_FAR_BIG - lowest line (dimension-0 index) holding such a row,
// [2] 1 + highest such line, [3] FK_FAR_BIG - lowest line their entries touch, [4] 1 + highest
// line their entries touch.  All fields grow by atomicAdd / atomicMax from 0.
#define FK_FAR_STRIDE 8
#define FK_FAR_BIG (1 << 30)

// Compact record of a near row (2-D): per dimension k the FK_NW = 2*FK_H+1 weights
// (alpha, beta) of the nodes i_k - FK_H .. i_k + FK_H around the row's own node i_k, zero where
// no quadrature point lands (or where the node does not exist); mask[k] has bit t set where
// slot t received an entry.  192 bytes, 16-byte aligned, so a line of records is one bulk copy.
struct FkRec2 {
  double c;               // absorbed constant (= g on Dirichlet nodes)
  int flags;              // FK_ROW_* in bits 0-7, mask[0] in bits 8-15, mask[1] in bits 16-23
  int mask[2];            // used slots per dimension (0 on Dirichlet rows)
  int pad[3];
  double2 w[2][FK_NW];
};

struct FkOperator {       // device pointers of one assembled A_nu
  double2* w;             // [J][RS] (alpha, beta)
  int* off;               // [J][RS] element offset i_k*stride_k*FK_CW inside a chunk
  int* cnt;               // [J][4]  entries used per dimension; [3] = FK_ROW_* flags
  double* c;              // [J]     absorbed constant (= g on Dirichlet nodes)
  FkRec2* rec;            // [J]     compact records (2-D grids only, else NULL)
};

// launchers (fk_kernels.cu); all asynchronous on `s`, return the launch's cudaError_t
cudaError_t fk_launch_fill_chi(const FkGrid& g, double* P, int n_chunks, cudaStream_t s);
cudaError_t fk_launch_assemble(const FkGrid& g, const double* b, const double* sigma,
                               FkOperator op, int* status, unsigned long long* work,
                               cudaStream_t s);
// operators of the steps nu_hi, nu_hi-1, ..., nu_hi-count+1 into consecutive operator-sized pieces
// of `op` (1-D multi-step path); work + 4*nu counts rows / non-zeros like fk_launch_assemble
cudaError_t fk_launch_assemble_batch(const FkGrid& g, const double* coef, int slots, int nu_hi,
                                     int count, int autonomous, FkOperator op, int* status,
                                     unsigned long long* work, cudaStream_t s);
// 1-D, many steps per launch (fk_line1d.cu): column groups of cg columns keep their line in shared
// memory over the steps n = n_hi .. n_hi-nsteps+1, operators from the batch `op`; reads Pcur, writes
// the final state of the touched columns to BOTH buffers
size_t fk_line1d_smem(const FkGrid& g, int cg);
int fk_line1d_group(const FkGrid& g, size_t smem_limit);
cudaError_t fk_line1d_setup(const FkGrid& g, int cg);
cudaError_t fk_launch_line1d(const FkGrid& g, FkOperator op, int cg, int nsteps, int n_hi,
                             int autonomous, double* Pcur, double* Pother, int n_chunks, int N,
                             cudaStream_t s);
// 2 x (iters x 8 chains) fused multiply-adds per thread on blocks x threads threads (fk_peak.cu)
cudaError_t fk_launch_dfma_peak(double* out, int blocks, int threads, int iters, cudaStream_t s);
// far_rows[slot] = number of rows of the step held in that coefficient slot that are not
// FK_ROW_NEAR (2-D only), for the `count` steps step0.. whose slices sit at
// coef + (step % slots) * 2*d*J (b then sigma); far_rows entries must be zeroed before
// far_line[slot * n[0] + i0] = how many of them sit on line i0 (zeroed before, like far_rows)
cudaError_t fk_launch_classify(const FkGrid& g, const double* coef, int slots, int step0,
                               int count, int* far_rows, int* far_line, cudaStream_t s);
// fused 2-D kernel: slopes + apply for the FK_ROW_NEAR and Dirichlet rows of every active
// column; P never leaves the chip between the two (fk_fused2d.cu)
// ... on the output lines line_lo .. line_hi-1 (rows elsewhere are not FK_ROW_NEAR, g.near_lo / near_hi)
cudaError_t fk_launch_fused2d(const FkGrid& g, FkOperator op, const double* Pold, double* Pnew,
                              int chunk0, int chunk1, int n, int N, int sm_count, int line_lo,
                              int line_hi, cudaStream_t s);
cudaError_t fk_fused2d_setup(void);
// slopes of the lines line0 .. line0+nlines-1 (a line = one run of the fastest dimension; J / n[d-1]
// lines in all); apply on the nodes j0 .. j0+jn-1 only (jn = J: all nodes)
cudaError_t fk_launch_slopes(const FkGrid& g, const double* P, double* dP, int n_chunks,
                             int chunk0, int chunk1, int line0, int nlines, cudaStream_t s);
cudaError_t fk_launch_apply(const FkGrid& g, FkOperator op, const double* Pold, const double* dP,
                            double* Pnew, int n_chunks, int chunk0, int chunk1, int n, int N,
                            int far_only, long long j0, long long jn, cudaStream_t s);
// 2-D apply of the rows that are not FK_ROW_NEAR on the lines line0 .. line0+nlines-1, four rows
// adjacent along dimension 1 per warp (fk_far2d.cu); near and Dirichlet rows are left to fk_fused2d
cudaError_t fk_launch_far2d(const FkGrid& g, FkOperator op, const double* Pold, const double* dP,
                            double* Pnew, int n_chunks, int chunk0, int chunk1, int n, int N,
                            int line0, int nlines, cudaStream_t s);
// 3-D apply, four rows adjacent along dimension 2 per warp (fk_rowblock3d.cu); all rows
cudaError_t fk_launch_rowblock3d(const FkGrid& g, FkOperator op, const double* Pold,
                                 const double* dP, double* Pnew, int n_chunks, int chunk0,
                                 int chunk1, int n, int N, cudaStream_t s);
// out[m - m0] = sum_j w[j] P(t_m, x_j) for the owned columns m0 <= m < m1; partial: scratch of
// FK_RED_BLOCKS * 32 doubles per chunk touched
#define FK_RED_BLOCKS 64
cudaError_t fk_launch_reduce(const FkGrid& g, const double* P, const double* w, int m0, int m1,
                             double* partial, double* out, cudaStream_t s);
// the same reduction with the partial sums in a fixed array inside the library image (no allocation):
// at most FK_REDUCE_STATIC_MAX_CHUNKS chunks touched by [m0, m1); `device` must be the current
// device; the first call on a device looks up the array's address on it (fk_kernels.cu)
#define FK_REDUCE_STATIC_MAX_CHUNKS 64   // == FK_REDUCE_STATIC_MAX_CHUNKS_ABI of include/fk.h
cudaError_t fk_launch_reduce_static(const FkGrid& g, const double* P, const double* w, int m0,
                                    int m1, double* out, int device, cudaStream_t s);
cudaError_t fk_launch_gather_columns(const FkGrid& g, const double* P, int m0, int m1,
                                     double* out, cudaStream_t s);

#endif
