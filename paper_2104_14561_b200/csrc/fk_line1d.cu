// fk_line1d.cu -- Algorithm 1 for 1-D problems, many steps per launch.
//
// The output-time columns never interact (Eq. 29), and a 1-D line of J nodes is
// small: a block owns a group of CG columns and keeps their whole line -- u, its Eq.-15 slopes du
// and the next state -- in shared memory across ALL the steps of a batch (J x CG x 24 bytes).  Per
// step it (i) recomputes the slopes (end nodes by R6), (ii) applies the rows of
// A_nu: a warp takes a row, its lanes are CG columns x 32/CG entry slices, and the
// slices are combined with shuffles.  Nothing goes back to HBM / L2 between steps and there is one
// launch per batch instead of two per step: several operators per pass over P (SURVEY.md section
// 8(f), temporal blocking).  The operators of a batch are assembled beforehand by one launch of
// fk_assemble_batch (fk_kernels.cu); an autonomous problem has a single operator.
// Opt-in (FK_FLAG_MULTISTEP).  Measured on the B200: config 1 (201 nodes) 2.2 ms against 2.9 ms
// step by step, config 2 (1025 nodes) 81 ms against 39 ms -- a column needs its steps one after
// the other, so the block that owns the last columns walks all N steps alone on its SM, one row's
// chain of dependent loads (operator row from L2, then shared memory) at a time, while the
// step-by-step kernels spread every step over all SMs.
//
// A column m is updated by the steps n <= m only (Algorithm 1's shrinking column range): a block
// skips the steps before its last column becomes active, lanes of columns that are not active yet
// keep chi.
#include "fk_device.cuh"

namespace {

constexpr int TH = 512;                    // threads per block

template <int CG>
__global__ void __launch_bounds__(TH, 1)
fk_line1d(FkGrid g, FkOperator op, int nsteps, int n_hi, int autonomous, double* __restrict__ Pa,
          double* __restrict__ Pb, int N) {
  extern __shared__ __align__(16) double sm1d[];
  constexpr int GPC = FK_CW / CG;          // column groups per chunk = entry slices per warp
  const int J = (int)g.J;
  const int chunk = blockIdx.x / GPC, sub = blockIdx.x - chunk * GPC;
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int cc = lane % CG, slice = lane / CG;
  const int m0 = fkd::column_of(g, chunk, sub * CG);            // first column of the group
  const int m_last = min(m0 + CG - 1, N);
  const int n_lo = n_hi - nsteps;                                // steps n = n_hi .. n_lo + 1
  if (m_last < n_lo + 1) return;                                 // no column of the group is touched
  double* u = sm1d;
  double* du = u + (size_t)J * CG;
  double* un = du + (size_t)J * CG;
  const size_t cbase = (size_t)chunk * J * FK_CW + sub * CG;
  for (int i = tid; i < J * CG; i += TH) {
    const int j = i / CG, c = i - j * CG;
    u[i] = Pa[cbase + (size_t)j * FK_CW + c];
  }
  __syncthreads();
  const double* __restrict__ ih = g.inv_h[0];
  const int m = m0 + cc;
  for (int s = 0; s < nsteps; ++s) {
    const int n = n_hi - s;
    if (m_last < n) continue;                                    // block-uniform
    // ---- slopes of every node (Eq. 15; the first / last node use the first / last two cells)
    for (int i = tid; i < J * CG; i += TH) {
      const int j = i / CG, c = i - j * CG;
      const int la = min(max(j - 1, 0), J - 3);
      const double va = u[la * CG + c], vb = u[(la + 1) * CG + c], vc = u[(la + 2) * CG + c];
      du[i] = fkd::harmonic((vb - va) * ih[la], (vc - vb) * ih[la + 1]);
    }
    __syncthreads();
    // ---- rows of A_nu (batch slot s; an autonomous problem has slot 0 only)
    const size_t slot = autonomous ? 0 : (size_t)s;
    const double2* __restrict__ W = op.w + slot * (size_t)J * g.RS;
    const int* __restrict__ O = op.off + slot * (size_t)J * g.RS;
    const int* __restrict__ C = op.cnt + slot * (size_t)J * 4;
    const double* __restrict__ K = op.c + slot * (size_t)J;
    const bool active = m >= n && m <= N;
    for (int j = warp; j < J; j += TH / 32) {
      const int4 cnt = *reinterpret_cast<const int4*>(C + (size_t)j * 4);
      if (cnt.w & FK_ROW_DIRICHLET) {                            // keeps g (R15)
        if (slice == 0) un[j * CG + cc] = u[j * CG + cc];
        continue;
      }
      const double2* __restrict__ w = W + (size_t)j * g.RS;
      const int* __restrict__ o = O + (size_t)j * g.RS;
      double a0 = 0.0, a1 = 0.0;
#pragma unroll 4
      for (int e = slice; e < cnt.x; e += GPC) {
        const double2 we = w[e];
        const int q = (o[e] / FK_CW) * CG + cc;
        a0 = fma(we.x, u[q], a0);
        a1 = fma(we.y, du[q], a1);
      }
      double acc = a0 + a1;
#pragma unroll
      for (int d = CG; d < 32; d <<= 1) acc += __shfl_xor_sync(0xffffffffu, acc, d);
      if (slice == 0) un[j * CG + cc] = active ? K[j] + acc : u[j * CG + cc];
    }
    __syncthreads();
    double* t = u; u = un; un = t;
  }
  for (int i = tid; i < J * CG; i += TH) {                        // both buffers: the parity of the
    const int j = i / CG, c = i - j * CG;                         // host's buffer index is then moot
    const size_t at = cbase + (size_t)j * FK_CW + c;
    const int mc = m0 + c;
    if (mc >= n_lo + 1 && mc <= N) { Pa[at] = u[i]; Pb[at] = u[i]; }
  }
}

}  // namespace

// shared memory of one block for column groups of cg columns
size_t fk_line1d_smem(const FkGrid& g, int cg) { return (size_t)3 * g.J * cg * sizeof(double); }

// column-group width to use on this grid (8 or 4), 0 if its lines do not fit shared memory
int fk_line1d_group(const FkGrid& g, size_t smem_limit) {
  if (g.d != 1 || g.general_slopes || g.J < 3) return 0;
  if (fk_line1d_smem(g, 8) <= smem_limit) return 8;
  if (fk_line1d_smem(g, 4) <= smem_limit) return 4;
  return 0;
}

cudaError_t fk_line1d_setup(const FkGrid& g, int cg) {
  const int bytes = (int)fk_line1d_smem(g, cg);
  return cg == 8 ? cudaFuncSetAttribute(fk_line1d<8>, cudaFuncAttributeMaxDynamicSharedMemorySize, bytes)
                 : cudaFuncSetAttribute(fk_line1d<4>, cudaFuncAttributeMaxDynamicSharedMemorySize, bytes);
}

cudaError_t fk_launch_line1d(const FkGrid& g, FkOperator op, int cg, int nsteps, int n_hi,
                             int autonomous, double* Pcur, double* Pother, int n_chunks, int N,
                             cudaStream_t s) {
  const unsigned blocks = (unsigned)(n_chunks * (FK_CW / cg));
  const size_t smem = fk_line1d_smem(g, cg);
  // the shared-memory limit is an attribute of the FUNCTION, shared by every context of the process:
  // another context with a shorter line may have lowered it since this one was created
  const cudaError_t e = fk_line1d_setup(g, cg);
  if (e != cudaSuccess) return e;
  if (cg == 8) fk_line1d<8><<<blocks, TH, smem, s>>>(g, op, nsteps, n_hi, autonomous, Pcur, Pother, N);
  else fk_line1d<4><<<blocks, TH, smem, s>>>(g, op, nsteps, n_hi, autonomous, Pcur, Pother, N);
  return cudaGetLastError();
}
