// fk_fused2d_tmem.cu -- variant of the fused 2-D step kernel (see fk_fused2d.cu for the scheme)
// that keeps the PCHIP slopes d0 / d1 in TENSOR MEMORY instead of shared memory.
//
// Why: the contraction needs one 8-byte operand per FMA and lane; with u, d0 and d1 all in
// shared memory the 128 B/clk/SM of the LSU path is the binding resource.  TMEM is a second,
// independent operand store (tcgen05.ld measured at > 200 B/clk/SM on B200), and its access
// shape 32x32b (thread i of a warp <-> TMEM lane i of the warp's quarter, N consecutive
// 32-bit columns) is exactly this library's layout: lane = output-time column.  A quarter of
// TMEM is private to the warps with the same (warp id mod 4): each contraction warp keeps, in
// its own quarter, the slopes of the 8 nodes its 4 rows can touch for the 6 resident lines.  The
// slope warps compute every slope of the strip once into a two-line shared exchange buffer;
// at the start of the next iteration each contraction warp moves its 8-node window of the new
// line into TMEM (16 LDS + 2 tcgen05.st.x16), and every line body then fetches d0 / d1 with two
// tcgen05.ld.x16 and only u through LDS (a third of the shared-memory operand traffic).
//
// Per block: T1 = 16 rows, 4 contraction + 4 slope warps, 256 TMEM columns (6 line slots x 32
// columns used), shared memory for the rolling u window, the exchange buffer and the records.
// Selected with FK_FUSED2D=tmem; measured on par with the shared-memory variant.
#include <cstdint>

#include "fk_device.cuh"

namespace {

using fkd::bulk_g2s;
using fkd::mbar_expect_tx;
using fkd::mbar_init;
using fkd::mbar_wait;
using fkd::smem_u32;

constexpr int H = FK_H;
constexpr int LBU = 2 * H + 4;      // resident u lines
constexpr int LBD = 2 * H + 2;      // resident slope lines (TMEM slots)
constexpr int RB = 4;               // rows per contraction warp
constexpr int T1 = 16;              // rows per strip
constexpr int NW = T1 / RB;         // warps per role
constexpr int THREADS = 2 * NW * 32;
constexpr int W1 = T1 + 2 * H;
constexpr int WU = W1 + 2;
constexpr int NQ = RB + FK_NW - 1;  // union nodes of a contraction warp (8)
constexpr int TMEM_COLS = 256;      // power of two >= LBD * NQ * 2 fields * 2 words
constexpr size_t U_ELEMS = (size_t)LBU * WU * FK_CW;
constexpr size_t X_LINE = (size_t)2 * W1 * FK_CW;    // slopes of one line: [field][node][lane]
constexpr size_t X_ELEMS = 2 * X_LINE;               // exchange buffer, two lines (by line parity)
constexpr int NIH = W1 + 4;                          // 1/h table of the strip (dimension 1)
constexpr size_t SMEM_BYTES = (U_ELEMS + X_ELEMS + NIH) * sizeof(double) + 2 * T1 * sizeof(FkRec2) + 48;
static_assert(LBD * NQ * 4 <= TMEM_COLS, "slope slots must fit the TMEM allocation");

#define FK_UPOS(i1) ((i1) - (s1 - H - 1))

__device__ __forceinline__ void tmem_st16(uint32_t taddr, const double (&v)[8]) {
  asm volatile(
      "tcgen05.st.sync.aligned.32x32b.x16.b32 [%0], {%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,"
      "%14,%15,%16};" ::"r"(taddr),
      "r"(__double2loint(v[0])), "r"(__double2hiint(v[0])), "r"(__double2loint(v[1])),
      "r"(__double2hiint(v[1])), "r"(__double2loint(v[2])), "r"(__double2hiint(v[2])),
      "r"(__double2loint(v[3])), "r"(__double2hiint(v[3])), "r"(__double2loint(v[4])),
      "r"(__double2hiint(v[4])), "r"(__double2loint(v[5])), "r"(__double2hiint(v[5])),
      "r"(__double2loint(v[6])), "r"(__double2hiint(v[6])), "r"(__double2loint(v[7])),
      "r"(__double2hiint(v[7]))
      : "memory");
}

__device__ __forceinline__ void tmem_ld16(uint32_t taddr, uint32_t (&r)[16]) {
  asm volatile(
      "tcgen05.ld.sync.aligned.32x32b.x16.b32 {%0,%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,"
      "%15}, [%16];"
      : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]),
        "=r"(r[7]), "=r"(r[8]), "=r"(r[9]), "=r"(r[10]), "=r"(r[11]), "=r"(r[12]), "=r"(r[13]),
        "=r"(r[14]), "=r"(r[15])
      : "r"(taddr)
      : "memory");
}

// Slopes of line l: the four slope warps split the strip's W1 = 20 slope nodes, five consecutive
// nodes each, everything in registers (as in fk_fused2d.cu), and put d0 / d1 into the exchange
// buffer sx[field][node][lane] of the line.  Positions outside the grid stay zero (the buffer is
// cleared once).
__device__ __forceinline__ void slopes_to_smem(const FkGrid& g, const double* __restrict__ su,
                                               double* __restrict__ sx,
                                               const double* __restrict__ sih, double iha,
                                               double ihb, int l, int s1, int w, int lane) {
  constexpr int NPW = W1 / NW;
  static_assert(NPW * NW == W1, "slope window must split evenly");
  const int n0 = g.n[0], n1 = g.n[1];
  const int la = min(max(l - 1, 0), n0 - 3);
  const double* __restrict__ ua = su + (((unsigned)la % LBU) * WU) * FK_CW + lane;
  const double* __restrict__ ub = su + (((unsigned)(la + 1) % LBU) * WU) * FK_CW + lane;
  const double* __restrict__ uc = su + (((unsigned)(la + 2) % LBU) * WU) * FK_CW + lane;
  const double* __restrict__ ul = su + (((unsigned)l % LBU) * WU) * FK_CW + lane;
  const int wlo = max(0, s1 - H - 1), whi = min(n1, s1 + T1 + H + 1) - 1;
  const int p0 = w * NPW;
  const int i_first = s1 - H + p0;
  double v[NPW + 4];
#pragma unroll
  for (int k = 0; k < NPW + 4; ++k) {
    const int i1 = min(max(i_first - 2 + k, wlo), whi);
    v[k] = ul[FK_UPOS(i1) * FK_CW];
  }
  double dl[NPW + 3];
#pragma unroll
  for (int k = 0; k < NPW + 3; ++k) {
    const int i1 = min(max(i_first - 2 + k, 0), n1 - 2);
    dl[k] = (v[k + 1] - v[k]) * sih[p0 + k];           // 1/h of the cell right of node i_first-2+k
  }
#pragma unroll
  for (int k = 0; k < NPW; ++k) {
    const int i1 = i_first + k;
    if (i1 >= 0 && i1 < n1) {
      const double a = i1 == 0 ? dl[k + 2] : (i1 == n1 - 1 ? dl[k] : dl[k + 1]);
      const double b = i1 == 0 ? dl[k + 3] : (i1 == n1 - 1 ? dl[k + 1] : dl[k + 2]);
      const int pu = FK_UPOS(i1) * FK_CW;
      const double va = ua[pu], vc = uc[pu];
      const double vb = (la + 1 == l) ? v[k + 2] : ub[pu];
      sx[(p0 + k) * FK_CW + lane] = fkd::harmonic((vb - va) * iha, (vc - vb) * ihb);
      sx[(W1 + p0 + k) * FK_CW + lane] = fkd::harmonic(a, b);
    }
  }
}

// Contraction warp w copies the slopes of the 8 nodes its rows can touch (slope-window positions
// 4w .. 4w+7) from the exchange buffer into the TMEM slot of the line: columns [4q, 4q+1] = d0,
// [4q+2, 4q+3] = d1.  Only this warp ever reads the slot, so no cross-warp TMEM fence is needed.
__device__ __forceinline__ void slopes_smem_to_tmem(const double* __restrict__ sx, uint32_t tslot,
                                                    int w, int lane) {
#pragma unroll
  for (int half = 0; half < 2; ++half) {
    double out[8];
#pragma unroll
    for (int k = 0; k < 4; ++k) {
      const int p = RB * w + 4 * half + k;
      out[2 * k] = sx[p * FK_CW + lane];
      out[2 * k + 1] = sx[(W1 + p) * FK_CW + lane];
    }
    tmem_st16(tslot + 16 * half, out);
  }
  asm volatile("tcgen05.wait::st.sync.aligned;" ::: "memory");
}

__device__ __forceinline__ void u_line_copy(const FkGrid& g, const double* __restrict__ Pc,
                                            double* su, int l, int s1, uint32_t bytes,
                                            uint64_t* bar) {
  const int a = max(0, s1 - H - 1);
  bulk_g2s(su + ((size_t)((unsigned)l % LBU) * WU + FK_UPOS(a)) * FK_CW,
           Pc + ((size_t)l * g.n[1] + a) * FK_CW, bytes, bar);
}


__global__ void __launch_bounds__(THREADS, 2)
fk_fused2d_tmem(FkGrid g, const FkRec2* __restrict__ rec, const double* __restrict__ Pold,
                double* __restrict__ Pnew, int chunk0, int n, int N, int nstrips, int seg_len) {
  extern __shared__ __align__(128) unsigned char smem_raw[];
  double* su = reinterpret_cast<double*>(smem_raw);
  double* sx = su + U_ELEMS;
  double* sih = sx + X_ELEMS;
  FkRec2* srec = reinterpret_cast<FkRec2*>(sih + NIH);
  uint64_t* ubar = reinterpret_cast<uint64_t*>(srec + 2 * T1);
  uint64_t* rbar = ubar + 2;                               // ubar[2], rbar[2]
  uint32_t* tbase_smem = reinterpret_cast<uint32_t*>(rbar + 2);

  const int lane = threadIdx.x;
  const bool contractor = (int)threadIdx.y < NW;
  const int warp = contractor ? threadIdx.y : threadIdx.y - NW;   // = TMEM quarter of the pair
  const bool leader = lane == 0 && (int)threadIdx.y == NW;
  const int n0 = g.n[0], n1 = g.n[1];
  const int strip = blockIdx.x % nstrips, seg = blockIdx.x / nstrips;
  const int s1 = strip * T1;
  const int L0 = seg * seg_len, L1 = min(n0, L0 + seg_len);
  const int chunk = chunk0 + blockIdx.y;
  const size_t chunk_elems = (size_t)g.J * FK_CW;
  const double* __restrict__ Pc = Pold + (size_t)chunk * chunk_elems;
  double* __restrict__ Pn = Pnew + (size_t)chunk * chunk_elems;
  const int rows = min(T1, n1 - s1);
  const uint32_t rec_bytes = (uint32_t)rows * sizeof(FkRec2);
  const uint32_t ubytes =
      (uint32_t)(min(n1, s1 + T1 + H + 1) - max(0, s1 - H - 1)) * FK_CW * sizeof(double);
  const int m = chunk * FK_CW + lane;
  const bool active = m >= n && m <= N;

  if (leader) {
    mbar_init(ubar, 1);
    mbar_init(ubar + 1, 1);
    mbar_init(rbar, 1);
    mbar_init(rbar + 1, 1);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  if (threadIdx.y == 0) {                                  // one warp allocates the block's TMEM
    asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(
                     smem_u32(tbase_smem)),
                 "n"(TMEM_COLS)
                 : "memory");
    asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
  }
  {  // clear the u window: positions outside the grid are read with zero weights
    double2* z = reinterpret_cast<double2*>(su);
    for (int i = threadIdx.y * FK_CW + threadIdx.x; i < (int)((U_ELEMS + X_ELEMS) / 2); i += THREADS)
      z[i] = make_double2(0.0, 0.0);
    // sih[p] = 1/h of the cell right of grid node s1 - H - 2 + p (index clamped to the grid)
    for (int p = threadIdx.y * FK_CW + threadIdx.x; p < NIH; p += THREADS)
      sih[p] = g.inv_h[1][min(max(s1 - H - 2 + p, 0), g.n[1] - 2)];
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
  }
  asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
  __syncthreads();
  asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
  const uint32_t tq = *tbase_smem + ((uint32_t)(warp * 32) << 16);   // this pair's quarter

  if (!contractor) {
    // ================= slope warps
    asm volatile("setmaxnreg.dec.sync.aligned.u32 88;");
    {  // prologue: u lines L0-H-1 .. L0+H+2, records of L0, slopes of L0-H .. L0+H
      const int a = max(0, L0 - H - 1), b = min(n0, L0 + H + 3);
      if (leader) {
        mbar_expect_tx(ubar, (uint32_t)(b - a) * ubytes);
        for (int l = a; l < b; ++l) u_line_copy(g, Pc, su, l, s1, ubytes, ubar);
        mbar_expect_tx(rbar + (L0 & 1), rec_bytes);
        bulk_g2s(srec + (L0 & 1) * T1, rec + (size_t)L0 * n1 + s1, rec_bytes, rbar + (L0 & 1));
      }
      mbar_wait(ubar, 0);
      // slopes of lines L0-H .. L0+H, one line per round: the slope warps fill the exchange
      // buffer of line l while the contraction warps move line l-1 into TMEM
      const int c = max(0, L0 - H), d = min(n0, L0 + H + 1);
      for (int l = c; l <= d; ++l) {
        if (l < d) {
          const int la = min(max(l - 1, 0), n0 - 3);
          slopes_to_smem(g, su, sx + (l & 1) * X_LINE, sih, g.inv_h[0][la], g.inv_h[0][la + 1], l,
                         s1, warp, lane);
        }
        asm volatile("bar.sync 1, %0;" ::"n"(THREADS) : "memory");
      }
    }
    uint32_t uparity = 1;                                  // bit b: parity to wait for on ubar[b]
    for (int i0 = L0; i0 < L1; ++i0) {
      const bool more = i0 + 1 < L1;
      const int lf = i0 + H + 3, ld = i0 + H + 1;
      // 1/h of the two line gaps around ld: issued before any wait so that the (L2) latency
      // of these two loads is off the critical path
      const int lda = min(max(ld - 1, 0), n0 - 3);
      const double iha = g.inv_h[0][lda], ihb = g.inv_h[0][lda + 1];
      if (more && i0 > L0 && ld + 1 < n0) {                // u(ld+1), fetched at iteration i0-1
        // two alternating barriers: a barrier is re-armed two iterations after its wait, with
        // a block barrier in between, so no warp can miss a phase
        const int b = (ld + 1) & 1;
        mbar_wait(ubar + b, (uparity >> b) & 1u);
        uparity ^= 1u << b;
      }
      if (leader) {
        if (more && i0 + 2 < L1 && lf < n0) {
          mbar_expect_tx(ubar + (lf & 1), ubytes);
          u_line_copy(g, Pc, su, lf, s1, ubytes, ubar + (lf & 1));
        }
        if (more) {
          uint64_t* rb = rbar + ((i0 + 1) & 1);
          mbar_expect_tx(rb, rec_bytes);
          bulk_g2s(srec + ((i0 + 1) & 1) * T1, rec + (size_t)(i0 + 1) * n1 + s1, rec_bytes, rb);
        }
      }
      if (more && ld < n0)
        slopes_to_smem(g, su, sx + (ld & 1) * X_LINE, sih, iha, ihb, ld, s1, warp, lane);
      asm volatile("bar.sync 1, %0;" ::"n"(THREADS) : "memory");
    }
    return;
  }

  // ================= contraction warps
  asm volatile("setmaxnreg.inc.sync.aligned.u32 168;");
  {  // prologue rounds (see the slope warps): line l-1 goes to TMEM while line l is computed
    const int c = max(0, L0 - H), d = min(n0, L0 + H + 1);
    for (int l = c; l <= d; ++l) {
      if (l > c)
        slopes_smem_to_tmem(sx + ((l - 1) & 1) * X_LINE, tq + ((unsigned)(l - 1) % LBD) * 32, warp,
                            lane);
      asm volatile("bar.sync 1, %0;" ::"n"(THREADS) : "memory");
    }
  }
  int ucol = (RB * warp + 1) * FK_CW + lane;
  asm volatile("" : "+r"(ucol));
  uint32_t rparity = 0;

  for (int i0 = L0; i0 < L1; ++i0) {
    // slopes of line i0+H, written to the exchange buffer during iteration i0-1
    if (i0 > L0 && i0 + H < n0)
      slopes_smem_to_tmem(sx + ((i0 + H) & 1) * X_LINE, tq + ((unsigned)(i0 + H) % LBD) * 32, warp,
                          lane);
    mbar_wait(rbar + (i0 & 1), (rparity >> (i0 & 1)) & 1u);
    rparity ^= 1u << (i0 & 1);
    {
      const FkRec2* __restrict__ rc = srec + (i0 & 1) * T1 + warp * RB;
      double2 w1[RB][FK_NW];
      double acc[RB];
      unsigned lines = 0;
      bool store[RB];
#pragma unroll
      for (int r = 0; r < RB; ++r) {
        const bool valid = warp * RB + r < rows;
        const int flags = valid ? rc[r].flags : 0;
        const bool mine = (flags & (FK_ROW_NEAR | FK_ROW_DIRICHLET)) != 0;
        store[r] = mine && active;
        lines |= mine ? (unsigned)rc[r].mask[0] : 0u;
        acc[r] = valid ? rc[r].c : 0.0;
#pragma unroll
        for (int t = 0; t < FK_NW; ++t)
          w1[r][t] = mine ? rc[r].w[1][t] : make_double2(0.0, 0.0);
      }
      lines = __reduce_or_sync(0xffffffffu, lines);
      int uslot = (unsigned)(i0 + LBU - H) % LBU, dslot = (unsigned)(i0 + LBD - H) % LBD;
      for (int t0 = 0; t0 < FK_NW; ++t0) {
        if ((lines >> t0) & 1u) {
          uint32_t dr[2][16];
          tmem_ld16(tq + dslot * 32, dr[0]);
          tmem_ld16(tq + dslot * 32 + 16, dr[1]);
          const double* __restrict__ up = su + (uslot * (WU * FK_CW) + ucol);
          double U[NQ];
#pragma unroll
          for (int q = 0; q < NQ; ++q) U[q] = up[q * FK_CW];
          asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
          double A[RB], A2[RB], B0[RB];
#pragma unroll
          for (int r = 0; r < RB; ++r) A[r] = A2[r] = B0[r] = 0.0;
#pragma unroll
          for (int q = 0; q < NQ; ++q) {
            const uint32_t* w = dr[q >> 2] + 4 * (q & 3);
            const double D0 = __hiloint2double((int)w[1], (int)w[0]);
            const double D1 = __hiloint2double((int)w[3], (int)w[2]);
#pragma unroll
            for (int r = 0; r < RB; ++r) {
              const int t = q - r;
              if (t >= 0 && t < FK_NW) {
                A[r] = fma(w1[r][t].x, U[q], A[r]);
                A2[r] = fma(w1[r][t].y, D1, A2[r]);
                B0[r] = fma(w1[r][t].x, D0, B0[r]);
              }
            }
          }
#pragma unroll
          for (int r = 0; r < RB; ++r) {
            const double2 w0 = rc[r].w[0][t0];
            acc[r] = fma(w0.x, A[r] + A2[r], acc[r]);
            acc[r] = fma(w0.y, B0[r], acc[r]);
          }
        }
        uslot = uslot + 1 == LBU ? 0 : uslot + 1;
        dslot = dslot + 1 == LBD ? 0 : dslot + 1;
      }
      double* __restrict__ out = Pn + ((size_t)i0 * n1 + s1 + warp * RB) * FK_CW + lane;
#pragma unroll
      for (int r = 0; r < RB; ++r)
        if (store[r]) out[r * FK_CW] = acc[r];
    }
    asm volatile("bar.sync 1, %0;" ::"n"(THREADS) : "memory");
  }
  if (threadIdx.y == 0)
    asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(*tbase_smem),
                 "n"(TMEM_COLS)
                 : "memory");
}

}  // namespace

cudaError_t fk_fused2d_tmem_setup(void) {
  return cudaFuncSetAttribute(fk_fused2d_tmem, cudaFuncAttributeMaxDynamicSharedMemorySize,
                              (int)SMEM_BYTES);
}

cudaError_t fk_launch_fused2d_tmem(const FkGrid& g, FkOperator op, const double* Pold,
                                   double* Pnew, int chunk0, int chunk1, int n, int N,
                                   int sm_count, cudaStream_t s) {
  const int n0 = g.n[0], n1 = g.n[1];
  const int nstrips = (n1 + T1 - 1) / T1;
  const int nchunks = chunk1 - chunk0;
  const long long want = 6LL * 2 * sm_count;
  long long nseg = (want + (long long)nstrips * nchunks - 1) / ((long long)nstrips * nchunks);
  const int max_seg = n0 / 16 > 1 ? n0 / 16 : 1;
  if (nseg > max_seg) nseg = max_seg;
  if (nseg < 1) nseg = 1;
  const int seg_len = (int)((n0 + nseg - 1) / nseg);
  nseg = (n0 + seg_len - 1) / seg_len;
  dim3 block(FK_CW, 2 * NW), grid((unsigned)(nstrips * nseg), (unsigned)nchunks);
  fk_fused2d_tmem<<<grid, block, SMEM_BYTES, s>>>(g, op.rec, Pold, Pnew, chunk0, n, N, nstrips,
                                                  seg_len);
  return cudaGetLastError();
}
