// fk_fused2d.cu -- the fused 2-D step kernel: PCHIP slopes (Eq. 15) and the
// row contraction P(:, n:N) <- A_nu [P; dP](:, n:N) in one pass, so that P is
// read once and written once per step (16 B per node-step update) and dP never exists in HBM.
//
// Work decomposition.  Lane = output-time column of a 32-column chunk (as everywhere in this
// library), so a node is one 256-byte row and the operator row is warp-uniform.  A block owns
// a strip of T1 nodes along dimension 1 (the fast one) and marches along dimension 0 over a
// segment of lines.  Shared memory holds a rolling window of lines:
//     u   LBU = 2H+3 lines of T1+2H+2 nodes      (TMA bulk copies, one line ahead)
//     d0  LBD = 2H+1 lines of T1+2H   nodes      (computed once per node of the strip + halo)
//     d1  same
//     rec 2 lines of T1 compact operator records (bulk copy, one line ahead)
// Per output line i0: [prefetch u(i0+H+2), rec(i0+1)] -> contraction of line i0 from shared
// memory -> wait/sync -> slopes of line i0+H+1 -> sync.  Slopes are recomputed only in the
// dimension-1 halo (2H nodes per T1) and in the H0+... lines of a segment's prologue.
//
// Rows whose entries leave the halo (not FK_ROW_NEAR) are skipped here; the host runs the
// generic slopes + apply kernels on them in the same step (fk_api.cu).
#include <cstdint>

#include "fk_device.cuh"

namespace {

constexpr int H = FK_H;
constexpr int LBU = 2 * H + 4;                // resident u lines: i0-H .. i0+H+3
constexpr int LBD = 2 * H + 2;                // resident slope lines: i0-H .. i0+H+1
constexpr int RB = 4;                         // rows per warp: adjacent nodes along dimension 1

template <int T1>
struct Tile {
  static constexpr int W1 = T1 + 2 * H;       // nodes of a slope line
  static constexpr int WU = W1 + 2;           // nodes of a u line
  static constexpr int NWARPS = T1 / RB;      // warps per role: one block of RB rows each
  static constexpr int THREADS = 2 * NWARPS * 32;   // contraction warps + slope warps
  static constexpr size_t U_ELEMS = (size_t)LBU * WU * FK_CW;
  static constexpr size_t D_ELEMS = (size_t)LBD * W1 * FK_CW;
  static constexpr size_t SMEM = (U_ELEMS + 2 * D_ELEMS) * sizeof(double) +
                                 2 * T1 * sizeof(FkRec2) + 48 + (W1 + 4) * sizeof(double);
};

using fkd::smem_u32;
using fkd::mbar_init;
using fkd::mbar_expect_tx;
using fkd::bulk_g2s;
using fkd::mbar_wait;

// position of grid node i1 inside a u line / a slope line of the strip starting at s1
#define FK_UPOS(i1) ((i1) - (s1 - H - 1))
#define FK_DPOS(i1) ((i1) - (s1 - H))

// Slopes of line l (Eq. 15 along both dimensions) for the strip's slope window.  Each warp
// owns NPW = ceil(W1 / NWARPS) consecutive nodes and sweeps them with everything in registers: the
// NPW + 4 values of line l around them give the dimension-1 differences once each, and the
// dimension-0 differences need two more loads per node.  Fully unrolled, so the 2 * NPW
// harmonic means (each a chain of ~10 dependent fp64 operations) overlap.
template <int T1>
__device__ __forceinline__ void slopes_line(const FkGrid& g, const double* __restrict__ su,
                                            double* __restrict__ sd0, double* __restrict__ sd1,
                                            const double* __restrict__ sih, double iha,
                                            double ihb, int l, int s1, int warp, int lane) {
  using T = Tile<T1>;
  constexpr int NPW = (T::W1 + T::NWARPS - 1) / T::NWARPS;
  const int n0 = g.n[0], n1 = g.n[1];
  // the three consecutive lines / nodes whose two divided differences give the slope:
  // (i-1, i, i+1) inside, the first / last three at the ends (R6)
  const int la = min(max(l - 1, 0), n0 - 3);
  const double* __restrict__ ua = su + (((unsigned)la % LBU) * T::WU) * FK_CW + lane;
  const double* __restrict__ ub = su + (((unsigned)(la + 1) % LBU) * T::WU) * FK_CW + lane;
  const double* __restrict__ uc = su + (((unsigned)(la + 2) % LBU) * T::WU) * FK_CW + lane;
  const double* __restrict__ ul = su + (((unsigned)l % LBU) * T::WU) * FK_CW + lane;
  double* __restrict__ o0 = sd0 + (((unsigned)l % LBD) * T::W1) * FK_CW + lane;
  double* __restrict__ o1 = sd1 + (((unsigned)l % LBD) * T::W1) * FK_CW + lane;
  const int p0 = warp * NPW;                       // first slope-window position of this warp
  const int i_first = s1 - H + p0;                 // its grid node
  // values of line l at nodes i_first-2 .. i_first+NPW+1 (u-window positions p0-1 ..), each
  // clamped into the part of the window that exists; clamped duplicates are never selected
  const int wlo = max(0, s1 - H - 1), whi = min(n1, s1 + T1 + H + 1) - 1;
  double v[NPW + 4];
#pragma unroll
  for (int k = 0; k < NPW + 4; ++k) {
    const int i1 = min(max(i_first - 2 + k, wlo), whi);
    v[k] = ul[FK_UPOS(i1) * FK_CW];
  }
  double dl[NPW + 3];                               // dl[k] = difference between v[k+1], v[k]
#pragma unroll
  for (int k = 0; k < NPW + 3; ++k) {
    const int i1 = min(max(i_first - 2 + k, 0), n1 - 2);
    dl[k] = (v[k + 1] - v[k]) * sih[p0 + k];   // 1/h of the cell right of node i_first-2+k
  }
#pragma unroll
  for (int k = 0; k < NPW; ++k) {
    const int i1 = i_first + k;
    if (i1 >= 0 && i1 < n1 && p0 + k < T::W1) {
      // node i1 is v[k+2]; inside: (dl[k+1], dl[k+2]); first node: (dl[k+2], dl[k+3]); last
      // node: (dl[k], dl[k+1])
      const double a = i1 == 0 ? dl[k + 2] : (i1 == n1 - 1 ? dl[k] : dl[k + 1]);
      const double b = i1 == 0 ? dl[k + 3] : (i1 == n1 - 1 ? dl[k + 1] : dl[k + 2]);
      const int pu = FK_UPOS(i1) * FK_CW;
      const double va = ua[pu], vc = uc[pu];
      const double vb = (la + 1 == l) ? v[k + 2] : ub[pu];
      const int pd = (p0 + k) * FK_CW;
      o0[pd] = fkd::harmonic((vb - va) * iha, (vc - vb) * ihb);
      o1[pd] = fkd::harmonic(a, b);
    }
  }
}

// The same for a line 1 <= l <= n0-2 of a strip whose slope window holds no first / last node of
// dimension 1 and lies inside the grid with its +-1 neighbours: no clamps, no end rules, no
// predicates -- straight-line code; ih[k] = 1/h of the cell right of node i_first-2+k is loop
// invariant and lives in registers.
template <int T1>
struct SlopeRegs {
  static constexpr int NPW = (Tile<T1>::W1 + Tile<T1>::NWARPS - 1) / Tile<T1>::NWARPS;
  double ih[NPW + 3];
};
template <int T1>
__device__ __forceinline__ void slopes_line_inner(const double* __restrict__ su,
                                                  double* __restrict__ sd0,
                                                  double* __restrict__ sd1,
                                                  const SlopeRegs<T1>& sr, double iha, double ihb,
                                                  int l, int warp, int lane) {
  using T = Tile<T1>;
  constexpr int NPW = SlopeRegs<T1>::NPW;
  static_assert(NPW * T::NWARPS == T::W1, "every warp owns exactly NPW nodes of the slope window");
  const int p0 = warp * NPW;
  // u-window position of slope-window position p is p + 1
  const double* __restrict__ ua = su + (((unsigned)(l - 1) % LBU) * T::WU + p0 + 1) * FK_CW + lane;
  const double* __restrict__ ul = su + (((unsigned)l % LBU) * T::WU + p0 - 1) * FK_CW + lane;
  const double* __restrict__ uc = su + (((unsigned)(l + 1) % LBU) * T::WU + p0 + 1) * FK_CW + lane;
  double* __restrict__ o0 = sd0 + (((unsigned)l % LBD) * T::W1 + p0) * FK_CW + lane;
  double* __restrict__ o1 = sd1 + (((unsigned)l % LBD) * T::W1 + p0) * FK_CW + lane;
  double v[NPW + 2];                                // nodes i_first-1 .. i_first+NPW
#pragma unroll
  for (int k = 0; k < NPW + 2; ++k) v[k] = ul[(k + 1) * FK_CW];
  double dl[NPW + 1];                               // dl[k]: cell right of node i_first-1+k
#pragma unroll
  for (int k = 0; k < NPW + 1; ++k) dl[k] = (v[k + 1] - v[k]) * sr.ih[k + 1];
#pragma unroll
  for (int k = 0; k < NPW; ++k) {
    const double va = ua[k * FK_CW], vc = uc[k * FK_CW], vb = v[k + 1];
    o0[k * FK_CW] = fkd::harmonic((vb - va) * iha, (vc - vb) * ihb);
    o1[k * FK_CW] = fkd::harmonic(dl[k], dl[k + 1]);
  }
}

// bytes and copies of one u line (nodes of the strip + halo + 1 that exist in the grid)
template <int T1>
__device__ __forceinline__ uint32_t u_line_bytes(const FkGrid& g, int s1) {
  const int a = max(0, s1 - H - 1), b = min(g.n[1], s1 + T1 + H + 1);
  return (uint32_t)(b - a) * FK_CW * sizeof(double);
}
template <int T1>
__device__ __forceinline__ void u_line_copy(const FkGrid& g, const double* __restrict__ Pc,
                                            double* su, int l, int s1, uint64_t* bar) {
  using T = Tile<T1>;
  const int a = max(0, s1 - H - 1);
  bulk_g2s(su + ((size_t)((unsigned)l % LBU) * T::WU + FK_UPOS(a)) * FK_CW,
           Pc + ((size_t)l * g.n[1] + a) * FK_CW, u_line_bytes<T1>(g, s1), bar);
}

// The lines t0 of a group's window that any of its RB rows uses, contracted with the rows'
// dimension-1 weights restricted to the slots TLO..THI (union nodes q = TLO .. RB-1+THI); all
// register indices are static.  Unused slots inside the range hold zero weights.
template <int T1, int TLO, int THI>
__device__ __forceinline__ void contract_lines(const double* __restrict__ su,
                                               const double* __restrict__ sd0,
                                               const FkRec2* __restrict__ rc,
                                               const double2 (&wc)[RB][3], unsigned lines,
                                               int i0, int ucol, int dcol, double (&acc)[RB]) {
  using T = Tile<T1>;
  // the centre slots 1..3 were fetched with the row heads (every variant needs them, and their
  // latency overlaps the mask reduction); the outer slots only where the variant has them
  double2 w1[RB][THI - TLO + 1];
#pragma unroll
  for (int r = 0; r < RB; ++r)
#pragma unroll
    for (int t = TLO; t <= THI; ++t) w1[r][t - TLO] = (t >= 1 && t <= 3) ? wc[r][t - 1] : rc[r].w[1][t];
  int uslot = (unsigned)(i0 + LBU - H) % LBU, dslot = (unsigned)(i0 + LBD - H) % LBD;
  for (int t0 = 0; t0 < FK_NW; ++t0) {
    if ((lines >> t0) & 1u) {
      const double* __restrict__ up = su + (uslot * (T::WU * FK_CW) + ucol);
      const double* __restrict__ d0p = sd0 + (dslot * (T::W1 * FK_CW) + dcol);
      const double* __restrict__ d1p = d0p + T::D_ELEMS;
      double A[RB], A2[RB], B0[RB];
#pragma unroll
      for (int r = 0; r < RB; ++r) A[r] = A2[r] = B0[r] = 0.0;
#pragma unroll
      for (int q = TLO; q < RB + THI; ++q) {
        // no per-node skipping: straight-line code lets the loads and the 3*RB
        // accumulation chains of a line overlap
        const double U = up[q * FK_CW], D0 = d0p[q * FK_CW], D1 = d1p[q * FK_CW];
#pragma unroll
        for (int r = 0; r < RB; ++r) {
          const int t = q - r;
          if (t >= TLO && t <= THI) {
            A[r] = fma(w1[r][t - TLO].x, U, A[r]);
            A2[r] = fma(w1[r][t - TLO].y, D1, A2[r]);
            B0[r] = fma(w1[r][t - TLO].x, D0, B0[r]);
          }
        }
      }
#pragma unroll
      for (int r = 0; r < RB; ++r) {
        const double2 w0 = rc[r].w[0][t0];           // zero if row r does not use the line
        acc[r] = fma(w0.x, A[r] + A2[r], acc[r]);
        acc[r] = fma(w0.y, B0[r], acc[r]);
      }
    }
    uslot = uslot + 1 == LBU ? 0 : uslot + 1;
    dslot = dslot + 1 == LBD ? 0 : dslot + 1;
  }
}

template <int T1>
__global__ void __launch_bounds__(Tile<T1>::THREADS, 2)
fk_fused2d(FkGrid g, const FkRec2* __restrict__ rec, const double* __restrict__ Pold,
           double* __restrict__ Pnew, int chunk0, int n, int N, int nstrips, int seg_len,
           int line_lo, int line_hi) {
  using T = Tile<T1>;
  extern __shared__ __align__(128) unsigned char smem_raw[];
  double* su = reinterpret_cast<double*>(smem_raw);
  double* sd0 = su + T::U_ELEMS;
  double* sd1 = sd0 + T::D_ELEMS;
  FkRec2* srec = reinterpret_cast<FkRec2*>(sd1 + T::D_ELEMS);
  uint64_t* ubar = reinterpret_cast<uint64_t*>(srec + 2 * T1);   // u lines landed
  uint64_t* rbar = ubar + 2;                                      // ubar[2], rbar[2]
  double* sih = reinterpret_cast<double*>(rbar + 2) + 1;          // 1/h table, dimension 1

  // roles: warps 0..NWARPS-1 contract (many registers), NWARPS..2*NWARPS-1 compute slopes and
  // drive the TMA copies (few registers); `warp` is the index inside the role
  const int lane = threadIdx.x;
  const bool contractor = (int)threadIdx.y < T::NWARPS;
  const int warp = contractor ? threadIdx.y : threadIdx.y - T::NWARPS;
  const bool leader = lane == 0 && (int)threadIdx.y == T::NWARPS;
  const int n0 = g.n[0], n1 = g.n[1];
  const int strip = blockIdx.x % nstrips, seg = blockIdx.x / nstrips;
  const int s1 = strip * T1;
  const int L0 = line_lo + seg * seg_len, L1 = min(line_hi, L0 + seg_len);   // output lines of this block
  const int chunk = chunk0 + blockIdx.y;
  const size_t chunk_elems = (size_t)g.J * FK_CW;
  const double* __restrict__ Pc = Pold + (size_t)chunk * chunk_elems;
  double* __restrict__ Pn = Pnew + (size_t)chunk * chunk_elems;
  const int rows = min(T1, n1 - s1);                      // rows of this strip
  const uint32_t rec_bytes = (uint32_t)rows * sizeof(FkRec2);
  const uint32_t ubytes = u_line_bytes<T1>(g, s1);
  const int m = fkd::column_of(g, chunk, lane);
  const bool active = m >= n && m <= N;

  // A last strip that holds nothing but the nodes of an ABSORB face (n1 = k*T1 + 1, e.g. 129 or
  // 257 nodes) has no row to contract: its rows are the constants g (R15), no window is needed.
  if (rows == 1 && s1 == n1 - 1 && g.face_kind[1][1] == 0) {
    if (active)
      for (int i0 = L0 + (int)threadIdx.y; i0 < L1; i0 += 2 * T::NWARPS) {
        const size_t j = (size_t)i0 * n1 + s1;
        Pn[j * FK_CW + lane] = rec[j].c;
      }
    return;
  }

  if (leader) {
    mbar_init(ubar, 1);
    mbar_init(ubar + 1, 1);
    mbar_init(rbar, 1);
    mbar_init(rbar + 1, 1);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  // Window positions that fall outside the grid are never written by the copies or the slope
  // sweep but are read (with zero weights) by the branch-free contraction: clear the window
  // once so that no stale NaN pattern can be multiplied by those zeros.
  {
    double2* z = reinterpret_cast<double2*>(su);
    const int nz = (int)((T::U_ELEMS + 2 * T::D_ELEMS) / 2);
    for (int i = threadIdx.y * FK_CW + threadIdx.x; i < nz; i += T::THREADS)
      z[i] = make_double2(0.0, 0.0);
    // sih[p] = 1/h of the cell right of grid node s1 - H - 2 + p (index clamped to the grid)
    for (int p = threadIdx.y * FK_CW + threadIdx.x; p < T::W1 + 4; p += T::THREADS)
      sih[p] = g.inv_h[1][min(max(s1 - H - 2 + p, 0), g.n[1] - 2)];
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");   // before the TMA writes
  }
  __syncthreads();

  // prologue: u lines L0-H-1 .. L0+H+2 and the records of line L0; slopes of L0-H .. L0+H
  {
    const int a = max(0, L0 - H - 1), b = min(n0, L0 + H + 3);
    if (leader) {
      mbar_expect_tx(ubar, (uint32_t)(b - a) * ubytes);
      for (int l = a; l < b; ++l) u_line_copy<T1>(g, Pc, su, l, s1, ubar);
      mbar_expect_tx(rbar + (L0 & 1), rec_bytes);
      bulk_g2s(srec + (L0 & 1) * T1, rec + (size_t)L0 * n1 + s1, rec_bytes, rbar + (L0 & 1));
    }
    mbar_wait(ubar, 0);
    const int c = max(0, L0 - H), d = min(n0, L0 + H + 1);
    for (int l = c + (contractor ? 0 : 1); l < d; l += 2)    // the two roles share the lines
    {
      const int la = min(max(l - 1, 0), n0 - 3);
      slopes_line<T1>(g, su, sd0, sd1, sih, g.inv_h[0][la], g.inv_h[0][la + 1], l, s1, warp, lane);
    }
    __syncthreads();
  }

  if (!contractor) {
    // ================= slope warps: per line i0, fetch u(i0+H+3) and rec(i0+1), then the
    // slopes of line i0+H+1 (needs u up to i0+H+2, fetched one iteration earlier)
    asm volatile("setmaxnreg.dec.sync.aligned.u32 96;");
    // strips whose slope window (nodes s1-H .. s1+T1+H-1) holds neither end node of dimension 1
    // take the straight-line sweep on every line that is not the first / last of dimension 0
    const bool inner1 = s1 - H >= 1 && s1 + T1 + H - 1 <= n1 - 2;
    SlopeRegs<T1> sr;
#pragma unroll
    for (int k = 0; k < SlopeRegs<T1>::NPW + 3; ++k) sr.ih[k] = sih[warp * SlopeRegs<T1>::NPW + k];
    uint32_t uparity = 1;                                  // bit b: parity to wait for on ubar[b]
    for (int i0 = L0; i0 < L1; ++i0) {
      const bool more = i0 + 1 < L1;                       // a next line exists in this segment
      const int lf = i0 + H + 3;                           // u line to fetch now
      const int ld = i0 + H + 1;                           // slopes of the next line to enter
      // 1/h of the two line gaps around ld, issued before any wait (off the critical path)
      const int lda = min(max(ld - 1, 0), n0 - 3);
      const double iha = g.inv_h[0][lda], ihb = g.inv_h[0][lda + 1];
      // an mbarrier phase must complete before the next one is armed: first wait for
      // u(ld+1), fetched during iteration i0-1, then arm the fetch of u(lf)
      if (more && i0 > L0 && ld + 1 < n0) {
        // two alternating barriers: a barrier is re-armed two iterations after its wait, with
        // a block barrier in between, so no warp can miss a phase
        const int b = (ld + 1) & 1;
        mbar_wait(ubar + b, (uparity >> b) & 1u);
        uparity ^= 1u << b;
      }
      if (leader) {
        if (more && i0 + 2 < L1 && lf < n0) {              // needed by the slopes of iteration i0+1
          mbar_expect_tx(ubar + (lf & 1), ubytes);
          u_line_copy<T1>(g, Pc, su, lf, s1, ubar + (lf & 1));
        }
        if (more) {                                        // barrier (i0+1)&1 was consumed at i0-1
          uint64_t* rb = rbar + ((i0 + 1) & 1);
          mbar_expect_tx(rb, rec_bytes);
          bulk_g2s(srec + ((i0 + 1) & 1) * T1, rec + (size_t)(i0 + 1) * n1 + s1, rec_bytes, rb);
        }
      }
      if (more && ld < n0) {
        if (inner1 && ld >= 1 && ld <= n0 - 2) slopes_line_inner<T1>(su, sd0, sd1, sr, iha, ihb, ld, warp, lane);
        else slopes_line<T1>(g, su, sd0, sd1, sih, iha, ihb, ld, s1, warp, lane);
      }
      asm volatile("bar.sync 1, %0;" ::"n"(T::THREADS) : "memory");
    }
    return;
  }

  // ================= contraction warps
  asm volatile("setmaxnreg.inc.sync.aligned.u32 160;");
  // union node q of a warp's RB rows is grid node s1 + RB*warp - H + q; element offsets of
  // q = 0 inside a u / slope line, made opaque so that they stay in registers
  int ucol = (RB * warp + 1) * FK_CW + lane, dcol = (RB * warp) * FK_CW + lane;
  asm volatile("" : "+r"(ucol), "+r"(dcol));
  uint32_t rparity = 0;                                    // bit b: parity to wait for on rbar[b]

  for (int i0 = L0; i0 < L1; ++i0) {
    mbar_wait(rbar + (i0 & 1), (rparity >> (i0 & 1)) & 1u);   // records of line i0
    rparity ^= 1u << (i0 & 1);

    // ---- contraction of line i0 (Eq. 13 with the quadrature weights folded in).  A warp
    // takes RB adjacent rows; their (2H+1)-node windows along dimension 1 overlap, so every
    // u / d0 / d1 value of the union window is loaded once and used by up to 2H+1 rows.  All
    // register indices are static: slot t of row r is union node q = r + t.
    {
      const FkRec2* __restrict__ rc = srec + (i0 & 1) * T1 + warp * RB;
      double acc[RB];
      double2 wc[RB][3];
      unsigned m1[RB];
      unsigned lines = 0;
      bool store[RB];
#pragma unroll
      for (int r = 0; r < RB; ++r) {
        const bool valid = warp * RB + r < rows;
        // c, flags and both masks of the row in one 16-byte load (FkRec2: c, then the flag word
        // with mask[0] in bits 8-15 and mask[1] in bits 16-23)
        const int4 head = *reinterpret_cast<const int4*>(&rc[r]);
        const int flags = valid ? head.z : 0;
        const bool mine = (flags & (FK_ROW_NEAR | FK_ROW_DIRICHLET)) != 0;
        store[r] = mine && active;
        m1[r] = mine ? ((unsigned)flags >> 16) & 0xffu : 0u;
        lines |= mine ? ((unsigned)flags >> 8) & 0xffu : 0u;
        acc[r] = valid ? __hiloint2double(head.y, head.x) : 0.0;
#pragma unroll
        for (int t = 0; t < 3; ++t) wc[r][t] = rc[r].w[1][t + 1];
      }
      // the masks are the same in every lane; the reductions tell the compiler so (uniform
      // registers, plain branches instead of divergence bookkeeping)
      lines = __reduce_or_sync(0xffffffffu, lines);
      // dimension-1 slots that carry a weight in any of the RB rows pick the variant of the sweep:
      // a group whose points stay within +-1 node reads 6 union nodes per line instead of 8
      unsigned slots = m1[0] | m1[1] | m1[2] | m1[3];
      slots = __reduce_or_sync(0xffffffffu, slots);
      if ((slots & ~0x0eu) == 0) contract_lines<T1, 1, 3>(su, sd0, rc, wc, lines, i0, ucol, dcol, acc);
      else if ((slots & ~0x0fu) == 0) contract_lines<T1, 0, 3>(su, sd0, rc, wc, lines, i0, ucol, dcol, acc);
      else if ((slots & ~0x1eu) == 0) contract_lines<T1, 1, 4>(su, sd0, rc, wc, lines, i0, ucol, dcol, acc);
      else contract_lines<T1, 0, 4>(su, sd0, rc, wc, lines, i0, ucol, dcol, acc);
      double* __restrict__ out = Pn + ((size_t)i0 * n1 + s1 + warp * RB) * FK_CW + lane;
#pragma unroll
      for (int r = 0; r < RB; ++r)
        if (store[r]) out[r * FK_CW] = acc[r];
    }

    asm volatile("bar.sync 1, %0;" ::"n"(T::THREADS) : "memory");
  }
}

}  // namespace

cudaError_t fk_fused2d_setup(void) {
  return cudaFuncSetAttribute(fk_fused2d<16>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                              (int)Tile<16>::SMEM);
}

cudaError_t fk_launch_fused2d(const FkGrid& g, FkOperator op, const double* Pold, double* Pnew,
                              int chunk0, int chunk1, int n, int N, int sm_count, int line_lo,
                              int line_hi, cudaStream_t s) {
  constexpr int T1 = 16;
  const int n1 = g.n[1];
  const int nl = line_hi - line_lo;                         // output lines line_lo .. line_hi-1
  if (nl <= 0) return cudaSuccess;
  const int nstrips = (n1 + T1 - 1) / T1;
  const int nchunks = chunk1 - chunk0;
  // enough blocks for about six waves of two blocks per SM, segments of at least 16 lines
  const long long want = 6LL * 2 * sm_count;
  long long nseg = (want + (long long)nstrips * nchunks - 1) / ((long long)nstrips * nchunks);
  const int max_seg = nl / 16 > 1 ? nl / 16 : 1;
  if (nseg > max_seg) nseg = max_seg;
  if (nseg < 1) nseg = 1;
  const int seg_len = (int)((nl + nseg - 1) / nseg);
  nseg = (nl + seg_len - 1) / seg_len;
  dim3 block(FK_CW, 2 * Tile<T1>::NWARPS), grid((unsigned)(nstrips * nseg), (unsigned)nchunks);
  fk_fused2d<T1><<<grid, block, Tile<T1>::SMEM, s>>>(g, op.rec, Pold, Pnew, chunk0, n, N,
                                                      nstrips, seg_len, line_lo, line_hi);
  return cudaGetLastError();
}
