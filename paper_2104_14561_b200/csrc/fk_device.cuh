// fk_device.cuh -- device helpers shared by the kernels of the CUDA path (not by oracle/).
#ifndef FK_DEVICE_CUH
#define FK_DEVICE_CUH

#include <cstdint>

#include "fk_internal.h"

namespace fkd {

__device__ __forceinline__ void unravel(const FkGrid& g, long long j, int idx[3]) {
  idx[0] = idx[1] = idx[2] = 0;
  unsigned r = (unsigned)j;                       // J * 32 < 2^31 is checked by fk_create
  for (int k = g.d - 1; k > 0; --k) {
    const unsigned n = (unsigned)g.n[k];
    const unsigned q = r / n;
    idx[k] = (int)(r - q * n);
    r = q;
  }
  idx[0] = (int)r;
}

// node on an ABSORB face?  lowest dimension decides the value (R9)
__device__ __forceinline__ bool dirichlet(const FkGrid& g, const int idx[3], double* val) {
  for (int k = 0; k < g.d; ++k) {
    if (idx[k] == 0 && g.face_kind[k][0] == 0) { *val = g.face_value[k][0]; return true; }
    if (idx[k] == g.n[k] - 1 && g.face_kind[k][1] == 0) { *val = g.face_value[k][1]; return true; }
  }
  return false;
}

// cell c with x[c] <= z < x[c+1], 0 <= c <= n-2 (z == x[n-1] falls in the last cell); z is
// inside [lo, hi] here.  The index is clamped whatever z is, so a NaN coefficient can only
// produce NaN values, never an out-of-range access.
__device__ __forceinline__ int locate(const FkGrid& g, int k, double z) {
  const double* __restrict__ x = g.x[k];
  const int n = g.n[k];
  int c;
  if (g.uniform[k]) {
    c = __double2int_rd((z - g.lo[k]) * g.inv_h0[k]);
    c = max(0, min(c, n - 2));
    while (c > 0 && z < x[c]) --c;
    while (c < n - 2 && z >= x[c + 1]) ++c;
  } else {
    int lo = 0, hi = n - 1;                 // invariant: x[lo] <= z (or lo == 0), z < x[hi] (or hi == n-1)
    while (hi - lo > 1) {
      int mid = (lo + hi) >> 1;
      if (z >= x[mid]) lo = mid; else hi = mid;
    }
    c = min(lo, n - 2);
  }
  return c;
}

// Eq. 21: z_q = (x + b dt) + (sigma sqrt(2 dt)) a_q, products and sums NOT fused
__device__ __forceinline__ double push_point(double centre, double spread, double a) {
  return __dadd_rn(centre, __dmul_rn(spread, a));
}

// Conservative node range [first, last] that the Q_k points of one node can touch along
// dimension k: the cells of the two extreme points (the points are ascending in q because
// sigma >= 0), each projected onto the box.  Used both by the classifier (does a step have rows
// that leave the fused kernel's halo?) and by fk_assemble (the per-row flag), so that the two
// always agree.
__device__ __forceinline__ void reach(const FkGrid& g, int k, double centre, double spread,
                                      int* first, int* last) {
  double z0 = push_point(centre, spread, g.gh_a[k][0]);
  double z1 = push_point(centre, spread, g.gh_a[k][g.Q[k] - 1]);
  z0 = fmin(fmax(z0, g.lo[k]), g.hi[k]);
  z1 = fmin(fmax(z1, g.lo[k]), g.hi[k]);
  *first = locate(g, k, fmin(z0, z1));
  *last = locate(g, k, fmax(z0, z1)) + 1;
}

// 1/s for a normal, finite s: MUFU seed + two Newton steps (error ~1 ulp)
__device__ __forceinline__ double rcp_newton(double s) {
  double r;
  asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(r) : "d"(s));
  double e = fma(-s, r, 1.0);
  r = fma(r, e, r);
  e = fma(-s, r, 1.0);
  r = fma(r, e, r);
  return r;
}

// Eq. 15: 0 if the two divided differences differ in sign or one is 0
// (R7), else their harmonic mean 2ab/(a+b).  p = ab > 0 implies |a+b| >= 2 sqrt(p) is a normal
// number, so the reciprocal needs no special cases; an underflowing product gives slope 0,
// which differs from the exact value by less than 1e-150.
__device__ __forceinline__ double harmonic(double a, double b) {
  const double p = a * b;
  const double r = rcp_newton(a + b);
  return p > 0.0 ? (p + p) * r : 0.0;
}

// One row of A_nu [P; dP] in factored form, contracted one dimension at a time (Eq. 13 with the
// quadrature weights folded in):
//   out = c_j + sum_{i0} [ alpha0 A'(i0) + beta0 B0'(i0) ]
//   A'(i0)  = sum_{i1} [ alpha1 A(i0,i1) + beta1 B1(i0,i1) ],  B0'(i0) = sum_{i1} alpha1 B0(i0,i1)
//   A(i0,i1)  = sum_{i2} [ alpha2 u + beta2 du2 ],  Bk(i0,i1) = sum_{i2} alpha2 du_k
// w / off: the row's entries (alpha, beta) and element offsets; u, d0, d1, d2: the lane's column
// of the chunk (base of the chunk + lane).
template <int D>
__device__ __forceinline__ double contract_row(const FkGrid& g, const double2* __restrict__ w,
                                               const int* __restrict__ off, int4 cnt, double c,
                                               const double* __restrict__ u,
                                               const double* __restrict__ d0,
                                               const double* __restrict__ d1,
                                               const double* __restrict__ d2) {
  double acc = c;
  if (D == 1) {
    double a0 = 0.0, a1 = 0.0;
#pragma unroll 8
    for (int e = 0; e < cnt.x; ++e) {
      const double2 w0 = w[e];
      const int o = off[e];
      a0 = fma(w0.x, u[o], a0);
      a1 = fma(w0.y, d0[o], a1);
    }
    acc += a0 + a1;
  } else if (D == 2) {
    const double2* __restrict__ w1p = w + g.qoff[1];
    const int* __restrict__ o1p = off + g.qoff[1];
    for (int e0 = 0; e0 < cnt.x; ++e0) {
      const double2 w0 = w[e0];
      const int o0 = off[e0];
      double A = 0.0, A2 = 0.0, B0 = 0.0;
#pragma unroll 4
      for (int e1 = 0; e1 < cnt.y; ++e1) {
        const double2 w1 = w1p[e1];
        const int o = o0 + o1p[e1];
        A = fma(w1.x, u[o], A);
        A2 = fma(w1.y, d1[o], A2);
        B0 = fma(w1.x, d0[o], B0);
      }
      acc = fma(w0.x, A + A2, acc);
      acc = fma(w0.y, B0, acc);
    }
  } else {
    const double2* __restrict__ w1p = w + g.qoff[1];
    const int* __restrict__ o1p = off + g.qoff[1];
    const double2* __restrict__ w2p = w + g.qoff[2];
    const int* __restrict__ o2p = off + g.qoff[2];
    for (int e0 = 0; e0 < cnt.x; ++e0) {
      const double2 w0 = w[e0];
      const int o0 = off[e0];
      double Ap = 0.0, B0p = 0.0;
      for (int e1 = 0; e1 < cnt.y; ++e1) {
        const double2 w1 = w1p[e1];
        const int o01 = o0 + o1p[e1];
        double A = 0.0, A2 = 0.0, B0 = 0.0, B1 = 0.0;
#pragma unroll 4
        for (int e2 = 0; e2 < cnt.z; ++e2) {
          const double2 w2 = w2p[e2];
          const int o = o01 + o2p[e2];
          A = fma(w2.x, u[o], A);
          A2 = fma(w2.y, d2[o], A2);
          B0 = fma(w2.x, d0[o], B0);
          B1 = fma(w2.x, d1[o], B1);
        }
        Ap = fma(w1.x, A + A2, Ap);
        Ap = fma(w1.y, B1, Ap);
        B0p = fma(w1.x, B0, B0p);
      }
      acc = fma(w0.x, Ap, acc);
      acc = fma(w0.y, B0p, acc);
    }
  }
  return acc;
}

// R22: weighted harmonic mean a b / (wa b + wb a), wa + wb = 1 the normalised Fritsch-Carlson
// weights attached to a and b (wa = wb = 1/2 is Eq. 15); 0 unless a and b have the same sign.
__device__ __forceinline__ double harmonic_w(double a, double b, double2 w) {
  const double p = a * b;
  const double r = rcp_newton(fma(w.x, b, w.y * a));
  return p > 0.0 ? p * r : 0.0;
}

// global output-time column of lane `lane` of the context's local chunk `chunk` (column sharding)
__device__ __forceinline__ int column_of(const FkGrid& g, int chunk, int lane) {
  return (chunk * g.shard_count + g.shard_index) * FK_CW + lane;
}

// ---- mbarrier / TMA bulk-copy primitives (sm_90+ PTX; SASS: SYNCS.*, UBLKCP)
__device__ __forceinline__ uint32_t smem_u32(const void* p) {
  return (uint32_t)__cvta_generic_to_shared(p);
}
__device__ __forceinline__ void mbar_init(uint64_t* bar, int count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count));
}
__device__ __forceinline__ void mbar_expect_tx(uint64_t* bar, uint32_t bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)),
               "r"(bytes)
               : "memory");
}
__device__ __forceinline__ void bulk_g2s(void* dst, const void* src, uint32_t bytes,
                                         uint64_t* bar) {
  asm volatile(
      "cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::
          "r"(smem_u32(dst)),
      "l"(src), "r"(bytes), "r"(smem_u32(bar))
      : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t* bar, uint32_t parity) {
  asm volatile(
      "{\n"
      ".reg .pred p;\n"
      "WAIT_LOOP:\n"
      "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
      "@p bra WAIT_DONE;\n"
      "bra WAIT_LOOP;\n"
      "WAIT_DONE:\n"
      "}\n" ::"r"(smem_u32(bar)),
      "r"(parity)
      : "memory");
}

}  // namespace fkd

#endif
