// fk_api.cu -- the C ABI of include/fk.h: validation, Gauss-Hermite tables, device state and
// the loop of Algorithm 1.  All arithmetic of the path runs in the kernels
// of fk_kernels.cu; this file only orders them on the caller's stream.
#include "../../include/fk.h"
#include "fk_internal.h"

#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <new>
#include <string>
#include <vector>

namespace {

thread_local std::string g_create_error;

struct EventPair { cudaEvent_t a, b; int cls; };

}  // namespace

struct fk_ctx {
  FkGrid g;
  int N = 0, slots = 0, device = 0;
  int n_chunks = 0;                    // chunks this context owns (all of them unless sharded)
  long long n_updated = 0;             // nodes that are not on an ABSORB face
  bool fused2d = false;                // 2-D: near rows go through fk_fused2d (else generic only)
  int line1d_cg = 0;                   // 1-D: column-group width of the multi-step kernel, 0 = step by step
  int batch_cap = 0;                   // ... operators its batch storage holds
  FkOperator opb = {nullptr, nullptr, nullptr, nullptr, nullptr};   // ... the batch storage
  double2* d_wgt[3] = {nullptr, nullptr, nullptr};
  double* d_red = nullptr;             // fk_reduce: weights [J], partial sums, result
  size_t red_bytes = 0;
  cudaStream_t stream = nullptr;
  double* d_x[3] = {nullptr, nullptr, nullptr};
  double* d_invh[3] = {nullptr, nullptr, nullptr};
  double* d_coef = nullptr;            // [slots][2][d][J]: b then sigma per slot
  std::vector<int> slot_step;          // step held by each slot, -2 = empty
  bool autonomous = false;
  bool auto_assembled = false;         // autonomous: A is the same every step and sits in op[0]
  int auto_nu = 0;                     // ... assembled (and counted in d_work) under this step index
  double* d_P[2] = {nullptr, nullptr};  // both point FK_GUARD_ROWS rows into their allocations
  void* raw_P[2] = {nullptr, nullptr};
  void* raw_dP = nullptr;
  int cur = 0;                         // buffer holding the current state
  double* d_dP = nullptr;
  // the operator of step nu is assembled on a side stream while the kernels of step nu+1 run:
  // two operator buffers (by parity of n), ready / free events between the two streams
  FkOperator op[2] = {{nullptr, nullptr, nullptr, nullptr, nullptr},
                      {nullptr, nullptr, nullptr, nullptr, nullptr}};
  cudaStream_t side = nullptr;
  cudaEvent_t ev_ready[2] = {nullptr, nullptr}, ev_free[2] = {nullptr, nullptr}, ev_coef = nullptr;
  cudaEvent_t ev_status = nullptr;     // recorded behind every queued refresh of h_status
  bool status_pending = false;         // ... one such refresh may still be in flight
  unsigned long long* d_work = nullptr; // [N][4] per step: rows / sum prod D_k, near and other (fk_assemble)
  double class_updates[FK_K_COUNT] = {0, 0, 0, 0, 0, 0, 0};   // node-step updates per kernel class
  unsigned long long* d_paths = nullptr; // FK_FLAG_COUNT_PATHS: FK_PATH_COUNT counters (== g.paths)
  int* d_status = nullptr;             // device status word: FK_BAD_* bits raised by fk_assemble
  int* h_status = nullptr;             // pinned host copy, refreshed at the end of every fk_evolve
  int* d_far = nullptr;                // [slots] rows per loaded step that leave the fused halo
  std::vector<int> h_far;              // host copy, valid when far_valid
  int* d_far_line = nullptr;           // [slots][n0] far rows per line of each loaded step
  std::vector<int> h_far_line;         // host copy, valid when far_valid
  bool far_valid = false;
  int sm_count = 148;
  double* d_stage = nullptr;           // fk_read staging for host destinations
  size_t stage_bytes = 0;
  int n_next = 0;                      // the n the next fk_evolve must start from
  long long launches = 0;
  bool profiling = false;
  std::vector<EventPair> events;
  std::vector<EventPair> event_pool;
  std::string err;
};

namespace {

int fail(fk_ctx* c, int code, const std::string& msg) {
  if (c) c->err = msg; else g_create_error = msg;
  return code;
}

int cuda_fail(fk_ctx* c, cudaError_t e, const char* what) {
  return fail(c, e == cudaErrorMemoryAllocation ? FK_ENOMEM : FK_ECUDA,
              std::string(what) + ": " + cudaGetErrorString(e));
}

// every entry point runs on the context's device and leaves the caller's current device alone
struct DeviceGuard {
  int prev = -1;
  explicit DeviceGuard(int dev) {
    if (cudaGetDevice(&prev) != cudaSuccess) prev = -1;
    if (prev != dev) cudaSetDevice(dev);
  }
  ~DeviceGuard() { if (prev >= 0) cudaSetDevice(prev); }
};

#define FK_CUDA(c, call)                                       \
  do {                                                         \
    cudaError_t e_ = (call);                                   \
    if (e_ != cudaSuccess) return cuda_fail((c), e_, #call);   \
  } while (0)

// ------------------------------------------------------------------------------------------
// Gauss-Hermite rule for the density pi^{-1/2} exp(-xi^2) by Golub-Welsch:
// the nodes are the eigenvalues of the Jacobi matrix with zero diagonal and off-diagonal
// sqrt(k/2), found by Sturm-sequence bisection and polished by Newton on the orthonormal
// polynomial p_Q; the weights are the Christoffel numbers 1 / sum_{k<Q} p_k(a)^2, which sum
// to 1 for this (normalised) density.
// ------------------------------------------------------------------------------------------
void orthonormal_hermite(int Q, long double x, long double* p /*Q+1*/) {
  p[0] = 1.0L;
  if (Q >= 1) p[1] = x * std::sqrt(2.0L);
  for (int k = 1; k < Q; ++k)
    p[k + 1] = (x * p[k] - std::sqrt(k / 2.0L) * p[k - 1]) / std::sqrt((k + 1) / 2.0L);
}

int sturm_count(int Q, long double x) {  // eigenvalues of the Jacobi matrix below x
  int count = 0;
  long double q = -x;
  if (q < 0) ++count;
  for (int k = 1; k < Q; ++k) {
    long double off2 = k / 2.0L;
    if (q == 0.0L) q = 1e-300L;
    q = -x - off2 / q;
    if (q < 0) ++count;
  }
  return count;
}

void gauss_hermite(int Q, double* a, double* w) {
  const long double bound = std::sqrt(2.0L * Q + 1.0L) + 1.0L;
  std::vector<long double> p(Q + 1);
  for (int i = 0; i < Q; ++i) {
    long double lo = -bound, hi = bound;
    for (int it = 0; it < 120; ++it) {
      long double mid = 0.5L * (lo + hi);
      if (sturm_count(Q, mid) <= i) lo = mid; else hi = mid;
    }
    long double r = 0.5L * (lo + hi);
    for (int it = 0; it < 3; ++it) {     // p_Q' = sqrt(2Q) p_{Q-1}
      orthonormal_hermite(Q, r, p.data());
      r -= p[Q] / (std::sqrt(2.0L * Q) * p[Q - 1]);
    }
    if (Q % 2 == 1 && i == Q / 2) r = 0.0L;
    orthonormal_hermite(Q, r, p.data());
    long double s = 0.0L;
    for (int k = 0; k < Q; ++k) s += p[k] * p[k];
    a[i] = (double)r;
    w[i] = (double)(1.0L / s);
  }
  for (int i = 0; i < Q / 2; ++i) {      // enforce the exact symmetry of the rule
    double am = 0.5 * (a[Q - 1 - i] - a[i]), wm = 0.5 * (w[i] + w[Q - 1 - i]);
    a[i] = -am; a[Q - 1 - i] = am;
    w[i] = wm; w[Q - 1 - i] = wm;
  }
}

void release(fk_ctx* c) {
  if (!c) return;
  DeviceGuard guard(c->device);
  for (int k = 0; k < 3; ++k) { cudaFree(c->d_x[k]); cudaFree(c->d_invh[k]); cudaFree(c->d_wgt[k]); }
  cudaFree(c->d_red);
  cudaFree(c->d_coef);
  cudaFree(c->raw_P[0]);
  cudaFree(c->raw_P[1]);
  cudaFree(c->raw_dP);
  for (int i = 0; i < 2; ++i) {
    cudaFree(c->op[i].w);
    cudaFree(c->op[i].off);
    cudaFree(c->op[i].cnt);
    cudaFree(c->op[i].c);
    cudaFree(c->op[i].rec);
    if (c->ev_ready[i]) cudaEventDestroy(c->ev_ready[i]);
    if (c->ev_free[i]) cudaEventDestroy(c->ev_free[i]);
  }
  if (c->ev_coef) cudaEventDestroy(c->ev_coef);
  if (c->ev_status) cudaEventDestroy(c->ev_status);
  if (c->side) cudaStreamDestroy(c->side);
  cudaFree(c->opb.w);
  cudaFree(c->opb.off);
  cudaFree(c->opb.cnt);
  cudaFree(c->opb.c);
  cudaFree(c->d_far);
  cudaFree(c->d_far_line);
  cudaFree(c->d_work);
  cudaFree(c->d_status);
  cudaFree(c->d_paths);
  if (c->h_status) cudaFreeHost(c->h_status);
  cudaFree(c->d_stage);
  for (auto& e : c->events) { cudaEventDestroy(e.a); cudaEventDestroy(e.b); }
  for (auto& e : c->event_pool) { cudaEventDestroy(e.a); cudaEventDestroy(e.b); }
  delete c;
}

}  // namespace

// ==========================================================================================
// entry points
// ==========================================================================================
extern "C" {

int fk_gauss_hermite(int Q, double* a, double* w) {
  if (Q < 1 || Q > FK_MAX_Q || !a || !w) return FK_EINVAL;
  gauss_hermite(Q, a, w);
  return FK_OK;
}

const char* fk_last_error(const fk_ctx* c) { return c ? c->err.c_str() : g_create_error.c_str(); }

long long fk_launch_count(const fk_ctx* c) { return c ? c->launches : 0; }

void fk_destroy(fk_ctx* c) { release(c); }

int fk_create(const fk_params* p, fk_ctx** out) {
  if (!out) return fail(nullptr, FK_EINVAL, "out is NULL");
  *out = nullptr;
  if (!p) return fail(nullptr, FK_EINVAL, "params is NULL");
  if (p->d < 1 || p->d > 3) return fail(nullptr, FK_EINVAL, "d must be 1..3");
  if (!(p->dt > 0.0) || !std::isfinite(p->dt)) return fail(nullptr, FK_EINVAL, "dt must be > 0");
  if (p->N < 1) return fail(nullptr, FK_EINVAL, "N must be >= 1");
  long long J = 1;
  for (int k = 0; k < p->d; ++k) {
    if (p->n[k] < 3) return fail(nullptr, FK_EINVAL, "each n[k] must be >= 3");
    if (!p->x[k]) return fail(nullptr, FK_EINVAL, "x[k] is NULL");
    if (p->Q[k] < 1 || p->Q[k] > FK_MAX_Q) return fail(nullptr, FK_EINVAL, "Q[k] must be 1..32");
    for (int i = 0; i < p->n[k]; ++i)
      if (!std::isfinite(p->x[k][i]) || (i > 0 && !(p->x[k][i] > p->x[k][i - 1])))
        return fail(nullptr, FK_EINVAL, "x[k] must be finite and strictly increasing");
    if ((p->face_kind[k][0] == FK_FACE_PERIODIC) != (p->face_kind[k][1] == FK_FACE_PERIODIC))
      return fail(nullptr, FK_EINVAL, "FK_FACE_PERIODIC must be set on both faces of a dimension");
    for (int s = 0; s < 2; ++s) {
      if (p->face_kind[k][s] != FK_FACE_ABSORB && p->face_kind[k][s] != FK_FACE_CLAMP &&
          p->face_kind[k][s] != FK_FACE_PERIODIC)
        return fail(nullptr, FK_EINVAL, "unknown face_kind");
      if (p->face_kind[k][s] == FK_FACE_ABSORB && !std::isfinite(p->face_value[k][s]))
        return fail(nullptr, FK_EINVAL, "face_value of an ABSORB face must be finite");
    }
    J *= p->n[k];
    if (J * FK_CW >= (1LL << 31)) return fail(nullptr, FK_EINVAL, "grid too large (J*32 must be < 2^31)");
  }
  int slots = p->coeff_slots;
  if (slots < 0 || slots > p->N) return fail(nullptr, FK_EINVAL, "coeff_slots must be 0..N");
  if (slots == 0) slots = p->N;

  int ndev = 0;
  if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev == 0)
    return fail(nullptr, FK_ECUDA, "no CUDA device: this library has no CPU path");
  if (p->device < 0 || p->device >= ndev) return fail(nullptr, FK_EINVAL, "bad device ordinal");
  int cc_major = 0;
  if (cudaDeviceGetAttribute(&cc_major, cudaDevAttrComputeCapabilityMajor, p->device) != cudaSuccess ||
      cc_major != 10)
    return fail(nullptr, FK_ECUDA, "device is not compute capability 10.x: the kernels are built for sm_100a only");
  if (p->flags & ~(unsigned)(FK_FLAG_VALIDATE | FK_FLAG_WEIGHTED_SLOPES | FK_FLAG_MULTISTEP | FK_FLAG_COUNT_PATHS))
    return fail(nullptr, FK_EINVAL, "unknown bits in flags");
  const int shard_count = p->shard_count <= 0 ? 1 : p->shard_count;
  if (p->shard_index < 0 || p->shard_index >= shard_count)
    return fail(nullptr, FK_EINVAL, "need 0 <= shard_index < shard_count");
  DeviceGuard guard(p->device);

  fk_ctx* c = new (std::nothrow) fk_ctx();
  if (!c) return fail(nullptr, FK_ENOMEM, "host allocation failed");
  c->device = p->device;
  c->stream = (cudaStream_t)p->stream;
  c->N = p->N;
  c->slots = slots;
  {
    const int all = p->N / FK_CW + 1;       // columns 0..N; this shard owns c = index, index+count, ...
    c->n_chunks = all > p->shard_index ? (all - p->shard_index + shard_count - 1) / shard_count : 0;
    if (c->n_chunks == 0) { delete c; return fail(nullptr, FK_EINVAL, "this shard owns no column: shard_count exceeds the number of 32-column chunks"); }
  }
  c->n_next = p->N;
  c->slot_step.assign(slots, -2);

  FkGrid& g = c->g;
  std::memset(&g, 0, sizeof(g));
  g.d = p->d;
  g.J = J;
  g.dt = p->dt;
  g.sq = std::sqrt(2.0 * p->dt);
  g.validate = (p->flags & FK_FLAG_VALIDATE) ? 1 : 0;
  g.weighted = (p->flags & FK_FLAG_WEIGHTED_SLOPES) ? 1 : 0;
  g.paths = nullptr;
  g.shard_index = p->shard_index;
  g.shard_count = shard_count;
  g.near_lo = 0;
  g.near_hi = p->n[0];
  int qoff = 0;
  for (int k = 0; k < 3; ++k) { g.n[k] = 1; g.Q[k] = 0; g.stride[k] = 0; }
  long long st = 1;
  for (int k = p->d - 1; k >= 0; --k) { g.stride[k] = st; st *= p->n[k]; }
  for (int k = 0; k < p->d; ++k) {
    g.n[k] = p->n[k];
    g.Q[k] = p->Q[k];
    g.qoff[k] = qoff;
    qoff += 2 * p->Q[k];
    g.lo[k] = p->x[k][0];
    g.hi[k] = p->x[k][p->n[k] - 1];
    g.inv_h0[k] = (p->n[k] - 1) / (g.hi[k] - g.lo[k]);
    const double h0 = (g.hi[k] - g.lo[k]) / (p->n[k] - 1);
    int uniform = 1;
    for (int i = 0; i < p->n[k]; ++i)
      if (std::fabs(p->x[k][i] - (g.lo[k] + i * h0)) > 1e-9 * h0) uniform = 0;
    g.uniform[k] = uniform;
    g.periodic[k] = p->face_kind[k][0] == FK_FACE_PERIODIC;
    for (int s = 0; s < 2; ++s) {
      g.face_kind[k][s] = p->face_kind[k][s];
      g.face_value[k][s] = p->face_value[k][s];
    }
    gauss_hermite(p->Q[k], g.gh_a[k], g.gh_w[k]);
  }
  g.RS = qoff;
  c->n_updated = 1;
  for (int k = 0; k < p->d; ++k)
    c->n_updated *= p->n[k] - (p->face_kind[k][0] == FK_FACE_ABSORB) - (p->face_kind[k][1] == FK_FACE_ABSORB);

#define FK_CREATE_CUDA(call)                                                    \
  do {                                                                          \
    cudaError_t e_ = (call);                                                    \
    if (e_ != cudaSuccess) {                                                    \
      int code_ = cuda_fail(nullptr, e_, #call);                                \
      release(c);                                                               \
      return code_;                                                             \
    }                                                                           \
  } while (0)

  for (int k = 0; k < p->d; ++k) {
    const int n = p->n[k];
    std::vector<double> ih(n - 1);
    for (int i = 0; i < n - 1; ++i) ih[i] = 1.0 / (p->x[k][i + 1] - p->x[k][i]);
    FK_CREATE_CUDA(cudaMalloc(&c->d_x[k], sizeof(double) * n));
    FK_CREATE_CUDA(cudaMalloc(&c->d_invh[k], sizeof(double) * (n - 1)));
    FK_CREATE_CUDA(cudaMemcpyAsync(c->d_x[k], p->x[k], sizeof(double) * n, cudaMemcpyHostToDevice, c->stream));
    FK_CREATE_CUDA(cudaMemcpyAsync(c->d_invh[k], ih.data(), sizeof(double) * (n - 1), cudaMemcpyHostToDevice, c->stream));
    FK_CREATE_CUDA(cudaStreamSynchronize(c->stream));   // ih is a local
    g.x[k] = c->d_x[k];
    g.inv_h[k] = c->d_invh[k];
    if (g.weighted) {
      // R22: per node the weights attached to the two divided differences of its slope window
      // (fk_kernels.cu slope_window): cells (ca, cb) of widths (ha, hb); the difference of ca
      // carries w = 2 hb + ha, that of cb carries hb + 2 ha -- except at the last node of a
      // non-periodic line, where the window is read in the opposite order (delta_{n-2} first)
      std::vector<double2> wg(n);
      for (int i = 0; i < n; ++i) {
        int ca, cb;
        if (g.periodic[k]) { ca = i == 0 ? n - 2 : i - 1; cb = i == n - 1 ? 0 : i; }
        else { const int la = i - 1 < 0 ? 0 : (i - 1 > n - 3 ? n - 3 : i - 1); ca = la; cb = la + 1; }
        const double ha = p->x[k][ca + 1] - p->x[k][ca], hb = p->x[k][cb + 1] - p->x[k][cb];
        double wa = 2.0 * hb + ha, wb = hb + 2.0 * ha;
        if (!g.periodic[k] && i == n - 1) { wa = ha + 2.0 * hb; wb = 2.0 * ha + hb; }
        wg[i] = make_double2(wa / (wa + wb), wb / (wa + wb));
      }
      FK_CREATE_CUDA(cudaMalloc(&c->d_wgt[k], sizeof(double2) * n));
      FK_CREATE_CUDA(cudaMemcpyAsync(c->d_wgt[k], wg.data(), sizeof(double2) * n, cudaMemcpyHostToDevice, c->stream));
      FK_CREATE_CUDA(cudaStreamSynchronize(c->stream));   // wg is a local
      g.wgt[k] = c->d_wgt[k];
    }
  }
  {
    bool any_periodic = false, all_uniform = true;
    for (int k = 0; k < p->d; ++k) { any_periodic = any_periodic || g.periodic[k]; all_uniform = all_uniform && g.uniform[k]; }
    g.general_slopes = (any_periodic || g.weighted) ? 1 : 0;
    // the fused 2-D kernel computes Eq. 15 itself, for box problems: periodic dimensions and the
    // weighted mean on a non-uniform grid go through the generic slopes / apply kernels
    c->fused2d = p->d == 2 && !any_periodic && !(g.weighted && !all_uniform);
  }
  const size_t buf = sizeof(double) * (size_t)c->n_chunks * J * FK_CW;
  // P and dP carry FK_GUARD_ROWS zeroed 256-byte rows at both ends, and dP is cleared once: the
  // row-blocked kernels read a few nodes past a line's ends with zero weights (fk_rowblock3d.cu),
  // which must then be finite numbers
  const size_t guard_bytes = sizeof(double) * FK_GUARD_ROWS * FK_CW;
  for (int i = 0; i < 2; ++i) {
    FK_CREATE_CUDA(cudaMalloc(&c->raw_P[i], buf + 2 * guard_bytes));
    FK_CREATE_CUDA(cudaMemsetAsync(c->raw_P[i], 0, buf + 2 * guard_bytes, c->stream));
    c->d_P[i] = reinterpret_cast<double*>(static_cast<char*>(c->raw_P[i]) + guard_bytes);
  }
  FK_CREATE_CUDA(cudaMalloc(&c->raw_dP, buf * p->d + 2 * guard_bytes));
  FK_CREATE_CUDA(cudaMemsetAsync(c->raw_dP, 0, buf * p->d + 2 * guard_bytes, c->stream));
  c->d_dP = reinterpret_cast<double*>(static_cast<char*>(c->raw_dP) + guard_bytes);
  FK_CREATE_CUDA(cudaMalloc(&c->d_coef, sizeof(double) * (size_t)slots * 2 * p->d * J));
  FK_CREATE_CUDA(cudaStreamCreateWithFlags(&c->side, cudaStreamNonBlocking));
  FK_CREATE_CUDA(cudaEventCreateWithFlags(&c->ev_coef, cudaEventDisableTiming));
  FK_CREATE_CUDA(cudaEventCreateWithFlags(&c->ev_status, cudaEventDisableTiming));
  for (int i = 0; i < 2; ++i) {
    FK_CREATE_CUDA(cudaMalloc(&c->op[i].w, sizeof(double2) * (size_t)J * g.RS));
    FK_CREATE_CUDA(cudaMalloc(&c->op[i].off, sizeof(int) * (size_t)J * g.RS));
    FK_CREATE_CUDA(cudaMalloc(&c->op[i].cnt, sizeof(int) * (size_t)J * 4));
    FK_CREATE_CUDA(cudaMalloc(&c->op[i].c, sizeof(double) * (size_t)J));
    FK_CREATE_CUDA(cudaEventCreateWithFlags(&c->ev_ready[i], cudaEventDisableTiming));
    FK_CREATE_CUDA(cudaEventCreateWithFlags(&c->ev_free[i], cudaEventDisableTiming));
  }
  FK_CREATE_CUDA(cudaMalloc(&c->d_work, sizeof(unsigned long long) * 4 * (size_t)p->N));
  FK_CREATE_CUDA(cudaMemsetAsync(c->d_work, 0, sizeof(unsigned long long) * 4 * (size_t)p->N, c->stream));
  if (p->flags & FK_FLAG_COUNT_PATHS) {
    FK_CREATE_CUDA(cudaMalloc(&c->d_paths, sizeof(unsigned long long) * FK_PATH_COUNT));
    FK_CREATE_CUDA(cudaMemsetAsync(c->d_paths, 0, sizeof(unsigned long long) * FK_PATH_COUNT, c->stream));
    c->g.paths = c->d_paths;
  }
  FK_CREATE_CUDA(cudaMalloc(&c->d_status, sizeof(int)));
  FK_CREATE_CUDA(cudaMemsetAsync(c->d_status, 0, sizeof(int), c->stream));
  FK_CREATE_CUDA(cudaHostAlloc(&c->h_status, sizeof(int), cudaHostAllocDefault));
  *c->h_status = 0;
  FK_CREATE_CUDA(cudaDeviceGetAttribute(&c->sm_count, cudaDevAttrMultiProcessorCount, c->device));
  if (c->fused2d) {                      // the fused 2-D kernel's records and step classification
    for (int i = 0; i < 2; ++i) {
      FK_CREATE_CUDA(cudaMalloc(&c->op[i].rec, sizeof(FkRec2) * (size_t)J));
      FK_CREATE_CUDA(cudaMemsetAsync(c->op[i].rec, 0, sizeof(FkRec2) * (size_t)J, c->stream));
    }
    FK_CREATE_CUDA(cudaMalloc(&c->d_far, sizeof(int) * (size_t)slots * FK_FAR_STRIDE));
    FK_CREATE_CUDA(cudaMemsetAsync(c->d_far, 0, sizeof(int) * (size_t)slots * FK_FAR_STRIDE, c->stream));
    FK_CREATE_CUDA(fk_fused2d_setup());
    c->h_far.assign((size_t)slots * FK_FAR_STRIDE, 0);
    FK_CREATE_CUDA(cudaMalloc(&c->d_far_line, sizeof(int) * (size_t)slots * p->n[0]));
    FK_CREATE_CUDA(cudaMemsetAsync(c->d_far_line, 0, sizeof(int) * (size_t)slots * p->n[0], c->stream));
    c->h_far_line.assign((size_t)slots * p->n[0], 0);
  }
  if (p->d == 1 && (p->flags & FK_FLAG_MULTISTEP)) {
    // the multi-step 1-D kernel: needs three copies of a column group's line in shared memory
    int smem_max = 0;
    FK_CREATE_CUDA(cudaDeviceGetAttribute(&smem_max, cudaDevAttrMaxSharedMemoryPerBlockOptin, c->device));
    c->line1d_cg = fk_line1d_group(g, (size_t)smem_max);
    if (c->line1d_cg) {
      const size_t per_step = (size_t)J * g.RS * (sizeof(double2) + sizeof(int)) + (size_t)J * (4 * sizeof(int) + sizeof(double));
      long long cap = (long long)(((size_t)256 << 20) / per_step);
      if (cap < 1) cap = 1;
      if (cap > slots) cap = slots;          // a batch never outruns the loaded coefficient slots
      c->batch_cap = (int)cap;
      FK_CREATE_CUDA(cudaMalloc(&c->opb.w, sizeof(double2) * (size_t)cap * J * g.RS));
      FK_CREATE_CUDA(cudaMalloc(&c->opb.off, sizeof(int) * (size_t)cap * J * g.RS));
      FK_CREATE_CUDA(cudaMalloc(&c->opb.cnt, sizeof(int) * (size_t)cap * J * 4));
      FK_CREATE_CUDA(cudaMalloc(&c->opb.c, sizeof(double) * (size_t)cap * J));
      FK_CREATE_CUDA(fk_line1d_setup(g, c->line1d_cg));
    }
  }
  FK_CREATE_CUDA(fk_launch_fill_chi(g, c->d_P[0], c->n_chunks, c->stream));
  FK_CREATE_CUDA(fk_launch_fill_chi(g, c->d_P[1], c->n_chunks, c->stream));
  c->launches += 2;
#undef FK_CREATE_CUDA
  *out = c;
  return FK_OK;
}

int fk_reset(fk_ctx* c) {
  if (!c) return FK_EINVAL;
  DeviceGuard guard(c->device);
  FK_CUDA(c, fk_launch_fill_chi(c->g, c->d_P[0], c->n_chunks, c->stream));
  FK_CUDA(c, fk_launch_fill_chi(c->g, c->d_P[1], c->n_chunks, c->stream));
  c->launches += 2;
  FK_CUDA(c, cudaMemsetAsync(c->d_status, 0, sizeof(int), c->stream));
  FK_CUDA(c, cudaMemsetAsync(c->d_work, 0, sizeof(unsigned long long) * 4 * (size_t)c->N, c->stream));
  for (int k = 0; k < FK_K_COUNT; ++k) c->class_updates[k] = 0.0;
  // a refresh of h_status queued by the last fk_evolve may not have landed yet: wait for it, or its
  // stale bits would overwrite the cleared word and fail the next call for no reason
  if (c->status_pending) {
    FK_CUDA(c, cudaEventSynchronize(c->ev_status));
    c->status_pending = false;
  }
  *c->h_status = 0;
  c->auto_assembled = false;           // its work counters were just cleared: assemble once more
  c->cur = 0;
  c->n_next = c->N;
  for (auto& e : c->events) c->event_pool.push_back(e);
  c->events.clear();
  return FK_OK;
}

int fk_set_coeffs_range(fk_ctx* c, int step0, int count, const double* b, const double* sigma,
                        int mem) {
  if (!c) return FK_EINVAL;
  if (!b || !sigma) return fail(c, FK_EINVAL, "b or sigma is NULL");
  if (mem != FK_MEM_HOST && mem != FK_MEM_DEVICE && mem != FK_MEM_HOST_PINNED) return fail(c, FK_EINVAL, "bad mem kind");
  if (count < 1 || count > c->slots) return fail(c, FK_EINVAL, "count must be 1..coeff_slots");
  if (step0 < 0 || step0 + count > c->N) return fail(c, FK_EINVAL, "step range outside 0..N-1");
  DeviceGuard guard(c->device);
  const size_t slice = (size_t)c->g.d * c->g.J;      // doubles per [d][J] array
  const cudaMemcpyKind kind = mem == FK_MEM_DEVICE ? cudaMemcpyDeviceToDevice : cudaMemcpyHostToDevice;
  for (int i = 0; i < count; ++i) {
    const int step = step0 + i, slot = step % c->slots;
    double* dst = c->d_coef + (size_t)slot * 2 * slice;
    FK_CUDA(c, cudaMemcpyAsync(dst, b + (size_t)i * slice, sizeof(double) * slice, kind, c->stream));
    FK_CUDA(c, cudaMemcpyAsync(dst + slice, sigma + (size_t)i * slice, sizeof(double) * slice, kind, c->stream));
    c->slot_step[slot] = step;
  }
  c->autonomous = false;
  if (c->fused2d) {                      // which of these steps have rows outside the fused halo
    const int s0 = step0 % c->slots;
    const int first = count < c->slots - s0 ? count : c->slots - s0;
    FK_CUDA(c, cudaMemsetAsync(c->d_far + (size_t)s0 * FK_FAR_STRIDE, 0, sizeof(int) * (size_t)first * FK_FAR_STRIDE, c->stream));
    if (count > first)
      FK_CUDA(c, cudaMemsetAsync(c->d_far, 0, sizeof(int) * (size_t)(count - first) * FK_FAR_STRIDE, c->stream));
    const size_t n0 = (size_t)c->g.n[0];
    FK_CUDA(c, cudaMemsetAsync(c->d_far_line + (size_t)s0 * n0, 0, sizeof(int) * (size_t)first * n0, c->stream));
    if (count > first)
      FK_CUDA(c, cudaMemsetAsync(c->d_far_line, 0, sizeof(int) * (size_t)(count - first) * n0, c->stream));
    FK_CUDA(c, fk_launch_classify(c->g, c->d_coef, c->slots, step0, count, c->d_far, c->d_far_line, c->stream));
    ++c->launches;
    c->far_valid = false;
  }
  if (mem == FK_MEM_HOST) FK_CUDA(c, cudaStreamSynchronize(c->stream));
  return FK_OK;
}

int fk_set_coeffs(fk_ctx* c, int step, const double* b, const double* sigma, int mem) {
  if (!c) return FK_EINVAL;
  if (step != FK_ALL_STEPS) return fk_set_coeffs_range(c, step, 1, b, sigma, mem);
  if (!b || !sigma) return fail(c, FK_EINVAL, "b or sigma is NULL");
  if (mem != FK_MEM_HOST && mem != FK_MEM_DEVICE && mem != FK_MEM_HOST_PINNED) return fail(c, FK_EINVAL, "bad mem kind");
  DeviceGuard guard(c->device);
  const size_t slice = (size_t)c->g.d * c->g.J;
  const cudaMemcpyKind kind = mem == FK_MEM_DEVICE ? cudaMemcpyDeviceToDevice : cudaMemcpyHostToDevice;
  FK_CUDA(c, cudaMemcpyAsync(c->d_coef, b, sizeof(double) * slice, kind, c->stream));
  FK_CUDA(c, cudaMemcpyAsync(c->d_coef + slice, sigma, sizeof(double) * slice, kind, c->stream));
  std::fill(c->slot_step.begin(), c->slot_step.end(), -2);
  c->autonomous = true;
  c->auto_assembled = false;
  if (c->fused2d) {
    FK_CUDA(c, cudaMemsetAsync(c->d_far, 0, sizeof(int) * FK_FAR_STRIDE, c->stream));
    FK_CUDA(c, cudaMemsetAsync(c->d_far_line, 0, sizeof(int) * (size_t)c->g.n[0], c->stream));
    FK_CUDA(c, fk_launch_classify(c->g, c->d_coef, c->slots, 0, 1, c->d_far, c->d_far_line, c->stream));
    ++c->launches;
    c->far_valid = false;
  }
  if (mem == FK_MEM_HOST) FK_CUDA(c, cudaStreamSynchronize(c->stream));
  return FK_OK;
}


}  // extern "C"

namespace {

// one kernel launch, optionally bracketed by a pair of events of class `cls`; the pair goes
// back to the pool when the launch fails
template <class Launch>
int launch_on(fk_ctx* c, cudaStream_t st, int cls, const char* what, Launch&& launch) {
  EventPair ep{};
  if (c->profiling) {
    if (!c->event_pool.empty()) { ep = c->event_pool.back(); c->event_pool.pop_back(); }
    else { FK_CUDA(c, cudaEventCreate(&ep.a)); FK_CUDA(c, cudaEventCreate(&ep.b)); }
    ep.cls = cls;
  }
  cudaError_t e = c->profiling ? cudaEventRecord(ep.a, st) : cudaSuccess;
  if (e == cudaSuccess) e = launch();
  if (e == cudaSuccess && c->profiling) e = cudaEventRecord(ep.b, st);
  if (e != cudaSuccess) {
    if (c->profiling) c->event_pool.push_back(ep);
    return cuda_fail(c, e, what);
  }
  ++c->launches;
  if (c->profiling) c->events.push_back(ep);
  return FK_OK;
}
#define FK_TRY(expr) do { int rc_ = (expr); if (rc_ != FK_OK) return rc_; } while (0)

const char* status_text(int bits) {
  if (bits & FK_BAD_NEG_SIGMA) return "negative sigma at an updated node (found on the device while assembling a step operator)";
  if (bits & FK_BAD_NONFINITE) return "NaN or Inf coefficient at an updated node (FK_FLAG_VALIDATE)";
  return "";
}

// 2-D: who takes which rows of one step.  The fused kernel costs the same per line whatever share
// of the line's rows it owns, so the lines at either end of dimension 0 on which at least half of
// the updated rows are far (config 4: p < ~12) are left to fk_far2d whole -- their near rows are
// assembled without the FK_ROW_NEAR flag (FkGrid::near_lo / near_hi) -- and the fused kernel runs on
// the output lines line_lo .. line_hi-1 only.  Lines of Dirichlet nodes need no kernel at all (both P
// buffers hold chi there from the start).
struct Plan2D {
  int line_lo = 0, line_hi = 0;   // output lines of the fused kernel
  double other_rows = 0.0;        // updated rows it leaves out (far rows + the near rows of skipped lines)
  int fl0 = 0, fl1 = 0;           // lines holding such rows: fl0 .. fl1-1 (fk_far2d)
  int sl0 = 0, sl1 = 0;           // lines their entries touch: sl0 .. sl1-1 (fk_slopes)
};

Plan2D plan_2d(const fk_ctx* c, int slot) {
  const FkGrid& g = c->g;
  const int n0 = g.n[0], n1 = g.n[1];
  const int* far = &c->h_far[(size_t)slot * FK_FAR_STRIDE];
  const int* fl = &c->h_far_line[(size_t)slot * n0];
  const int upl = n1 - (g.face_kind[1][0] == FK_FACE_ABSORB) - (g.face_kind[1][1] == FK_FACE_ABSORB);
  const int first = g.face_kind[0][0] == FK_FACE_ABSORB ? 1 : 0;          // updated lines: first .. last-1
  const int last = g.face_kind[0][1] == FK_FACE_ABSORB ? n0 - 1 : n0;
  Plan2D p;
  int lo = first, hi = last;
  while (lo < hi && 2 * fl[lo] >= upl) ++lo;
  while (hi > lo && 2 * fl[hi - 1] >= upl) --hi;
  p.line_lo = lo;
  p.line_hi = hi;
  p.other_rows = far[0];
  p.fl0 = p.sl0 = n0;
  if (far[0] > 0) {
    p.fl0 = FK_FAR_BIG - far[1]; p.fl1 = far[2];
    p.sl0 = FK_FAR_BIG - far[3]; p.sl1 = far[4];
  }
  auto hand_over = [&](int a, int b) {               // lines a .. b-1 go to fk_far2d whole
    if (a >= b) return;
    for (int l = a; l < b; ++l) p.other_rows += upl - fl[l];
    p.fl0 = a < p.fl0 ? a : p.fl0;
    p.fl1 = b > p.fl1 ? b : p.fl1;
    const int s0 = a - FK_H > 0 ? a - FK_H : 0, s1 = b + FK_H < n0 ? b + FK_H : n0;   // near rows reach FK_H lines
    p.sl0 = s0 < p.sl0 ? s0 : p.sl0;
    p.sl1 = s1 > p.sl1 ? s1 : p.sl1;
  };
  hand_over(first, lo);
  hand_over(hi, last);
  return p;
}

// one step of Algorithm 1: assemble A_nu (nu = n-1) on the side stream,
// update columns n..N on the caller's stream
int evolve_step(fk_ctx* c, int n) {
  const size_t slice = (size_t)c->g.d * c->g.J;
  const int last_chunk = c->n_chunks;                  // one past the (local) chunk of column N
  const int nu = n - 1;
  int slot = 0;
  if (!c->autonomous) {
    slot = nu % c->slots;
    if (c->slot_step[slot] != nu) {
      char msg[96];
      std::snprintf(msg, sizeof msg, "coefficients of step %d are not loaded", nu);
      return fail(c, FK_ESTATE, msg);
    }
  }
  const double* b = c->d_coef + (size_t)slot * 2 * slice;
  // first local chunk with an active column: local chunk l is global chunk l * count + index
  int chunk0 = (n / FK_CW - c->g.shard_index + c->g.shard_count - 1) / c->g.shard_count;
  if (n / FK_CW < c->g.shard_index) chunk0 = 0;
  const double* Pold = c->d_P[c->cur];
  double* Pnew = c->d_P[c->cur ^ 1];
  if (chunk0 >= last_chunk) return FK_OK;              // (sharded) none of this context's columns is active yet
  // assemble A_nu into buffer n & 1 on the side stream as soon as the kernels of step n + 2
  // (the buffer's previous users) are done; the kernels of this step wait for it
  // (an autonomous problem has one operator: assembled at the first step after a reset, reused)
  const int ob = c->autonomous ? 0 : (n & 1);
  const FkOperator& op = c->op[ob];
  cudaStream_t st = c->stream;
  const bool fused = c->fused2d;
  const Plan2D plan = fused ? plan_2d(c, slot) : Plan2D();
  if (!(c->autonomous && c->auto_assembled)) {
    FkGrid gs = c->g;                                  // this step's range of lines with FK_ROW_NEAR rows
    if (fused) { gs.near_lo = plan.line_lo; gs.near_hi = plan.line_hi; }
    FK_CUDA(c, cudaStreamWaitEvent(c->side, c->ev_free[ob], 0));
    FK_TRY(launch_on(c, c->side, FK_K_ASSEMBLE, "fk_assemble", [&] {
      return fk_launch_assemble(gs, b, b + slice, op, c->d_status, c->d_work + 4 * (size_t)nu, c->side); }));
    FK_CUDA(c, cudaEventRecord(c->ev_ready[ob], c->side));
    FK_CUDA(c, cudaStreamWaitEvent(st, c->ev_ready[ob], 0));
    if (c->autonomous) { c->auto_assembled = true; c->auto_nu = nu; }
    c->class_updates[FK_K_ASSEMBLE] += (double)c->n_updated;
  }
  const bool generic = !fused || plan.other_rows > 0;  // rows the fused kernel leaves out
  {                                                    // bookkeeping for fk_profile_updates
    double cols = 0.0;                                 // active columns this context owns
    for (int l = chunk0; l < last_chunk; ++l) {
      const int m_lo = (l * c->g.shard_count + c->g.shard_index) * FK_CW;
      const int a = m_lo > n ? m_lo : n, e = m_lo + FK_CW - 1 < c->N ? m_lo + FK_CW - 1 : c->N;
      if (e >= a) cols += e - a + 1;
    }
    if (fused) c->class_updates[FK_K_FUSED] += ((double)c->n_updated - plan.other_rows) * cols;
    if (generic) {
      c->class_updates[FK_K_SLOPES] += (fused ? (double)(plan.sl1 - plan.sl0) * c->g.n[1] : (double)c->g.J) * cols;
      c->class_updates[c->g.d == 3 ? FK_K_ROWBLOCK : fused ? FK_K_FAR2D : FK_K_APPLY] += (fused ? plan.other_rows : (double)c->n_updated) * cols;
    }
  }
  if (fused && plan.line_hi > plan.line_lo)
    FK_TRY(launch_on(c, st, FK_K_FUSED, "fk_fused2d", [&] {
      return fk_launch_fused2d(c->g, op, Pold, Pnew, chunk0, last_chunk, n, c->N, c->sm_count, plan.line_lo,
                               plan.line_hi, st); }));
  if (generic) {
    // all nodes, or (2-D) only the lines that hold rows outside the fused kernel / that their entries touch
    int sl0 = 0, sln = (int)(c->g.J / c->g.n[c->g.d - 1]);
    if (fused) {
      sl0 = plan.sl0;
      sln = plan.sl1 - plan.sl0;
    }
    FK_TRY(launch_on(c, st, FK_K_SLOPES, "fk_slopes", [&] {
      return fk_launch_slopes(c->g, Pold, c->d_dP, c->n_chunks, chunk0, last_chunk, sl0, sln, st); }));
    if (c->g.d == 3)
      FK_TRY(launch_on(c, st, FK_K_ROWBLOCK, "fk_rowblock3d", [&] {
        return fk_launch_rowblock3d(c->g, op, Pold, c->d_dP, Pnew, c->n_chunks, chunk0, last_chunk, n,
                                    c->N, st); }));
    else if (fused)                                    // the rows the fused kernel left out
      FK_TRY(launch_on(c, st, FK_K_FAR2D, "fk_far2d", [&] {
        return fk_launch_far2d(c->g, op, Pold, c->d_dP, Pnew, c->n_chunks, chunk0, last_chunk, n, c->N,
                               plan.fl0, plan.fl1 - plan.fl0, st); }));
    else
      FK_TRY(launch_on(c, st, FK_K_APPLY, "fk_apply", [&] {
        return fk_launch_apply(c->g, op, Pold, c->d_dP, Pnew, c->n_chunks, chunk0, last_chunk, n, c->N,
                               0, 0, c->g.J, st); }));
  }
  if (!c->autonomous) FK_CUDA(c, cudaEventRecord(c->ev_free[ob], st));
  return FK_OK;
}

// active columns this context owns at step n (bookkeeping for fk_profile_updates)
double active_columns(const fk_ctx* c, int n) {
  double cols = 0.0;
  for (int l = 0; l < c->n_chunks; ++l) {
    const int m_lo = (l * c->g.shard_count + c->g.shard_index) * FK_CW;
    const int a = m_lo > n ? m_lo : n, e = m_lo + FK_CW - 1 < c->N ? m_lo + FK_CW - 1 : c->N;
    if (e >= a) cols += e - a + 1;
  }
  return cols;
}

// 1-D: the steps n, n-1, ..., n-count+1 of Algorithm 1 in two launches -- their operators into the
// batch storage, then fk_line1d with every column group resident in shared memory over all of them
int evolve_batch1d(fk_ctx* c, int n, int count) {
  cudaStream_t st = c->stream;
  if (!c->autonomous)
    for (int k = 0; k < count; ++k) {
      const int nu = n - 1 - k;
      if (c->slot_step[nu % c->slots] != nu) {
        char msg[96];
        std::snprintf(msg, sizeof msg, "coefficients of step %d are not loaded", nu);
        return fail(c, FK_ESTATE, msg);
      }
    }
  if (!(c->autonomous && c->auto_assembled)) {
    const int na = c->autonomous ? 1 : count;
    FK_TRY(launch_on(c, st, FK_K_ASSEMBLE, "fk_assemble_batch", [&] {
      return fk_launch_assemble_batch(c->g, c->d_coef, c->slots, n - 1, na, c->autonomous ? 1 : 0, c->opb,
                                      c->d_status, c->d_work, st); }));
    if (c->autonomous) { c->auto_assembled = true; c->auto_nu = n - 1; }
    c->class_updates[FK_K_ASSEMBLE] += (double)c->n_updated * na;
  }
  for (int k = 0; k < count; ++k) c->class_updates[FK_K_LINE1D] += (double)c->n_updated * active_columns(c, n - k);
  FK_TRY(launch_on(c, st, FK_K_LINE1D, "fk_line1d", [&] {
    return fk_launch_line1d(c->g, c->opb, c->line1d_cg, count, n, c->autonomous ? 1 : 0, c->d_P[c->cur],
                            c->d_P[c->cur ^ 1], c->n_chunks, c->N, st); }));
  return FK_OK;
}

// after a failure inside a step: make the caller's stream wait for whatever the side stream
// still has queued, so that the two never run unordered past the failing call (best effort)
void join_side(fk_ctx* c) {
  if (cudaEventRecord(c->ev_coef, c->side) == cudaSuccess) cudaStreamWaitEvent(c->stream, c->ev_coef, 0);
}

}  // namespace

extern "C" {

int fk_evolve(fk_ctx* c, int n_from, int n_to) {
  if (!c) return FK_EINVAL;
  if (n_from != c->n_next) return fail(c, FK_ESTATE, "n_from must continue where the last fk_evolve stopped (N after create/reset)");
  if (n_to < 0 || n_to > n_from) return fail(c, FK_EINVAL, "need 0 <= n_to <= n_from");
  if (*c->h_status) return fail(c, FK_EINVAL, status_text(*c->h_status));
  DeviceGuard guard(c->device);
  if (c->fused2d && !c->far_valid && n_from > n_to) {  // one small read-back per coefficient load
    FK_CUDA(c, cudaMemcpyAsync(c->h_far.data(), c->d_far, sizeof(int) * (size_t)c->slots * FK_FAR_STRIDE,
                               cudaMemcpyDeviceToHost, c->stream));
    FK_CUDA(c, cudaMemcpyAsync(c->h_far_line.data(), c->d_far_line, sizeof(int) * c->h_far_line.size(),
                               cudaMemcpyDeviceToHost, c->stream));
    FK_CUDA(c, cudaStreamSynchronize(c->stream));
    c->far_valid = true;
  }
  // the side stream must see the coefficient copies queued on the caller's stream so far
  FK_CUDA(c, cudaEventRecord(c->ev_coef, c->stream));
  FK_CUDA(c, cudaStreamWaitEvent(c->side, c->ev_coef, 0));
  if (c->line1d_cg) {                 // 1-D: batches of steps, both P buffers end up current
    for (int n = n_from; n > n_to;) {
      const int left = n - n_to;
      const int count = c->autonomous ? left : (left < c->batch_cap ? left : c->batch_cap);
      const int rc = evolve_batch1d(c, n, count);
      if (rc != FK_OK) { c->n_next = n; return rc; }
      n -= count;
      c->n_next = n;
    }
    if (n_from > n_to) {
      FK_CUDA(c, cudaMemcpyAsync(c->h_status, c->d_status, sizeof(int), cudaMemcpyDeviceToHost, c->stream));
      FK_CUDA(c, cudaEventRecord(c->ev_status, c->stream));
      c->status_pending = true;
    }
    return FK_OK;
  }
  for (int n = n_from; n > n_to; --n) {
    const int rc = evolve_step(c, n);
    if (rc != FK_OK) {
      join_side(c);
      c->n_next = n;                 // the step was not completed; P still holds the state of n
      return rc;
    }
    c->cur ^= 1;
    c->n_next = n - 1;
  }
  if (n_from > n_to) {               // refresh the host copy of the device status word
    FK_CUDA(c, cudaMemcpyAsync(c->h_status, c->d_status, sizeof(int), cudaMemcpyDeviceToHost, c->stream));
    FK_CUDA(c, cudaEventRecord(c->ev_status, c->stream));
    c->status_pending = true;
  }
  return FK_OK;
}

int fk_check(fk_ctx* c) {
  if (!c) return FK_EINVAL;
  DeviceGuard guard(c->device);
  FK_CUDA(c, cudaMemcpyAsync(c->h_status, c->d_status, sizeof(int), cudaMemcpyDeviceToHost, c->stream));
  FK_CUDA(c, cudaStreamSynchronize(c->stream));
  if (*c->h_status) return fail(c, FK_EINVAL, status_text(*c->h_status));
  return FK_OK;
}

int fk_read(fk_ctx* c, int m0, int m1, double* out, int mem) {
  if (!c) return FK_EINVAL;
  if (!out) return fail(c, FK_EINVAL, "out is NULL");
  if (mem != FK_MEM_HOST && mem != FK_MEM_DEVICE) return fail(c, FK_EINVAL, "bad mem kind");
  if (m0 < 0 || m1 > c->N + 1 || m0 >= m1) return fail(c, FK_EINVAL, "need 0 <= m0 < m1 <= N+1");
  if (c->n_next != 0 && m1 > 1) return fail(c, FK_ESTATE, "columns other than 0 are final only after fk_evolve reached n_to = 0");
  if (*c->h_status) return fail(c, FK_EINVAL, status_text(*c->h_status));
  DeviceGuard guard(c->device);
  const double* P = c->d_P[c->cur];
  const size_t col = sizeof(double) * (size_t)c->g.J;
  if (mem == FK_MEM_DEVICE) {
    FK_CUDA(c, fk_launch_gather_columns(c->g, P, m0, m1, out, c->stream));
    ++c->launches;
    return FK_OK;
  }
  // host destination: gather into a bounded device staging buffer, copy out batch by batch
  // (a shard copies chunk by chunk, its own chunks only: the other rows of `out` are not its)
  const bool sharded = c->g.shard_count > 1;
  const size_t want = (size_t)256 << 20;
  int batch = (int)(want / col);
  if (batch < FK_CW || sharded) batch = FK_CW;
  batch -= batch % FK_CW;
  if (batch > m1 - m0 && !sharded) batch = m1 - m0;
  if (c->stage_bytes < (size_t)batch * col) {
    cudaFree(c->d_stage);
    c->d_stage = nullptr;
    c->stage_bytes = 0;
    FK_CUDA(c, cudaMalloc(&c->d_stage, (size_t)batch * col));
    c->stage_bytes = (size_t)batch * col;
  }
  for (int a = m0; a < m1;) {
    int e = a + batch < m1 ? a + batch : m1;
    if (sharded) {                                       // [a, e) = the part of one chunk inside [m0, m1)
      e = (a / FK_CW + 1) * FK_CW < m1 ? (a / FK_CW + 1) * FK_CW : m1;
      if ((a / FK_CW) % c->g.shard_count != c->g.shard_index) { a = e; continue; }
    }
    FK_CUDA(c, fk_launch_gather_columns(c->g, P, a, e, c->d_stage, c->stream));
    ++c->launches;
    FK_CUDA(c, cudaMemcpyAsync(out + (size_t)(a - m0) * c->g.J, c->d_stage, (size_t)(e - a) * col,
                               cudaMemcpyDeviceToHost, c->stream));
    FK_CUDA(c, cudaStreamSynchronize(c->stream));
    a = e;
  }
  if (*c->h_status) return fail(c, FK_EINVAL, status_text(*c->h_status));   // refreshed by fk_evolve
  return FK_OK;
}

int fk_reduce(fk_ctx* c, const double* weights, int m0, int m1, double* out, int mem) {
  if (!c) return FK_EINVAL;
  if (!weights || !out) return fail(c, FK_EINVAL, "weights or out is NULL");
  if (mem != FK_MEM_HOST && mem != FK_MEM_DEVICE) return fail(c, FK_EINVAL, "bad mem kind");
  if (m0 < 0 || m1 > c->N + 1 || m0 >= m1) return fail(c, FK_EINVAL, "need 0 <= m0 < m1 <= N+1");
  if (c->n_next != 0 && m1 > 1) return fail(c, FK_ESTATE, "columns other than 0 are final only after fk_evolve reached n_to = 0");
  if (*c->h_status) return fail(c, FK_EINVAL, status_text(*c->h_status));
  DeviceGuard guard(c->device);
  const size_t J = (size_t)c->g.J;
  const int chunks = (m1 - 1) / FK_CW - m0 / FK_CW + 1;
  // scratch: [J] weights (host sources), [chunks][FK_RED_BLOCKS][32] partial sums, [m1-m0] result
  const size_t need = sizeof(double) * (J + (size_t)chunks * FK_RED_BLOCKS * FK_CW + (size_t)(m1 - m0));
  if (c->red_bytes < need) {
    cudaFree(c->d_red);
    c->d_red = nullptr;
    c->red_bytes = 0;
    FK_CUDA(c, cudaMalloc(&c->d_red, need));
    c->red_bytes = need;
  }
  double* d_w = c->d_red;
  double* d_partial = d_w + J;
  double* d_out = d_partial + (size_t)chunks * FK_RED_BLOCKS * FK_CW;
  const double* w = weights;
  if (mem == FK_MEM_HOST) {
    FK_CUDA(c, cudaMemcpyAsync(d_w, weights, sizeof(double) * J, cudaMemcpyHostToDevice, c->stream));
    // a shard writes only its own columns: start from the caller's values
    FK_CUDA(c, cudaMemcpyAsync(d_out, out, sizeof(double) * (size_t)(m1 - m0), cudaMemcpyHostToDevice, c->stream));
    w = d_w;
  }
  FK_CUDA(c, fk_launch_reduce(c->g, c->d_P[c->cur], w, m0, m1, d_partial,
                              mem == FK_MEM_HOST ? d_out : out, c->stream));
  c->launches += 2;
  if (mem == FK_MEM_HOST) {
    FK_CUDA(c, cudaMemcpyAsync(out, d_out, sizeof(double) * (size_t)(m1 - m0), cudaMemcpyDeviceToHost, c->stream));
    FK_CUDA(c, cudaStreamSynchronize(c->stream));
    if (*c->h_status) return fail(c, FK_EINVAL, status_text(*c->h_status));
  }
  return FK_OK;
}

// fk_reduce for callers that cannot allocate device memory (include/fk.h): device buffers only, the
// partial sums live in the library's fixed scratch array.  No cudaMalloc / cudaFree here or below.
int fk_reduce_static(fk_ctx* c, const double* weights, int m0, int m1, double* out) {
  if (!c) return FK_EINVAL;
  if (!weights || !out) return fail(c, FK_EINVAL, "weights or out is NULL");
  if (m0 < 0 || m1 > c->N + 1 || m0 >= m1) return fail(c, FK_EINVAL, "need 0 <= m0 < m1 <= N+1");
  const int chunks = (m1 - 1) / FK_CW - m0 / FK_CW + 1;
  if (chunks > FK_REDUCE_STATIC_MAX_CHUNKS) {
    char msg[200];
    std::snprintf(msg, sizeof msg,
                  "fk_reduce_static: columns %d..%d touch %d chunks of 32 columns, the fixed scratch "
                  "holds %d; split the range or use fk_reduce",
                  m0, m1 - 1, chunks, FK_REDUCE_STATIC_MAX_CHUNKS);
    return fail(c, FK_EINVAL, msg);
  }
  static_assert(FK_REDUCE_STATIC_MAX_CHUNKS == FK_REDUCE_STATIC_MAX_CHUNKS_ABI, "fk.h and fk_internal.h disagree");
  if (c->n_next != 0 && m1 > 1) return fail(c, FK_ESTATE, "columns other than 0 are final only after fk_evolve reached n_to = 0");
  if (*c->h_status) return fail(c, FK_EINVAL, status_text(*c->h_status));
  DeviceGuard guard(c->device);
  // both buffers are read / written by kernels: a host pointer would fault there, refuse it here
  const void* ptrs[2] = {weights, out};
  for (const void* p : ptrs) {
    cudaPointerAttributes at;
    FK_CUDA(c, cudaPointerGetAttributes(&at, p));
    if (at.type != cudaMemoryTypeDevice && at.type != cudaMemoryTypeManaged)
      return fail(c, FK_EINVAL, "fk_reduce_static: weights and out must be device memory");
  }
  FK_CUDA(c, fk_launch_reduce_static(c->g, c->d_P[c->cur], weights, m0, m1, out, c->device, c->stream));
  c->launches += 2;
  return FK_OK;
}

int fk_profile_updates(fk_ctx* c, double* updates) {
  if (!c) return FK_EINVAL;
  if (!updates) return fail(c, FK_EINVAL, "updates is NULL");
  for (int k = 0; k < FK_K_COUNT; ++k) updates[k] = c->class_updates[k];
  return FK_OK;
}

int fk_paths(fk_ctx* c, long long counts[FK_PATH_COUNT]) {
  if (!c) return FK_EINVAL;
  if (!counts) return fail(c, FK_EINVAL, "counts is NULL");
  if (!c->d_paths) return fail(c, FK_ESTATE, "fk_paths needs FK_FLAG_COUNT_PATHS at fk_create");
  DeviceGuard guard(c->device);
  unsigned long long h[FK_PATH_COUNT];
  FK_CUDA(c, cudaMemcpyAsync(h, c->d_paths, sizeof h, cudaMemcpyDeviceToHost, c->stream));
  FK_CUDA(c, cudaStreamSynchronize(c->stream));
  for (int k = 0; k < FK_PATH_COUNT; ++k) counts[k] = (long long)h[k];
  return FK_OK;
}

int fk_work(fk_ctx* c, double work[4]) {
  if (!c) return FK_EINVAL;
  if (!work) return fail(c, FK_EINVAL, "work is NULL");
  DeviceGuard guard(c->device);
  std::vector<unsigned long long> h((size_t)4 * c->N);
  FK_CUDA(c, cudaMemcpyAsync(h.data(), c->d_work, sizeof(unsigned long long) * h.size(), cudaMemcpyDeviceToHost, c->stream));
  FK_CUDA(c, cudaStreamSynchronize(c->stream));
  for (int k = 0; k < 4; ++k) work[k] = 0.0;
  for (int nu = 0; nu < c->N; ++nu) {                  // operator nu acts on the columns nu+1 .. N
    const double cols = c->N - nu;
    // autonomous: one operator, counted where it was assembled, applied at every evolved step
    const size_t at = 4 * (size_t)((c->autonomous && c->auto_assembled && nu >= c->n_next) ? c->auto_nu : nu);
    work[0] += (double)h[at + 0] * cols;
    work[1] += (double)h[at + 1] * cols * (c->g.d + 1);
    work[2] += (double)h[at + 2] * cols;
    work[3] += (double)h[at + 3] * cols * (c->g.d + 1);
  }
  return FK_OK;
}

int fk_peak_fp64(int device, void* stream, int iters, double* tflops, double* ms) {
  if (!tflops || !ms || iters < 1) return FK_EINVAL;
  int ndev = 0;
  if (cudaGetDeviceCount(&ndev) != cudaSuccess || device < 0 || device >= ndev) return FK_ECUDA;
  DeviceGuard guard(device);
  int sms = 0;
  if (cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, device) != cudaSuccess) return FK_ECUDA;
  const int blocks = 4 * sms, threads = 512;
  cudaStream_t st = (cudaStream_t)stream;
  double* out = nullptr;
  cudaEvent_t e0 = nullptr, e1 = nullptr;
  int rc = FK_ECUDA;
  float t = 0.f;
  if (cudaMalloc(&out, sizeof(double) * (size_t)blocks * threads) != cudaSuccess) return FK_ENOMEM;
  if (cudaEventCreate(&e0) == cudaSuccess && cudaEventCreate(&e1) == cudaSuccess &&
      fk_launch_dfma_peak(out, blocks, threads, iters, st) == cudaSuccess &&      // warm-up
      cudaEventRecord(e0, st) == cudaSuccess &&
      fk_launch_dfma_peak(out, blocks, threads, iters, st) == cudaSuccess &&
      cudaEventRecord(e1, st) == cudaSuccess && cudaEventSynchronize(e1) == cudaSuccess &&
      cudaEventElapsedTime(&t, e0, e1) == cudaSuccess && t > 0.f) {
    *ms = t;
    *tflops = 2.0 * 8.0 * iters * (double)blocks * threads / (t * 1e-3) * 1e-12;
    rc = FK_OK;
  }
  if (e0) cudaEventDestroy(e0);
  if (e1) cudaEventDestroy(e1);
  cudaFree(out);
  return rc;
}

int fk_profile(fk_ctx* c, int on) {
  if (!c) return FK_EINVAL;
  c->profiling = on != 0;
  return FK_OK;
}

int fk_profile_read(fk_ctx* c, double* ms, long long* launches) {
  if (!c) return FK_EINVAL;
  if (!ms || !launches) return fail(c, FK_EINVAL, "ms or launches is NULL");
  DeviceGuard guard(c->device);
  FK_CUDA(c, cudaStreamSynchronize(c->stream));
  for (int k = 0; k < FK_K_COUNT; ++k) { ms[k] = 0.0; launches[k] = 0; }
  for (auto& e : c->events) {
    float t = 0.f;
    FK_CUDA(c, cudaEventElapsedTime(&t, e.a, e.b));
    ms[e.cls] += t;
    ++launches[e.cls];
  }
  return FK_OK;
}

}  // extern "C"
