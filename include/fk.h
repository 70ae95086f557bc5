/* fk.h -- C ABI of the B200-native Feynman-Kac exit-time hot path (arXiv 2104.14561).
 *
 * The path: for every time step, push each grid node one Euler-Maruyama step to its
 * tensor-product Gauss-Hermite points (Eq. 11, 21), interpolate the exit
 * probability there with piecewise cubic Hermite polynomials (Eq. 13-15),
 * give points that left the box the absorbing value, fold the quadrature weights into the
 * sparse step operator A_nu = Q Psi^nu (Eq. 24-27), and apply the operators
 * to all output-time columns in one backward pass (Algorithm 1), which
 * yields P(t_m, x_j) for every t_m in [0, T_max].
 *
 * Every step of that path runs in CUDA kernels for sm_100a inside this library; there is no
 * CPU fallback.  All entry points return an int code (FK_OK = 0) and never throw.  The library
 * COPIES what it is given.  A HOST buffer may be freed or reused as soon as the call returns.
 * A DEVICE buffer (FK_MEM_DEVICE) is copied by work queued on the context's stream: it must
 * stay valid and unmodified until that stream has reached the copy (order your own work on the
 * same stream, or synchronise it -- fk_check does).  Device work is ordered on the stream given to
 * fk_create (the library also owns a side stream on which it assembles the next step's operator
 * while the current step's kernels run; it is joined to the caller's stream with events, so
 * everything a caller can observe is ordered on the caller's stream); calls on one context must
 * not be made concurrently from several threads.
 *
 * Index conventions.  d = dimension (1..3); n[k] nodes along dimension k; node index
 * j = ((i0*n[1])+i1)*n[2]+i2 (last dimension fastest); J = prod n[k].  Steps: dt, N,
 * T_max = N*dt, t_nu = nu*dt.  Operator nu (0..N-1) uses the coefficients sampled at t_nu
 * (explicit Euler).  Column m (0..N) is P(t_m, .); column 0 is chi (Eq. 28,
 * PAPER.md:268); column m = A_0 A_1 ... A_{m-1} chi (Eq. 29).
 */
#ifndef FK_B200_H
#define FK_B200_H

#ifdef __cplusplus
extern "C" {
#endif

typedef struct fk_ctx fk_ctx; /* opaque; owned by the library; free with fk_destroy */

enum { FK_OK = 0, FK_EINVAL = 1, FK_ENOMEM = 2, FK_ECUDA = 3, FK_ESTATE = 4 };

/* Face rule for a quadrature point that leaves the box through that face (R8/R9):
 * ABSORB: the point contributes face_value (1 = "exit", the paper's absorbing value); grid
 *         nodes lying on an ABSORB face are Dirichlet nodes held at face_value.
 * CLAMP : the point is projected back onto the face and interpolated there; nodes on a CLAMP
 *         face are updated like interior nodes.
 * CLAMP dimensions are projected first; among the remaining dimensions that are outside, the
 * lowest dimension index decides the value. */
/* PERIODIC (both faces of a dimension or neither; R21; "periodic in x1"):
 *         x[k][n-1] is the image of x[k][0] one period L = beta - alpha later; a point is
 *         wrapped into [alpha, beta) before it is located; Eq. 15 uses the cell across the seam
 *         at the first / last node; both end nodes are updated like interior nodes (give them the
 *         same coefficients).  Problems with a periodic dimension run on the generic kernels. */
enum { FK_FACE_ABSORB = 0, FK_FACE_CLAMP = 1, FK_FACE_PERIODIC = 2 };

/* FK_MEM_HOST_PINNED (fk_set_coeffs / fk_set_coeffs_range only): a page-locked HOST buffer that the
 * caller keeps valid and unmodified until the context's stream has reached the copy, exactly like a
 * device buffer.  The call then only queues the copies and returns without synchronising, so the
 * upload of the next ring piece overlaps the kernels of the current one (config 5 streams 81 GB of
 * coefficients through its ring).  With pageable memory the copies are still correct but no longer
 * asynchronous. */
enum { FK_MEM_HOST = 0, FK_MEM_DEVICE = 1, FK_MEM_HOST_PINNED = 2 };

/* fk_params.flags */
enum {
  FK_FLAG_VALIDATE = 1,  /* check every coefficient read by an updated node for NaN / Inf on the
                            device while the operator is assembled (costs two compares per
                            value); a hit is reported like a negative sigma, see fk_check */
  FK_FLAG_MULTISTEP = 4, /* 1-D problems (no periodic face, Eq. 15 as printed, a line that fits shared
                            memory): run the steps of an fk_evolve call in batches -- one launch
                            assembles the operators of up to a few hundred steps, one launch applies
                            them with each group of columns resident in shared memory (several
                            operators per pass over P: SURVEY.md section 8(f)'s temporal blocking).
                            Same results up to summation order.  Off by default: measured faster
                            only on short lines */
  FK_FLAG_COUNT_PATHS = 8, /* testing aid: count, per group of four rows and step, which contraction path
                            of the blocked 2-D / 3-D apply kernels the group took (fk_paths); one
                            predicated atomic per group */
  FK_FLAG_WEIGHTED_SLOPES = 2  /* nodal slopes by the Fritsch-Carlson weighted harmonic mean
                            (ref [17]; R22) instead of Eq. 15 as printed:
                            (w1+w2)/(w1/d_{j-1} + w2/d_j), w1 = 2h_j + h_{j-1}, w2 = h_j + 2h_{j-1};
                            equal to Eq. 15 on uniform grids, meant for non-uniform ones */
};

#define FK_ALL_STEPS (-1)
#define FK_MAX_Q 32

/* Problem statement (PAPER.md:49-51 box and SDE; 117-123 time partition; 134 tensor mesh;
 * 197-204 Gauss-Hermite rule).  All pointers are HOST pointers read during fk_create only. */
typedef struct {
  int d;                   /* 1..3 */
  int n[3];                /* nodes per dimension, each >= 3 (Eq. 15's end rule needs two
                              divided differences); unused entries ignored */
  const double* x[3];      /* x[k][0..n[k]-1], strictly increasing; x[k][0] = alpha_k and
                              x[k][n[k]-1] = beta_k are the faces of the box; may be
                              non-uniform */
  double dt;               /* > 0 */
  int N;                   /* >= 1 time steps; N+1 output columns */
  int Q[3];                /* Gauss-Hermite points per dimension, 1..FK_MAX_Q */
  int face_kind[3][2];     /* [dim][0 = lower face, 1 = upper face] */
  double face_value[3][2]; /* g of ABSORB faces; ignored for CLAMP */
  int coeff_slots;         /* number of per-step coefficient slots kept on the device:
                              N (or 0) = the full table; 1 <= s < N = a ring, step nu lives in
                              slot nu % s and must be (re)loaded before fk_evolve needs it */
  int device;              /* CUDA device ordinal (compute capability 10.x) */
  void* stream;            /* cudaStream_t (e.g. from torch); NULL = the legacy default stream */
  unsigned flags;          /* FK_FLAG_* or 0 */
  int shard_index;         /* column sharding (the columns are independent): this */
  int shard_count;         /* context keeps and updates only the 32-column chunks c with
                              c % shard_count == shard_index; 0 or 1 = all columns.  Shards never
                              exchange data; fk_read / fk_reduce of a shard write only the columns
                              it owns and leave the other entries of `out` untouched */
} fk_params;

/* Validate, build the Gauss-Hermite tables, allocate device state and fill both P buffers
 * with chi (Algorithm 1's "P = repmat(chi)").  On failure *out is NULL and the
 * code says why (FK_EINVAL: bad parameter; FK_ENOMEM: device allocation; FK_ECUDA). */
int fk_create(const fk_params* p, fk_ctx** out);

/* Drift b and per-dimension noise amplitude sigma (diagonal sigma of Eq. 1)
 * sampled on the nodes at t_step: b[d][J], sigma[d][J], fp64, in host (mem = FK_MEM_HOST) or
 * device (FK_MEM_DEVICE, same device) memory.  step in 0..N-1 fills slot step % coeff_slots;
 * step = FK_ALL_STEPS declares the problem autonomous: the one slice is used by every step.
 * Values at Dirichlet nodes are never read.  sigma must be >= 0 at updated nodes: a negative
 * sigma (it would reverse the order of the quadrature points) is detected on the device when
 * the step's operator is assembled and reported as FK_EINVAL by fk_check, by the next fk_read
 * to host memory, or by a later fk_evolve / fk_read that finds the flag already raised; the
 * columns computed from such a step are undefined.  Non-finite values are reported the same
 * way when FK_FLAG_VALIDATE is set, and are undefined (they propagate as NaN) otherwise.
 * Copies are stream-ordered; a host buffer may be reused when the call returns (the call
 * synchronises the stream for FK_MEM_HOST sources; FK_MEM_HOST_PINNED sources are not waited for,
 * see above). */
int fk_set_coeffs(fk_ctx* c, int step, const double* b, const double* sigma, int mem);

/* Same for `count` consecutive steps step0..step0+count-1: b and sigma are [count][d][J].
 * count must not exceed coeff_slots. */
int fk_set_coeffs_range(fk_ctx* c, int step0, int count, const double* b, const double* sigma,
                        int mem);

/* Algorithm 1's loop for n = n_from, n_from-1, ..., n_to+1: assemble the
 * operator nu = n-1 once and update columns n..N.  The first call after fk_create/fk_reset
 * must have n_from = N; later calls continue where the previous one stopped (n_from = its
 * n_to); after n_to = 0 all columns are final.  With FK_FLAG_MULTISTEP a 1-D problem
 * runs its steps in batches (see the flag).  Kernels are queued on the stream and the call
 * returns without waiting for them, with one exception: on 2-D grids the first fk_evolve after
 * a coefficient load synchronises the stream once to read back, per loaded step, which rows
 * leave the fused kernel's halo (a few integers), so that the kernels of each step can be
 * chosen on the host.  FK_ESTATE: wrong n_from, or a needed coefficient slot does not hold that
 * step.  FK_EINVAL: a coefficient error found on the device by an earlier step (see fk_check). */
int fk_evolve(fk_ctx* c, int n_from, int n_to);

/* Refill P with chi and rewind to n = N; coefficient slots are kept.  Clears the device's error
 * flag (see fk_check); to do that safely the call waits until the kernels of the last fk_evolve on
 * this context have finished (not for anything queued after them). */
int fk_reset(fk_ctx* c);

/* Copy columns m0..m1-1 out as out[(m1-m0)][J] (row m-m0 = P(t_m, .), node index fastest),
 * to host or device memory.  Valid for any column once fk_evolve has reached n_to = 0; before
 * that only column 0 and, after reaching n, nothing else is final (FK_ESTATE).  The call
 * synchronises the stream when `mem` is FK_MEM_HOST. */
int fk_read(fk_ctx* c, int m0, int m1, double* out, int mem);

/* Weighted reduction over the nodes of every requested column, straight from the device layout:
 * out[m - m0] = sum_j weights[j] * P(t_m, x_j) for m0 <= m < m1 (weights[J] and out[m1-m0] in
 * host or device memory, same kind `mem` for both).  With w_j = (quadrature weight of node j) *
 * P_init(x_j) this is the exit probability for initial conditions distributed as P_init,
 * int P(t,x) P_init(x) dx; with w_j = 2 pi n_0 f_M(p_j) * (quadrature weight)
 * on the nodes of the slice r = r_0 and 0 elsewhere it is the moment n_RE(r_0, t) of Eq. 42
 * (PAPER.md:453).  The sum over nodes runs in a fixed order (reproducible).  State rules as
 * fk_read; synchronises the stream when `mem` is FK_MEM_HOST. */
int fk_reduce(fk_ctx* c, const double* weights, int m0, int m1, double* out, int mem);

/* fk_reduce without any device allocation: same sums, same fixed summation order (the results are
 * bit-identical to fk_reduce on device buffers), for callers that must not -- or cannot -- call
 * cudaMalloc at this point.  Who that is: a program whose device memory is already fully handed out
 * (a framework's caching allocator that has taken the rest of the GPU, or simply config-5-sized
 * contexts that leave no room: a late cudaMalloc there fails with out-of-memory), and a program
 * that reduces inside a loop it cannot afford to stall (cudaMalloc and cudaFree make the whole
 * device wait, other streams included; fk_reduce grows its scratch with them whenever a call needs
 * more than the one before).
 *
 * How: fk_reduce's only scratch, the per-block partial sums of its first pass, sits in a fixed
 * array compiled into the library: FK_REDUCE_STATIC_MAX_CHUNKS_ABI x 64 x 32 doubles = 1 MiB of
 * device memory on every GPU that loads the library, kept until the process exits whether or not
 * this call is ever used.  That bounds what one call can take: the columns m0..m1-1 may touch at
 * most FK_REDUCE_STATIC_MAX_CHUNKS_ABI = 64 of the 32-column chunks (chunk = m / 32), i.e. any range
 * of up to 2017 columns, 2048 when m0 is a multiple of 32 (configs 1, 2, 3 and 5 in one call;
 * config 4's 5001 columns in three).  A wider range is refused with FK_EINVAL and a message that
 * says so; nothing is launched then.
 *
 * weights[J] and out[m1-m0] are the caller's and must both be DEVICE memory on the context's device
 * (anything else is refused with FK_EINVAL: there is no room to stage a host array without
 * allocating).  The call queues two kernels on the context's stream and returns without waiting;
 * `out` is ready when the stream has passed them.  State rules and shard behaviour as fk_reduce.
 *
 * Shared state, read this: the array belongs to the library, not to a context.  Every call on a
 * device, from whatever context or stream, uses the same memory, so two calls whose kernels can be
 * on the GPU at the same time (different streams, different contexts, different threads) corrupt
 * each other's sums -- keep them on one stream or order them with events.  Calls that run one
 * after the other are safe: nothing in the array needs to start at zero, the second pass reads only
 * what the first pass of the same call wrote, so leftovers of an earlier call never count.
 *
 * First call on each device: looks up the device address of the array (cudaGetSymbolAddress, once
 * per device, with that device current) and remembers it; later calls only launch.  Make that
 * first call during start-up, before any stream capture begins on that device. */
#define FK_REDUCE_STATIC_MAX_CHUNKS_ABI 64
int fk_reduce_static(fk_ctx* c, const double* weights, int m0, int m1, double* out);

/* Synchronise the context's stream and report what the device found since the last fk_reset:
 * FK_OK, or FK_EINVAL with fk_last_error naming the first kind of bad coefficient (negative
 * sigma at an updated node; NaN / Inf with FK_FLAG_VALIDATE). */
int fk_check(fk_ctx* c);

/* Per-kernel-class device time of the fk_evolve calls since the last fk_reset, measured with
 * CUDA events on the launching stream when profiling is on (fk_profile(c, 1)); ms[FK_K_COUNT]
 * and launches[FK_K_COUNT] are indexed FK_K_ASSEMBLE, FK_K_SLOPES, FK_K_APPLY (the generic
 * slopes / apply pair), FK_K_FUSED (the fused 2-D slopes+apply kernel), FK_K_ROWBLOCK (the
 * 3-D apply kernel that contracts four rows at a time), FK_K_FAR2D (the 2-D apply kernel of the
 * rows the fused kernel leaves out) and FK_K_LINE1D (the 1-D kernel that runs a batch of steps per
 * launch; its batch assembly is booked under FK_K_ASSEMBLE).  Synchronises the
 * stream.  FK_K_ASSEMBLE is timed on the side stream, overlapped with other kernels: the classes
 * do not add up to the duration of the step. */
enum { FK_K_ASSEMBLE = 0, FK_K_SLOPES = 1, FK_K_APPLY = 2, FK_K_FUSED = 3, FK_K_ROWBLOCK = 4,
       FK_K_FAR2D = 5, FK_K_LINE1D = 6, FK_K_COUNT = 7 };
int fk_profile(fk_ctx* c, int on);
int fk_profile_read(fk_ctx* c, double* ms, long long* launches);

/* Node-step updates each kernel class processed since the last fk_reset (rows it owns x active
 * columns, Dirichlet rows excluded), host-side bookkeeping of fk_evolve: updates[FK_K_COUNT].
 * FK_K_ASSEMBLE counts operator rows assembled (one per updated node and step). */
int fk_profile_updates(fk_ctx* c, double* updates);

/* With FK_FLAG_COUNT_PATHS: how many (group of four adjacent rows, step) pairs each contraction path
 * of the blocked apply kernels served since fk_create (synchronises the stream).  3-D (fk_rowblock3d):
 * SAME = the four rows put their dimension-0 / 1 entries on the same nodes, static dimension-2 slots;
 * MERGED = contracted on the union of the rows' entry lists; WIDE / WIDE_MERGED = the same two with
 * the dimension-2 weights spread over a dense union window (rows that reach beyond two nodes along a
 * non-uniform last dimension); ROWWISE = one row at a time (lists too long for the staging, a
 * periodic or too wide dimension 2).  2-D (fk_far2d): BANDED = dense union window along dimension 1,
 * SCATTERED = entry by entry.  FK_ESTATE without the flag.  The tests use it to prove that the path a
 * parity case is meant for actually ran. */
enum { FK_PATH_3D_SAME = 0, FK_PATH_3D_MERGED = 1, FK_PATH_3D_WIDE = 2, FK_PATH_3D_WIDE_MERGED = 3,
       FK_PATH_3D_ROWWISE = 4, FK_PATH_2D_BANDED = 5, FK_PATH_2D_SCATTERED = 6, FK_PATH_COUNT = 8 };
int fk_paths(fk_ctx* c, long long counts[FK_PATH_COUNT]);

/* Algorithmic work of the steps evolved since the last fk_reset, counted on the device while the
 * operators are assembled (synchronises the stream): work[0] = node-step updates on rows the fused
 * 2-D kernel owns, work[1] = their row-contraction multiply-adds, sum over steps of (active
 * columns) x sum over rows of (d+1) prod_k D_k with D_k the distinct nodes the row touches along
 * dimension k (the non-zeros of a row of Q Psi), work[2], work[3] = the same for
 * all other updated rows.  The slopes of Eq. 15 cost about 14 d more operations per update
 * (SURVEY.md section 8(d)). */
int fk_work(fk_ctx* c, double work[4]);

/* Measurement only, no context: the device's fp64 fused-multiply-add rate.  Launches
 * 4 x (SM count) blocks x 512 threads, each thread running 8 independent chains of `iters`
 * dependent fma; timed with CUDA events on `stream`, second of two launches.
 * *tflops = 2 flops x 8 x iters x threads / time; *ms = that time. */
int fk_peak_fp64(int device, void* stream, int iters, double* tflops, double* ms);

/* Total kernels launched by this context since fk_create (all entry points). */
long long fk_launch_count(const fk_ctx* c);

void fk_destroy(fk_ctx* c);

/* Text of the last error on this context ("" if none); for a failed fk_create pass NULL. */
const char* fk_last_error(const fk_ctx* c);

/* Gauss-Hermite rule the library uses (a ascending, weights summing to 1); for inspection. */
int fk_gauss_hermite(int Q, double* a, double* w);

#ifdef __cplusplus
}
#endif
#endif /* FK_B200_H */
