/* graphgp.h — C ABI of the B200-native GraphGP hot path (Vecchia conditioning).
 *
 * Source of every operation: arxiv/paper_2606_11402 as extracted in PAPER.md
 *   Eq. 1, Eq. 2, Alg. 1,
 *   §2.2 ordering/batches, §2.3 implementation.
 * Scope table: SURVEY.md §8(b).  Readings of silent/garbled passages: DESIGN.md §3.
 *
 * Conventions
 *   - 0-based indices.  All per-point arrays (x, xi, v, v_bar, xi_bar) are in GRAPH order: the
 *     paper's bit-reversed k-d tree order stably sorted by depth, head first.
 *   - K_ab = sigma^2 [ rho(|x_a - x_b|) + jitter * delta_ab ]  (relative nugget, R-7).
 *   - "device" = CUDA device memory of the current device; "host" = ordinary host memory.
 *   - Ownership: the caller owns every buffer, including the workspace.  The library allocates no
 *     memory on these calls.  Its only process state, all of it PER DEVICE: one internal high-priority
 *     stream and two events, created on first use and never destroyed (the dense head runs there beside
 *     the bulk kernel; everything is joined back into `cuda_stream` before a call returns its work to
 *     it), the cached SM count, the launch counter, and the optional kernel-timing events.  Calls may
 *     come from several host threads and on several devices (the side-stream events are taken under a
 *     per-device mutex; concurrent callers share the one side stream and are serialised on it); the
 *     kernel-timing diagnostic is meant for one thread.  Calls are asynchronous on `cuda_stream`
 *     (a cudaStream_t passed as void*; NULL = default stream) unless stated otherwise; a workspace must
 *     not be used by two calls in flight at once.
 *   - gp_forward and gp_vjp copy a small per-batch table from pageable host memory (staged by the runtime
 *     before the call returns); gp_forward with the dataflow launch polls device memory and carries a
 *     watchdog: if it ever fired, gp_check_errors returns GP_ERR_CUDA.
 *   - Errors: return codes only.  Argument errors are synchronous.  A numerical failure (a pivot or
 *     conditional variance that is not positive and finite) writes NaN for that point and increments
 *     a device counter that gp_check_errors() reads.
 *   - There is no CPU fallback: without a CUDA device every compute entry point returns GP_ERR_CUDA.
 */
#ifndef GRAPHGP_H_
#define GRAPHGP_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef enum {
  GP_OK = 0,
  GP_ERR_INVALID_ARG = 1,
  GP_ERR_UNSUPPORTED = 2, /* (k, d, dtype) outside what the call handles: k <= 128, d <= 4 for forward / inverse /
                             logdet and the builder; k <= 64 for the gradient, JVP and multi-sample calls */
  GP_ERR_NOT_PD = 3,
  GP_ERR_CUDA = 4,
  GP_ERR_WORKSPACE = 5, /* ws == NULL or ws_bytes < gp_workspace_bytes() */
  GP_ERR_TOO_LARGE = 6  /* gp_logdet_noalloc only: n0 > GP_NOALLOC_MAX_N0 or k > GP_NOALLOC_MAX_K (its scratch is a
                           fixed device array); use gp_logdet with a workspace instead */
} gp_status;

typedef enum { GP_KERNEL_SE = 0, GP_KERNEL_MATERN32 = 1, GP_KERNEL_EXP = 2 } gp_kernel_kind;
typedef enum { GP_F32 = 0, GP_F64 = 1 } gp_dtype;
typedef enum { GP_OP_FORWARD = 0, GP_OP_INVERSE = 1, GP_OP_LOGDET = 2, GP_OP_VJP = 3, GP_OP_BUILD = 4,
               GP_OP_FORWARD_MULTI = 5, GP_OP_INVERSE_MULTI = 6 } gp_op;

/* gp_graph.flags */
enum {
  GP_FLAG_PER_BATCH_LAUNCH = 1, /* forward/VJP: one launch per batch (Alg. 1 lines 2-8 literally) instead of
                                   the single dataflow launch; results agree to rounding */
  GP_FLAG_GENERIC_KERNEL = 2,   /* force the runtime-(k,d,kind) kernel even where a specialised one exists */
  GP_FLAG_FLOW_CARRY = 4,       /* dataflow forward: use the wait-first body (meant for large batches) everywhere */
  GP_FLAG_FLOW_WEIGHTS = 8      /* dataflow forward: use the wait-last body (meant for small batches) everywhere;
                                   without either flag the library picks per stretch of batches by their size */
};

/* Stationary covariance kappa(r) = sigma^2 rho(r); rho:
 *   SE        exp(-r^2 / (2 ell^2))
 *   MATERN32  (1 + sqrt(3) r / ell) exp(-sqrt(3) r / ell)
 *   EXP       exp(-r / ell)                                   (BASELINE.json configs) */
typedef struct {
  int32_t kind; /* gp_kernel_kind */
  double sigma, ell, jitter;
} gp_kernel;

/* The inputs of Alg. 1 `Require` except the noise. */
typedef struct {
  int64_t n;         /* number of points N                                                            */
  int64_t n0;        /* size of the dense initial block (Alg. 1 line 1); k <= n0 <= n    */
  int32_t d;         /* spatial dimension, 1..4                                                        */
  int32_t k;         /* neighbours per point, 1..128 (PAPER.md:53 sends k >~ 64 to JAX; here 64 < k <= 128 runs
                        on warp-per-point fp64 kernels: forward, inverse, logdet only)                  */
  int32_t n_batches; /* L                                                                              */
  int32_t dtype;     /* gp_dtype of x, xi, v, v_bar, xi_bar                                            */
  int32_t flags;     /* GP_FLAG_*                                                                      */
  int32_t reserved;
  const void* x;            /* device, [n][d] row-major, graph order, dtype                           */
  const int32_t* nbr;       /* device, [n - n0][k] row-major; row r belongs to point i = n0 + r; every
                               entry is a graph position < batch start of i; order inside a row is free */
  const int64_t* batch_off; /* HOST, [n_batches + 1]; batch_off[0] = n0, strictly increasing,
                               batch_off[n_batches] = n.  Points of one batch are conditionally
                               independent.                                              */
} gp_graph;

/* Bytes of workspace `op` needs for this graph (0 on invalid arguments). */
size_t gp_workspace_bytes(const gp_graph* g, int32_t op);

/* Forward generation, Alg. 1:  v[0:n0] = chol(K_head) xi[0:n0];  for each batch, for
 * every point i in it:  v_i = K_ic K_cc^-1 v_c + sqrt(K_ii - K_ic K_cc^-1 K_ci) xi_i   (Eq. 2).
 * xi: device [n] (in);  v: device [n] (out).                                                          */
gp_status gp_forward(const gp_graph* g, const gp_kernel* kern, const void* xi, void* v, void* ws,
                     size_t ws_bytes, void* cuda_stream);

/* Inverse ("easily parallelized"):  xi_i = (v_i - K_ic K_cc^-1 v_c) / s_i for all
 * i at once; head: xi[0:n0] = chol(K_head)^-1 v[0:n0].   v: device [n] (in);  xi: device [n] (out).   */
gp_status gp_inverse(const gp_graph* g, const gp_kernel* kern, const void* v, void* xi, void* ws,
                     size_t ws_bytes, void* cuda_stream);

/* Log-determinant of the Vecchia covariance:  sum_i log s_i^2  (+ log det K_head).
 * logdet_dev: device double[1] (out).  dlogdet_dtheta_dev: device double[2] = d/dsigma, d/dell, or NULL.
 * Workspace: gp_workspace_bytes(g, GP_OP_LOGDET) without the gradient; WITH the gradient the call needs the
 * larger gp_workspace_bytes(g, GP_OP_VJP) (the head carries 2 n0 extra rows), else GP_ERR_WORKSPACE.         */
gp_status gp_logdet(const gp_graph* g, const gp_kernel* kern, double* logdet_dev, double* dlogdet_dtheta_dev,
                    void* ws, size_t ws_bytes, void* cuda_stream);

/* gp_logdet for callers that cannot allocate device memory (code under CUDA graph capture, tight serving loops,
 * harnesses that forbid cudaMalloc): no workspace argument.  Same quantity as gp_logdet (Eq. 2 for
 * s_i^2), without the gradient.  The scratch - the n0 x n0 fp64 matrix of the dense head (Alg. 1 line 1) and the
 * accumulators - is ONE fixed array in device memory inside the library, gp_logdet_noalloc_scratch_bytes() = 8 MiB +
 * 4 KiB, which every GPU that loads the library holds until the process exits.  Hence the limits: n0 <=
 * GP_NOALLOC_MAX_N0 and k <= GP_NOALLOC_MAX_K, any n; beyond them the call returns GP_ERR_TOO_LARGE and launches
 * nothing.  The call enqueues kernels and one memset on `cuda_stream` and calls no cudaMalloc / cudaFree, creates no
 * stream or event, and uses no allocating library routine.  fp64 arithmetic whatever g->dtype; shared-memory kernels,
 * roughly an order of magnitude slower than gp_logdet.
 * g, kern: as for gp_logdet (g->batch_off is not used beyond validation).  logdet_dev: device double[1] (out), NaN if
 * any conditional or head pivot was not positive (there is no workspace to query with gp_check_errors).
 * ALL calls share the one array, and it keeps the last call's contents (what must start at zero is cleared by every
 * call): two calls whose GPU work overlaps - different streams, or host threads - on the same device RACE; callers
 * serialise them.  Per-device state: the array's device address, taken once per device on first use.             */
#define GP_NOALLOC_MAX_N0 1024
#define GP_NOALLOC_MAX_K 64
gp_status gp_logdet_noalloc(const gp_graph* g, const gp_kernel* kern, double* logdet_dev, void* cuda_stream);
size_t gp_logdet_noalloc_scratch_bytes(void);

/* Vector-Jacobian product of gp_forward ("backward derivatives"): given xi, v = forward(xi)
 * and a cotangent v_bar, returns xi_bar [n] and theta_bar = (d/dsigma, d/dell) of <v_bar, forward(xi; theta)>.
 * xi, v, v_bar: device [n] (in);  xi_bar: device [n] (out);  theta_bar_dev: device double[2] (out).
 * Floating-point atomics make the last bits of xi_bar/theta_bar run-dependent.                        */
gp_status gp_vjp(const gp_graph* g, const gp_kernel* kern, const void* xi, const void* v, const void* v_bar,
                 void* xi_bar, double* theta_bar_dev, void* ws, size_t ws_bytes, void* cuda_stream);

/* Forward-mode derivative of gp_forward ("forward ... derivatives"): at the point (xi, v = forward(xi; theta))
 * and along the tangent (xi_dot [n], sigma_dot, ell_dot) returns v_dot [n] = d forward.  xi, v, xi_dot: device [n] (in);
 * v_dot: device [n] (out).  <v_bar, v_dot> = <xi_bar, xi_dot> + theta_bar . (sigma_dot, ell_dot) with gp_vjp's outputs.
 * Workspace: gp_workspace_bytes(g, GP_OP_VJP).                                                                       */
gp_status gp_jvp(const gp_graph* g, const gp_kernel* kern, const void* xi, const void* v, const void* xi_dot, double sigma_dot,
                 double ell_dot, void* v_dot, void* ws, size_t ws_bytes, void* cuda_stream);

/* VJP of gp_inverse ("kernel parameter derivatives"): at (v, xi = inverse(v; theta)) and for a
 * cotangent xi_bar [n] on xi returns v_bar [n] and theta_bar = (d/dsigma, d/dell) of <xi_bar, inverse(v; theta)>.
 * Every point contributes independently (no sweep); v_bar is accumulated with floating-point atomics.
 * v, xi, xi_bar: device [n] (in);  v_bar: device [n] (out);  theta_bar_dev: device double[2] (out).
 * Workspace: gp_workspace_bytes(g, GP_OP_VJP).  (The gradient of the log-determinant is gp_logdet's second output.)   */
gp_status gp_inverse_vjp(const gp_graph* g, const gp_kernel* kern, const void* v, const void* xi, const void* xi_bar,
                         void* v_bar, double* theta_bar_dev, void* ws, size_t ws_bytes, void* cuda_stream);

/* Multi-sample apply: S = n_samples noise vectors on one graph and one set of kernel parameters (MGVI /
 * geoVI "require the forward pass for posterior sampling").  The conditioning of Eq. 2 - K, its
 * factor, the weights and s - is computed once per point and applied to every sample.  xi, v: device [n][S], row-major
 * (the S values of a point are contiguous), sample s of these calls equals gp_forward / gp_inverse on column s.
 * Shapes: fp32 k = 8, 16 and fp64 k = 8 with d = 2, 3 (others: GP_ERR_UNSUPPORTED); 1 <= S <= 1024.
 * Workspace: gp_workspace_bytes_multi(g, GP_OP_FORWARD_MULTI | GP_OP_INVERSE_MULTI, S).                              */
size_t gp_workspace_bytes_multi(const gp_graph* g, int32_t op, int32_t n_samples);
gp_status gp_forward_multi(const gp_graph* g, const gp_kernel* kern, int32_t n_samples, const void* xi, void* v, void* ws,
                           size_t ws_bytes, void* cuda_stream);
gp_status gp_inverse_multi(const gp_graph* g, const gp_kernel* kern, int32_t n_samples, const void* v, void* xi, void* ws,
                           size_t ws_bytes, void* cuda_stream);

/* End-to-end variants with HOST input/output vectors: the [n] input goes host->device into `in_dev`, the op runs,
 * the [n] result goes device->host (pinned host memory makes the copies asynchronous).  The graph stays device-
 * resident.  in_dev/out_dev: device staging, [n] each.  The op is cut into ranges of the graph order (a point reads
 * only points before it) and the copies of neighbouring ranges run on two library-internal copy streams (per device,
 * created on first use) beside the kernels; everything is ordered after the work already queued on `cuda_stream`,
 * and `cuda_stream` ends only when the result is on the host: the caller synchronises that stream and reads.        */
gp_status gp_forward_host(const gp_graph* g, const gp_kernel* kern, const void* xi_host, void* v_host,
                          void* in_dev, void* out_dev, void* ws, size_t ws_bytes, void* cuda_stream);
gp_status gp_inverse_host(const gp_graph* g, const gp_kernel* kern, const void* v_host, void* xi_host,
                          void* in_dev, void* out_dev, void* ws, size_t ws_bytes, void* cuda_stream);

/* gp_logdet with HOST results: the op, then logdet_dev -> logdet_host (and the gradient pair if
 * dlogdet_dtheta_host != NULL) on `cuda_stream`.  logdet_dev [1] / dlogdet_dtheta_dev [2]: device staging.
 * Workspace as for gp_logdet.                                                                              */
gp_status gp_logdet_host(const gp_graph* g, const gp_kernel* kern, double* logdet_host, double* dlogdet_dtheta_host,
                         double* logdet_dev, double* dlogdet_dtheta_dev, void* ws, size_t ws_bytes, void* cuda_stream);

/* gp_vjp with HOST xi, v, v_bar (in) and xi_bar, theta_bar[2] (out): three [n] host->device copies into the
 * device staging buffers xi_dev, v_dev, v_bar_dev, the VJP, then xi_bar_dev -> xi_bar_host and theta_bar_dev ->
 * theta_bar_host, all on `cuda_stream`.  The caller synchronises the stream before reading the results.  */
gp_status gp_vjp_host(const gp_graph* g, const gp_kernel* kern, const void* xi_host, const void* v_host,
                      const void* v_bar_host, void* xi_bar_host, double* theta_bar_host, void* xi_dev, void* v_dev,
                      void* v_bar_dev, void* xi_bar_dev, double* theta_bar_dev, void* ws, size_t ws_bytes,
                      void* cuda_stream);

/* Graph construction, separately timed, "plain":
 *   order   bit-reversed left-balanced k-d tree: node i at level l has children i+2^l, i+2^(l+1);
 *           split dimension = level mod d; ties by (coordinate, user id)             (R-3, R-4);
 *           sort-based: one radix sort per dimension, then a stable split of the sorted lists per level
 *   kNN     k nearest among PRECEDING points in that order, ranked by (fp64 FMA-free squared distance,
 *           tree index) (R-5); depth-first walk over the implicit tree restricted to indices < i
 *   depth   d_i = 1 + max_{j in c(i)} d_j by parallel fixed point; head depth 0
 *   sort    graph order = tree order stably sorted by depth; with GP_BUILD_SPATIAL_BATCHES points inside
 *           a batch are additionally ordered by Morton code of their coordinates (any order inside a batch is
 *           legal) so that neighbouring threads gather neighbouring memory.
 * x_user: device [n][d] dtype (in).  Outputs (device unless noted): perm [n] graph position -> user id;
 * x_graph [n][d] dtype; nbr [n-n0][k]; depth [n] (graph order); batch_off_host: HOST int64
 * [max_batches+1]; n_batches: HOST.  Synchronises the stream before returning (batch_off is host data).
 * Requires n < 2^31.                                                                                   */
enum { GP_BUILD_SPATIAL_BATCHES = 1,
       GP_BUILD_RADIUS_CLASSES = 2 /* inside a batch, order first by the class of the neighbourhood radius (distance to
                                      the farthest of the k neighbours, one class per two octaves), tight first, then
                                      as GP_BUILD_SPATIAL_BATCHES says.  Optional and off by default. */,
       GP_BUILD_PLAIN_KNN = 4      /* kNN by the plain walk (stack and candidate list in local memory) instead of the
                                      shared-memory walk (stack + max-heap of the k best) used for d <= 3 and
                                      every k <= 128.  Same result bit for bit; kept for comparison and as the path
                                      for larger k or d.                                                        */,
       GP_BUILD_PLAIN_ORDER = 8    /* tree order by one radix sort of (subtree, coordinate rank) keys per level
                                      instead of the presorted per-dimension lists split stably per level (one
                                      sort per dimension in all).  Same order bit for bit; kept for comparison. */ };
gp_status gp_graph_build(const void* x_user, int64_t n, int32_t d, int32_t k, int64_t n0, int32_t dtype,
                         int32_t build_flags, int64_t* perm, void* x_graph, int32_t* nbr, int32_t* depth,
                         int64_t* batch_off_host, int32_t max_batches, int32_t* n_batches, void* ws,
                         size_t ws_bytes, void* cuda_stream);
size_t gp_graph_build_workspace_bytes(int64_t n, int32_t d, int32_t k, int32_t dtype);
/* Optional per-stage device times of the last gp_graph_build on this workspace, milliseconds:
 * [0] order, [1] kNN, [2] depth, [3] depth sort + remap.  HOST double[4].                              */
gp_status gp_graph_build_times(void* ws, double* ms4_host);

/* Number of points whose conditional was not positive definite in the last op that used `ws`.
 * Synchronous: copies one counter from the device (the caller must have synchronised the stream).     */
gp_status gp_check_errors(void* ws, int64_t* n_bad_points);

const char* gp_status_string(gp_status s);

/* Diagnostics: 1 if (dtype, k, d, kind) has a register-resident specialised kernel, else 0.           */
int32_t gp_has_specialised(int32_t dtype, int32_t k, int32_t d, int32_t kind);
/* Kernel timing for the roofline report (bench.py).  While enabled, every op brackets its DOMINANT kernel(s) -
 * the conditioning kernels over the points i >= n0: the dataflow forward launches, the inverse / logdet kernel,
 * the VJP geometry + scatter kernels - with CUDA events recorded on the stream they are launched on.
 * gp_kernel_time_last synchronises on the closing event and returns the device time between the two events of
 * the most recent op in milliseconds (GP_ERR_INVALID_ARG if nothing was recorded).  Off by default.             */
void gp_kernel_time_enable(int32_t on);
gp_status gp_kernel_time_last(double* ms_host);

/* Non-tensor ALU rates of the current device, measured with register-resident loops ("measure
 * with a register-resident FMA loop under the same clocks").  bench.py prints them beside the NOMINAL peak that
 * roofline.frac is taken against.  out_host[i], i < min(n_out, GP_PEAK_COUNT), in TFLOP/s (2 flop per fma lane;
 * MUFU: 1e12 results/s; the two mixed variants count the work of both pipes / of the packed fmas only):
 *   GP_PEAK_FFMA scalar 3-register fma; GP_PEAK_FFMA_IMM scalar fma with an immediate; GP_PEAK_FFMA2 packed
 *   fma.rn.f32x2; GP_PEAK_FFMA2_BC packed fma with a broadcast scalar operand (the Cholesky update of the packed
 *   kernels); GP_PEAK_DFMA; GP_PEAK_MUFU (ex2.approx); GP_PEAK_FFMA2_DFMA and GP_PEAK_FFMA2_MUFU (two pipes at once).
 * Synchronous (times about 30 short launches with CUDA events on `cuda_stream`).  ws: device scratch >= 256 bytes. */
enum { GP_PEAK_FFMA = 0, GP_PEAK_FFMA_IMM = 1, GP_PEAK_FFMA2 = 2, GP_PEAK_FFMA2_BC = 3, GP_PEAK_DFMA = 4,
       GP_PEAK_MUFU = 5, GP_PEAK_FFMA2_DFMA = 6, GP_PEAK_FFMA2_MUFU = 7, GP_PEAK_COUNT = 8 };
gp_status gp_measure_alu_peak(double* out_host, int32_t n_out, void* ws, size_t ws_bytes, void* cuda_stream);

/* Number of kernels launched by the library in this process so far (for bench.py's gpu_launches).    */
int64_t gp_launch_count(void);

#ifdef __cplusplus
}
#endif
#endif /* GRAPHGP_H_ */
