// Shared device/host definitions for the GraphGP sm_100a kernels.
// Nothing here is shared with oracle/ (which has its own, independent arithmetic).
#pragma once
#include <cuda_runtime.h>
#include <math.h>
#include <stddef.h>
#include <stdint.h>

#include "../../include/graphgp.h"

namespace gp {

constexpr int kMaxK = 128;       // 64 < k <= 128: warp-per-point kernels (gp_large.cu), forward / inverse / logdet only
constexpr int kMaxKGrad = 64;    // gradients, JVP, multi-sample calls
constexpr int kMaxD = 4;
constexpr int kCtrlBytes = 2048;
constexpr int kAccSlots = 64;
constexpr int kMaxBatches = 1 << 20;
constexpr int kFlowTickets = 32;   // dataflow forward: launches (stretches of batches) with their own ticket counter

// First kCtrlBytes of every workspace; zeroed by the library at the start of each op.
struct Control {
  unsigned long long n_bad;    // points whose conditional was not positive definite
  unsigned long long ticket;   // dataflow forward: next chunk to hand out
  unsigned long long timeout;  // dataflow watchdog fired (a bug, never expected)
  unsigned long long done;     // dataflow VJP: points whose cotangent scatter is complete (reverse order)
  double acc[8];               // [0] logdet  [1] dlogdet/dsigma  [2] dlogdet/dell  [3] theta_bar sigma  [4] theta_bar ell
  double build_ms[4];          // graph builder stage times
  unsigned long long pad[4];
  double slots[2][kAccSlots];  // dataflow VJP: per-warp partial sums of sigma_bar / ell_bar, spread to avoid one hot address
  unsigned long long flow_ticket[kFlowTickets];  // dataflow forward: next 128-point group of each launch
};
static_assert(sizeof(Control) <= kCtrlBytes, "control block");

// Packed per-point record the register-resident kernels gather: coordinates (d <= 3, unused slots 0)
// and the point's value in ONE aligned 4-scalar record, so a neighbour costs one 16 B (fp32) / 32 B
// (fp64) load = one L2 sector, instead of d+1 scattered 4 B loads.
template <typename T> struct alignas(4 * sizeof(T)) Rec { T x0, x1, x2, v; };

// Kernel parameters in the working precision, unit-sigma form:  K/sigma^2 = rho + eps*delta.
// q = qscale * |x_a - x_b|^2 is the argument the correlation needs (see rho_from_q); the difference
// is taken on the RAW coordinates (exact for nearby points), the scale applied afterwards.
template <typename T>
struct KParams {
  T qscale;  // fp32 (base-2 exponent): SE log2e/(2 ell^2); Matern-3/2 3 log2e^2/ell^2; EXP log2e^2/ell^2
             // fp64 (natural exponent): SE 1/(2 ell^2);   Matern-3/2 3/ell^2;          EXP 1/ell^2
  T eps;     // relative jitter
  T sigma;
  T diag;    // 1 + eps
  T inv_ell;
  T sq;      // sqrt(qscale): the packed fp32 path scales the centred coordinates once instead of every q
  T inv_diag;  // 1 / (1 + eps)
};

template <typename T> __host__ inline KParams<T> make_kparams(const gp_kernel& k);
template <> __host__ inline KParams<float> make_kparams<float>(const gp_kernel& k) {
  const double log2e = 1.4426950408889634074;
  KParams<float> p;
  double s = 0;
  switch (k.kind) {
    case GP_KERNEL_SE: s = 0.5 * log2e / (k.ell * k.ell); break;
    case GP_KERNEL_MATERN32: s = 3.0 * log2e * log2e / (k.ell * k.ell); break;
    default: s = log2e * log2e / (k.ell * k.ell); break;
  }
  p.qscale = (float)s; p.eps = (float)k.jitter; p.sigma = (float)k.sigma; p.diag = (float)(1.0 + k.jitter);
  p.inv_ell = (float)(1.0 / k.ell);
  p.sq = (float)sqrt(s);
  p.inv_diag = (float)(1.0 / (1.0 + k.jitter));
  return p;
}
template <> __host__ inline KParams<double> make_kparams<double>(const gp_kernel& k) {
  KParams<double> p;
  double s = 0;
  switch (k.kind) {
    case GP_KERNEL_SE: s = 0.5 / (k.ell * k.ell); break;
    case GP_KERNEL_MATERN32: s = 3.0 / (k.ell * k.ell); break;
    default: s = 1.0 / (k.ell * k.ell); break;
  }
  p.qscale = s; p.eps = k.jitter; p.sigma = k.sigma; p.diag = 1.0 + k.jitter; p.inv_ell = 1.0 / k.ell;
  p.sq = sqrt(s);
  p.inv_diag = 1.0 / (1.0 + k.jitter);
  return p;
}

// ---- per-precision math -------------------------------------------------------------------------
template <typename T> struct Math;
template <> struct Math<float> {
  static __device__ __forceinline__ float rsqrt_approx(float x) { float y; asm("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x)); return y; }
  // MUFU.RSQ (about 2 ulp) + one Newton step: error well below the fp32 rounding of the factor itself
  static __device__ __forceinline__ float rsqrt(float x) {
    float y = rsqrt_approx(x);
    float h = 0.5f * y;
    float e = fmaf(-x * y, h, 0.5f);   // 0.5 - 0.5 x y^2
    return fmaf(y, e, y);
  }
  static __device__ __forceinline__ float sqrt_approx(float x) { float y; asm("sqrt.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x)); return y; }
  static __device__ __forceinline__ float sqrt(float x) { return sqrtf(x); }
  static __device__ __forceinline__ float ex2(float x) { float y; asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x)); return y; }
  static __device__ __forceinline__ float fma(float a, float b, float c) { return fmaf(a, b, c); }
  static __device__ __forceinline__ float log(float x) { return logf(x); }
  static __device__ __forceinline__ float fmin(float a, float b) { return fminf(a, b); }
  // rho as a function of q = qscale * |x_a - x_b|^2 (base-2 exponent folded in).
  template <int KIND> static __device__ __forceinline__ float rho_from_q(float q) {
    if (KIND == GP_KERNEL_SE) return ex2(-q);
    float t = sqrt_approx(q);                            // MUFU.SQRT: sqrt(0) = 0, no guard needed
    if (KIND == GP_KERNEL_MATERN32) return fmaf(t, 0.69314718055994530942f, 1.0f) * ex2(-t);
    return ex2(-t);
  }
  // ell * d rho / d ell  as a function of q (dimensionless; the caller divides by ell).
  template <int KIND> static __device__ __forceinline__ float drho_from_q(float q) {
    const float ln2 = 0.69314718055994530942f;
    if (KIND == GP_KERNEL_SE) return 2.0f * ln2 * q * ex2(-q);            // rho * r^2/ell^2
    float t = sqrt_approx(q);
    if (KIND == GP_KERNEL_MATERN32) { float a = t * ln2; return a * a * ex2(-t); }   // a^2 e^-a
    return t * ln2 * ex2(-t);                                               // rho * r/ell
  }
};
// e^-a for a >= 0 in double, branch-free, coefficients in constant memory (operands of the DFMAs themselves).  The
// library exp costs the fp64 lane-group kernels a quarter of their instructions in constants moved through uniform
// registers at every call site and in the branches around its special cases (profiles/r2_ncu_full.md).  Cody-Waite
// reduction a = n ln2 + r', |r'| <= ln2 / 2, degree-13 Taylor polynomial of e^-r' (truncation 6e-18), scaling by the
// exponent field; a > 700 gives 0.  Error about 1 ulp, as the library's.
__constant__ double kExpNegC[14] = {1.0, 1.0, 0.5, 1.0 / 6, 1.0 / 24, 1.0 / 120, 1.0 / 720, 1.0 / 5040, 1.0 / 40320,
                                    1.0 / 362880, 1.0 / 3628800, 1.0 / 39916800, 1.0 / 479001600, 1.0 / 6227020800.0};
__device__ __forceinline__ double exp_neg(double a) {
  const double shift = 6755399441055744.0;                      // 1.5 * 2^52: round to nearest integer in the low bits
  const double t = ::fma(a, 1.4426950408889634074, shift);
  const int n = __double2loint(t);
  const double nf = t - shift;
  double r = ::fma(nf, 6.93147180369123816490e-01, -a);         // r = n ln2 - a = -r'
  r = ::fma(nf, 1.90821492927058770002e-10, r);
  double p = kExpNegC[13];
#pragma unroll
  for (int q = 12; q >= 0; --q) p = ::fma(p, r, kExpNegC[q]);
  const double scale = __hiloint2double((1023 - n) << 20, 0);   // 2^-n, n <= 1010 where it is used
  return a > 700.0 ? 0.0 : p * scale;
}

// sqrt(q) for q >= 0 in double without the library's special-case branch: fp32 MUFU seed of 1 / sqrt(q), two Newton
// steps (2^-22 -> 2^-44 -> 2^-88), one residual correction of q y.  q below 1e-30 (squared distances of points that
// coincide to 15 digits) gives 0: an absolute error of 1e-15 in a, far below everything else.
__device__ __forceinline__ double sqrt_pos(double q) {
  double y = (double)rsqrtf((float)q);
  const double h = 0.5 * q;
  y = y * ::fma(-h * y, y, 1.5);
  y = y * ::fma(-h * y, y, 1.5);
  double a = q * y;
  a = ::fma(::fma(-a, a, q), 0.5 * y, a);
  return q < 1e-30 ? 0.0 : a;
}

template <> struct Math<double> {
  static __device__ __forceinline__ double rsqrt(double x) { return 1.0 / ::sqrt(x); }
  static __device__ __forceinline__ double sqrt(double x) { return ::sqrt(x); }
  static __device__ __forceinline__ double fma(double a, double b, double c) { return ::fma(a, b, c); }
  static __device__ __forceinline__ double log(double x) { return ::log(x); }
  static __device__ __forceinline__ double fmin(double a, double b) { return ::fmin(a, b); }
  template <int KIND> static __device__ __forceinline__ double rho_from_q(double q) {
    if (KIND == GP_KERNEL_SE) return exp_neg(q);
    double a = sqrt_pos(q);
    if (KIND == GP_KERNEL_MATERN32) return (1.0 + a) * exp_neg(a);
    return exp_neg(a);
  }
  template <int KIND> static __device__ __forceinline__ double drho_from_q(double q) {
    if (KIND == GP_KERNEL_SE) return 2.0 * q * ::exp(-q);
    double a = ::sqrt(q);
    if (KIND == GP_KERNEL_MATERN32) return a * a * ::exp(-a);
    return a * ::exp(-a);
  }
};

// runtime-kind versions (generic kernel, dense head)
template <typename T> __device__ __forceinline__ T rho_rt(int kind, T q) {
  switch (kind) {
    case GP_KERNEL_SE: return Math<T>::template rho_from_q<GP_KERNEL_SE>(q);
    case GP_KERNEL_MATERN32: return Math<T>::template rho_from_q<GP_KERNEL_MATERN32>(q);
    default: return Math<T>::template rho_from_q<GP_KERNEL_EXP>(q);
  }
}
template <typename T> __device__ __forceinline__ T drho_rt(int kind, T q) {
  switch (kind) {
    case GP_KERNEL_SE: return Math<T>::template drho_from_q<GP_KERNEL_SE>(q);
    case GP_KERNEL_MATERN32: return Math<T>::template drho_from_q<GP_KERNEL_MATERN32>(q);
    default: return Math<T>::template drho_from_q<GP_KERNEL_EXP>(q);
  }
}

// ---- host-side helpers ---------------------------------------------------------------------------
void count_launch(int n = 1);

#define GP_CUDA_OK(expr)                                   \
  do {                                                     \
    cudaError_t e__ = (expr);                              \
    if (e__ != cudaSuccess) return GP_ERR_CUDA;            \
  } while (0)
#define GP_OK_OR_RETURN(expr)                              \
  do {                                                     \
    gp_status s__ = (expr);                                \
    if (s__ != GP_OK) return s__;                          \
  } while (0)
#define GP_LAUNCH_CHECK()                                  \
  do {                                                     \
    gp::count_launch();                                    \
    if (cudaGetLastError() != cudaSuccess) return GP_ERR_CUDA; \
  } while (0)

inline size_t align_up(size_t v, size_t a) { return (v + a - 1) / a * a; }
inline size_t dtype_bytes(int dtype) { return dtype == GP_F64 ? 8 : 4; }

// Workspace layout (byte offsets from ws).  The head is always factored in fp64.
//   ctrl     Control
//   boff     dataflow VJP: per batch in reverse order {first chunk, first point, end point, end chunk} (int64 x 4)
//   gtab     dataflow forward: per 128-point group {first point, end of its batch} (int64 x 2)
//   head     (n0 + carried) x n0 doubles: factor of K_head/sigma^2 + carried rows (+ n0 doubles for the VJP)
//   rec      packed records Rec<T>[n]                          (register-resident kernels only)
//   g        VJP: running cotangent, T[n]
struct WsLayout {
  size_t ctrl_off, boff_off, gtab_off, head_off, rec_off, g_off, wbuf_off, total;
  size_t head_rows;
};
inline WsLayout ws_layout(const gp_graph* g, int op) {
  WsLayout w{};
  size_t B = dtype_bytes(g->dtype);
  size_t n0 = (size_t)g->n0, n = (size_t)g->n;
  size_t off = 0;
  w.ctrl_off = off; off += kCtrlBytes;
  w.boff_off = off; off += align_up(4 * ((size_t)g->n_batches + 1) * sizeof(int64_t), 256);
  // dataflow forward: one {first point, batch end} entry per 128-point group, groups aligned to batches
  w.gtab_off = off;
  if (op == GP_OP_FORWARD) off += align_up(((n - n0) / 128 + (size_t)g->n_batches + 1) * 2 * sizeof(int64_t), 256);
  // carried rows: inverse 1 (v_head); gradients 2 n0 (identity -> L^-T, and ell dM/dell -> its L^-1 image)
  size_t carried = (op == GP_OP_INVERSE) ? 1 : (op == GP_OP_VJP ? 2 * n0 : 0);
  w.head_rows = n0 + carried;
  size_t head_elems = w.head_rows * n0;
  if (op == GP_OP_VJP) head_elems += n0;  // p = L^T g_head
  w.head_off = off; off += align_up(head_elems * sizeof(double), 256);
  w.rec_off = off; off += align_up(n * 4 * B, 256);
  w.g_off = off;
  if (op == GP_OP_VJP) off += align_up(n * B, 256);
  // per conditioned point the k weights and {s, A_i, B_i, ok} (two-phase VJP, JVP, inverse VJP), working dtype
  w.wbuf_off = off;
  if (op == GP_OP_VJP) off += align_up((n - n0) * ((size_t)g->k + 4) * B, 256);
  w.total = off;
  return w;
}

// Host-buffer variants (gp_*_host): the [n] inputs live in (pinned) host memory and the result goes back to it.  The
// op is cut into ranges of the graph order (a point only reads points before it) so that the host->device copy of a
// later range and the device->host copy of an earlier one run on two library-internal copy streams beside the kernels.
struct HostIO {
  const void* in_host[3] = {nullptr, nullptr, nullptr};   // forward: xi; inverse: v; vjp: xi, v, v_bar
  void* out_host = nullptr;
  cudaStream_t cin = nullptr, cout = nullptr;
};
gp_status copy_streams(cudaStream_t* cin, cudaStream_t* cout);   // per device, created on first use, never destroyed

// events of one call (no timing); destroyed when the call returns (CUDA releases them once they have completed)
struct EventBag {
  cudaEvent_t ev[64];
  int used = 0;
  cudaEvent_t make() {
    if (used >= 64) return nullptr;
    if (cudaEventCreateWithFlags(&ev[used], cudaEventDisableTiming) != cudaSuccess) return nullptr;
    return ev[used++];
  }
  ~EventBag() { for (int i = 0; i < used; ++i) cudaEventDestroy(ev[i]); }
};
// `waiter` waits for everything queued on `src` so far
inline gp_status stream_after(EventBag& bag, cudaStream_t waiter, cudaStream_t src) {
  cudaEvent_t e = bag.make();
  if (!e) return GP_ERR_CUDA;
  if (cudaEventRecord(e, src) != cudaSuccess) return GP_ERR_CUDA;
  if (cudaStreamWaitEvent(waiter, e, 0) != cudaSuccess) return GP_ERR_CUDA;
  return GP_OK;
}

struct OpCtx {
  const gp_graph* g;
  const gp_kernel* kern;
  char* ws;
  WsLayout lay;
  cudaStream_t st;
  const HostIO* io = nullptr;
  Control* ctrl() const { return (Control*)(ws + lay.ctrl_off); }
  int64_t* boff_dev() const { return (int64_t*)(ws + lay.boff_off); }
  void* gtab() const { return ws + lay.gtab_off; }
  double* head() const { return (double*)(ws + lay.head_off); }
  void* rec() const { return ws + lay.rec_off; }
  void* gbar() const { return ws + lay.g_off; }
  float* wbuf() const { return (float*)(ws + lay.wbuf_off); }
};

// Fork/join helper: the dense head is independent of the bulk conditioning in gp_inverse / gp_logdet / gp_vjp,
// so it runs on a library-internal high-priority stream between a fork event (recorded on the caller's
// stream) and a join event (waited on by the caller's stream).  One stream and two events per device are
// created lazily on first use and never destroyed; everything stays ordered with respect to the caller's stream.
// Thread-safe (per-device mutex around creation and around each record + wait pair).
struct SideStream {
  cudaStream_t stream = nullptr;
  cudaEvent_t fork = nullptr, join = nullptr;
  int device = 0;
};
int device_sm_count();   // SMs of the current device (cached per device), 0 on error
gp_status side_stream(SideStream** out);
gp_status side_fork(const SideStream* s, cudaStream_t main);   // side waits for everything queued on main so far
gp_status side_join(const SideStream* s, cudaStream_t main);   // main waits for everything queued on side so far

// bench.py's roofline: events around the dominant kernel(s) of the current op, on the launching stream
gp_status ktime_begin(cudaStream_t st);
gp_status ktime_end(cudaStream_t st);

// ---- entry points implemented across the .cu files ------------------------------------------------
// dense head (gp_head.cu)
// overlapped: the factorisation runs beside the bulk kernel on the side stream -> use few CTAs so that most
// SMs keep their full bulk occupancy; otherwise (forward: the head is on the critical path) one CTA per SM.
gp_status head_factor(const OpCtx& c, const void* carried_src /*dtype [n0] or null*/, int n_carried, bool overlapped = false);
// build + factor with `n_carried` extra rows that the caller has already written below the square part
gp_status head_factor_preinit(const OpCtx& c, int n_carried, bool overlapped);
gp_status head_forward(const OpCtx& c, const void* xi, void* v, void* rec, bool rec_is_packed);
gp_status validate_graph(const gp_graph* g, const gp_kernel* kern);   // gp_api.cu: synchronous argument checks
gp_status head_inverse_out(const OpCtx& c, void* xi);
gp_status head_logdet(const OpCtx& c, double* acc /*device: acc[0] += logdet head*/,
                      double* grad_ell_acc /*device or null: += ell * d/dell, needs head_factor(c, nullptr, 2 n0)*/);
gp_status head_vjp(const OpCtx& c, const void* xi, const void* gbar, void* xibar,
                   double* acc /*device: acc[0] += sigma_bar, acc[1] += ell * ell_bar*/);

// conditioning (gp_ops.cu, gp_vjp.cu)
gp_status run_forward(const OpCtx& c, const void* xi, void* v);
gp_status run_inverse(const OpCtx& c, const void* v, void* xi);
gp_status run_logdet(const OpCtx& c, double* logdet, double* grad);
gp_status run_vjp(const OpCtx& c, const void* xi, const void* v, const void* vbar, void* xibar, double* thetabar);
gp_status run_logdet_grad(const OpCtx& c);   // conditioning part of d logdet / d ell into ctrl->acc[2]
// gp_vjp.cu: packs the records and writes, for every point i >= n0, the k weights w = K_cc^-1 K_ci (wbuf [n - n0][k]) and
// {s (unit sigma), A_i = ell dv_i/dell, B_i = dv_i/dsigma, ok} (sab [n - n0][4], after the weights), all in the working dtype
gp_status run_geometry(const OpCtx& c, const void* xi, const void* v);
// gp_jvp.cu
gp_status run_jvp(const OpCtx& c, const void* xi, const void* v, const void* xi_dot, double sigma_dot, double ell_dot, void* v_dot);
gp_status run_inverse_vjp(const OpCtx& c, const void* v, const void* xi, const void* xi_bar, void* v_bar, double* theta_bar);
bool has_specialised(int dtype, int k, int d, int kind);
// gp_large.cu: k > 64; op = GP_OP_FORWARD / INVERSE (in -> out) / LOGDET (logdet_dev)
gp_status run_large(const OpCtx& c, int op, const void* in, void* out, double* logdet);

}  // namespace gp
