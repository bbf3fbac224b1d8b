// C ABI of include/graphgp.h: argument validation, workspace carving, dispatch.  No torch types,
// no allocation, no global state except the launch counter used by bench.py's gpu_launches.
#include <atomic>
#include <cstring>
#include <mutex>

#include "gp_common.cuh"

namespace gp {
static std::atomic<long long> g_launches{0};
void count_launch(int n) { g_launches.fetch_add(n, std::memory_order_relaxed); }

// Per-device state, safe for several host threads: creation and every record + wait pair run under the device's
// mutex (an event may be re-recorded as soon as the wait on its previous record has been enqueued, so the pair only
// has to be atomic with respect to other callers).  Work of concurrent callers shares the one side stream of the
// device and is serialised on it; each caller's fork / join still orders it against that caller's own stream.
static std::mutex g_dev_mutex[64];

int device_sm_count() {
  static std::atomic<int> sms[64];
  int dev = 0;
  if (cudaGetDevice(&dev) != cudaSuccess || dev < 0 || dev >= 64) return 0;
  int v = sms[dev].load(std::memory_order_relaxed);
  if (v == 0) {
    if (cudaDeviceGetAttribute(&v, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess) return 0;
    sms[dev].store(v, std::memory_order_relaxed);
  }
  return v;
}

gp_status side_stream(SideStream** out) {
  static SideStream per_dev[64];
  int dev = 0;
  GP_CUDA_OK(cudaGetDevice(&dev));
  if (dev < 0 || dev >= 64) return GP_ERR_CUDA;
  std::lock_guard<std::mutex> lock(g_dev_mutex[dev]);
  SideStream& s = per_dev[dev];
  if (!s.stream) {
    int lo = 0, hi = 0;
    GP_CUDA_OK(cudaDeviceGetStreamPriorityRange(&lo, &hi));
    GP_CUDA_OK(cudaStreamCreateWithPriority(&s.stream, cudaStreamNonBlocking, hi));
    GP_CUDA_OK(cudaEventCreateWithFlags(&s.fork, cudaEventDisableTiming));
    GP_CUDA_OK(cudaEventCreateWithFlags(&s.join, cudaEventDisableTiming));
    s.device = dev;
  }
  *out = &s;
  return GP_OK;
}
gp_status copy_streams(cudaStream_t* cin, cudaStream_t* cout) {
  static cudaStream_t per_dev[64][2];
  int dev = 0;
  GP_CUDA_OK(cudaGetDevice(&dev));
  if (dev < 0 || dev >= 64) return GP_ERR_CUDA;
  std::lock_guard<std::mutex> lock(g_dev_mutex[dev]);
  if (!per_dev[dev][0]) {
    GP_CUDA_OK(cudaStreamCreateWithFlags(&per_dev[dev][0], cudaStreamNonBlocking));
    GP_CUDA_OK(cudaStreamCreateWithFlags(&per_dev[dev][1], cudaStreamNonBlocking));
  }
  *cin = per_dev[dev][0];
  *cout = per_dev[dev][1];
  return GP_OK;
}
gp_status side_fork(const SideStream* s, cudaStream_t main) {
  std::lock_guard<std::mutex> lock(g_dev_mutex[s->device]);
  GP_CUDA_OK(cudaEventRecord(s->fork, main));
  GP_CUDA_OK(cudaStreamWaitEvent(s->stream, s->fork, 0));
  return GP_OK;
}
gp_status side_join(const SideStream* s, cudaStream_t main) {
  std::lock_guard<std::mutex> lock(g_dev_mutex[s->device]);
  GP_CUDA_OK(cudaEventRecord(s->join, s->stream));
  GP_CUDA_OK(cudaStreamWaitEvent(main, s->join, 0));
  return GP_OK;
}

// Kernel timing (a diagnostic for bench.py, off by default): one event pair per device; meant for one host thread.
static std::atomic<int> g_ktime_on{0};
struct KTime { cudaEvent_t e0 = nullptr, e1 = nullptr; bool recorded = false; };
static KTime g_kt[64];
static KTime* ktime_slot() {
  int dev = 0;
  if (cudaGetDevice(&dev) != cudaSuccess || dev < 0 || dev >= 64) return nullptr;
  return &g_kt[dev];
}
gp_status ktime_begin(cudaStream_t st) {
  if (!g_ktime_on.load(std::memory_order_relaxed)) return GP_OK;
  KTime* k = ktime_slot();
  if (!k) return GP_ERR_CUDA;
  if (!k->e0) { GP_CUDA_OK(cudaEventCreate(&k->e0)); GP_CUDA_OK(cudaEventCreate(&k->e1)); }
  GP_CUDA_OK(cudaEventRecord(k->e0, st));
  return GP_OK;
}
gp_status ktime_end(cudaStream_t st) {
  if (!g_ktime_on.load(std::memory_order_relaxed)) return GP_OK;
  KTime* k = ktime_slot();
  if (!k || !k->e0) return GP_OK;
  GP_CUDA_OK(cudaEventRecord(k->e1, st));
  k->recorded = true;
  return GP_OK;
}

gp_status validate_graph(const gp_graph* g, const gp_kernel* kern) {
  if (!g || !kern) return GP_ERR_INVALID_ARG;
  if (g->n <= 0 || g->n0 < 0 || g->n0 > g->n) return GP_ERR_INVALID_ARG;
  if (g->dtype != GP_F32 && g->dtype != GP_F64) return GP_ERR_INVALID_ARG;
  if (g->d < 1 || g->k < 1) return GP_ERR_INVALID_ARG;
  if (g->d > kMaxD || g->k > kMaxK) return GP_ERR_UNSUPPORTED;
  if (g->n >= (1LL << 31)) return GP_ERR_UNSUPPORTED;
  if (g->n0 < g->k && g->n0 < g->n) return GP_ERR_INVALID_ARG;  // every row needs k predecessors
  if (g->n_batches < 0 || g->n_batches > kMaxBatches) return GP_ERR_INVALID_ARG;
  if (!g->x) return GP_ERR_INVALID_ARG;
  if (g->n > g->n0) {
    if (!g->nbr || !g->batch_off || g->n_batches < 1) return GP_ERR_INVALID_ARG;
    if (g->batch_off[0] != g->n0 || g->batch_off[g->n_batches] != g->n) return GP_ERR_INVALID_ARG;
    for (int b = 0; b < g->n_batches; ++b)
      if (g->batch_off[b + 1] <= g->batch_off[b]) return GP_ERR_INVALID_ARG;
  } else if (g->n_batches != 0 && !g->batch_off) {
    return GP_ERR_INVALID_ARG;
  }
  if (kern->kind < 0 || kern->kind > 2) return GP_ERR_INVALID_ARG;
  if (!(kern->sigma > 0.0) || !(kern->ell > 0.0) || !(kern->jitter >= 0.0)) return GP_ERR_INVALID_ARG;
  return GP_OK;
}

static gp_status make_ctx(const gp_graph* g, const gp_kernel* kern, int op, void* ws, size_t ws_bytes,
                          void* stream, OpCtx* out) {
  GP_OK_OR_RETURN(validate_graph(g, kern));
  WsLayout lay = ws_layout(g, op);
  if (!ws || ws_bytes < lay.total || (((uintptr_t)ws) & 255) != 0) return GP_ERR_WORKSPACE;
  int ndev = 0;
  if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev == 0) return GP_ERR_CUDA;
  out->g = g; out->kern = kern; out->ws = (char*)ws; out->lay = lay; out->st = (cudaStream_t)stream;
  return GP_OK;
}
}  // namespace gp

using namespace gp;

extern "C" {

size_t gp_workspace_bytes(const gp_graph* g, int32_t op) {
  if (!g || g->n <= 0 || g->n0 < 0 || g->n0 > g->n || g->n_batches < 0 || op < GP_OP_FORWARD || op > GP_OP_VJP)
    return 0;
  return ws_layout(g, op).total;
}

gp_status gp_forward(const gp_graph* g, const gp_kernel* kern, const void* xi, void* v, void* ws, size_t ws_bytes,
                     void* cuda_stream) {
  OpCtx c;
  GP_OK_OR_RETURN(make_ctx(g, kern, GP_OP_FORWARD, ws, ws_bytes, cuda_stream, &c));
  if (!xi || !v) return GP_ERR_INVALID_ARG;
  return run_forward(c, xi, v);
}

gp_status gp_inverse(const gp_graph* g, const gp_kernel* kern, const void* v, void* xi, void* ws, size_t ws_bytes,
                     void* cuda_stream) {
  OpCtx c;
  GP_OK_OR_RETURN(make_ctx(g, kern, GP_OP_INVERSE, ws, ws_bytes, cuda_stream, &c));
  if (!xi || !v) return GP_ERR_INVALID_ARG;
  return run_inverse(c, v, xi);
}

gp_status gp_logdet(const gp_graph* g, const gp_kernel* kern, double* logdet_dev, double* dlogdet_dtheta_dev,
                    void* ws, size_t ws_bytes, void* cuda_stream) {
  OpCtx c;
  GP_OK_OR_RETURN(make_ctx(g, kern, dlogdet_dtheta_dev ? GP_OP_VJP : GP_OP_LOGDET, ws, ws_bytes, cuda_stream, &c));
  if (!logdet_dev) return GP_ERR_INVALID_ARG;
  return run_logdet(c, logdet_dev, dlogdet_dtheta_dev);
}

gp_status gp_vjp(const gp_graph* g, const gp_kernel* kern, const void* xi, const void* v, const void* v_bar,
                 void* xi_bar, double* theta_bar_dev, void* ws, size_t ws_bytes, void* cuda_stream) {
  OpCtx c;
  GP_OK_OR_RETURN(make_ctx(g, kern, GP_OP_VJP, ws, ws_bytes, cuda_stream, &c));
  if (!xi || !v || !v_bar || !xi_bar || !theta_bar_dev) return GP_ERR_INVALID_ARG;
  if (g->k > kMaxKGrad) return GP_ERR_UNSUPPORTED;
  return run_vjp(c, xi, v, v_bar, xi_bar, theta_bar_dev);
}

gp_status gp_jvp(const gp_graph* g, const gp_kernel* kern, const void* xi, const void* v, const void* xi_dot, double sigma_dot,
                 double ell_dot, void* v_dot, void* ws, size_t ws_bytes, void* cuda_stream) {
  OpCtx c;
  GP_OK_OR_RETURN(make_ctx(g, kern, GP_OP_VJP, ws, ws_bytes, cuda_stream, &c));
  if (!xi || !v || !xi_dot || !v_dot) return GP_ERR_INVALID_ARG;
  if (g->k > kMaxKGrad) return GP_ERR_UNSUPPORTED;
  return run_jvp(c, xi, v, xi_dot, sigma_dot, ell_dot, v_dot);
}

gp_status gp_inverse_vjp(const gp_graph* g, const gp_kernel* kern, const void* v, const void* xi, const void* xi_bar,
                         void* v_bar, double* theta_bar_dev, void* ws, size_t ws_bytes, void* cuda_stream) {
  OpCtx c;
  GP_OK_OR_RETURN(make_ctx(g, kern, GP_OP_VJP, ws, ws_bytes, cuda_stream, &c));
  if (!xi || !v || !xi_bar || !v_bar || !theta_bar_dev) return GP_ERR_INVALID_ARG;
  if (g->k > kMaxKGrad) return GP_ERR_UNSUPPORTED;
  return run_inverse_vjp(c, v, xi, xi_bar, v_bar, theta_bar_dev);
}

gp_status gp_forward_host(const gp_graph* g, const gp_kernel* kern, const void* xi_host, void* v_host, void* in_dev,
                          void* out_dev, void* ws, size_t ws_bytes, void* cuda_stream) {
  if (!g || !xi_host || !v_host || !in_dev || !out_dev) return GP_ERR_INVALID_ARG;
  OpCtx c;
  GP_OK_OR_RETURN(make_ctx(g, kern, GP_OP_FORWARD, ws, ws_bytes, cuda_stream, &c));
  HostIO io;
  io.in_host[0] = xi_host;
  io.out_host = v_host;
  GP_OK_OR_RETURN(copy_streams(&io.cin, &io.cout));
  c.io = &io;
  return run_forward(c, in_dev, out_dev);
}

gp_status gp_inverse_host(const gp_graph* g, const gp_kernel* kern, const void* v_host, void* xi_host, void* in_dev,
                          void* out_dev, void* ws, size_t ws_bytes, void* cuda_stream) {
  if (!g || !xi_host || !v_host || !in_dev || !out_dev) return GP_ERR_INVALID_ARG;
  OpCtx c;
  GP_OK_OR_RETURN(make_ctx(g, kern, GP_OP_INVERSE, ws, ws_bytes, cuda_stream, &c));
  HostIO io;
  io.in_host[0] = v_host;
  io.out_host = xi_host;
  GP_OK_OR_RETURN(copy_streams(&io.cin, &io.cout));
  c.io = &io;
  return run_inverse(c, in_dev, out_dev);
}

gp_status gp_logdet_host(const gp_graph* g, const gp_kernel* kern, double* logdet_host, double* dlogdet_dtheta_host,
                         double* logdet_dev, double* dlogdet_dtheta_dev, void* ws, size_t ws_bytes, void* cuda_stream) {
  if (!g || !logdet_host || !logdet_dev || (dlogdet_dtheta_host && !dlogdet_dtheta_dev)) return GP_ERR_INVALID_ARG;
  cudaStream_t st = (cudaStream_t)cuda_stream;
  GP_OK_OR_RETURN(gp_logdet(g, kern, logdet_dev, dlogdet_dtheta_host ? dlogdet_dtheta_dev : nullptr, ws, ws_bytes, cuda_stream));
  GP_CUDA_OK(cudaMemcpyAsync(logdet_host, logdet_dev, sizeof(double), cudaMemcpyDeviceToHost, st));
  if (dlogdet_dtheta_host)
    GP_CUDA_OK(cudaMemcpyAsync(dlogdet_dtheta_host, dlogdet_dtheta_dev, 2 * sizeof(double), cudaMemcpyDeviceToHost, st));
  return GP_OK;
}

gp_status gp_vjp_host(const gp_graph* g, const gp_kernel* kern, const void* xi_host, const void* v_host,
                      const void* v_bar_host, void* xi_bar_host, double* theta_bar_host, void* xi_dev, void* v_dev,
                      void* v_bar_dev, void* xi_bar_dev, double* theta_bar_dev, void* ws, size_t ws_bytes,
                      void* cuda_stream) {
  if (!g || !xi_host || !v_host || !v_bar_host || !xi_bar_host || !theta_bar_host || !xi_dev || !v_dev || !v_bar_dev ||
      !xi_bar_dev || !theta_bar_dev)
    return GP_ERR_INVALID_ARG;
  OpCtx c;
  GP_OK_OR_RETURN(make_ctx(g, kern, GP_OP_VJP, ws, ws_bytes, cuda_stream, &c));
  if (g->k > kMaxKGrad) return GP_ERR_UNSUPPORTED;
  HostIO io;
  io.in_host[0] = xi_host;
  io.in_host[1] = v_host;
  io.in_host[2] = v_bar_host;
  io.out_host = xi_bar_host;
  GP_OK_OR_RETURN(copy_streams(&io.cin, &io.cout));
  c.io = &io;
  GP_OK_OR_RETURN(run_vjp(c, xi_dev, v_dev, v_bar_dev, xi_bar_dev, theta_bar_dev));
  GP_CUDA_OK(cudaMemcpyAsync(theta_bar_host, theta_bar_dev, 2 * sizeof(double), cudaMemcpyDeviceToHost, (cudaStream_t)cuda_stream));
  return GP_OK;
}

gp_status gp_check_errors(void* ws, int64_t* n_bad_points) {
  if (!ws || !n_bad_points) return GP_ERR_INVALID_ARG;
  Control h;
  GP_CUDA_OK(cudaMemcpy(&h, ws, sizeof(Control), cudaMemcpyDeviceToHost));
  *n_bad_points = (int64_t)h.n_bad;
  if (h.timeout) return GP_ERR_CUDA;
  return h.n_bad ? GP_ERR_NOT_PD : GP_OK;
}

const char* gp_status_string(gp_status s) {
  switch (s) {
    case GP_OK: return "ok";
    case GP_ERR_INVALID_ARG: return "invalid argument";
    case GP_ERR_UNSUPPORTED: return "unsupported (k, d, dtype) or size";
    case GP_ERR_NOT_PD: return "a conditional covariance was not positive definite";
    case GP_ERR_CUDA: return "CUDA error or no CUDA device";
    case GP_ERR_WORKSPACE: return "workspace missing, misaligned or too small";
    case GP_ERR_TOO_LARGE: return "size beyond the fixed scratch of gp_logdet_noalloc (n0 <= 1024, k <= 64): use gp_logdet";
  }
  return "unknown status";
}

int32_t gp_has_specialised(int32_t dtype, int32_t k, int32_t d, int32_t kind) {
  return has_specialised(dtype, k, d, kind) ? 1 : 0;
}

void gp_kernel_time_enable(int32_t on) { g_ktime_on.store(on ? 1 : 0, std::memory_order_relaxed); }
gp_status gp_kernel_time_last(double* ms_host) {
  KTime* k = ktime_slot();
  if (!ms_host || !k || !k->recorded) return GP_ERR_INVALID_ARG;
  GP_CUDA_OK(cudaEventSynchronize(k->e1));
  float ms = 0.f;
  GP_CUDA_OK(cudaEventElapsedTime(&ms, k->e0, k->e1));
  *ms_host = (double)ms;
  return GP_OK;
}

int64_t gp_launch_count(void) { return (int64_t)g_launches.load(std::memory_order_relaxed); }

}  // extern "C"
