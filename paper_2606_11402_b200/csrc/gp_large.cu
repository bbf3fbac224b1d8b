// Large-k path: the paper keeps the conditioning matrices in registers and says "k cannot be
// arbitrarily large ... for applications that require k >~ 64, the JAX version should be used".  Here
// 64 < k <= 128 runs on the GPU as well: ONE CTA (256 threads) per point, the joint (k + 2) x (k + 1) triangle of Alg. 1
// (rows 0..k-1 the neighbours, row k the point itself, row k + 1 the carried values) in shared memory,
// rows dealt to the warps and columns to the lanes in every right-looking step (a warp per point left the GPU idle:
// 71 KB of triangle per warp = 2 warps per SM, 2.45 s for 2^20 points at k = 128).  The arithmetic is fp64 whatever the working
// dtype: at this size the triangle no longer fits registers anyway, the FP64 pipe of sm_100a runs at half the FP32
// rate, and the fp32 accuracy question (gamma form) does not arise.  Forward: one launch per batch (Alg. 1 lines 2-8).
// Gradients, JVP and the multi-sample calls are not provided for k > 64 (GP_ERR_UNSUPPORTED).
#include "gp_cond.cuh"

namespace gp {

enum { LOP_FORWARD = 0, LOP_INVERSE = 1, LOP_LOGDET = 2 };

__host__ __device__ inline size_t large_warp_doubles(int k, int d) {
  return (size_t)(k + 2) * (k + 3) / 2 + (size_t)(k + 1) * d;      // triangle + coordinates
}

constexpr int kLargeThreads = 256;

template <typename T, int OP>
__global__ void __launch_bounds__(kLargeThreads)
cond_cta_kernel(const T* __restrict__ x, const T* vals, const int32_t* __restrict__ nbr, const T* in, T* out,
                int64_t start, int64_t n0, int d, int k, int kind, KParams<double> kp, Control* ctrl) {
  extern __shared__ double smem_large[];
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5, nwarp = kLargeThreads / 32;
  const int64_t i = start + blockIdx.x;                            // one point per CTA
  double* A = smem_large;                                          // tri(r, c), rows 0 .. k + 1
  double* X = A + (size_t)(k + 2) * (k + 3) / 2;                   // [k + 1][d], row k = the point itself
  const int32_t* row = nbr + (i - n0) * k;
  for (int r = tid; r <= k; r += kLargeThreads) {
    const int64_t p = r == k ? i : (int64_t)row[r];
    for (int t = 0; t < d; ++t) X[r * d + t] = (double)x[p * d + t];
    if (r < k) A[tri(k + 1, r)] = OP == LOP_LOGDET ? 0.0 : (double)vals[p];
  }
  if (tid == 0) A[tri(k + 1, k)] = 0.0;
  __syncthreads();
  // joint matrix M = K / sigma^2: rows dealt to warps, columns to lanes
  for (int r = warp; r <= k; r += nwarp) {
    for (int c = lane; c < r; c += 32) {
      double d2 = 0.0;
      for (int t = 0; t < d; ++t) { const double dx = X[r * d + t] - X[c * d + t]; d2 = fma(dx, dx, d2); }
      A[tri(r, c)] = rho_rt<double>(kind, d2 * kp.qscale);
    }
    if (lane == 0) A[tri(r, r)] = kp.diag;
  }
  __syncthreads();
  // right-looking Cholesky, values row carried; column k is not scaled:
  // A[k][k] = s^2, A[k + 1][k] = -m.  Per step: scale column j, then rows j+1 .. k+1 dealt to warps, columns to lanes.
  double minpiv = kp.diag;
  for (int j = 0; j < k; ++j) {
    const double piv = A[tri(j, j)];
    minpiv = fmin(minpiv, piv);
    const double inv = 1.0 / sqrt(piv);
    __syncthreads();                                               // everyone has read the pivot before column j changes
    for (int r = j + 1 + tid; r <= k + 1; r += kLargeThreads) A[tri(r, j)] *= inv;
    __syncthreads();
    for (int r = j + 1 + warp; r <= k + 1; r += nwarp) {
      const double lrj = A[tri(r, j)];
      const int cmax = r < k ? r : k;
      for (int c = j + 1 + lane; c <= cmax; c += 32) A[tri(r, c)] = fma(-lrj, A[tri(c, j)], A[tri(r, c)]);
    }
    __syncthreads();
  }
  if (tid == 0) {
    const double s2 = A[tri(k, k)], m = -A[tri(k + 1, k)];
    minpiv = fmin(minpiv, s2);
    const bool ok = minpiv > 0.0 && s2 == s2 && s2 < 1e300;
    const double ss = kp.sigma * sqrt(s2);
    if (!ok) atomicAdd(&ctrl->n_bad, 1ULL);
    const double nanv = __longlong_as_double(0x7ff8000000000000LL);
    if (OP == LOP_FORWARD) out[i] = (T)(ok ? fma(ss, (double)in[i], m) : nanv);
    else if (OP == LOP_INVERSE) out[i] = (T)(ok ? ((double)in[i] - m) / ss : nanv);
    else if (ok) atomicAdd(&ctrl->slots[0][blockIdx.x % kAccSlots], 2.0 * log(ss));   // spread: one hot address otherwise
  }
}

__global__ void large_logdet_sum_kernel(Control* ctrl) {
  if (threadIdx.x == 0 && blockIdx.x == 0) {
    double a = 0.0;
    for (int q = 0; q < kAccSlots; ++q) a += ctrl->slots[0][q];
    atomicAdd(&ctrl->acc[0], a);
  }
}

template <typename T, int OP>
static gp_status launch_large(const OpCtx& c, const T* vals, const T* in, T* out, int64_t start, int64_t end) {
  const int64_t cnt = end - start;
  if (cnt <= 0) return GP_OK;
  if (cnt > 0x7fffffffLL) return GP_ERR_UNSUPPORTED;
  const int k = c.g->k, d = c.g->d;
  const size_t smem = large_warp_doubles(k, d) * sizeof(double);
  if (smem > 220 * 1024) return GP_ERR_UNSUPPORTED;
  GP_CUDA_OK(cudaFuncSetAttribute(cond_cta_kernel<T, OP>, cudaFuncAttributeMaxDynamicSharedMemorySize, 220 * 1024));
  const KParams<double> kp = make_kparams<double>(*c.kern);
  cond_cta_kernel<T, OP><<<(unsigned)cnt, kLargeThreads, smem, c.st>>>((const T*)c.g->x, vals, c.g->nbr, in, out, start, c.g->n0, d, k,
                                                                      c.kern->kind, kp, c.ctrl());
  GP_LAUNCH_CHECK();
  return GP_OK;
}

template <typename T>
static gp_status large_t(const OpCtx& c, int op, const T* in, T* out, double* logdet) {
  const int64_t n = c.g->n, n0 = c.g->n0;
  GP_CUDA_OK(cudaMemsetAsync(c.ctrl(), 0, kCtrlBytes, c.st));
  if (c.io && op != GP_OP_LOGDET)      // host-buffer variants: plain copies around the op (no pipelining at this size)
    GP_CUDA_OK(cudaMemcpyAsync((T*)in, c.io->in_host[0], (size_t)n * sizeof(T), cudaMemcpyHostToDevice, c.st));
  SideStream* side = nullptr;
  GP_OK_OR_RETURN(side_stream(&side));
  if (op == GP_OP_FORWARD) {
    GP_OK_OR_RETURN(head_factor(c, nullptr, 0));
    GP_OK_OR_RETURN(head_forward(c, in, out, nullptr, false));
    GP_OK_OR_RETURN(ktime_begin(c.st));
    const int64_t* off = c.g->batch_off;
    for (int b = 0; b < c.g->n_batches; ++b)
      GP_OK_OR_RETURN((launch_large<T, LOP_FORWARD>(c, out, in, out, off[b], off[b + 1])));
    GP_OK_OR_RETURN(ktime_end(c.st));
    if (c.io) GP_CUDA_OK(cudaMemcpyAsync(c.io->out_host, out, (size_t)n * sizeof(T), cudaMemcpyDeviceToHost, c.st));
    return GP_OK;
  }
  GP_OK_OR_RETURN(side_fork(side, c.st));
  OpCtx hc = c;
  hc.st = side->stream;
  if (op == GP_OP_INVERSE) {
    GP_OK_OR_RETURN(head_factor(hc, in, 1, true));
    GP_OK_OR_RETURN(head_inverse_out(hc, out));
    GP_OK_OR_RETURN(ktime_begin(c.st));
    GP_OK_OR_RETURN((launch_large<T, LOP_INVERSE>(c, in, in, out, n0, n)));
    GP_OK_OR_RETURN(ktime_end(c.st));
    GP_OK_OR_RETURN(side_join(side, c.st));
    if (c.io) GP_CUDA_OK(cudaMemcpyAsync(c.io->out_host, out, (size_t)n * sizeof(T), cudaMemcpyDeviceToHost, c.st));
    return GP_OK;
  }
  GP_OK_OR_RETURN(head_factor(hc, nullptr, 0, true));
  GP_OK_OR_RETURN(head_logdet(hc, &c.ctrl()->acc[0], nullptr));
  GP_OK_OR_RETURN(ktime_begin(c.st));
  GP_OK_OR_RETURN((launch_large<T, LOP_LOGDET>(c, nullptr, nullptr, nullptr, n0, n)));
  large_logdet_sum_kernel<<<1, 32, 0, c.st>>>(c.ctrl());
  GP_LAUNCH_CHECK();
  GP_OK_OR_RETURN(ktime_end(c.st));
  GP_OK_OR_RETURN(side_join(side, c.st));
  GP_CUDA_OK(cudaMemcpyAsync(logdet, &c.ctrl()->acc[0], sizeof(double), cudaMemcpyDeviceToDevice, c.st));
  return GP_OK;
}

gp_status run_large(const OpCtx& c, int op, const void* in, void* out, double* logdet) {
  return c.g->dtype == GP_F64 ? large_t<double>(c, op, (const double*)in, (double*)out, logdet)
                              : large_t<float>(c, op, (const float*)in, (float*)out, logdet);
}

}  // namespace gp
