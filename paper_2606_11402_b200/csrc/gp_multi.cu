// Multi-sample apply (MGVI / geoVI "require the forward pass for posterior sampling"):
// S noise vectors on ONE graph and ONE set of kernel parameters.  Everything that does not depend on the values -
// indices, coordinates, K, its factor, the weights w = K_cc^-1 K_ci and s of Eq. 2 - is computed once
// per point; only the k-term apply  v_i = w . v_c + sigma s xi_i  (inverse: xi_i = (v_i - w . v_c) / (sigma s))  repeats
// per sample.  Vectors are POINT-MAJOR, [n][S]: the S values of a neighbour are contiguous, one gather serves them all.
//
//   gp_forward_multi   (1) multi_weights_kernel over all points at once (no dependency on values) -> w, s in the
//                          workspace;  (2) the dense head for S right-hand sides;  (3) multi_apply_kernel batch by
//                          batch (Alg. 1 lines 2-8): a light, gather-bound kernel.
//   gp_inverse_multi   the same weights kernel, then ONE apply launch over all points (every point at once).
#include <type_traits>

#include "gp_cond_pk.cuh"

namespace gp {

constexpr int kMultiThreads = 128;

template <typename T> __device__ __forceinline__ T mnan();
template <> __device__ __forceinline__ float mnan<float>() { return __int_as_float(0x7fc00000); }
template <> __device__ __forceinline__ double mnan<double>() { return __longlong_as_double(0x7ff8000000000000LL); }

template <typename T>
__global__ void multi_pack_kernel(const T* __restrict__ x, Rec<T>* __restrict__ rec, int64_t n, int d) {
  int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  Rec<T> r;
  r.x0 = x[i * d];
  r.x1 = d >= 2 ? x[i * d + 1] : T(0);
  r.x2 = d >= 3 ? x[i * d + 2] : T(0);
  r.v = T(0);
  rec[i] = r;
}

// weights and s of one point (unit sigma), the v-independent half of the conditioning
template <typename T, int K, int D, int KIND>
__device__ __forceinline__ Cond<T> point_weights(const Rec<T>* __restrict__ rec, const int32_t* __restrict__ row, int64_t i,
                                                 const KParams<T>& kp, T (&w)[K]) {
  Rec<T> self = load_rec<false>(rec + i);
  int32_t idx[K];
  Rec<T> R[K];
  gather_reg<T, K, false>(rec, row, idx, R);
  if constexpr (std::is_same<T, float>::value && K % 2 == 0) return weights_pk<K, D, KIND>(R, self, kp, w);
  else return weights_reg<T, K, D, KIND>(R, self, kp, w);
}

// wbuf[(i - n0) * (K + 1)] = {w_0 .. w_{K-1}, sigma s}  (sigma s = NaN marks a point that was not positive definite)
template <typename T, int K, int D, int KIND>
__global__ void __launch_bounds__(kMultiThreads, 2)
multi_weights_kernel(const Rec<T>* __restrict__ rec, const int32_t* __restrict__ nbr, T* __restrict__ wbuf, int64_t n0,
                     int64_t n, KParams<T> kp, Control* ctrl) {
  const int64_t i = n0 + (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  T w[K];
  Cond<T> c = point_weights<T, K, D, KIND>(rec, nbr + (i - n0) * K, i, kp, w);
  if (!c.ok) atomicAdd(&ctrl->n_bad, 1ULL);
  T* dst = wbuf + (i - n0) * (K + 1);
#pragma unroll
  for (int j = 0; j < K; ++j) dst[j] = w[j];
  dst[K] = c.ok ? kp.sigma * c.s : mnan<T>();
}

// One thread per (point, sample).  The K + 1 weights and K indices of a point are read by its S threads (consecutive
// threads: broadcast out of L1); the S values of a neighbour are contiguous.
template <typename T, int K, bool INVERSE>
__global__ void __launch_bounds__(256)
multi_apply_kernel(const int32_t* __restrict__ nbr, const T* __restrict__ wbuf, const T* in, T* out, const T* vals,
                   int S, int64_t start, int64_t end, int64_t n0) {
  const int64_t t = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  const int64_t i = start + t / S;
  const int s = (int)(t % S);
  if (i >= end) return;
  const int32_t* row = nbr + (i - n0) * K;
  const T* w = wbuf + (i - n0) * (K + 1);
  T m = T(0);
#pragma unroll
  for (int j = 0; j < K; ++j) m = Math<T>::fma(__ldg(w + j), vals[(int64_t)__ldg(row + j) * S + s], m);
  const T ss = __ldg(w + K);
  if (INVERSE) out[i * S + s] = (in[i * S + s] - m) / ss;
  else out[i * S + s] = Math<T>::fma(ss, in[i * S + s], m);   // NaN sigma s -> NaN
}

// ---- dense head for S right-hand sides --------------------------------------------------------------------------
// forward: v_head[:, s] = sigma L xi_head[:, s]   (one warp per row, loop over the samples)
template <typename T>
__global__ void multi_head_forward_kernel(const double* __restrict__ L, const T* __restrict__ xi, T* __restrict__ v,
                                          int n0, int S, double sigma) {
  const int r = blockIdx.x * (blockDim.x / 32) + threadIdx.x / 32;
  const int lane = threadIdx.x & 31;
  if (r >= n0) return;
  for (int s = 0; s < S; ++s) {
    double acc = 0.0;
    for (int cc = lane; cc <= r; cc += 32) acc = fma(L[(size_t)r * n0 + cc], (double)xi[(size_t)cc * S + s], acc);
    acc = warp_sum(acc);
    if (lane == 0) v[(size_t)r * S + s] = (T)(sigma * acc);
  }
}
// inverse: carried row s of the head factorisation starts as v_head[:, s]^T and ends as (L^-1 v_head[:, s])^T
template <typename T>
__global__ void multi_head_carry_init_kernel(const T* __restrict__ v, int n0, int S, double* __restrict__ A) {
  const int64_t e = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (e >= (int64_t)n0 * S) return;
  const int s = (int)(e / n0), p = (int)(e % n0);
  A[(size_t)n0 * n0 + e] = (double)v[(size_t)p * S + s];
}
template <typename T>
__global__ void multi_head_inverse_out_kernel(const double* __restrict__ carried, T* __restrict__ xi, int n0, int S,
                                              double inv_sigma) {
  const int64_t e = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (e >= (int64_t)n0 * S) return;
  const int s = (int)(e / n0), p = (int)(e % n0);
  xi[(size_t)p * S + s] = (T)(carried[e] * inv_sigma);
}

// ---- host side ------------------------------------------------------------------------------------------------
// workspace: ctrl | head (n0 + carried) x n0 doubles | records | weights
struct MultiLayout { size_t ctrl_off, head_off, rec_off, w_off, total; };
static MultiLayout multi_layout(const gp_graph* g, int op, int S) {
  MultiLayout m{};
  const size_t B = dtype_bytes(g->dtype), n0 = (size_t)g->n0, n = (size_t)g->n;
  size_t off = 0;
  m.ctrl_off = off; off += kCtrlBytes;
  const size_t carried = op == GP_OP_INVERSE_MULTI ? (size_t)S : 0;
  m.head_off = off; off += align_up((n0 + carried) * n0 * sizeof(double), 256);
  m.rec_off = off; off += align_up(n * 4 * B, 256);
  m.w_off = off;
  off += align_up((n - n0) * ((size_t)g->k + 1) * B, 256);
  m.total = off;
  return m;
}

#define GP_MULTI_TABLE(X) X(float, 8, 3) X(float, 16, 3) X(float, 8, 2) X(float, 16, 2) X(double, 8, 3) X(double, 8, 2)

static bool multi_supported(const gp_graph* g) {
#define X(T, K, D) \
  if ((g->dtype == GP_F64) == (sizeof(T) == 8) && g->k == K && g->d == D) return true;
  GP_MULTI_TABLE(X)
#undef X
  return false;
}

template <typename T, int K, int D>
static gp_status multi_run(const OpCtx& c, const MultiLayout& lay, bool inverse, int S, const T* in, T* out) {
  const int64_t n = c.g->n, n0 = c.g->n0, cnt = n - n0;
  const KParams<T> kp = make_kparams<T>(*c.kern);
  Rec<T>* rec = (Rec<T>*)(c.ws + lay.rec_off);
  T* wbuf = (T*)(c.ws + lay.w_off);
  Control* ctrl = c.ctrl();
  GP_CUDA_OK(cudaMemsetAsync(ctrl, 0, kCtrlBytes, c.st));
  multi_pack_kernel<T><<<(unsigned)((n + 255) / 256), 256, 0, c.st>>>((const T*)c.g->x, rec, n, c.g->d);
  GP_LAUNCH_CHECK();
  const unsigned wgrid = (unsigned)((cnt + kMultiThreads - 1) / kMultiThreads);
  // the dense head (fp64, R-19) on the side stream beside the weights / inverse kernel
  SideStream* side = nullptr;
  GP_OK_OR_RETURN(side_stream(&side));
  GP_OK_OR_RETURN(side_fork(side, c.st));
  OpCtx hc = c;
  hc.st = side->stream;
  if (n0 > 0) {
    if (inverse) {
      const int64_t tot = n0 * S;
      multi_head_carry_init_kernel<T><<<(unsigned)((tot + 255) / 256), 256, 0, hc.st>>>(in, (int)n0, S, c.head());
      GP_LAUNCH_CHECK();
      GP_OK_OR_RETURN(head_factor_preinit(hc, S, cnt > 0));
      multi_head_inverse_out_kernel<T><<<(unsigned)((tot + 255) / 256), 256, 0, hc.st>>>(c.head() + (size_t)n0 * n0, out, (int)n0, S,
                                                                                        1.0 / c.kern->sigma);
      GP_LAUNCH_CHECK();
    } else {
      GP_OK_OR_RETURN(head_factor_preinit(hc, 0, cnt > 0));
      multi_head_forward_kernel<T><<<(unsigned)((n0 + 3) / 4), 128, 0, hc.st>>>(c.head(), in, out, (int)n0, S, c.kern->sigma);
      GP_LAUNCH_CHECK();
    }
  }
  GP_OK_OR_RETURN(ktime_begin(c.st));
  if (cnt > 0) {
#define GP_MK(KIND) multi_weights_kernel<T, K, D, KIND><<<wgrid, kMultiThreads, 0, c.st>>>(rec, c.g->nbr, wbuf, n0, n, kp, ctrl);
    switch (c.kern->kind) {
      case GP_KERNEL_SE: GP_MK(GP_KERNEL_SE) break;
      case GP_KERNEL_MATERN32: GP_MK(GP_KERNEL_MATERN32) break;
      default: GP_MK(GP_KERNEL_EXP) break;
    }
#undef GP_MK
    GP_LAUNCH_CHECK();
  }
  GP_OK_OR_RETURN(side_join(side, c.st));
  if (inverse && cnt > 0) {
    const int64_t work = cnt * S;
    multi_apply_kernel<T, K, true><<<(unsigned)((work + 255) / 256), 256, 0, c.st>>>(c.g->nbr, wbuf, in, out, in, S, n0, n, n0);
    GP_LAUNCH_CHECK();
  }
  if (!inverse && cnt > 0) {
    const int64_t* off = c.g->batch_off;
    for (int b = 0; b < c.g->n_batches; ++b) {          // Alg. 1 lines 2-8: batches in order, points in parallel
      const int64_t work = (off[b + 1] - off[b]) * S;
      multi_apply_kernel<T, K, false><<<(unsigned)((work + 255) / 256), 256, 0, c.st>>>(c.g->nbr, wbuf, in, out, out, S, off[b],
                                                                                        off[b + 1], n0);
      GP_LAUNCH_CHECK();
    }
  }
  return ktime_end(c.st);
}

static gp_status multi_dispatch(const gp_graph* g, const gp_kernel* kern, int op, int S, const void* in, void* out,
                                void* ws, size_t ws_bytes, void* stream) {
  if (!g || !kern || !in || !out) return GP_ERR_INVALID_ARG;
  if (S < 1 || S > 1024) return GP_ERR_INVALID_ARG;
  gp_status vs = validate_graph(g, kern);
  if (vs != GP_OK) return vs;
  if (!multi_supported(g) || (((uintptr_t)g->nbr) & 15) != 0) return GP_ERR_UNSUPPORTED;
  const MultiLayout lay = multi_layout(g, op, S);
  if (!ws || ws_bytes < lay.total || (((uintptr_t)ws) & 255) != 0) return GP_ERR_WORKSPACE;
  int ndev = 0;
  if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev == 0) return GP_ERR_CUDA;
  OpCtx c;
  c.g = g; c.kern = kern; c.ws = (char*)ws; c.st = (cudaStream_t)stream;
  c.lay = WsLayout{};
  c.lay.ctrl_off = lay.ctrl_off;
  c.lay.head_off = lay.head_off;
  c.lay.rec_off = lay.rec_off;
  const bool inverse = op == GP_OP_INVERSE_MULTI;
#define X(T, K, D) \
  if ((g->dtype == GP_F64) == (sizeof(T) == 8) && g->k == K && g->d == D) \
    return multi_run<T, K, D>(c, lay, inverse, S, (const T*)in, (T*)out);
  GP_MULTI_TABLE(X)
#undef X
  return GP_ERR_UNSUPPORTED;
}

}  // namespace gp

using namespace gp;

extern "C" {

size_t gp_workspace_bytes_multi(const gp_graph* g, int32_t op, int32_t n_samples) {
  if (!g || g->n <= 0 || g->n0 < 0 || g->n0 > g->n || n_samples < 1 || (op != GP_OP_FORWARD_MULTI && op != GP_OP_INVERSE_MULTI))
    return 0;
  return multi_layout(g, op, n_samples).total;
}

gp_status gp_forward_multi(const gp_graph* g, const gp_kernel* kern, int32_t n_samples, const void* xi, void* v, void* ws,
                           size_t ws_bytes, void* cuda_stream) {
  return multi_dispatch(g, kern, GP_OP_FORWARD_MULTI, n_samples, xi, v, ws, ws_bytes, cuda_stream);
}

gp_status gp_inverse_multi(const gp_graph* g, const gp_kernel* kern, int32_t n_samples, const void* v, void* xi, void* ws,
                           size_t ws_bytes, void* cuda_stream) {
  return multi_dispatch(g, kern, GP_OP_INVERSE_MULTI, n_samples, v, xi, ws, ws_bytes, cuda_stream);
}

}  // extern "C"
