// Forward-mode derivative of gp_forward and the VJP of gp_inverse ("forward and backward derivatives of
// GraphGP").  Both reuse the geometry pass of the VJP (gp_vjp.cu: run_geometry), which
// leaves per point the weights w = K_cc^-1 K_ci and three scalars
//     s,   A_i = ell dv_i/dell,   B_i = dv_i/dsigma      (derivatives at fixed neighbour values v_c),
// because  v_i = w . v_c + sigma s xi_i  gives
//   JVP of forward      dv_i = w . dv_c + sigma s dxi_i + (dell / ell) A_i + dsigma B_i          (a forward sweep)
//   VJP of inverse      xi_i = (v_i - w . v_c) / (sigma s):   with h_i = xi_bar_i / (sigma s)
//                       v_bar_i += h_i,  v_bar_c -= h_i w,  ell_bar -= h_i A_i / ell,  sigma_bar -= h_i B_i
//                       (no sweep: every point contributes independently)
// Dense head, M = K_head / sigma^2 = L L^T:  dL = (dell / ell) L Phi(Z),  Z = L^-1 D L^-T,  D = ell dM/dell,  Phi = lower
// triangle with the diagonal halved.  The head factorisation carries two blocks of rows (gp_head.cu):
// C1[b][a] = Linv[a][b] and C2[b][a] = (Linv D)[a][b], so  Z_ab = sum_c C2[c][a] C1[c][b]  and
//     p_a := (Phi(Z) xi_h)_a = sum_c C2[c][a] ( sum_{b < a} C1[c][b] xi_b + C1[c][a] xi_a / 2 )            O(n0^2)
//   JVP   dv_h = (dsigma / sigma) v_h + sigma L (dxi_h + (dell / ell) p)
//   VJP   xi_h = L^-1 v_h / sigma:  v_bar_h = L^-T h_h / sigma,  ell_bar -= h_h . p / ell,  sigma_bar -= h_h . xi_h / sigma
#include <type_traits>

#include "gp_cond.cuh"

namespace gp {

// p = Phi(Z) xi_h.  One warp per carried row c: running prefix of C1[c][b] xi_b over b, contributions added to p[a].
template <typename T>
__global__ void head_pxi_kernel(const double* __restrict__ C1, const double* __restrict__ C2, const T* __restrict__ xi,
                                double* __restrict__ p, int n0) {
  const int c = blockIdx.x * (blockDim.x / 32) + threadIdx.x / 32;
  const int lane = threadIdx.x & 31;
  if (c >= n0) return;
  const double* c1 = C1 + (size_t)c * n0;
  const double* c2 = C2 + (size_t)c * n0;
  double carry = 0.0;                                           // sum_{b < chunk} C1[c][b] xi_b
  for (int a0 = (c / 32) * 32; a0 < n0; a0 += 32) {             // Linv[a][c] = 0 for a < c
    const int a = a0 + lane;
    const double t = a < n0 ? c1[a] * (double)xi[a] : 0.0;
    double incl = t;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
      double up = __shfl_up_sync(0xffffffffu, incl, o);
      if (lane >= o) incl += up;
    }
    if (a < n0) atomicAdd(p + a, c2[a] * (carry + incl - 0.5 * t));
    carry += __shfl_sync(0xffffffffu, incl, 31);
  }
}

// dv_h = (dsigma / sigma) v_h + sigma L (dxi_h + (dell / ell) p)     (one warp per row)
template <typename T>
__global__ void head_jvp_kernel(const double* __restrict__ L, const double* __restrict__ p, const T* __restrict__ v,
                                const T* __restrict__ dxi, T* __restrict__ dv, int n0, double sigma, double dsig_over_sig,
                                double dell_over_ell) {
  const int r = blockIdx.x * (blockDim.x / 32) + threadIdx.x / 32;
  const int lane = threadIdx.x & 31;
  if (r >= n0) return;
  double acc = 0.0;
  for (int cc = lane; cc <= r; cc += 32) acc = fma(L[(size_t)r * n0 + cc], (double)dxi[cc] + dell_over_ell * p[cc], acc);
  acc = warp_sum(acc);
  if (lane == 0) dv[r] = (T)(dsig_over_sig * (double)v[r] + sigma * acc);
}

// forward sweep of the JVP over one batch (runtime k)
template <typename T>
__global__ void jvp_apply_kernel(const int32_t* __restrict__ nbr, const T* __restrict__ wbuf, const T* __restrict__ sab,
                                 const T* __restrict__ dxi, T* dv, int k, int64_t start, int64_t end, int64_t n0, T sigma,
                                 T dsig, T dell_over_ell) {
  const int64_t i = start + (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= end) return;
  const int32_t* row = nbr + (i - n0) * k;
  const T* w = wbuf + (i - n0) * k;
  const T* o = sab + (i - n0) * 4;
  T m = T(0);
  for (int j = 0; j < k; ++j) m = Math<T>::fma(w[j], dv[row[j]], m);
  T out = m + sigma * o[0] * dxi[i] + dell_over_ell * o[1] + dsig * o[2];
  if (o[3] == T(0)) out = sizeof(T) == 8 ? (T)__longlong_as_double(0x7ff8000000000000LL) : (T)__int_as_float(0x7fc00000);
  dv[i] = out;
}

// VJP of the inverse, conditioned points: scatter into v_bar, block sums of the two parameter cotangents
template <typename T>
__global__ void __launch_bounds__(256)
inverse_vjp_kernel(const int32_t* __restrict__ nbr, const T* __restrict__ wbuf, const T* __restrict__ sab,
                   const T* __restrict__ xibar, T* vbar, int k, int64_t n0, int64_t n, T sigma, Control* ctrl) {
  __shared__ double red[32];
  const int64_t i = n0 + (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  double acc_sigma = 0.0, acc_ell = 0.0;
  if (i < n) {
    const T* o = sab + (i - n0) * 4;
    if (o[3] != T(0)) {
      const T h = xibar[i] / (sigma * o[0]);
      const int32_t* row = nbr + (i - n0) * k;
      const T* w = wbuf + (i - n0) * k;
      atomicAdd(vbar + i, h);
      for (int j = 0; j < k; ++j) atomicAdd(vbar + row[j], -h * w[j]);
      acc_ell = -(double)(h * o[1]);
      acc_sigma = -(double)(h * o[2]);
    }
  }
  block_atomic_add(acc_sigma, &ctrl->acc[3], red);
  block_atomic_add(acc_ell, &ctrl->acc[4], red);
}

// head of the inverse VJP: v_bar_h[b] += (1 / sigma) sum_a C1[b][a] h_a;  acc_ell -= h_h . p;  acc_sigma -= h_h . xi_h / sigma
template <typename T>
__global__ void head_inverse_vjp_kernel(const double* __restrict__ C1, const double* __restrict__ p, const T* __restrict__ xi,
                                        const T* __restrict__ xibar, T* vbar, int n0, double sigma, double* acc) {
  __shared__ double red[32];
  const int b = blockIdx.x * (blockDim.x / 32) + threadIdx.x / 32;
  const int lane = threadIdx.x & 31;
  double cs = 0.0, cl = 0.0;
  if (b < n0) {
    double s = 0.0;
    for (int a = b + lane; a < n0; a += 32) s = fma(C1[(size_t)b * n0 + a], (double)xibar[a], s);   // Linv[a][b] = 0 for a < b
    s = warp_sum(s);
    if (lane == 0) {
      atomicAdd(vbar + b, (T)(s / sigma));
      cl = -(double)xibar[b] * p[b];
      cs = -(double)xibar[b] * (double)xi[b] / sigma;
    }
  }
  block_atomic_add(cs, acc, red);
  block_atomic_add(cl, acc + 1, red);
}

__global__ void finalize_theta_kernel(const Control* ctrl, double inv_ell, double* out2) {
  if (threadIdx.x == 0 && blockIdx.x == 0) {
    out2[0] = ctrl->acc[3];
    out2[1] = ctrl->acc[4] * inv_ell;
  }
}

template <typename T>
static gp_status head_pxi(const OpCtx& c, const T* xi, double** p_out) {
  const int n0 = (int)c.g->n0;
  const double* C1 = c.head() + (size_t)n0 * n0;
  const double* C2 = C1 + (size_t)n0 * n0;
  double* p = c.head() + (size_t)3 * n0 * n0;
  GP_CUDA_OK(cudaMemsetAsync(p, 0, (size_t)n0 * sizeof(double), c.st));
  head_pxi_kernel<T><<<(unsigned)((n0 + 3) / 4), 128, 0, c.st>>>(C1, C2, xi, p, n0);
  GP_LAUNCH_CHECK();
  *p_out = p;
  return GP_OK;
}

template <typename T>
static gp_status jvp_t(const OpCtx& c, const T* xi, const T* v, const T* dxi, double dsig, double dell, T* dv) {
  const int64_t n = c.g->n, n0 = c.g->n0, cnt = n - n0;
  const int k = c.g->k;
  GP_CUDA_OK(cudaMemsetAsync(c.ctrl(), 0, kCtrlBytes, c.st));
  // the head factorisation (two carried blocks) on the side stream beside the geometry pass
  SideStream* side = nullptr;
  GP_OK_OR_RETURN(side_stream(&side));
  GP_OK_OR_RETURN(side_fork(side, c.st));
  if (n0 > 0) {
    OpCtx hc = c;
    hc.st = side->stream;
    GP_OK_OR_RETURN(head_factor(hc, nullptr, 2 * (int)n0, cnt > 0));
    double* p = nullptr;
    GP_OK_OR_RETURN(head_pxi<T>(hc, xi, &p));
    head_jvp_kernel<T><<<(unsigned)((n0 + 3) / 4), 128, 0, hc.st>>>(c.head(), p, v, dxi, dv, (int)n0, c.kern->sigma,
                                                                   dsig / c.kern->sigma, dell / c.kern->ell);
    GP_LAUNCH_CHECK();
  }
  GP_OK_OR_RETURN(ktime_begin(c.st));
  GP_OK_OR_RETURN(run_geometry(c, xi, v));
  GP_OK_OR_RETURN(side_join(side, c.st));
  if (cnt > 0) {
    const T* wbuf = (const T*)c.wbuf();
    const T* sab = wbuf + (size_t)cnt * k;
    const int64_t* off = c.g->batch_off;
    for (int b = 0; b < c.g->n_batches; ++b) {                 // batches in order, points in parallel
      const int64_t m = off[b + 1] - off[b];
      jvp_apply_kernel<T><<<(unsigned)((m + 255) / 256), 256, 0, c.st>>>(c.g->nbr, wbuf, sab, dxi, dv, k, off[b], off[b + 1], n0,
                                                                        (T)c.kern->sigma, (T)dsig, (T)(dell / c.kern->ell));
      GP_LAUNCH_CHECK();
    }
  }
  return ktime_end(c.st);
}

template <typename T>
static gp_status inverse_vjp_t(const OpCtx& c, const T* v, const T* xi, const T* xibar, T* vbar, double* thetabar) {
  const int64_t n = c.g->n, n0 = c.g->n0, cnt = n - n0;
  const int k = c.g->k;
  GP_CUDA_OK(cudaMemsetAsync(c.ctrl(), 0, kCtrlBytes, c.st));
  GP_CUDA_OK(cudaMemsetAsync(vbar, 0, (size_t)n * sizeof(T), c.st));
  SideStream* side = nullptr;
  GP_OK_OR_RETURN(side_stream(&side));
  GP_OK_OR_RETURN(side_fork(side, c.st));
  double* p = nullptr;
  if (n0 > 0) {
    OpCtx hc = c;
    hc.st = side->stream;
    GP_OK_OR_RETURN(head_factor(hc, nullptr, 2 * (int)n0, cnt > 0));
    GP_OK_OR_RETURN(head_pxi<T>(hc, xi, &p));
  }
  GP_OK_OR_RETURN(ktime_begin(c.st));
  GP_OK_OR_RETURN(run_geometry(c, xi, v));
  if (cnt > 0) {
    const T* wbuf = (const T*)c.wbuf();
    inverse_vjp_kernel<T><<<(unsigned)((cnt + 255) / 256), 256, 0, c.st>>>(c.g->nbr, wbuf, wbuf + (size_t)cnt * k, xibar, vbar, k,
                                                                          n0, n, (T)c.kern->sigma, c.ctrl());
    GP_LAUNCH_CHECK();
  }
  GP_OK_OR_RETURN(ktime_end(c.st));
  GP_OK_OR_RETURN(side_join(side, c.st));
  if (n0 > 0) {
    head_inverse_vjp_kernel<T><<<(unsigned)((n0 + 3) / 4), 128, 0, c.st>>>(c.head() + (size_t)n0 * n0, p, xi, xibar, vbar, (int)n0,
                                                                          c.kern->sigma, &c.ctrl()->acc[3]);
    GP_LAUNCH_CHECK();
  }
  finalize_theta_kernel<<<1, 32, 0, c.st>>>(c.ctrl(), 1.0 / c.kern->ell, thetabar);
  GP_LAUNCH_CHECK();
  return GP_OK;
}

gp_status run_jvp(const OpCtx& c, const void* xi, const void* v, const void* xi_dot, double sigma_dot, double ell_dot,
                  void* v_dot) {
  return c.g->dtype == GP_F64
             ? jvp_t<double>(c, (const double*)xi, (const double*)v, (const double*)xi_dot, sigma_dot, ell_dot, (double*)v_dot)
             : jvp_t<float>(c, (const float*)xi, (const float*)v, (const float*)xi_dot, sigma_dot, ell_dot, (float*)v_dot);
}
gp_status run_inverse_vjp(const OpCtx& c, const void* v, const void* xi, const void* xi_bar, void* v_bar, double* theta_bar) {
  return c.g->dtype == GP_F64
             ? inverse_vjp_t<double>(c, (const double*)v, (const double*)xi, (const double*)xi_bar, (double*)v_bar, theta_bar)
             : inverse_vjp_t<float>(c, (const float*)v, (const float*)xi, (const float*)xi_bar, (float*)v_bar, theta_bar);
}

}  // namespace gp
