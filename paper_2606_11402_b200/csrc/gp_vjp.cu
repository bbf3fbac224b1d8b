// Kernel-parameter derivatives ("backward derivatives"):
//   gp_vjp     VJP of the forward map (xi, sigma, ell) -> v for a cotangent v_bar
//   gp_logdet  gradient d/d(sigma, ell) of sum_i log s_i^2
//
// Per point, in unit-sigma form M = K / sigma^2 with joint factor L (Alg. 1):
//   l = L[k][0:k], s = L[k][k], z = L_cc^-1 v_c,   v_i = l.z + sigma s xi_i
//   w = L_cc^-T l  (= K_cc^-1 K_ci),  alpha = L_cc^-T z  (= M_cc^-1 v_c),  u = (-w, 1)
//   y = (dM/dell) u  where dM_ab/dell = drho/dell(r_ab), zero on the diagonal
// For the total cotangent g on v_i (all later batches already scattered into it):
//   xi_bar_i   = g sigma s
//   g_c       += g w                                     (k floating-point atomics)
//   sigma_bar += g s xi_i                                (v_i depends on sigma only through sigma s xi_i)
//   ell_bar   += g ( y[0:k].alpha + sigma xi_i (y.u) / (2 s) )
// and for the log-determinant  d/dell log s_i^2 = (y.u) / s^2,  d/dsigma sum_i log(sigma^2 s_i^2) = 2 N / sigma.
// These are the differentials dm = u^T dM [alpha; 0], d(s^2) = u^T dM u of Eq. 2 (R-14); the oracle
// reaches the same numbers by summing K_bar_ab dK_ab/dtheta over the full joint matrix in the solve form.
//
// Batches run in REVERSE order: a point's cotangent is complete once every later batch has scattered into it, and
// points of one batch never touch each other's cotangent.  fp32 shapes with a packed kernel: two
// launches (vjp_geom_kernel, then the ticketed reverse dataflow of vjp_scatter_kernel); every other shape, and
// GP_FLAG_PER_BATCH_LAUNCH: one grad_kernel launch per batch.
#include <type_traits>

#include <vector>

#include "gp_grad_pk.cuh"

namespace gp {

enum { GRAD_VJP = 0, GRAD_LOGDET = 1 };
constexpr int kGradThreads = 128;
#ifndef GP_GRAD_MIN_CTAS
#define GP_GRAD_MIN_CTAS 2
#endif

template <typename T> __device__ __forceinline__ T qnan();
template <> __device__ __forceinline__ float qnan<float>() { return __int_as_float(0x7fc00000); }
template <> __device__ __forceinline__ double qnan<double>() { return __longlong_as_double(0x7ff8000000000000LL); }

// rec[i] = {x_i, vals_i or 0}  (same packed record the forward kernels gather)
template <typename T>
__global__ void grad_pack_kernel(const T* __restrict__ x, const T* __restrict__ vals, Rec<T>* __restrict__ rec,
                                 int64_t n, int d) {
  int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  Rec<T> r;
  r.x0 = x[i * d];
  r.x1 = d >= 2 ? x[i * d + 1] : T(0);
  r.x2 = d >= 3 ? x[i * d + 2] : T(0);
  r.v = vals ? vals[i] : T(0);
  rec[i] = r;
}

// ---- register-resident gradient kernel -----------------------------------------------------------------
template <typename T, int K, int D, int KIND, int MODE>
__global__ void __launch_bounds__(kGradThreads)
grad_kernel(const Rec<T>* __restrict__ rec, const int32_t* __restrict__ nbr, const T* __restrict__ xi,
            T* gbar, T* __restrict__ xibar, int64_t start, int64_t end, int64_t n0, KParams<T> kp, Control* ctrl) {
  __shared__ double red[32];
  int64_t i = start + (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  double acc_sigma = 0.0, acc_ell = 0.0;
  if (i < end) {
    Rec<T> self = load_rec<false>(rec + i);
    int32_t idx[K];
    Rec<T> R[K];
    gather_reg<T, K, false>(rec, nbr + (i - n0) * K, idx, R);
    constexpr int NT = (K + 1) * (K + 2) / 2;
    T A[NT];
    build_joint_reg<T, K, D, KIND>(R, self, kp, A);
    T cv[K];
#pragma unroll
    for (int j = 0; j < K; ++j) cv[j] = R[j].v;
    Cond<T> c = factor_joint_reg<T, K, true>(A, cv, kp);
    // back-substitution, in place:  A[K][j] <- w_j,  cv[j] <- alpha_j
#pragma unroll
    for (int j = K - 1; j >= 0; --j) {
      T w = A[tri(K, j)], a = cv[j];
#pragma unroll
      for (int r = j + 1; r < K; ++r) {
        w = Math<T>::fma(-A[tri(r, j)], A[tri(K, r)], w);
        a = Math<T>::fma(-A[tri(r, j)], cv[r], a);
      }
      A[tri(K, j)] = w * A[tri(j, j)];
      cv[j] = a * A[tri(j, j)];
    }
    // y = (ell dM/dell) u, u = (-w, 1); the triangle of L_cc is dead from here on
    T y[K + 1];
#pragma unroll
    for (int j = 0; j <= K; ++j) y[j] = T(0);
#pragma unroll
    for (int r = 1; r <= K; ++r) {
      T ur = (r == K) ? T(1) : -A[tri(K, r)];
#pragma unroll
      for (int cc = 0; cc < r; ++cc) {
        T q = (r == K) ? pair_q<T, D>(self, R[cc], kp.qscale) : pair_q<T, D>(R[r], R[cc], kp.qscale);
        T dq = Math<T>::template drho_from_q<KIND>(q);
        y[r] = Math<T>::fma(-dq, A[tri(K, cc)], y[r]);   // dq * u_cc
        y[cc] = Math<T>::fma(dq, ur, y[cc]);
      }
    }
    T yu = y[K], ya = T(0);
#pragma unroll
    for (int j = 0; j < K; ++j) {
      yu = Math<T>::fma(-y[j], A[tri(K, j)], yu);
      ya = Math<T>::fma(y[j], cv[j], ya);
    }
    if (!c.ok) atomicAdd(&ctrl->n_bad, 1ULL);
    if (MODE == GRAD_VJP) {
      T g = gbar[i];
      T xi_i = xi[i];
      T gs = g * c.s;
      T out = kp.sigma * gs;
      if (!c.ok) out = qnan<T>();
      xibar[i] = out;
      if (c.ok) {
#pragma unroll
        for (int j = 0; j < K; ++j) atomicAdd(gbar + idx[j], g * A[tri(K, j)]);
        acc_sigma = (double)(gs * xi_i);
        acc_ell = (double)(g * (ya + T(0.5) * kp.sigma * xi_i * yu / c.s));
      }
    } else {
      if (c.ok) acc_ell = (double)(yu / (c.s * c.s));
    }
  }
  if (MODE == GRAD_VJP) block_atomic_add(acc_sigma, &ctrl->acc[3], red);
  block_atomic_add(acc_ell, &ctrl->acc[MODE == GRAD_VJP ? 4 : 2], red);
}

// ---- packed fp32 gradient kernels ----------------------------------------------------------------------------
// Everything that does not depend on the incoming cotangent (weights w, s, and the two scalars
//   A_i = y[0:k].alpha + sigma xi_i (y.u) / (2 s),   B_i = s xi_i      (ell_bar += g A_i, sigma_bar += g B_i))
// is computed first; only then does the point need its total cotangent g.
template <int K, int D, int KIND>
__device__ __forceinline__ bool grad_geometry_pk(const Rec<float>* __restrict__ rec, const int32_t* __restrict__ row,
                                                 const Rec<float>& self, const KParams<float>& kp, const DqStore<K>& dq,
                                                 f2 (&W)[K / 2], f2 (&AL)[K / 2], float& s) {
  f2 P[pk_pairs(K)];
  {
    int32_t idx[K];
    Rec<float> R[K];
    gather_reg<float, K, false>(rec, row, idx, R);
    PkCoords<K> X;
    centre_pk<K, D>(R, self, kp.sq, X);
    float vals[K];
#pragma unroll
    for (int j = 0; j < K; ++j) vals[j] = R[j].v;
    build_joint_grad_pk<K, D, KIND>(X, vals, kp, P, dq);
  }
  eliminate0_pk<K>(P, kp);
  bool ok = factor_joint_pk<K, true>(P, kp.diag);
  s = Math<float>::sqrt(P[pk(K / 2, K)].x * kp.inv_diag);
  backsub2_pk<K>(P, kp, W, AL);
  return ok;
}

template <int K>
__device__ __forceinline__ DqStore<K> dq_store_of(void* smem) {
  DqStore<K> dq;
  dq.p2 = reinterpret_cast<float2*>(smem) + threadIdx.x;
  dq.p1 = reinterpret_cast<float*>(reinterpret_cast<float2*>(smem) + (size_t)dq_full_total(K) * blockDim.x) + threadIdx.x;
  dq.stride = blockDim.x;
  return dq;
}

// gradient of the log-determinant, conditioning part: every point at once
template <int K, int D, int KIND>
__global__ void __launch_bounds__(kGradThreads, GP_GRAD_MIN_CTAS)
logdet_grad_pk_kernel(const Rec<float>* __restrict__ rec, const int32_t* __restrict__ nbr, int64_t start, int64_t end,
                      int64_t n0, KParams<float> kp, Control* ctrl) {
  extern __shared__ float4 dq_raw[];
  __shared__ double red[32];
  int64_t i = start + (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  double acc_ell = 0.0;
  if (i < end) {
    DqStore<K> dq = dq_store_of<K>(dq_raw);
    Rec<float> self = load_rec<false>(rec + i);
    f2 W[K / 2], AL[K / 2];
    float s;
    bool ok = grad_geometry_pk<K, D, KIND>(rec, nbr + (i - n0) * K, self, kp, dq, W, AL, s);
#pragma unroll
    for (int rp = 0; rp < K / 2; ++rp) AL[rp] = make_float2(0.0f, 0.0f);
    float half_yu = grad_sweep_pk<K>(W, AL, 1.0f, dq);
    if (!ok) atomicAdd(&ctrl->n_bad, 1ULL);
    else acc_ell = (double)(2.0f * half_yu / (s * s));
  }
  block_atomic_add(acc_ell, &ctrl->acc[2], red);
}

// VJP of the forward pass in two launches.
//  (1) vjp_geom_kernel: everything that does not depend on the incoming cotangent, for all points at once (no
//      ordering constraint, register-heavy): writes the k weights and {s, A_i, B_i, ok} of every point.
//  (2) vjp_scatter_kernel: the reverse sweep proper, a light kernel at full occupancy.  CTAs take batch-aligned
//      chunks through a ticket, last batch first.  A chunk of batch b may read its cotangents once every point
//      of every later batch has scattered: ctrl->done counts finished points (done >= n - batch_off[b + 1]).
//      Lower tickets have always started and never wait on higher ones, so polling cannot deadlock.
template <int K, int D, int KIND>
__global__ void __launch_bounds__(kGradThreads, GP_GRAD_MIN_CTAS)
vjp_geom_kernel(const Rec<float>* __restrict__ rec, const int32_t* __restrict__ nbr, const float* __restrict__ xi,
                float* __restrict__ wbuf, float4* __restrict__ sab, int64_t n0, int64_t first, int64_t n, KParams<float> kp,
                Control* ctrl) {
  extern __shared__ float4 dq_raw[];
  const int64_t i = first + (int64_t)blockIdx.x * blockDim.x + threadIdx.x;   // points [first, n) of this launch
  if (i >= n) return;
  DqStore<K> dq = dq_store_of<K>(dq_raw);
  Rec<float> self = load_rec<false>(rec + i);
  f2 W[K / 2], AL[K / 2];
  float s;
  bool ok = grad_geometry_pk<K, D, KIND>(rec, nbr + (i - n0) * K, self, kp, dq, W, AL, s);
  const float xi_i = xi[i];
  const float Ai = grad_sweep_pk<K>(W, AL, kp.sigma * xi_i / s, dq);
  if (!ok) atomicAdd(&ctrl->n_bad, 1ULL);
  float4* wrow = reinterpret_cast<float4*>(wbuf + (i - n0) * K);
#pragma unroll
  for (int q = 0; q < K / 4; ++q) wrow[q] = make_float4(W[2 * q].x, W[2 * q].y, W[2 * q + 1].x, W[2 * q + 1].y);
  sab[i - n0] = make_float4(s, Ai, s * xi_i, ok ? 1.0f : 0.0f);
}

constexpr int kScatterThreads = 256;

template <int K>
__global__ void __launch_bounds__(kScatterThreads, 4)
vjp_scatter_kernel(const int32_t* __restrict__ nbr, const float* __restrict__ wbuf, const float4* __restrict__ sab,
                   float* gbar, float* __restrict__ xibar, const longlong4* __restrict__ tab, int L,
                   unsigned long long* ticket, int64_t n0, int64_t n, float sigma, Control* ctrl) {
  __shared__ double red[32];
  __shared__ long long s_info[3];
  __shared__ long long s_ticket;
  if (threadIdx.x == 0) s_ticket = (long long)atomicAdd(ticket, 1ULL);
  __syncthreads();
  {
    const long long t = s_ticket;
    for (int q = threadIdx.x; q < L; q += blockDim.x) {
      const longlong2 e01 = __ldg(reinterpret_cast<const longlong2*>(tab + q));
      const longlong2 e23 = __ldg(reinterpret_cast<const longlong2*>(tab + q) + 1);
      if (e01.x <= t && t < e23.y) {   // {first chunk, first point, end point, end chunk} of reverse batch q
        s_info[0] = e01.y + (t - e01.x) * (long long)blockDim.x;
        s_info[1] = e23.x;
        s_info[2] = n - e23.x;
      }
    }
  }
  __syncthreads();
  const int64_t i = s_info[0] + threadIdx.x;
  const int64_t end = s_info[1];
  const bool active = i < end;
  // everything that does not depend on the cotangent is fetched before waiting
  int32_t idx[K];
  float w[K];
  float4 q4 = make_float4(0.f, 0.f, 0.f, 0.f);
  if (active) {
    load_row<K>(nbr + (i - n0) * K, idx);
    const float4* wrow = reinterpret_cast<const float4*>(wbuf + (i - n0) * K);
#pragma unroll
    for (int q = 0; q < K / 4; ++q) {
      float4 t = __ldcs(wrow + q);
      w[4 * q] = t.x; w[4 * q + 1] = t.y; w[4 * q + 2] = t.z; w[4 * q + 3] = t.w;
    }
    q4 = __ldcs(sab + (i - n0));
  }
  if (threadIdx.x == 0) {
    const unsigned long long need = (unsigned long long)s_info[2];
    const long long t0 = clock64();
    unsigned spins = 0;
    while (true) {
      unsigned long long d;
      asm volatile("ld.relaxed.gpu.global.u64 %0, [%1];" : "=l"(d) : "l"(&ctrl->done) : "memory");
      if (d >= need) break;
      if (++spins > 16) __nanosleep(32);
      if ((spins & 1023u) == 0 && clock64() - t0 > 8000000000LL) { atomicAdd(&ctrl->timeout, 1ULL); break; }
    }
    __threadfence();   // acquire side of the done counter: the scatters counted in `d` are visible before gbar is read
  }
  __syncthreads();
  double acc_sigma = 0.0, acc_ell = 0.0;
  if (active) {
    const float g = __ldcg(gbar + i);           // L2: the cotangent was accumulated there by atomics
    const bool ok = q4.w != 0.0f;
    xibar[i] = ok ? sigma * g * q4.x : qnan<float>();
    if (ok) {
#pragma unroll
      for (int j = 0; j < K; ++j) atomicAdd(gbar + idx[j], g * w[j]);
      acc_sigma = (double)(g * q4.z);
      acc_ell = (double)(g * q4.y);
    }
  }
  // publish first (the next batch is waiting on it), reduce afterwards: the barrier orders every thread's scatter
  // before thread 0's fence.  (Summing the CTA's contributions per target in a shared-memory hash table first was
  // tried: 4.5 ms against 2.95 ms - the table costs more than the L2 atomics it saves.)
  __syncthreads();
  if (threadIdx.x == 0) {
    long long cnt = end - s_info[0];
    if (cnt > (long long)blockDim.x) cnt = blockDim.x;
    __threadfence();
    atomicAdd(&ctrl->done, (unsigned long long)cnt);
  }
  const int slot = (int)(blockIdx.x % kAccSlots);
  block_atomic_add(acc_sigma, &ctrl->slots[0][slot], red);
  block_atomic_add(acc_ell, &ctrl->slots[1][slot], red);
}

// ---- generic gradient kernel: triangle in shared memory, any k <= 64, d <= 4 -----------------------------
template <typename T, int MODE>
__global__ void grad_generic_kernel(const T* __restrict__ x, const T* __restrict__ vals, const int32_t* __restrict__ nbr,
                                    const T* __restrict__ xi, T* gbar, T* __restrict__ xibar, int64_t start, int64_t end,
                                    int64_t n0, int d, int k, int kind, KParams<T> kp, Control* ctrl, int active) {
  extern __shared__ double smem_raw[];
  __shared__ double red[32];
  int tid = threadIdx.x;
  int64_t i = start + (int64_t)blockIdx.x * active + tid;
  double acc_sigma = 0.0, acc_ell = 0.0;
  if (tid < active && i < end) {
    Scratch<T> A{reinterpret_cast<T*>(smem_raw) + tid, active};
    const int32_t* row = nbr + (i - n0) * k;
    const int NT = (k + 1) * (k + 2) / 2;
    Cond<T> c = condition_generic<T>(x, MODE == GRAD_VJP ? vals : nullptr, d, k, kind, row, i, kp, A);
    // back-substitution: A[k][j] <- w_j, A[NT + j] <- alpha_j   (A[j][j] = L_jj)
    for (int j = k - 1; j >= 0; --j) {
      T w = A[tri(k, j)], a = A[NT + j];
      for (int r = j + 1; r < k; ++r) {
        T lrj = A[tri(r, j)];
        w = Math<T>::fma(-lrj, A[tri(k, r)], w);
        a = Math<T>::fma(-lrj, A[NT + r], a);
      }
      T inv = T(1) / A[tri(j, j)];
      A[tri(k, j)] = w * inv;
      A[NT + j] = a * inv;
    }
    const int YO = NT + k;
    for (int j = 0; j <= k; ++j) A[YO + j] = T(0);
    for (int r = 1; r <= k; ++r) {
      int64_t pr = (r == k) ? i : (int64_t)row[r];
      T ur = (r == k) ? T(1) : -A[tri(k, r)];
      T yr = T(0);
      for (int cc = 0; cc < r; ++cc) {
        T dq = drho_rt<T>(kind, dist_q<T>(x, d, pr, (int64_t)row[cc], kp.qscale));
        yr = Math<T>::fma(-dq, A[tri(k, cc)], yr);
        A[YO + cc] = Math<T>::fma(dq, ur, A[YO + cc]);
      }
      A[YO + r] += yr;
    }
    T yu = A[YO + k], ya = T(0);
    for (int j = 0; j < k; ++j) {
      yu = Math<T>::fma(-A[YO + j], A[tri(k, j)], yu);
      ya = Math<T>::fma(A[YO + j], A[NT + j], ya);
    }
    if (!c.ok) atomicAdd(&ctrl->n_bad, 1ULL);
    if (MODE == GRAD_VJP) {
      T g = gbar[i];
      T xi_i = xi[i];
      T gs = g * c.s;
      T out = kp.sigma * gs;
      if (!c.ok) out = qnan<T>();
      xibar[i] = out;
      if (c.ok) {
        for (int j = 0; j < k; ++j) atomicAdd(gbar + row[j], g * A[tri(k, j)]);
        acc_sigma = (double)(gs * xi_i);
        acc_ell = (double)(g * (ya + T(0.5) * kp.sigma * xi_i * yu / c.s));
      }
    } else {
      if (c.ok) acc_ell = (double)(yu / (c.s * c.s));
    }
  }
  if (MODE == GRAD_VJP) block_atomic_add(acc_sigma, &ctrl->acc[3], red);
  block_atomic_add(acc_ell, &ctrl->acc[MODE == GRAD_VJP ? 4 : 2], red);
}

// ---- generic geometry kernel: what vjp_geom_kernel writes, for any (k, d, kind, dtype) ---------------------------------
// w = K_cc^-1 K_ci, s, A_i = y[0:k].alpha + sigma xi_i (y.u) / (2 s) (= ell dv_i/dell at fixed v_c), B_i = s xi_i
template <typename T>
__global__ void geom_generic_kernel(const T* __restrict__ x, const T* __restrict__ vals, const int32_t* __restrict__ nbr,
                                    const T* __restrict__ xi, T* __restrict__ wbuf, T* __restrict__ sab, int64_t n0,
                                    int64_t n, int d, int k, int kind, KParams<T> kp, Control* ctrl, int active) {
  extern __shared__ double smem_raw[];
  const int tid = threadIdx.x;
  const int64_t i = n0 + (int64_t)blockIdx.x * active + tid;
  if (tid >= active || i >= n) return;
  Scratch<T> A{reinterpret_cast<T*>(smem_raw) + tid, active};
  const int32_t* row = nbr + (i - n0) * k;
  const int NT = (k + 1) * (k + 2) / 2;
  Cond<T> c = condition_generic<T>(x, vals, d, k, kind, row, i, kp, A);
  for (int j = k - 1; j >= 0; --j) {        // back-substitution: A[k][j] <- w_j, A[NT + j] <- alpha_j
    T w = A[tri(k, j)], a = A[NT + j];
    for (int r = j + 1; r < k; ++r) {
      T lrj = A[tri(r, j)];
      w = Math<T>::fma(-lrj, A[tri(k, r)], w);
      a = Math<T>::fma(-lrj, A[NT + r], a);
    }
    T inv = T(1) / A[tri(j, j)];
    A[tri(k, j)] = w * inv;
    A[NT + j] = a * inv;
  }
  const int YO = NT + k;
  for (int j = 0; j <= k; ++j) A[YO + j] = T(0);
  for (int r = 1; r <= k; ++r) {            // y = (ell dM/dell) u, u = (-w, 1)
    int64_t pr = (r == k) ? i : (int64_t)row[r];
    T ur = (r == k) ? T(1) : -A[tri(k, r)];
    T yr = T(0);
    for (int cc = 0; cc < r; ++cc) {
      T dq = drho_rt<T>(kind, dist_q<T>(x, d, pr, (int64_t)row[cc], kp.qscale));
      yr = Math<T>::fma(-dq, A[tri(k, cc)], yr);
      A[YO + cc] = Math<T>::fma(dq, ur, A[YO + cc]);
    }
    A[YO + r] += yr;
  }
  T yu = A[YO + k], ya = T(0);
  for (int j = 0; j < k; ++j) {
    yu = Math<T>::fma(-A[YO + j], A[tri(k, j)], yu);
    ya = Math<T>::fma(A[YO + j], A[NT + j], ya);
  }
  if (!c.ok) atomicAdd(&ctrl->n_bad, 1ULL);
  T* wrow = wbuf + (i - n0) * k;
  for (int j = 0; j < k; ++j) wrow[j] = A[tri(k, j)];
  const T xi_i = xi[i];
  T* o = sab + (i - n0) * 4;
  o[0] = c.s;
  o[1] = ya + T(0.5) * kp.sigma * xi_i * yu / c.s;
  o[2] = c.s * xi_i;
  o[3] = c.ok ? T(1) : T(0);
}

// ---- host side --------------------------------------------------------------------------------------------
int generic_active_threads(int k, size_t elem_bytes, bool with_vjp);   // gp_ops.cu

// fp64 gradients go through the shared-memory kernel: with 2 x 36 inlined double exp/sqrt the register-resident
// form makes ptxas fall back to a spill-everything allocation (32 registers, 7 KB of local memory per thread).
#define GP_GRAD_SPEC_TABLE(X) X(float, 8, 3) X(float, 16, 3) X(float, 8, 2) X(float, 16, 2)

template <typename T, int K, int D, int MODE>
static gp_status launch_grad_spec(const OpCtx& c, const T* xi, T* gbar, T* xibar, int64_t start, int64_t end) {
  int64_t cnt = end - start;
  if (cnt <= 0) return GP_OK;
  unsigned grid = (unsigned)((cnt + kGradThreads - 1) / kGradThreads);
  KParams<T> kp = make_kparams<T>(*c.kern);
  const Rec<T>* rec = (const Rec<T>*)c.rec();
  switch (c.kern->kind) {
    case GP_KERNEL_SE:
      grad_kernel<T, K, D, GP_KERNEL_SE, MODE><<<grid, kGradThreads, 0, c.st>>>(rec, c.g->nbr, xi, gbar, xibar, start, end, c.g->n0, kp, c.ctrl());
      break;
    case GP_KERNEL_MATERN32:
      grad_kernel<T, K, D, GP_KERNEL_MATERN32, MODE><<<grid, kGradThreads, 0, c.st>>>(rec, c.g->nbr, xi, gbar, xibar, start, end, c.g->n0, kp, c.ctrl());
      break;
    default:
      grad_kernel<T, K, D, GP_KERNEL_EXP, MODE><<<grid, kGradThreads, 0, c.st>>>(rec, c.g->nbr, xi, gbar, xibar, start, end, c.g->n0, kp, c.ctrl());
      break;
  }
  GP_LAUNCH_CHECK();
  return GP_OK;
}

template <typename T, int MODE>
static gp_status launch_grad_generic(const OpCtx& c, const T* vals, const T* xi, T* gbar, T* xibar, int64_t start,
                                     int64_t end) {
  int64_t cnt = end - start;
  if (cnt <= 0) return GP_OK;
  int k = c.g->k;
  int active = generic_active_threads(k, sizeof(T), true);
  int threads = (active + 31) / 32 * 32;
  size_t smem = (size_t)generic_scratch_elems(k, true) * sizeof(T) * active;
  GP_CUDA_OK(cudaFuncSetAttribute(grad_generic_kernel<T, MODE>, cudaFuncAttributeMaxDynamicSharedMemorySize, 220 * 1024));
  unsigned grid = (unsigned)((cnt + active - 1) / active);
  KParams<T> kp = make_kparams<T>(*c.kern);
  grad_generic_kernel<T, MODE><<<grid, threads, smem, c.st>>>((const T*)c.g->x, vals, c.g->nbr, xi, gbar, xibar, start, end,
                                                            c.g->n0, c.g->d, k, c.kern->kind, kp, c.ctrl(), active);
  GP_LAUNCH_CHECK();
  return GP_OK;
}

static bool grad_use_spec(const OpCtx& c) {
  if (c.g->flags & GP_FLAG_GENERIC_KERNEL) return false;
  bool have = false;
#define X(T, K, D) \
  if ((c.g->dtype == GP_F64) == (sizeof(T) == 8) && c.g->k == K && c.g->d == D) have = true;
  GP_GRAD_SPEC_TABLE(X)
#undef X
  return have && (((uintptr_t)c.g->nbr) & 15) == 0;
}

template <typename T, int MODE>
static gp_status launch_grad_range(const OpCtx& c, bool spec, const T* vals, const T* xi, T* gbar, T* xibar,
                                   int64_t start, int64_t end) {
  if (spec) {
#define X(TT, K, D) \
    if constexpr (std::is_same<TT, T>::value) {                    \
      if (c.g->k == K && c.g->d == D) return launch_grad_spec<T, K, D, MODE>(c, xi, gbar, xibar, start, end); \
    }
    GP_GRAD_SPEC_TABLE(X)
#undef X
  }
  return launch_grad_generic<T, MODE>(c, vals, xi, gbar, xibar, start, end);
}

template <typename T>
static gp_status grad_pack(const OpCtx& c, const T* vals) {
  int64_t n = c.g->n;
  grad_pack_kernel<T><<<(unsigned)((n + 255) / 256), 256, 0, c.st>>>((const T*)c.g->x, vals, (Rec<T>*)c.rec(), n, c.g->d);
  GP_LAUNCH_CHECK();
  return GP_OK;
}

// theta_bar[0] = sigma_bar, theta_bar[1] = ell_bar; the kernels accumulate ell * d/dell
__global__ void finalize_grad_kernel(const Control* ctrl, int slot_sigma, int slot_ell, double inv_ell, double* out2) {
  if (threadIdx.x == 0 && blockIdx.x == 0) {
    double a = ctrl->acc[slot_sigma], b = ctrl->acc[slot_ell];
    for (int q = 0; q < kAccSlots; ++q) { a += ctrl->slots[0][q]; b += ctrl->slots[1][q]; }
    out2[0] = a;
    out2[1] = b * inv_ell;
  }
}

// ---- packed fp32 host side ------------------------------------------------------------------------------------
template <typename KernelT> static gp_status set_dq_smem(KernelT kern, size_t bytes) {
  GP_CUDA_OK(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bytes));
  return GP_OK;
}

template <int K, int D>
static gp_status launch_logdet_grad_pk(const OpCtx& c) {
  int64_t cnt = c.g->n - c.g->n0;
  if (cnt <= 0) return GP_OK;
  unsigned grid = (unsigned)((cnt + kGradThreads - 1) / kGradThreads);
  KParams<float> kp = make_kparams<float>(*c.kern);
  const Rec<float>* rec = (const Rec<float>*)c.rec();
  size_t smem = dq_smem_bytes(K, kGradThreads);
#define GP_LD(KIND)                                                                                              \
  GP_OK_OR_RETURN(set_dq_smem(logdet_grad_pk_kernel<K, D, KIND>, smem));                                        \
  logdet_grad_pk_kernel<K, D, KIND><<<grid, kGradThreads, smem, c.st>>>(rec, c.g->nbr, c.g->n0, c.g->n, c.g->n0, kp, c.ctrl());
  switch (c.kern->kind) {
    case GP_KERNEL_SE: GP_LD(GP_KERNEL_SE) break;
    case GP_KERNEL_MATERN32: GP_LD(GP_KERNEL_MATERN32) break;
    default: GP_LD(GP_KERNEL_EXP) break;
  }
#undef GP_LD
  GP_LAUNCH_CHECK();
  return GP_OK;
}

// geometry of the points [first, end): everything of the VJP that does not depend on the incoming cotangent
template <int K, int D>
static gp_status launch_vjp_geom(const OpCtx& c, const float* xi, int64_t first, int64_t end) {
  const int64_t cnt = end - first, total = c.g->n - c.g->n0;
  if (cnt <= 0) return GP_OK;
  KParams<float> kp = make_kparams<float>(*c.kern);
  const Rec<float>* rec = (const Rec<float>*)c.rec();
  float* wbuf = c.wbuf();
  float4* sab = reinterpret_cast<float4*>(wbuf + (size_t)total * K);
  size_t smem = dq_smem_bytes(K, kGradThreads);
  unsigned ggrid = (unsigned)((cnt + kGradThreads - 1) / kGradThreads);
#define GP_VF(KIND)                                                                                              \
  GP_OK_OR_RETURN(set_dq_smem(vjp_geom_kernel<K, D, KIND>, smem));                                              \
  vjp_geom_kernel<K, D, KIND><<<ggrid, kGradThreads, smem, c.st>>>(rec, c.g->nbr, xi, wbuf, sab, c.g->n0, first, end, kp, c.ctrl());
  switch (c.kern->kind) {
    case GP_KERNEL_SE: GP_VF(GP_KERNEL_SE) break;
    case GP_KERNEL_MATERN32: GP_VF(GP_KERNEL_MATERN32) break;
    default: GP_VF(GP_KERNEL_EXP) break;
  }
#undef GP_VF
  GP_LAUNCH_CHECK();
  return GP_OK;
}

// the reverse sweep proper over all batches (ticketed dataflow, last batch first)
template <int K>
static gp_status launch_vjp_scatter(const OpCtx& c, float* gbar, float* xibar, EventBag* bag = nullptr) {
  const int L = c.g->n_batches;
  const int64_t cnt = c.g->n - c.g->n0;
  if (L <= 0 || cnt <= 0) return GP_OK;
  // Host-buffer variant (bag != nullptr): the reverse sweep is cut into up to kScatterParts launches at batch
  // boundaries, each with its own ticket counter (`done` keeps counting across them), and the xi_bar of a part goes
  // home on the copy-out stream while the next part runs.  Otherwise one launch.
  constexpr int kScatterParts = 4;
  const int parts = bag ? kScatterParts : 1;
  // device table, one entry per batch in REVERSE order: {first chunk, first point, end point, end chunk}; chunk
  // numbers restart with every part
  std::vector<int64_t> tab(4 * (size_t)L);
  const int64_t* off = c.g->batch_off;
  struct Part { int r0, r1; int64_t chunks; };
  std::vector<Part> plan;
  int64_t chunks = 0, pts = 0;
  int r0 = 0;
  for (int rb = 0; rb < L; ++rb) {
    int b = L - 1 - rb;
    int64_t nc = (off[b + 1] - off[b] + kScatterThreads - 1) / kScatterThreads;
    tab[4 * rb + 0] = chunks;
    tab[4 * rb + 1] = off[b];
    tab[4 * rb + 2] = off[b + 1];
    tab[4 * rb + 3] = chunks + nc;
    chunks += nc;
    pts += off[b + 1] - off[b];
    const bool last = rb == L - 1;
    if (last || ((int)plan.size() < parts - 1 && pts >= cnt * ((int64_t)plan.size() + 1) / parts)) {
      if (chunks > 0x7fffffffLL) return GP_ERR_UNSUPPORTED;
      plan.push_back({r0, rb + 1, chunks});
      r0 = rb + 1;
      chunks = 0;
    }
  }
  // pageable source: the runtime stages it before returning, so the vector may die afterwards
  GP_CUDA_OK(cudaMemcpyAsync(c.boff_dev(), tab.data(), tab.size() * sizeof(int64_t), cudaMemcpyHostToDevice, c.st));
  float* wbuf = c.wbuf();
  float4* sab = reinterpret_cast<float4*>(wbuf + (size_t)cnt * K);
  int slot = 0;
  for (const Part& p : plan) {
    if (p.chunks <= 0) continue;
    const longlong4* tab_d = (const longlong4*)c.boff_dev() + p.r0;
    unsigned long long* ticket = plan.size() == 1 ? &c.ctrl()->ticket : &c.ctrl()->flow_ticket[slot++];
    vjp_scatter_kernel<K><<<(unsigned)p.chunks, kScatterThreads, 0, c.st>>>(c.g->nbr, wbuf, sab, gbar, xibar, tab_d, p.r1 - p.r0,
                                                                          ticket, c.g->n0, c.g->n, (float)c.kern->sigma, c.ctrl());
    GP_LAUNCH_CHECK();
    if (bag) {                                 // points of reverse batches [r0, r1) = graph positions [lo, hi)
      const int64_t lo = off[L - p.r1], hi = off[L - p.r0];
      GP_OK_OR_RETURN(stream_after(*bag, c.io->cout, c.st));
      GP_CUDA_OK(cudaMemcpyAsync((float*)c.io->out_host + lo, xibar + lo, (size_t)(hi - lo) * sizeof(float),
                                 cudaMemcpyDeviceToHost, c.io->cout));
    }
  }
  return GP_OK;
}

// (K, D) pairs with packed fp32 gradient kernels (K even)
#define GP_GRAD_PK_TABLE(X) X(8, 3) X(16, 3) X(8, 2) X(16, 2)

template <typename T>
static gp_status vjp_t(const OpCtx& c, const T* xi, const T* v, const T* vbar, T* xibar, double* thetabar) {
  bool spec = grad_use_spec(c);
  const int64_t n = c.g->n, n0 = c.g->n0;
  T* gbar = (T*)c.gbar();
  bool flow = false;                          // two-phase packed fp32 path
  if constexpr (std::is_same<T, float>::value) {
    if (spec && !(c.g->flags & GP_FLAG_PER_BATCH_LAUNCH)) {
#define X(K, D) \
      if (c.g->k == K && c.g->d == D) flow = true;
      GP_GRAD_PK_TABLE(X)
#undef X
    }
  }
  GP_CUDA_OK(cudaMemsetAsync(c.ctrl(), 0, kCtrlBytes, c.st));
  // host-buffer variant: v and xi arrive range by range beside the geometry kernel (a point reads only points before
  // it), then v_bar; xi_bar goes home at the end
  EventBag bag;
  constexpr int kVjpChunks = 8;
  const int chunks = (c.io && flow) ? kVjpChunks : 1;
  int64_t cut[kVjpChunks + 1];
  for (int q = 0; q <= chunks; ++q) cut[q] = q == 0 ? 0 : (q == chunks ? n : n0 + (n - n0) * q / chunks);
  cudaEvent_t arrived[kVjpChunks] = {}, vbar_arrived = nullptr;
  if (c.io) {
    GP_OK_OR_RETURN(stream_after(bag, c.io->cin, c.st));
    for (int q = 0; q < chunks; ++q) {
      const size_t bytes = (size_t)(cut[q + 1] - cut[q]) * sizeof(T);
      GP_CUDA_OK(cudaMemcpyAsync((T*)v + cut[q], (const T*)c.io->in_host[1] + cut[q], bytes, cudaMemcpyHostToDevice, c.io->cin));
      GP_CUDA_OK(cudaMemcpyAsync((T*)xi + cut[q], (const T*)c.io->in_host[0] + cut[q], bytes, cudaMemcpyHostToDevice, c.io->cin));
      arrived[q] = bag.make();
      if (!arrived[q]) return GP_ERR_CUDA;
      GP_CUDA_OK(cudaEventRecord(arrived[q], c.io->cin));
    }
    GP_CUDA_OK(cudaMemcpyAsync((T*)vbar, c.io->in_host[2], (size_t)n * sizeof(T), cudaMemcpyHostToDevice, c.io->cin));
    vbar_arrived = bag.make();
    if (!vbar_arrived) return GP_ERR_CUDA;
    GP_CUDA_OK(cudaEventRecord(vbar_arrived, c.io->cin));
  }
  // the head factorisation does not depend on the cotangents: side stream, overlapped with the reverse sweep
  SideStream* side = nullptr;
  GP_OK_OR_RETURN(side_stream(&side));
  GP_OK_OR_RETURN(side_fork(side, c.st));
  if (n0 > 0) {
    OpCtx hc = c;
    hc.st = side->stream;
    GP_OK_OR_RETURN(head_factor(hc, nullptr, 2 * (int)n0, true));
  }
  GP_OK_OR_RETURN(ktime_begin(c.st));
  if (flow) {
    if constexpr (std::is_same<T, float>::value) {
      for (int q = 0; q < chunks; ++q) {
        if (c.io) GP_CUDA_OK(cudaStreamWaitEvent(c.st, arrived[q], 0));
        grad_pack_kernel<T><<<(unsigned)((cut[q + 1] - cut[q] + 255) / 256), 256, 0, c.st>>>(
            (const T*)c.g->x + cut[q] * c.g->d, v + cut[q], (Rec<T>*)c.rec() + cut[q], cut[q + 1] - cut[q], c.g->d);
        GP_LAUNCH_CHECK();
#define X(K, D) \
        if (c.g->k == K && c.g->d == D) GP_OK_OR_RETURN((launch_vjp_geom<K, D>(c, xi, cut[q] < n0 ? n0 : cut[q], cut[q + 1])));
        GP_GRAD_PK_TABLE(X)
#undef X
      }
      if (c.io) GP_CUDA_OK(cudaStreamWaitEvent(c.st, vbar_arrived, 0));
      GP_CUDA_OK(cudaMemcpyAsync(gbar, vbar, (size_t)n * sizeof(T), cudaMemcpyDeviceToDevice, c.st));
      if (c.g->k == 8) GP_OK_OR_RETURN((launch_vjp_scatter<8>(c, gbar, xibar, c.io ? &bag : nullptr)));
      else GP_OK_OR_RETURN((launch_vjp_scatter<16>(c, gbar, xibar, c.io ? &bag : nullptr)));
    }
  } else {
    if (c.io) {
      GP_CUDA_OK(cudaStreamWaitEvent(c.st, arrived[0], 0));
      GP_CUDA_OK(cudaStreamWaitEvent(c.st, vbar_arrived, 0));
    }
    GP_CUDA_OK(cudaMemcpyAsync(gbar, vbar, (size_t)n * sizeof(T), cudaMemcpyDeviceToDevice, c.st));
    if (spec) GP_OK_OR_RETURN(grad_pack<T>(c, v));
    const int64_t* off = c.g->batch_off;
    for (int b = c.g->n_batches - 1; b >= 0; --b)
      GP_OK_OR_RETURN((launch_grad_range<T, GRAD_VJP>(c, spec, v, xi, gbar, xibar, off[b], off[b + 1])));
  }
  GP_OK_OR_RETURN(ktime_end(c.st));
  GP_OK_OR_RETURN(side_join(side, c.st));
  if (n0 > 0) GP_OK_OR_RETURN(head_vjp(c, xi, gbar, xibar, &c.ctrl()->acc[3]));
  finalize_grad_kernel<<<1, 32, 0, c.st>>>(c.ctrl(), 3, 4, 1.0 / c.kern->ell, thetabar);
  GP_LAUNCH_CHECK();
  if (c.io) {
    // the dataflow path has sent xi_bar[n0:] home part by part already: only the head's xi_bar is left
    const int64_t cnt_out = (flow && n > n0) ? n0 : n;
    GP_CUDA_OK(cudaMemcpyAsync(c.io->out_host, xibar, (size_t)cnt_out * sizeof(T), cudaMemcpyDeviceToHost, c.st));
    GP_OK_OR_RETURN(stream_after(bag, c.st, c.io->cout));   // the caller's stream ends when all of xi_bar is on the host
  }
  return GP_OK;
}

template <typename T>
static gp_status geometry_t(const OpCtx& c, const T* xi, const T* v) {
  const int64_t n = c.g->n, n0 = c.g->n0, cnt = n - n0;
  if (cnt <= 0) return GP_OK;
  if constexpr (std::is_same<T, float>::value) {
    if (grad_use_spec(c)) {
      bool pk = false;
#define X(K, D) \
      if (c.g->k == K && c.g->d == D) pk = true;
      GP_GRAD_PK_TABLE(X)
#undef X
      if (pk) {
        GP_OK_OR_RETURN(grad_pack<T>(c, v));
#define X(K, D) \
        if (c.g->k == K && c.g->d == D) return launch_vjp_geom<K, D>(c, xi, n0, n);
        GP_GRAD_PK_TABLE(X)
#undef X
      }
    }
  }
  const int k = c.g->k;
  int active = generic_active_threads(k, sizeof(T), true);
  int threads = (active + 31) / 32 * 32;
  size_t smem = (size_t)generic_scratch_elems(k, true) * sizeof(T) * active;
  GP_CUDA_OK(cudaFuncSetAttribute(geom_generic_kernel<T>, cudaFuncAttributeMaxDynamicSharedMemorySize, 220 * 1024));
  unsigned grid = (unsigned)((cnt + active - 1) / active);
  KParams<T> kp = make_kparams<T>(*c.kern);
  T* wbuf = (T*)c.wbuf();
  geom_generic_kernel<T><<<grid, threads, smem, c.st>>>((const T*)c.g->x, v, c.g->nbr, xi, wbuf, wbuf + (size_t)cnt * k, n0, n,
                                                       c.g->d, k, c.kern->kind, kp, c.ctrl(), active);
  GP_LAUNCH_CHECK();
  return GP_OK;
}
gp_status run_geometry(const OpCtx& c, const void* xi, const void* v) {
  return c.g->dtype == GP_F64 ? geometry_t<double>(c, (const double*)xi, (const double*)v)
                              : geometry_t<float>(c, (const float*)xi, (const float*)v);
}

gp_status run_vjp(const OpCtx& c, const void* xi, const void* v, const void* vbar, void* xibar, double* thetabar) {
  return c.g->dtype == GP_F64 ? vjp_t<double>(c, (const double*)xi, (const double*)v, (const double*)vbar, (double*)xibar, thetabar)
                              : vjp_t<float>(c, (const float*)xi, (const float*)v, (const float*)vbar, (float*)xibar, thetabar);
}

// gradient of the log-determinant: acc[1] = d/dsigma, acc[2] = ell * d/dell (conditioning part)
template <typename T>
static gp_status logdet_grad_t(const OpCtx& c) {
  bool spec = grad_use_spec(c);
  if constexpr (std::is_same<T, float>::value) {
    if (spec) {
#define X(K, D) \
      if (c.g->k == K && c.g->d == D) return launch_logdet_grad_pk<K, D>(c);
      GP_GRAD_PK_TABLE(X)
#undef X
    }
  }
  return launch_grad_range<T, GRAD_LOGDET>(c, spec, nullptr, nullptr, nullptr, nullptr, c.g->n0, c.g->n);
}
gp_status run_logdet_grad(const OpCtx& c) {
  return c.g->dtype == GP_F64 ? logdet_grad_t<double>(c) : logdet_grad_t<float>(c);
}

}  // namespace gp
