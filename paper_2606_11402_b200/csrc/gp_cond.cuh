// Per-point Gaussian conditioning (Eq. 2) in Alg. 1's joint-Cholesky form
// (PAPER.md:70-77):  M = K/sigma^2 over [c(i), i];  L = chol(M);  l = L[k][0:k], s = L[k][k];
// z = L_cc^-1 v_c carried through the factorisation as one more row;  K_ic K_cc^-1 v_c = l.z.
// No back-substitution is needed for forward / inverse / logdet.
//
// Two realisations:
//   condition_reg      compile-time (K, D, KIND): the (K+1)(K+2)/2 triangle, the K carried values and the
//                      K+1 coordinate records live in registers, every loop fully unrolled
//                      so no register array is ever indexed dynamically (no local-memory spill).
//   condition_generic  run-time (k, d, kind): the triangle lives in shared memory, one column of
//                      the per-thread scratch per thread (bank-conflict free), any k <= 64, d <= 4.
#pragma once
#include "gp_common.cuh"

namespace gp {

__host__ __device__ constexpr int tri(int r, int c) { return r * (r + 1) / 2 + c; }

// ---- record loads ------------------------------------------------------------------------------
// COHERENT = false: read-only path (ld.global.nc).  COHERENT = true: L2-coherent load (ld.global.cg),
// needed when another CTA of the SAME launch produced the value (dataflow forward).
template <bool COHERENT> __device__ __forceinline__ Rec<float> load_rec(const Rec<float>* p) {
  float4 t = COHERENT ? __ldcg(reinterpret_cast<const float4*>(p)) : __ldg(reinterpret_cast<const float4*>(p));
  Rec<float> r; r.x0 = t.x; r.x1 = t.y; r.x2 = t.z; r.v = t.w; return r;
}
template <bool COHERENT> __device__ __forceinline__ Rec<double> load_rec(const Rec<double>* p) {
  const double2* q = reinterpret_cast<const double2*>(p);
  double2 a = COHERENT ? __ldcg(q) : __ldg(q);
  double2 b = COHERENT ? __ldcg(q + 1) : __ldg(q + 1);
  Rec<double> r; r.x0 = a.x; r.x1 = a.y; r.x2 = b.x; r.v = b.y; return r;
}

// Ordinary (L1-allocating) load of a record that a CTA of the same launch may still be writing: the
// coordinates never change, and the value word is either "pending" or final (see forward_flow_kernel).
__device__ __forceinline__ Rec<float> load_rec_l1(const Rec<float>* p) {
  float4 t;
  asm volatile("ld.global.ca.v4.f32 {%0, %1, %2, %3}, [%4];" : "=f"(t.x), "=f"(t.y), "=f"(t.z), "=f"(t.w) : "l"(p));
  Rec<float> r; r.x0 = t.x; r.x1 = t.y; r.x2 = t.z; r.v = t.w; return r;
}
__device__ __forceinline__ Rec<double> load_rec_l1(const Rec<double>* p) {
  double a, b, c, d;
  asm volatile("ld.global.ca.v2.f64 {%0, %1}, [%2];" : "=d"(a), "=d"(b) : "l"(p));
  asm volatile("ld.global.ca.v2.f64 {%0, %1}, [%2];" : "=d"(c), "=d"(d) : "l"(reinterpret_cast<const double*>(p) + 2));
  Rec<double> r; r.x0 = a; r.x1 = b; r.x2 = c; r.v = d; return r;
}

__device__ __forceinline__ float load_val_l1(const float* p) {
  float v; asm volatile("ld.global.ca.f32 %0, [%1];" : "=f"(v) : "l"(p)); return v;
}
__device__ __forceinline__ double load_val_l1(const double* p) {
  double v; asm volatile("ld.global.ca.f64 %0, [%1];" : "=d"(v) : "l"(p)); return v;
}

template <typename T, int D> __device__ __forceinline__ T pair_q(const Rec<T>& a, const Rec<T>& b, T qscale) {
  T dx = a.x0 - b.x0;
  T d2 = dx * dx;
  if (D >= 2) { T dy = a.x1 - b.x1; d2 = Math<T>::fma(dy, dy, d2); }
  if (D >= 3) { T dz = a.x2 - b.x2; d2 = Math<T>::fma(dz, dz, d2); }
  return d2 * qscale;
}

// Load the K neighbour indices of one row (streaming: every index is read exactly once per op).
template <int K> __device__ __forceinline__ void load_row(const int32_t* __restrict__ row, int32_t (&idx)[K]) {
  if (K % 4 == 0) {
    const int4* r4 = reinterpret_cast<const int4*>(row);
#pragma unroll
    for (int j = 0; j < K / 4; ++j) {
      int4 t = __ldcs(r4 + j);
      idx[4 * j + 0] = t.x; idx[4 * j + 1] = t.y; idx[4 * j + 2] = t.z; idx[4 * j + 3] = t.w;
    }
  } else {
#pragma unroll
    for (int j = 0; j < K; ++j) idx[j] = __ldcs(row + j);
  }
}

// Result of one conditioning in unit-sigma form.
template <typename T> struct Cond {
  T m;   // K_ic K_cc^-1 v_c
  T s;   // sqrt(M_ii - M_ic M_cc^-1 M_ci)   (multiply by sigma for the conditional std)
  bool ok;
};

// Register-resident conditioning, in three pieces so that the gradient kernels (gp_vjp.cu) can keep the
// factor.  Every loop is fully unrolled: no register array is ever indexed dynamically.
template <typename T, int K, bool COHERENT>
__device__ __forceinline__ void gather_reg(const Rec<T>* __restrict__ rec, const int32_t* __restrict__ row,
                                           int32_t (&idx)[K], Rec<T> (&R)[K]) {
  load_row<K>(row, idx);
#pragma unroll
  for (int j = 0; j < K; ++j) R[j] = load_rec<COHERENT>(rec + idx[j]);
}

// joint matrix M = K / sigma^2, lower triangle, rows 0..K-1 = neighbours, row K = the point itself
template <typename T, int K, int D, int KIND>
__device__ __forceinline__ void build_joint_reg(const Rec<T> (&R)[K], const Rec<T>& self, const KParams<T>& kp,
                                                T (&A)[(K + 1) * (K + 2) / 2]) {
#pragma unroll
  for (int r = 0; r <= K; ++r) {
#pragma unroll
    for (int c = 0; c < r; ++c) {
      T q = (r == K) ? pair_q<T, D>(self, R[c], kp.qscale) : pair_q<T, D>(R[r], R[c], kp.qscale);
      A[tri(r, c)] = Math<T>::template rho_from_q<KIND>(q);
    }
    A[tri(r, r)] = kp.diag;
  }
}

// in-place right-looking Cholesky with the values row cv carried along.
// On return A holds L below the diagonal, cv = z = L_cc^-1 v_c.  KEEP_INV: A[j][j] = 1 / L_jj (j < K).
template <typename T, int K, bool KEEP_INV, bool CARRY = true>
__device__ __forceinline__ Cond<T> factor_joint_reg(T (&A)[(K + 1) * (K + 2) / 2], T (&cv)[K], const KParams<T>& kp) {
  T m = T(0);
  T minpiv = kp.diag;
#pragma unroll
  for (int j = 0; j < K; ++j) {
    T piv = A[tri(j, j)];
    minpiv = Math<T>::fmin(minpiv, piv);
    T inv = Math<T>::rsqrt(piv);
    if (KEEP_INV) A[tri(j, j)] = inv;
#pragma unroll
    for (int r = j + 1; r <= K; ++r) A[tri(r, j)] *= inv;
    T zj = T(0);
    if (CARRY) { zj = cv[j] * inv; cv[j] = zj; }
#pragma unroll
    for (int r = j + 1; r <= K; ++r) {
#pragma unroll
      for (int c = j + 1; c <= r; ++c) A[tri(r, c)] = Math<T>::fma(-A[tri(r, j)], A[tri(c, j)], A[tri(r, c)]);
    }
    if (CARRY) {
#pragma unroll
      for (int c = j + 1; c < K; ++c) cv[c] = Math<T>::fma(-zj, A[tri(c, j)], cv[c]);
      m = Math<T>::fma(zj, A[tri(K, j)], m);
    }
  }
  T s2 = A[tri(K, K)];
  minpiv = Math<T>::fmin(minpiv, s2);
  Cond<T> out;
  out.ok = (minpiv > T(0)) && (s2 < T(3.0e38));
  out.m = m;
  out.s = Math<T>::sqrt(s2);
  return out;
}

template <typename T, int K, int D, int KIND, bool COHERENT>
__device__ __forceinline__ Cond<T> condition_reg(const Rec<T>* __restrict__ rec, const int32_t* __restrict__ row,
                                                 const Rec<T>& self, const KParams<T>& kp) {
  int32_t idx[K];
  Rec<T> R[K];
  gather_reg<T, K, COHERENT>(rec, row, idx, R);
  T A[(K + 1) * (K + 2) / 2];
  build_joint_reg<T, K, D, KIND>(R, self, kp, A);
  T cv[K];
#pragma unroll
  for (int j = 0; j < K; ++j) cv[j] = R[j].v;
  return factor_joint_reg<T, K, false>(A, cv, kp);
}

// v-independent half of the conditioning (dataflow forward): factor the joint matrix WITHOUT a carried values
// row, then back-substitute  w = L_cc^-T l  (= K_cc^-1 K_ci, Eq. 2), so that all that is left once the
// neighbour values exist is the dot product  m = w . v_c.
template <typename T, int K, int D, int KIND>
__device__ __forceinline__ Cond<T> weights_reg(const Rec<T> (&R)[K], const Rec<T>& self, const KParams<T>& kp,
                                               T (&w)[K]) {
  T A[(K + 1) * (K + 2) / 2];
  build_joint_reg<T, K, D, KIND>(R, self, kp, A);
  Cond<T> c = factor_joint_reg<T, K, true, false>(A, w, kp);
#pragma unroll
  for (int j = K - 1; j >= 0; --j) {
    T t = A[tri(K, j)];
#pragma unroll
    for (int r = j + 1; r < K; ++r) t = Math<T>::fma(-A[tri(r, j)], w[r], t);
    w[j] = t * A[tri(j, j)];
  }
  return c;
}

// ---- generic: triangle in shared memory ------------------------------------------------------------
// Per-thread scratch column: element e of thread t lives at base[e * stride + t].
template <typename T> struct Scratch {
  T* p;
  int stride;
  __device__ __forceinline__ T& operator[](int e) const { return p[(size_t)e * stride]; }
};

__host__ __device__ inline int generic_scratch_elems(int k, bool with_vjp) {
  int e = (k + 1) * (k + 2) / 2 + k;       // triangle + carried values
  if (with_vjp) e += (k + 1);              // y = D u
  return e;
}

template <typename T>
__device__ __forceinline__ T dist_q(const T* __restrict__ x, int d, int64_t a, int64_t b, T qscale) {
  T d2 = T(0);
  for (int t = 0; t < d; ++t) { T dx = x[a * d + t] - x[b * d + t]; d2 = Math<T>::fma(dx, dx, d2); }
  return d2 * qscale;
}

// vals may be null (logdet).  Leaves L in A (triangle) and z in A[NT + j].
template <typename T>
__device__ Cond<T> condition_generic(const T* __restrict__ x, const T* vals, int d, int k, int kind,
                                     const int32_t* __restrict__ row, int64_t i, const KParams<T>& kp,
                                     const Scratch<T>& A) {
  const int NT = (k + 1) * (k + 2) / 2;
  for (int r = 0; r <= k; ++r) {
    int64_t pr = (r == k) ? i : (int64_t)row[r];
    for (int c = 0; c < r; ++c) A[tri(r, c)] = rho_rt<T>(kind, dist_q<T>(x, d, pr, (int64_t)row[c], kp.qscale));
    A[tri(r, r)] = kp.diag;
  }
  for (int j = 0; j < k; ++j) A[NT + j] = vals ? vals[row[j]] : T(0);
  T m = T(0);
  T minpiv = kp.diag;
  for (int j = 0; j < k; ++j) {
    T piv = A[tri(j, j)];
    minpiv = Math<T>::fmin(minpiv, piv);
    T inv = Math<T>::rsqrt(piv);
    A[tri(j, j)] = piv * inv;              // L_jj (the specialised path never needs it; VJP does)
    for (int r = j + 1; r <= k; ++r) A[tri(r, j)] *= inv;
    T zj = A[NT + j] * inv;
    A[NT + j] = zj;
    for (int r = j + 1; r <= k; ++r) {
      T lrj = A[tri(r, j)];
      for (int c = j + 1; c <= r; ++c) A[tri(r, c)] = Math<T>::fma(-lrj, A[tri(c, j)], A[tri(r, c)]);
    }
    for (int c = j + 1; c < k; ++c) A[NT + c] = Math<T>::fma(-zj, A[tri(c, j)], A[NT + c]);
    m = Math<T>::fma(zj, A[tri(k, j)], m);
  }
  T s2 = A[tri(k, k)];
  minpiv = Math<T>::fmin(minpiv, s2);
  Cond<T> out;
  out.ok = (minpiv > T(0)) && (s2 < T(1e300) || sizeof(T) == 4) && (s2 == s2);
  out.m = m;
  out.s = Math<T>::sqrt(s2);
  A[tri(k, k)] = out.s;
  return out;
}

// ---- block reduction of doubles (logdet, theta_bar) ---------------------------------------------------
__device__ __forceinline__ double warp_sum(double v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v += __shfl_down_sync(0xffffffffu, v, o);
  return v;
}
// Sums `v` over the block and adds the total to *dst with one atomic.  All threads must call it.
__device__ __forceinline__ void block_atomic_add(double v, double* dst, double* red /* shared, >= 32 doubles */) {
  v = warp_sum(v);
  int lane = threadIdx.x & 31, w = threadIdx.x >> 5, nw = (blockDim.x + 31) >> 5;
  if (lane == 0) red[w] = v;
  __syncthreads();
  if (w == 0) {
    double t = (lane < nw) ? red[lane] : 0.0;
    t = warp_sum(t);
    if (lane == 0) atomicAdd(dst, t);
  }
  __syncthreads();
}

}  // namespace gp
