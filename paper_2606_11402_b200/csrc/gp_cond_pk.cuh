// Packed-fp32 (FFMA2 / FMUL2 / FADD2) realisation of the per-point conditioning for sm_100a.
//
// Blackwell's FMA pipe retires a 3-register scalar FFMA at about 72 lanes/clk/SM but a packed fma.rn.f32x2
// at about 112 FMA-lanes/clk/SM (measured on B200), and a packed instruction takes one issue
// slot for two results.  The joint (k+1) x (k+1) matrix of Alg. 1 is therefore held as
// VERTICAL pairs: pair (rp, c) = (A[2 rp][c], A[2 rp + 1][c]).  In a right-looking step j the update
//     A[r][c] -= L[r][j] L[c][j]
// becomes, for two rows at once,   P[rp][c] -= P[rp][j] * bcast(L[c][j]),
// where the second factor is ONE scalar register (the SASS operand form `Rn.F32` broadcasts it to both
// halves), so no shuffling or duplicating moves are needed.  Row k is the point itself and row k + 1 the
// carried values row: they form the last pair, whose column k ends as (s^2, -m).
// The triangle costs k/2 (k/2 + 1) + k + 1 register pairs (89 for k = 16).  k must be even.
#pragma once
#include "gp_cond.cuh"

namespace gp {

typedef float2 f2;
__device__ __forceinline__ f2 bc(float a) { return make_float2(a, a); }
__device__ __forceinline__ f2 neg2(f2 a) { return make_float2(-a.x, -a.y); }
__device__ __forceinline__ f2 fma2(f2 a, f2 b, f2 c) { return __ffma2_rn(a, b, c); }
__device__ __forceinline__ f2 mul2(f2 a, f2 b) { return __fmul2_rn(a, b); }
__device__ __forceinline__ f2 add2(f2 a, f2 b) { return __fadd2_rn(a, b); }

__host__ __device__ constexpr int pk_pairs(int K) { return (K / 2) * (K / 2 + 1) + K + 1; }
// pair rp holds columns 0 .. min(2 rp + 1, K)
__host__ __device__ constexpr int pk(int rp, int c) { return rp * (rp + 1) + c; }

template <int KIND> __device__ __forceinline__ f2 rho2_from_q(f2 q) {
  if (KIND == GP_KERNEL_SE) return make_float2(Math<float>::ex2(-q.x), Math<float>::ex2(-q.y));
  f2 t = make_float2(Math<float>::sqrt_approx(q.x), Math<float>::sqrt_approx(q.y));
  f2 e = make_float2(Math<float>::ex2(-t.x), Math<float>::ex2(-t.y));
  if (KIND == GP_KERNEL_MATERN32) return mul2(fma2(t, bc(0.69314718055994530942f), bc(1.0f)), e);
  return e;
}

template <int K> struct PkCoords { f2 x0[K / 2], x1[K / 2], x2[K / 2]; };

// Coordinates relative to the point itself, scaled by sqrt(qscale), rows paired vertically.  The difference
// is taken on the raw coordinates first (exact for nearby points), the scale applied afterwards.
template <int K, int D>
__device__ __forceinline__ void centre_pk(const Rec<float> (&R)[K], const Rec<float>& self, float sq, PkCoords<K>& X) {
#pragma unroll
  for (int rp = 0; rp < K / 2; ++rp) {
    X.x0[rp] = mul2(add2(make_float2(R[2 * rp].x0, R[2 * rp + 1].x0), bc(-self.x0)), bc(sq));
    if (D >= 2) X.x1[rp] = mul2(add2(make_float2(R[2 * rp].x1, R[2 * rp + 1].x1), bc(-self.x1)), bc(sq));
    if (D >= 3) X.x2[rp] = mul2(add2(make_float2(R[2 * rp].x2, R[2 * rp + 1].x2), bc(-self.x2)), bc(sq));
  }
}

__device__ __forceinline__ float half_of(const f2& p, int odd) { return odd ? p.y : p.x; }

// Joint matrix M = K / sigma^2 over [c(i), i] plus the values row, in vertical pairs.
template <int K, int D, int KIND>
__device__ __forceinline__ void build_joint_pk(const PkCoords<K>& X, const float (&vals)[K], const KParams<float>& kp,
                                               f2 (&P)[pk_pairs(K)]) {
  constexpr int H = K / 2;
#pragma unroll
  for (int c = 0; c < K; ++c) {
    const int cp = c / 2, odd = c & 1;
    const float c0 = half_of(X.x0[cp], odd);
    const float c1 = D >= 2 ? half_of(X.x1[cp], odd) : 0.0f;
    const float c2 = D >= 3 ? half_of(X.x2[cp], odd) : 0.0f;
    if (!odd) {   // rows (c, c + 1): diagonal of c, and the entry (c + 1, c)
      float dx = X.x0[cp].y - c0;
      float q = dx * dx;
      if (D >= 2) { float dy = X.x1[cp].y - c1; q = fmaf(dy, dy, q); }
      if (D >= 3) { float dz = X.x2[cp].y - c2; q = fmaf(dz, dz, q); }
      P[pk(cp, c)] = make_float2(kp.diag, Math<float>::template rho_from_q<KIND>(q));
    } else {      // rows (c - 1, c): above the diagonal (never read), diagonal of c
      P[pk(cp, c)] = make_float2(0.0f, kp.diag);
    }
#pragma unroll
    for (int rp = cp + 1; rp < H; ++rp) {
      f2 dx = add2(X.x0[rp], bc(-c0));
      f2 q = mul2(dx, dx);
      if (D >= 2) { f2 dy = add2(X.x1[rp], bc(-c1)); q = fma2(dy, dy, q); }
      if (D >= 3) { f2 dz = add2(X.x2[rp], bc(-c2)); q = fma2(dz, dz, q); }
      P[pk(rp, c)] = rho2_from_q<KIND>(q);
    }
    // last pair: (the point itself, the carried value); centred coordinates ARE the differences
    float qs = c0 * c0;
    if (D >= 2) qs = fmaf(c1, c1, qs);
    if (D >= 3) qs = fmaf(c2, c2, qs);
    P[pk(H, c)] = make_float2(Math<float>::template rho_from_q<KIND>(qs), vals[c]);
  }
  P[pk(H, K)] = make_float2(kp.diag, 0.0f);
}

// In-place right-looking Cholesky on the paired triangle, values row carried.
// On return column j holds L[.][j] (rows > j); P[pk(K/2, K)] = (s^2, -m).  KEEP_INV: the diagonal slot of
// column j holds 1 / L_jj.  Returns false if a pivot or s^2 was not positive and finite.
template <int K, bool KEEP_INV>
__device__ __forceinline__ bool factor_joint_pk(f2 (&P)[pk_pairs(K)], float diag) {
  constexpr int H = K / 2;
  float minpiv = diag;
#pragma unroll
  for (int j = 0; j < K; ++j) {
    const int jp = j / 2, odd = j & 1;
    const float piv = half_of(P[pk(jp, j)], odd);
    minpiv = fminf(minpiv, piv);
    const float inv = Math<float>::rsqrt(piv);
    if (!odd) {
      P[pk(jp, j)] = mul2(P[pk(jp, j)], bc(inv));
      if (KEEP_INV) P[pk(jp, j)].x = inv;
    } else if (KEEP_INV) {
      P[pk(jp, j)].y = inv;
    }
#pragma unroll
    for (int rp = jp + 1; rp <= H; ++rp) P[pk(rp, j)] = mul2(P[pk(rp, j)], bc(inv));
#pragma unroll
    for (int c = j + 1; c <= K; ++c) {
      const float lc = half_of(P[pk(c / 2, j)], c & 1);
#pragma unroll
      for (int rp = c / 2; rp <= H; ++rp) P[pk(rp, c)] = fma2(neg2(P[pk(rp, j)]), bc(lc), P[pk(rp, c)]);
    }
  }
  const float s2 = P[pk(H, K)].x;
  minpiv = fminf(minpiv, s2);
  return (minpiv > 0.0f) && (s2 < 3.0e38f);
}

// forward / inverse / logdet body on gathered records: build, factor.
template <int K, int D, int KIND>
__device__ __forceinline__ Cond<float> condition_pk_rec(const Rec<float> (&R)[K], const Rec<float>& self,
                                                        const KParams<float>& kp) {
  f2 P[pk_pairs(K)];
  {
    PkCoords<K> X;
    centre_pk<K, D>(R, self, kp.sq, X);
    float vals[K];
#pragma unroll
    for (int j = 0; j < K; ++j) vals[j] = R[j].v;
    build_joint_pk<K, D, KIND>(X, vals, kp, P);
  }
  Cond<float> out;
  out.ok = factor_joint_pk<K, false>(P, kp.diag);
  out.m = -P[pk(K / 2, K)].y;
  out.s = Math<float>::sqrt(P[pk(K / 2, K)].x);
  return out;
}

template <int K, int D, int KIND, bool COHERENT>
__device__ __forceinline__ Cond<float> condition_pk(const Rec<float>* __restrict__ rec, const int32_t* __restrict__ row,
                                                    const Rec<float>& self, const KParams<float>& kp) {
  int32_t idx[K];
  Rec<float> R[K];
  gather_reg<float, K, COHERENT>(rec, row, idx, R);
  return condition_pk_rec<K, D, KIND>(R, self, kp);
}

// v-independent half for the dataflow forward: weights w = L_cc^-T l (= K_cc^-1 K_ci, Eq. 2) and s.
template <int K, int D, int KIND>
__device__ __forceinline__ Cond<float> weights_pk(const Rec<float> (&R)[K], const Rec<float>& self,
                                                  const KParams<float>& kp, float (&w)[K]) {
  constexpr int H = K / 2;
  f2 P[pk_pairs(K)];
  {
    PkCoords<K> X;
    centre_pk<K, D>(R, self, kp.sq, X);
    float vals[K];
#pragma unroll
    for (int j = 0; j < K; ++j) vals[j] = 0.0f;
    build_joint_pk<K, D, KIND>(X, vals, kp, P);
  }
  Cond<float> out;
  out.ok = factor_joint_pk<K, true>(P, kp.diag);
  out.m = 0.0f;
  out.s = Math<float>::sqrt(P[pk(H, K)].x);
  // back-substitution with W[rp] = (w[2 rp], w[2 rp + 1]):  w_j = (l_j - sum_{r > j} L[r][j] w_r) / L_jj
  f2 W[H];
#pragma unroll
  for (int j = K - 1; j >= 0; --j) {
    const int jp = j / 2, odd = j & 1;
    f2 acc = make_float2(0.0f, 0.0f);
#pragma unroll
    for (int rp = jp + 1; rp < H; ++rp) acc = fma2(P[pk(rp, j)], W[rp], acc);
    float t = P[pk(H, j)].x - (acc.x + acc.y);
    if (!odd) t = fmaf(-P[pk(jp, j)].y, W[jp].y, t);       // row j + 1 shares the pair of row j
    const float inv = half_of(P[pk(jp, j)], odd);
    const float wj = t * inv;
    if (odd) W[jp].y = wj; else W[jp].x = wj;
  }
#pragma unroll
  for (int rp = 0; rp < H; ++rp) { w[2 * rp] = W[rp].x; w[2 * rp + 1] = W[rp].y; }
  return out;
}

}  // namespace gp
