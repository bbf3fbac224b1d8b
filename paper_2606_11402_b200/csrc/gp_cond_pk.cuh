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

// ---- gamma form -----------------------------------------------------------------------------------------
// In fp32 the entries rho = 1 - gamma of a tight neighbourhood (r << ell) all round to "1 - a few ulp", and the
// first elimination step subtracts O(1) numbers to leave O(gamma + eps) ones: the information is gone before
// the factorisation starts (measured: max |dv| = 1.8e-4 std(v) on config 3, above the 1e-4 bar).  So the
// packed path never forms rho.  It evaluates gamma = 1 - rho WITHOUT cancellation (a short series below a
// threshold, 1 - rho above it, where gamma is no longer small), and performs the elimination of neighbour 0
// analytically on the gammas (eliminate0_pk); the factorisation then starts at column 1 on a matrix whose
// entries are O(gamma + eps).  This is Eq. 2 / Alg. 1 unchanged - the same Cholesky, its first step done in
// exact arithmetic - so the oracle (which works in fp64 on rho) is still the reference.
// Branch selection without predicated moves: w = 1.0f where the series applies, else 0.0f (FSET on the ALU pipe),
// then gamma = big + w (small - big) as packed arithmetic.
__device__ __forceinline__ f2 below2(f2 a, float thr) { return make_float2(a.x < thr ? 1.0f : 0.0f, a.y < thr ? 1.0f : 0.0f); }
__device__ __forceinline__ f2 blend2(f2 w, f2 small, f2 big) { return fma2(w, add2(small, neg2(big)), big); }

// gamma(q), q = qscale |dx|^2 (base-2 scaling: rho = 2^-q (SE), (1 + t ln2) 2^-t (Matern-3/2), 2^-t (exp), t = sqrt q).
// Below the threshold the series is used; its truncation and, above the threshold, the 2^-22 relative error of
// MUFU.EX2 in 1 - rho both stay below about 4e-6 relative to gamma (against 1e-7 / gamma for 1 - rho alone).
// Measured on config 3 at N = 2^23: max |dv| / std(v) = 1.8e-4 (rho form), 1.05e-4 (threshold 0.17, 3 terms),
// 7.5e-5 (threshold 0.25, 5 terms), 5.4e-5 (threshold 0.5, 7 terms, series in a), 7.4e-5 (the same series written
// in t, one packed instruction less per pair: the one kept), 1.4e-4 (threshold 0.5 with 6 terms: the dropped term is
// 5e-6 of gamma at the threshold, and that is already too much); the bar is 1e-4.  What is left is the fp32 Cholesky
// itself (condition number ~ 1 / eps times the fp32 epsilon).
template <int KIND> __device__ __forceinline__ f2 gamma2_from_q(f2 q) {
  const float ln2 = 0.69314718055994530942f;
  if (KIND == GP_KERNEL_SE) {
    const f2 u = mul2(q, bc(ln2));                                  // r^2 / (2 ell^2)
    const f2 big = make_float2(1.0f - Math<float>::ex2(-q.x), 1.0f - Math<float>::ex2(-q.y));
    f2 p = fma2(u, bc(1.0f / 120.0f), bc(-1.0f / 24.0f));           // 1 - e^-u = u (1 - u/2 + u^2/6 - u^3/24 + u^4/120 ...)
    p = fma2(u, p, bc(1.0f / 6.0f));
    p = fma2(u, p, bc(-0.5f));
    p = fma2(u, p, bc(1.0f));
    return blend2(below2(u, 0.125f), mul2(u, p), big);
  }
  // the series are written in t = a / ln2 (coefficients carry the powers of ln2) so that a itself is never formed
  const f2 t = make_float2(Math<float>::sqrt_approx(q.x), Math<float>::sqrt_approx(q.y));
  const f2 e = make_float2(Math<float>::ex2(-t.x), Math<float>::ex2(-t.y));
  constexpr double L1 = 0.69314718055994530942, L2 = L1 * L1, L3 = L2 * L1, L4 = L3 * L1, L5 = L4 * L1, L6 = L5 * L1,
                   L7 = L6 * L1, L8 = L7 * L1;   // coefficients rounded to fp32 once
  constexpr float l1 = (float)L1;
  if (KIND == GP_KERNEL_MATERN32) {
    const f2 big = fma2(neg2(fma2(t, bc(l1), bc(1.0f))), e, bc(1.0f));     // 1 - (1 + a) e^-a
    // 1 - (1 + a) e^-a = a^2 (1/2 - a/3 + a^2/8 - a^3/30 + a^4/144 - a^5/840 + a^6/5760 - ...)
    f2 p = fma2(t, bc((float)(L8 / 5760.0)), bc((float)(-L7 / 840.0)));
    p = fma2(t, p, bc((float)(L6 / 144.0)));
    p = fma2(t, p, bc((float)(-L5 / 30.0)));
    p = fma2(t, p, bc((float)(L4 * 0.125)));
    p = fma2(t, p, bc((float)(-L3 / 3.0)));
    p = fma2(t, p, bc((float)(L2 * 0.5)));
    return blend2(below2(t, 0.5f / l1), mul2(mul2(t, t), p), big);
  }
  const f2 big = add2(bc(1.0f), neg2(e));
  f2 p = fma2(t, bc((float)(L5 / 120.0)), bc((float)(-L4 / 24.0)));                        // 1 - e^-a = a (1 - a/2 + a^2/6 - ...)
  p = fma2(t, p, bc((float)(L3 / 6.0)));
  p = fma2(t, p, bc((float)(-L2 * 0.5)));
  p = fma2(t, p, bc(l1));
  return blend2(below2(t, 0.125f / l1), mul2(t, p), big);
}
// scalar twin (lane-group kernel): same series, same thresholds
template <int KIND> __device__ __forceinline__ float gamma_from_q(float q) {
  const float ln2 = 0.69314718055994530942f;
  if (KIND == GP_KERNEL_SE) {
    const float u = q * ln2;
    const float big = 1.0f - Math<float>::ex2(-q);
    float p = fmaf(u, 1.0f / 120.0f, -1.0f / 24.0f);
    p = fmaf(u, p, 1.0f / 6.0f);
    p = fmaf(u, p, -0.5f);
    p = fmaf(u, p, 1.0f);
    return u < 0.125f ? u * p : big;
  }
  const float t = Math<float>::sqrt_approx(q);
  const float a = t * ln2;
  const float e = Math<float>::ex2(-t);
  if (KIND == GP_KERNEL_MATERN32) {
    const float big = fmaf(-(1.0f + a), e, 1.0f);
    float p = fmaf(a, 1.0f / 5760.0f, -1.0f / 840.0f);
    p = fmaf(a, p, 1.0f / 144.0f);
    p = fmaf(a, p, -1.0f / 30.0f);
    p = fmaf(a, p, 0.125f);
    p = fmaf(a, p, -1.0f / 3.0f);
    p = fmaf(a, p, 0.5f);
    return a < 0.5f ? a * a * p : big;
  }
  const float big = 1.0f - e;
  float p = fmaf(a, 1.0f / 120.0f, -1.0f / 24.0f);
  p = fmaf(a, p, 1.0f / 6.0f);
  p = fmaf(a, p, -0.5f);
  p = fmaf(a, p, 1.0f);
  return a < 0.125f ? a * p : big;
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

// GAMMAS of the joint matrix M = K / sigma^2 over [c(i), i] (M_rc = 1 - gamma_rc off the diagonal)
// plus the values row, in vertical pairs.  Diagonal slots are placeholders: eliminate0_pk writes them.
template <int K, int D, int KIND>
__device__ __forceinline__ void build_joint_pk(const PkCoords<K>& X, const float (&vals)[K], const KParams<float>& kp,
                                               f2 (&P)[pk_pairs(K)]) {
  constexpr int H = K / 2;
  // entries (c + 1, c), c even (the two rows of one pair), two pairs per packed evaluation
  float gh[H];
#pragma unroll
  for (int cp = 0; cp < H; cp += 2) {
    const int c2 = cp + 1 < H ? cp + 1 : cp;
    f2 dx = make_float2(X.x0[cp].y - X.x0[cp].x, X.x0[c2].y - X.x0[c2].x);
    f2 q = mul2(dx, dx);
    if (D >= 2) { f2 dy = make_float2(X.x1[cp].y - X.x1[cp].x, X.x1[c2].y - X.x1[c2].x); q = fma2(dy, dy, q); }
    if (D >= 3) { f2 dz = make_float2(X.x2[cp].y - X.x2[cp].x, X.x2[c2].y - X.x2[c2].x); q = fma2(dz, dz, q); }
    const f2 g = gamma2_from_q<KIND>(q);
    gh[cp] = g.x;
    if (cp + 1 < H) gh[cp + 1] = g.y;
  }
  // entries (self, c): the centred coordinates ARE the differences; columns (2 cp, 2 cp + 1) per evaluation
  float gs[K];
#pragma unroll
  for (int cp = 0; cp < H; ++cp) {
    f2 q = mul2(X.x0[cp], X.x0[cp]);
    if (D >= 2) q = fma2(X.x1[cp], X.x1[cp], q);
    if (D >= 3) q = fma2(X.x2[cp], X.x2[cp], q);
    const f2 g = gamma2_from_q<KIND>(q);
    gs[2 * cp] = g.x;
    gs[2 * cp + 1] = g.y;
  }
#pragma unroll
  for (int c = 0; c < K; ++c) {
    const int cp = c / 2, odd = c & 1;
    const float c0 = half_of(X.x0[cp], odd);
    const float c1 = D >= 2 ? half_of(X.x1[cp], odd) : 0.0f;
    const float c2 = D >= 3 ? half_of(X.x2[cp], odd) : 0.0f;
    P[pk(cp, c)] = make_float2(0.0f, odd ? 0.0f : gh[cp]);   // diagonal slots: eliminate0_pk
#pragma unroll
    for (int rp = cp + 1; rp < H; ++rp) {
      f2 dx = add2(X.x0[rp], bc(-c0));
      f2 q = mul2(dx, dx);
      if (D >= 2) { f2 dy = add2(X.x1[rp], bc(-c1)); q = fma2(dy, dy, q); }
      if (D >= 3) { f2 dz = add2(X.x2[rp], bc(-c2)); q = fma2(dz, dz, q); }
      P[pk(rp, c)] = gamma2_from_q<KIND>(q);
    }
    P[pk(H, c)] = make_float2(gs[c], vals[c]);               // last pair: (the point itself, the carried value)
  }
  P[pk(H, K)] = make_float2(0.0f, 0.0f);
}

// Analytic elimination of neighbour 0 (the first Cholesky step in exact arithmetic on the gammas).  With
// g_r = gamma_r0 it leaves, for rows and columns >= 1, S' = (1 + eps) x (Schur complement of M_00):
//   S'_rc = eps + g_r + g_c - g_r g_c - (1 + eps) gamma_rc        S'_rr = (eps + g_r)(2 + eps - g_r)
// the carried values  u_c = (v_c - v_0) + v_0 (g_c + eps) / (1 + eps)  (difference first: values are smooth),
// and the entry (values row, column K) = -v_0 (1 - g_K) / (1 + eps), the first term of -m.
// Scaling S by (1 + eps) leaves m and the weights unchanged and multiplies s^2 by (1 + eps).
// Column 0 of P keeps the gammas g_r (and v_0 in the last pair): the back-substitutions need them.
template <int K>
__device__ __forceinline__ void eliminate0_pk(f2 (&P)[pk_pairs(K)], const KParams<float>& kp) {
  constexpr int H = K / 2;
  const float eps = kp.eps, ope = kp.diag, inv_ope = kp.inv_diag;
  const float gK = P[pk(H, 0)].x, v0 = P[pk(H, 0)].y;
#pragma unroll
  for (int c = 1; c < K; ++c) {
    const int cp = c / 2, odd = c & 1;
    const float gc = half_of(P[pk(cp, 0)], odd);
    const float a = 1.0f - gc, b = eps + gc;
    const float dg = b * (ope + a);
    if (!odd) {
      const float g1 = P[pk(cp, 0)].y;
      P[pk(cp, c)] = make_float2(dg, fmaf(-ope, P[pk(cp, c)].y, fmaf(g1, a, b)));
    } else {
      P[pk(cp, c)] = make_float2(0.0f, dg);
    }
#pragma unroll
    for (int rp = cp + 1; rp < H; ++rp) P[pk(rp, c)] = fma2(P[pk(rp, c)], bc(-ope), fma2(P[pk(rp, 0)], bc(a), bc(b)));
    const float x = fmaf(-ope, P[pk(H, c)].x, fmaf(gK, a, b));
    const float y = fmaf(v0 * inv_ope, b, P[pk(H, c)].y - v0);
    P[pk(H, c)] = make_float2(x, y);
  }
  const float aK = 1.0f - gK;
  P[pk(H, K)] = make_float2((eps + gK) * (ope + aK), -v0 * aK * inv_ope);
}

// In-place right-looking Cholesky on the paired triangle, values row carried.
// Starts at column J0 = 1 (column 0 was eliminated analytically).  On return column j >= 1 holds L'[.][j]
// (rows > j) of S' = L' L'^T;  P[pk(K/2, K)] = ((1 + eps) s^2, -m).  KEEP_INV: the diagonal slot of
// column j holds 1 / L_jj.  Returns false if a pivot or s^2 was not positive and finite.
template <int K, bool KEEP_INV, int J0 = 1>
__device__ __forceinline__ bool factor_joint_pk(f2 (&P)[pk_pairs(K)], float diag) {
  constexpr int H = K / 2;
  float minpiv = diag;
#pragma unroll
  for (int j = J0; j < K; ++j) {
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
  eliminate0_pk<K>(P, kp);
  Cond<float> out;
  out.ok = factor_joint_pk<K, false>(P, kp.diag);
  out.m = -P[pk(K / 2, K)].y;
  out.s = Math<float>::sqrt(P[pk(K / 2, K)].x * kp.inv_diag);
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

// top - sum_{r >= 1} (1 - g_r) Y_r  for a vector Y held as vertical pairs (row 0 of the back-substitutions)
template <int K>
__device__ __forceinline__ float w0_pk(const f2 (&P)[pk_pairs(K)], const f2 (&Y)[K / 2], float top) {
  f2 acc = make_float2(0.0f, 0.0f);
#pragma unroll
  for (int rp = 1; rp < K / 2; ++rp) acc = fma2(add2(bc(1.0f), neg2(P[pk(rp, 0)])), Y[rp], acc);
  return fmaf(-(1.0f - P[pk(0, 0)].y), Y[0].y, top - (acc.x + acc.y));
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
  eliminate0_pk<K>(P, kp);
  Cond<float> out;
  out.ok = factor_joint_pk<K, true>(P, kp.diag);
  out.m = 0.0f;
  out.s = Math<float>::sqrt(P[pk(H, K)].x * kp.inv_diag);
  // back-substitution with W[rp] = (w[2 rp], w[2 rp + 1]):  w_j = (l_j - sum_{r > j} L[r][j] w_r) / L_jj, j >= 1
  // (scale free: L' and l' carry the same factor), then  w_0 = ((1 - g_K) - sum_{r >= 1} (1 - g_r) w_r) / (1 + eps)
  f2 W[H];
  W[0] = make_float2(0.0f, 0.0f);
#pragma unroll
  for (int j = K - 1; j >= 1; --j) {
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
  W[0].x = w0_pk<K>(P, W, 1.0f - P[pk(H, 0)].x) * kp.inv_diag;
#pragma unroll
  for (int rp = 0; rp < H; ++rp) { w[2 * rp] = W[rp].x; w[2 * rp + 1] = W[rp].y; }
  return out;
}

}  // namespace gp
