// Packed-fp32 building blocks of the gradient kernels (formulas: header of gp_vjp.cu).
// Same vertical-pair layout as gp_cond_pk.cuh.  The pair derivatives D_rc = ell d rho / d ell (r_rc) are
// evaluated in the same pass as rho (they share the MUFU results) and parked in shared memory, one column
// per thread, because the factorisation overwrites the triangle in place and the coordinates are dead by
// the time the weights u = (-w, 1) and alpha exist.
#pragma once
#include "gp_cond_pk.cuh"

namespace gp {

// number of full row-pairs in columns < c, and the slot of (rp, c), rp in c/2 + 1 .. K/2 - 1
__host__ __device__ constexpr int dq_full_before(int K, int c) {
  int s = 0;
  for (int q = 0; q < c; ++q) s += K / 2 - 1 - q / 2;
  return s;
}
__host__ __device__ constexpr int dq_full_total(int K) { return dq_full_before(K, K); }
__host__ __device__ constexpr int dq_slot(int K, int rp, int c) { return dq_full_before(K, c) + rp - (c / 2 + 1); }
// scalar slots: [0, K/2) entry (c + 1, c) for even c; [K/2, K/2 + K) entry (self, c)
__host__ __device__ constexpr int dq_scalar_total(int K) { return K / 2 + K; }
__host__ __device__ constexpr size_t dq_smem_bytes(int K, int threads) {
  return (size_t)threads * (dq_full_total(K) * sizeof(float2) + dq_scalar_total(K) * sizeof(float));
}

template <int K> struct DqStore {
  float2* p2;   // [dq_full_total][threads], this thread's column
  float* p1;    // [dq_scalar_total][threads]
  int stride;
  __device__ __forceinline__ float2& full(int slot) const { return p2[(size_t)slot * stride]; }
  __device__ __forceinline__ float& scalar(int slot) const { return p1[(size_t)slot * stride]; }
};

// gamma = 1 - rho and D = ell d rho / d ell for a pair of q's; the MUFU results are shared.  gamma for small arguments
// is the degree-4 minimax polynomial of gp_cond_jit.cuh (same coefficients, same threshold a = 0.5; relative error
// 1.4e-7 / 7.7e-8) instead of the 7-term Taylor series of gamma2_from_q: four packed instructions fewer per pair of pairs.
template <int KIND> __device__ __forceinline__ void gamma_drho2(f2 q, f2& gam, f2& dr) {
  const float ln2 = 0.69314718055994530942f;
  constexpr float thr = (float)(0.5 / 0.69314718055994530942);
  f2 x, z;   // polynomial variable, outer factor: gamma = z p(x) below the threshold
  if (KIND == GP_KERNEL_SE) { x = q; z = q; }
  else {
    x = make_float2(Math<float>::sqrt_approx(q.x), Math<float>::sqrt_approx(q.y));
    z = KIND == GP_KERNEL_MATERN32 ? q : x;
  }
  f2 p;
  if (KIND == GP_KERNEL_MATERN32) {
    p = fma2(x, bc(0.00062144729987298388f), bc(-0.0052416320720599019f));
    p = fma2(x, p, bc(0.028830641441173678f));
    p = fma2(x, p, bc(-0.11100602753190689f));
    p = fma2(x, p, bc(0.24022647391618276f));
  } else {
    p = fma2(x, bc(0.0010833843510131165f), bc(-0.0094645342465443268f));
    p = fma2(x, p, bc(0.055464640197308061f));
    p = fma2(x, p, bc(-0.24022290282841074f));
    p = fma2(x, p, bc(0.69314712699668024f));
  }
  const f2 e = make_float2(Math<float>::ex2(-x.x), Math<float>::ex2(-x.y));
  const f2 a = mul2(x, bc(ln2));                       // SE: r^2 / (2 ell^2); else sqrt(3) r / ell or r / ell
  f2 rho = e;
  if (KIND == GP_KERNEL_MATERN32) rho = mul2(add2(a, bc(1.0f)), e);
  gam = blend2(below2(x, thr), mul2(z, p), add2(bc(1.0f), neg2(rho)));
  if (KIND == GP_KERNEL_SE) dr = mul2(mul2(a, bc(2.0f)), e);
  else if (KIND == GP_KERNEL_MATERN32) dr = mul2(mul2(a, a), e);
  else dr = mul2(a, e);
}
template <int KIND> __device__ __forceinline__ void gamma_drho1(float q, float& gam, float& dr) {
  f2 g2, d2;
  gamma_drho2<KIND>(make_float2(q, q), g2, d2);   // the compiler drops the duplicate half
  gam = g2.x;
  dr = d2.x;
}

// build_joint_pk + derivative store
template <int K, int D, int KIND>
__device__ __forceinline__ void build_joint_grad_pk(const PkCoords<K>& X, const float (&vals)[K], const KParams<float>& kp,
                                                    f2 (&P)[pk_pairs(K)], const DqStore<K>& dq) {
  constexpr int H = K / 2;
#pragma unroll
  for (int c = 0; c < K; ++c) {
    const int cp = c / 2, odd = c & 1;
    const float c0 = half_of(X.x0[cp], odd);
    const float c1 = D >= 2 ? half_of(X.x1[cp], odd) : 0.0f;
    const float c2 = D >= 3 ? half_of(X.x2[cp], odd) : 0.0f;
    if (!odd) {
      float dx = X.x0[cp].y - c0;
      float q = dx * dx;
      if (D >= 2) { float dy = X.x1[cp].y - c1; q = fmaf(dy, dy, q); }
      if (D >= 3) { float dz = X.x2[cp].y - c2; q = fmaf(dz, dz, q); }
      float r, d;
      gamma_drho1<KIND>(q, r, d);
      P[pk(cp, c)] = make_float2(0.0f, r);
      dq.scalar(cp) = d;
    } else {
      P[pk(cp, c)] = make_float2(0.0f, 0.0f);
    }
#pragma unroll
    for (int rp = cp + 1; rp < H; ++rp) {
      f2 dx = add2(X.x0[rp], bc(-c0));
      f2 q = mul2(dx, dx);
      if (D >= 2) { f2 dy = add2(X.x1[rp], bc(-c1)); q = fma2(dy, dy, q); }
      if (D >= 3) { f2 dz = add2(X.x2[rp], bc(-c2)); q = fma2(dz, dz, q); }
      f2 r, d;
      gamma_drho2<KIND>(q, r, d);
      P[pk(rp, c)] = r;
      dq.full(dq_slot(K, rp, c)) = d;
    }
    float qs = c0 * c0;
    if (D >= 2) qs = fmaf(c1, c1, qs);
    if (D >= 3) qs = fmaf(c2, c2, qs);
    float r, d;
    gamma_drho1<KIND>(qs, r, d);
    P[pk(H, c)] = make_float2(r, vals[c]);
    dq.scalar(H + c) = d;
  }
  P[pk(H, K)] = make_float2(0.0f, 0.0f);
}

// After eliminate0_pk and factor_joint_pk<K, true>:  W[rp] = (w[2rp], w[2rp+1]) with w = M_cc^-1 M_ci, AL likewise
// with alpha = M_cc^-1 v_c.  Rows >= 1 come from the back-substitution on S' = (1 + eps) S (w is scale free; the
// carried values were not scaled, so alpha picks up the factor 1 + eps), row 0 from the eliminated equation.
template <int K>
__device__ __forceinline__ void backsub2_pk(const f2 (&P)[pk_pairs(K)], const KParams<float>& kp, f2 (&W)[K / 2],
                                            f2 (&AL)[K / 2]) {
  constexpr int H = K / 2;
  W[0] = make_float2(0.0f, 0.0f);
  AL[0] = make_float2(0.0f, 0.0f);
#pragma unroll
  for (int j = K - 1; j >= 1; --j) {
    const int jp = j / 2, odd = j & 1;
    f2 accw = make_float2(0.0f, 0.0f), acca = make_float2(0.0f, 0.0f);
#pragma unroll
    for (int rp = jp + 1; rp < H; ++rp) {
      accw = fma2(P[pk(rp, j)], W[rp], accw);
      acca = fma2(P[pk(rp, j)], AL[rp], acca);
    }
    float tw = P[pk(H, j)].x - (accw.x + accw.y);
    float ta = P[pk(H, j)].y - (acca.x + acca.y);
    if (!odd) {
      tw = fmaf(-P[pk(jp, j)].y, W[jp].y, tw);
      ta = fmaf(-P[pk(jp, j)].y, AL[jp].y, ta);
    }
    const float inv = half_of(P[pk(jp, j)], odd);
    if (odd) { W[jp].y = tw * inv; AL[jp].y = ta * inv; }
    else { W[jp].x = tw * inv; AL[jp].x = ta * inv; }
  }
#pragma unroll
  for (int rp = 0; rp < H; ++rp) AL[rp] = mul2(AL[rp], bc(kp.diag));
  W[0].x = w0_pk<K>(P, W, 1.0f - P[pk(H, 0)].x) * kp.inv_diag;
  AL[0].x = w0_pk<K>(P, AL, P[pk(H, 0)].y) * kp.inv_diag;
}

// sum_{r > c} D_rc [ u_r (alpha'_c + two_coef u_c) + alpha'_r u_c ]   with u = (-w, 1), alpha' = (alpha, 0).
//   VJP:     two_coef = sigma xi_i / s   ->  y[0:k].alpha + (sigma xi_i / 2 s) (y.u)
//   logdet:  AL = 0, two_coef = 1        ->  y.u / 2 ... so the caller doubles it
template <int K>
__device__ __forceinline__ float grad_sweep_pk(const f2 (&W)[K / 2], const f2 (&AL)[K / 2], float two_coef,
                                               const DqStore<K>& dq) {
  constexpr int H = K / 2;
  f2 acc = make_float2(0.0f, 0.0f);
  float accs = 0.0f;
#pragma unroll
  for (int c = 0; c < K; ++c) {
    const int cp = c / 2, odd = c & 1;
    const float uc = -half_of(W[cp], odd);
    const float bcoef = fmaf(two_coef, uc, half_of(AL[cp], odd));
    if (!odd) {   // entry (c + 1, c)
      float t = fmaf(-W[cp].y, bcoef, AL[cp].y * uc);
      accs = fmaf(dq.scalar(cp), t, accs);
    }
#pragma unroll
    for (int rp = cp + 1; rp < H; ++rp) {
      f2 t = fma2(neg2(W[rp]), bc(bcoef), mul2(AL[rp], bc(uc)));
      acc = fma2(dq.full(dq_slot(K, rp, c)), t, acc);
    }
    accs = fmaf(dq.scalar(H + c), bcoef, accs);   // entry (self, c): u = 1, alpha' = 0
  }
  return accs + (acc.x + acc.y);
}

}  // namespace gp
