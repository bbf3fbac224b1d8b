// Left-looking, just-in-time realisation of the packed fp32 conditioning (Eq. 2; Alg. 1 lines 4-6,
// PAPER.md:70-77) for sm_100a.  Same mathematics as gp_cond_pk.cuh (vertical register pairs, gamma form, neighbour 0
// eliminated analytically), organised around what the round-1 profiles and gp_measure_alu_peak showed:
//
//  * The FMA pipe is the bound, and what it delivers is set by REGISTER OPERAND WORDS, about two 32-bit words per
//    lane per cycle: a packed fma with three register-pair operands takes 3.0 cycles, with a broadcast scalar or a
//    uniform-register operand 2.0-2.3, a scalar fma with an immediate 1.0.  So the K build — two thirds
//    of the packed instructions — is written to read few words: minimax coefficients live in uniform registers,
//    -(1 + eps) is folded into them, and the analytic first elimination step enters as the addend of the last
//    Horner-type fma (S'_rc = base_rc + q p(t)) instead of a separate pass over the triangle.
//  * gamma(a) = 1 - rho(a) for small a is a degree-4 minimax polynomial (relative error 1.4e-7 on a <= 0.5, where the
//    Taylor series of round 1 needed 7 terms).  A second, polynomial-only body for warps whose 32 neighbourhoods all
//    lie below a = 1 (with the builder ordering each batch by neighbourhood radius so that such warps are the rule)
//    was built and measured: alone it runs the inverse in 1.9 ms against 2.65 ms, but a kernel holding both bodies
//    ran at 2.5 ms for a 60 % share of small warps (ptxas re-loads the uniform-register constants, the two bodies
//    do not fit the 32 KB instruction cache together, the radius order halves the L1 hit rate of the gathers), and
//    BASELINE's other configurations have almost no such warps: dropped.
//  * LEFT-LOOKING order: column c of S' is built when the factorisation reaches it, then receives the updates of
//    columns 1..c-1 and is scaled.  Rows < c of the earlier columns are dead by then, so the live triangle peaks at
//    about 40 register pairs instead of 89, the coordinates of row c die after column c, and nothing spills
//    ("registers only"; the right-looking form of round 1 kept 84 bytes per thread in local memory).
//
// Row K is the point itself and row K + 1 the carried values row: the last pair of every column.
#pragma once
#include "gp_cond_pk.cuh"

namespace gp {

// Host-prepared constants of the gamma evaluation, all in uniform registers.  With z = q (Matern-3/2, SE) or
// t = sqrt(q) (exponential) and the polynomial variable x = t (Matern-3/2, exponential) or q (SE):
//   -(1 + eps) gamma = z (c0 + c1 x + ... + c4 x^4)      where x < thr (a < 0.5), else -(1 + eps)(1 - rho)
struct JitParams {
  float c0, c1, c2, c3, c4;       // degree-4 minimax coefficients times -(1 + eps)
  float thr;                      // threshold in the polynomial variable
  float ope, neg_ope;             // 1 + eps, -(1 + eps)
  float neg_inv_ope;              // -1 / (1 + eps): turns the scaled value back into gamma
};

inline JitParams make_jit_params(const gp_kernel& k) {
  // degree-4 minimax fits on a <= 0.5 (Lawson iteration on Chebyshev nodes, RELATIVE error of gamma, checked in the
  // fp32 Horner form too):   Matern-3/2:  gamma / t^2, gamma = 1 - (1 + a) e^-a, a = t ln 2:  1.4e-7 (fp32: 2.4e-7)
  //                          exp, SE:     gamma / x,   gamma = 1 - e^-a,         a = x ln 2:  7.7e-8 (fp32: 1.6e-7)
  // (the 7-term Taylor series of round 1 had 3.4e-7 at the same threshold)
  static const double m32_c[5] = {0.24022647391618276, -0.11100602753190689, 0.028830641441173678,
                                  -0.0052416320720599019, 0.00062144729987298388};
  static const double ex_c[5] = {0.69314712699668024, -0.24022290282841074, 0.055464640197308061,
                                 -0.0094645342465443268, 0.0010833843510131165};
  const double* c = k.kind == GP_KERNEL_MATERN32 ? m32_c : ex_c;
  const double ope = 1.0 + k.jitter, ln2 = 0.69314718055994530942;
  JitParams p;
  p.c0 = (float)(-ope * c[0]); p.c1 = (float)(-ope * c[1]); p.c2 = (float)(-ope * c[2]);
  p.c3 = (float)(-ope * c[3]); p.c4 = (float)(-ope * c[4]);
  p.thr = (float)(0.5 / ln2);
  p.ope = (float)ope; p.neg_ope = (float)(-ope); p.neg_inv_ope = (float)(-1.0 / ope);
  return p;
}

__device__ __forceinline__ f2 sqrt2_approx(f2 q) {
  return make_float2(Math<float>::sqrt_approx(q.x), Math<float>::sqrt_approx(q.y));
}
__device__ __forceinline__ f2 ex2_neg2(f2 t) { return make_float2(Math<float>::ex2(-t.x), Math<float>::ex2(-t.y)); }

// base + (-(1 + eps)) gamma(q) for a pair of q's.
template <int KIND>
__device__ __forceinline__ f2 scaled_neg_gamma2(f2 q, const JitParams& jp, f2 base) {
  f2 x, z;   // polynomial variable, outer factor
  if (KIND == GP_KERNEL_SE) { x = q; z = q; }
  else { x = sqrt2_approx(q); z = KIND == GP_KERNEL_MATERN32 ? q : x; }
  f2 p = fma2(x, bc(jp.c4), bc(jp.c3));
  p = fma2(x, p, bc(jp.c2));
  p = fma2(x, p, bc(jp.c1));
  p = fma2(x, p, bc(jp.c0));
  // above the threshold gamma is no longer small: 1 - rho with rho from MUFU.EX2 is accurate enough there.  The two
  // forms are blended arithmetically (w = 1 where the polynomial applies: FSET on the ALU pipe): selects on the
  // halves of a register pair cost moves, measured 2.95 ms against 2.56 ms for the whole inverse kernel.
  const f2 e = ex2_neg2(x);
  f2 rho = e;
  if (KIND == GP_KERNEL_MATERN32) rho = mul2(fma2(x, bc(0.69314718055994530942f), bc(1.0f)), e);
  const f2 big = fma2(rho, bc(jp.ope), bc(jp.neg_ope));          // -(1 + eps)(1 - rho)
  const f2 small = mul2(z, p);
  return fma2(below2(x, jp.thr), add2(small, neg2(big)), add2(big, base));
}

// q(self, c) for two columns per packed evaluation: the centred coordinates ARE the differences.
template <int K, int D>
__device__ __forceinline__ void self_q_jit(const PkCoords<K>& X, f2 (&qS)[K / 2], float& qmax) {
  qmax = 0.0f;
#pragma unroll
  for (int cp = 0; cp < K / 2; ++cp) {
    f2 q = mul2(X.x0[cp], X.x0[cp]);
    if (D >= 2) q = fma2(X.x1[cp], X.x1[cp], q);
    if (D >= 3) q = fma2(X.x2[cp], X.x2[cp], q);
    qS[cp] = q;
    qmax = fmaxf(qmax, fmaxf(q.x, q.y));
  }
}

template <int K, int D>
__device__ __forceinline__ f2 pair_q_jit(const PkCoords<K>& X, int rp, float c0, float c1, float c2) {
  f2 dx = add2(X.x0[rp], bc(-c0));
  f2 q = mul2(dx, dx);
  if (D >= 2) { f2 dy = add2(X.x1[rp], bc(-c1)); q = fma2(dy, dy, q); }
  if (D >= 3) { f2 dz = add2(X.x2[rp], bc(-c2)); q = fma2(dz, dz, q); }
  return q;
}

// Build, eliminate neighbour 0, factor: returns m = K_ic K_cc^-1 v_c and s (unit sigma).  X: centred, scaled
// coordinates in vertical pairs; V: neighbour values; qS: q(self, c) from self_q_jit.
template <int K, int D, int KIND>
__device__ __forceinline__ Cond<float> condition_jit(const PkCoords<K>& X, const float (&V)[K], const f2 (&qS)[K / 2],
                                                     const KParams<float>& kp, const JitParams& jp) {
  constexpr int H = K / 2;
  const f2 zero2 = make_float2(0.0f, 0.0f);
  // gammas of the point itself (row K) and of column 0 (neighbour 0): the analytic elimination needs them raw
  float gS[K];
#pragma unroll
  for (int cp = 0; cp < H; ++cp) {
    const f2 g = mul2(scaled_neg_gamma2<KIND>(qS[cp], jp, zero2), bc(jp.neg_inv_ope));
    gS[2 * cp] = g.x;
    gS[2 * cp + 1] = g.y;
  }
  f2 G[H];
  {
    const float c0 = X.x0[0].x, c1 = D >= 2 ? X.x1[0].x : 0.0f, c2 = D >= 3 ? X.x2[0].x : 0.0f;
#pragma unroll
    for (int rp = 0; rp < H; ++rp)
      G[rp] = mul2(scaled_neg_gamma2<KIND>(pair_q_jit<K, D>(X, rp, c0, c1, c2), jp, zero2), bc(jp.neg_inv_ope));
    G[0].x = 0.0f;
  }
  const float eps = kp.eps, ope = kp.diag, inv_ope = kp.inv_diag;
  const float gK = gS[0], v0 = V[0], v0s = v0 * inv_ope;

  f2 P[pk_pairs(K)];
  float minpiv = ope;
#pragma unroll
  for (int c = 1; c < K; ++c) {
    const int cp = c / 2, odd = c & 1;
    const float gc = half_of(G[cp], odd);
    const float a = 1.0f - gc, b = eps + gc;
    // ---- column c of S' = (1 + eps) x (Schur complement of neighbour 0), rows > c
    {
      const float c0 = half_of(X.x0[cp], odd);
      const float c1 = D >= 2 ? half_of(X.x1[cp], odd) : 0.0f;
      const float c2 = D >= 3 ? half_of(X.x2[cp], odd) : 0.0f;
#pragma unroll
      for (int rp = odd ? cp + 1 : cp; rp < H; ++rp) {
        const f2 base = fma2(G[rp], bc(a), bc(b));                 // eps + g_r + g_c - g_r g_c
        P[pk(rp, c)] = scaled_neg_gamma2<KIND>(pair_q_jit<K, D>(X, rp, c0, c1, c2), jp, base);
      }
    }
    const float dg = b * (ope + a);                                 // S'_cc = (eps + g_c)(2 + eps - g_c)
    if (!odd) P[pk(cp, c)].x = dg;
    else P[pk(cp, c)] = make_float2(0.0f, dg);                      // .x lies above the diagonal: never read
    P[pk(H, c)] = make_float2(fmaf(jp.neg_ope, gS[c], fmaf(gK, a, b)),   // S'_Kc
                              fmaf(v0s, b, V[c] - v0));                  // u_c = (v_c - v_0) + v_0 (g_c + eps)/(1 + eps)
    // ---- left-looking update with columns 1 .. c-1, then the pivot
#pragma unroll
    for (int j = 1; j < c; ++j) {
      const float l = half_of(P[pk(cp, j)], odd);
#pragma unroll
      for (int rp = cp; rp <= H; ++rp) P[pk(rp, c)] = fma2(neg2(P[pk(rp, j)]), bc(l), P[pk(rp, c)]);
    }
    const float piv = half_of(P[pk(cp, c)], odd);
    minpiv = fminf(minpiv, piv);
    const float inv = Math<float>::rsqrt(piv);
#pragma unroll
    for (int rp = cp; rp <= H; ++rp) P[pk(rp, c)] = mul2(P[pk(rp, c)], bc(inv));
  }
  // ---- column K: ((1 + eps) s^2, -m), two partial sums to halve the dependent chain
  const float aK = 1.0f - gK;
  f2 acc0 = make_float2((eps + gK) * (ope + aK), -v0s * aK), acc1 = zero2;
#pragma unroll
  for (int j = 1; j < K; ++j) {
    if (j & 1) acc0 = fma2(neg2(P[pk(H, j)]), bc(P[pk(H, j)].x), acc0);
    else acc1 = fma2(neg2(P[pk(H, j)]), bc(P[pk(H, j)].x), acc1);
  }
  const f2 last = add2(acc0, acc1);
  minpiv = fminf(minpiv, last.x);
  Cond<float> out;
  out.ok = (minpiv > 0.0f) && (last.x < 3.0e38f);
  out.m = -last.y;
  out.s = Math<float>::sqrt(last.x * inv_ope);
  return out;
}

// Gathered records -> conditioning.
template <int K, int D, int KIND>
__device__ __forceinline__ Cond<float> condition_jit_rec(const Rec<float> (&R)[K], const Rec<float>& self,
                                                         const KParams<float>& kp, const JitParams& jp) {
  PkCoords<K> X;
  centre_pk<K, D>(R, self, kp.sq, X);
  float V[K];
#pragma unroll
  for (int j = 0; j < K; ++j) V[j] = R[j].v;
  f2 qS[K / 2];
  float qmax;
  self_q_jit<K, D>(X, qS, qmax);
  return condition_jit<K, D, KIND>(X, V, qS, kp, jp);
}

}  // namespace gp
