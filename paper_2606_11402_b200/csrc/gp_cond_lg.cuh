// Lane-group conditioning: one point split over L consecutive lanes of a warp (PAPER.md:53 says the register
// budget (k+1)[d+1+(k+2)/2] limits one thread to k <~ 64 on the paper's GPU; on sm_100a one thread per point
// stops paying at k = 16 in fp32 and k = 8 in fp64: 255 registers).  Used for k = 32 fp32 and k = 16 fp64.
//
// Rows of the joint matrix plus the carried values row - K + 2 rows, row K
// the point itself, row K + 1 the values - are dealt cyclically to the lanes: row r lives in lane r % L, slot
// r / L, so every register index below is a compile-time constant and nothing spills.  A right-looking step j
// needs L[c][j] for all c > j in every lane: one width-L shuffle per (j, c) from the lane that owns row c.
// Entries above the diagonal inside a slot are computed as harmless finite junk and never read.
#pragma once
#include <type_traits>

#include "gp_cond_pk.cuh"

namespace gp {

template <typename T> __device__ __forceinline__ T shfl_grp(T v, int src, int width) {
  return __shfl_sync(0xffffffffu, v, src, width);
}

template <typename T, int K, int L> struct LgShape {
  static constexpr int ROWS = K + 2;
  static constexpr int S = (ROWS + L - 1) / L;
  // columns a slot needs: rows of slot s reach s L + L - 1, capped at K
  __host__ __device__ static constexpr int cols(int s) { return (s * L + L - 1 < K ? s * L + L - 1 : K) + 1; }
};

// Result in every lane of the group: m, s (unit sigma), ok, and the point's own value.
template <typename T> struct LgCond { T m, s, self_v; bool ok; };

// Build and factor.  a: the factor (column j >= J0, rows > j), column 0 keeps the gammas in the gamma form; with
// KEEP_INV the diagonal slot of column j holds 1 / L_jj.  CARRY: the values row is carried (else zeros).
template <typename T, int K, int D, int KIND, int L, bool COHERENT, bool KEEP_INV, bool CARRY>
__device__ __forceinline__ void lg_factor(const Rec<T>* __restrict__ rec, const int32_t* __restrict__ row, int64_t i, int l,
                                          const KParams<T>& kp, T (&a)[LgShape<T, K, L>::S][K + 1],
                                          T (&V)[LgShape<T, K, L>::S], T& minpiv) {
  using Sh = LgShape<T, K, L>;
  constexpr int S = Sh::S;
  T X0[S], X1[S], X2[S];
#pragma unroll
  for (int s = 0; s < S; ++s) {
    const int r = s * L + l;
    Rec<T> R;
    R.x0 = R.x1 = R.x2 = R.v = T(0);
    if (r < K) R = load_rec<COHERENT>(rec + row[r]);
    else if (r == K) R = load_rec<COHERENT>(rec + i);
    X0[s] = R.x0; X1[s] = R.x1; X2[s] = R.x2; V[s] = CARRY ? R.v : T(0);
  }
  // fp32 works in the gamma form of gp_cond_pk.cuh: gammas instead of rho, neighbour 0 eliminated analytically
  // (S' = (1 + eps) x Schur complement), factorisation from column 1.  fp64 keeps the plain form.
  constexpr bool GAMMA = std::is_same<T, float>::value;
  constexpr int J0 = GAMMA ? 1 : 0;
  const T v0 = shfl_grp(V[0], 0, L);
  T gK = T(0);
#pragma unroll
  for (int c = 0; c < K; ++c) {
    const int cs = c / L, co = c % L;
    const T c0 = shfl_grp(X0[cs], co, L);
    const T c1 = D >= 2 ? shfl_grp(X1[cs], co, L) : T(0);
    const T c2 = D >= 3 ? shfl_grp(X2[cs], co, L) : T(0);
    const T vc = shfl_grp(V[cs], co, L);
    T gc = T(0);
    if (GAMMA && c >= 1) gc = shfl_grp(a[cs][0], co, L);        // gamma_c0 from the lane that owns row c
    constexpr int SV = (K + 1) / L;   // the slot that holds the values row (in lane (K + 1) % L)
#pragma unroll
    for (int s = cs; s < S; ++s) {
      const int r = s * L + l;
      T dx = X0[s] - c0;
      T d2 = dx * dx;
      if (D >= 2) { T dy = X1[s] - c1; d2 = Math<T>::fma(dy, dy, d2); }
      if (D >= 3) { T dz = X2[s] - c2; d2 = Math<T>::fma(dz, dz, d2); }
      // rows of a slot s > cs are all below row c: only slot cs needs the r > c / r == c selects, only slot SV the
      // values-row select (s and cs are compile-time after unrolling)
      T val;
      if constexpr (GAMMA) {
        const float gam = gamma_from_q<KIND>(d2 * kp.qscale);
        if (c == 0) {
          val = gam;                                             // column 0 keeps the gammas g_r
        } else {
          const float gr = a[s][0];
          const float b = kp.eps + gc;
          val = fmaf(-kp.diag, gam, fmaf(gr, 1.0f - gc, b));                          // S'_rc
          if (s == SV) val = (r == K + 1) ? fmaf(v0 * kp.inv_diag, b, vc - v0) : val;  // u_c
          if (s == cs) val = r > c ? val : (r == c ? b * (kp.diag + (1.0f - gc)) : 0.0f);   // S'_cc, above: 0
        }
      } else {
        val = Math<T>::template rho_from_q<KIND>(d2 * kp.qscale);
        if (s == SV) val = (r == K + 1) ? vc : val;
        if (s == cs) val = r > c ? val : (r == c ? kp.diag : T(0));
      }
      a[s][c] = val;
    }
  }
  if constexpr (GAMMA) {
    gK = shfl_grp(a[K / L][0], K % L, L);
#pragma unroll
    for (int s = K / L; s < S; ++s) {
      const int r = s * L + l;
      T val = T(0);
      if (r == K) val = (kp.eps + gK) * (kp.diag + (1.0f - gK));
      else if (r == K + 1) val = -v0 * (1.0f - gK) * kp.inv_diag;
      a[s][K] = val;
    }
  } else {
#pragma unroll
    for (int s = K / L; s < S; ++s) a[s][K] = (s * L + l == K) ? kp.diag : T(0);
  }

  minpiv = kp.diag;
#pragma unroll
  for (int j = J0; j < K; ++j) {
    const int js = j / L, jo = j % L;
    const T piv = shfl_grp(a[js][j], jo, L);
    minpiv = Math<T>::fmin(minpiv, piv);
    const T inv = Math<T>::rsqrt(piv);
#pragma unroll
    for (int s = js; s < S; ++s) a[s][j] *= inv;
    if (KEEP_INV) a[js][j] = (l == jo) ? inv : a[js][j];
#pragma unroll
    for (int c = j + 1; c <= K; ++c) {
      const T lc = shfl_grp(a[c / L][j], c % L, L);
#pragma unroll
      for (int s = c / L; s < S; ++s) a[s][c] = Math<T>::fma(-a[s][j], lc, a[s][c]);
    }
  }
}

template <typename T, int K, int D, int KIND, int L, bool COHERENT>
__device__ __forceinline__ LgCond<T> condition_lg(const Rec<T>* __restrict__ rec, const int32_t* __restrict__ row,
                                                  int64_t i, int l, const KParams<T>& kp) {
  constexpr int S = LgShape<T, K, L>::S;
  constexpr bool GAMMA = std::is_same<T, float>::value;
  T a[S][K + 1], V[S], minpiv;            // a[s][c], c < cols(s): every index is a compile-time constant
  lg_factor<T, K, D, KIND, L, COHERENT, false, true>(rec, row, i, l, kp, a, V, minpiv);
  LgCond<T> out;
  const T s2 = shfl_grp(a[K / L][K], K % L, L) * (GAMMA ? kp.inv_diag : T(1));
  const T negm = shfl_grp(a[(K + 1) / L][K], (K + 1) % L, L);
  out.self_v = shfl_grp(V[K / L], K % L, L);
  minpiv = Math<T>::fmin(minpiv, s2);
  out.ok = (minpiv > T(0)) && (s2 == s2) && (s2 < T(3.0e38));
  out.m = -negm;
  out.s = Math<T>::sqrt(s2);
  return out;
}

// v-independent half for the dataflow forward: every lane ends with the weights of ITS rows (w[s] for row s L + l
// < K, else 0), s and ok.  Back-substitution  w_j = (l_j - sum_{r > j} L[r][j] w_r) / L_jj : every lane sums over
// its own rows, the group adds the partial sums with log2 L shuffles, the owner of row j keeps w_j.
template <typename T> __device__ __forceinline__ T group_sum(T p, int L) {
  for (int o = L >> 1; o > 0; o >>= 1) p += __shfl_xor_sync(0xffffffffu, p, o, L);
  return p;
}

template <typename T, int K, int D, int KIND, int L, bool COHERENT>
__device__ __forceinline__ void weights_lg(const Rec<T>* __restrict__ rec, const int32_t* __restrict__ row, int64_t i, int l,
                                           const KParams<T>& kp, T (&w)[LgShape<T, K, L>::S], T& s_out, bool& ok) {
  constexpr int S = LgShape<T, K, L>::S;
  constexpr bool GAMMA = std::is_same<T, float>::value;
  constexpr int J0 = GAMMA ? 1 : 0;
  T a[S][K + 1], V[S], minpiv;
  lg_factor<T, K, D, KIND, L, COHERENT, true, false>(rec, row, i, l, kp, a, V, minpiv);
  const T s2 = shfl_grp(a[K / L][K], K % L, L) * (GAMMA ? kp.inv_diag : T(1));
  minpiv = Math<T>::fmin(minpiv, s2);
  ok = (minpiv > T(0)) && (s2 == s2) && (s2 < T(3.0e38));
  s_out = Math<T>::sqrt(s2);
#pragma unroll
  for (int s = 0; s < S; ++s) w[s] = T(0);
#pragma unroll
  for (int j = K - 1; j >= J0; --j) {
    const int js = j / L, jo = j % L;
    T p = T(0);
#pragma unroll
    for (int s = js; s < S; ++s) {
      // rows of slots > js are all below row j; rows >= K have w = 0; in slot js only rows > j count
      const T wr = (s == js) ? ((s * L + l > j) ? w[s] : T(0)) : w[s];
      p = Math<T>::fma(a[s][j], wr, p);
    }
    p = group_sum(p, L);
    const T lj = shfl_grp(a[K / L][j], K % L, L);
    const T invj = shfl_grp(a[js][j], jo, L);
    const T wj = (lj - p) * invj;
    w[js] = (l == jo) ? wj : w[js];
  }
  if (GAMMA) {   // row 0 of the eliminated system:  w_0 = ((1 - g_K) - sum_{r >= 1} (1 - g_r) w_r) / (1 + eps)
    T p = T(0);
#pragma unroll
    for (int s = 0; s < S; ++s) {
      const int r = s * L + l;
      p = Math<T>::fma(T(1) - a[s][0], (r >= 1 && r < K) ? w[s] : T(0), p);
    }
    p = group_sum(p, L);
    const T gK = shfl_grp(a[K / L][0], K % L, L);
    const T w0 = ((T(1) - gK) - p) * kp.inv_diag;
    w[0] = (l == 0) ? w0 : w[0];
  }
}

}  // namespace gp
