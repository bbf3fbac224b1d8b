// Lane-group conditioning: one point split over L consecutive lanes of a warp (PAPER.md:53 says the register
// budget (k+1)[d+1+(k+2)/2] limits one thread to k <~ 64 on the paper's GPU; on sm_100a one thread per point
// stops paying at k = 16 in fp32 and k = 8 in fp64: 255 registers).  Used for k = 32 fp32 and k = 16 fp64.
//
// The K neighbour rows of the joint matrix are dealt cyclically to the lanes: row r lives in lane
// r % L, slot r / L (K is a multiple of L), so every register index below is a compile-time constant and nothing
// spills.  A right-looking step j needs L[c][j] for all c > j in every lane: one width-L shuffle per (j, c) from the
// lane that owns row c.  Entries above the diagonal inside a slot are computed as harmless finite junk and never read.
// The two remaining rows - row K, the point itself, and the carried values row K + 1 - are stored
// BY COLUMN: their column-c entries live in the lane that owns neighbour row c (lane c % L, slot c / L).  That lane
// already holds everything their build needs (the coordinates and the value of neighbour c) and, in step j, the factor
// L[c][j] their update needs, so the two rows cost one kernel evaluation per neighbour and two shuffles per step,
// where a fifth, nearly empty slot (2 of L lanes busy) cost a full slot of evaluations and updates per column
// (config 4: 112 -> 84 kernel evaluations per lane).  Their column-K entries ((1 + eps) s^2 and -m at the end) are
// scalars every lane carries.
#pragma once
#include <type_traits>

#include "gp_cond_pk.cuh"

namespace gp {

template <typename T> __device__ __forceinline__ T shfl_grp(T v, int src, int width) {
  return __shfl_sync(0xffffffffu, v, src, width);
}

template <typename T, int K, int L> struct LgShape {
  static_assert(K % L == 0, "lane-group kernels need K to be a multiple of the group width");
  static constexpr int S = K / L;
};

// Result in every lane of the group: m, s (unit sigma), ok, and the point's own value.
template <typename T> struct LgCond { T m, s, self_v; bool ok; };

// What lg_factor leaves besides the factor: rows K and K + 1 by column (sK[s], sV[s]: column s L + l; with KEEP_ROWS
// the final L[K][c], else partly updated values), their column-K entries dKK, dVK, and gK = gamma(point, neighbour 0).
template <typename T, int S> struct LgTail { T sK[S], sV[S], dKK, dVK, gK, self_v; };

// One right-looking step (column J) of the factorisation, as a template recursion: the loop over J with this body is
// too large for the compiler to unroll fully, and a step whose J is not a compile-time constant puts `a` into
// local memory.
template <typename T, int K, int L, bool KEEP_INV, int J>
__device__ __forceinline__ void lg_step(T (&a)[LgShape<T, K, L>::S][K], LgTail<T, LgShape<T, K, L>::S>& t, int l, T& minpiv) {
  if constexpr (J < K) {
    constexpr int S = LgShape<T, K, L>::S;
    constexpr int js = J / L, jo = J % L;
    const T piv = shfl_grp(a[js][J], jo, L);
    minpiv = Math<T>::fmin(minpiv, piv);
    const T inv = Math<T>::rsqrt(piv);
#pragma unroll
    for (int s = js; s < S; ++s) a[s][J] *= inv;
    if (KEEP_INV) a[js][J] = (l == jo) ? inv : a[js][J];
    // L[K][J], L[K + 1][J]: from the lane that owns column J; kept there in final form
    const T lKj = shfl_grp(t.sK[js], jo, L) * inv;
    const T lVj = shfl_grp(t.sV[js], jo, L) * inv;
    t.sK[js] = (l == jo) ? lKj : t.sK[js];
    t.dKK = Math<T>::fma(-lKj, lKj, t.dKK);
    t.dVK = Math<T>::fma(-lVj, lKj, t.dVK);
#pragma unroll
    for (int c = J + 1; c < K; ++c) {
      const T lc = shfl_grp(a[c / L][J], c % L, L);
#pragma unroll
      for (int s = c / L; s < S; ++s) a[s][c] = Math<T>::fma(-a[s][J], lc, a[s][c]);
    }
    // rows K, K + 1 at this lane's columns c = s L + l > J: the factor L[c][J] is a[s][J], already here
#pragma unroll
    for (int s = js; s < S; ++s) {
      const bool upd = (s > js) || (l > jo);
      const T nk = Math<T>::fma(-lKj, a[s][J], t.sK[s]);
      const T nv = Math<T>::fma(-lVj, a[s][J], t.sV[s]);
      t.sK[s] = upd ? nk : t.sK[s];
      t.sV[s] = upd ? nv : t.sV[s];
    }
    lg_step<T, K, L, KEEP_INV, J + 1>(a, t, l, minpiv);
  }
}

// Build and factor.  a: the factor (column j >= J0, rows > j), column 0 keeps the gammas in the gamma form; with
// KEEP_INV the diagonal slot of column j holds 1 / L_jj.  CARRY: the values row is carried (else zeros).
template <typename T, int K, int D, int KIND, int L, bool COHERENT, bool KEEP_INV, bool CARRY>
__device__ __forceinline__ void lg_factor(const Rec<T>* __restrict__ rec, const int32_t* __restrict__ row, int64_t i, int l,
                                          const KParams<T>& kp, T (&a)[LgShape<T, K, L>::S][K],
                                          LgTail<T, LgShape<T, K, L>::S>& t, T& minpiv) {
  constexpr int S = LgShape<T, K, L>::S;
  T X0[S], X1[S], X2[S], V[S];
#pragma unroll
  for (int s = 0; s < S; ++s) {
    const Rec<T> R = load_rec<COHERENT>(rec + row[s * L + l]);
    X0[s] = R.x0; X1[s] = R.x1; X2[s] = R.x2; V[s] = CARRY ? R.v : T(0);
  }
  const Rec<T> self = load_rec<COHERENT>(rec + i);          // every lane of the group: one address, one transaction
  t.self_v = self.v;
  // fp32 works in the gamma form of gp_cond_pk.cuh: gammas instead of rho, neighbour 0 eliminated analytically
  // (S' = (1 + eps) x Schur complement), factorisation from column 1.  fp64 keeps the plain form.
  constexpr bool GAMMA = std::is_same<T, float>::value;
  constexpr int J0 = GAMMA ? 1 : 0;
  T kS[S];                                                   // kernel between the point itself and this lane's rows
#pragma unroll
  for (int s = 0; s < S; ++s) {
    T dx = X0[s] - self.x0;
    T d2 = dx * dx;
    if (D >= 2) { T dy = X1[s] - self.x1; d2 = Math<T>::fma(dy, dy, d2); }
    if (D >= 3) { T dz = X2[s] - self.x2; d2 = Math<T>::fma(dz, dz, d2); }
    if constexpr (GAMMA) kS[s] = gamma_from_q<KIND>(d2 * kp.qscale);
    else kS[s] = Math<T>::template rho_from_q<KIND>(d2 * kp.qscale);
  }
  const T v0 = shfl_grp(V[0], 0, L);
#pragma unroll
  for (int c = 0; c < K; ++c) {
    const int cs = c / L, co = c % L;
    const T c0 = shfl_grp(X0[cs], co, L);
    const T c1 = D >= 2 ? shfl_grp(X1[cs], co, L) : T(0);
    const T c2 = D >= 3 ? shfl_grp(X2[cs], co, L) : T(0);
    T gc = T(0);
    if (GAMMA && c >= 1) gc = shfl_grp(a[cs][0], co, L);        // gamma_c0 from the lane that owns row c
#pragma unroll
    for (int s = cs; s < S; ++s) {
      const int r = s * L + l;
      T dx = X0[s] - c0;
      T d2 = dx * dx;
      if (D >= 2) { T dy = X1[s] - c1; d2 = Math<T>::fma(dy, dy, d2); }
      if (D >= 3) { T dz = X2[s] - c2; d2 = Math<T>::fma(dz, dz, d2); }
      // rows of a slot s > cs are all below row c: only slot cs needs the r > c / r == c selects (s and cs are
      // compile-time after unrolling)
      T val;
      if constexpr (GAMMA) {
        const float gam = gamma_from_q<KIND>(d2 * kp.qscale);
        if (c == 0) {
          val = gam;                                             // column 0 keeps the gammas g_r
        } else {
          const float gr = a[s][0];
          const float b = kp.eps + gc;
          val = fmaf(-kp.diag, gam, fmaf(gr, 1.0f - gc, b));                          // S'_rc
          if (s == cs) val = r > c ? val : (r == c ? b * (kp.diag + (1.0f - gc)) : 0.0f);   // S'_cc, above: 0
        }
      } else {
        val = Math<T>::template rho_from_q<KIND>(d2 * kp.qscale);
        if (s == cs) val = r > c ? val : (r == c ? kp.diag : T(0));
      }
      a[s][c] = val;
    }
  }
  // rows K and K + 1, column s L + l in this lane
  if constexpr (GAMMA) {
    const float gK = shfl_grp(kS[0], 0, L);                      // gamma(point, neighbour 0)
    t.gK = gK;
#pragma unroll
    for (int s = 0; s < S; ++s) {
      const float gcl = a[s][0];                                 // g_c of this lane's column (column 0 itself: unused)
      const float b = kp.eps + gcl;
      t.sK[s] = fmaf(-kp.diag, kS[s], fmaf(gK, 1.0f - gcl, b));  // S'_Kc
      t.sV[s] = fmaf(v0 * kp.inv_diag, b, V[s] - v0);            // u_c = (v_c - v_0) + v_0 (g_c + eps) / (1 + eps)
    }
    t.dKK = (kp.eps + gK) * (kp.diag + (1.0f - gK));
    t.dVK = -v0 * (1.0f - gK) * kp.inv_diag;
  } else {
    t.gK = T(0);
#pragma unroll
    for (int s = 0; s < S; ++s) { t.sK[s] = kS[s]; t.sV[s] = V[s]; }
    t.dKK = kp.diag;
    t.dVK = T(0);
  }

  minpiv = kp.diag;
  lg_step<T, K, L, KEEP_INV, J0>(a, t, l, minpiv);
}

template <typename T, int K, int D, int KIND, int L, bool COHERENT>
__device__ __forceinline__ LgCond<T> condition_lg(const Rec<T>* __restrict__ rec, const int32_t* __restrict__ row,
                                                  int64_t i, int l, const KParams<T>& kp) {
  constexpr int S = LgShape<T, K, L>::S;
  constexpr bool GAMMA = std::is_same<T, float>::value;
  T a[S][K], minpiv;                      // a[s][c], c <= s L + L - 1: every index is a compile-time constant
  LgTail<T, S> t;
  lg_factor<T, K, D, KIND, L, COHERENT, false, true>(rec, row, i, l, kp, a, t, minpiv);
  LgCond<T> out;
  const T s2 = t.dKK * (GAMMA ? kp.inv_diag : T(1));
  out.self_v = t.self_v;
  minpiv = Math<T>::fmin(minpiv, s2);
  out.ok = (minpiv > T(0)) && (s2 == s2) && (s2 < T(3.0e38));
  out.m = -t.dVK;
  out.s = Math<T>::sqrt(s2);
  return out;
}

// v-independent half for the dataflow forward: every lane ends with the weights of ITS rows (w[s] for row s L + l),
// s and ok.  Back-substitution  w_j = (l_j - sum_{r > j} L[r][j] w_r) / L_jj : every lane sums over
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
  T a[S][K], minpiv;
  LgTail<T, S> t;
  lg_factor<T, K, D, KIND, L, COHERENT, true, false>(rec, row, i, l, kp, a, t, minpiv);
  const T s2 = t.dKK * (GAMMA ? kp.inv_diag : T(1));
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
      // rows of slots > js are all below row j; in slot js only rows > j count
      const T wr = (s == js) ? ((l > jo) ? w[s] : T(0)) : w[s];
      p = Math<T>::fma(a[s][j], wr, p);
    }
    p = group_sum(p, L);
    const T lj = shfl_grp(t.sK[js], jo, L);                  // L[K][j], final since step j
    const T invj = shfl_grp(a[js][j], jo, L);
    const T wj = (lj - p) * invj;
    w[js] = (l == jo) ? wj : w[js];
  }
  if (GAMMA) {   // row 0 of the eliminated system:  w_0 = ((1 - g_K) - sum_{r >= 1} (1 - g_r) w_r) / (1 + eps)
    T p = T(0);
#pragma unroll
    for (int s = 0; s < S; ++s) {
      const int r = s * L + l;
      p = Math<T>::fma(T(1) - a[s][0], r >= 1 ? w[s] : T(0), p);
    }
    p = group_sum(p, L);
    const T w0 = ((T(1) - t.gK) - p) * kp.inv_diag;
    w[0] = (l == 0) ? w0 : w[0];
  }
}

}  // namespace gp
