// GraphGP oracle — TEST INFRASTRUCTURE ONLY.
//
// A plain, slow, obviously-correct CPU implementation of what the hot path of
// GraphGP's Vecchia approximation computes (arxiv/paper_2606_11402, PAPER.md).
// It exists to judge the CUDA path in paper_2606_11402_b200/; it shares no code,
// header, table or helper with that path and must never be called by it.  Only
// tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference
// legs may load this library.
//
// Everything is fp64 (a `long double` re-run of the conditioning is available for
// pin P-14).  No blocking, fusion or re-ordering beyond what the definitions state.
// Build: g++ -O2 -fopenmp -ffp-contract=off -shared -fPIC  (no FMA contraction, so
// the canonical squared distance below is reproducible bit for bit).
//
// Passages followed (PAPER.md line numbers):
//   Eq. 1   p(v) ~= prod_i p(v_i | v_c(i)),  c(i) subset of preceding points
//   Eq. 2   v_i | v_c ~ N(K_ic K_cc^-1 v_c, K_ii - K_ic K_cc^-1 K_ci)
//   PAPER.md:33               c(i) = k nearest among preceding points; all preceding => dense Cholesky
//   PAPER.md:39-41            bit-reversed left-balanced k-d tree order, children i+2^l and i+2^(l+1)
//   PAPER.md:43               depth d_i = 1 + max_{j in c(i)} d_j, depth-sorted batches, dense head of n0
//   PAPER.md:59               parallel depth fixed point
//   Alg. 1   forward pass
//   PAPER.md:57               kernel-parameter derivatives (here: closed forms of DESIGN.md §3 R-14)
//
// Pins (tests/test_oracle_*.py, all `-m "not gpu"`): dense-Cholesky equivalence against
// LAPACK (P-1), inverse∘forward = id (P-2), VJP vs central differences (P-3), brute-force
// neighbour invariants (P-4), k=1 closed form (P-5), sigma scaling (P-6), power-of-two scale
// invariance (P-7), 1-d Markov exponential closed form (P-8), logdet monotonicity (P-9),
// order worked examples and k-d invariants (P-11), depth sequential = parallel (P-12),
// long-double agreement (P-14), JVP and inverse-VJP against central differences and against the VJP by duality (P-15).  Nothing is "parity unpinned" except absolute fp32 values
// at N >= 2^24, which no formula in the paper fixes.
#include <algorithm>
#include <cmath>
#include <cstdint>
#include <cstring>
#include <numeric>
#include <vector>
#ifdef _OPENMP
#include <omp.h>
#endif

extern "C" {
typedef struct {
  int32_t kind;  // 0 squared-exponential, 1 Matern-3/2, 2 exponential
  double sigma, ell, jitter;  // K_ab = sigma^2 [ rho(r_ab) + jitter * delta_ab ]   (relative nugget)
} orc_kernel;
}

namespace {

// ---------------------------------------------------------------------------------------
// Canonical squared distance (R-5): double, per-coordinate difference, products
// summed left to right, round-to-nearest, no FMA.  Used for neighbour ranking AND as the
// r^2 that enters kappa.
// ---------------------------------------------------------------------------------------
inline double d2_canon(const double* a, const double* b, int d) {
  double dx = a[0] - b[0];
  double s = dx * dx;
  for (int j = 1; j < d; ++j) {
    dx = a[j] - b[j];
    double p = dx * dx;
    s = s + p;
  }
  return s;
}

// rho(r) = kappa(r) / sigma^2  (BASELINE.json configs; "stationary covariance kappa(r)")
template <class T>
inline T rho_of(int kind, T r, T ell) {
  switch (kind) {
    case 0: return std::exp(-(r * r) / (T(2) * ell * ell));
    case 1: { T a = std::sqrt(T(3)) * r / ell; return (T(1) + a) * std::exp(-a); }
    default: return std::exp(-r / ell);
  }
}
// d rho / d ell
template <class T>
inline T drho_dell(int kind, T r, T ell) {
  switch (kind) {
    case 0: return rho_of<T>(0, r, ell) * r * r / (ell * ell * ell);
    case 1: { T a = std::sqrt(T(3)) * r / ell; return T(3) * r * r / (ell * ell * ell) * std::exp(-a); }
    default: return rho_of<T>(2, r, ell) * r / (ell * ell);
  }
}

template <class T>
inline T kappa_pair(const double* x, int d, const orc_kernel& kp, int64_t a, int64_t b) {
  T s2 = T(kp.sigma) * T(kp.sigma);
  if (a == b) return s2 * (T(1) + T(kp.jitter));
  T r = std::sqrt(T(d2_canon(x + a * d, x + b * d, d)));
  return s2 * rho_of<T>(kp.kind, r, T(kp.ell));
}

// Textbook row-oriented Cholesky A = L L^T of a dense symmetric m x m matrix (row-major,
// lower part read, L written in place in the lower part).  Returns 0, or 1+row on a
// non-positive pivot.
template <class T>
int cholesky_lower(T* A, int64_t m) {
  for (int64_t a = 0; a < m; ++a) {
    for (int64_t b = 0; b <= a; ++b) {
      T sum = A[a * m + b];
      for (int64_t p = 0; p < b; ++p) sum -= A[a * m + p] * A[b * m + p];
      if (a == b) {
        if (!(sum > T(0))) return int(1 + a);
        A[a * m + a] = std::sqrt(sum);
      } else {
        A[a * m + b] = sum / A[b * m + b];
      }
    }
  }
  return 0;
}
template <class T>
void solve_lower(const T* L, int64_t m, T* y) {  // y <- L^-1 y
  for (int64_t a = 0; a < m; ++a) {
    T sum = y[a];
    for (int64_t p = 0; p < a; ++p) sum -= L[a * m + p] * y[p];
    y[a] = sum / L[a * m + a];
  }
}
template <class T>
void solve_lower_t(const T* L, int64_t m, T* y) {  // y <- L^-T y
  for (int64_t a = m - 1; a >= 0; --a) {
    T sum = y[a];
    for (int64_t p = a + 1; p < m; ++p) sum -= L[p * m + a] * y[p];
    y[a] = sum / L[a * m + a];
  }
}

// Per-point Gaussian conditioning, Eq. 2, in the SOLVE form (deliberately not
// Alg. 1's joint-Cholesky last-row form, so the CUDA kernels are checked by a different formula).
template <class T>
struct Cond {
  std::vector<T> L;     // m x m: K_cc, then its Cholesky factor
  std::vector<T> kci;   // K_ci
  std::vector<T> w;     // K_cc^-1 K_ci
  std::vector<T> tmp;
  T kii = 0, s2 = 0;
  int m = 0;
  // returns 0 ok, else non-PD
  int run(const double* x, int d, const orc_kernel& kp, int64_t i, const int32_t* c, int m_) {
    m = m_;
    L.assign(size_t(m) * m, T(0));
    kci.resize(m);
    w.resize(m);
    for (int a = 0; a < m; ++a) {
      for (int b = 0; b <= a; ++b) L[size_t(a) * m + b] = kappa_pair<T>(x, d, kp, c[a], (a == b) ? c[a] : c[b]);
      kci[a] = kappa_pair<T>(x, d, kp, c[a], i);
    }
    kii = T(kp.sigma) * T(kp.sigma) * (T(1) + T(kp.jitter));
    int rc = cholesky_lower<T>(L.data(), m);
    if (rc) return rc;
    for (int a = 0; a < m; ++a) w[a] = kci[a];
    solve_lower<T>(L.data(), m, w.data());
    solve_lower_t<T>(L.data(), m, w.data());
    T dot = 0;
    for (int a = 0; a < m; ++a) dot += kci[a] * w[a];
    s2 = kii - dot;
    if (!(s2 > T(0))) return -1;
    return 0;
  }
  // alpha = K_cc^-1 vc
  void solve_kcc(T* y) {
    solve_lower<T>(L.data(), m, y);
    solve_lower_t<T>(L.data(), m, y);
  }
};

// A graph as the drivers see it: either "regular" (dense head of n0 + k neighbours per row,
// Alg. 1 `Require`) or "ragged" (CSR, every point through Eq. 2; used by pins).
struct Graph {
  int64_t n = 0, n0 = 0;
  int k = 0;
  const int32_t* nbr = nullptr;     // regular
  const int64_t* rowptr = nullptr;  // ragged
  const int32_t* col = nullptr;
  bool ragged() const { return rowptr != nullptr; }
  int64_t first() const { return ragged() ? 0 : n0; }  // first point handled per-point
  void row(int64_t i, const int32_t*& c, int& m) const {
    if (ragged()) { c = col + rowptr[i]; m = int(rowptr[i + 1] - rowptr[i]); }
    else { c = nbr + (i - n0) * int64_t(k); m = k; }
  }
};

// Batches: batch_off[0..L]; when absent every point is its own batch (purely sequential).
struct Batches {
  const int64_t* off; int64_t L; int64_t first, n;
  int64_t count() const { return off ? L : (n - first); }
  int64_t lo(int64_t b) const { return off ? off[b] : first + b; }
  int64_t hi(int64_t b) const { return off ? off[b + 1] : first + b + 1; }
};

// Dense head (Alg. 1 line 1): K0 = kappa(|x_a - x_b|) over the first n0 points, L0 = chol K0.
template <class T>
int head_factor(const double* x, int d, const orc_kernel& kp, int64_t n0, std::vector<T>& L0) {
  L0.assign(size_t(n0) * n0, T(0));
  for (int64_t a = 0; a < n0; ++a)
    for (int64_t b = 0; b <= a; ++b) L0[a * n0 + b] = kappa_pair<T>(x, d, kp, a, b);
  return cholesky_lower<T>(L0.data(), n0);
}

template <class T>
int forward_impl(const double* x, int d, const Graph& g, const Batches& B, const orc_kernel& kp,
                 const double* xi, double* v) {
  int bad = 0;
  if (!g.ragged() && g.n0 > 0) {
    std::vector<T> L0;
    if (head_factor<T>(x, d, kp, g.n0, L0)) return 3;
    for (int64_t a = 0; a < g.n0; ++a) {  // v_head = L0 xi_head
      T sum = 0;
      for (int64_t b = 0; b <= a; ++b) sum += L0[a * g.n0 + b] * T(xi[b]);
      v[a] = double(sum);
    }
  }
  for (int64_t b = 0; b < B.count(); ++b) {
    int64_t lo = B.lo(b), hi = B.hi(b);
#pragma omp parallel if (hi - lo > 64)
    {
      Cond<T> C;
#pragma omp for schedule(static)
      for (int64_t i = lo; i < hi; ++i) {
        const int32_t* c; int m;
        g.row(i, c, m);
        if (C.run(x, d, kp, i, c, m)) {
#pragma omp atomic write
          bad = 1;
          v[i] = NAN;
          continue;
        }
        T mean = 0;
        for (int a = 0; a < m; ++a) mean += C.w[a] * T(v[c[a]]);
        v[i] = double(mean + std::sqrt(C.s2) * T(xi[i]));   // v_i = w.v_c + s xi_i
      }
    }
  }
  return bad ? 3 : 0;
}

template <class T>
int inverse_impl(const double* x, int d, const Graph& g, const orc_kernel& kp, const double* v, double* xi) {
  int bad = 0;
  if (!g.ragged() && g.n0 > 0) {
    std::vector<T> L0, y(g.n0);
    if (head_factor<T>(x, d, kp, g.n0, L0)) return 3;
    for (int64_t a = 0; a < g.n0; ++a) y[a] = T(v[a]);
    solve_lower<T>(L0.data(), g.n0, y.data());              // xi_head = L0^-1 v_head
    for (int64_t a = 0; a < g.n0; ++a) xi[a] = double(y[a]);
  }
#pragma omp parallel
  {
    Cond<T> C;
#pragma omp for schedule(static)
    for (int64_t i = g.first(); i < g.n; ++i) {
      const int32_t* c; int m;
      g.row(i, c, m);
      if (C.run(x, d, kp, i, c, m)) {
#pragma omp atomic write
        bad = 1;
        xi[i] = NAN;
        continue;
      }
      T mean = 0;
      for (int a = 0; a < m; ++a) mean += C.w[a] * T(v[c[a]]);
      xi[i] = double((T(v[i]) - mean) / std::sqrt(C.s2));    // xi_i = (v_i - w.v_c) / s
    }
  }
  return bad ? 3 : 0;
}

// logdet = sum_i log s_i^2 (+ 2 sum log L0_jj for the dense head); optional gradient w.r.t.
// (sigma, ell):  d/dtheta sum log s^2 = sum_i u^T (dK/dtheta) u / s_i^2,  u = (-w, 1);
// head: tr(K0^-1 dK0/dtheta).
template <class T>
int logdet_impl(const double* x, int d, const Graph& g, const orc_kernel& kp, double* logdet, double* grad) {
  long double acc = 0, gs = 0, gl = 0;
  int bad = 0;
  if (!g.ragged() && g.n0 > 0) {
    int64_t n0 = g.n0;
    std::vector<T> L0;
    if (head_factor<T>(x, d, kp, n0, L0)) return 3;
    for (int64_t a = 0; a < n0; ++a) acc += 2.0L * std::log((long double)L0[a * n0 + a]);
    if (grad) {
      // K0^-1 column by column; tr(K0^-1 dK0)
      std::vector<T> e(n0);
      for (int64_t bcol = 0; bcol < n0; ++bcol) {
        std::fill(e.begin(), e.end(), T(0));
        e[bcol] = 1;
        solve_lower<T>(L0.data(), n0, e.data());
        solve_lower_t<T>(L0.data(), n0, e.data());          // e = K0^-1[:, bcol]
        for (int64_t a = 0; a < n0; ++a) {
          T kab = kappa_pair<T>(x, d, kp, a, bcol);
          gs += (long double)(e[a] * T(2) * kab / T(kp.sigma));
          if (a != bcol) {
            T r = std::sqrt(T(d2_canon(x + a * d, x + bcol * d, d)));
            gl += (long double)(e[a] * T(kp.sigma) * T(kp.sigma) * drho_dell<T>(kp.kind, r, T(kp.ell)));
          }
        }
      }
    }
  }
  int64_t first = g.first();
  std::vector<long double> pl(g.n - first), ps, pe;
  if (grad) { ps.assign(g.n - first, 0); pe.assign(g.n - first, 0); }
#pragma omp parallel
  {
    Cond<T> C;
    std::vector<T> u;
#pragma omp for schedule(static)
    for (int64_t i = first; i < g.n; ++i) {
      const int32_t* c; int m;
      g.row(i, c, m);
      if (C.run(x, d, kp, i, c, m)) {
#pragma omp atomic write
        bad = 1;
        pl[i - first] = NAN;
        continue;
      }
      pl[i - first] = std::log((long double)C.s2);
      if (grad) {
        u.resize(m + 1);
        for (int a = 0; a < m; ++a) u[a] = -C.w[a];
        u[m] = 1;
        T qs = 0, ql = 0;
        for (int a = 0; a <= m; ++a)
          for (int b = 0; b <= m; ++b) {
            int64_t pa = (a < m) ? c[a] : i, pb = (b < m) ? c[b] : i;
            T kab = kappa_pair<T>(x, d, kp, pa, pb);
            qs += u[a] * u[b] * T(2) * kab / T(kp.sigma);
            if (a != b) {
              T r = std::sqrt(T(d2_canon(x + pa * d, x + pb * d, d)));
              ql += u[a] * u[b] * T(kp.sigma) * T(kp.sigma) * drho_dell<T>(kp.kind, r, T(kp.ell));
            }
          }
        ps[i - first] = (long double)(qs / C.s2);
        pe[i - first] = (long double)(ql / C.s2);
      }
    }
  }
  for (size_t t = 0; t < pl.size(); ++t) acc += pl[t];
  if (grad) {
    for (size_t t = 0; t < ps.size(); ++t) { gs += ps[t]; gl += pe[t]; }
    grad[0] = double(gs);
    grad[1] = double(gl);
  }
  *logdet = double(acc);
  return bad ? 3 : 0;
}

// VJP of the forward map (xi, theta) -> v for a cotangent v_bar (R-14).
// Reverse sweep.  Per point, with w = K_cc^-1 K_ci, alpha = K_cc^-1 v_c, u = (-w, 1), g = total
// cotangent on v_i:   xi_bar_i = g s;  g_c += g w;  K_bar = g ( u [alpha;0]^T + (xi_i / 2s) u u^T );
// theta_bar += sum_{a,b} K_bar_ab dK_ab/dtheta over the full joint matrix, dK/dsigma = 2K/sigma,
// dK_ab/dell = sigma^2 drho/dell(r_ab).
// Dense head: v_h = L0 xi_h;  xi_bar_h = L0^T g_h;  L_bar = tril(g_h xi_h^T);
// S = L0^-T Phi(L0^T L_bar) L0^-1 (Phi: lower triangle, diagonal halved);  theta_bar += sum S_ab dK_ab/dtheta.
template <class T>
int vjp_impl(const double* x, int d, const Graph& g, const Batches& B, const orc_kernel& kp,
             const double* xi, const double* v, const double* vbar, double* xibar, double* thetabar) {
  std::vector<long double> gacc(vbar, vbar + g.n);   // running cotangent on v
  long double ts = 0, tl = 0;
  int bad = 0;
  const T sig = T(kp.sigma), s2g = sig * sig;
  for (int64_t b = B.count() - 1; b >= 0; --b) {
    int64_t lo = B.lo(b), hi = B.hi(b), cnt = hi - lo;
    int kk = 0;
    for (int64_t i = lo; i < hi; ++i) { const int32_t* c; int m; g.row(i, c, m); kk = std::max(kk, m); }
    std::vector<T> wst(size_t(cnt) * std::max(kk, 1));
    std::vector<long double> cs(cnt, 0), cl(cnt, 0);
#pragma omp parallel if (cnt > 64)
    {
      Cond<T> C;
      std::vector<T> alpha, u;
#pragma omp for schedule(static)
      for (int64_t i = lo; i < hi; ++i) {
        const int32_t* c; int m;
        g.row(i, c, m);
        if (C.run(x, d, kp, i, c, m)) {
#pragma omp atomic write
          bad = 1;
          continue;
        }
        T s = std::sqrt(C.s2);
        T gi = T(gacc[i]);
        xibar[i] = double(gi * s);
        alpha.resize(m + 1); u.resize(m + 1);
        for (int a = 0; a < m; ++a) { alpha[a] = T(v[c[a]]); u[a] = -C.w[a]; }
        C.solve_kcc(alpha.data());
        alpha[m] = 0; u[m] = 1;
        T coef = T(xi[i]) / (T(2) * s);
        T qs = 0, ql = 0;
        for (int a = 0; a <= m; ++a)
          for (int bb = 0; bb <= m; ++bb) {
            T kbar = gi * (u[a] * alpha[bb] + coef * u[a] * u[bb]);
            int64_t pa = (a < m) ? c[a] : i, pb = (bb < m) ? c[bb] : i;
            qs += kbar * T(2) * kappa_pair<T>(x, d, kp, pa, pb) / sig;
            if (a != bb) {
              T r = std::sqrt(T(d2_canon(x + pa * d, x + pb * d, d)));
              ql += kbar * s2g * drho_dell<T>(kp.kind, r, T(kp.ell));
            }
          }
        cs[i - lo] = (long double)qs;
        cl[i - lo] = (long double)ql;
        for (int a = 0; a < m; ++a) wst[size_t(i - lo) * kk + a] = gi * C.w[a];
      }
    }
    for (int64_t i = lo; i < hi; ++i) {          // sequential, deterministic scatter: g_c += g_i w
      const int32_t* c; int m;
      g.row(i, c, m);
      for (int a = 0; a < m; ++a) gacc[c[a]] += (long double)wst[size_t(i - lo) * kk + a];
      ts += cs[i - lo];
      tl += cl[i - lo];
    }
  }
  if (!g.ragged() && g.n0 > 0) {
    int64_t n0 = g.n0;
    std::vector<T> L0;
    if (head_factor<T>(x, d, kp, n0, L0)) return 3;
    std::vector<T> gh(n0);
    for (int64_t a = 0; a < n0; ++a) gh[a] = T(gacc[a]);
    for (int64_t bcol = 0; bcol < n0; ++bcol) {            // xi_bar_h = L0^T g_h
      T sum = 0;
      for (int64_t a = bcol; a < n0; ++a) sum += L0[a * n0 + bcol] * gh[a];
      xibar[bcol] = double(sum);
    }
    // M = L0^T L_bar,  L_bar_ab = g_a xi_b (a >= b);  only the lower part of M is used.
    std::vector<T> M(size_t(n0) * n0, T(0));
    for (int64_t p = 0; p < n0; ++p) {
      T sum = 0;
      for (int64_t a = p; a < n0; ++a) sum += L0[a * n0 + p] * gh[a];     // sum_{a >= p} L0_ap g_a
      for (int64_t q = 0; q <= p; ++q) M[p * n0 + q] = sum * T(xi[q]);    // (a >= p >= q)
    }
    for (int64_t p = 0; p < n0; ++p) M[p * n0 + p] *= T(0.5);            // Phi
    // S = L0^-T Phi L0^-1 :  first columns (L0^-T Phi), then rows (. L0^-1)
#pragma omp parallel for schedule(static)
    for (int64_t q = 0; q < n0; ++q) {                                     // column q of Phi -> L0^-T col
      std::vector<T> colv(n0);
      for (int64_t p = 0; p < n0; ++p) colv[p] = (p >= q) ? M[p * n0 + q] : T(0);
      solve_lower_t<T>(L0.data(), n0, colv.data());
      for (int64_t p = 0; p < n0; ++p) M[p * n0 + q] = colv[p];
    }
#pragma omp parallel for schedule(static)
    for (int64_t p = 0; p < n0; ++p) {                                     // row p: r L0^-1  <=>  L0^-T r^T
      solve_lower_t<T>(L0.data(), n0, &M[p * n0]);
    }
    for (int64_t a = 0; a < n0; ++a)
      for (int64_t bb = 0; bb < n0; ++bb) {
        T S = M[a * n0 + bb];
        ts += (long double)(S * T(2) * kappa_pair<T>(x, d, kp, a, bb) / sig);
        if (a != bb) {
          T r = std::sqrt(T(d2_canon(x + a * d, x + bb * d, d)));
          tl += (long double)(S * s2g * drho_dell<T>(kp.kind, r, T(kp.ell)));
        }
      }
  }
  thetabar[0] = double(ts);
  thetabar[1] = double(tl);
  return bad ? 3 : 0;
}

// dK_ab/dtheta along the direction (dsigma, dell):  dK = dsigma 2K/sigma + dell sigma^2 drho/dell(r_ab) (zero on the diagonal
// for the ell part: the nugget is relative, K_aa = sigma^2 (1 + eps)).
template <class T>
inline T dkappa_pair(const double* x, int d, const orc_kernel& kp, int64_t a, int64_t b, T dsig, T dell) {
  T out = dsig * T(2) * kappa_pair<T>(x, d, kp, a, b) / T(kp.sigma);
  if (a != b) {
    T r = std::sqrt(T(d2_canon(x + a * d, x + b * d, d)));
    out += dell * T(kp.sigma) * T(kp.sigma) * drho_dell<T>(kp.kind, r, T(kp.ell));
  }
  return out;
}

// Forward-mode derivative of the dense factor (textbook): K0 = L L^T, dK0 given => dL = L Phi(L^-1 dK0 L^-T), Phi = lower
// triangle with the diagonal halved.  dK (n0 x n0, full symmetric, row-major) is overwritten by dL (lower part).
template <class T>
void chol_forward_mode(const T* L, int64_t n0, T* dK) {
  // W = L^-1 dK  (column by column), then Z = W L^-T  (row by row: L^-1 applied to the rows), then Phi, then dL = L Phi
  std::vector<T> colv(n0);
  for (int64_t q = 0; q < n0; ++q) {
    for (int64_t p = 0; p < n0; ++p) colv[p] = dK[p * n0 + q];
    solve_lower<T>(L, n0, colv.data());
    for (int64_t p = 0; p < n0; ++p) dK[p * n0 + q] = colv[p];
  }
  for (int64_t p = 0; p < n0; ++p) solve_lower<T>(L, n0, &dK[p * n0]);      // row p: (W L^-T)[p][:] = L^-1 W[p][:]^T
  for (int64_t p = 0; p < n0; ++p)
    for (int64_t q = 0; q < n0; ++q) dK[p * n0 + q] = (q < p) ? dK[p * n0 + q] : (q == p ? T(0.5) * dK[p * n0 + q] : T(0));
  std::vector<T> out(size_t(n0) * n0, T(0));
  for (int64_t p = 0; p < n0; ++p)
    for (int64_t q = 0; q <= p; ++q) {
      T sum = 0;
      for (int64_t t = q; t <= p; ++t) sum += L[p * n0 + t] * dK[t * n0 + q];
      out[p * n0 + q] = sum;
    }
  std::memcpy(dK, out.data(), sizeof(T) * size_t(n0) * n0);
}

// JVP of the forward map (xi, sigma, ell) -> v along (dxi, dsigma, dell)  ("forward ... derivatives";
// DESIGN.md R-14).  Differentials of Eq. 2 with w = K_cc^-1 K_ci, alpha = K_cc^-1 v_c, u = (-w, 1):
//   dm = u^T dK [alpha; 0] + w . dv_c,    d(s^2) = u^T dK u,    dv_i = dm + d(s^2) xi_i / (2 s) + s dxi_i.
// Dense head: v_h = L0 xi_h  =>  dv_h = dL0 xi_h + L0 dxi_h.
template <class T>
int jvp_impl(const double* x, int d, const Graph& g, const Batches& B, const orc_kernel& kp, const double* xi,
             const double* v, const double* dxi, double dsig, double dell, double* dv) {
  int bad = 0;
  if (!g.ragged() && g.n0 > 0) {
    int64_t n0 = g.n0;
    std::vector<T> L0;
    if (head_factor<T>(x, d, kp, n0, L0)) return 3;
    std::vector<T> dL(size_t(n0) * n0);
    for (int64_t a = 0; a < n0; ++a)
      for (int64_t b = 0; b < n0; ++b) dL[a * n0 + b] = dkappa_pair<T>(x, d, kp, a, b, T(dsig), T(dell));
    chol_forward_mode<T>(L0.data(), n0, dL.data());
    for (int64_t a = 0; a < n0; ++a) {
      T sum = 0;
      for (int64_t b = 0; b <= a; ++b) sum += dL[a * n0 + b] * T(xi[b]) + L0[a * n0 + b] * T(dxi[b]);
      dv[a] = double(sum);
    }
  }
  for (int64_t b = 0; b < B.count(); ++b) {
    int64_t lo = B.lo(b), hi = B.hi(b);
#pragma omp parallel if (hi - lo > 64)
    {
      Cond<T> C;
      std::vector<T> alpha, u;
#pragma omp for schedule(static)
      for (int64_t i = lo; i < hi; ++i) {
        const int32_t* c; int m;
        g.row(i, c, m);
        if (C.run(x, d, kp, i, c, m)) {
#pragma omp atomic write
          bad = 1;
          dv[i] = NAN;
          continue;
        }
        T s = std::sqrt(C.s2);
        alpha.resize(m + 1); u.resize(m + 1);
        for (int a = 0; a < m; ++a) { alpha[a] = T(v[c[a]]); u[a] = -C.w[a]; }
        C.solve_kcc(alpha.data());
        alpha[m] = 0; u[m] = 1;
        T dm = 0, ds2 = 0;
        for (int a = 0; a <= m; ++a)
          for (int bb = 0; bb <= m; ++bb) {
            int64_t pa = (a < m) ? c[a] : i, pb = (bb < m) ? c[bb] : i;
            T dk = dkappa_pair<T>(x, d, kp, pa, pb, T(dsig), T(dell));
            dm += u[a] * dk * alpha[bb];
            ds2 += u[a] * dk * u[bb];
          }
        for (int a = 0; a < m; ++a) dm += C.w[a] * T(dv[c[a]]);
        dv[i] = double(dm + ds2 * T(xi[i]) / (T(2) * s) + s * T(dxi[i]));
      }
    }
  }
  return bad ? 3 : 0;
}

// VJP of the inverse map (v, sigma, ell) -> xi for a cotangent xi_bar = h  (R-14):
//   xi_i = (v_i - w . v_c) / s:   v_bar_i += h_i / s,   v_bar_c -= (h_i / s) w,
//   K_bar = -(h_i / s) u [alpha; 0]^T - (h_i xi_i / (2 s^2)) u u^T,   theta_bar += sum_ab K_bar_ab dK_ab/dtheta.
// No sweep is needed: every point contributes independently.  Dense head: xi_h = L0^-1 v_h =>
// v_bar_h += L0^-T h_h and, parameter by parameter, theta_bar_p -= h_h . L0^-1 dL0_p xi_h (forward mode of the factor).
template <class T>
int inverse_vjp_impl(const double* x, int d, const Graph& g, const orc_kernel& kp, const double* v, const double* xi,
                     const double* h, double* vbar, double* thetabar) {
  std::vector<long double> acc(g.n, 0.0L);
  long double ts = 0, tl = 0;
  int bad = 0;
  int64_t first = g.first();
  if (!g.ragged() && g.n0 > 0) {
    int64_t n0 = g.n0;
    std::vector<T> L0, y(n0);
    if (head_factor<T>(x, d, kp, n0, L0)) return 3;
    for (int64_t a = 0; a < n0; ++a) y[a] = T(h[a]);
    solve_lower_t<T>(L0.data(), n0, y.data());                 // L0^-T h_h
    for (int64_t a = 0; a < n0; ++a) acc[a] += (long double)y[a];
    for (int p = 0; p < 2; ++p) {
      std::vector<T> dL(size_t(n0) * n0);
      for (int64_t a = 0; a < n0; ++a)
        for (int64_t b = 0; b < n0; ++b) dL[a * n0 + b] = dkappa_pair<T>(x, d, kp, a, b, T(p == 0), T(p == 1));
      chol_forward_mode<T>(L0.data(), n0, dL.data());
      std::vector<T> t(n0);
      for (int64_t a = 0; a < n0; ++a) {
        T sum = 0;
        for (int64_t b = 0; b <= a; ++b) sum += dL[a * n0 + b] * T(xi[b]);
        t[a] = sum;
      }
      solve_lower<T>(L0.data(), n0, t.data());                 // L0^-1 dL0 xi_h
      long double dot = 0;
      for (int64_t a = 0; a < n0; ++a) dot += (long double)(T(h[a]) * t[a]);
      (p == 0 ? ts : tl) -= dot;
    }
  }
  // sequential over points (deterministic scatter); the per-point work is the oracle's usual conditioning
  Cond<T> C;
  std::vector<T> alpha, u;
  for (int64_t i = first; i < g.n; ++i) {
    const int32_t* c; int m;
    g.row(i, c, m);
    if (C.run(x, d, kp, i, c, m)) { bad = 1; continue; }
    T s = std::sqrt(C.s2), hs = T(h[i]) / s;
    acc[i] += (long double)hs;
    alpha.resize(m + 1); u.resize(m + 1);
    for (int a = 0; a < m; ++a) { alpha[a] = T(v[c[a]]); u[a] = -C.w[a]; acc[c[a]] -= (long double)(hs * C.w[a]); }
    C.solve_kcc(alpha.data());
    alpha[m] = 0; u[m] = 1;
    T coef = T(h[i]) * T(xi[i]) / (T(2) * C.s2);
    T qs = 0, ql = 0;
    for (int a = 0; a <= m; ++a)
      for (int bb = 0; bb <= m; ++bb) {
        T kbar = -hs * u[a] * alpha[bb] - coef * u[a] * u[bb];
        int64_t pa = (a < m) ? c[a] : i, pb = (bb < m) ? c[bb] : i;
        qs += kbar * dkappa_pair<T>(x, d, kp, pa, pb, T(1), T(0));
        ql += kbar * dkappa_pair<T>(x, d, kp, pa, pb, T(0), T(1));
      }
    ts += (long double)qs;
    tl += (long double)ql;
  }
  for (int64_t i = 0; i < g.n; ++i) vbar[i] = double(acc[i]);
  thetabar[0] = double(ts);
  thetabar[1] = double(tl);
  return bad ? 3 : 0;
}

// ---- order ---------------------------------------------------------------------------
inline int level_of(int64_t i) {  // floor(log2(i+1))
  int l = 0;
  uint64_t t = uint64_t(i) + 1;
  while (t >>= 1) ++l;
  return l;
}

struct OrderCtx {
  const double* x; int64_t n; int d;
  std::vector<int64_t> sz;   // subtree sizes from the child formula alone
  int64_t* perm;
};

void assign_node(OrderCtx& C, int64_t node, int64_t* idx, int64_t cnt) {
  // `idx[0..cnt)` are the user ids of the points that form the subtree rooted at `node`.
  if (node >= C.n || cnt == 0) return;
  int l = level_of(node);
  int dim = l % C.d;
  int64_t left = node + (int64_t(1) << l), right = node + (int64_t(1) << (l + 1));
  int64_t nl = (left < C.n) ? C.sz[left] : 0;
  auto cmp = [&](int64_t a, int64_t b) {
    double xa = C.x[a * C.d + dim], xb = C.x[b * C.d + dim];
    return (xa < xb) || (xa == xb && a < b);                 // key (coordinate, user id), reading R-4
  };
  std::nth_element(idx, idx + nl, idx + cnt, cmp);           // first nl keys -> left, next one is the node
  C.perm[node] = idx[nl];
#pragma omp task shared(C) firstprivate(left, idx, nl) if (cnt > 4096)
  assign_node(C, left, idx, nl);
#pragma omp task shared(C) firstprivate(right, idx, nl, cnt) if (cnt > 4096)
  assign_node(C, right, idx + nl + 1, cnt - nl - 1);
}

}  // namespace

extern "C" {

int orc_num_threads() {
#ifdef _OPENMP
  return omp_get_max_threads();
#else
  return 1;
#endif
}

// O-2: bit-reversed left-balanced k-d tree order.  perm_tree[node] = user id.
// Split dimension = level mod d (R-3); ties by (coordinate, user id) (R-4).
int orc_order(const double* x, int64_t n, int32_t d, int64_t* perm_tree) {
  OrderCtx C{x, n, d, std::vector<int64_t>(size_t(n), 1), perm_tree};
  for (int64_t i = n - 1; i >= 0; --i) {                     // subtree sizes, bottom up
    int l = level_of(i);
    int64_t left = i + (int64_t(1) << l), right = i + (int64_t(1) << (l + 1));
    int64_t s = 1;
    if (left < n) s += C.sz[left];
    if (right < n) s += C.sz[right];
    C.sz[i] = s;
  }
  std::vector<int64_t> idx(n);
  std::iota(idx.begin(), idx.end(), int64_t(0));
#pragma omp parallel
#pragma omp single
  assign_node(C, 0, idx.data(), n);
  return 0;
}

// subtree sizes only (for tests of the closed form used by the GPU builder)
void orc_subtree_sizes(int64_t n, int64_t* sz) {
  for (int64_t i = n - 1; i >= 0; --i) {
    int l = level_of(i);
    int64_t left = i + (int64_t(1) << l), right = i + (int64_t(1) << (l + 1));
    int64_t s = 1;
    if (left < n) s += sz[left];
    if (right < n) s += sz[right];
    sz[i] = s;
  }
}

// O-3: preceding k nearest neighbours by brute force.  For each listed row i,
// the k smallest (d2_canon(i,j), j), j < i, in lexicographic order; written nearest first.
// Rows with i < k get the i available predecessors followed by -1.
void orc_knn_rows(const double* x, int64_t n, int32_t d, int32_t k, const int64_t* rows, int64_t nrows,
                  int32_t* out) {
  (void)n;
#pragma omp parallel for schedule(dynamic, 4)
  for (int64_t t = 0; t < nrows; ++t) {
    int64_t i = rows[t];
    std::vector<double> bd(k);
    std::vector<int32_t> bj(k);
    int cnt = 0;
    for (int64_t j = 0; j < i; ++j) {
      double dd = d2_canon(x + i * d, x + j * d, d);
      if (cnt == k && !(dd < bd[k - 1])) continue;           // j increases, so equal d2 never displaces
      int pos = (cnt < k) ? cnt : k - 1;
      while (pos > 0 && dd < bd[pos - 1]) { bd[pos] = bd[pos - 1]; bj[pos] = bj[pos - 1]; --pos; }
      bd[pos] = dd; bj[pos] = int32_t(j);
      if (cnt < k) ++cnt;
    }
    for (int a = 0; a < k; ++a) out[t * k + a] = (a < cnt) ? bj[a] : -1;
  }
}

// O-4: depth[i] = 0 for i < n0, else 1 + max_{j in c(i)} depth[j], one sequential pass.
void orc_depth(const int32_t* nbr, int64_t n, int64_t n0, int32_t k, int32_t* depth) {
  for (int64_t i = 0; i < n0; ++i) depth[i] = 0;
  for (int64_t i = n0; i < n; ++i) {
    int32_t m = 0;
    for (int a = 0; a < k; ++a) m = std::max(m, depth[nbr[(i - n0) * k + a]]);
    depth[i] = 1 + m;
  }
}
// The parallel fixed point of PAPER.md:59: apply the update to all points at once (Jacobi),
// repeat until nothing changes.  Returns the number of sweeps.
int64_t orc_depth_fixed_point(const int32_t* nbr, int64_t n, int64_t n0, int32_t k, int32_t* depth) {
  std::vector<int32_t> cur(n, 0), nxt(n, 0);
  for (int64_t i = n0; i < n; ++i) cur[i] = 1;
  int64_t sweeps = 0;
  for (;;) {
    bool changed = false;
    for (int64_t i = 0; i < n0; ++i) nxt[i] = 0;
    for (int64_t i = n0; i < n; ++i) {
      int32_t m = 0;
      for (int a = 0; a < k; ++a) m = std::max(m, cur[nbr[(i - n0) * k + a]]);
      nxt[i] = 1 + m;
      if (nxt[i] != cur[i]) changed = true;
    }
    ++sweeps;
    cur.swap(nxt);
    if (!changed) break;
  }
  std::memcpy(depth, cur.data(), n * sizeof(int32_t));
  return sweeps;
}

// Per-point conditioning (Eq. 2): w[m], s2.
int orc_condition(const double* x, int32_t d, const orc_kernel* kp, int64_t i, const int32_t* c, int32_t m,
                  double* w, double* s2) {
  Cond<double> C;
  int rc = C.run(x, d, *kp, i, c, m);
  if (rc) return 3;
  for (int a = 0; a < m; ++a) w[a] = C.w[a];
  *s2 = C.s2;
  return 0;
}

// Conditional standard deviations s_i = sqrt(K_ii - K_ic K_cc^-1 K_ci) of Eq. 2 for every point:
// the diagonal of the dense head factor for i < n0 (Alg. 1 line 1: v_head = L0 xi_head, so dv_i/dxi_i = L0_ii),
// Cond::run for the rest.  Tests use it to express an error of the inverse in units of v (R-16).
int orc_cond_std(const double* x, int64_t n, int32_t d, int64_t n0, int32_t k, const int32_t* nbr,
                 const int64_t* rowptr, const int32_t* col, const orc_kernel* kp, double* s_out) {
  Graph g; g.n = n; g.n0 = n0; g.k = k; g.nbr = nbr; g.rowptr = rowptr; g.col = col;
  int bad = 0;
  if (!g.ragged() && n0 > 0) {
    std::vector<double> L0;
    if (head_factor<double>(x, d, *kp, n0, L0)) return 3;
    for (int64_t a = 0; a < n0; ++a) s_out[a] = L0[a * n0 + a];
  }
#pragma omp parallel
  {
    Cond<double> C;
#pragma omp for schedule(static)
    for (int64_t i = g.first(); i < n; ++i) {
      const int32_t* c; int m;
      g.row(i, c, m);
      if (C.run(x, d, *kp, i, c, m)) {
#pragma omp atomic write
        bad = 1;
        s_out[i] = NAN;
        continue;
      }
      s_out[i] = std::sqrt(C.s2);
    }
  }
  return bad ? 3 : 0;
}

double orc_rho(int32_t kind, double r, double ell) { return rho_of<double>(kind, r, ell); }
double orc_drho_dell(int32_t kind, double r, double ell) { return drho_dell<double>(kind, r, ell); }
double orc_d2(const double* a, const double* b, int32_t d) { return d2_canon(a, b, d); }

#define ORC_GRAPH_ARGS const double *x, int64_t n, int32_t d, int64_t n0, int32_t k, const int32_t *nbr, \
                       const int64_t *rowptr, const int32_t *col, const int64_t *batch_off, int64_t n_batches
#define ORC_MAKE_GRAPH                                                            \
  Graph g; g.n = n; g.n0 = n0; g.k = k; g.nbr = nbr; g.rowptr = rowptr; g.col = col; \
  Batches B{batch_off, n_batches, g.first(), n};

// Regular graph: rowptr = col = NULL.  Ragged graph: nbr = NULL, n0/k ignored.
int orc_forward(ORC_GRAPH_ARGS, const orc_kernel* kp, const double* xi, double* v, int32_t use_long_double) {
  ORC_MAKE_GRAPH
  return use_long_double ? forward_impl<long double>(x, d, g, B, *kp, xi, v)
                         : forward_impl<double>(x, d, g, B, *kp, xi, v);
}
int orc_inverse(ORC_GRAPH_ARGS, const orc_kernel* kp, const double* v, double* xi, int32_t use_long_double) {
  ORC_MAKE_GRAPH
  (void)B;
  return use_long_double ? inverse_impl<long double>(x, d, g, *kp, v, xi) : inverse_impl<double>(x, d, g, *kp, v, xi);
}
int orc_logdet(ORC_GRAPH_ARGS, const orc_kernel* kp, double* logdet, double* grad2, int32_t use_long_double) {
  ORC_MAKE_GRAPH
  (void)B;
  return use_long_double ? logdet_impl<long double>(x, d, g, *kp, logdet, grad2)
                         : logdet_impl<double>(x, d, g, *kp, logdet, grad2);
}
int orc_vjp(ORC_GRAPH_ARGS, const orc_kernel* kp, const double* xi, const double* v, const double* vbar,
            double* xibar, double* thetabar2, int32_t use_long_double) {
  ORC_MAKE_GRAPH
  return use_long_double ? vjp_impl<long double>(x, d, g, B, *kp, xi, v, vbar, xibar, thetabar2)
                         : vjp_impl<double>(x, d, g, B, *kp, xi, v, vbar, xibar, thetabar2);
}

int orc_jvp(ORC_GRAPH_ARGS, const orc_kernel* kp, const double* xi, const double* v, const double* dxi, double dsigma,
            double dell, double* dv) {
  ORC_MAKE_GRAPH
  return jvp_impl<double>(x, d, g, B, *kp, xi, v, dxi, dsigma, dell, dv);
}
int orc_inverse_vjp(ORC_GRAPH_ARGS, const orc_kernel* kp, const double* v, const double* xi, const double* h, double* vbar,
                    double* thetabar2) {
  ORC_MAKE_GRAPH
  (void)B;
  return inverse_vjp_impl<double>(x, d, g, *kp, v, xi, h, vbar, thetabar2);
}

}  // extern "C"
