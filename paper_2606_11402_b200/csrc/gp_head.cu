// Dense initial block (Alg. 1 line 1): the first n0 values come from a dense
// Cholesky of K_head.  Always factored in fp64 (n0^3/3 flops are negligible next to the N k^3 of the
// conditioning, and the head feeds every later point), whatever the working dtype.
//
// Right-looking blocked Cholesky of M = K_head / sigma^2 (row-major, lower part), NB = 32, with
// `carried` extra rows below the square part that receive the same panel solves and trailing updates:
// a carried row that starts as r^T ends as (L^-1 r)^T, exactly the values row of Alg. 1.
//   inverse : 1 carried row  = v_head^T      ->  (L^-1 v_head)^T = sigma * xi_head^T
//   VJP     : n0 carried rows = identity     ->  L^-T
#include <cooperative_groups.h>

#include "gp_cond.cuh"

namespace cg = cooperative_groups;

namespace gp {

constexpr int NB = 32;

template <typename T>
__global__ void head_build_kernel(const T* __restrict__ x, int d, int n0, int kind, KParams<double> kp,
                                  double* __restrict__ A) {
  int c = blockIdx.x * blockDim.x + threadIdx.x;
  int r = blockIdx.y * blockDim.y + threadIdx.y;
  if (r >= n0 || c > r) return;
  double val;
  if (r == c) {
    val = kp.diag;
  } else {
    double d2 = 0.0;
    for (int t = 0; t < d; ++t) {
      double dx = (double)x[(size_t)r * d + t] - (double)x[(size_t)c * d + t];
      d2 = fma(dx, dx, d2);
    }
    val = rho_rt<double>(kind, d2 * kp.qscale);
  }
  A[(size_t)r * n0 + c] = val;
}

// gradient mode: rows n0..2n0-1 = identity, rows 2n0..3n0-1 = ell * dM/dell (symmetric, zero diagonal)
template <typename T>
__global__ void head_carry_grad_init_kernel(const T* __restrict__ x, int d, int n0, int kind, KParams<double> kp,
                                            double* __restrict__ A) {
  int c = blockIdx.x * blockDim.x + threadIdx.x;
  int r = blockIdx.y * blockDim.y + threadIdx.y;
  if (r >= n0 || c >= n0) return;
  double* C1 = A + (size_t)n0 * n0;
  double* C2 = C1 + (size_t)n0 * n0;
  C1[(size_t)r * n0 + c] = r == c ? 1.0 : 0.0;
  double val = 0.0;
  if (r != c) {
    double d2 = 0.0;
    for (int t = 0; t < d; ++t) {
      double dx = (double)x[(size_t)r * d + t] - (double)x[(size_t)c * d + t];
      d2 = fma(dx, dx, d2);
    }
    val = drho_rt<double>(kind, d2 * kp.qscale);
  }
  C2[(size_t)r * n0 + c] = val;
}

// carried rows: mode 1 = one row holding src[0:n0]; mode 2 = identity (n0 rows)
template <typename T>
__global__ void head_carry_init_kernel(const T* __restrict__ src, int n0, int mode, double* __restrict__ A) {
  int64_t e = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  int64_t total = mode == 1 ? n0 : (int64_t)n0 * n0;
  if (e >= total) return;
  double* C = A + (size_t)n0 * n0;
  if (mode == 1) C[e] = (double)src[e];
  else C[e] = (e / n0 == e % n0) ? 1.0 : 0.0;
}

// The whole blocked factorisation in ONE cooperative launch (the per-panel launches of a host loop cost more
// than the arithmetic: n0 = 1024 is 32 panels, each a strictly serial step).  Per panel two grid barriers:
//   phase 1  every CTA that owns panel rows factors the 32 x 32 diagonal block (one warp, rows in registers,
//            pivots broadcast by shuffles), then one WARP per row solves its panel row; CTA 0 writes the factored
//            block back after the barrier (the other CTAs read the unfactored one until then);
//   phase 2  64 x 64 trailing tiles, dealt round-robin to the CTAs.
__device__ __forceinline__ double shfl_d(double v, int src) { return __shfl_sync(0xffffffffu, v, src); }

// 1 / sqrt(x) in full double precision from the fp32 MUFU seed and two Newton steps (2^-22 -> 2^-44 -> 2^-88):
// a much shorter dependent chain than the library's rsqrt(double), and this chain is what the head waits on.
__device__ __forceinline__ double rsqrt_fast(double x) {
  double y = (double)rsqrtf((float)x);
  double h = 0.5 * x;
  y = y * fma(-h * y, y, 1.5);
  y = y * fma(-h * y, y, 1.5);
  return y;
}

// Pivot J of the in-register 32 x 32 factorisation (lane r holds row r); a template recursion so that every
// index into a[] is a compile-time constant (a loop this size is not unrolled reliably -> local memory).
// The scaled column is broadcast through shared memory (one store per lane, then broadcast loads) rather than
// by two shuffles per element, and entries above the diagonal are updated too (junk that is never read) so that
// no select is needed: measured, the shuffle version spent 9 us per 32 x 32 block, 45 % of the whole head.
template <int J> struct DiagStep {
  static __device__ __forceinline__ void run(double (&a)[NB], int lane, double* invd, double* col, bool& bad) {
    double piv = shfl_d(a[J], J);
    bad |= !(piv > 0.0);
    double inv = rsqrt_fast(piv);
    double lj = a[J] * inv;                           // lane J: sqrt(piv); lanes > J: L[lane][J]
    a[J] = lj;
    if (lane == J) invd[J] = inv;
    if (J + 1 < NB) {
      col[lane] = lj;
      __syncwarp();
#pragma unroll
      for (int c = J + 1; c < NB; ++c) a[c] = fma(-lj, col[c], a[c]);
      __syncwarp();
    }
    DiagStep<J + 1>::run(a, lane, invd, col, bad);
  }
};
template <> struct DiagStep<NB> {
  static __device__ __forceinline__ void run(double (&)[NB], int, double*, double*, bool&) {}
};

// Two entry points (below): head_chol_kernel_128 is capped at 128 registers (a few spills) - beside the VJP's geometry pass,
// 255 registers x 128 threads, one geometry CTA must still fit on an SM that holds a head CTA, or the geometry pass loses
// those SMs (VJP 8.27 against 8.38 ms); head_chol_kernel is unconstrained (142 registers, no spill).  An explicit minimum
// of one CTA per SM made the compiler take 255 registers, and then no bulk CTA fits beside the head at all.
static __device__ __forceinline__ void head_chol_body(double* __restrict__ A, int n0, int rows_total, int lookahead,
                                                      Control* ctrl) {
  cg::grid_group grid = cg::this_grid();
  __shared__ double Ds[NB][NB + 1];
  __shared__ double invd[NB];
  __shared__ double colbuf[NB];
  __shared__ __align__(16) double Pr[NB][64 + 2];
  __shared__ __align__(16) double Pc[NB][64 + 2];
  const int tid = threadIdx.x, lane = tid & 31;
  const int G = gridDim.x;
  // LOOK-AHEAD (G >= 2): the last CTA takes no tiles; during phase 2 of panel p it updates the NEXT 32 x 32 diagonal
  // block, factors it and writes the factor to A, so that in phase 1 of panel p + 1 every CTA just reads the factored
  // block instead of all of them repeating its 32-step pivot chain on the critical path (profiles/r2_head_samples.md:
  // 27 % of the warp samples sat in the barrier behind that chain).  The tile owners leave that block alone.
  const bool la = lookahead && G >= 2;
  const int GT = la ? G - 1 : G;                      // CTAs that take tiles
  for (int j0 = 0; j0 < n0; j0 += NB) {
    const int nb = min(NB, n0 - j0);
    const int j1 = j0 + nb;
    const int below = rows_total - j1;
    // ---- phase 1 --------------------------------------------------------------------------------------
    // panel rows are dealt to WARPS (one row per warp at a time, lane = column): coalesced 256 B row loads, and a
    // 32-step chain per row instead of one thread grinding through 496 dependent FMAs
    const int warp = tid >> 5, nwarp = blockDim.x >> 5;
    const int first_row = j1 + (int)blockIdx.x * nwarp + warp;
    if ((int)blockIdx.x * nwarp < below || blockIdx.x == 0) {
      if (!la || j0 == 0) {
        if (tid < 32) {
          double a[NB];
#pragma unroll
          for (int c = 0; c < NB; ++c)
            a[c] = (lane < nb && c <= lane && c < nb) ? A[(size_t)(j0 + lane) * n0 + j0 + c] : (c == lane ? 1.0 : 0.0);
          bool bad = false;
          DiagStep<0>::run(a, lane, invd, colbuf, bad);
          if (bad && blockIdx.x == 0 && lane == 0) atomicAdd(&ctrl->n_bad, 1ULL);
#pragma unroll
          for (int c = 0; c < NB; ++c) Ds[lane][c] = c <= lane ? a[c] : 0.0;
        }
      } else {
        // the factored block is in A already (look-ahead CTA, previous phase 2)
        for (int e = tid; e < NB * NB; e += blockDim.x) {
          const int r = e / NB, cc = e % NB;
          Ds[r][cc] = (r < nb && cc <= r) ? A[(size_t)(j0 + r) * n0 + j0 + cc] : (r == cc ? 1.0 : 0.0);
        }
        __syncthreads();
        if (tid < NB) invd[tid] = 1.0 / Ds[tid][tid];
      }
      __syncthreads();
      for (int r = first_row; r < rows_total; r += G * nwarp) {
        double* arow = A + (size_t)r * n0 + j0;
        double a = lane < nb ? arow[lane] : 0.0;
#pragma unroll
        for (int c = 0; c < NB; ++c) {
          const double xc = shfl_d(a, c) * invd[c];
          if (lane == c) a = xc;
          else if (lane > c) a = fma(-xc, Ds[lane][c], a);
        }
        if (lane < nb) arow[lane] = a;
      }
    }
    grid.sync();
    // ---- phase 2 --------------------------------------------------------------------------------------
    // Without look-ahead (and for the first panel) CTA 0 writes the factored diagonal block back only now: during phase 1
    // the other CTAs were still reading the unfactored block from A (every CTA factors its own copy), and nothing in
    // this kernel reads it again.
    if (blockIdx.x == 0 && (!la || j0 == 0)) {
      for (int e = tid; e < NB * NB; e += blockDim.x) {
        const int r = e / NB, cc = e % NB;
        if (r < nb && cc <= r) A[(size_t)(j0 + r) * n0 + j0 + cc] = Ds[r][cc];
      }
    }
    const int cols = n0 - j1;
    if (cols > 0 && la && blockIdx.x == G - 1) {
      // next diagonal block: D = A[j1 : j1 + nb2][j1 : j1 + nb2] - P P^T with P = the panel rows just solved, then factor
      const int nb2 = min(NB, n0 - j1);
      __syncthreads();
      for (int e = tid; e < NB * NB; e += blockDim.x) {
        const int row = e / NB, tt = e % NB;
        Pr[tt][row] = (row < nb2 && tt < nb) ? A[(size_t)(j1 + row) * n0 + j0 + tt] : 0.0;
      }
      __syncthreads();
      for (int e = tid; e < NB * NB; e += blockDim.x) {
        const int r = e / NB, cc = e % NB;
        double v = r == cc ? 1.0 : 0.0;                // padding of a short last block: identity
        if (r < nb2 && cc <= r) {
          double acc = 0.0;
#pragma unroll 8
          for (int tt = 0; tt < NB; ++tt) acc = fma(Pr[tt][r], Pr[tt][cc], acc);
          v = A[(size_t)(j1 + r) * n0 + j1 + cc] - acc;
        } else if (cc > r) {
          v = 0.0;
        }
        Ds[r][cc] = v;
      }
      __syncthreads();
      if (tid < 32) {
        double a[NB];
#pragma unroll
        for (int c = 0; c < NB; ++c) a[c] = Ds[lane][c];
        bool bad = false;
        DiagStep<0>::run(a, lane, invd, colbuf, bad);
        if (bad && lane == 0) atomicAdd(&ctrl->n_bad, 1ULL);
#pragma unroll
        for (int c = 0; c < NB; ++c)
          if (lane < nb2 && c <= lane) A[(size_t)(j1 + lane) * n0 + j1 + c] = a[c];
      }
    } else if (cols > 0) {
      const int ntc = (cols + 63) / 64, ntr = (below + 63) / 64;
      const int nb2t = min(NB, n0 - j1);             // size of the next diagonal block
      // valid tiles only: for a row tile inside the square part, column tiles up to the diagonal
      for (int t = blockIdx.x;; t += GT) {
        // map t to the t-th valid tile: rows tr < ntc are triangular (tr + 1 tiles), the rest are full
        int tr, tc;
        const int tri_tiles = ntc * (ntc + 1) / 2;
        if (t < tri_tiles) {
          tr = (int)((sqrt(8.0 * t + 1.0) - 1.0) * 0.5);
          while (tr * (tr + 1) / 2 > t) --tr;
          while ((tr + 1) * (tr + 2) / 2 <= t) ++tr;
          tc = t - tr * (tr + 1) / 2;
        } else {
          int u = t - tri_tiles;
          tr = ntc + u / ntc;
          tc = u % ntc;
        }
        if (tr >= ntr) break;
        const int r0 = j1 + tr * 64, c0 = j1 + tc * 64;
        __syncthreads();
        for (int e = tid; e < 64 * NB; e += 256) {
          int row = e / NB, tt = e % NB;
          int rr = r0 + row, cc = c0 + row;
          Pr[tt][row] = (rr < rows_total && tt < nb) ? A[(size_t)rr * n0 + j0 + tt] : 0.0;
          Pc[tt][row] = (cc < n0 && tt < nb) ? A[(size_t)cc * n0 + j0 + tt] : 0.0;
        }
        __syncthreads();
        const int tx = tid % 16, ty = tid / 16;
        double acc[4][4];
#pragma unroll
        for (int a_ = 0; a_ < 4; ++a_)
#pragma unroll
          for (int b_ = 0; b_ < 4; ++b_) acc[a_][b_] = 0.0;
#pragma unroll 8
        for (int tt = 0; tt < NB; ++tt) {
          double pr[4], pc[4];                       // 16 B-aligned: rows are 66 doubles, offsets multiples of 4
          const double2 r01 = *reinterpret_cast<const double2*>(&Pr[tt][ty * 4]);
          const double2 r23 = *reinterpret_cast<const double2*>(&Pr[tt][ty * 4 + 2]);
          const double2 c01 = *reinterpret_cast<const double2*>(&Pc[tt][tx * 4]);
          const double2 c23 = *reinterpret_cast<const double2*>(&Pc[tt][tx * 4 + 2]);
          pr[0] = r01.x; pr[1] = r01.y; pr[2] = r23.x; pr[3] = r23.y;
          pc[0] = c01.x; pc[1] = c01.y; pc[2] = c23.x; pc[3] = c23.y;
#pragma unroll
          for (int a_ = 0; a_ < 4; ++a_)
#pragma unroll
            for (int b_ = 0; b_ < 4; ++b_) acc[a_][b_] = fma(pr[a_], pc[b_], acc[a_][b_]);
        }
#pragma unroll
        for (int a_ = 0; a_ < 4; ++a_) {
          int r = r0 + ty * 4 + a_;
          if (r >= rows_total) continue;
#pragma unroll
          for (int b_ = 0; b_ < 4; ++b_) {
            int cidx = c0 + tx * 4 + b_;
            if (cidx >= n0 || (r < n0 && cidx > r)) continue;
            if (la && r < j1 + nb2t) continue;         // the next diagonal block (rows j1 .. j1 + nb2t - 1, all their
                                                       // columns >= j1) belongs to the look-ahead CTA
            A[(size_t)r * n0 + cidx] -= acc[a_][b_];
          }
        }
      }
    }
    grid.sync();
  }
}

__global__ void __launch_bounds__(256) head_chol_kernel(double* __restrict__ A, int n0, int rows_total, int lookahead,
                                                        Control* ctrl) {
  head_chol_body(A, n0, rows_total, lookahead, ctrl);
}
__global__ void __launch_bounds__(256, 2) head_chol_kernel_128(double* __restrict__ A, int n0, int rows_total,
                                                               int lookahead, Control* ctrl) {
  head_chol_body(A, n0, rows_total, lookahead, ctrl);
}

static gp_status head_build(const OpCtx& c) {
  const int n0 = (int)c.g->n0;
  KParams<double> kp = make_kparams<double>(*c.kern);
  dim3 bb(16, 16), bg((n0 + 15) / 16, (n0 + 15) / 16);
  if (c.g->dtype == GP_F64)
    head_build_kernel<double><<<bg, bb, 0, c.st>>>((const double*)c.g->x, c.g->d, n0, c.kern->kind, kp, c.head());
  else
    head_build_kernel<float><<<bg, bb, 0, c.st>>>((const float*)c.g->x, c.g->d, n0, c.kern->kind, kp, c.head());
  GP_LAUNCH_CHECK();
  return GP_OK;
}

static gp_status head_chol(const OpCtx& c, int n_carried, bool overlapped) {
  const int n0 = (int)c.g->n0;
  double* A = c.head();
  int rows_total = n0 + n_carried;
  const int grid_ctas = device_sm_count();                  // one CTA per SM: all co-resident
  if (grid_ctas <= 0) return GP_ERR_CUDA;
  int n0_arg = n0;
  Control* ctrl = c.ctrl();
  int lookahead = 1;
  void* args[] = {(void*)&A, (void*)&n0_arg, (void*)&rows_total, (void*)&lookahead, (void*)&ctrl};
  int ctas = grid_ctas;
  // beside a LONG bulk kernel the head takes a quarter of the SMs (more when many rows are carried) and is hidden;
  // beside a short one (config 2: 2^20 points, 0.2 ms of bulk work) it is the critical path and takes every SM
  if (overlapped && c.g->n - c.g->n0 >= ((int64_t)1 << (c.g->dtype == GP_F64 ? 19 : 22))) {
    ctas = n_carried > n0 ? grid_ctas / 2 : grid_ctas / 4;
    if (ctas < 1) ctas = 1;
  }
  const void* fn = n_carried > 1 ? (const void*)head_chol_kernel_128 : (const void*)head_chol_kernel;
  GP_CUDA_OK(cudaLaunchCooperativeKernel(fn, dim3(ctas), dim3(256), args, 0, c.st));
  GP_LAUNCH_CHECK();
  return GP_OK;
}

gp_status head_factor_preinit(const OpCtx& c, int n_carried, bool overlapped) {
  if (c.g->n0 <= 0) return GP_OK;
  GP_OK_OR_RETURN(head_build(c));
  return head_chol(c, n_carried, overlapped);
}

gp_status head_factor(const OpCtx& c, const void* carried_src, int n_carried, bool overlapped) {
  const int n0 = (int)c.g->n0;
  if (n0 <= 0) return GP_OK;
  double* A = c.head();
  KParams<double> kp = make_kparams<double>(*c.kern);
  dim3 bb(16, 16), bg((n0 + 15) / 16, (n0 + 15) / 16);
  GP_OK_OR_RETURN(head_build(c));
  if (n_carried == 2 * n0 && n_carried > 1) {
    if (c.g->dtype == GP_F64)
      head_carry_grad_init_kernel<double><<<bg, bb, 0, c.st>>>((const double*)c.g->x, c.g->d, n0, c.kern->kind, kp, A);
    else
      head_carry_grad_init_kernel<float><<<bg, bb, 0, c.st>>>((const float*)c.g->x, c.g->d, n0, c.kern->kind, kp, A);
    GP_LAUNCH_CHECK();
  } else if (n_carried > 0) {
    int mode = n_carried == 1 ? 1 : 2;
    int64_t total = mode == 1 ? n0 : (int64_t)n0 * n0;
    unsigned grid = (unsigned)((total + 255) / 256);
    if (c.g->dtype == GP_F64)
      head_carry_init_kernel<double><<<grid, 256, 0, c.st>>>((const double*)carried_src, n0, mode, A);
    else
      head_carry_init_kernel<float><<<grid, 256, 0, c.st>>>((const float*)carried_src, n0, mode, A);
    GP_LAUNCH_CHECK();
  }
  return head_chol(c, n_carried, overlapped);
}

// v_head = sigma * L xi_head  (one warp per row)
template <typename T>
__global__ void head_forward_kernel(const double* __restrict__ L, const T* __restrict__ xi, T* __restrict__ v,
                                    Rec<T>* rec, int n0, double sigma) {
  int r = blockIdx.x * (blockDim.x / 32) + threadIdx.x / 32;
  int lane = threadIdx.x & 31;
  if (r >= n0) return;
  double acc = 0.0;
  for (int cc = lane; cc <= r; cc += 32) acc = fma(L[(size_t)r * n0 + cc], (double)xi[cc], acc);
  acc = warp_sum(acc);
  if (lane == 0) {
    T out = (T)(sigma * acc);
    v[r] = out;
    if (rec) rec[r].v = out;
  }
}

gp_status head_forward(const OpCtx& c, const void* xi, void* v, void* rec, bool rec_is_packed) {
  const int n0 = (int)c.g->n0;
  if (n0 <= 0) return GP_OK;
  unsigned grid = (unsigned)((n0 + 3) / 4);
  if (c.g->dtype == GP_F64)
    head_forward_kernel<double><<<grid, 128, 0, c.st>>>(c.head(), (const double*)xi, (double*)v,
                                                      rec_is_packed ? (Rec<double>*)rec : nullptr, n0, c.kern->sigma);
  else
    head_forward_kernel<float><<<grid, 128, 0, c.st>>>(c.head(), (const float*)xi, (float*)v,
                                                     rec_is_packed ? (Rec<float>*)rec : nullptr, n0, c.kern->sigma);
  GP_LAUNCH_CHECK();
  return GP_OK;
}

template <typename T>
__global__ void head_inverse_out_kernel(const double* __restrict__ carried, T* __restrict__ xi, int n0, double inv_sigma) {
  int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i < n0) xi[i] = (T)(carried[i] * inv_sigma);
}

gp_status head_inverse_out(const OpCtx& c, void* xi) {
  const int n0 = (int)c.g->n0;
  if (n0 <= 0) return GP_OK;
  const double* carried = c.head() + (size_t)n0 * n0;
  unsigned grid = (unsigned)((n0 + 255) / 256);
  if (c.g->dtype == GP_F64)
    head_inverse_out_kernel<double><<<grid, 256, 0, c.st>>>(carried, (double*)xi, n0, 1.0 / c.kern->sigma);
  else
    head_inverse_out_kernel<float><<<grid, 256, 0, c.st>>>(carried, (float*)xi, n0, 1.0 / c.kern->sigma);
  GP_LAUNCH_CHECK();
  return GP_OK;
}

__global__ void head_logdet_kernel(const double* __restrict__ L, int n0, double sigma, double* acc) {
  __shared__ double red[32];
  double s = 0.0;
  for (int j = threadIdx.x; j < n0; j += blockDim.x) s += 2.0 * log(sigma * L[(size_t)j * n0 + j]);
  block_atomic_add(s, acc, red);
}

// tr(M^-1 D) = sum_{e,b} Linv[e][b] (Linv D)[e][b] = sum over the two carried blocks, element by element
__global__ void head_trace_kernel(const double* __restrict__ C1, const double* __restrict__ C2, int64_t total, double* acc) {
  __shared__ double red[32];
  double s = 0.0;
  for (int64_t e = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; e < total; e += (int64_t)gridDim.x * blockDim.x)
    s = fma(C1[e], C2[e], s);
  block_atomic_add(s, acc, red);
}

gp_status head_logdet(const OpCtx& c, double* acc, double* grad_ell_acc) {
  const int n0 = (int)c.g->n0;
  if (n0 <= 0) return GP_OK;
  head_logdet_kernel<<<1, 256, 0, c.st>>>(c.head(), n0, c.kern->sigma, acc);
  GP_LAUNCH_CHECK();
  if (grad_ell_acc) {
    const double* C1 = c.head() + (size_t)n0 * n0;
    const double* C2 = C1 + (size_t)n0 * n0;
    int64_t total = (int64_t)n0 * n0;
    unsigned grid = (unsigned)((total + 255) / 256);
    if (grid > 1184) grid = 1184;
    head_trace_kernel<<<grid, 256, 0, c.st>>>(C1, C2, total, grad_ell_acc);
    GP_LAUNCH_CHECK();
  }
  return GP_OK;
}

// ---- VJP through the head:  v_h = sigma L xi_h --------------------------------------------
//   p = L^T g_h;  xi_bar_h = sigma p;  sigma_bar += g_h . (L xi_h) = p . xi_h
//   L_bar = sigma tril(g_h xi_h^T);  M_bar = L^-T Phi(L^T L_bar) L^-1, Phi = lower triangle with the diagonal
//   halved;  L^T L_bar = sigma p xi^T on the lower part.  With T1 = Phi L^-1, i.e.
//     T1[a][b] = sigma p_a ( sum_{b' <= a} xi_b' Linv[b'][b]  -  xi_a Linv[a][b] / 2 ),
//   ell_bar = sum_ab M_bar_ab dM_ab/dell = sum_{a,b} T1[a][b] (Linv dM/dell)[a][b]: both factors come out of
//   the factorisation as carried rows (C1[b][a] = Linv[a][b], C2[b][a] = (Linv D)[a][b]), so no dense
//   triangular solve or GEMM is needed beyond the factorisation itself.
template <typename T>
__global__ void head_vjp_p_kernel(const double* __restrict__ L, const T* __restrict__ gbar, const T* __restrict__ xi,
                                  T* __restrict__ xibar, double* __restrict__ p, int n0, double sigma, double* acc_sigma) {
  __shared__ double red[32];
  int e = blockIdx.x * (blockDim.x / 32) + threadIdx.x / 32;   // one warp per column e
  int lane = threadIdx.x & 31;
  double contrib = 0.0;
  if (e < n0) {
    double s = 0.0;
    for (int a = e + lane; a < n0; a += 32) s = fma(L[(size_t)a * n0 + e], (double)gbar[a], s);
    s = warp_sum(s);
    if (lane == 0) {
      p[e] = s;
      xibar[e] = (T)(sigma * s);
      contrib = s * (double)xi[e];
    }
  }
  block_atomic_add(contrib, acc_sigma, red);
}

template <typename T>
__global__ void head_vjp_ell_kernel(const double* __restrict__ C1, const double* __restrict__ C2,
                                    const double* __restrict__ p, const T* __restrict__ xi, int n0, double sigma,
                                    double* acc_ell) {
  __shared__ double red[32];
  int b = blockIdx.x * (blockDim.x / 32) + threadIdx.x / 32;   // one warp per carried row b
  int lane = threadIdx.x & 31;
  double total = 0.0;
  if (b < n0) {
    const double* c1 = C1 + (size_t)b * n0;
    const double* c2 = C2 + (size_t)b * n0;
    double carry = 0.0;                                         // sum_{a' < chunk} xi_a' Linv[a'][b]
    for (int a0 = (b / 32) * 32; a0 < n0; a0 += 32) {          // Linv[a][b] = 0 for a < b
      int a = a0 + lane;
      double t = a < n0 ? (double)xi[a] * c1[a] : 0.0;
      double incl = t;
#pragma unroll
      for (int o = 1; o < 32; o <<= 1) {
        double up = __shfl_up_sync(0xffffffffu, incl, o);
        if (lane >= o) incl += up;
      }
      if (a < n0) total = fma(p[a] * (carry + incl - 0.5 * t), c2[a], total);
      carry += __shfl_sync(0xffffffffu, incl, 31);
    }
    total = warp_sum(total);
    if (lane != 0) total = 0.0;
  }
  block_atomic_add(sigma * total, acc_ell, red);
}

gp_status head_vjp(const OpCtx& c, const void* xi, const void* gbar, void* xibar, double* acc) {
  const int n0 = (int)c.g->n0;
  if (n0 <= 0) return GP_OK;
  const double* L = c.head();
  const double* C1 = L + (size_t)n0 * n0;
  const double* C2 = C1 + (size_t)n0 * n0;
  double* p = c.head() + (size_t)3 * n0 * n0;
  unsigned grid = (unsigned)((n0 + 3) / 4);
  if (c.g->dtype == GP_F64) {
    head_vjp_p_kernel<double><<<grid, 128, 0, c.st>>>(L, (const double*)gbar, (const double*)xi, (double*)xibar, p, n0, c.kern->sigma, acc);
    GP_LAUNCH_CHECK();
    head_vjp_ell_kernel<double><<<grid, 128, 0, c.st>>>(C1, C2, p, (const double*)xi, n0, c.kern->sigma, acc + 1);
  } else {
    head_vjp_p_kernel<float><<<grid, 128, 0, c.st>>>(L, (const float*)gbar, (const float*)xi, (float*)xibar, p, n0, c.kern->sigma, acc);
    GP_LAUNCH_CHECK();
    head_vjp_ell_kernel<float><<<grid, 128, 0, c.st>>>(C1, C2, p, (const float*)xi, n0, c.kern->sigma, acc + 1);
  }
  GP_LAUNCH_CHECK();
  return GP_OK;
}

}  // namespace gp
