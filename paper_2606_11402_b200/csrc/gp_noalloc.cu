// gp_logdet_noalloc: the log-determinant (sum_i log s_i^2 + log det K_head, Eq. 2 / PAPER.md:30-31 for
// s_i^2) for callers that cannot allocate device memory - code under CUDA graph capture, tight serving loops, harnesses
// that forbid cudaMalloc.  Every other entry point takes a caller-allocated workspace; this one takes none: its scratch
// (the n0 x n0 matrix of the dense head, Alg. 1 line 1 / PAPER.md:66, and the accumulators of the sum over points) is
// the file-scope device array below, of a fixed modest size, resident on every GPU that loads the library until the
// process exits.  Hence the limits n0 <= kNaMaxN0, k <= kNaMaxK; larger sizes are rejected (GP_ERR_TOO_LARGE).
//
// The call launches kernels and one cudaMemsetAsync on the caller's stream and nothing else: no cudaMalloc / cudaFree,
// no stream or event creation, no library that allocates.  All calls share the array and it keeps the last call's
// contents; what must start at zero (the accumulators) is cleared at the start of every call.  Two calls that overlap
// on the GPU (different streams, or different host threads on one device) RACE on it: callers serialise them.
//
// The bulk kernel is a variant of the large-k logdet kernel (gp_large.cu): fp64 whatever the working dtype, the joint
// (k + 1) x (k + 1) triangle in shared memory, here one WARP per point and any k <= 64.  This is a convenience path,
// about an order of magnitude slower than gp_logdet's register kernels; it changes no existing code path.
#include <mutex>

#include "gp_cond.cuh"

namespace gp {

constexpr int kNaMaxN0 = 1024;
constexpr int kNaMaxK = 64;
constexpr int kNaCtrlBytes = 4096;
constexpr size_t kNaScratchBytes = (size_t)kNaCtrlBytes + (size_t)kNaMaxN0 * kNaMaxN0 * sizeof(double);   // 8 MiB + 4 KiB

// In HOST code this name is a host-side stand-in, not a device address: the host passes kernels the pointer that
// cudaGetSymbolAddress returns (na_scratch_ptr below), never the name.
static __device__ __align__(256) unsigned char g_na_scratch[kNaScratchBytes];

struct NaControl {
  double slots[kAccSlots];        // partial sums of log s_i^2 over the conditioned points (spread: no single hot address)
  double head;                    // log det K_head
  unsigned long long n_bad;       // pivots that were not positive (head or conditionals)
};
static_assert(sizeof(NaControl) <= kNaCtrlBytes, "control block of the no-alloc scratch");

constexpr int kNaNB = 32;         // panel width of the head factorisation

// ---- dense head in the scratch matrix A [n0][n0] (row-major, lower triangle used), unit sigma ----------------------
template <typename T>
__global__ void na_head_build_kernel(const T* __restrict__ x, int d, int n0, int kind, KParams<double> kp,
                                     double* __restrict__ A) {
  const int64_t e = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (e >= (int64_t)n0 * n0) return;
  const int r = (int)(e / n0), c = (int)(e % n0);
  if (c > r) return;
  double v = kp.diag;
  if (c < r) {
    double d2 = 0.0;
    for (int t = 0; t < d; ++t) { const double dx = (double)x[(int64_t)r * d + t] - (double)x[(int64_t)c * d + t]; d2 = fma(dx, dx, d2); }
    v = rho_rt<double>(kind, d2 * kp.qscale);
  }
  A[e] = v;
}

// one warp: Cholesky of the nb x nb diagonal block at (j0, j0), in place; adds its part of log det (sigma^2 M)
__global__ void __launch_bounds__(32)
na_head_diag_kernel(double* __restrict__ A, int n0, int j0, int nb, double sigma, NaControl* ctl) {
  __shared__ double S[kNaNB][kNaNB + 1];
  const int lane = threadIdx.x;
  for (int c = 0; c < nb; ++c) S[lane][c] = (lane < nb && c <= lane) ? A[(size_t)(j0 + lane) * n0 + j0 + c] : 0.0;
  __syncwarp();
  double ld = 0.0;
  bool bad = false;
  for (int j = 0; j < nb; ++j) {
    const double piv = S[j][j];
    bad |= !(piv > 0.0);
    const double ljj = sqrt(piv);
    __syncwarp();
    if (lane == j) { S[j][j] = ljj; ld = 2.0 * log(sigma * ljj); }
    if (lane > j && lane < nb) S[lane][j] /= ljj;
    __syncwarp();
    if (lane > j && lane < nb) {
      const double lrj = S[lane][j];
      for (int c = j + 1; c <= lane; ++c) S[lane][c] = fma(-lrj, S[c][j], S[lane][c]);
    }
    __syncwarp();
  }
  for (int c = 0; c < nb; ++c)
    if (lane < nb && c <= lane) A[(size_t)(j0 + lane) * n0 + j0 + c] = S[lane][c];
  for (int o = 16; o > 0; o >>= 1) ld += __shfl_xor_sync(0xffffffffu, ld, o);
  if (lane == 0) {
    if (bad) atomicAdd(&ctl->n_bad, 1ULL);
    else atomicAdd(&ctl->head, ld);
  }
}

// rows below the diagonal block: L[r][j0 : j0 + nb] = A[r][j0 : j0 + nb] L_diag^-T, one thread per row
__global__ void __launch_bounds__(128)
na_head_solve_kernel(double* __restrict__ A, int n0, int j0, int nb) {
  __shared__ double Ld[kNaNB][kNaNB + 1];
  __shared__ double R[128][kNaNB + 1];
  for (int e = threadIdx.x; e < nb * nb; e += blockDim.x) Ld[e / nb][e % nb] = A[(size_t)(j0 + e / nb) * n0 + j0 + e % nb];
  const int r = j0 + nb + blockIdx.x * blockDim.x + threadIdx.x;
  if (r < n0)
    for (int j = 0; j < nb; ++j) R[threadIdx.x][j] = A[(size_t)r * n0 + j0 + j];
  __syncthreads();
  if (r >= n0) return;
  for (int j = 0; j < nb; ++j) {
    double a = R[threadIdx.x][j];
    for (int t = 0; t < j; ++t) a = fma(-R[threadIdx.x][t], Ld[j][t], a);
    a /= Ld[j][j];
    R[threadIdx.x][j] = a;
    A[(size_t)r * n0 + j0 + j] = a;
  }
}

// trailing update, lower-triangle tiles of 32 x 32:  A[r][c] -= sum_j L[r][j0 + j] L[c][j0 + j],  r, c >= j0 + nb
__global__ void __launch_bounds__(256)
na_head_update_kernel(double* __restrict__ A, int n0, int j0, int nb) {
  if (blockIdx.x > blockIdx.y) return;                 // tile column <= tile row
  __shared__ double Lr[kNaNB][kNaNB + 1], Lc[kNaNB][kNaNB + 1];
  const int base = j0 + nb, r0 = base + blockIdx.y * kNaNB, c0 = base + blockIdx.x * kNaNB;
  for (int e = threadIdx.x; e < kNaNB * kNaNB; e += blockDim.x) {
    const int a = e / kNaNB, j = e % kNaNB;
    Lr[a][j] = (r0 + a < n0 && j < nb) ? A[(size_t)(r0 + a) * n0 + j0 + j] : 0.0;
    Lc[a][j] = (c0 + a < n0 && j < nb) ? A[(size_t)(c0 + a) * n0 + j0 + j] : 0.0;
  }
  __syncthreads();
  const int tc = threadIdx.x % kNaNB;
  for (int tr = threadIdx.x / kNaNB; tr < kNaNB; tr += 256 / kNaNB) {
    const int r = r0 + tr, c = c0 + tc;
    if (r >= n0 || c > r) continue;
    double acc = 0.0;
    for (int j = 0; j < kNaNB; ++j) acc = fma(Lr[tr][j], Lc[tc][j], acc);
    A[(size_t)r * n0 + c] -= acc;
  }
}

// ---- conditioned points: one warp per point, joint triangle in shared memory ---------------------------------------
// Local index 0 is the point itself, 1..k its neighbours; entry (a, b), a <= b, lives at b (b + 1) / 2 + a.  The
// elimination runs from b = k down to 1 (the point itself last, as in Alg. 1 where it is row k + 1):
// with this numbering the trailing matrix of every step is the PREFIX [0, m (m + 1) / 2) of the array and the scaled
// column the m entries behind it, so the lanes sweep a contiguous range; pa / pb map a prefix position to (a, b).
// After the last step entry 0 is s_i^2 = K_ii - K_ic K_cc^-1 K_ci in unit sigma (Eq. 2).
constexpr int kNaWarps = 4;

__host__ __device__ inline int na_tri(int k) { return (k + 1) * (k + 2) / 2; }
__host__ inline size_t na_cond_smem(int k, int d) {
  return (size_t)kNaWarps * ((size_t)na_tri(k) + (size_t)(k + 1) * d) * sizeof(double) + 2 * (size_t)na_tri(k);
}

template <typename T>
__global__ void __launch_bounds__(kNaWarps * 32)
na_cond_logdet_kernel(const T* __restrict__ x, const int32_t* __restrict__ nbr, int64_t n0, int64_t n, int d, int k,
                      int kind, KParams<double> kp, NaControl* ctl) {
  extern __shared__ double na_smem[];
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const int NT = na_tri(k);
  double* A = na_smem + (size_t)warp * (NT + (k + 1) * d);
  double* X = A + NT;                                               // [k + 1][d]
  unsigned char* pa = reinterpret_cast<unsigned char*>(na_smem + (size_t)kNaWarps * (NT + (k + 1) * d));
  unsigned char* pb = pa + NT;
  for (int b = threadIdx.x; b <= k; b += blockDim.x)
    for (int a = 0; a <= b; ++a) { pa[b * (b + 1) / 2 + a] = (unsigned char)a; pb[b * (b + 1) / 2 + a] = (unsigned char)b; }
  __syncthreads();
  double sum = 0.0;
  unsigned long long bad = 0;
  for (int64_t i = n0 + (int64_t)blockIdx.x * kNaWarps + warp; i < n; i += (int64_t)gridDim.x * kNaWarps) {
    const int32_t* row = nbr + (i - n0) * k;
    for (int q = lane; q <= k; q += 32) {
      const int64_t p = q == 0 ? i : (int64_t)row[q - 1];
      for (int t = 0; t < d; ++t) X[q * d + t] = (double)x[p * d + t];
    }
    __syncwarp();
    for (int e = lane; e < NT; e += 32) {
      const int a = pa[e], b = pb[e];
      double v = kp.diag;
      if (a != b) {
        double d2 = 0.0;
        for (int t = 0; t < d; ++t) { const double dx = X[a * d + t] - X[b * d + t]; d2 = fma(dx, dx, d2); }
        v = rho_rt<double>(kind, d2 * kp.qscale);
      }
      A[e] = v;
    }
    __syncwarp();
    double minpiv = kp.diag;
    for (int m = k; m >= 1; --m) {
      const int P = m * (m + 1) / 2;                                // prefix = trailing matrix; column m behind it
      double* col = A + P;
      const double piv = col[m];
      minpiv = fmin(minpiv, piv);
      const double inv = 1.0 / sqrt(piv);
      for (int a = lane; a < m; a += 32) col[a] *= inv;
      __syncwarp();
      for (int e = lane; e < P; e += 32) A[e] = fma(-col[pa[e]], col[pb[e]], A[e]);
      __syncwarp();
    }
    const double s2 = A[0];
    minpiv = fmin(minpiv, s2);
    const bool ok = minpiv > 0.0 && s2 < 1e300;
    if (ok) sum += log(kp.sigma * kp.sigma * s2);
    else ++bad;
    __syncwarp();                                                   // A and X are rewritten by the next point
  }
  if (lane == 0) {
    atomicAdd(&ctl->slots[(blockIdx.x * kNaWarps + warp) % kAccSlots], sum);
    if (bad) atomicAdd(&ctl->n_bad, bad);
  }
}

// logdet = head + the slots; NaN if any pivot was not positive (this entry point has no workspace to query afterwards)
__global__ void na_finalize_kernel(const NaControl* ctl, double* __restrict__ logdet) {
  if (threadIdx.x != 0 || blockIdx.x != 0) return;
  double a = ctl->head;
  for (int q = 0; q < kAccSlots; ++q) a += ctl->slots[q];
  *logdet = ctl->n_bad ? __longlong_as_double(0x7ff8000000000000LL) : a;
}

// ---- host side ----------------------------------------------------------------------------------------------------
// Device address of the scratch array, taken ONCE PER DEVICE with that device current (cudaGetSymbolAddress answers
// for the current device); the shared-memory opt-in of the bulk kernel is set at the same time.
constexpr int kNaMaxDevices = 64;
static gp_status na_scratch_ptr(unsigned char** out) {
  static std::mutex mu;
  static unsigned char* ptr[kNaMaxDevices] = {};
  int dev = 0;
  GP_CUDA_OK(cudaGetDevice(&dev));
  if (dev < 0 || dev >= kNaMaxDevices) return GP_ERR_UNSUPPORTED;
  std::lock_guard<std::mutex> lock(mu);
  if (!ptr[dev]) {
    unsigned char* p = nullptr;
    GP_CUDA_OK(cudaGetSymbolAddress((void**)&p, g_na_scratch));
    if (!p) return GP_ERR_CUDA;
    const int smem_max = (int)na_cond_smem(kNaMaxK, kMaxD);
    GP_CUDA_OK(cudaFuncSetAttribute(na_cond_logdet_kernel<float>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem_max));
    GP_CUDA_OK(cudaFuncSetAttribute(na_cond_logdet_kernel<double>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem_max));
    ptr[dev] = p;
  }
  *out = ptr[dev];
  return GP_OK;
}

template <typename T>
static gp_status logdet_noalloc_t(const gp_graph* g, const gp_kernel* kern, double* logdet_dev, cudaStream_t st) {
  unsigned char* scratch = nullptr;
  GP_OK_OR_RETURN(na_scratch_ptr(&scratch));
  NaControl* ctl = reinterpret_cast<NaControl*>(scratch);
  double* A = reinterpret_cast<double*>(scratch + kNaCtrlBytes);
  const int n0 = (int)g->n0, d = g->d, k = g->k;
  const KParams<double> kp = make_kparams<double>(*kern);
  const T* x = (const T*)g->x;
  GP_CUDA_OK(cudaMemsetAsync(ctl, 0, kNaCtrlBytes, st));           // the accumulators must start at zero
  if (n0 > 0) {
    na_head_build_kernel<T><<<(unsigned)(((int64_t)n0 * n0 + 255) / 256), 256, 0, st>>>(x, d, n0, kern->kind, kp, A);
    GP_LAUNCH_CHECK();
    for (int j0 = 0; j0 < n0; j0 += kNaNB) {
      const int nb = n0 - j0 < kNaNB ? n0 - j0 : kNaNB;
      na_head_diag_kernel<<<1, 32, 0, st>>>(A, n0, j0, nb, kern->sigma, ctl);
      GP_LAUNCH_CHECK();
      const int rest = n0 - j0 - nb;
      if (rest <= 0) break;
      na_head_solve_kernel<<<(rest + 127) / 128, 128, 0, st>>>(A, n0, j0, nb);
      GP_LAUNCH_CHECK();
      const unsigned tiles = (unsigned)((rest + kNaNB - 1) / kNaNB);
      na_head_update_kernel<<<dim3(tiles, tiles), 256, 0, st>>>(A, n0, j0, nb);
      GP_LAUNCH_CHECK();
    }
  }
  if (g->n > g->n0) {
    const int sms = device_sm_count();
    if (sms <= 0) return GP_ERR_CUDA;
    const int64_t want = (g->n - g->n0 + kNaWarps - 1) / kNaWarps;
    const int64_t cap = (int64_t)sms * 16;
    na_cond_logdet_kernel<T><<<(unsigned)(want < cap ? want : cap), kNaWarps * 32, na_cond_smem(k, d), st>>>(
        x, g->nbr, g->n0, g->n, d, k, kern->kind, kp, ctl);
    GP_LAUNCH_CHECK();
  }
  na_finalize_kernel<<<1, 32, 0, st>>>(ctl, logdet_dev);
  GP_LAUNCH_CHECK();
  return GP_OK;
}

}  // namespace gp

extern "C" {

size_t gp_logdet_noalloc_scratch_bytes(void) { return gp::kNaScratchBytes; }

gp_status gp_logdet_noalloc(const gp_graph* g, const gp_kernel* kern, double* logdet_dev, void* cuda_stream) {
  if (!g || !kern || !logdet_dev) return GP_ERR_INVALID_ARG;
  gp_status vs = gp::validate_graph(g, kern);
  if (vs != GP_OK) return vs;
  if (g->n0 > gp::kNaMaxN0 || g->k > gp::kNaMaxK) return GP_ERR_TOO_LARGE;
  cudaStream_t st = (cudaStream_t)cuda_stream;
  return g->dtype == GP_F64 ? gp::logdet_noalloc_t<double>(g, kern, logdet_dev, st)
                            : gp::logdet_noalloc_t<float>(g, kern, logdet_dev, st);
}

}  // extern "C"
