// Forward / inverse / logdet kernels of the Vecchia conditioning path.
//   forward  Alg. 1 lines 2-8: ticketed dataflow launches over stretches of batches (forward_flow_kernel);
//            the literal launch per batch is kept behind GP_FLAG_PER_BATCH_LAUNCH and for the lane-group / generic shapes
//   inverse  PAPER.md:91: every point at once
//   logdet   PAPER.md:9:  sum_i log s_i^2, fp64 accumulation
#include <type_traits>
#include <vector>

#include "gp_cond_jit.cuh"
#include "gp_cond_lg.cuh"
#include "gp_cond_pk.cuh"

namespace gp {

enum { OPK_FORWARD = 0, OPK_INVERSE = 1, OPK_LOGDET = 2 };
constexpr int kCondThreads = 128;
#ifndef GP_COND_MIN_CTAS
#define GP_COND_MIN_CTAS 3
#endif
#ifndef GP_FLOW_MIN_CTAS
#define GP_FLOW_MIN_CTAS 3
#endif

// rec[i] = {x_i, vals_i or 0}
// "value not produced yet" marker of the dataflow forward: an all-ones NaN.  The kernels never write it
// (every NaN result is canonicalised to the quiet NaN 0x7fc0... first).
template <typename T> struct Pending;
template <> struct Pending<float> {
  static __device__ __forceinline__ float make() { return __uint_as_float(0xffffffffu); }
  static __device__ __forceinline__ bool is(float v) { return __float_as_uint(v) == 0xffffffffu; }
  static __device__ __forceinline__ float load(const float* p) {
    float v; asm volatile("ld.relaxed.gpu.global.f32 %0, [%1];" : "=f"(v) : "l"(p) : "memory"); return v;
  }
  static __device__ __forceinline__ void store(float* p, float v) {
    asm volatile("st.relaxed.gpu.global.f32 [%0], %1;" ::"l"(p), "f"(v) : "memory");
  }
};
template <> struct Pending<double> {
  static __device__ __forceinline__ double make() { return __longlong_as_double(-1LL); }
  static __device__ __forceinline__ bool is(double v) { return __double_as_longlong(v) == -1LL; }
  static __device__ __forceinline__ double load(const double* p) {
    double v; asm volatile("ld.relaxed.gpu.global.f64 %0, [%1];" : "=d"(v) : "l"(p) : "memory"); return v;
  }
  static __device__ __forceinline__ void store(double* p, double v) {
    asm volatile("st.relaxed.gpu.global.f64 [%0], %1;" ::"l"(p), "d"(v) : "memory");
  }
};

// rec[i] = {x_i, vals_i | 0 | pending}
template <typename T>
__global__ void pack_kernel(const T* __restrict__ x, const T* __restrict__ vals, Rec<T>* __restrict__ rec,
                            int64_t n, int d, int pending) {
  int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  Rec<T> r;
  r.x0 = x[i * d];
  r.x1 = d >= 2 ? x[i * d + 1] : T(0);
  r.x2 = d >= 3 ? x[i * d + 2] : T(0);
  r.v = vals ? vals[i] : (pending ? Pending<T>::make() : T(0));
  rec[i] = r;
}

template <typename T> __device__ __forceinline__ T quiet_nan();
template <> __device__ __forceinline__ float quiet_nan<float>() { return __int_as_float(0x7fc00000); }
template <> __device__ __forceinline__ double quiet_nan<double>() { return __longlong_as_double(0x7ff8000000000000LL); }

template <typename T, int K, int D, int KIND, int OP>
__global__ void __launch_bounds__(kCondThreads, GP_COND_MIN_CTAS)
cond_kernel(Rec<T>* __restrict__ rec, const int32_t* __restrict__ nbr, const T* __restrict__ in,
            T* __restrict__ out, int64_t start, int64_t end, int64_t n0, KParams<T> kp, JitParams jp, Control* ctrl) {
  __shared__ double red[32];
  int64_t i = start + (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  double ld = 0.0;
  if (i < end) {
    Rec<T> self = load_rec<false>(rec + i);
    Cond<T> c;
    if constexpr (std::is_same<T, float>::value && K % 2 == 0) {
      int32_t idx[K];
      Rec<T> R[K];
      gather_reg<T, K, false>(rec, nbr + (i - n0) * K, idx, R);
      c = condition_jit_rec<K, D, KIND>(R, self, kp, jp);
    } else {
      c = condition_reg<T, K, D, KIND, false>(rec, nbr + (i - n0) * K, self, kp);
    }
    T ss = kp.sigma * c.s;
    if (!c.ok) atomicAdd(&ctrl->n_bad, 1ULL);
    if (OP == OPK_FORWARD) {
      T v = Math<T>::fma(ss, in[i], c.m);
      if (!c.ok) v = quiet_nan<T>();
      out[i] = v;
      rec[i].v = v;
    } else if (OP == OPK_INVERSE) {
      T xi = (self.v - c.m) / ss;
      if (!c.ok) xi = quiet_nan<T>();
      out[i] = xi;
    } else {
      ld = c.ok ? 2.0 * (double)Math<T>::log(ss) : 0.0;
    }
  }
  if (OP == OPK_LOGDET) block_atomic_add(ld, &ctrl->acc[0], red);
}

// ---- lane-group kernel: one point per L lanes (k = 32 fp32, k = 16 fp64) -----------------------------------
template <typename T, int K, int D, int KIND, int L, int OP>
__global__ void __launch_bounds__(kCondThreads, sizeof(T) == 8 ? 4 : 3)
cond_lg_kernel(Rec<T>* __restrict__ rec, const int32_t* __restrict__ nbr, const T* __restrict__ in, T* __restrict__ out,
               int64_t start, int64_t end, int64_t n0, KParams<T> kp, Control* ctrl) {
  __shared__ double red[32];
  constexpr int PPB = kCondThreads / L;
  const int l = threadIdx.x % L;
  int64_t i = start + (int64_t)blockIdx.x * PPB + threadIdx.x / L;
  const bool live = i < end;
  if (!live) i = end - 1;                     // every lane takes part in the shuffles; the result is dropped
  LgCond<T> c = condition_lg<T, K, D, KIND, L, false>(rec, nbr + (i - n0) * K, i, l, kp);
  double ld = 0.0;
  if (live && l == 0) {
    const T ss = kp.sigma * c.s;
    if (!c.ok) atomicAdd(&ctrl->n_bad, 1ULL);
    if (OP == OPK_FORWARD) {
      T v = Math<T>::fma(ss, in[i], c.m);
      if (!c.ok) v = quiet_nan<T>();
      out[i] = v;
      rec[i].v = v;
    } else if (OP == OPK_INVERSE) {
      T xi = (c.self_v - c.m) / ss;
      if (!c.ok) xi = quiet_nan<T>();
      out[i] = xi;
    } else {
      ld = c.ok ? 2.0 * (double)Math<T>::log(ss) : 0.0;
    }
  }
  if (OP == OPK_LOGDET) block_atomic_add(ld, &ctrl->acc[0], red);
}

// Dataflow forward for the lane-group shapes (wait-last body only): CTAs take BATCH-ALIGNED chunks of PPB points
// through a ticket - the groups of one warp then belong to one batch and never wait on each other, so the
// full-mask shuffles cannot deadlock - weights first, then every lane polls the values of its own rows.
template <typename T, int K, int D, int KIND, int L>
__global__ void __launch_bounds__(kCondThreads, 3)
lg_flow_kernel(Rec<T>* rec, const int32_t* __restrict__ nbr, const T* __restrict__ xi, T* __restrict__ out,
               const longlong4* __restrict__ tab, int nb, unsigned long long* ticket, int64_t n0, KParams<T> kp,
               Control* ctrl) {
  constexpr int PPB = kCondThreads / L;
  constexpr int S = LgShape<T, K, L>::S;
  __shared__ long long s_info[3];
  __shared__ long long s_ticket;
  if (threadIdx.x == 0) s_ticket = (long long)atomicAdd(ticket, 1ULL);
  __syncthreads();
  {
    const long long t = s_ticket;
    for (int q = threadIdx.x; q < nb; q += blockDim.x) {
      const longlong2 e01 = __ldg(reinterpret_cast<const longlong2*>(tab + q));
      const longlong2 e23 = __ldg(reinterpret_cast<const longlong2*>(tab + q) + 1);
      if (e01.x <= t && t < e23.y) {   // {first chunk, rounds << 40 | first point, end point, end chunk} of batch q
        const long long rounds = e01.y >> 40, first = e01.y & ((1LL << 40) - 1);
        s_info[0] = first + (t - e01.x) * PPB * rounds;
        s_info[1] = e23.x;
        s_info[2] = rounds;
      }
    }
  }
  __syncthreads();
  const int l = threadIdx.x % L;
  const int64_t end = s_info[1];
  // a ticket covers `rounds` consecutive groups of PPB points of ONE batch (large batches: the ticket and the table
  // lookup are amortised; small batches: rounds = 1, every point gets its own CTA slot at once)
  for (int rd = 0; rd < (int)s_info[2]; ++rd) {
  int64_t i = s_info[0] + (int64_t)rd * PPB + threadIdx.x / L;
  if (s_info[0] + (int64_t)rd * PPB >= end) break;
  const bool live = i < end;
  if (!live) i = end - 1;                     // every lane takes part in the shuffles; the result is dropped
  const int32_t* row = nbr + (i - n0) * K;
  T w[S], s;
  bool ok;
  weights_lg<T, K, D, KIND, L, true>(rec, row, i, l, kp, w, s, ok);
  // values of the own rows: all loads in flight first, then poll only what is still pending
  T vv[S];
#pragma unroll
  for (int q = 0; q < S; ++q) vv[q] = (q * L + l < K) ? Pending<T>::load(&rec[row[q * L + l]].v) : T(0);
  {
    bool missing = false;
#pragma unroll
    for (int q = 0; q < S; ++q) missing |= Pending<T>::is(vv[q]);
    const long long t0 = clock64();
    unsigned spins = 0;
    while (missing) {
      missing = false;
#pragma unroll
      for (int q = 0; q < S; ++q) {
        if (Pending<T>::is(vv[q])) {
          vv[q] = Pending<T>::load(&rec[row[q * L + l]].v);
          missing |= Pending<T>::is(vv[q]);
        }
      }
      if (!missing) break;
      if (++spins > 8) __nanosleep(spins > 64 ? 256 : 32);
      if ((spins & 1023u) == 0 && clock64() - t0 > 8000000000LL) {   // watchdog: a bug, never expected
        atomicAdd(&ctrl->timeout, 1ULL);
        ok = false;
        break;
      }
    }
  }
  T part = T(0);
#pragma unroll
  for (int q = 0; q < S; ++q) part = Math<T>::fma(w[q], vv[q], part);
  const T m = group_sum(part, L);
  int oki = ok ? 1 : 0;                       // a lane's watchdog may have fired: AND over the group
  for (int o = L >> 1; o > 0; o >>= 1) oki &= __shfl_xor_sync(0xffffffffu, oki, o, L);
  ok = oki != 0;
  if (live && l == 0) {
    T v = Math<T>::fma(kp.sigma * s, xi[i], m);
    if (!ok) atomicAdd(&ctrl->n_bad, 1ULL);
    if (!ok || v != v) v = quiet_nan<T>();
    out[i] = v;
    Pending<T>::store(&rec[i].v, v);
  }
  }
}

// ---- dataflow forward: ONE launch for all batches (Alg. 1 lines 2-8) --------------------
// Every point i >= n0 is one thread.  CTAs take chunks of the graph order through a ticket, so a chunk with a
// lower number has always started: its threads are resident and depend only on still earlier chunks, hence
// polling cannot deadlock.  A thread first does everything that does not depend on values (indices,
// coordinates, K, its factor, the weights w and s), then waits until the k neighbour values are no longer
// "pending", and applies  v_i = w . v_c + sigma s xi_i.  In steady state the neighbours were produced long
// ago and the first gather already returns them; only at the frontier (and in the small early batches, where
// the per-batch latency chain of a launch-per-batch loop is what costs) does a thread poll.  The value word
// is its own ready flag, so no fence or counter is involved.
//
// Two bodies share the scheme.  FLOW_WEIGHTS (above) is for the stretches of SMALL batches, where the chain of
// dependent batches is what costs: the wait comes last, after all the arithmetic.  FLOW_CARRY is for the
// stretches of LARGE batches (larger than what the GPU holds in flight, so a neighbour is almost never
// pending): it waits first - almost always zero iterations - and then runs exactly the inverse's body, values
// row carried through the factorisation, no back-substitution.  The host cuts the graph
// order into such stretches (at batch boundaries) and launches one kernel per stretch; tickets keep counting
// across launches, `chunk0` is the number handed out before this launch.
enum { FLOW_WEIGHTS = 0, FLOW_CARRY = 1 };

template <typename T, int K>
__device__ __forceinline__ bool wait_values(Rec<T>* rec, const int32_t (&idx)[K], T (&vv)[K], Control* ctrl) {
  bool missing = false;
#pragma unroll
  for (int j = 0; j < K; ++j) missing |= Pending<T>::is(vv[j]);
  if (!missing) return true;
  const long long t0 = clock64();
  unsigned spins = 0;
  while (true) {
    missing = false;
#pragma unroll
    for (int j = 0; j < K; ++j) {
      if (Pending<T>::is(vv[j])) {
        vv[j] = Pending<T>::load(&rec[idx[j]].v);
        missing |= Pending<T>::is(vv[j]);
      }
    }
    if (!missing) return true;
    if (++spins > 8) __nanosleep(spins > 64 ? 256 : 32);
    if ((spins & 1023u) == 0 && clock64() - t0 > 8000000000LL) {   // watchdog (about 4 s): a bug, never expected
      atomicAdd(&ctrl->timeout, 1ULL);
      return false;
    }
  }
}

// one entry per 128-point group of the graph order: {first point, end of its batch}
__global__ void flow_groups_kernel(const longlong2* __restrict__ btab, int L, longlong2* __restrict__ gtab, long long groups) {
  const long long g = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (g >= groups) return;
  int lo = 0, hi = L;                               // largest b in [0, L) with btab[b].x <= g
  while (hi - lo > 1) {
    const int mid = (lo + hi) >> 1;
    if (__ldg(&btab[mid]).x <= g) lo = mid; else hi = mid;
  }
  const longlong2 e = __ldg(&btab[lo]);
  gtab[g] = make_longlong2(e.y + (g - e.x) * (long long)kCondThreads, __ldg(&btab[lo + 1]).y);
}

template <typename T, int K, int D, int KIND, int MODE>
__global__ void __launch_bounds__(kCondThreads, GP_FLOW_MIN_CTAS)
forward_flow_kernel(Rec<T>* rec, const int32_t* __restrict__ nbr, const T* __restrict__ xi, T* __restrict__ out,
                    int64_t n0, const longlong2* __restrict__ gtab, unsigned long long* ticket,
                    KParams<T> kp, JitParams jp, Control* ctrl) {
  // CTAs take 128-point groups of this launch through `ticket`, so a group with a lower number has always started:
  // its threads are resident and depend only on still earlier groups, hence polling cannot deadlock.
  // gtab[t] = {first point, end of its batch}: groups are BATCH-ALIGNED, so the lanes of a warp belong to one batch
  // and never wait on one another (points of a batch are conditionally independent): the polling does
  // not lean on independent thread scheduling.  (A persistent variant that draws the next ticket and table entry
  // while the current group is computed was measured: 2.33 ms against 2.24 ms for the large batches.)
  __shared__ long long s_first, s_end;
  if (threadIdx.x == 0) {
    const long long t = (long long)atomicAdd(ticket, 1ULL);
    const longlong2 e = __ldg(&gtab[t]);
    s_first = e.x;
    s_end = e.y;
  }
  __syncthreads();
  const int64_t i = s_first + threadIdx.x;
  if (i >= s_end) return;
  Cond<T> c;
  T m = T(0);
  const int32_t* row = nbr + (i - n0) * K;
  if (MODE == FLOW_CARRY) {
    Rec<T> self = load_rec_l1(rec + i);
    int32_t idx[K];
    Rec<T> R[K];
    T vv[K];
    load_row<K>(row, idx);
#pragma unroll
    for (int j = 0; j < K; ++j) R[j] = load_rec_l1(rec + idx[j]);
#pragma unroll
    for (int j = 0; j < K; ++j) vv[j] = R[j].v;
    bool got = wait_values<T, K>(rec, idx, vv, ctrl);
#pragma unroll
    for (int j = 0; j < K; ++j) R[j].v = vv[j];
    if constexpr (std::is_same<T, float>::value && K % 2 == 0) {
      c = condition_jit_rec<K, D, KIND>(R, self, kp, jp);
    } else {
      T A[(K + 1) * (K + 2) / 2];
      build_joint_reg<T, K, D, KIND>(R, self, kp, A);
      c = factor_joint_reg<T, K, false>(A, vv, kp);
    }
    c.ok = c.ok && got;
    m = c.m;
  } else {
    T w[K];
    {
      Rec<T> self = load_rec_l1(rec + i);
      int32_t idx[K];
      Rec<T> R[K];
      load_row<K>(row, idx);
#pragma unroll
      for (int j = 0; j < K; ++j) R[j] = load_rec_l1(rec + idx[j]);
      if constexpr (std::is_same<T, float>::value && K % 2 == 0) c = weights_pk<K, D, KIND>(R, self, kp, w);
      else c = weights_reg<T, K, D, KIND>(R, self, kp, w);
    }
    // values: read again now (the lines are in L1 from the gather above; a stale "pending" is re-read from L2)
    T vv[K];
    int32_t idx[K];
    load_row<K>(row, idx);
#pragma unroll
    for (int j = 0; j < K; ++j) vv[j] = load_val_l1(&rec[idx[j]].v);
    bool got = wait_values<T, K>(rec, idx, vv, ctrl);
    c.ok = c.ok && got;
    m = T(0);
#pragma unroll
    for (int j = 0; j < K; ++j) m = Math<T>::fma(w[j], vv[j], m);
  }
  T v = Math<T>::fma(kp.sigma * c.s, xi[i], m);
  if (!c.ok) atomicAdd(&ctrl->n_bad, 1ULL);
  if (!c.ok || v != v) v = quiet_nan<T>();
  out[i] = v;
  Pending<T>::store(&rec[i].v, v);
}

template <typename T, int OP>
__global__ void cond_generic_kernel(const T* __restrict__ x, const T* vals, const int32_t* __restrict__ nbr,
                                    const T* in, T* out, int64_t start, int64_t end, int64_t n0, int d, int k,
                                    int kind, KParams<T> kp, Control* ctrl, int active) {
  extern __shared__ double smem_raw[];
  __shared__ double red[32];
  int tid = threadIdx.x;
  int64_t i = start + (int64_t)blockIdx.x * active + tid;
  double ld = 0.0;
  if (tid < active && i < end) {
    Scratch<T> A{reinterpret_cast<T*>(smem_raw) + tid, active};
    Cond<T> c = condition_generic<T>(x, OP == OPK_LOGDET ? nullptr : vals, d, k, kind, nbr + (i - n0) * k, i, kp, A);
    T ss = kp.sigma * c.s;
    if (!c.ok) atomicAdd(&ctrl->n_bad, 1ULL);
    if (OP == OPK_FORWARD) {
      T v = Math<T>::fma(ss, in[i], c.m);
      if (!c.ok) v = quiet_nan<T>();
      out[i] = v;
    } else if (OP == OPK_INVERSE) {
      T xi = (in[i] - c.m) / ss;
      if (!c.ok) xi = quiet_nan<T>();
      out[i] = xi;
    } else {
      ld = c.ok ? 2.0 * (double)Math<T>::log(ss) : 0.0;
    }
  }
  if (OP == OPK_LOGDET) block_atomic_add(ld, &ctrl->acc[0], red);
}

// Threads of a generic block that own a scratch column (the block is padded to a multiple of 32).
int generic_active_threads(int k, size_t elem_bytes, bool with_vjp) {
  size_t per = (size_t)generic_scratch_elems(k, with_vjp) * elem_bytes;
  size_t budget = 200 * 1024;
  size_t a = budget / per;
  if (a > 128) a = 128;
  if (a >= 32) a = a / 32 * 32;
  if (a < 1) a = 1;
  return (int)a;
}

// ---- specialisation table ------------------------------------------------------------------------
// (dtype, K, D) triples with a register-resident kernel; every KIND is instantiated for each.
#define GP_SPEC_TABLE(X) \
  X(float, 8, 3) X(float, 16, 3) X(float, 8, 2) X(float, 16, 2) X(double, 8, 3) X(double, 8, 2)

// (dtype, K, D, L): lane-group kernels
#define GP_LG_TABLE(X) X(float, 32, 2, 8) X(float, 32, 3, 8) X(double, 16, 3, 4) X(double, 16, 2, 4)

bool has_specialised(int dtype, int k, int d, int kind) {
  if (kind < 0 || kind > 2) return false;
#define X(T, K, D, L) \
  if ((dtype == GP_F64) == (sizeof(T) == 8) && k == K && d == D) return true;
  GP_LG_TABLE(X)
#undef X
#define X(T, K, D) \
  if ((dtype == GP_F64) == (sizeof(T) == 8) && k == K && d == D) return true;
  GP_SPEC_TABLE(X)
#undef X
  return false;
}

template <typename T, int K, int D, int OP>
static gp_status launch_spec_kind(const OpCtx& c, const T* in, T* out, int64_t start, int64_t end) {
  int64_t cnt = end - start;
  if (cnt <= 0) return GP_OK;
  unsigned grid = (unsigned)((cnt + kCondThreads - 1) / kCondThreads);
  KParams<T> kp = make_kparams<T>(*c.kern);
  const JitParams jp = make_jit_params(*c.kern);
  Rec<T>* rec = (Rec<T>*)c.rec();
  switch (c.kern->kind) {
    case GP_KERNEL_SE:
      cond_kernel<T, K, D, GP_KERNEL_SE, OP><<<grid, kCondThreads, 0, c.st>>>(rec, c.g->nbr, in, out, start, end, c.g->n0, kp, jp, c.ctrl());
      break;
    case GP_KERNEL_MATERN32:
      cond_kernel<T, K, D, GP_KERNEL_MATERN32, OP><<<grid, kCondThreads, 0, c.st>>>(rec, c.g->nbr, in, out, start, end, c.g->n0, kp, jp, c.ctrl());
      break;
    default:
      cond_kernel<T, K, D, GP_KERNEL_EXP, OP><<<grid, kCondThreads, 0, c.st>>>(rec, c.g->nbr, in, out, start, end, c.g->n0, kp, jp, c.ctrl());
      break;
  }
  GP_LAUNCH_CHECK();
  return GP_OK;
}

template <typename T, int K, int D, int L, int OP>
static gp_status launch_lg(const OpCtx& c, const T* in, T* out, int64_t start, int64_t end) {
  int64_t cnt = end - start;
  if (cnt <= 0) return GP_OK;
  constexpr int PPB = kCondThreads / L;
  unsigned grid = (unsigned)((cnt + PPB - 1) / PPB);
  KParams<T> kp = make_kparams<T>(*c.kern);
  Rec<T>* rec = (Rec<T>*)c.rec();
  switch (c.kern->kind) {
    case GP_KERNEL_SE:
      cond_lg_kernel<T, K, D, GP_KERNEL_SE, L, OP><<<grid, kCondThreads, 0, c.st>>>(rec, c.g->nbr, in, out, start, end, c.g->n0, kp, c.ctrl());
      break;
    case GP_KERNEL_MATERN32:
      cond_lg_kernel<T, K, D, GP_KERNEL_MATERN32, L, OP><<<grid, kCondThreads, 0, c.st>>>(rec, c.g->nbr, in, out, start, end, c.g->n0, kp, c.ctrl());
      break;
    default:
      cond_lg_kernel<T, K, D, GP_KERNEL_EXP, L, OP><<<grid, kCondThreads, 0, c.st>>>(rec, c.g->nbr, in, out, start, end, c.g->n0, kp, c.ctrl());
      break;
  }
  GP_LAUNCH_CHECK();
  return GP_OK;
}

template <typename T, int OP>
static gp_status launch_generic(const OpCtx& c, const T* vals, const T* in, T* out, int64_t start, int64_t end) {
  int64_t cnt = end - start;
  if (cnt <= 0) return GP_OK;
  int k = c.g->k;
  int active = generic_active_threads(k, sizeof(T), false);
  int threads = (active + 31) / 32 * 32;
  size_t smem = (size_t)generic_scratch_elems(k, false) * sizeof(T) * active;
  // a per-device attribute: set on every launch (cheap next to this kernel) rather than cached per process
  GP_CUDA_OK(cudaFuncSetAttribute(cond_generic_kernel<T, OP>, cudaFuncAttributeMaxDynamicSharedMemorySize, 220 * 1024));
  unsigned grid = (unsigned)((cnt + active - 1) / active);
  KParams<T> kp = make_kparams<T>(*c.kern);
  cond_generic_kernel<T, OP><<<grid, threads, smem, c.st>>>((const T*)c.g->x, vals, c.g->nbr, in, out, start, end,
                                                          c.g->n0, c.g->d, k, c.kern->kind, kp, c.ctrl(), active);
  GP_LAUNCH_CHECK();
  return GP_OK;
}

static bool use_spec(const OpCtx& c) {
  if (c.g->flags & GP_FLAG_GENERIC_KERNEL) return false;
  if (!has_specialised(c.g->dtype, c.g->k, c.g->d, c.kern->kind)) return false;
  return (((uintptr_t)c.g->nbr) & 15) == 0;  // vectorised index loads need 16 B alignment
}

template <typename T, int OP>
static gp_status launch_range(const OpCtx& c, bool spec, const T* vals, const T* in, T* out, int64_t start, int64_t end) {
  if (spec) {
#define X(TT, K, D) \
    if constexpr (std::is_same<TT, T>::value) {                    \
      if (c.g->k == K && c.g->d == D) return launch_spec_kind<T, K, D, OP>(c, in, out, start, end); \
    }
    GP_SPEC_TABLE(X)
#undef X
#define X(TT, K, D, L) \
    if constexpr (std::is_same<TT, T>::value) {                    \
      if (c.g->k == K && c.g->d == D) return launch_lg<T, K, D, L, OP>(c, in, out, start, end); \
    }
    GP_LG_TABLE(X)
#undef X
  }
  return launch_generic<T, OP>(c, vals, in, out, start, end);
}

template <typename T>
static gp_status pack(const OpCtx& c, const T* vals, bool pending = false, int64_t lo = 0, int64_t hi = -1) {
  if (hi < 0) hi = c.g->n;
  const int64_t cnt = hi - lo;
  if (cnt <= 0) return GP_OK;
  unsigned grid = (unsigned)((cnt + 255) / 256);
  pack_kernel<T><<<grid, 256, 0, c.st>>>((const T*)c.g->x + lo * c.g->d, vals ? vals + lo : nullptr, (Rec<T>*)c.rec() + lo, cnt,
                                         c.g->d, pending ? 1 : 0);
  GP_LAUNCH_CHECK();
  return GP_OK;
}

// ranges of the graph order for the host-buffer variants: about kHostChunks pieces, the first starting at 0
constexpr int kHostChunks = 4;

// grad = d/d(sigma, ell):  every point contributes log sigma^2 + log s_i^2, so d/dsigma = 2 N / sigma exactly;
// acc[2] holds ell * d/dell (gp_vjp.cu).
__global__ void finalize_logdet_kernel(const Control* ctrl, double* logdet, double* grad, double two_n_over_sigma,
                                       double inv_ell) {
  if (threadIdx.x == 0 && blockIdx.x == 0) {
    logdet[0] = ctrl->acc[0];
    if (grad) { grad[0] = two_n_over_sigma; grad[1] = ctrl->acc[2] * inv_ell; }
  }
}

// host-buffer forward: xi[0 : cut) has arrived when the first kernel starts, the rest when `arrived_rest` fires; v leaves
// stretch by stretch on the copy-out stream
struct ForwardPipe {
  int64_t cut;
  cudaEvent_t arrived_rest;
  EventBag* bag;
  bool waited;
};
static int64_t forward_pipe_cut(const OpCtx& c) {
  // first batch boundary past an eighth of the conditioned points, or the first batch larger than twice what the GPU
  // holds in flight (where launch_flow starts its large-batch stretch), whichever comes first
  const int L = c.g->n_batches;
  const int64_t* off = c.g->batch_off;
  const int64_t n = c.g->n, n0 = c.g->n0;
  const int64_t large = 2 * (int64_t)device_sm_count() * GP_FLOW_MIN_CTAS * kCondThreads;
  for (int b = 0; b < L; ++b)
    if (off[b + 1] - off[b] >= large || off[b] - n0 >= (n - n0) / 8) return off[b];
  return n;
}

template <typename T, int K, int D, int MODE>
static gp_status launch_flow_segment(const OpCtx& c, const T* xi, T* v, int64_t group0, int64_t groups, int slot) {
  if (groups <= 0) return GP_OK;
  if (groups > 0x7fffffffLL) return GP_ERR_UNSUPPORTED;
  unsigned grid = (unsigned)groups;
  KParams<T> kp = make_kparams<T>(*c.kern);
  const JitParams jp = make_jit_params(*c.kern);
  Rec<T>* rec = (Rec<T>*)c.rec();
  const longlong2* gtab = (const longlong2*)c.gtab() + group0;
  unsigned long long* ticket = &c.ctrl()->flow_ticket[slot];
  switch (c.kern->kind) {
    case GP_KERNEL_SE:
      forward_flow_kernel<T, K, D, GP_KERNEL_SE, MODE><<<grid, kCondThreads, 0, c.st>>>(rec, c.g->nbr, xi, v, c.g->n0, gtab, ticket, kp, jp, c.ctrl());
      break;
    case GP_KERNEL_MATERN32:
      forward_flow_kernel<T, K, D, GP_KERNEL_MATERN32, MODE><<<grid, kCondThreads, 0, c.st>>>(rec, c.g->nbr, xi, v, c.g->n0, gtab, ticket, kp, jp, c.ctrl());
      break;
    default:
      forward_flow_kernel<T, K, D, GP_KERNEL_EXP, MODE><<<grid, kCondThreads, 0, c.st>>>(rec, c.g->nbr, xi, v, c.g->n0, gtab, ticket, kp, jp, c.ctrl());
      break;
  }
  GP_LAUNCH_CHECK();
  return GP_OK;
}

// Cut the graph order into stretches of small and of large batches (see forward_flow_kernel) and launch each with its
// own ticket counter.  The per-batch table {first group, first point} goes to the workspace (pageable source: staged
// by the runtime before the copy call returns); flow_groups_kernel expands it to one entry per 128-point group.
template <typename T, int K, int D>
static gp_status launch_flow(const OpCtx& c, const T* xi, T* v, ForwardPipe* fp) {
  const int L = c.g->n_batches;
  if (L <= 0) return GP_OK;
  const int64_t* off = c.g->batch_off;
  const int sms = device_sm_count();
  if (sms <= 0) return GP_ERR_CUDA;
  const int64_t in_flight = (int64_t)sms * GP_FLOW_MIN_CTAS * kCondThreads;   // points the GPU holds at once
  const int64_t large = 2 * in_flight;
  std::vector<int64_t> tab(2 * ((size_t)L + 1));
  int64_t groups = 0;
  for (int b = 0; b < L; ++b) {
    tab[2 * b] = groups;
    tab[2 * b + 1] = off[b];
    groups += (off[b + 1] - off[b] + kCondThreads - 1) / kCondThreads;
  }
  tab[2 * L] = groups;
  tab[2 * L + 1] = off[L];
  GP_CUDA_OK(cudaMemcpyAsync(c.boff_dev(), tab.data(), tab.size() * sizeof(int64_t), cudaMemcpyHostToDevice, c.st));
  flow_groups_kernel<<<(unsigned)((groups + 255) / 256), 256, 0, c.st>>>((const longlong2*)c.boff_dev(), L,
                                                                        (longlong2*)c.gtab(), groups);
  GP_LAUNCH_CHECK();
  int b = 0, slot = 0;
  while (b < L) {
    auto is_big = [&](int q) {
      if (c.g->flags & GP_FLAG_FLOW_CARRY) return true;
      if (c.g->flags & GP_FLAG_FLOW_WEIGHTS) return false;
      return off[q + 1] - off[q] >= large;
    };
    const bool big = is_big(b);
    int e = b + 1;
    // the last ticket counter takes everything that is left (the wait-last body is right for any batch size)
    if (slot == kFlowTickets - 1) e = L;
    else while (e < L && is_big(e) == big && !(fp && big && off[e] - off[b] >= (c.g->n - c.g->n0) / 5)) ++e;
    if (fp && !fp->waited && off[e] > fp->cut) {              // this stretch reads xi beyond what has arrived
      GP_CUDA_OK(cudaStreamWaitEvent(c.st, fp->arrived_rest, 0));
      fp->waited = true;
    }
    const int64_t g0 = tab[2 * b], ng = tab[2 * e] - tab[2 * b];
    if (big && slot != kFlowTickets - 1) GP_OK_OR_RETURN((launch_flow_segment<T, K, D, FLOW_CARRY>(c, xi, v, g0, ng, slot)));
    else GP_OK_OR_RETURN((launch_flow_segment<T, K, D, FLOW_WEIGHTS>(c, xi, v, g0, ng, slot)));
    if (fp) {                                                 // v of this stretch (and of the head) goes home
      const int64_t lo = b == 0 ? 0 : off[b], hi = off[e];
      GP_OK_OR_RETURN(stream_after(*fp->bag, c.io->cout, c.st));
      GP_CUDA_OK(cudaMemcpyAsync((T*)c.io->out_host + lo, v + lo, (size_t)(hi - lo) * sizeof(T), cudaMemcpyDeviceToHost, c.io->cout));
    }
    b = e;
    ++slot;
  }
  return GP_OK;
}

// Lane-group shapes: the wait-last dataflow body costs about twice the arithmetic of the plain per-point body (the
// back-substitution runs on group-wide shuffles), so it pays only where the chain of dependent batches is what costs.
// Stretches of SMALL batches go through lg_flow_kernel (one launch per stretch, own ticket counter), every LARGE batch
// (at least one wave of CTAs) is one plain launch of cond_lg_kernel.  Measured, config 4 (k = 32, 651 batches):
// a launch per batch 30.4 ms, dataflow everywhere 37.8 ms, this split 28.3 ms; config 2 fp64: 3.24 / 2.72 / 2.49 ms.
template <typename T, int K, int D, int L>
static gp_status launch_lg_flow(const OpCtx& c, const T* xi, T* v) {
  const int nb = c.g->n_batches;
  if (nb <= 0) return GP_OK;
  constexpr int PPB = kCondThreads / L;
  const int64_t* off = c.g->batch_off;
  const int sms = device_sm_count();
  if (sms <= 0) return GP_ERR_CUDA;
  const int64_t resident = (int64_t)sms * 3;   // CTAs the GPU holds at once
  const int64_t large = resident * PPB;        // one full wave; measured flat between 1 and 4 waves, worse beyond
  auto is_big = [&](int q) {
    if (c.g->flags & GP_FLAG_FLOW_WEIGHTS) return false;
    return off[q + 1] - off[q] >= large;
  };
  struct Stretch { int b, e; bool big; int64_t chunks; };
  std::vector<Stretch> plan;
  std::vector<int64_t> tab(4 * (size_t)nb);    // per batch {first chunk, rounds << 40 | first point, end point, end chunk}
  for (int b = 0; b < nb;) {
    const bool big = is_big(b);
    int e = b + 1;
    if ((int)plan.size() >= kFlowTickets - 1 && !big) e = nb;   // the last ticket counter takes everything that is left
    else if (!big) while (e < nb && !is_big(e)) ++e;
    int64_t chunks = 0;
    if (!big) {
      for (int q = b; q < e; ++q) {              // chunk numbers restart with every stretch
        const int64_t cnt = off[q + 1] - off[q];
        int64_t rounds = cnt / (2 * resident * PPB);   // keep at least two waves of tickets per batch
        rounds = rounds < 1 ? 1 : (rounds > 8 ? 8 : rounds);
        const int64_t nc = (cnt + PPB * rounds - 1) / (PPB * rounds);
        tab[4 * q + 0] = chunks;
        tab[4 * q + 1] = (rounds << 40) | off[q];
        tab[4 * q + 2] = off[q + 1];
        tab[4 * q + 3] = chunks + nc;
        chunks += nc;
      }
      if (chunks > 0x7fffffffLL) return GP_ERR_UNSUPPORTED;
    }
    plan.push_back({b, e, big, chunks});
    b = e;
  }
  // pageable source: the runtime stages it before returning, so the vector may die afterwards
  GP_CUDA_OK(cudaMemcpyAsync(c.boff_dev(), tab.data(), tab.size() * sizeof(int64_t), cudaMemcpyHostToDevice, c.st));
  KParams<T> kp = make_kparams<T>(*c.kern);
  Rec<T>* rec = (Rec<T>*)c.rec();
  int slot = 0;
  for (const Stretch& s : plan) {
    if (s.big) {
      GP_OK_OR_RETURN((launch_range<T, OPK_FORWARD>(c, true, v, xi, v, off[s.b], off[s.e])));
      continue;
    }
    const longlong4* tab_d = (const longlong4*)c.boff_dev() + s.b;
    const int cnt = s.e - s.b;
    unsigned long long* ticket = &c.ctrl()->flow_ticket[slot < kFlowTickets ? slot : kFlowTickets - 1];
    ++slot;
    switch (c.kern->kind) {
      case GP_KERNEL_SE:
        lg_flow_kernel<T, K, D, GP_KERNEL_SE, L><<<(unsigned)s.chunks, kCondThreads, 0, c.st>>>(rec, c.g->nbr, xi, v, tab_d, cnt, ticket, c.g->n0, kp, c.ctrl());
        break;
      case GP_KERNEL_MATERN32:
        lg_flow_kernel<T, K, D, GP_KERNEL_MATERN32, L><<<(unsigned)s.chunks, kCondThreads, 0, c.st>>>(rec, c.g->nbr, xi, v, tab_d, cnt, ticket, c.g->n0, kp, c.ctrl());
        break;
      default:
        lg_flow_kernel<T, K, D, GP_KERNEL_EXP, L><<<(unsigned)s.chunks, kCondThreads, 0, c.st>>>(rec, c.g->nbr, xi, v, tab_d, cnt, ticket, c.g->n0, kp, c.ctrl());
        break;
    }
    GP_LAUNCH_CHECK();
  }
  return GP_OK;
}

template <typename T>
static gp_status forward_t(const OpCtx& c, const T* xi, T* v) {
  bool spec = use_spec(c);
  bool flow = false;                          // single-launch dataflow: one-thread-per-point shapes only
  if (spec && !(c.g->flags & GP_FLAG_PER_BATCH_LAUNCH)) {
#define X(TT, K, D) \
    if (std::is_same<TT, T>::value && c.g->k == K && c.g->d == D) flow = true;
    GP_SPEC_TABLE(X)
#undef X
    // lane-group shapes: dataflow launches for the stretches of small batches, a plain launch per large batch
#define X(TT, K, D, L) \
    if (std::is_same<TT, T>::value && c.g->k == K && c.g->d == D) flow = true;
    GP_LG_TABLE(X)
#undef X
  }
  GP_CUDA_OK(cudaMemsetAsync(c.ctrl(), 0, kCtrlBytes, c.st));
  EventBag bag;
  ForwardPipe pipe{c.g->n, nullptr, &bag, false};
  if (c.io) {   // host-buffer variant: xi arrives in two parts on the copy-in stream
    const int64_t n = c.g->n;
    pipe.cut = forward_pipe_cut(c);
    GP_OK_OR_RETURN(stream_after(bag, c.io->cin, c.st));
    GP_CUDA_OK(cudaMemcpyAsync((T*)xi, c.io->in_host[0], (size_t)pipe.cut * sizeof(T), cudaMemcpyHostToDevice, c.io->cin));
    GP_OK_OR_RETURN(stream_after(bag, c.st, c.io->cin));
    if (pipe.cut < n)
      GP_CUDA_OK(cudaMemcpyAsync((T*)xi + pipe.cut, (const T*)c.io->in_host[0] + pipe.cut, (size_t)(n - pipe.cut) * sizeof(T),
                                 cudaMemcpyHostToDevice, c.io->cin));
    pipe.arrived_rest = bag.make();
    if (!pipe.arrived_rest) return GP_ERR_CUDA;
    GP_CUDA_OK(cudaEventRecord(pipe.arrived_rest, c.io->cin));
  }
  ForwardPipe* fp = c.io ? &pipe : nullptr;
  // the head is on the critical path (every batch depends on it); packing the records is not: side stream
  SideStream* side = nullptr;
  GP_OK_OR_RETURN(side_stream(&side));
  if (spec) {
    GP_OK_OR_RETURN(side_fork(side, c.st));
    OpCtx pc = c;
    pc.st = side->stream;
    GP_OK_OR_RETURN(pack<T>(pc, nullptr, flow));
  }
  GP_OK_OR_RETURN(head_factor(c, nullptr, 0));
  if (spec) GP_OK_OR_RETURN(side_join(side, c.st));
  GP_OK_OR_RETURN(head_forward(c, xi, v, c.rec(), spec));
  GP_OK_OR_RETURN(ktime_begin(c.st));
  if (flow) {
#define X(TT, K, D) \
    if constexpr (std::is_same<TT, T>::value) {                    \
      if (c.g->k == K && c.g->d == D) {                            \
        GP_OK_OR_RETURN((launch_flow<T, K, D>(c, xi, v, fp)));     \
        GP_OK_OR_RETURN(ktime_end(c.st));                          \
        if (fp) GP_OK_OR_RETURN(stream_after(bag, c.st, c.io->cout)); \
        return GP_OK;                                              \
      }                                                            \
    }
    GP_SPEC_TABLE(X)
#undef X
#define X(TT, K, D, L) \
    if constexpr (std::is_same<TT, T>::value) {                    \
      if (c.g->k == K && c.g->d == D) {                            \
        if (fp) GP_CUDA_OK(cudaStreamWaitEvent(c.st, fp->arrived_rest, 0)); \
        GP_OK_OR_RETURN((launch_lg_flow<T, K, D, L>(c, xi, v)));   \
        GP_OK_OR_RETURN(ktime_end(c.st));                          \
        if (fp) GP_CUDA_OK(cudaMemcpyAsync(c.io->out_host, v, (size_t)c.g->n * sizeof(T), cudaMemcpyDeviceToHost, c.st)); \
        return GP_OK;                                              \
      }                                                            \
    }
    GP_LG_TABLE(X)
#undef X
  }
  const int64_t* off = c.g->batch_off;
  if (fp) GP_CUDA_OK(cudaStreamWaitEvent(c.st, fp->arrived_rest, 0));
  for (int b = 0; b < c.g->n_batches; ++b)
    GP_OK_OR_RETURN((launch_range<T, OPK_FORWARD>(c, spec, v, xi, v, off[b], off[b + 1])));
  GP_OK_OR_RETURN(ktime_end(c.st));
  if (fp) GP_CUDA_OK(cudaMemcpyAsync(c.io->out_host, v, (size_t)c.g->n * sizeof(T), cudaMemcpyDeviceToHost, c.st));
  return GP_OK;
}

template <typename T>
static gp_status inverse_t(const OpCtx& c, const T* v, T* xi) {
  bool spec = use_spec(c);
  const int64_t n = c.g->n, n0 = c.g->n0;
  GP_CUDA_OK(cudaMemsetAsync(c.ctrl(), 0, kCtrlBytes, c.st));
  EventBag bag;
  // host-buffer variant: v arrives range by range (a point reads only points before it), xi leaves range by range
  const int chunks = c.io ? kHostChunks : 1;
  int64_t cut[kHostChunks + 1];
  for (int q = 0; q <= chunks; ++q) cut[q] = q == 0 ? 0 : (q == chunks ? n : n0 + (n - n0) * q / chunks);
  cudaEvent_t arrived[kHostChunks] = {};
  if (c.io) {
    GP_OK_OR_RETURN(stream_after(bag, c.io->cin, c.st));       // the staging buffer may still be read by earlier work
    for (int q = 0; q < chunks; ++q) {
      GP_CUDA_OK(cudaMemcpyAsync((T*)v + cut[q], (const T*)c.io->in_host[0] + cut[q], (size_t)(cut[q + 1] - cut[q]) * sizeof(T),
                                 cudaMemcpyHostToDevice, c.io->cin));
      arrived[q] = bag.make();
      if (!arrived[q]) return GP_ERR_CUDA;
      GP_CUDA_OK(cudaEventRecord(arrived[q], c.io->cin));
    }
  }
  // the head (xi[0:n0]) and the bulk (xi[n0:n]) are independent: head on the side stream, submitted first
  SideStream* side = nullptr;
  GP_OK_OR_RETURN(side_stream(&side));
  if (c.io) GP_CUDA_OK(cudaStreamWaitEvent(c.st, arrived[0], 0));
  GP_OK_OR_RETURN(side_fork(side, c.st));
  OpCtx hc = c;
  hc.st = side->stream;
  GP_OK_OR_RETURN(head_factor(hc, v, 1, true));
  GP_OK_OR_RETURN(head_inverse_out(hc, xi));
  GP_OK_OR_RETURN(ktime_begin(c.st));
  for (int q = 0; q < chunks; ++q) {
    if (c.io && q > 0) GP_CUDA_OK(cudaStreamWaitEvent(c.st, arrived[q], 0));
    if (spec) GP_OK_OR_RETURN(pack<T>(c, v, false, cut[q], cut[q + 1]));
    GP_OK_OR_RETURN((launch_range<T, OPK_INVERSE>(c, spec, v, v, xi, cut[q] < n0 ? n0 : cut[q], cut[q + 1])));
    if (q == 0) GP_OK_OR_RETURN(side_join(side, c.st));
    if (c.io) {
      GP_OK_OR_RETURN(stream_after(bag, c.io->cout, c.st));
      GP_CUDA_OK(cudaMemcpyAsync((T*)c.io->out_host + cut[q], xi + cut[q], (size_t)(cut[q + 1] - cut[q]) * sizeof(T),
                                 cudaMemcpyDeviceToHost, c.io->cout));
    }
  }
  GP_OK_OR_RETURN(ktime_end(c.st));
  if (c.io) GP_OK_OR_RETURN(stream_after(bag, c.st, c.io->cout));   // the caller's stream ends when the result is on the host
  return GP_OK;
}

template <typename T>
static gp_status logdet_t(const OpCtx& c, double* logdet, double* grad) {
  bool spec = use_spec(c);
  GP_CUDA_OK(cudaMemsetAsync(c.ctrl(), 0, kCtrlBytes, c.st));
  SideStream* side = nullptr;
  GP_OK_OR_RETURN(side_stream(&side));
  GP_OK_OR_RETURN(side_fork(side, c.st));
  OpCtx hc = c;
  hc.st = side->stream;
  GP_OK_OR_RETURN(head_factor(hc, nullptr, grad ? 2 * (int)c.g->n0 : 0, true));
  GP_OK_OR_RETURN(head_logdet(hc, &c.ctrl()->acc[0], grad ? &c.ctrl()->acc[2] : nullptr));
  if (spec) GP_OK_OR_RETURN(pack<T>(c, nullptr));
  GP_OK_OR_RETURN(ktime_begin(c.st));
  GP_OK_OR_RETURN((launch_range<T, OPK_LOGDET>(c, spec, nullptr, nullptr, nullptr, c.g->n0, c.g->n)));
  GP_OK_OR_RETURN(ktime_end(c.st));
  if (grad) GP_OK_OR_RETURN(run_logdet_grad(c));
  GP_OK_OR_RETURN(side_join(side, c.st));
  finalize_logdet_kernel<<<1, 32, 0, c.st>>>(c.ctrl(), logdet, grad, 2.0 * (double)c.g->n / c.kern->sigma,
                                             1.0 / c.kern->ell);
  GP_LAUNCH_CHECK();
  return GP_OK;
}

gp_status run_forward(const OpCtx& c, const void* xi, void* v) {
  if (c.g->k > kMaxKGrad) return run_large(c, GP_OP_FORWARD, xi, v, nullptr);
  return c.g->dtype == GP_F64 ? forward_t<double>(c, (const double*)xi, (double*)v)
                              : forward_t<float>(c, (const float*)xi, (float*)v);
}
gp_status run_inverse(const OpCtx& c, const void* v, void* xi) {
  if (c.g->k > kMaxKGrad) return run_large(c, GP_OP_INVERSE, v, xi, nullptr);
  return c.g->dtype == GP_F64 ? inverse_t<double>(c, (const double*)v, (double*)xi)
                              : inverse_t<float>(c, (const float*)v, (float*)xi);
}
gp_status run_logdet(const OpCtx& c, double* logdet, double* grad) {
  if (c.g->k > kMaxKGrad) return grad ? GP_ERR_UNSUPPORTED : run_large(c, GP_OP_LOGDET, nullptr, nullptr, logdet);
  return c.g->dtype == GP_F64 ? logdet_t<double>(c, logdet, grad) : logdet_t<float>(c, logdet, grad);
}

}  // namespace gp
