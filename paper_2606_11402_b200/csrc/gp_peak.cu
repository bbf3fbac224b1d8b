// gp_measure_alu_peak: non-tensor ALU rates of the current device, measured with register-resident loops.
// SURVEY.md §8(d) asks for the FP32 / FP64 non-tensor peak "measured with a register-resident FMA loop under the same
// clocks"; bench.py prints these numbers (roofline.peak_measured) beside the nominal peak that roofline.frac uses.
// Every variant is the instruction shape one of the conditioning kernels leans on, so the numbers also say which
// pipe bounds them:
//   FFMA      scalar fma, three register operands                     (lane-group and fp64-free scalar code)
//   FFMA_IMM  scalar fma with an immediate addend                     (Horner steps with literal coefficients)
//   FFMA2     packed fma.rn.f32x2, three register-pair operands       (K build of the packed kernels)
//   FFMA2_BC  packed fma with one scalar operand broadcast to both halves, accumulator updated in place
//             (the right-/left-looking Cholesky update  P[rp][c] -= P[rp][j] * L[c][j])
//   DFMA      double fma                                              (fp64 kernels, dense head)
//   MUFU      ex2.approx                                              (one per pair in rho / gamma)
//   FFMA2_DFMA, FFMA2_MUFU  two pipes fed from one instruction stream (does the second pipe come for free?)
#include "gp_cond_pk.cuh"

namespace gp {

constexpr int kPeakThreads = 256;
constexpr int kPeakChains = 8;
constexpr int kPeakInner = 16;   // unrolled steps per loop trip; every step touches all chains

template <int V>
__global__ void __launch_bounds__(kPeakThreads)
peak_kernel(float* __restrict__ sink, int trips, float a, float b, double da, double db) {
  const float t0 = (float)threadIdx.x * 1e-3f;
  float acc = 0.0f;
  if constexpr (V == GP_PEAK_FFMA) {
    float x[kPeakChains], y[kPeakChains], z[kPeakChains];
#pragma unroll
    for (int i = 0; i < kPeakChains; ++i) { x[i] = t0 + i; y[i] = a + t0 * i; z[i] = b - t0 * i; }
#pragma unroll 1
    for (int t = 0; t < trips; ++t) {
#pragma unroll
      for (int s = 0; s < kPeakInner; ++s) {
#pragma unroll
        for (int i = 0; i < kPeakChains; ++i) x[i] = fmaf(x[i], y[(i + s) % kPeakChains], z[(i + 3 * s) % kPeakChains]);
      }
    }
#pragma unroll
    for (int i = 0; i < kPeakChains; ++i) acc += x[i];
  } else if constexpr (V == GP_PEAK_FFMA_IMM) {
    float x[kPeakChains], y[kPeakChains];                  // a Horner step: p = fma(t, p, literal)
#pragma unroll
    for (int i = 0; i < kPeakChains; ++i) { x[i] = t0 + i; y[i] = a + t0 * i; }
#pragma unroll 1
    for (int t = 0; t < trips; ++t) {
#pragma unroll
      for (int s = 0; s < kPeakInner; ++s) {
#pragma unroll
        for (int i = 0; i < kPeakChains; ++i) x[i] = fmaf(y[i], x[i], 0.33333334f);
      }
    }
#pragma unroll
    for (int i = 0; i < kPeakChains; ++i) acc += x[i];
  } else if constexpr (V == GP_PEAK_FFMA2) {
    f2 x[kPeakChains], y[kPeakChains], z[kPeakChains];
#pragma unroll
    for (int i = 0; i < kPeakChains; ++i) {
      x[i] = make_float2(t0 + i, t0 - i);
      y[i] = make_float2(a + t0 * i, a - t0 * i);
      z[i] = make_float2(b + t0 * i, b - t0 * i);
    }
#pragma unroll 1
    for (int t = 0; t < trips; ++t) {
#pragma unroll
      for (int s = 0; s < kPeakInner; ++s) {
#pragma unroll
        for (int i = 0; i < kPeakChains; ++i) x[i] = fma2(x[i], y[(i + s) % kPeakChains], z[(i + 3 * s) % kPeakChains]);
      }
    }
#pragma unroll
    for (int i = 0; i < kPeakChains; ++i) acc += x[i].x + x[i].y;
  } else if constexpr (V == GP_PEAK_FFMA2_BC) {
    // x[i] -= y[i] * bc(l[s]): the Cholesky trailing update (accumulator in place, scalar broadcast operand)
    f2 x[kPeakChains], y[kPeakChains];
    float l[4];
#pragma unroll
    for (int i = 0; i < kPeakChains; ++i) { x[i] = make_float2(t0 + i, t0 - i); y[i] = make_float2(a + t0 * i, a - t0 * i); }
#pragma unroll
    for (int i = 0; i < 4; ++i) l[i] = b + t0 * i;
#pragma unroll 1
    for (int t = 0; t < trips; ++t) {
#pragma unroll
      for (int s = 0; s < kPeakInner; ++s) {
#pragma unroll
        for (int i = 0; i < kPeakChains; ++i) x[i] = fma2(neg2(y[i]), bc(l[s % 4]), x[i]);
      }
    }
#pragma unroll
    for (int i = 0; i < kPeakChains; ++i) acc += x[i].x + x[i].y;
  } else if constexpr (V == GP_PEAK_DFMA) {
    double x[kPeakChains];
#pragma unroll
    for (int i = 0; i < kPeakChains; ++i) x[i] = (double)t0 + i;
#pragma unroll 1
    for (int t = 0; t < trips; ++t) {
#pragma unroll
      for (int s = 0; s < kPeakInner; ++s) {
#pragma unroll
        for (int i = 0; i < kPeakChains; ++i) x[i] = fma(x[i], da, db);
      }
    }
#pragma unroll
    for (int i = 0; i < kPeakChains; ++i) acc += (float)x[i];
  } else if constexpr (V == GP_PEAK_MUFU) {
    float x[kPeakChains];
#pragma unroll
    for (int i = 0; i < kPeakChains; ++i) x[i] = -t0 - i;
#pragma unroll 1
    for (int t = 0; t < trips; ++t) {
#pragma unroll
      for (int s = 0; s < kPeakInner; ++s) {
#pragma unroll
        for (int i = 0; i < kPeakChains; ++i) x[i] = Math<float>::ex2(x[i]);
      }
    }
#pragma unroll
    for (int i = 0; i < kPeakChains; ++i) acc += x[i];
  } else if constexpr (V == GP_PEAK_FFMA2_DFMA) {
    // per step: kPeakChains packed fmas and kPeakChains / 2 double fmas
    f2 x[kPeakChains], y[kPeakChains];
    double w[kPeakChains / 2];
#pragma unroll
    for (int i = 0; i < kPeakChains; ++i) { x[i] = make_float2(t0 + i, t0 - i); y[i] = make_float2(a + t0 * i, a - t0 * i); }
#pragma unroll
    for (int i = 0; i < kPeakChains / 2; ++i) w[i] = (double)t0 + i;
#pragma unroll 1
    for (int t = 0; t < trips; ++t) {
#pragma unroll
      for (int s = 0; s < kPeakInner; ++s) {
#pragma unroll
        for (int i = 0; i < kPeakChains; ++i) {
          x[i] = fma2(x[i], y[(i + s) % kPeakChains], bc(b));
          if (i % 2 == 0) w[i / 2] = fma(w[i / 2], da, db);
        }
      }
    }
#pragma unroll
    for (int i = 0; i < kPeakChains; ++i) acc += x[i].x + x[i].y;
#pragma unroll
    for (int i = 0; i < kPeakChains / 2; ++i) acc += (float)w[i];
  } else if constexpr (V == GP_PEAK_FFMA2_MUFU) {
    // per step: kPeakChains packed fmas and kPeakChains / 4 MUFU.EX2
    f2 x[kPeakChains], y[kPeakChains];
    float w[kPeakChains / 4];
#pragma unroll
    for (int i = 0; i < kPeakChains; ++i) { x[i] = make_float2(t0 + i, t0 - i); y[i] = make_float2(a + t0 * i, a - t0 * i); }
#pragma unroll
    for (int i = 0; i < kPeakChains / 4; ++i) w[i] = -t0 - i;
#pragma unroll 1
    for (int t = 0; t < trips; ++t) {
#pragma unroll
      for (int s = 0; s < kPeakInner; ++s) {
#pragma unroll
        for (int i = 0; i < kPeakChains; ++i) {
          x[i] = fma2(x[i], y[(i + s) % kPeakChains], bc(b));
          if (i % 4 == 0) w[i / 4] = Math<float>::ex2(w[i / 4]);
        }
      }
    }
#pragma unroll
    for (int i = 0; i < kPeakChains; ++i) acc += x[i].x + x[i].y;
#pragma unroll
    for (int i = 0; i < kPeakChains / 4; ++i) acc += w[i];
  }
  if (acc == 123.456f) sink[0] = acc;   // never true in practice: keeps the loops alive
}

// lane-operations per thread per loop trip, and flop per lane-operation
static void peak_shape(int v, double* ops_per_trip, double* flop_per_op) {
  const double base = (double)kPeakInner * kPeakChains;
  switch (v) {
    case GP_PEAK_FFMA: case GP_PEAK_FFMA_IMM: case GP_PEAK_DFMA: *ops_per_trip = base; *flop_per_op = 2; break;
    case GP_PEAK_FFMA2: case GP_PEAK_FFMA2_BC: *ops_per_trip = 2 * base; *flop_per_op = 2; break;
    case GP_PEAK_MUFU: *ops_per_trip = base; *flop_per_op = 1; break;
    case GP_PEAK_FFMA2_DFMA: *ops_per_trip = 2 * base + base / 2; *flop_per_op = 2; break;
    default: *ops_per_trip = 2 * base; *flop_per_op = 2; break;   // FFMA2_MUFU: the packed fmas only are counted
  }
}

template <int V>
static gp_status run_peak(double* out, cudaStream_t st, float* sink, int sms) {
  const int trips = 4096;
  const int grid = sms * 8;
  cudaEvent_t e0, e1;
  GP_CUDA_OK(cudaEventCreate(&e0));
  GP_CUDA_OK(cudaEventCreate(&e1));
  peak_kernel<V><<<grid, kPeakThreads, 0, st>>>(sink, trips / 8, 1.0001f, 0.5f, 1.0001, 0.5);   // warm-up
  GP_LAUNCH_CHECK();
  double best = 1e30;
  for (int rep = 0; rep < 3; ++rep) {
    GP_CUDA_OK(cudaEventRecord(e0, st));
    peak_kernel<V><<<grid, kPeakThreads, 0, st>>>(sink, trips, 1.0001f, 0.5f, 1.0001, 0.5);
    GP_LAUNCH_CHECK();
    GP_CUDA_OK(cudaEventRecord(e1, st));
    GP_CUDA_OK(cudaEventSynchronize(e1));
    float ms = 0.f;
    GP_CUDA_OK(cudaEventElapsedTime(&ms, e0, e1));
    if (ms < best) best = ms;
  }
  cudaEventDestroy(e0);
  cudaEventDestroy(e1);
  double ops, fl;
  peak_shape(V, &ops, &fl);
  *out = ops * fl * (double)trips * (double)grid * kPeakThreads / (best * 1e-3) / 1e12;
  return GP_OK;
}

}  // namespace gp

using namespace gp;

extern "C" gp_status gp_measure_alu_peak(double* out_host, int32_t n_out, void* ws, size_t ws_bytes, void* cuda_stream) {
  if (!out_host || n_out < 1) return GP_ERR_INVALID_ARG;
  if (!ws || ws_bytes < 256) return GP_ERR_WORKSPACE;
  int dev = 0, sms = 0;
  GP_CUDA_OK(cudaGetDevice(&dev));
  GP_CUDA_OK(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
  cudaStream_t st = (cudaStream_t)cuda_stream;
  float* sink = (float*)ws;
  double r[GP_PEAK_COUNT] = {0};
  GP_OK_OR_RETURN(run_peak<GP_PEAK_FFMA>(&r[GP_PEAK_FFMA], st, sink, sms));
  GP_OK_OR_RETURN(run_peak<GP_PEAK_FFMA_IMM>(&r[GP_PEAK_FFMA_IMM], st, sink, sms));
  GP_OK_OR_RETURN(run_peak<GP_PEAK_FFMA2>(&r[GP_PEAK_FFMA2], st, sink, sms));
  GP_OK_OR_RETURN(run_peak<GP_PEAK_FFMA2_BC>(&r[GP_PEAK_FFMA2_BC], st, sink, sms));
  GP_OK_OR_RETURN(run_peak<GP_PEAK_DFMA>(&r[GP_PEAK_DFMA], st, sink, sms));
  GP_OK_OR_RETURN(run_peak<GP_PEAK_MUFU>(&r[GP_PEAK_MUFU], st, sink, sms));
  GP_OK_OR_RETURN(run_peak<GP_PEAK_FFMA2_DFMA>(&r[GP_PEAK_FFMA2_DFMA], st, sink, sms));
  GP_OK_OR_RETURN(run_peak<GP_PEAK_FFMA2_MUFU>(&r[GP_PEAK_FFMA2_MUFU], st, sink, sms));
  for (int i = 0; i < n_out && i < GP_PEAK_COUNT; ++i) out_host[i] = r[i];
  return GP_OK;
}
