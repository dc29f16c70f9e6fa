// aw_probe.cu — TEST AND MEASUREMENT SUPPORT (tests/aw_probe.h): the library's device routines behind elementwise
// kernels, and the fp64 micro-benchmarks.  Built into tests/libaw_probe.so; nothing in libaw.so depends on it.
#include <cuda_runtime.h>
#include <stdint.h>

#include "../paper_1107_4107_b200/csrc/aw_internal.cuh"
#include "../paper_1107_4107_b200/csrc/aw_model.cuh"
#include "../paper_1107_4107_b200/csrc/aw_trig.cuh"
#include "../paper_1107_4107_b200/csrc/aw_tsincos.cuh"
#include "aw_probe.h"

namespace {

using aw::hamiltonian_dev;
using aw::sincos;
using aw::uniform01;

__global__ void uniform_kernel(uint64_t seed, uint64_t k0, int64_t n, uint32_t slot, double *out) {
  const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i < n) out[i] = uniform01(seed, k0 + (uint64_t)i, slot);
}

__global__ void sincos_kernel(const double *x, int64_t n, double *s, double *c) {
  const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i < n) {
    double sn, cs;
    sincos(x[i], sn, cs);
    s[i] = sn;
    c[i] = cs;
  }
}

__global__ void tsincos_kernel(const double *x, int64_t n, double *s, double *c) {
  __shared__ double2 tab_s[aw::kTab * aw::kTabCopies];
  for (int i = threadIdx.x; i < aw::kTab * aw::kTabCopies; i += blockDim.x)
    tab_s[i] = make_double2(aw_trig_table[2 * (i / aw::kTabCopies)], aw_trig_table[2 * (i / aw::kTabCopies) + 1]);
  __syncthreads();
  const aw::TrigTable tab = {reinterpret_cast<const char *>(tab_s), (threadIdx.x & (aw::kTabCopies - 1)) * 16u};
  const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i < n) {
    double sn, cs;
    aw::tsincos(tab, x[i], sn, cs);
    s[i] = sn;
    c[i] = cs;
  }
}

__global__ void hamiltonian_kernel(const double *q, int64_t n, int64_t P, double eps, double *out) {
  const int64_t k = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (k < n) out[k] = hamiltonian_dev(q[k], q[P + k], q[2 * P + k], q[3 * P + k], q[4 * P + k], q[5 * P + k], eps);
}

template <int CH>
__global__ void dfma_peak_kernel(int64_t iters, double *sink) {
  double v[CH];
  const double a = 1.0 - 1e-9 * (double)(threadIdx.x & 7), b = 1e-12;
#pragma unroll
  for (int c = 0; c < CH; ++c) v[c] = (double)(threadIdx.x + c);
#pragma unroll 1
  for (int64_t i = 0; i < iters; i += 8) {
#pragma unroll
    for (int u = 0; u < 8; ++u) {
#pragma unroll
      for (int c = 0; c < CH; ++c) v[c] = fma(v[c], a, b);
    }
  }
  double acc = 0.0;
#pragma unroll
  for (int c = 0; c < CH; ++c) acc += v[c];
  if (acc == 123.456) sink[0] = acc;  // never true in practice; keeps the chains alive
}

// fp64 issue rate by operand shape: 8 independent chains per thread, 32 instructions per loop trip.
//   0: fma(v, u0, w0)    three registers, two of them shared by neighbouring instructions (reuse cache)
//   1: fma(v, u_c, w_c)  three distinct registers, nothing shared with the neighbours
//   2: fma(v, u_c, imm)  two registers + an immediate
//   3: fma(v, v, w_c)    three register operands, two distinct
//   4: v * u_c           DMUL, two registers
//   5: fma(u_c, w_c', v) accumulate form, three distinct registers
template <int SHAPE>
__global__ void dfma_shape_kernel(int64_t iters, double *sink, const double *in) {
  constexpr int CH = 8;
  double v[CH], u[CH], w[CH];
#pragma unroll
  for (int c = 0; c < CH; ++c) {
    v[c] = in[(threadIdx.x + c) & 127];
    u[c] = in[(threadIdx.x + 32 + c) & 127];
    w[c] = in[(threadIdx.x + 64 + c) & 127];
  }
#pragma unroll 1
  for (int64_t i = 0; i < iters; ++i) {
#pragma unroll
    for (int r = 0; r < 4; ++r) {
#pragma unroll
      for (int c = 0; c < CH; ++c) {
        if (SHAPE == 0) v[c] = fma(v[c], u[0], w[0]);
        if (SHAPE == 1) v[c] = fma(v[c], u[c], w[c]);
        if (SHAPE == 2) v[c] = fma(v[c], u[c], 1e-12);
        if (SHAPE == 3) v[c] = fma(v[c], v[c], w[c]);
        if (SHAPE == 4) v[c] = v[c] * u[c];
        if (SHAPE == 5) v[c] = fma(u[c], w[(c + 1) % CH], v[c]);
      }
    }
  }
  double acc = 0.0;
#pragma unroll
  for (int c = 0; c < CH; ++c) acc += v[c];
  if (acc == 123.456) sink[0] = acc;
}

int done(cudaStream_t st) {
  if (cudaGetLastError() != cudaSuccess) return -2;
  return cudaStreamSynchronize(st) == cudaSuccess ? 0 : -2;
}

template <typename F, typename G>
int timed(cudaStream_t st, F &&warm, G &&run, double *ms_host) {
  cudaEvent_t e0, e1;
  if (cudaEventCreate(&e0) != cudaSuccess || cudaEventCreate(&e1) != cudaSuccess) return -2;
  warm();
  cudaEventRecord(e0, st);
  run();
  cudaEventRecord(e1, st);
  cudaError_t err = cudaEventSynchronize(e1);
  float ms = 0.f;
  if (err == cudaSuccess) err = cudaEventElapsedTime(&ms, e0, e1);
  if (err == cudaSuccess) err = cudaGetLastError();
  cudaEventDestroy(e0);
  cudaEventDestroy(e1);
  *ms_host = (double)ms;
  return err == cudaSuccess ? 0 : -2;
}

template <int CH>
void peak(int blocks, int threads, int64_t iters, double *sink, cudaStream_t st) {
  dfma_peak_kernel<CH><<<blocks, threads, 0, st>>>(iters, sink);
}
void peak_any(int chains, int blocks, int threads, int64_t iters, double *sink, cudaStream_t st) {
  switch (chains) {
    case 1: peak<1>(blocks, threads, iters, sink, st); break;
    case 2: peak<2>(blocks, threads, iters, sink, st); break;
    case 4: peak<4>(blocks, threads, iters, sink, st); break;
    case 8: peak<8>(blocks, threads, iters, sink, st); break;
    default: peak<16>(blocks, threads, iters, sink, st); break;
  }
}
void shape_any(int shape, int blocks, int threads, int64_t iters, double *sink, const double *in, cudaStream_t st) {
  switch (shape) {
    case 0: dfma_shape_kernel<0><<<blocks, threads, 0, st>>>(iters, sink, in); break;
    case 1: dfma_shape_kernel<1><<<blocks, threads, 0, st>>>(iters, sink, in); break;
    case 2: dfma_shape_kernel<2><<<blocks, threads, 0, st>>>(iters, sink, in); break;
    case 3: dfma_shape_kernel<3><<<blocks, threads, 0, st>>>(iters, sink, in); break;
    case 4: dfma_shape_kernel<4><<<blocks, threads, 0, st>>>(iters, sink, in); break;
    default: dfma_shape_kernel<5><<<blocks, threads, 0, st>>>(iters, sink, in); break;
  }
}

}  // namespace

extern "C" {

int awp_sincos(const double *x_dev, int64_t n, double *sin_dev, double *cos_dev, void *stream) {
  if (!x_dev || !sin_dev || !cos_dev || n < 0) return -1;
  if (n == 0) return 0;
  cudaStream_t st = (cudaStream_t)stream;
  sincos_kernel<<<(unsigned)((n + 255) / 256), 256, 0, st>>>(x_dev, n, sin_dev, cos_dev);
  return done(st);
}

int awp_tsincos(const double *x_dev, int64_t n, double *sin_dev, double *cos_dev, void *stream) {
  if (!x_dev || !sin_dev || !cos_dev || n < 0) return -1;
  if (n == 0) return 0;
  cudaStream_t st = (cudaStream_t)stream;
  tsincos_kernel<<<(unsigned)((n + 255) / 256), 256, 0, st>>>(x_dev, n, sin_dev, cos_dev);
  return done(st);
}

int awp_uniform(uint64_t seed, uint64_t k0, int64_t n, uint32_t slot, double *out_dev, void *stream) {
  if (!out_dev || n < 0 || slot > 15) return -1;
  if (n == 0) return 0;
  cudaStream_t st = (cudaStream_t)stream;
  uniform_kernel<<<(unsigned)((n + 255) / 256), 256, 0, st>>>(seed, k0, n, slot, out_dev);
  return done(st);
}

int awp_hamiltonian(const double *q_dev, int64_t n, int64_t pitch, double eps, double *out_dev, void *stream) {
  if (!q_dev || !out_dev || n < 0 || pitch < n) return -1;
  if (n == 0) return 0;
  cudaStream_t st = (cudaStream_t)stream;
  hamiltonian_kernel<<<(unsigned)((n + 255) / 256), 256, 0, st>>>(q_dev, n, pitch, eps, out_dev);
  return done(st);
}

int awp_dfma_peak(int blocks, int threads, int chains, int64_t iters, double *sink_dev, double *ms_host,
                  double *dfma_host, void *stream) {
  if (blocks <= 0 || threads <= 0 || threads > 1024 || iters <= 0 || !sink_dev || !ms_host || !dfma_host) return -1;
  if (chains != 1 && chains != 2 && chains != 4 && chains != 8 && chains != 16) return -1;
  iters = (iters + 7) / 8 * 8;
  cudaStream_t st = (cudaStream_t)stream;
  const int rc = timed(st, [&] { peak_any(chains, blocks, threads, 128, sink_dev, st); },
                       [&] { peak_any(chains, blocks, threads, iters, sink_dev, st); }, ms_host);
  *dfma_host = (double)blocks * (double)threads * (double)chains * (double)iters;
  return rc;
}

int awp_dfma_shape(int blocks, int threads, int shape, int64_t iters, double *work_dev, double *ms_host,
                   double *inst_host, void *stream) {
  if (blocks <= 0 || threads <= 0 || threads > 1024 || iters <= 0 || !work_dev || !ms_host || !inst_host) return -1;
  if (shape < 0 || shape > 5) return -1;
  cudaStream_t st = (cudaStream_t)stream;
  double host[128];
  for (int i = 0; i < 128; ++i) host[i] = 1.0 - 1e-9 * (double)(i % 97);
  if (cudaMemcpyAsync(work_dev, host, sizeof host, cudaMemcpyHostToDevice, st) != cudaSuccess) return -2;
  const int rc = timed(st, [&] { shape_any(shape, blocks, threads, 64, work_dev + 128, work_dev, st); },
                       [&] { shape_any(shape, blocks, threads, iters, work_dev + 128, work_dev, st); }, ms_host);
  *inst_host = (double)blocks * (double)threads * (double)iters * 32.0;
  return rc;
}

}  // extern "C"
