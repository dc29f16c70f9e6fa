// aw_reduce.cu — §8(a) a5 (indicator image) and a6 (visited-cell density histogram); DESIGN.md §6.3-6.4.
#include "aw_internal.cuh"

namespace aw {

namespace {

// ------------------------------------------------------------------------------------------- a5
// Elementwise, HBM bound: reads 8 (+1) bytes, writes 8 (or 1) bytes per trajectory.
__global__ void __launch_bounds__(256) indicator_kernel(const double *__restrict__ acc,
                                                        const uint8_t *__restrict__ status, int64_t n,
                                                        int64_t P, int kind, double thr, double t,
                                                        void *out) {
  const int64_t k = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (k >= n) return;
  const bool live = status[k] == AW_ST_LIVE;
  const double nan = __longlong_as_double(0x7ff8000000000000ll);
  if (kind == AW_IND_CLASS) {
    uint8_t v = 255;
    if (live) v = acc[P + k] > thr ? 1 : 0;
    static_cast<uint8_t *>(out)[k] = v;
    return;
  }
  double v = nan;
  if (live) {
    if (kind == AW_IND_FLI) v = acc[P + k];
    else if (kind == AW_IND_FTLE) v = __ddiv_rn(acc[k], t);
    else v = acc[3 * P + k];
  }
  static_cast<double *>(out)[k] = v;
}

// ------------------------------------------------------------------------------------------- a6
// The histogram (1024 x 1024 uint32 = 4 MiB at configs[4]) does not fit in shared memory, so the
// privatisation is a per-block open-addressing table of (bin, count) pairs in shared memory:
//   1. each thread turns its point into a bin index (two roundings: subtract, multiply; no FMA — R20);
//   2. lanes of a warp holding the same bin elect one leader (__match_any_sync) that carries the count;
//   3. the leader adds into the block's shared table (atomicCAS on the key, atomicAdd on the count);
//      a table miss after kProbe probes goes straight to the global histogram;
//   4. one merge per block: every occupied slot is added to the global histogram once.
// configs[4] starts with 2^20 points in <= 4 bins: steps 2-3 turn 2^20 same-address global atomics
// into <= 4 per block.  Counts are exact integers, so the result is independent of the order.
constexpr int kTable = 2048;  // slots per block (power of two)
constexpr int kProbe = 8;
constexpr int kDensityBlock = 256;
constexpr int kItems = 16;  // points per thread
constexpr unsigned kEmpty = 0xffffffffu;

__global__ void __launch_bounds__(kDensityBlock)
    density_kernel(const double *__restrict__ px, const double *__restrict__ py,
                   const uint8_t *__restrict__ status, int64_t n, uint32_t *hist, int32_t gx, int32_t gy,
                   double lo, double fx, double fy, unsigned long long *dropped) {
  __shared__ unsigned keys[kTable];
  __shared__ unsigned counts[kTable];
  __shared__ unsigned block_dropped;
  for (int s = threadIdx.x; s < kTable; s += kDensityBlock) { keys[s] = kEmpty; counts[s] = 0; }
  if (threadIdx.x == 0) block_dropped = 0;
  __syncthreads();

  const int64_t base = (int64_t)blockIdx.x * (kDensityBlock * kItems);
  const double dgx = (double)gx, dgy = (double)gy;
  unsigned my_dropped = 0;
#pragma unroll 4
  for (int it = 0; it < kItems; ++it) {
    const int64_t k = base + (int64_t)it * kDensityBlock + threadIdx.x;  // warp-uniform trip count
    unsigned bin = kEmpty;
    if (k < n && status[k] == AW_ST_LIVE) {
      const double ax = floor(__dmul_rn(__dsub_rn(px[k], lo), fx));
      const double ay = floor(__dmul_rn(__dsub_rn(py[k], lo), fy));
      if (ax >= 0.0 && ax < dgx && ay >= 0.0 && ay < dgy) bin = (unsigned)((int64_t)ay * gx + (int64_t)ax);
      else ++my_dropped;
    }
    const unsigned peers = __match_any_sync(0xffffffffu, bin);
    if (bin != kEmpty && (__ffs(peers) - 1) == (int)(threadIdx.x & 31)) {
      const unsigned cnt = __popc(peers);
      unsigned slot = (bin * 2654435761u) >> 21;  // top 11 bits -> [0, 2048)
      bool done = false;
#pragma unroll 1
      for (int pr = 0; pr < kProbe; ++pr) {
        const unsigned prev = atomicCAS(&keys[slot], kEmpty, bin);
        if (prev == kEmpty || prev == bin) { atomicAdd(&counts[slot], cnt); done = true; break; }
        slot = (slot + 1) & (kTable - 1);
      }
      if (!done) atomicAdd(&hist[bin], cnt);
    }
  }
  // dropped: warp sum, one shared atomic per warp, one global atomic per block
  for (int off = 16; off > 0; off >>= 1) my_dropped += __shfl_down_sync(0xffffffffu, my_dropped, off);
  if ((threadIdx.x & 31) == 0 && my_dropped) atomicAdd(&block_dropped, my_dropped);
  __syncthreads();
  for (int s = threadIdx.x; s < kTable; s += kDensityBlock)
    if (keys[s] != kEmpty) atomicAdd(&hist[keys[s]], counts[s]);
  if (threadIdx.x == 0 && dropped && block_dropped) atomicAdd(dropped, (unsigned long long)block_dropped);
}

// ------------------------------------------------------------------------------- fp64 peak probe
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

}  // namespace

cudaError_t launch_indicator(const double *acc, const uint8_t *status, int64_t n, int64_t pitch, int kind,
                             double thr, double t, void *out, cudaStream_t st) {
  indicator_kernel<<<(unsigned)((n + 255) / 256), 256, 0, st>>>(acc, status, n, pitch, kind, thr, t, out);
  count_launch();
  return cudaGetLastError();
}

cudaError_t launch_density(const double *px, const double *py, const uint8_t *status, int64_t n,
                           uint32_t *hist, int32_t gx, int32_t gy, double lo, double fx, double fy,
                           unsigned long long *dropped, cudaStream_t st) {
  const int64_t per_block = (int64_t)kDensityBlock * kItems;
  density_kernel<<<(unsigned)((n + per_block - 1) / per_block), kDensityBlock, 0, st>>>(
      px, py, status, n, hist, gx, gy, lo, fx, fy, dropped);
  count_launch();
  return cudaGetLastError();
}

cudaError_t launch_dfma_peak(int blocks, int threads, int chains, int64_t iters, double *sink,
                             cudaStream_t st) {
  switch (chains) {
    case 1: dfma_peak_kernel<1><<<blocks, threads, 0, st>>>(iters, sink); break;
    case 2: dfma_peak_kernel<2><<<blocks, threads, 0, st>>>(iters, sink); break;
    case 4: dfma_peak_kernel<4><<<blocks, threads, 0, st>>>(iters, sink); break;
    case 8: dfma_peak_kernel<8><<<blocks, threads, 0, st>>>(iters, sink); break;
    case 16: dfma_peak_kernel<16><<<blocks, threads, 0, st>>>(iters, sink); break;
    default: return cudaErrorInvalidValue;
  }
  count_launch();
  return cudaGetLastError();
}

}  // namespace aw
