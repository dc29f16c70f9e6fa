// aw_reduce.cu — §8(a) a5 (indicator image) and a6 (visited-cell density histogram); DESIGN.md §6.3-6.4.
#include <cstring>
#include <mutex>

#include "aw_internal.cuh"
#include "aw_model.cuh"

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

// ---------------------------------------------------------------------- §8(f) 1-2: the paper's indicator
// Averaged finite-time velocity over the window since aw_mark and its central projection on S (P:67,
// P:171 fn. 26; R26, R27).  Every operation is rounded separately, in the order include/aw.h states (the
// explicit-rounding intrinsics stop the compiler from contracting them into FMAs), so that the bin a
// point falls in is decided by the same fp64 numbers on both sides of the parity test.
constexpr double kTwoPiHi = 6.283185307179586;  // double nearest 2 pi

__device__ __forceinline__ bool averaged_velocity(const VelocityArgs &v, int64_t k, double vh[3]) {
  double V[3];
#pragma unroll
  for (int a = 0; a < 3; ++a) {
    const double dxw = __dsub_rn(v.q[a * v.pitch + k], v.qref[a * v.pitch + k]);
    const int dk = v.wind ? v.wind[a * v.pitch + k] - v.windref[a * v.pitch + k] : 0;
    const double dX = __dadd_rn(__dmul_rn((double)dk, kTwoPiHi), dxw);
    V[a] = __ddiv_rn(dX, v.Dt);
  }
  double n2 = __dmul_rn(V[0], V[0]);
  n2 = __dadd_rn(n2, __dmul_rn(V[1], V[1]));
  n2 = __dadd_rn(n2, __dmul_rn(V[2], V[2]));
  const double nrm = __dsqrt_rn(n2);
  if (!(nrm > 0.0) || !isfinite(nrm)) return false;
  const double scale = __ddiv_rn(v.radius, nrm);
#pragma unroll
  for (int a = 0; a < 3; ++a) vh[a] = __dmul_rn(V[a], scale);
  return true;
}

__global__ void __launch_bounds__(256) indicator_ref_kernel(const __grid_constant__ VelocityArgs v,
                                                            const uint8_t *__restrict__ status, int64_t n,
                                                            int kind, double *__restrict__ out) {
  const int64_t k = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (k >= n) return;
  double r = __longlong_as_double(0x7ff8000000000000ll);
  if (status[k] == AW_ST_LIVE) {
    if (kind == AW_IND_DP) {  // |P(t) - P(0)|
      const int64_t P = v.pitch;
      const double d0 = __dsub_rn(v.q[3 * P + k], v.qref[3 * P + k]);
      const double d1 = __dsub_rn(v.q[4 * P + k], v.qref[4 * P + k]);
      const double d2 = __dsub_rn(v.q[5 * P + k], v.qref[5 * P + k]);
      double s2 = __dmul_rn(d0, d0);
      s2 = __dadd_rn(s2, __dmul_rn(d1, d1));
      s2 = __dadd_rn(s2, __dmul_rn(d2, d2));
      r = __dsqrt_rn(s2);
    } else {
      double vh[3];
      if (averaged_velocity(v, k, vh)) r = kind == AW_IND_VX ? vh[0] : (kind == AW_IND_VY ? vh[1] : vh[2]);
    }
  }
  out[k] = r;
}

// ------------------------------------------------------------ energy-drift statistics (BJ:configs[2]; R29)
// Over the live trajectories: count, max / sum / sum of squares of dH_max (acc plane 3), sum / sum of squares /
// max |.| of the signed error of the current state H(X,P) - H0, and the first index attaining max dH_max.
// Deterministic: fixed block partials (warp shuffles in a fixed order), then one block folds the partials in a
// fixed order, so the result does not depend on scheduling (no floating-point atomics).
struct EnergyPartial {
  double cnt, mx, idx, sum, sq, ssum, ssq, smax;
};
__device__ __forceinline__ void fold(EnergyPartial &a, const EnergyPartial &b) {
  if (b.cnt > 0.0 && (a.cnt == 0.0 || b.mx > a.mx || (b.mx == a.mx && b.idx < a.idx))) { a.mx = b.mx; a.idx = b.idx; }
  a.cnt += b.cnt; a.sum += b.sum; a.sq += b.sq; a.ssum += b.ssum; a.ssq += b.ssq;
  a.smax = fmax(a.smax, b.smax);
}
__device__ __forceinline__ EnergyPartial shuffle_down(const EnergyPartial &a, int off) {
  EnergyPartial b;
  b.cnt = __shfl_down_sync(0xffffffffu, a.cnt, off); b.mx = __shfl_down_sync(0xffffffffu, a.mx, off);
  b.idx = __shfl_down_sync(0xffffffffu, a.idx, off); b.sum = __shfl_down_sync(0xffffffffu, a.sum, off);
  b.sq = __shfl_down_sync(0xffffffffu, a.sq, off); b.ssum = __shfl_down_sync(0xffffffffu, a.ssum, off);
  b.ssq = __shfl_down_sync(0xffffffffu, a.ssq, off); b.smax = __shfl_down_sync(0xffffffffu, a.smax, off);
  return b;
}
constexpr int kStatsBlock = 256;
constexpr int kStatsItems = 8;

__device__ __forceinline__ void block_fold(EnergyPartial &a, EnergyPartial *sh) {
#pragma unroll
  for (int off = 16; off > 0; off >>= 1) { const EnergyPartial b = shuffle_down(a, off); fold(a, b); }
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  if (lane == 0) sh[warp] = a;
  __syncthreads();
  if (warp == 0) {
    EnergyPartial z = {0, 0, -1, 0, 0, 0, 0, 0};
    a = lane < kStatsBlock / 32 ? sh[lane] : z;
#pragma unroll
    for (int off = 4; off > 0; off >>= 1) { const EnergyPartial b = shuffle_down(a, off); fold(a, b); }
  }
}

__global__ void __launch_bounds__(kStatsBlock)
    energy_partial_kernel(const double *__restrict__ q, const double *__restrict__ acc,
                          const uint8_t *__restrict__ status, int64_t n, int64_t P, double eps,
                          EnergyPartial *partials) {
  __shared__ EnergyPartial sh[kStatsBlock / 32];
  EnergyPartial a = {0, 0, -1, 0, 0, 0, 0, 0};
  const int64_t base = (int64_t)blockIdx.x * (kStatsBlock * kStatsItems);
  for (int it = 0; it < kStatsItems; ++it) {
    const int64_t k = base + (int64_t)it * kStatsBlock + threadIdx.x;
    if (k < n && status[k] == AW_ST_LIVE) {
      const double sd = hamiltonian_dev(q[k], q[P + k], q[2 * P + k], q[3 * P + k], q[4 * P + k], q[5 * P + k], eps) -
                        acc[2 * P + k];
      const double d = acc[3 * P + k];
      EnergyPartial b = {1.0, d, (double)k, d, d * d, sd, sd * sd, fabs(sd)};
      fold(a, b);
    }
  }
  block_fold(a, sh);
  if (threadIdx.x == 0) partials[blockIdx.x] = a;
}

__global__ void __launch_bounds__(kStatsBlock)
    energy_final_kernel(const EnergyPartial *partials, int64_t nblocks, double *out) {
  __shared__ EnergyPartial sh[kStatsBlock / 32];
  EnergyPartial a = {0, 0, -1, 0, 0, 0, 0, 0};
  for (int64_t b = threadIdx.x; b < nblocks; b += kStatsBlock) fold(a, partials[b]);
  block_fold(a, sh);
  if (threadIdx.x == 0) {
    const double nan = __longlong_as_double(0x7ff8000000000000ll);
    const bool any = a.cnt > 0.0;
    out[0] = a.cnt; out[1] = a.mx; out[6] = any ? a.idx : -1.0; out[7] = a.smax;
    out[2] = any ? a.sum / a.cnt : nan;
    out[3] = any ? sqrt(a.sq / a.cnt) : nan;
    out[4] = any ? a.ssum / a.cnt : nan;
    out[5] = any ? sqrt(a.ssq / a.cnt) : nan;
  }
}

// signed energy error of the current state, H(X,P) - H0 (NaN where not live)
__global__ void __launch_bounds__(256) signed_dh_kernel(const double *__restrict__ q, const double *__restrict__ acc,
                                                        const uint8_t *__restrict__ status, int64_t n, int64_t P,
                                                        double eps, double *__restrict__ out) {
  const int64_t k = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (k >= n) return;
  double r = __longlong_as_double(0x7ff8000000000000ll);
  if (status[k] == AW_ST_LIVE)
    r = hamiltonian_dev(q[k], q[P + k], q[2 * P + k], q[3 * P + k], q[4 * P + k], q[5 * P + k], eps) - acc[2 * P + k];
  out[k] = r;
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

// MODE 0: the point is the instantaneous (px, py); MODE 1: (Vhat_x, Vhat_y), hemisphere chosen by `hemi`.
template <int MODE>
__global__ void __launch_bounds__(kDensityBlock)
    density_kernel(const __grid_constant__ VelocityArgs v, int hemi,
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
      double bx, by;
      bool in = true;
      if (MODE == 0) {
        bx = v.q[3 * v.pitch + k];
        by = v.q[4 * v.pitch + k];
      } else {
        double vh[3];
        in = averaged_velocity(v, k, vh);
        if (in) in = (hemi == AW_DENS_VEL_BOTH) || (hemi == AW_DENS_VEL_UPPER ? vh[2] >= 0.0 : vh[2] < 0.0);
        bx = vh[0];
        by = vh[1];
      }
      if (in) {
        const double ax = floor(__dmul_rn(__dsub_rn(bx, lo), fx));
        const double ay = floor(__dmul_rn(__dsub_rn(by, lo), fy));
        in = ax >= 0.0 && ax < dgx && ay >= 0.0 && ay < dgy;
        if (in) bin = (unsigned)((int64_t)ay * gx + (int64_t)ax);
      }
      if (!in) ++my_dropped;
    }
    const unsigned peers = __match_any_sync(0xffffffffu, bin);
    // spread input: when no two lanes of the warp share a bin the block table would only add a shared-memory
    // round trip in front of the same global atomic, so the points go straight to the histogram
    if (__all_sync(0xffffffffu, bin == kEmpty || __popc(peers) == 1)) {
      if (bin != kEmpty) atomicAdd(&hist[bin], 1u);
      continue;
    }
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

// ------------------------------------------------------------------------------- precondition of aw_integrate
// Enforced, not assumed (include/aw.h, aw_state.Emax): P^2 <= 2(H + 2|eps|) on the whole orbit, so the largest
// drift angle of a trajectory is bounded by its energy; one whose energy exceeds what the Taylor degrees of the chosen
// trigonometry level (and the angle range of R7) were sized for is flagged AW_ST_RANGE before the integrator runs
// and is never touched.  A non-finite H is the checkpoint's business (status 2).  Runs once per aw_integrate call:
// 49 bytes per trajectory, HBM bound, ~1e-4 of a 20 000-step launch.
__global__ void __launch_bounds__(256) range_check_kernel(const double *__restrict__ q, uint8_t *__restrict__ status,
                                                          int64_t n, int64_t P, double eps, double hmax) {
  const int64_t k = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (k >= n || status[k] != AW_ST_LIVE) return;
  const double h = hamiltonian_dev(q[k], q[P + k], q[2 * P + k], q[3 * P + k], q[4 * P + k], q[5 * P + k], eps);
  if (h > hmax && h <= 1.7976931348623157e308) status[k] = (uint8_t)AW_ST_RANGE;
}

// ------------------------------------------------------------------------------- aw_bound_energy
// max over live trajectories of H(X,P) (finite values only): doubles map to 64-bit keys whose unsigned order is the
// numeric order, so one atomicMax per block on an 8-byte scratch word gives an order-independent, exact maximum.
__device__ __forceinline__ unsigned long long energy_key(double h) {
  const unsigned long long b = (unsigned long long)__double_as_longlong(h);
  return (b >> 63) ? ~b : (b | 0x8000000000000000ull);
}

__global__ void __launch_bounds__(256) energy_bound_kernel(const double *__restrict__ q,
                                                           const uint8_t *__restrict__ status, int64_t n, int64_t P,
                                                           double eps, unsigned long long *key_out) {
  __shared__ unsigned long long sh[8];
  unsigned long long key = 0ull;
  for (int64_t k = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; k < n; k += (int64_t)gridDim.x * blockDim.x) {
    if (status[k] != AW_ST_LIVE) continue;
    const double h = hamiltonian_dev(q[k], q[P + k], q[2 * P + k], q[3 * P + k], q[4 * P + k], q[5 * P + k], eps);
    if (isfinite(h)) { const unsigned long long kk = energy_key(h); key = kk > key ? kk : key; }
  }
#pragma unroll
  for (int off = 16; off > 0; off >>= 1) {
    const unsigned long long o = __shfl_down_sync(0xffffffffu, key, off);
    key = o > key ? o : key;
  }
  if ((threadIdx.x & 31) == 0) sh[threadIdx.x >> 5] = key;
  __syncthreads();
  if (threadIdx.x == 0) {
    for (int w = 1; w < 8; ++w) key = sh[w] > key ? sh[w] : key;
    if (key) atomicMax(key_out, key);
  }
}

}  // namespace

cudaError_t launch_indicator(const double *acc, const uint8_t *status, int64_t n, int64_t pitch, int kind,
                             double thr, double t, void *out, cudaStream_t st) {
  indicator_kernel<<<(unsigned)((n + 255) / 256), 256, 0, st>>>(acc, status, n, pitch, kind, thr, t, out);
  count_launch();
  return cudaGetLastError();
}

int64_t energy_stats_blocks(int64_t n) {
  const int64_t per = (int64_t)kStatsBlock * kStatsItems;
  return (n + per - 1) / per;
}
size_t energy_partial_bytes() { return sizeof(EnergyPartial); }

cudaError_t launch_energy_stats(const double *q, const double *acc, const uint8_t *status, int64_t n, int64_t pitch,
                                double eps, void *scratch, double *out, cudaStream_t st) {
  const int64_t nb = energy_stats_blocks(n);
  EnergyPartial *part = static_cast<EnergyPartial *>(scratch);
  if (nb > 0) {
    energy_partial_kernel<<<(unsigned)nb, kStatsBlock, 0, st>>>(q, acc, status, n, pitch, eps, part);
    count_launch();
  }
  energy_final_kernel<<<1, kStatsBlock, 0, st>>>(part, nb, out);
  count_launch();
  return cudaGetLastError();
}

cudaError_t launch_signed_dh(const double *q, const double *acc, const uint8_t *status, int64_t n, int64_t pitch,
                             double eps, double *out, cudaStream_t st) {
  signed_dh_kernel<<<(unsigned)((n + 255) / 256), 256, 0, st>>>(q, acc, status, n, pitch, eps, out);
  count_launch();
  return cudaGetLastError();
}

cudaError_t launch_indicator_ref(const VelocityArgs &v, const uint8_t *status, int64_t n, int kind, double *out,
                                 cudaStream_t st) {
  indicator_ref_kernel<<<(unsigned)((n + 255) / 256), 256, 0, st>>>(v, status, n, kind, out);
  count_launch();
  return cudaGetLastError();
}

cudaError_t launch_density(const VelocityArgs &v, int mode, const uint8_t *status, int64_t n,
                           uint32_t *hist, int32_t gx, int32_t gy, double lo, double fx, double fy,
                           unsigned long long *dropped, cudaStream_t st) {
  const int64_t per_block = (int64_t)kDensityBlock * kItems;
  const unsigned blocks = (unsigned)((n + per_block - 1) / per_block);
  if (mode == AW_DENS_ACTION)
    density_kernel<0><<<blocks, kDensityBlock, 0, st>>>(v, mode, status, n, hist, gx, gy, lo, fx, fy, dropped);
  else
    density_kernel<1><<<blocks, kDensityBlock, 0, st>>>(v, mode, status, n, hist, gx, gy, lo, fx, fy, dropped);
  count_launch();
  return cudaGetLastError();
}

cudaError_t launch_range_check(const double *q, uint8_t *status, int64_t n, int64_t pitch, double eps, double hmax,
                               cudaStream_t st) {
  range_check_kernel<<<(unsigned)((n + 255) / 256), 256, 0, st>>>(q, status, n, pitch, eps, hmax);
  count_launch();
  return cudaGetLastError();
}

cudaError_t launch_energy_bound(const double *q, const uint8_t *status, int64_t n, int64_t pitch, double eps,
                                unsigned long long *key_out, cudaStream_t st) {
  int64_t blocks = (n + 255) / 256;
  if (blocks > 148 * 8) blocks = 148 * 8;
  energy_bound_kernel<<<(unsigned)blocks, 256, 0, st>>>(q, status, n, pitch, eps, key_out);
  count_launch();
  return cudaGetLastError();
}

double energy_key_decode(unsigned long long key, bool *any) {
  *any = key != 0ull;
  const unsigned long long b = (key >> 63) ? (key & 0x7fffffffffffffffull) : ~key;
  double h;
  static_assert(sizeof h == sizeof b, "fp64");
  memcpy(&h, &b, sizeof h);
  return h;
}

// ------------------------------------------------------------ aw_energy_stats_noalloc: scratch held by the library
// The block partials of the energy statistics live in this file-scope device array instead of caller memory, so the
// call needs no allocation from anybody (CUDA graph capture, serving loops).  Every device that loads the library
// holds the 512 KiB until the process exits.  The name below is only a host-side handle in host code: the device
// address is taken once per device with cudaGetSymbolAddress, with that device current, and handed to the kernels.
// Nothing has to start at zero — energy_partial_kernel overwrites partials [0, nb) and energy_final_kernel reads
// exactly those — so the previous call's contents are never seen.  All calls on a device share the array: two calls
// whose kernels overlap on the GPU (different streams) race.
constexpr int64_t kNoAllocMaxBlocks = (AW_NOALLOC_MAX_N + kStatsBlock * kStatsItems - 1) / (kStatsBlock * kStatsItems);
static __device__ __align__(256) EnergyPartial g_noalloc_partials[kNoAllocMaxBlocks];

namespace {
constexpr int kNoAllocMaxDevices = 64;
std::mutex g_noalloc_mutex;
EnergyPartial *g_noalloc_addr[kNoAllocMaxDevices] = {};

cudaError_t noalloc_scratch(EnergyPartial **out) {
  int dev = -1;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) return e;
  if (dev < 0 || dev >= kNoAllocMaxDevices) return cudaErrorInvalidDevice;
  std::lock_guard<std::mutex> lock(g_noalloc_mutex);
  if (!g_noalloc_addr[dev]) {
    void *p = nullptr;
    e = cudaGetSymbolAddress(&p, g_noalloc_partials);
    if (e != cudaSuccess) return e;
    g_noalloc_addr[dev] = static_cast<EnergyPartial *>(p);
  }
  *out = g_noalloc_addr[dev];
  return cudaSuccess;
}
}  // namespace

int64_t energy_stats_noalloc_max_n() { return kNoAllocMaxBlocks * kStatsBlock * kStatsItems; }

cudaError_t launch_energy_stats_noalloc(const double *q, const double *acc, const uint8_t *status, int64_t n,
                                        int64_t pitch, double eps, double *out, cudaStream_t st) {
  EnergyPartial *part = nullptr;
  const cudaError_t e = noalloc_scratch(&part);
  if (e != cudaSuccess) return e;
  const int64_t nb = energy_stats_blocks(n);
  if (nb > kNoAllocMaxBlocks) return cudaErrorInvalidValue;   // the C entry rejects this before coming here
  if (nb > 0) {
    energy_partial_kernel<<<(unsigned)nb, kStatsBlock, 0, st>>>(q, acc, status, n, pitch, eps, part);
    count_launch();
  }
  energy_final_kernel<<<1, kStatsBlock, 0, st>>>(part, nb, out);
  count_launch();
  return cudaGetLastError();
}

}  // namespace aw
