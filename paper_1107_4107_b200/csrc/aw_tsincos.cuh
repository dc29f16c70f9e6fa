// aw_tsincos.cuh — the table-driven sincos of the integrator's step loop (DESIGN.md §6.1 (ii)).
#pragma once
#include "aw_trig.cuh"
#include "aw_trig_table.h"

namespace aw {

// Table-driven sincos for the kicks that follow a drift too long to rotate through (from level 5 on, and at every
// stage of level 0): the angle is split as x = k (2 pi / T) + r, |r| <= pi / T, the pair of the grid point k mod T comes
// from a table of T = 256 correctly rounded (sin, cos) values in shared memory (csrc/aw_trig_table.h, whole circle),
// and is rotated by the residual r with the same short Taylor series as the drift rotations (|r| <= 0.0123: sin to
// r^5, truncation 8e-18; cos - 1 to r^6, truncation 1e-20).
// Against the device sincos of aw_trig.cuh (19 fp64 + ~12 integer-pipe instructions for the quadrant swap and signs)
// this is 15 fp64 + 3 (shift, mask-or, 16-byte shared load): there is no quadrant logic, and it was the integer
// work, one issue cycle each, that held the sincos-bound kernels at ~80 % of the fp64 pipe (profiles/r2a_*).
// Shared-memory layout: the lanes of a warp look up unrelated entries, and a 16-byte load is served a quarter-warp
// (8 lanes) at a time, so a plain array costs ~10 wavefronts per load in bank conflicts and the kernel becomes
// shared-memory bound (profiles/r2b_*: l1tex data-pipe wavefronts 99.7 % of peak).  The table is therefore stored 8
// times, row k = the 8 copies of entry k (128 bytes = all 32 banks), and lane l reads copy l mod 8: the 8 lanes of a
// quarter-warp hit 8 different bank groups whatever their k, i.e. 4 wavefronts per load, the minimum.  32 KB per block.
// Accuracy: |error| <= 2 ulp(max(|result|, sin(2 pi / T) = 0.0123)): 2 ulp wherever |result| >= 0.0123, and an absolute
// 3.5e-18 (0.016 ulp of the amplitude) nearer a zero of the function, where the result is the difference of a table
// entry and a correction of the same size (tests/test_gpu_parity_r2.py, test_table_sincos_within_2ulp).
// Exact at x = 0 (r = 0, entry 0 = (0, 1)); the table is mirror-symmetric, so sin stays bit-odd and cos bit-even.
constexpr int kTab = 1 << AW_TAB_LOG2;
constexpr int kTabCopies = 4;
static_assert(AW_TAB_LOG2 == 9, "tsincos: the polynomial degrees below are sized for T = 512");

// The table handle a thread carries: the shared array and the byte offset of its copy, (lane mod 8) * 16.  The entry
// address is base + (((q << 7) & ((T - 1) << 7)) | lane_off): one shift, one three-input logic op, one load.
struct TrigTable {
  const char *base;
  unsigned lane_off;
};

__device__ __forceinline__ void tsincos(const TrigTable &tab, double x, double &s, double &c) {
  const double j = fma(x, AW_TAB_INV_STEP, kRintMagic);  // round-to-nearest-even of x T / 2 pi in the low mantissa bits
  const int q = __double2loint(j);
  const double k = j - kRintMagic;
  double r = fma(-k, AW_TAB_STEP_HI, x);                 // exact: the difference is representable (|x| < 1024, R7)
  r = fma(-k, AW_TAB_STEP_LO, r);
  const unsigned off = (((unsigned)q << 6) & ((unsigned)(kTab - 1) << 6)) | tab.lane_off;
  const double2 e = *reinterpret_cast<const double2 *>(tab.base + off);
  const double z = r * r;
  const double pg = fma(z, 0x1.1111111111111p-7, -0x1.5555555555555p-3);      //  1/120, -1/6
  const double pm = fma(z, AW_TAB_COS_C1, -0.5);                             //  1/24 adjusted (economised), -1/2
  // sin r = r (1 + z pg): the rounding of 1 + z pg (1 ulp of a correction below 0.013) is far below ulp(sin x), and
  // the product form keeps every instruction at two register operands (a three-register DFMA issues in 3 cycles)
  const double g = r * fma(z, pg, 1.0);
  const double m = z * pm;                               // cos r - 1
  const double t1 = fma(e.x, m, e.x), t2 = fma(e.y, m, e.y);
  s = fma(e.y, g, t1);
  c = fma(-e.x, g, t2);
}

// How a kernel sets the table up (written out where the __shared__ array is declared: through helper functions the
// compiler loses the shared address space of the array and adds the base with an extra instruction per load):
//     __shared__ double2 tab_s[kTab * kTabCopies];
//     for (int i = threadIdx.x; i < kTab * kTabCopies; i += blockDim.x)
//       tab_s[i] = make_double2(aw_trig_table[2 * (i / kTabCopies)], aw_trig_table[2 * (i / kTabCopies) + 1]);
//     __syncthreads();
//     const TrigTable tab = {reinterpret_cast<const char *>(tab_s), (threadIdx.x & (kTabCopies - 1)) * 16u};

}  // namespace aw
