// aw_trig.cuh — the integrator's own fp64 sincos.
//
// Why not the CUDA library sincos(): it carries a Payne-Hanek slow path (local memory, a branch) for
// arguments the integrator never produces — angles are wrapped to [-pi, pi] at every checkpoint (R7)
// and aw_integrate refuses strides that let |x| reach 1024 rad — and a three-constant reduction.
// This one is branch-free, FMA-only on the fp64 pipe, with the quadrant logic on the integer pipes:
//
//   j = fma(x, 2/pi, 1.5*2^52)            round-to-nearest-even of x*2/pi lands in the low mantissa bits
//   k = j - 1.5*2^52 ; q = lo32(j)        k exact integer as double, q the same integer mod 2^32
//   r = fma(-k, PIO2_HI, x)               exact for |k| < 2^11 (the difference is representable)
//   r = fma(-k, PIO2_LO, r)               |error| <= ulp(r)/2 + |k| * 2^-109
//   sin r = r + (r z) S(z), cos r = fma(z, fma(z, C(z), -1/2), 1),   z = r^2   (csrc/aw_trig_coeffs.h)
//   quadrant: q odd -> swap;  q & 2 -> negate sin;  (q + 1) & 2 -> negate cos.
//
// 19 fp64 instructions (16 DFMA, 2 DMUL, 1 DADD) per sincos.  Exact at 0; sin bit-odd, cos bit-even.
#pragma once
#include "aw_trig_coeffs.h"

namespace aw {

constexpr double kTwoOverPi = 0x1.45f306dc9c883p-1;  // double nearest 2/pi
constexpr double kPio2Hi = 0x1.921fb54442d18p+0;     // double nearest pi/2
constexpr double kPio2Lo = 0x1.1a62633145c07p-54;    // pi/2 - kPio2Hi, rounded
constexpr double kRintMagic = 6755399441055744.0;    // 1.5 * 2^52

__device__ __forceinline__ void sincos_core(double x, double &sn, double &cs, int &q) {
  const double j = fma(x, kTwoOverPi, kRintMagic);
  q = __double2loint(j);
  const double k = j - kRintMagic;
  double r = fma(-k, kPio2Hi, x);
  r = fma(-k, kPio2Lo, r);
  const double z = r * r;
  double ps = fma(z, AW_SIN_S6, AW_SIN_S5);
  double pc = fma(z, AW_COS_C6, AW_COS_C5);
  ps = fma(ps, z, AW_SIN_S4);
  pc = fma(pc, z, AW_COS_C4);
  ps = fma(ps, z, AW_SIN_S3);
  pc = fma(pc, z, AW_COS_C3);
  ps = fma(ps, z, AW_SIN_S2);
  pc = fma(pc, z, AW_COS_C2);
  ps = fma(ps, z, AW_SIN_S1);
  pc = fma(pc, z, AW_COS_C1);
  const double rz = r * z;
  pc = fma(pc, z, -0.5);
  sn = fma(rz, ps, r);
  cs = fma(pc, z, 1.0);
}

// Conditional negate by flipping the sign bit of the high word (integer pipe, not fp64).
__device__ __forceinline__ double flip_sign_if(double v, unsigned bit31) {
  return __hiloint2double(__double2hiint(v) ^ (int)bit31, __double2loint(v));
}

__device__ __forceinline__ void sincos(double x, double &s, double &c) {
  double sn, cs;
  int q;
  sincos_core(x, sn, cs, q);
  const bool odd = q & 1;
  const double s0 = odd ? cs : sn;
  const double c0 = odd ? sn : cs;
  s = flip_sign_if(s0, ((unsigned)q & 2u) << 30);
  c = flip_sign_if(c0, ((unsigned)(q + 1) & 2u) << 30);
}

}  // namespace aw
