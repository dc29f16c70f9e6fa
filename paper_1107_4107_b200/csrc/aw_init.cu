// aw_init.cu — §8(a) a1: initial conditions on the energy shell (R6, R8-R12, R17, R18).
//
// One thread per trajectory, one pass, HBM-write bound (48 + 48 + 32 + 12 + 1 bytes per trajectory).
// The grid arithmetic uses the explicit-rounding intrinsics (__dmul_rn, ...) so that no product/sum is
// contracted into an FMA: px, py are then bit-equal to the plain definition
//   px = lo_x + ((i + 1/2) (hi_x - lo_x)) / gx          (cell-centred, k = j*gx + i; R6).
#include "aw_internal.cuh"
#include "aw_model.cuh"

namespace aw {

namespace {

constexpr double kTwoPiHi = 6.283185307179586;  // double nearest 2 pi

// two standard normals from slots (slot, slot+1): Box-Muller on (1 - u_a, u_b)
__device__ __forceinline__ void normal_pair(uint64_t seed, uint64_t k, uint64_t slot, double &n1, double &n2) {
  const double ua = uniform01(seed, k, slot), ub = uniform01(seed, k, slot + 1);
  const double rad = sqrt(-2.0 * log(1.0 - ua));
  double sn, cs;
  sincos(kTwoPiHi * ub, sn, cs);
  n1 = rad * cs;
  n2 = rad * sn;
}

__global__ void __launch_bounds__(256) init_shell_kernel(const __grid_constant__ InitParams p) {
  const int64_t k = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (k >= p.n) return;
  const int64_t P = p.pitch;
  const aw_grid &g = p.g;
  // K: index in the whole ensemble the grid describes (grid position, random-number counter); k: slot in the planes
  const int64_t K = g.k0 + k;
  const int64_t i = K % g.gx, j = K / g.gx;
  const uint64_t uk = (uint64_t)K;

  const double nan = __longlong_as_double(0x7ff8000000000000ll);
  const double sgn = g.pz_sign < 0 ? -1.0 : 1.0;
  double x = 0.0, y = 0.0, z = 0.0, px = nan, py = nan, pz = nan, H0 = nan;
  bool live = false;
  // cloud shapes with resample > 0: draw again until the point has a real third action (R31; include/aw.h)
  const int attempts =
      (g.shape == AW_SHAPE_DISK || g.shape == AW_SHAPE_GAUSS || g.shape == AW_SHAPE_RECT) && g.resample > 0 ? g.resample + 1 : 1;
  for (int a = 0; a < attempts && !live; ++a) {
    const uint64_t sd = p.seed + (uint64_t)a * 0xD1B54A32D192ED03ull;
    if (g.angle_mode == 1) {
      x = kTwoPiHi * uniform01(sd, uk, 0);
      y = kTwoPiHi * uniform01(sd, uk, 1);
      z = kTwoPiHi * uniform01(sd, uk, 2);
    }
    if (g.shape == AW_SHAPE_SPHERE) {
      // direction uniform on the unit sphere, |P| from the energy condition (R28); always on the shell
      const double u1 = uniform01(sd, uk, 3), u2 = uniform01(sd, uk, 4);
      const double ct = __dsub_rn(1.0, __dmul_rn(2.0, u1));
      const double sth = sqrt(__dmul_rn(__dsub_rn(1.0, ct), __dadd_rn(1.0, ct)));
      double sn, cs;
      sincos(kTwoPiHi * u2, sn, cs);
      const double pn = sqrt(__dmul_rn(2.0, __dsub_rn(p.E, __dmul_rn(p.eps, hp_dev(x, y, z)))));
      px = __dmul_rn(pn, __dmul_rn(sth, cs));
      py = __dmul_rn(pn, __dmul_rn(sth, sn));
      pz = sgn * __dmul_rn(pn, ct);
      live = true;
    } else {
      if (g.shape == AW_SHAPE_GRID) {
        px = __dadd_rn(g.lo_x, __ddiv_rn(__dmul_rn(__dadd_rn((double)i, 0.5), __dsub_rn(g.hi_x, g.lo_x)), (double)g.gx));
        py = __dadd_rn(g.lo_y, __ddiv_rn(__dmul_rn(__dadd_rn((double)j, 0.5), __dsub_rn(g.hi_y, g.lo_y)), (double)g.gy));
      } else if (g.shape == AW_SHAPE_RECT) {
        // uniform random points of a rectangle in (px, py) (R33)
        const double u1 = uniform01(sd, uk, 3), u2 = uniform01(sd, uk, 4);
        px = __dadd_rn(g.lo_x, __dmul_rn(u1, __dsub_rn(g.hi_x, g.lo_x)));
        py = __dadd_rn(g.lo_y, __dmul_rn(u2, __dsub_rn(g.hi_y, g.lo_y)));
      } else {
        const double u1 = uniform01(sd, uk, 3), u2 = uniform01(sd, uk, 4);
        const double rad = (g.shape == AW_SHAPE_DISK) ? __dmul_rn(g.r, sqrt(u1))
                                                      : __dmul_rn(g.r, sqrt(-2.0 * log(1.0 - u1)));
        double sn, cs;
        sincos(kTwoPiHi * u2, sn, cs);
        px = __dadd_rn(g.cx, __dmul_rn(rad, cs));
        py = __dadd_rn(g.cy, __dmul_rn(rad, sn));
      }
      // third action from the energy condition H = E: pz^2 = 2(E - eps H_p) - px^2 - py^2
      double R = __dmul_rn(2.0, __dsub_rn(p.E, __dmul_rn(p.eps, hp_dev(x, y, z))));
      R = __dsub_rn(R, __dmul_rn(px, px));
      R = __dsub_rn(R, __dmul_rn(py, py));
      live = R >= 0.0;  // false for NaN too
      if (live) pz = sgn * sqrt(R);
    }
  }
  if (live) {
    H0 = hamiltonian_dev(x, y, z, px, py, pz, p.eps);
  } else {
    x = y = z = px = py = nan;
  }
  p.q[k] = x; p.q[P + k] = y; p.q[2 * P + k] = z;
  p.q[3 * P + k] = px; p.q[4 * P + k] = py; p.q[5 * P + k] = pz;
  p.acc[k] = 0.0; p.acc[P + k] = 0.0; p.acc[2 * P + k] = H0; p.acc[3 * P + k] = 0.0;
  p.status[k] = live ? AW_ST_LIVE : AW_ST_OFFSHELL;
  if (p.wind) { p.wind[k] = 0; p.wind[P + k] = 0; p.wind[2 * P + k] = 0; }
  if (p.w) {
    double t[6];
    if (g.tangent_mode == 1) {
      normal_pair(p.seed, uk, 5, t[0], t[1]);
      normal_pair(p.seed, uk, 7, t[2], t[3]);
      normal_pair(p.seed, uk, 9, t[4], t[5]);
      double s2 = 0.0;
#pragma unroll
      for (int c = 0; c < 6; ++c) s2 = __dadd_rn(s2, __dmul_rn(t[c], t[c]));
      const double nu = sqrt(s2);
#pragma unroll
      for (int c = 0; c < 6; ++c) t[c] = t[c] / nu;
    } else {
#pragma unroll
      for (int c = 0; c < 6; ++c) t[c] = p.tcommon[c];
    }
#pragma unroll
    for (int c = 0; c < 6; ++c) p.w[c * P + k] = t[c];
  }
}

}  // namespace

cudaError_t launch_init(const InitParams &p, cudaStream_t st) {
  init_shell_kernel<<<(unsigned)((p.n + 255) / 256), 256, 0, st>>>(p);
  count_launch();
  return cudaGetLastError();
}

}  // namespace aw
