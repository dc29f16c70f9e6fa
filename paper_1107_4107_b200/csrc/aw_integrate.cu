// aw_integrate.cu — §8(a) a2 + a3 + a4: the integrator kernel.
//
// One trajectory per thread ("complete parallelisation"), the six state words and the six tangent
// words live in registers for the whole launch; HBM is touched at launch start and end, plus one
// read-modify-write of the accumulator planes per checkpoint.  The stage loop is fully unrolled so
// a_s, 2b_s, 4b_s are constant-bank operands.  Bound by the fp64 pipe: per stage 3 sincos (57 fp64
// instructions) + 3 drift + 11 kick (+ 3 + 16 with the tangent map).
//
// Scheme (ref. 25; R2): for s = 1..S { X += a_s P ; P -= b_s grad H_p(X) }  X += a_{S+1} P.
// Inside a block of `stride` steps the closing drift of a step and the opening drift of the next are
// one FMA with the constant a_{S+1} + a_1 (same map, one rounding fewer; DESIGN.md §7 D3).
// Model (eq. 2) with u = cos^2 z, d = sin z cos z:  H_p = 2 cx cy u,
//   grad H_p = (-2 sx cy u, -2 cx sy u, -4 cx cy d),  Hessian in SURVEY.md Appendix A.2.
#include "aw_internal.cuh"
#include "aw_model.cuh"
#include "aw_trig.cuh"

#ifndef AW_BLOCK
#define AW_BLOCK 128
#endif
#ifndef AW_MIN_BLOCKS
#define AW_MIN_BLOCKS 4
#endif

namespace aw {

namespace {

constexpr double kInv2Pi = 0.15915494309189535;       // double nearest 1/(2 pi)
constexpr double kTwoPiHi = 6.283185307179586;        // double nearest 2 pi
constexpr double kTwoPiLo = 2.4492935982947064e-16;   // 2 pi - kTwoPiHi

__device__ __forceinline__ double wrap_angle(double x, int &turns) {
  const double k = rint(x * kInv2Pi);
  turns = (int)k;
  return fma(-k, kTwoPiLo, fma(-k, kTwoPiHi, x));
}

template <int S, bool TAN>
__global__ void __launch_bounds__(AW_BLOCK, AW_MIN_BLOCKS)
    integrate_kernel(const __grid_constant__ IntegrateParams p) {
  const int64_t k = (int64_t)blockIdx.x * AW_BLOCK + threadIdx.x;
  if (k >= p.n) return;
  if (p.status[k] != AW_ST_LIVE) return;
  const int64_t P = p.pitch;

  double x = p.q[k], y = p.q[P + k], z = p.q[2 * P + k];
  double px = p.q[3 * P + k], py = p.q[4 * P + k], pz = p.q[5 * P + k];
  double dx = 0, dy = 0, dz = 0, dpx = 0, dpy = 0, dpz = 0;
  if (TAN) {
    dx = p.w[k]; dy = p.w[P + k]; dz = p.w[2 * P + k];
    dpx = p.w[3 * P + k]; dpy = p.w[4 * P + k]; dpz = p.w[5 * P + k];
  }
  int status = AW_ST_LIVE;

  for (int chk = 0; chk < p.nchk; ++chk) {
    // opening drift of the block
    x = fma(p.a_first, px, x); y = fma(p.a_first, py, y); z = fma(p.a_first, pz, z);
    if (TAN) { dx = fma(p.a_first, dpx, dx); dy = fma(p.a_first, dpy, dy); dz = fma(p.a_first, dpz, dz); }

#pragma unroll 1
    for (int i = p.stride; i > 0; --i) {
#pragma unroll
      for (int s = 0; s < S; ++s) {
        double sx, cx, sy, cy, sz, cz;
        sincos(x, sx, cx);
        sincos(y, sy, cy);
        sincos(z, sz, cz);
        const double u = cz * cz, d = sz * cz;
        const double U = p.b2[s] * u;  // 2 b u
        const double D = p.b4[s] * d;  // 4 b d
        const double c = cx * cy, sc = sx * cy, cs = cx * sy;
        // kick: P -= b grad H_p
        px = fma(sc, U, px);
        py = fma(cs, U, py);
        pz = fma(c, D, pz);
        if (TAN) {
          // tangent kick: dP -= b Hess H_p dX, rows (e1,-e2,-e3), (-e2,e1,-e4), (-e3,-e4,e5)
          const double ss = sx * sy;
          const double e1 = c * U, e2 = ss * U, e3 = sc * D, e4 = cs * D;
          const double e5 = c * fma(4.0, U, -p.b4[s]);  // 4 b c (2u - 1)
          dpx = fma(e1, dx, dpx); dpx = fma(-e2, dy, dpx); dpx = fma(-e3, dz, dpx);
          dpy = fma(e1, dy, dpy); dpy = fma(-e2, dx, dpy); dpy = fma(-e4, dz, dpy);
          dpz = fma(e5, dz, dpz); dpz = fma(-e3, dx, dpz); dpz = fma(-e4, dy, dpz);
        }
        if (s < S - 1) {
          const double a = p.a_mid[s];
          x = fma(a, px, x); y = fma(a, py, y); z = fma(a, pz, z);
          if (TAN) { dx = fma(a, dpx, dx); dy = fma(a, dpy, dy); dz = fma(a, dpz, dz); }
        }
      }
      const double a = (i == 1) ? p.a_last : p.a_merge;
      x = fma(a, px, x); y = fma(a, py, y); z = fma(a, pz, z);
      if (TAN) { dx = fma(a, dpx, dx); dy = fma(a, dpy, dy); dz = fma(a, dpz, dz); }
    }

    // ---- fused checkpoint (R4): (i) renormalise + log growth, (ii) energy error, (iii) wrap
    bool finite = true;
    if (TAN) {
      double s2 = dx * dx;
      s2 = fma(dy, dy, s2); s2 = fma(dz, dz, s2);
      s2 = fma(dpx, dpx, s2); s2 = fma(dpy, dpy, s2); s2 = fma(dpz, dpz, s2);
      const double nu = sqrt(s2);
      const double inv = 1.0 / nu;
      dx *= inv; dy *= inv; dz *= inv; dpx *= inv; dpy *= inv; dpz *= inv;
      const double logsum = p.acc[k] + log(nu);
      p.acc[k] = logsum;
      if (logsum > p.acc[P + k]) p.acc[P + k] = logsum;
      finite = isfinite(dx) && isfinite(dy) && isfinite(dz) && isfinite(dpx) && isfinite(dpy) &&
               isfinite(dpz);
    }
    const double dH = fabs(hamiltonian_dev(x, y, z, px, py, pz, p.eps) - p.acc[2 * P + k]);
    if (dH > p.acc[3 * P + k]) p.acc[3 * P + k] = dH;
    int tx, ty, tz;
    x = wrap_angle(x, tx); y = wrap_angle(y, ty); z = wrap_angle(z, tz);
    if (p.wind) {
      p.wind[k] += tx; p.wind[P + k] += ty; p.wind[2 * P + k] += tz;
    }
    finite = finite && isfinite(x) && isfinite(y) && isfinite(z) && isfinite(px) && isfinite(py) &&
             isfinite(pz);
    if (!finite) { status = AW_ST_NONFINITE; break; }
  }

  p.q[k] = x; p.q[P + k] = y; p.q[2 * P + k] = z;
  p.q[3 * P + k] = px; p.q[4 * P + k] = py; p.q[5 * P + k] = pz;
  if (TAN) {
    p.w[k] = dx; p.w[P + k] = dy; p.w[2 * P + k] = dz;
    p.w[3 * P + k] = dpx; p.w[4 * P + k] = dpy; p.w[5 * P + k] = dpz;
  }
  if (status != AW_ST_LIVE) p.status[k] = (uint8_t)status;
}

template <int S, bool TAN>
cudaError_t launch_one(const IntegrateParams &p, cudaStream_t st) {
  const int64_t blocks = (p.n + AW_BLOCK - 1) / AW_BLOCK;
  integrate_kernel<S, TAN><<<(unsigned)blocks, AW_BLOCK, 0, st>>>(p);
  count_launch();
  return cudaGetLastError();
}

}  // namespace

cudaError_t launch_integrate(const IntegrateParams &p, int order, bool tangent, cudaStream_t st) {
  if (order == 4) return tangent ? launch_one<3, true>(p, st) : launch_one<3, false>(p, st);
  return tangent ? launch_one<7, true>(p, st) : launch_one<7, false>(p, st);
}

__global__ void hamiltonian_probe_kernel(const double *q, int64_t n, int64_t P, double eps, double *out) {
  const int64_t k = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (k < n) out[k] = hamiltonian_dev(q[k], q[P + k], q[2 * P + k], q[3 * P + k], q[4 * P + k], q[5 * P + k], eps);
}

cudaError_t launch_hamiltonian_probe(const double *q, int64_t n, int64_t pitch, double eps, double *out,
                                     cudaStream_t st) {
  hamiltonian_probe_kernel<<<(unsigned)((n + 255) / 256), 256, 0, st>>>(q, n, pitch, eps, out);
  count_launch();
  return cudaGetLastError();
}

}  // namespace aw
