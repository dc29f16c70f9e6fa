// aw_integrate.cu — §8(a) a2 + a3 + a4: the integrator kernel.
//
// One trajectory per thread ("complete parallelisation"); the six state words, the six tangent
// words and the running (sin, cos) pairs live in registers for the whole launch; HBM is touched at launch
// start and end, plus one read-modify-write of the accumulator planes per checkpoint.  The stage loop is
// fully unrolled so a_s, b_s, 2b_s, 4b_s are constant-bank operands.  Bound by the fp64 pipe.
//
// Scheme (ref. 25; R2): for s = 1..S { X += a_s P ; P -= b_s grad H_p(X) }  X += a_{S+1} P.
// Inside a block of `stride` steps the closing drift of a step and the opening drift of the next are
// one FMA with the constant a_{S+1} + a_1 (same map, one rounding fewer; DESIGN.md §7 D3).  A block is
//   X += a_1 P;  stride x { for s: kick_s; X += a_loop[s] P };  X -= a_1 P;  checkpoint
// (a_1 = a_{S+1} for the palindromic stage lists, so the last merged drift minus a_1 P is the closing drift).
// Model (eq. 2) with F = 1 + cos 2z:  H_p = cx cy F,
//   grad H_p = (-sx cy F, -cx sy F, -2 cx cy sin 2z),  Hessian in SURVEY.md Appendix A.2.
//
// Trigonometry.  LEVEL 0: the device sincos (aw_trig.cuh) of x, y, z at every stage.
// LEVEL >= 1: the pairs (sin x, cos x), (sin y, cos y), (sin 2z, cos 2z) are carried in registers and
// advanced through every drift X += a P by the rotation with the drift angle d = a p (2 a pz for 2z):
//     s' = s + (s m + c g),  c' = c + (c m - s g),   g = sin d = p G(p^2),  m = cos d - 1 = p^2 M(p^2),
// G and M being the Taylor polynomials of sin and cos - 1 with the powers of a folded into their
// coefficients on the host (constant-bank operands); the degree is picked on the host from the largest
// possible |d| so that the truncation error stays below 2^-60 (trig_level_for).  The pairs are
// re-synchronised from the tracked angles with the full sincos after the opening drift of every block and
// at least every kMaxChunk steps, which bounds the rounding random walk of the rotations at a few 1e-15.
//
// Instruction shapes (profiles/r1c_dfma_operands.md): on sm_100 a DFMA that reads three distinct 64-bit
// registers issues every 3 cycles instead of 2 unless one operand comes from the operand-reuse cache, the
// constant bank or an immediate.  The code below therefore keeps polynomial coefficients and stage
// constants in the constant bank and writes the remaining three-register FMAs in groups that share an
// operand in the same slot (the rotation's g, the kick's F, the tangent map's column vector).
#include <cmath>

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

// g = sin(A p), m = cos(A p) - 1 as p G(z), z M(z), z = p^2: N + (N-1) FMA with constant-bank coefficients,
// 3 DMUL.  Truncation: |d|^(2N+3)/(2N+3)! in g, |d|^(2N+2)/(2N+2)! in m (d = A p).
template <int N>
__device__ __forceinline__ void small_sincos(double p, const double (&G)[kTrigTerms + 1],
                                             const double (&M)[kTrigTerms], double &g, double &m) {
  static_assert(N >= 1 && N <= kTrigTerms, "degree");
  const double z = p * p;
  double pg = G[N], pm = M[N - 1];
#pragma unroll
  for (int i = N - 1; i >= 0; --i) pg = fma(pg, z, G[i]);
#pragma unroll
  for (int i = N - 2; i >= 0; --i) pm = fma(pm, z, M[i]);
  g = p * pg;
  m = z * pm;
}

// The same two functions of the angle d itself, with the universal Taylor coefficients: used by the 7-stage
// scheme, whose four distinct drift constants would otherwise need four sets of leading coefficients in
// registers (a DFMA takes one constant-bank operand at most).  N + (N-1) FMA, 3 DMUL, plus d = A p outside.
template <int N>
__device__ __forceinline__ void small_sincos_angle(double d, double &g, double &m) {
  constexpr double Sc[5] = {-1.0 / 6.0, 1.0 / 120.0, -1.0 / 5040.0, 1.0 / 362880.0, -1.0 / 39916800.0};
  constexpr double Cc[5] = {-1.0 / 2.0, 1.0 / 24.0, -1.0 / 720.0, 1.0 / 40320.0, -1.0 / 3628800.0};
  static_assert(N >= 1 && N <= 5, "degree");
  const double z = d * d;
  double pg = Sc[N - 1], pm = Cc[N - 1];
#pragma unroll
  for (int i = N - 2; i >= 0; --i) {
    pg = fma(pg, z, Sc[i]);
    pm = fma(pm, z, Cc[i]);
  }
  pg = fma(pg, z, 1.0);
  g = d * pg;
  m = z * pm;
}

// (s, c) <- rotation of (s, c) by the angle whose sine is g and cosine is 1 + m; <= 1 ulp each.
__device__ __forceinline__ void rotate(double &s, double &c, double g, double m) {
  const double t1 = fma(s, m, s), t2 = fma(c, m, c);
  const double s1 = fma(c, g, t1), c1 = fma(-s, g, t2);
  s = s1;
  c = c1;
}

// Degrees (x/y pair, 2z pair) of the trigonometry levels; the angle of the 2z pair is twice as large.
template <int LEVEL> struct Deg;
template <> struct Deg<0> { static constexpr int xy = 1, z = 1; };  // unused
template <> struct Deg<1> { static constexpr int xy = 3, z = 3; };
template <> struct Deg<2> { static constexpr int xy = 3, z = 4; };
template <> struct Deg<3> { static constexpr int xy = 4, z = 4; };
template <> struct Deg<4> { static constexpr int xy = 4, z = 5; };

// Everything a thread carries between stages.
template <bool TAN>
struct Traj {
  double x, y, z, px, py, pz;
  double dx, dy, dz, dpx, dpy, dpz;
  double sx, cx, sy, cy, s2, c2;  // sin x, cos x, sin y, cos y, sin 2z, cos 2z (LEVEL >= 1)
};

// angles (and tangent angles) only: X += a P
template <bool TAN>
__device__ __forceinline__ void drift_angles(Traj<TAN> &t, double a) {
  t.x = fma(a, t.px, t.x); t.y = fma(a, t.py, t.y); t.z = fma(a, t.pz, t.z);
  if (TAN) { t.dx = fma(a, t.dpx, t.dx); t.dy = fma(a, t.dpy, t.dy); t.dz = fma(a, t.dpz, t.dz); }
}

// drift after kick s of the step loop: angles and, for LEVEL >= 1, the running pairs.  The stage lists are
// palindromic, so a_loop[s] == a_loop[S-2-s] for s < S-1: both use the coefficient set of the smaller index
// (fewer distinct constants for the compiler to keep at hand).
template <int S, bool TAN, int LEVEL, int s>
__device__ __forceinline__ void drift(Traj<TAN> &t, const IntegrateParams &p) {
  constexpr int cs = (s == S - 1) ? s : (s < S - 2 - s ? s : S - 2 - s);
  if (LEVEL > 0) {
    double g, m;
    if (S <= 3) {
      small_sincos<Deg<LEVEL>::xy>(t.px, p.gxy[cs], p.mxy[cs], g, m);
      rotate(t.sx, t.cx, g, m);
      small_sincos<Deg<LEVEL>::xy>(t.py, p.gxy[cs], p.mxy[cs], g, m);
      rotate(t.sy, t.cy, g, m);
      small_sincos<Deg<LEVEL>::z>(t.pz, p.gz[cs], p.mz[cs], g, m);
      rotate(t.s2, t.c2, g, m);
    } else {
      small_sincos_angle<Deg<LEVEL>::xy>(p.a_loop[cs] * t.px, g, m);
      rotate(t.sx, t.cx, g, m);
      small_sincos_angle<Deg<LEVEL>::xy>(p.a_loop[cs] * t.py, g, m);
      rotate(t.sy, t.cy, g, m);
      small_sincos_angle<Deg<LEVEL>::z>(p.a2_loop[cs] * t.pz, g, m);
      rotate(t.s2, t.c2, g, m);
    }
  }
  drift_angles<TAN>(t, p.a_loop[cs]);
}

template <bool TAN, int LEVEL>
__device__ __forceinline__ void resync(Traj<TAN> &t) {
  if (LEVEL > 0) {
    sincos(t.x, t.sx, t.cx);
    sincos(t.y, t.sy, t.cy);
    sincos(2.0 * t.z, t.s2, t.c2);
  }
}

// kick of stage s: P -= b grad H_p(X), dP -= b Hess H_p(X) dX (R3), b1 = b, b2 = 2b, b4 = 4b
template <bool TAN, int LEVEL>
__device__ __forceinline__ void kick(Traj<TAN> &t, double b1, double b2, double b4) {
  if (LEVEL == 0) {
    double sz, cz;
    sincos(t.x, t.sx, t.cx);
    sincos(t.y, t.sy, t.cy);
    sincos(t.z, sz, cz);
    t.c2 = fma(cz + cz, cz, -1.0);  // cos 2z = 2 cz^2 - 1
    t.s2 = (sz + sz) * cz;          // sin 2z
  }
  const double F = fma(b1, t.c2, b1);  // b (1 + cos 2z)
  const double G = b2 * t.s2;          // 2 b sin 2z
  const double c = t.cx * t.cy, sc = t.sx * t.cy, cs = t.cx * t.sy;
  t.px = fma(sc, F, t.px);
  t.py = fma(cs, F, t.py);
  t.pz = fma(c, G, t.pz);
  if (TAN) {
    // rows of -b Hess H_p: (e1,-e2,-e3), (-e2,e1,-e4), (-e3,-e4,e5); applied column by column so that
    // consecutive FMAs share the tangent component (operand-reuse cache) and are independent
    const double ss = t.sx * t.sy;
    const double e1 = c * F, e2 = ss * F, e3 = sc * G, e4 = cs * G;
    const double e5 = c * (b4 * t.c2);  // 4 b cx cy cos 2z
    t.dpx = fma(e1, t.dx, t.dpx); t.dpy = fma(-e2, t.dx, t.dpy); t.dpz = fma(-e3, t.dx, t.dpz);
    t.dpx = fma(-e2, t.dy, t.dpx); t.dpy = fma(e1, t.dy, t.dpy); t.dpz = fma(-e4, t.dy, t.dpz);
    t.dpx = fma(-e3, t.dz, t.dpx); t.dpy = fma(-e4, t.dz, t.dpy); t.dpz = fma(e5, t.dz, t.dpz);
  }
}

// stages s, s+1, ..., S-1 of one step: kick_s then the drift after it
template <int S, bool TAN, int LEVEL, int s>
__device__ __forceinline__ void stages(Traj<TAN> &t, const IntegrateParams &p) {
  if constexpr (s < S) {
    kick<TAN, LEVEL>(t, p.b1[s], p.b2[s], p.b4[s]);
    drift<S, TAN, LEVEL, s>(t, p);
    stages<S, TAN, LEVEL, s + 1>(t, p);
  }
}

template <int S, bool TAN, int LEVEL>
__global__ void __launch_bounds__(AW_BLOCK, AW_MIN_BLOCKS)
    integrate_kernel(const __grid_constant__ IntegrateParams p) {
  const int64_t k = (int64_t)blockIdx.x * AW_BLOCK + threadIdx.x;
  if (k >= p.n) return;
  if (p.status[k] != AW_ST_LIVE) return;
  const int64_t P = p.pitch;

  Traj<TAN> t;
  t.x = p.q[k]; t.y = p.q[P + k]; t.z = p.q[2 * P + k];
  t.px = p.q[3 * P + k]; t.py = p.q[4 * P + k]; t.pz = p.q[5 * P + k];
  if (TAN) {
    t.dx = p.w[k]; t.dy = p.w[P + k]; t.dz = p.w[2 * P + k];
    t.dpx = p.w[3 * P + k]; t.dpy = p.w[4 * P + k]; t.dpz = p.w[5 * P + k];
  }
  int status = AW_ST_LIVE;

  for (int chk = 0; chk < p.nchk; ++chk) {
    drift_angles<TAN>(t, p.a_open);  // opening drift of the block
    resync<TAN, LEVEL>(t);           // pairs from the angles: the same values a new launch would start from

#pragma unroll 1
    for (int rem = p.stride; rem > 0;) {
      const int m = rem < p.chunk ? rem : p.chunk;
      rem -= m;
#pragma unroll 1
      for (int i = m; i > 0; --i) stages<S, TAN, LEVEL, 0>(t, p);
      if (rem > 0) resync<TAN, LEVEL>(t);
    }
    drift_angles<TAN>(t, -p.a_open);  // last merged drift -> closing drift of the block

    // ---- fused checkpoint (R4): (i) renormalise + log growth, (ii) energy error, (iii) wrap
    bool finite = true;
    if (TAN) {
      double s2 = t.dx * t.dx;
      s2 = fma(t.dy, t.dy, s2); s2 = fma(t.dz, t.dz, s2);
      s2 = fma(t.dpx, t.dpx, s2); s2 = fma(t.dpy, t.dpy, s2); s2 = fma(t.dpz, t.dpz, s2);
      const double nu = sqrt(s2);
      const double inv = 1.0 / nu;
      t.dx *= inv; t.dy *= inv; t.dz *= inv; t.dpx *= inv; t.dpy *= inv; t.dpz *= inv;
      const double logsum = p.acc[k] + log(nu);
      p.acc[k] = logsum;
      if (logsum > p.acc[P + k]) p.acc[P + k] = logsum;
      finite = isfinite(t.dx) && isfinite(t.dy) && isfinite(t.dz) && isfinite(t.dpx) && isfinite(t.dpy) &&
               isfinite(t.dpz);
    }
    const double dH = fabs(hamiltonian_dev(t.x, t.y, t.z, t.px, t.py, t.pz, p.eps) - p.acc[2 * P + k]);
    if (dH > p.acc[3 * P + k]) p.acc[3 * P + k] = dH;
    int tx, ty, tz;
    t.x = wrap_angle(t.x, tx); t.y = wrap_angle(t.y, ty); t.z = wrap_angle(t.z, tz);
    if (p.wind) {
      p.wind[k] += tx; p.wind[P + k] += ty; p.wind[2 * P + k] += tz;
    }
    finite = finite && isfinite(t.x) && isfinite(t.y) && isfinite(t.z) && isfinite(t.px) && isfinite(t.py) &&
             isfinite(t.pz);
    if (!finite) { status = AW_ST_NONFINITE; break; }
    // survivor filter (R25): outside the launch rectangle at a checkpoint -> dropped, frozen here
    if (p.survive && !(t.px >= p.surv[0] && t.px < p.surv[1] && t.py >= p.surv[2] && t.py < p.surv[3])) {
      status = AW_ST_LEFT;
      break;
    }
  }

  p.q[k] = t.x; p.q[P + k] = t.y; p.q[2 * P + k] = t.z;
  p.q[3 * P + k] = t.px; p.q[4 * P + k] = t.py; p.q[5 * P + k] = t.pz;
  if (TAN) {
    p.w[k] = t.dx; p.w[P + k] = t.dy; p.w[2 * P + k] = t.dz;
    p.w[3 * P + k] = t.dpx; p.w[4 * P + k] = t.dpy; p.w[5 * P + k] = t.dpz;
  }
  if (status != AW_ST_LIVE) p.status[k] = (uint8_t)status;
}

template <int S, bool TAN, int LEVEL>
cudaError_t launch_one(const IntegrateParams &p, cudaStream_t st) {
  const int64_t blocks = (p.n + AW_BLOCK - 1) / AW_BLOCK;
  integrate_kernel<S, TAN, LEVEL><<<(unsigned)blocks, AW_BLOCK, 0, st>>>(p);
  count_launch();
  return cudaGetLastError();
}

template <int S, bool TAN>
cudaError_t launch_level(const IntegrateParams &p, cudaStream_t st) {
  switch (p.level) {
    case 1: return launch_one<S, TAN, 1>(p, st);
    case 2: return launch_one<S, TAN, 2>(p, st);
    case 3: return launch_one<S, TAN, 3>(p, st);
    case 4: return launch_one<S, TAN, 4>(p, st);
    default: return launch_one<S, TAN, 0>(p, st);
  }
}

}  // namespace

// Largest |d| each level may see on the x/y pairs (the 2z pair sees 2|d|) with both Taylor truncations
// below 2^-60 ~ 8.7e-19 (they are systematic, so 300 of them still sum to < 3e-16):
//   m of degree N truncates at |d|^(2N+2)/(2N+2)!, g at |d|^(2N+3)/(2N+3)!:
//   N = 3: |d| <= 0.0208 (m), 0.0408 (g);  N = 4: 0.0708, 0.112;  N = 5: 0.165, 0.23.
// level 1 = (3,3): 2|d| <= 0.0208;  level 2 = (3,4): |d| <= 0.0208;  level 3 = (4,4): 2|d| <= 0.0708;
// level 4 = (4,5): |d| <= 0.0708;  beyond: level 0 (full sincos every stage).
int trig_level_for(double d) {
  if (!(d == d)) return 0;
  if (d <= 0.0104) return 1;
  if (d <= 0.0208) return 2;
  if (d <= 0.0354) return 3;
  if (d <= 0.0708) return 4;
  return 0;
}

cudaError_t launch_integrate(const IntegrateParams &p, int order, bool tangent, cudaStream_t st) {
  if (order == 4) return tangent ? launch_level<3, true>(p, st) : launch_level<3, false>(p, st);
  return tangent ? launch_level<7, true>(p, st) : launch_level<7, false>(p, st);
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
