// aw_integrate.cu — §8(a) a2 + a3 + a4: the integrator kernel.
//
// One trajectory per thread ("complete parallelisation"); the six state words, the six tangent
// words and the running (sin, cos) pairs live in registers for the whole launch; HBM is touched at launch
// start and end, plus one read-modify-write of the accumulator planes per checkpoint.  The stage loop is
// fully unrolled; the stage constants reach the fp64 instructions through uniform registers.  Bound by the
// fp64 pipe.
//
// Scheme (ref. 25; R2): for s = 1..S { X += a_s P ; P -= b_s grad H_p(X) }  X += a_{S+1} P.
// Inside a block of `stride` steps the closing drift of a step and the opening drift of the next are
// one FMA with the constant a_{S+1} + a_1 (same map, one rounding fewer; DESIGN.md §7 D3).  A block is
//   X += a_1 P;  stride x { for s: kick_s; X += a_loop[s] P };  X -= a_1 P;  checkpoint
// (a_1 = a_{S+1} for the palindromic stage lists, so the last merged drift minus a_1 P is the closing drift).
//
// Model (eq. 2): H_p = cos x cos y (1 + cos 2z) = (cos u + cos v)(1 + cos zeta)/2 in the working
// variables u = x + y, v = x - y, zeta = 2z the kernel holds inside a block, every momentum-like variable doubled
// (struct Traj below), so
//   grad H_p = -(F sin u, F sin v, (cos u + cos v) sin zeta),  F = 1 + cos zeta   (d/du, d/dv, d/dz),
// and the Hessian-vector product is the sum and difference of the x and y rows of SURVEY.md Appendix A.2; with the
// zeta pair carried scaled by 2 b_0 the kick of the first and last stage needs no constant multiplies (kick()).
//
// Trigonometry, two mechanisms chosen per drift and per pair type at compile time from the LEVEL the
// host picks (largest possible drift angle |d|) and the drift's ratio to the longest one:
// (i) the pairs (sin u, cos u), (sin v, cos v), (sin zeta, cos zeta) are carried in registers and advanced through a
// drift by the rotation with the drift angle d = A p:
//     s' = s + (s m + c g),  c' = c + (c m - s g),   g = sin d = p G(p^2),  m = cos d - 1 = p^2 M(p^2),
// G and M being the Taylor polynomials of sin and cos - 1 with the powers of A folded into their coefficients on the
// host, of the smallest degree (<= 5) that keeps the truncation below 2^-60 (rotation_degree, trig_level_for).  A
// pair type every drift rotates is re-synchronised from the tracked angle with the full sincos after the opening
// drift of every block and at least every kMaxChunk steps, which bounds the rounding random walk of the rotations at
// a few 1e-15.  (ii) After a drift too long for that, the kick evaluates the pair from the angle with the
// table-driven sincos of aw_tsincos.cuh (LEVEL 0: at every stage).
//
// Instruction shapes (profiles/r1c_dfma_operand_shapes.md): on sm_100 a DFMA that reads three distinct 64-bit
// registers issues every 3 cycles instead of 2 unless one operand comes from the operand-reuse cache, a
// uniform register or an immediate, and every non-fp64 instruction takes an issue cycle the fp64 pipe also
// needs.  The code below therefore minimises register reads and integer work, not just fp64 instructions:
// coefficients and stage constants in uniform registers, the working variables above (16 three-register
// multiply-adds per stage instead of 21), three-register FMAs written in groups that share an operand, no quadrant
// logic anywhere in the step loop.
#include <cmath>

#include "aw_internal.cuh"
#include "aw_model.cuh"
#include "aw_trig.cuh"
#include "aw_tsincos.cuh"

#ifndef AW_BLOCK
#define AW_BLOCK 128
#endif
// Register cap: __launch_bounds__(128, 3) allows 168 registers per thread; the kernels take 94-144, which still
// places 3-5 blocks per SM, and 3 warps per sub-partition already saturate the fp64 pipe.  With the cap at 128 ptxas finds fewer operand-reuse pairs in most instantiations
// (measured: configs[3] -1.1 %), except the level-4 ones (configs[2]: +1.8 % at 128), which keep 4.
#ifndef AW_MIN_BLOCKS
#define AW_MIN_BLOCKS(LEVEL) ((LEVEL) == 4 ? 4 : 3)
#endif

// This file is compiled twice (build.py), the same source and the same arithmetic under two ptxas schedules:
//   AW_LEVEL_GROUP 1, -Xptxas -O1: the lighter scheduler stays close to source order, which keeps the three-register
//     FMAs that share an operand next to each other, so more of them hit the operand-reuse cache (measured on B200:
//     configs[3] +3.5 %, configs[2] +3.5 %, order 6 +2.9 %; the table kernel of the E = 400 workload +1.9 %), and needs
//     fewer registers.  This is the THROUGHPUT flavour: best when the fp64 pipe is saturated (>= 3 warps per
//     sub-partition).
//   AW_LEVEL_GROUP 0, default flags: ptxas interleaves the independent chains of a stage (the three pairs' polynomials,
//     the three table look-ups), which is what a warp needs when it has a sub-partition almost to itself.  This is the
//     LATENCY flavour, used for small ensembles (the paper's Fig. 4 ensemble, 32 000 trajectories = 1.7 warps per
//     sub-partition: 2.94e10 -> 3.56e10 traj-steps/s; configs[0], 4096 trajectories: 1.46e10 -> 2.28e10; the same
//     kernels on 6e5 trajectories: -1 to -3 %).  It also holds the host-side functions.
// ptxas does not reassociate floating-point arithmetic, so both flavours give the same bits (tested).
#ifndef AW_LEVEL_GROUP
#define AW_LEVEL_GROUP 0
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

// g = sin(A p), m = cos(A p) - 1 as p G(z), z M(z), z = p^2: N + (N-1) FMA with uniform-register coefficients,
// 3 DMUL.  Truncation: |d|^(2N+3)/(2N+3)! in g, |d|^(2N+2)/(2N+2)! in m (d = A p).
// G[0] = A exactly, and A is the drift constant the angle FMAs of the same drift already hold in a uniform register:
// it is passed separately so that ptxas keeps ONE copy (the loop's constants do not all fit the uniform registers; the
// overflow lives in ordinary registers, where a polynomial FMA becomes a three-register one).
template <int N>
__device__ __forceinline__ void small_sincos(double p, double A, const double (&G)[kTrigTerms + 1],
                                             const double (&M)[kTrigTerms], double &g, double &m) {
  static_assert(N >= 1 && N <= kTrigTerms, "degree");
  const double z = p * p;
  double pg = G[N], pm = M[N - 1];
#pragma unroll
  for (int i = N - 1; i >= 1; --i) pg = fma(pg, z, G[i]);
  pg = fma(pg, z, A);
#pragma unroll
  for (int i = N - 2; i >= 0; --i) pm = fma(pm, z, M[i]);
  g = p * pg;
  m = z * pm;
}

// (s, c) <- rotation of (s, c) by the angle whose sine is g and cosine is 1 + m; <= 1 ulp each.
__device__ __forceinline__ void rotate(double &s, double &c, double g, double m) {
  const double t1 = fma(s, m, s), t2 = fma(c, m, c);
  const double s1 = fma(c, g, t1), c1 = fma(-s, g, t2);
  s = s1;
  c = c1;
}

// Taylor degrees of the drift rotations.  A trigonometry level L is picked on the host from
// |d| = max_s |a_s| max|P| <= kLevelMaxD[L] (trig_level_for).  The drift after kick s has its own constant
// a_loop[s]; its ratio to the largest one is fixed by the scheme (kDriftRatio, checked on the host), so each
// drift gets the smallest degree N whose truncation stays below 2^-60 for ITS largest angle: the u and v pairs
// rotate by up to sqrt(2) |a_loop[s]| max|P|, the zeta = 2z pair by up to 2 |a_loop[s]| max|P|, and a degree-N
// pair truncates at t^(2N+2)/(2N+2)! (cos - 1; the sine's t^(2N+3)/(2N+3)! is smaller) for an angle t:
//   N = 1: t <= 6.8e-5;  2: 0.00293;  3: 0.0208;  4: 0.0708;  5: 0.165;  6: 0.310;  7: 0.505;  8: 0.750.
// The largest drift (the merged one) gets degrees (3,3), (3,4), (4,4), (4,5), (5,6), (6,7), (7,8) at levels
// 1..7; the short inner drifts of the triple jump (ratio 0.13) and of the 7-stage scheme (0.088) one or two less.
// A drift whose own largest angle needs more than degree kMaxRotDegree leaves that pair type stale, and the kick that
// follows evaluates the table-driven sincos instead (degree 0 below); the decision is per drift and per pair type, so
// from level 5 on the kernels are mixed: the short inner drifts rotate, the long ones (first the zeta pair, which
// turns sqrt(2) faster) go through tsincos.  A pair type with a stale drift is recomputed in every step and needs no
// re-synchronisation.
constexpr double kLevelMaxD[10] = {0.0, 0.0104, 0.0147, 0.0354, 0.0500, 0.1166, 0.2192, 0.3570, 0.5400, 2.0};
constexpr double kDegreeMaxAngle[9] = {0.0, 6.8e-5, 0.00293, 0.0208, 0.0708, 0.165, 0.310, 0.505, 0.750};

// upper bounds of |a_loop[cs]| / max_s |a_loop[s]| for the coefficient sets cs of drift() (cs = S-1: merged drift)
template <int S> struct DriftRatio;
template <> struct DriftRatio<3> { static constexpr double r[3] = {0.1300, 0.1300, 1.0}; };
template <> struct DriftRatio<7> { static constexpr double r[7] = {0.6502, 0.6005, 0.08765, 0.08765, 0.6005, 0.6502, 1.0}; };

// A degree-N rotation costs 2N + 6 fp64 instructions per pair, the table-driven sincos 14 + 3 light ones: beyond
// degree kMaxRotDegree the drift leaves the pairs stale and the kick that follows evaluates tsincos instead.
#ifndef AW_MAX_ROT_DEGREE
#define AW_MAX_ROT_DEGREE 5
#endif
constexpr int kMaxRotDegree = AW_MAX_ROT_DEGREE;

template <int S, int LEVEL, int cs, bool ZETA>
__host__ __device__ constexpr int rotation_degree() {
  if (LEVEL == 0) return 0;  // no rotation: table-driven sincos at every stage
  const double t = (ZETA ? 2.0 : 1.4142135623730951) * kLevelMaxD[LEVEL] * DriftRatio<S>::r[cs];
  int n = 1;
  while (n < kMaxRotDegree && kDegreeMaxAngle[n] < t) ++n;
  return kDegreeMaxAngle[n] < t ? 0 : n;  // 0: the angle is too large for a rotation of degree <= kMaxRotDegree
}

// Does the drift after kick s rotate the u and v pairs (ZETA = false) / the zeta pair (ZETA = true)?  Decided per
// pair type: the zeta = 2z pair turns by sqrt(2) more than the other two, so it goes stale one level earlier.
template <int S, int LEVEL, int s, bool ZETA>
__host__ __device__ constexpr bool drift_rotates() {
  constexpr int cs = (s == S - 1) ? s : (s < S - 2 - s ? s : S - 2 - s);
  return rotation_degree<S, LEVEL, cs, ZETA>() > 0;
}
// Do all drifts of a step rotate this pair type?  Then it lives on rotations alone and is re-synchronised from the
// angles every chunk; otherwise every step contains a kick that recomputes it from the angle (tsincos).
template <int S, int LEVEL, bool ZETA, int s = 0>
__host__ __device__ constexpr bool all_drifts_rotate() {
  if constexpr (s == S) return true;
  else return drift_rotates<S, LEVEL, s, ZETA>() && all_drifts_rotate<S, LEVEL, ZETA, s + 1>();
}

// Everything a thread carries between stages.  Inside a block of `stride` steps the state is held in the
// rotated and scaled variables
//     u = x + y,  v = x - y,  zeta = 2 z,   pu = 2 (px + py),  pv = 2 (px - py),  pzt = 2 pz  (4 pz for S = 7, below)
// (tangent vector: du, dv, dzt = 2 dz, dpu = 2 (dpx + dpy), dpv = 2 (dpx - dpy), dpz = 2 dpz), in which
//     H_p = (cos u + cos v)(1 + cos zeta)/2:
// the kick needs no products of the x and y functions, the tangent kick is seven multiply-adds instead of nine
// (kick()), and with every momentum-like variable doubled the kick's coefficients are exactly the quantities the
// carried pairs provide (no constant multiplies on the native stages, see kick()).  u and v then advance with a/2
// per unit of pu, pv and zeta with a per unit of pzt, so the rotations take two coefficient sets (A = a/2 and A = a).
// The 7-stage scheme has four distinct drift constants, and two sets for each do not fit the uniform registers
// (ptxas then reloads constants inside the loop: +45..57 issue cycles per step); there pzt = 4 pz, so that zeta too
// advances with a/2 per unit of pzt and one set serves the three pairs, at the price of a factor 2 in the pzt kick.
// The change of variables is linear, so the map is the same map; halving and doubling are exact; the state is
// converted back to (x, y, z) for every checkpoint and for the store.
template <bool TAN>
struct Traj {
  double u, v, zt, pu, pv, pzt;
  double du, dv, dzt, dpu, dpv, dpz;
  // sin u, cos u, sin v, cos v; (s2, c2) = kz (sin zeta, cos zeta) with kz = 2 b_0 when the zeta pair lives on
  // rotations (every drift rotates it), kz = 1 when a kick of every step recomputes it from the angle
  double su, cu, sv, cv, s2, c2;
};

// (x, y) -> (x + y, x - y) and back, in place, for every pair of the first two degrees of freedom
__device__ __forceinline__ void to_sum_diff(double &a, double &b) {
  const double s = a + b, d = a - b;
  a = s;
  b = d;
}
__device__ __forceinline__ void from_sum_diff(double &a, double &b, double half) {
  const double x = half * (a + b), y = half * (a - b);
  a = x;
  b = y;
}
// pzt = kPzScale<S> pz
template <int S> constexpr double kPzScale = (S == 3) ? 2.0 : 4.0;

template <int S, bool TAN>
__device__ __forceinline__ void rotate_in(Traj<TAN> &t) {
  to_sum_diff(t.u, t.v);
  to_sum_diff(t.pu, t.pv);
  t.pu *= 2.0; t.pv *= 2.0;
  t.zt *= 2.0;
  t.pzt *= kPzScale<S>;
  if (TAN) {
    to_sum_diff(t.du, t.dv); to_sum_diff(t.dpu, t.dpv);
    t.dpu *= 2.0; t.dpv *= 2.0; t.dzt *= 2.0; t.dpz *= 2.0;
  }
}
// The momenta come back as px = px0 + ((pu - pu0) + (pv - pv0))/4 with (px0, py0) the values the block started
// from and pu0 = 2 (px0 + py0), pv0 = 2 (px0 - py0) as rotate_in rounded them: the differences are exact (or nearly),
// so the rounding of the forward conversion cancels and P stays bit-constant when the kicks vanish (eps = 0).
template <int S, bool TAN>
__device__ __forceinline__ void rotate_out(Traj<TAN> &t, double px0, double py0) {
  from_sum_diff(t.u, t.v, 0.5);
  const double du = t.pu - 2.0 * (px0 + py0), dv = t.pv - 2.0 * (px0 - py0);
  t.pu = fma(0.25, du + dv, px0);
  t.pv = fma(0.25, du - dv, py0);
  t.zt *= 0.5;
  t.pzt *= 1.0 / kPzScale<S>;
  if (TAN) { from_sum_diff(t.du, t.dv, 0.5); from_sum_diff(t.dpu, t.dpv, 0.25); t.dzt *= 0.5; t.dpz *= 0.5; }
}

// angles (and tangent angles) only: X += a P with ah = a/2 for the u, v variables (momenta doubled), a for dzt (and
// for zeta when pzt = 2 pz; a/2 when pzt = 4 pz)
template <int S, bool TAN>
__device__ __forceinline__ void drift_angles(Traj<TAN> &t, double ah, double a) {
  t.u = fma(ah, t.pu, t.u); t.v = fma(ah, t.pv, t.v); t.zt = fma(S == 3 ? a : ah, t.pzt, t.zt);
  if (TAN) { t.du = fma(ah, t.dpu, t.du); t.dv = fma(ah, t.dpv, t.dv); t.dzt = fma(a, t.dpz, t.dzt); }
}

// drift after kick s of the step loop: angles and, for LEVEL >= 1, the running pairs.  The stage lists are
// palindromic, so a_loop[s] == a_loop[S-2-s] for s < S-1: both use the coefficient set of the smaller index
// (fewer distinct constants for the compiler to keep at hand).
template <int S, bool TAN, int LEVEL, int s>
__device__ __forceinline__ void drift(Traj<TAN> &t, const IntegrateParams &p) {
  constexpr int cs = (s == S - 1) ? s : (s < S - 2 - s ? s : S - 2 - s);
  // the angle FMAs first: they depend only on the kick just done, and in the -O1 unit (source order) they fill
  // the latency of the kick's tail before the polynomial chains start (measured +0.8 to +1.6 %)
  drift_angles<S, TAN>(t, p.ah_loop[cs], p.a_loop[cs]);
  constexpr int nuv = rotation_degree<S, LEVEL, cs, false>(), nz = rotation_degree<S, LEVEL, cs, true>();
  double g, m;
  if constexpr (nuv > 0) {
    small_sincos<nuv>(t.pu, p.ah_loop[cs], p.grot_uv[cs], p.mrot_uv[cs], g, m);
    rotate(t.su, t.cu, g, m);
    small_sincos<nuv>(t.pv, p.ah_loop[cs], p.grot_uv[cs], p.mrot_uv[cs], g, m);
    rotate(t.sv, t.cv, g, m);
  }
  if constexpr (nz > 0) {
    if constexpr (S == 3) small_sincos<nz>(t.pzt, p.a_loop[cs], p.grot_z[cs], p.mrot_z[cs], g, m);    // A = a,   pzt = 2 pz
    else small_sincos<nz>(t.pzt, p.ah_loop[cs], p.grot_uv[cs], p.mrot_uv[cs], g, m);                // A = a/2, pzt = 4 pz
    rotate(t.s2, t.c2, g, m);
  }
}

// Is the zeta pair carried scaled by 2 b_0 (it lives on rotations, which are linear) or plain?
template <int S, int LEVEL>
__host__ __device__ constexpr bool zeta_pair_scaled() { return all_drifts_rotate<S, LEVEL, true>(); }

template <int S, bool TAN, int LEVEL>
__device__ __forceinline__ void resync(Traj<TAN> &t, const IntegrateParams &p) {
  // The merged drift is the longest of the step: if it rotates a pair type, every drift does, and that type lives on
  // rotations alone (re-synchronised here); if not, the first kick of every step recomputes it from the angle.
  static_assert(all_drifts_rotate<S, LEVEL, false>() == drift_rotates<S, LEVEL, S - 1, false>() &&
                all_drifts_rotate<S, LEVEL, true>() == drift_rotates<S, LEVEL, S - 1, true>(), "drift ratios");
  if constexpr (all_drifts_rotate<S, LEVEL, false>()) {
    sincos(t.u, t.su, t.cu);
    sincos(t.v, t.sv, t.cv);
  }
  if constexpr (zeta_pair_scaled<S, LEVEL>()) {
    sincos(t.zt, t.s2, t.c2);
    t.s2 *= p.b2[0];
    t.c2 *= p.b2[0];
  }
}

// kick of stage s in the rotated variables: P -= b grad H_p(X), dP -= b Hess H_p(X) dX (R3).  In natural variables,
// with W = cos u + cos v (the sum and difference of the x and y rows of SURVEY.md Appendix A.2, dzeta = 2 dz):
//   d(px+py) = b (1 + cos zeta) sin u,   d(px-py) = b (1 + cos zeta) sin v,   d(pz) = b W sin zeta
//   d(dpx+dpy) = b ((1 + cos zeta) cos u du - sin zeta sin u dzeta),   likewise v
//   d(dpz) = b (-sin zeta (sin u du + sin v dv) + W cos zeta dzeta)
// With every momentum-like variable doubled and (Sz, Cz) = 2b (sin zeta, cos zeta), F = Cz + 2b:
//   pu += F su,  pv += F sv,  pzt += W Sz
//   dpu += (F cu) du - (Sz su) dzt,  dpv += (F cv) dv - (Sz sv) dzt,  dpz += -(Sz su) du - (Sz sv) dv + (Cz W) dzt
// i.e. 2 adds + 5 products + 10 multiply-adds with no constant multiplies at all when the carried pair already is
// (Sz, Cz) — ZMODE 0: the pair lives on rotations scaled by 2 b_0 and this stage's weight is b_0 (the first and
// last stage of the palindromic schemes).  ZMODE 1: scaled pair, other weight: Sz = rho s2, Cz = rho c2 with
// rho = b_s / b_0, folded as F = fma(rho, c2, 2b), W' = rho W.  ZMODE 2: plain pair (recomputed by tsincos in every
// step): the same with kz = 2 b_s in place of rho.
// PZ4 (the 7-stage scheme): pzt = 4 pz takes 2 W Sz, i.e. its own product with the constant 2 kz (2 when ZMODE 0).
// FRESH_UV / FRESH_Z: the running pairs are valid (the drift before this kick rotated them); otherwise they are
// evaluated here from the angles.
template <bool TAN, bool FRESH_UV, bool FRESH_Z, int ZMODE, bool PZ4>
__device__ __forceinline__ void kick(Traj<TAN> &t, double b2, double kz, double kz2, const TrigTable &tab) {
  if (!FRESH_UV) {
    tsincos(tab, t.u, t.su, t.cu);
    tsincos(tab, t.v, t.sv, t.cv);
  }
  if (!FRESH_Z) tsincos(tab, t.zt, t.s2, t.c2);
  const double W = t.cu + t.cv;                                   // 2 cos x cos y
  const double F = ZMODE == 0 ? t.c2 + b2 : fma(kz, t.c2, b2);    // 2 b (1 + cos zeta)
  const double Wk = (ZMODE == 0 || (PZ4 && !TAN)) ? W : kz * W;   // feeds e5 (and pzt unless PZ4)
  const double Wz = !PZ4 ? Wk : (ZMODE == 0 ? 2.0 * W : kz2 * W);
  t.pu = fma(t.su, F, t.pu);
  t.pv = fma(t.sv, F, t.pv);
  t.pzt = fma(Wz, t.s2, t.pzt);
  if (TAN) {
    const double Sz = ZMODE == 0 ? t.s2 : kz * t.s2;              // 2 b sin zeta
    const double a1 = F * t.cu, a2 = F * t.cv, k1 = Sz * t.su, k2 = Sz * t.sv;
    const double e5 = t.c2 * Wk;                                  // 2 b cos zeta W
    // Seven all-register multiply-adds, grouped by the operand they share in the same slot (du, dv, dzt): in the -O1
    // unit ptxas keeps this order, and the operand-reuse cache then serves the repeated operand (a DFMA with three
    // fresh register operands issues in 3 cycles instead of 2).  Measured on configs[3] against five other orders:
    // +1.0 % over the round-1 order (a1, a2, e5 first), the others within -0.8 .. +0.8 %.
    t.dpu = fma(a1, t.du, t.dpu); t.dpz = fma(-k1, t.du, t.dpz);
    t.dpv = fma(a2, t.dv, t.dpv); t.dpz = fma(-k2, t.dv, t.dpz);
    t.dpu = fma(-k1, t.dzt, t.dpu); t.dpv = fma(-k2, t.dzt, t.dpv); t.dpz = fma(e5, t.dzt, t.dpz);
  }
}

// stages s, s+1, ..., S-1 of one step: kick_s then the drift after it
template <int S, bool TAN, int LEVEL, int s>
__device__ __forceinline__ void stages(Traj<TAN> &t, const IntegrateParams &p, const TrigTable &tab) {
  if constexpr (s < S) {
    // the drift before kick s is the one after kick s-1, or for s = 0 the merged drift that closed the last step
    constexpr int prev = (s == 0 ? S - 1 : s - 1);
    constexpr int zmode = !zeta_pair_scaled<S, LEVEL>() ? 2 : ((s == 0 || s == S - 1) ? 0 : 1);
    kick<TAN, drift_rotates<S, LEVEL, prev, false>(), drift_rotates<S, LEVEL, prev, true>(), zmode, S != 3>(
        t, p.b2[s], zmode == 2 ? p.b2[s] : p.rho[s], zmode == 2 ? p.b4[s] : p.rho2[s], tab);
    drift<S, TAN, LEVEL, s>(t, p);
    stages<S, TAN, LEVEL, s + 1>(t, p, tab);
  }
}

// SCHEDULE = AW_LEVEL_GROUP: 1 = the throughput flavour (-Xptxas -O1 unit), 0 = the latency flavour (default flags).  It
// changes nothing in the code; it only gives the two compilations of the same kernel different names.
template <int S, bool TAN, int LEVEL, int SCHEDULE>
__global__ void __launch_bounds__(AW_BLOCK, AW_MIN_BLOCKS(LEVEL))
    integrate_kernel(const __grid_constant__ IntegrateParams p) {
  // the (sin, cos) table of tsincos, 4 interleaved copies, 32 KB of shared memory (kernels with a stale drift only)
  constexpr bool kUsesTable = !(all_drifts_rotate<S, LEVEL, false>() && all_drifts_rotate<S, LEVEL, true>());
  __shared__ double2 tab_s[kUsesTable ? kTab * kTabCopies : 1];
  if constexpr (kUsesTable) {
    for (int i = threadIdx.x; i < kTab * kTabCopies; i += blockDim.x)
      tab_s[i] = make_double2(aw_trig_table[2 * (i / kTabCopies)], aw_trig_table[2 * (i / kTabCopies) + 1]);
    __syncthreads();
  }
  const TrigTable tab = {reinterpret_cast<const char *>(tab_s), (threadIdx.x & (kTabCopies - 1)) * 16u};
  // blocks of 32, 64 or 128 threads (launch_one): the arithmetic is per trajectory, so the result does not depend on it
  const int64_t k = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (k >= p.n) return;
  if (p.status[k] != AW_ST_LIVE) return;
  const int64_t P = p.pitch;

  // between blocks the fields of t hold x, y, z, px, py, pz (and the plain tangent vector)
  Traj<TAN> t;
  t.u = p.q[k]; t.v = p.q[P + k]; t.zt = p.q[2 * P + k];
  t.pu = p.q[3 * P + k]; t.pv = p.q[4 * P + k]; t.pzt = p.q[5 * P + k];
  if (TAN) {
    t.du = p.w[k]; t.dv = p.w[P + k]; t.dzt = p.w[2 * P + k];
    t.dpu = p.w[3 * P + k]; t.dpv = p.w[4 * P + k]; t.dpz = p.w[5 * P + k];
  }
  int status = AW_ST_LIVE;

  for (int chk = 0; chk < p.nchk; ++chk) {
    const double px0 = t.pu, py0 = t.pv;
    rotate_in<S, TAN>(t);                           // (x, y, z) -> (u, v, zeta)
    drift_angles<S, TAN>(t, 0.5 * p.a_open, p.a_open);  // opening drift of the block
    resync<S, TAN, LEVEL>(t, p);     // pairs from the angles: the same values a new launch would start from

#pragma unroll 1
    for (int rem = p.stride; rem > 0;) {
      const int m = rem < p.chunk ? rem : p.chunk;
      rem -= m;
#pragma unroll 1
      for (int i = m; i > 0; --i) stages<S, TAN, LEVEL, 0>(t, p, tab);
      if (rem > 0) resync<S, TAN, LEVEL>(t, p);
    }
    drift_angles<S, TAN>(t, -0.5 * p.a_open, -p.a_open);  // last merged drift -> closing drift of the block
    rotate_out<S, TAN>(t, px0, py0);                   // (u, v, zeta) -> (x, y, z)
    double &x = t.u, &y = t.v, &z = t.zt, &px = t.pu, &py = t.pv, &pz = t.pzt;
    double &dx = t.du, &dy = t.dv, &dz = t.dzt, &dpx = t.dpu, &dpy = t.dpv;

    // ---- fused checkpoint (R4): (i) renormalise + log growth, (ii) energy error, (iii) wrap
    bool finite = true;
    if (TAN) {
      double s2 = dx * dx;
      s2 = fma(dy, dy, s2); s2 = fma(dz, dz, s2);
      s2 = fma(dpx, dpx, s2); s2 = fma(dpy, dpy, s2); s2 = fma(t.dpz, t.dpz, s2);
      const double nu = sqrt(s2);
      const double inv = 1.0 / nu;
      dx *= inv; dy *= inv; dz *= inv; dpx *= inv; dpy *= inv; t.dpz *= inv;
      const double logsum = p.acc[k] + log(nu);
      p.acc[k] = logsum;
      if (logsum > p.acc[P + k]) p.acc[P + k] = logsum;
      finite = isfinite(dx) && isfinite(dy) && isfinite(dz) && isfinite(dpx) && isfinite(dpy) &&
               isfinite(t.dpz);
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
    // survivor filter (R25): outside the launch rectangle at a checkpoint -> dropped, frozen here
    if (p.survive && !(px >= p.surv[0] && px < p.surv[1] && py >= p.surv[2] && py < p.surv[3])) {
      status = AW_ST_LEFT;
      break;
    }
  }

  p.q[k] = t.u; p.q[P + k] = t.v; p.q[2 * P + k] = t.zt;
  p.q[3 * P + k] = t.pu; p.q[4 * P + k] = t.pv; p.q[5 * P + k] = t.pzt;
  if (TAN) {
    p.w[k] = t.du; p.w[P + k] = t.dv; p.w[2 * P + k] = t.dzt;
    p.w[3 * P + k] = t.dpu; p.w[4 * P + k] = t.dpv; p.w[5 * P + k] = t.dpz;
  }
  if (status != AW_ST_LIVE) p.status[k] = (uint8_t)status;
}

template <int S, bool TAN, int LEVEL>
cudaError_t launch_one(const IntegrateParams &p, cudaStream_t st) {
  const int block = p.block;
  const int64_t blocks = (p.n + block - 1) / block;
  integrate_kernel<S, TAN, LEVEL, AW_LEVEL_GROUP><<<(unsigned)blocks, block, 0, st>>>(p);
  count_launch();
  return cudaGetLastError();
}

template <int S, bool TAN>
cudaError_t launch_level(const IntegrateParams &p, cudaStream_t st) {
  switch (p.level) {
#if AW_LEVEL_GROUP == 1
    case 1: return launch_one<S, TAN, 1>(p, st);
    case 2: return launch_one<S, TAN, 2>(p, st);
    case 3: return launch_one<S, TAN, 3>(p, st);
    case 4: return launch_one<S, TAN, 4>(p, st);
    case 5: return launch_one<S, TAN, 5>(p, st);
    case 6: return launch_one<S, TAN, 6>(p, st);
    case 7: return launch_one<S, TAN, 7>(p, st);
    case 8: return launch_one<S, TAN, 8>(p, st);
    case 9: return launch_one<S, TAN, 9>(p, st);
    case 0: return launch_one<S, TAN, 0>(p, st);
    default: return cudaErrorInvalidValue;
#else  // the latency flavour: every level
    case 1: return launch_one<S, TAN, 1>(p, st);
    case 2: return launch_one<S, TAN, 2>(p, st);
    case 3: return launch_one<S, TAN, 3>(p, st);
    case 4: return launch_one<S, TAN, 4>(p, st);
    case 5: return launch_one<S, TAN, 5>(p, st);
    case 6: return launch_one<S, TAN, 6>(p, st);
    case 7: return launch_one<S, TAN, 7>(p, st);
    case 8: return launch_one<S, TAN, 8>(p, st);
    case 9: return launch_one<S, TAN, 9>(p, st);
    default: return launch_one<S, TAN, 0>(p, st);
#endif
  }
}

}  // namespace

#if AW_LEVEL_GROUP == 1

cudaError_t launch_integrate_low(const IntegrateParams &p, int order, bool tangent, cudaStream_t st) {
  if (order == 4) return tangent ? launch_level<3, true>(p, st) : launch_level<3, false>(p, st);
  return tangent ? launch_level<7, true>(p, st) : launch_level<7, false>(p, st);
}

#else

// Largest |d| = max_s |a_s| max|P| each level may see, with both Taylor truncations below 2^-60 ~ 8.7e-19 (they
// are systematic, so 300 of them still sum to < 3e-16):
//   m of degree N truncates at |t|^(2N+2)/(2N+2)!, g at |t|^(2N+3)/(2N+3)! for a rotation angle t; the m bound
//   is the tighter one:  N = 3: |t| <= 0.0208;  4: 0.0708;  5: 0.165;  6: 0.310;  7: 0.505;  8: 0.750.
// The u and v pairs rotate by up to sqrt(2) |d|, the 2z pair by up to 2 |d|:
//   level 1 = (3,3): 2|d| <= 0.0208;       level 2 = (3,4): sqrt(2)|d| <= 0.0208;   level 3 = (4,4): 2|d| <= 0.0708;
//   level 4 = (4,5): sqrt(2)|d| <= 0.0708;  level 5 = (5,6): sqrt(2)|d| <= 0.165;    level 6 = (6,7): sqrt(2)|d| <= 0.310;
//   level 7 = (7,8): sqrt(2)|d| <= 0.505 (and 2|d| <= 0.750);  levels 8 (|d| <= 0.54) and 9 (|d| <= 2): mixed, see kLevelMaxD;
//   beyond: level 0 (full sincos every stage).  A degree-(8,9) rotation of the merged drift would cost more fp64
//   instructions than the sincos it replaces, which is why the pure rotation levels stop at 7.
int trig_level_for(double d) {
  if (!(d == d)) return 0;
  for (int level = 1; level <= 9; ++level)
    if (d <= kLevelMaxD[level]) return level;
  return 0;
}

double trig_level_max_angle(int level) {
  return (level >= 1 && level <= 9) ? kLevelMaxD[level] : INFINITY;
}

// Does integrate_kernel<S, *, level> carry the 32 KB sincos table in shared memory?
template <int S, int LEVEL = 0>
bool uses_table_at(int level) {
  if constexpr (LEVEL > 9) return true;
  else return level == LEVEL ? !(all_drifts_rotate<S, LEVEL, false>() && all_drifts_rotate<S, LEVEL, true>())
                             : uses_table_at<S, LEVEL + 1>(level);
}
bool kernel_uses_table(int order, int level) { return order == 4 ? uses_table_at<3>(level) : uses_table_at<7>(level); }

// Threads per block from the ensemble size: 128 (the tuned shape) once that fills every SM with its
// 4 resident blocks; smaller ensembles get 64- or 32-thread blocks so that their warps spread over all SMs (and
// over the four sub-partitions of each) instead of piling 4 warps on a quarter of the chip — as long as all blocks
// stay resident at once: 16 per SM by registers, 6 per SM for the kernels that hold the 32 KB table in shared memory
// (measured on the Fig. 4 ensemble, 32 000 trajectories: 1000 blocks of 32 threads do not fit 148 x 6 and run in two
// waves, 1.6e10 traj-steps/s; 500 blocks of 64 threads 3.0e10).
int integrate_block_size(int64_t n, int forced, bool uses_table) {
  if (forced == 32 || forced == 64 || forced == 128) return forced;
  static int sms[64] = {0};
  int dev = 0;
  if (cudaGetDevice(&dev) != cudaSuccess || dev < 0 || dev >= 64) dev = 0;
  if (sms[dev] == 0) {
    int v = 0;
    if (cudaDeviceGetAttribute(&v, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess || v <= 0) v = 148;
    sms[dev] = v;
  }
  const int64_t full = (int64_t)sms[dev] * 4;   // blocks of one full wave at 4 resident 128-thread blocks per SM
  const int64_t resident = (int64_t)sms[dev] * (uses_table ? 6 : 16);
  if ((n + 127) / 128 >= full) return 128;
  if ((n + 31) / 32 <= resident) return 32;
  if ((n + 63) / 64 <= resident) return 64;
  return 128;
}

// Throughput or latency flavour (see AW_LEVEL_GROUP above).  Measured on B200 (latency / throughput flavour, four kernels:
// order 4 and 6, with and without tangent, levels 1, 3, 7): x 1.4-1.9 below one warp per sub-partition (n <= 16 000),
// x 1.0-1.2 at 1.7-5 warps, x 1.00-1.05 at 8 warps (n = 150 000), x 0.97-0.99 at 32 warps (n = 600 000): latency up
// to 8 warps per sub-partition on average (n <= 8 x 4 x SMs x 32 = 151 552 trajectories on a B200).
bool integrate_latency_flavour(int64_t n, int forced) {
  if (forced == 1) return false;
  if (forced == 2) return true;
  int dev = 0, v = 0;
  if (cudaGetDevice(&dev) != cudaSuccess || cudaDeviceGetAttribute(&v, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess ||
      v <= 0)
    v = 148;
  return (n + 31) / 32 <= (int64_t)v * 32;
}

// The per-drift degrees assume the ratios |a_loop[cs]| / max |a_loop| of the two built-in stage lists.
bool drift_ratios_hold(int S, const double *a_loop) {
  double amax = 0.0;
  for (int s = 0; s < S; ++s) amax = fmax(amax, fabs(a_loop[s]));
  for (int s = 0; s < S; ++s) {
    const double r = (S == 3) ? DriftRatio<3>::r[s] : DriftRatio<7>::r[s];
    if (fabs(a_loop[s]) > r * amax) return false;
  }
  return true;
}

cudaError_t launch_integrate_low(const IntegrateParams &p, int order, bool tangent, cudaStream_t st);

cudaError_t launch_integrate(const IntegrateParams &p, int order, bool tangent, bool latency, cudaStream_t st) {
  if (!latency) return launch_integrate_low(p, order, tangent, st);
  if (order == 4) return tangent ? launch_level<3, true>(p, st) : launch_level<3, false>(p, st);
  return tangent ? launch_level<7, true>(p, st) : launch_level<7, false>(p, st);
}

#endif  // AW_LEVEL_GROUP

}  // namespace aw
