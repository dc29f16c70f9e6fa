// aw_oracle.cpp — TEST INFRASTRUCTURE ONLY.
//
// Plain, slow, single-threaded, obviously-correct fp64 restatement of the hot path of
// arXiv 1107.4107 ("Mapping the Arnold web with a GPU-supercomputer"), written from the paper text
// (/root/reference/PAPER.md, cited below as P:<line>) and the readings listed in DESIGN.md §3
// (cited as R<n>).  It is the parity oracle for the CUDA library in paper_1107_4107_b200/csrc and
// shares NO code, header, table or constant generator with it.  Only tests/, __graft_entry__.smoke()
// and bench.py's cpu_baseline / --impl reference legs may load this file's shared object.
//
// Build: g++ -std=c++17 -O2 -ffp-contract=off -fPIC -shared   (no FMA contraction: every product and
// sum below is rounded separately, exactly as written; std::fma appears ONLY in the angle wrap, R7).
//
// Every function follows the paper's algorithm step by step, in the paper's order and notation:
//   P:33 eq.(1)  H(P,X) = P^2/2 + eps*H_p(X)
//   P:43 eq.(2)  H_p(x,y,z) = cos(x) cos(y) [1 + cos(2z)]
//   P:55         fixed-step symplectic composition integrator (Yoshida 1990, ref. 25)
//   P:85,87,97   initial conditions on the energy shell; third momentum from the energy condition
//   P:67,97      histogram of the ensemble over the momentum (action) space, accumulated over time
// The tangent map / FLI is not in the paper (P:111 only names the concept); it follows BASELINE.json's
// north_star: the exact derivative of the discrete map applied to one tangent vector (R3, R13).
//
// Pins (tests/test_oracle_pins.py, run with -m "not gpu"): eps=0 closed form, energy-error order
// 4 / 6, order conditions of the weights, reversibility, symplectic 6x6 tangent map, tangent
// vs finite differences, pendulum reduction vs the complete elliptic integral, invariant subspaces
// (P:79), shell layer, IC energy, histogram brute force; averaged velocity vs eps=0 closed
// form, vs an unwrapped brute-force run and vs the pendulum rotation frequency 2 pi / T(h); central
// projection on a hand case; survivor filter vs a stepwise brute force; the indicator kinds and masks on a
// hand-made table (strict FLI > thr, 255 / NaN for every status != 1); slices by global index against the whole
// and the cell-centre definition; the Gaussian cloud's Rayleigh law; cloud resampling against plain ensembles of the
// attempt seeds.  tests/test_oracle_sanitizers.py runs this file under -fsanitize=address,undefined.  No function
// here is "parity unpinned" except where DESIGN.md §3 says so (the paper's figures and its dE<1e-8 remark).

#include <cmath>
#include <cstdint>
#include <cstring>
#include <limits>

namespace {

// ---------------------------------------------------------------- model: eq.(1), eq.(2)

inline double Hp(double x, double y, double z) {
  return std::cos(x) * std::cos(y) * (1.0 + std::cos(2.0 * z));
}

// gradient of H_p, term by term from eq.(2)
inline void gradHp(double x, double y, double z, double g[3]) {
  const double f = 1.0 + std::cos(2.0 * z);
  g[0] = -std::sin(x) * std::cos(y) * f;
  g[1] = -std::cos(x) * std::sin(y) * f;
  g[2] = -2.0 * std::cos(x) * std::cos(y) * std::sin(2.0 * z);
}

// Hessian of H_p (symmetric), row-major 3x3, second derivatives of eq.(2)
inline void hessHp(double x, double y, double z, double h[9]) {
  const double sx = std::sin(x), cx = std::cos(x);
  const double sy = std::sin(y), cy = std::cos(y);
  const double s2 = std::sin(2.0 * z), c2 = std::cos(2.0 * z);
  const double f = 1.0 + c2;
  h[0] = -cx * cy * f;         // xx
  h[4] = -cx * cy * f;         // yy
  h[8] = -4.0 * cx * cy * c2;  // zz
  h[1] = h[3] = sx * sy * f;          // xy
  h[2] = h[6] = 2.0 * sx * cy * s2;   // xz
  h[5] = h[7] = 2.0 * cx * sy * s2;   // yz
}

// eq.(1): H = P^2/2 + eps * H_p(X)
inline double Hamiltonian(const double q[6], double eps) {
  const double kin = 0.5 * (q[3] * q[3] + q[4] * q[4] + q[5] * q[5]);
  return kin + eps * Hp(q[0], q[1], q[2]);
}

// ---------------------------------------------------------------- scheme: P:55, ref. 25 (R1, R2)
//
// Symmetric composition of the 2nd-order drift-kick-drift map S2(tau):
//   X += (tau/2) P ; P -= eps tau grad H_p(X) ; X += (tau/2) P
// as S(dt) = S2(w_S dt) o ... o S2(w_1 dt), adjacent half drifts merged inside one step:
//   for s = 1..S { X += a_s P ; P -= b_s grad H_p(X) }   X += a_{S+1} P
// with c_1 = w_1/2, c_s = (w_{s-1} + w_s)/2, c_{S+1} = w_S/2, a_s = c_s dt, b_s = (eps w_s) dt.
//
// order 4, S = 3 (triple jump): w_1 = w_3 = 1/(2 - 2^(1/3)), w_2 = -2^(1/3)/(2 - 2^(1/3)).
// order 6, S = 7 (Yoshida 1990 "solution A", palindromic w3 w2 w1 w0 w1 w2 w3).  The paper prints no
// coefficients; the values below are the root of the four order conditions
//   sum g = 1, sum g^3 = 0, sum g^5 = 0, sum_i g_i^3 (sum_{j<i} g_j + g_i/2)^2 = 0
// nearest to the published 6-digit values, polished to 20 digits by oracle/derive_yoshida6.py
// (mpmath Newton); tests re-evaluate the four conditions on these doubles.
const double Y6_W0 = 1.31518632068391121888;
const double Y6_W1 = -1.17767998417887100695;
const double Y6_W2 = 0.23557321335935813368;
const double Y6_W3 = 0.78451361047755726382;

int stage_list(int order, double w[9]) {
  if (order == 4) {
    const double cbrt2 = std::cbrt(2.0);
    w[0] = 1.0 / (2.0 - cbrt2);
    w[1] = -cbrt2 / (2.0 - cbrt2);
    w[2] = w[0];
    return 3;
  }
  if (order == 6) {
    w[0] = Y6_W3; w[1] = Y6_W2; w[2] = Y6_W1; w[3] = Y6_W0; w[4] = Y6_W1; w[5] = Y6_W2; w[6] = Y6_W3;
    return 7;
  }
  if (order == 2) { w[0] = 1.0; return 1; }   // plain S2, used by tests only
  if (order == 66) {
    // closed-form 6th-order cross-check (oracle only): triple jump of the order-4 triple jump,
    // z_1 = 1/(2 - 2^(1/5)), z_0 = -2^(1/5)/(2 - 2^(1/5)); 9 stages
    const double cbrt2 = std::cbrt(2.0);
    const double v1 = 1.0 / (2.0 - cbrt2), v0 = -cbrt2 / (2.0 - cbrt2);
    const double r5 = std::pow(2.0, 0.2);
    const double z1 = 1.0 / (2.0 - r5), z0 = -r5 / (2.0 - r5);
    const double v[3] = {v1, v0, v1};
    const double zz[3] = {z1, z0, z1};
    for (int i = 0; i < 3; ++i)
      for (int j = 0; j < 3; ++j) w[3 * i + j] = zz[i] * v[j];
    return 9;
  }
  return 0;
}

// a[0..S] drift constants, b[0..S-1] kick constants, evaluated in exactly this order in fp64
int stage_constants(int order, double dt, double eps, double a[10], double b[9]) {
  double w[9];
  const int S = stage_list(order, w);
  if (S == 0) return 0;
  for (int s = 0; s <= S; ++s) {
    double c;
    if (s == 0) c = w[0] / 2.0;
    else if (s == S) c = w[S - 1] / 2.0;
    else c = (w[s - 1] + w[s]) / 2.0;
    a[s] = c * dt;
  }
  for (int s = 0; s < S; ++s) b[s] = (eps * w[s]) * dt;
  return S;
}

// One full step of the composition on the state q = (x,y,z,px,py,pz) and, if tw != nullptr, on the
// tangent vector tw = (dx,dy,dz,dpx,dpy,dpz) through the exact derivative of the same map (R3):
//   dX += a_s dP ; dP -= b_s Hess H_p(X) dX   with X taken AFTER the stage's drift.
inline void one_step(double q[6], double *tw, int S, const double a[10], const double b[9]) {
  double g[3], h[9];
  for (int s = 0; s < S; ++s) {
    q[0] += a[s] * q[3];
    q[1] += a[s] * q[4];
    q[2] += a[s] * q[5];
    if (tw) {
      tw[0] += a[s] * tw[3];
      tw[1] += a[s] * tw[4];
      tw[2] += a[s] * tw[5];
    }
    gradHp(q[0], q[1], q[2], g);
    q[3] -= b[s] * g[0];
    q[4] -= b[s] * g[1];
    q[5] -= b[s] * g[2];
    if (tw) {
      hessHp(q[0], q[1], q[2], h);
      const double r0 = h[0] * tw[0] + h[1] * tw[1] + h[2] * tw[2];
      const double r1 = h[3] * tw[0] + h[4] * tw[1] + h[5] * tw[2];
      const double r2 = h[6] * tw[0] + h[7] * tw[1] + h[8] * tw[2];
      tw[3] -= b[s] * r0;
      tw[4] -= b[s] * r1;
      tw[5] -= b[s] * r2;
    }
  }
  q[0] += a[S] * q[3];
  q[1] += a[S] * q[4];
  q[2] += a[S] * q[5];
  if (tw) {
    tw[0] += a[S] * tw[3];
    tw[1] += a[S] * tw[4];
    tw[2] += a[S] * tw[5];
  }
}

// ---------------------------------------------------------------- checkpoint (R4, R7, R13, R16)

const double INV_2PI = 0.15915494309189535;      // double nearest 1/(2 pi)
const double TWO_PI_HI = 6.283185307179586;      // double nearest 2 pi  (0x1.921fb54442d18p+2)
const double TWO_PI_LO = 2.4492935982947064e-16; // 2 pi - TWO_PI_HI

// acc = {logsum, fli_max, H0, dH_max}; wind may be nullptr; returns the new status.
// surv (may be nullptr) = {lo_x, hi_x, lo_y, hi_y}: the survivor filter of P:99 ("tracked only those
// trajectories which remained within the area during the whole observation time"; R25): a trajectory
// whose (px, py) is outside the half-open rectangle at a checkpoint gets status 3 and is frozen there.
inline int checkpoint(double q[6], double *tw, double acc[4], int32_t *wind, double eps,
                      const double *surv = nullptr) {
  // (i) renormalise the tangent vector and accumulate the log of its growth
  if (tw) {
    double s2 = tw[0] * tw[0];
    s2 = s2 + tw[1] * tw[1];
    s2 = s2 + tw[2] * tw[2];
    s2 = s2 + tw[3] * tw[3];
    s2 = s2 + tw[4] * tw[4];
    s2 = s2 + tw[5] * tw[5];
    const double nu = std::sqrt(s2);
    acc[0] += std::log(nu);
    for (int i = 0; i < 6; ++i) tw[i] = tw[i] / nu;
    if (acc[0] > acc[1]) acc[1] = acc[0];
  }
  // (ii) energy error against the value the same routine returned at t = 0
  const double dH = std::fabs(Hamiltonian(q, eps) - acc[2]);
  if (dH > acc[3]) acc[3] = dH;
  // (iii) wrap the angles to [-pi, pi] and count whole turns
  for (int i = 0; i < 3; ++i) {
    const double k = std::nearbyint(q[i] * INV_2PI);
    q[i] = std::fma(-k, TWO_PI_LO, std::fma(-k, TWO_PI_HI, q[i]));
    if (wind) wind[i] += (int32_t)k;
  }
  bool finite = true;
  for (int i = 0; i < 6; ++i) finite = finite && std::isfinite(q[i]);
  if (tw)
    for (int i = 0; i < 6; ++i) finite = finite && std::isfinite(tw[i]);
  if (!finite) return 2;
  if (surv && !(q[3] >= surv[0] && q[3] < surv[1] && q[4] >= surv[2] && q[4] < surv[3])) return 3;
  return 1;
}

// ---------------------------------------------------------------- counter-based randomness (R11)
//
// mix64(seed, ctr): z = seed + ctr * 0x9E3779B97F4A7C15 (mod 2^64), followed by two
// xorshift-multiply rounds and a final xorshift.  u = (z >> 11) * 2^-53 in [0, 1).
inline uint64_t mix64(uint64_t seed, uint64_t ctr) {
  uint64_t z = seed + ctr * 0x9E3779B97F4A7C15ull;
  z ^= z >> 30; z *= 0xBF58476D1CE4E5B9ull;
  z ^= z >> 27; z *= 0x94D049BB133111EBull;
  z ^= z >> 31;
  return z;
}
inline double uniform01(uint64_t seed, uint64_t k, uint64_t slot) {
  return (double)(mix64(seed, 16ull * k + slot) >> 11) * (1.0 / 9007199254740992.0);
}
// slots a, b -> two independent standard normals (Box-Muller on (1 - u_a, u_b))
inline void normal_pair(uint64_t seed, uint64_t k, uint64_t slot, double &n1, double &n2) {
  const double ua = uniform01(seed, k, slot), ub = uniform01(seed, k, slot + 1);
  const double rad = std::sqrt(-2.0 * std::log(1.0 - ua));
  const double ang = TWO_PI_HI * ub;
  n1 = rad * std::cos(ang);
  n2 = rad * std::sin(ang);
}
// unit tangent vector from slots 5..10 of counter k
inline void unit_tangent(uint64_t seed, uint64_t k, double t[6]) {
  normal_pair(seed, k, 5, t[0], t[1]);
  normal_pair(seed, k, 7, t[2], t[3]);
  normal_pair(seed, k, 9, t[4], t[5]);
  double s2 = 0.0;
  for (int i = 0; i < 6; ++i) s2 = s2 + t[i] * t[i];
  const double nu = std::sqrt(s2);
  for (int i = 0; i < 6; ++i) t[i] = t[i] / nu;
}

}  // namespace

// ======================================================================================== C interface
extern "C" {

struct awo_grid {
  int32_t gx, gy;
  double lo_x, hi_x, lo_y, hi_y;
  int32_t angle_mode;    // 0: all angles 0; 1: U[0,2pi) from seed
  int32_t shape;         // 0: grid; 1: uniform disk (cx,cy,r); 2: Gaussian (cx,cy,sigma=r);
                         // 3: uniform on the whole sphere S (R28);
                         // 4: uniform random points of the rectangle [lo_x,hi_x) x [lo_y,hi_y) (R33)
  double cx, cy, r;
  int32_t pz_sign;       // +1 or -1
  int32_t tangent_mode;  // 0: one common seeded unit vector; 1: per trajectory
  int64_t k0;            // the state holds trajectories [k0, k0 + n) of the gx*gy ensemble the grid describes
                         // (independent realisations, so any contiguous slice can be generated alone)
  int32_t resample;      // random shapes 1, 2, 4: redraw a trajectory whose (px, py, X) has no real v_z, up to this many
                         // times (R31); 0: mask it (status 0, R8)
  int32_t reserved_;
};

double awo_hp(double x, double y, double z) { return Hp(x, y, z); }
void awo_grad(double x, double y, double z, double *g) { gradHp(x, y, z, g); }
void awo_hess(double x, double y, double z, double *h) { hessHp(x, y, z, h); }
double awo_hamiltonian(const double *q, double eps) { return Hamiltonian(q, eps); }
int awo_stage_list(int order, double *w) { return stage_list(order, w); }
int awo_stage_constants(int order, double dt, double eps, double *a, double *b) {
  return stage_constants(order, dt, eps, a, b);
}
uint64_t awo_mix64(uint64_t seed, uint64_t ctr) { return mix64(seed, ctr); }
double awo_uniform(uint64_t seed, uint64_t k, uint64_t slot) { return uniform01(seed, k, slot); }
void awo_common_tangent(uint64_t seed, double *t) { unit_tangent(seed, 0x7FFFFFFFFFFFFFFFull, t); }

// `nsteps` plain steps on ONE trajectory held as q[6] (+ tw[6] or NULL): no checkpoint, no wrap.
int awo_steps(double *q, double *tw, int order, double dt, double eps, int64_t nsteps) {
  double a[10], b[9];
  const int S = stage_constants(order, dt, eps, a, b);
  if (S == 0) return -1;
  for (int64_t i = 0; i < nsteps; ++i) one_step(q, tw, S, a, b);
  return 0;
}

// One checkpoint on ONE trajectory (exposed so tests can exercise the wrap and renormalisation alone).
int awo_checkpoint(double *q, double *tw, double *acc, int32_t *wind, double eps, const double *surv) {
  return checkpoint(q, tw, acc, wind, eps, surv);
}

// a1: initial conditions on the energy shell (R6, R8-R12, R17, R18).
// SoA planes: q[6*pitch], w[6*pitch] or NULL, acc[4*pitch], wind[3*pitch] or NULL, status[n].
int awo_init_shell(const awo_grid *g, double E, double eps, uint64_t seed, int64_t n, int64_t pitch,
                   double *q, double *w, double *acc, int32_t *wind, uint8_t *status) {
  if (!g || !q || !acc || !status || pitch < n) return -1;
  if (g->k0 < 0 || n < 0 || g->k0 + n > (int64_t)g->gx * g->gy) return -1;
  double tcommon[6];
  unit_tangent(seed, 0x7FFFFFFFFFFFFFFFull, tcommon);
  const double nan = std::numeric_limits<double>::quiet_NaN();
  for (int64_t k = 0; k < n; ++k) {
    // K: index in the whole ensemble (grid position and random-number counter); k: slot in this state's planes
    const int64_t K = g->k0 + k;
    const int64_t i = K % g->gx, j = K / g->gx;
    double st[6];
    // P:97 "the corresponding initial velocity v_z was calculated from the fixed energy condition": a draw of
    // (v_x, v_y, X) with 2(E - eps H_p(X)) < v_x^2 + v_y^2 has no real v_z.  Reading R31: with resample > 0 the
    // trajectory is drawn again — attempt a takes ALL its draws (angles and cloud point) from the seed
    // seed_a = seed + a * 0xD1B54A32D192ED03 (mod 2^64) — until it lies on the shell; the accepted points are
    // distributed exactly like the unmasked points of the plain ensemble (rejection sampling).
    const int attempts = (g->shape == 1 || g->shape == 2 || g->shape == 4) && g->resample > 0 ? g->resample + 1 : 1;
    for (int a = 0; a < attempts; ++a) {
      const uint64_t sd = seed + (uint64_t)a * 0xD1B54A32D192ED03ull;
      double X[3] = {0.0, 0.0, 0.0};
      if (g->angle_mode == 1)
        for (int al = 0; al < 3; ++al) X[al] = TWO_PI_HI * uniform01(sd, (uint64_t)K, (uint64_t)al);
      if (g->shape == 3) {
        // P:85 "initial conditions uniformly distributed over the sphere S": direction uniform on the unit
        // sphere (cos(theta) = 1 - 2 u3 uniform in (-1, 1], phi = 2 pi u4), |P| from the energy condition
        // H = E: |P|^2 = 2 (E - eps H_p(X)) > 0 always (E > 2|eps|), so no point is off the shell (R28).
        const double u1 = uniform01(sd, (uint64_t)K, 3), u2 = uniform01(sd, (uint64_t)K, 4);
        const double ct = 1.0 - 2.0 * u1;
        const double sth = std::sqrt((1.0 - ct) * (1.0 + ct));
        const double ang = TWO_PI_HI * u2;
        const double pn = std::sqrt(2.0 * (E - eps * Hp(X[0], X[1], X[2])));
        status[k] = 1;
        st[0] = X[0]; st[1] = X[1]; st[2] = X[2];
        st[3] = pn * (sth * std::cos(ang));
        st[4] = pn * (sth * std::sin(ang));
        st[5] = (g->pz_sign < 0 ? -1.0 : 1.0) * (pn * ct);
      } else {
        double px, py;
        if (g->shape == 0) {
          px = g->lo_x + ((double)i + 0.5) * (g->hi_x - g->lo_x) / (double)g->gx;
          py = g->lo_y + ((double)j + 0.5) * (g->hi_y - g->lo_y) / (double)g->gy;
        } else if (g->shape == 4) {
          // P:87 "initial conditions uniformly distributed within a small segment of the sphere (enclosed by the two
          // squares in Fig. 2 (a))": the segment is a square in the view of S along the third axis, i.e. a rectangle
          // in (px, py), sampled uniformly at random (R33); v_z from the energy condition as for the clouds
          const double u1 = uniform01(sd, (uint64_t)K, 3), u2 = uniform01(sd, (uint64_t)K, 4);
          px = g->lo_x + u1 * (g->hi_x - g->lo_x);
          py = g->lo_y + u2 * (g->hi_y - g->lo_y);
        } else {
          const double u1 = uniform01(sd, (uint64_t)K, 3), u2 = uniform01(sd, (uint64_t)K, 4);
          const double ang = TWO_PI_HI * u2;
          const double rad = (g->shape == 1) ? g->r * std::sqrt(u1)
                                             : g->r * std::sqrt(-2.0 * std::log(1.0 - u1));
          px = g->cx + rad * std::cos(ang);
          py = g->cy + rad * std::sin(ang);
        }
        // third action from the energy condition H = E
        double R = 2.0 * (E - eps * Hp(X[0], X[1], X[2]));
        R = R - px * px;
        R = R - py * py;
        if (R < 0.0 || !(R == R)) {
          status[k] = 0;
          for (int c = 0; c < 6; ++c) st[c] = nan;
        } else {
          status[k] = 1;
          st[0] = X[0]; st[1] = X[1]; st[2] = X[2];
          st[3] = px; st[4] = py;
          st[5] = (g->pz_sign < 0 ? -1.0 : 1.0) * std::sqrt(R);
        }
      }
      if (status[k] == 1) break;
    }
    for (int c = 0; c < 6; ++c) q[c * pitch + k] = st[c];
    acc[0 * pitch + k] = 0.0;                                          // logsum
    acc[1 * pitch + k] = 0.0;                                          // fli_max
    acc[2 * pitch + k] = status[k] ? Hamiltonian(st, eps) : nan;       // H0
    acc[3 * pitch + k] = 0.0;                                          // dH_max
    if (w) {
      double t[6];
      if (g->tangent_mode == 1) unit_tangent(seed, (uint64_t)K, t);
      else std::memcpy(t, tcommon, sizeof t);
      for (int c = 0; c < 6; ++c) w[c * pitch + k] = t[c];
    }
    if (wind)
      for (int c = 0; c < 3; ++c) wind[c * pitch + k] = 0;
  }
  return 0;
}

// a2 + a3 + a4: integrate trajectories k in [k0, k1) for `steps` steps, checkpoint every `stride`.
// surv = NULL or the survivor rectangle {lo_x, hi_x, lo_y, hi_y} (R25).
int awo_integrate(int64_t n, int64_t pitch, double *q, double *w, double *acc, int32_t *wind,
                  uint8_t *status, double eps, int order, int64_t steps, double dt, int64_t stride,
                  int64_t k0, int64_t k1, const double *surv) {
  if (!q || !acc || !status || stride <= 0 || steps < 0 || steps % stride != 0) return -1;
  if (k0 < 0 || k1 > n || pitch < n) return -1;
  double a[10], b[9];
  const int S = stage_constants(order, dt, eps, a, b);
  if (S == 0) return -1;
  for (int64_t k = k0; k < k1; ++k) {
    if (status[k] != 1) continue;
    double s[6], t[6], ac[4];
    int32_t wd[3] = {0, 0, 0};
    for (int c = 0; c < 6; ++c) s[c] = q[c * pitch + k];
    if (w) for (int c = 0; c < 6; ++c) t[c] = w[c * pitch + k];
    for (int c = 0; c < 4; ++c) ac[c] = acc[c * pitch + k];
    if (wind) for (int c = 0; c < 3; ++c) wd[c] = wind[c * pitch + k];
    int stt = 1;
    for (int64_t c0 = 0; c0 < steps; c0 += stride) {
      for (int64_t i = 0; i < stride; ++i) one_step(s, w ? t : nullptr, S, a, b);
      stt = checkpoint(s, w ? t : nullptr, ac, wd, eps, surv);
      if (stt != 1) break;
    }
    status[k] = (uint8_t)stt;
    for (int c = 0; c < 6; ++c) q[c * pitch + k] = s[c];
    if (w) for (int c = 0; c < 6; ++c) w[c * pitch + k] = t[c];
    for (int c = 0; c < 4; ++c) acc[c * pitch + k] = ac[c];
    if (wind) for (int c = 0; c < 3; ++c) wind[c * pitch + k] = wd[c];
  }
  return 0;
}

// a5: indicator image (R13, R14).  kind 0 FLI, 1 FTLE (= logsum / t), 2 DH -> out_f64[n];
// kind 3 CLASS -> out_u8[n] (1 if FLI > thr else 0; 255 for trajectories that are not live).
int awo_indicator(int64_t n, int64_t pitch, const double *acc, const uint8_t *status, double t,
                  int kind, double thr, double *out_f64, uint8_t *out_u8) {
  const double nan = std::numeric_limits<double>::quiet_NaN();
  for (int64_t k = 0; k < n; ++k) {
    const bool live = status[k] == 1;
    if (kind == 0) out_f64[k] = live ? acc[1 * pitch + k] : nan;
    else if (kind == 1) out_f64[k] = live ? acc[0 * pitch + k] / t : nan;
    else if (kind == 2) out_f64[k] = live ? acc[3 * pitch + k] : nan;
    else if (kind == 3) out_u8[k] = live ? (acc[1 * pitch + k] > thr ? 1 : 0) : 255;
    else return -1;
  }
  return 0;
}

// a6: visited-cell density over the first two actions (R19, R20).  Adds into hist.
int awo_density(int64_t n, int64_t pitch, const double *q, const uint8_t *status, uint32_t *hist,
                int32_t gx, int32_t gy, double lo, double hi, uint64_t *dropped) {
  if (!(hi > lo) || gx <= 0 || gy <= 0) return -1;
  const double fx = (double)gx / (hi - lo), fy = (double)gy / (hi - lo);
  for (int64_t k = 0; k < n; ++k) {
    if (status[k] != 1) continue;
    const double px = q[3 * pitch + k], py = q[4 * pitch + k];
    const double ax = std::floor((px - lo) * fx), ay = std::floor((py - lo) * fy);
    if (ax >= 0.0 && ax < (double)gx && ay >= 0.0 && ay < (double)gy)
      hist[(int64_t)ay * gx + (int64_t)ax] += 1u;
    else if (dropped) *dropped += 1ull;
  }
  return 0;
}

// ---------------------------------------------------------------- the paper's own indicator
//
// "For every trajectory from the ensemble we calculate the vector of the averaged finite-time velocity
//  V^i(t) with the components V_a(t) = [X_a(t + Dt) - X_a(t)] / Dt", where X is the unwrapped
// coordinate: the checkpoint wraps the angles and counts whole turns (R7), so
//   X_a(t + Dt) - X_a(t) = (x_a - xref_a) + 2 pi (wind_a - windref_a)                        (R27)
// with (xref, windref) the snapshot taken at time t (awo_mark).  "Finally we use the central projection
// of the point V on the surface of the sphere" S: P^2 = 2E (P:171 fn. 26): Vhat = sqrt(2E) V / |V|.
// Every product, sum, quotient and root below is rounded separately, in exactly this order.

// snapshot of the state at the start of an averaging window: qref <- q (6 planes), windref <- wind
int awo_mark(int64_t pitch, const double *q, const int32_t *wind, double *qref, int32_t *windref) {
  if (!q || !qref) return -1;
  std::memcpy(qref, q, sizeof(double) * 6 * (size_t)pitch);
  if (wind && windref) std::memcpy(windref, wind, sizeof(int32_t) * 3 * (size_t)pitch);
  return 0;
}

namespace {
// V (averaged velocity) and Vhat (its central projection on S) of trajectory k; false if |V| is zero
// or not finite (nothing to project).
inline bool averaged_velocity(int64_t k, int64_t pitch, const double *q, const int32_t *wind,
                              const double *qref, const int32_t *windref, double E, double Dt,
                              double V[3], double Vhat[3]) {
  for (int a = 0; a < 3; ++a) {
    const double dxw = q[a * pitch + k] - qref[a * pitch + k];
    const int32_t dk = (wind && windref) ? wind[a * pitch + k] - windref[a * pitch + k] : 0;
    const double dX = (double)dk * TWO_PI_HI + dxw;
    V[a] = dX / Dt;
  }
  double n2 = V[0] * V[0];
  n2 = n2 + V[1] * V[1];
  n2 = n2 + V[2] * V[2];
  const double nrm = std::sqrt(n2);
  if (!(nrm > 0.0) || !std::isfinite(nrm)) return false;
  const double scale = std::sqrt(2.0 * E) / nrm;
  for (int a = 0; a < 3; ++a) Vhat[a] = V[a] * scale;
  return true;
}
}  // namespace

// out[3*n] (planes of n): kind 0 -> V, kind 1 -> Vhat; NaN where the trajectory is not live or |V| = 0
int awo_velocity(int64_t n, int64_t pitch, const double *q, const int32_t *wind, const double *qref,
                 const int32_t *windref, const uint8_t *status, double E, double Dt, int kind, double *out) {
  if (!q || !qref || !status || !out || !(Dt > 0.0)) return -1;
  const double nan = std::numeric_limits<double>::quiet_NaN();
  for (int64_t k = 0; k < n; ++k) {
    double V[3], Vh[3];
    const bool ok = status[k] == 1 && averaged_velocity(k, pitch, q, wind, qref, windref, E, Dt, V, Vh);
    for (int a = 0; a < 3; ++a) out[a * n + k] = ok ? (kind == 0 ? V[a] : Vh[a]) : nan;
  }
  return 0;
}

// Density F_Dt(V; t) of the projected averaged velocity on the sphere S, as the sphere seen along
// the third axis (R26): bins over (Vhat_x, Vhat_y) exactly as awo_density bins (px, py); hemi = 1 counts
// the hemisphere Vhat_z >= 0, hemi = 2 the hemisphere Vhat_z < 0, hemi = 3 both (folded).  Points of
// the other hemisphere, outside [lo, hi)^2, or with |V| = 0 go to *dropped.  Adds into hist.
int awo_density_velocity(int64_t n, int64_t pitch, const double *q, const int32_t *wind, const double *qref,
                         const int32_t *windref, const uint8_t *status, double E, double Dt, int hemi,
                         uint32_t *hist, int32_t gx, int32_t gy, double lo, double hi, uint64_t *dropped) {
  if (!(hi > lo) || gx <= 0 || gy <= 0 || !(Dt > 0.0) || hemi < 1 || hemi > 3) return -1;
  const double fx = (double)gx / (hi - lo), fy = (double)gy / (hi - lo);
  for (int64_t k = 0; k < n; ++k) {
    if (status[k] != 1) continue;
    double V[3], Vh[3];
    bool in = averaged_velocity(k, pitch, q, wind, qref, windref, E, Dt, V, Vh);
    if (in) in = (hemi == 3) || (hemi == 1 ? Vh[2] >= 0.0 : Vh[2] < 0.0);
    if (in) {
      const double ax = std::floor((Vh[0] - lo) * fx), ay = std::floor((Vh[1] - lo) * fy);
      in = ax >= 0.0 && ax < (double)gx && ay >= 0.0 && ay < (double)gy;
      if (in) hist[(int64_t)ay * gx + (int64_t)ax] += 1u;
    }
    if (!in && dropped) *dropped += 1ull;
  }
  return 0;
}

// Drift detector of P:37: dP(t) = ||P(t) - P(0)||, with P(0) the marked snapshot.  out[n], NaN if not live.
int awo_delta_p(int64_t n, int64_t pitch, const double *q, const double *qref, const uint8_t *status,
                double *out) {
  if (!q || !qref || !status || !out) return -1;
  const double nan = std::numeric_limits<double>::quiet_NaN();
  for (int64_t k = 0; k < n; ++k) {
    if (status[k] != 1) { out[k] = nan; continue; }
    const double d0 = q[3 * pitch + k] - qref[3 * pitch + k];
    const double d1 = q[4 * pitch + k] - qref[4 * pitch + k];
    const double d2 = q[5 * pitch + k] - qref[5 * pitch + k];
    double s2 = d0 * d0;
    s2 = s2 + d1 * d1;
    s2 = s2 + d2 * d2;
    out[k] = std::sqrt(s2);
  }
  return 0;
}

// "Energy-drift statistics" of BJ:configs[2] (R29): over the live trajectories, from the checkpointed maximum
// dH_max = max_t |H(t) - H0| (acc plane 3) and the signed error of the CURRENT state, H(X, P) - H0:
//   out[0] live count   out[1] max dH_max   out[2] mean dH_max   out[3] rms dH_max
//   out[4] mean signed  out[5] rms signed   out[6] index of the trajectory with the largest dH_max (first one)
//   out[7] max |signed|
// A symplectic scheme shows no secular growth: the signed mean stays at the rounding level and
// dH_max does not grow with t.  Plain left-to-right sums.  signed_out (may be NULL): the signed image, NaN
// where the trajectory is not live.
int awo_energy_stats(int64_t n, int64_t pitch, const double *q, const double *acc, const uint8_t *status,
                     double eps, double *out, double *signed_out) {
  if (!q || !acc || !status || !out) return -1;
  const double nan = std::numeric_limits<double>::quiet_NaN();
  double cnt = 0.0, mx = 0.0, sum = 0.0, sq = 0.0, ssum = 0.0, ssq = 0.0, smax = 0.0, worst = -1.0;
  for (int64_t k = 0; k < n; ++k) {
    if (status[k] != 1) { if (signed_out) signed_out[k] = nan; continue; }
    double st[6];
    for (int c = 0; c < 6; ++c) st[c] = q[c * pitch + k];
    const double sd = Hamiltonian(st, eps) - acc[2 * pitch + k];
    const double d = acc[3 * pitch + k];
    if (signed_out) signed_out[k] = sd;
    cnt += 1.0;
    if (d > mx || worst < 0.0) { mx = d; worst = (double)k; }
    sum += d;
    sq += d * d;
    ssum += sd;
    ssq += sd * sd;
    if (std::fabs(sd) > smax) smax = std::fabs(sd);
  }
  out[0] = cnt; out[1] = mx; out[6] = worst; out[7] = smax;
  out[2] = cnt > 0.0 ? sum / cnt : nan;
  out[3] = cnt > 0.0 ? std::sqrt(sq / cnt) : nan;
  out[4] = cnt > 0.0 ? ssum / cnt : nan;
  out[5] = cnt > 0.0 ? std::sqrt(ssq / cnt) : nan;
  return 0;
}

}  // extern "C"
