// aw_api.cu — the C ABI of include/aw.h: host-side validation, stage constants, launch chaining.
// Every entry validates on the host before any launch and returns an aw_status; nothing here touches
// trajectory data on the CPU (there is no CPU fallback — without a device the calls return AW_ECUDA).
#include <atomic>
#include <cmath>
#include <cstring>
#include <mutex>

#include "aw_internal.cuh"

namespace aw {

static thread_local int g_last_cuda = 0;
static std::atomic<uint64_t> g_launches{0};

void count_launch() { g_launches.fetch_add(1, std::memory_order_relaxed); }

static int cuda_fail(cudaError_t e) {
  g_last_cuda = (int)e;
  return AW_ECUDA;
}
#define AW_CUDA(call)                                  \
  do {                                                 \
    cudaError_t e_ = (call);                           \
    if (e_ != cudaSuccess) return ::aw::cuda_fail(e_); \
  } while (0)

// ---- stage weights of the composition (R1, R2) -----------------------------------------------------
//
// order 4: triple jump, closed form.  order 6: 7-stage palindromic composition (w3 w2 w1 w0 w1 w2 w3);
// the paper prints no coefficients, so they are obtained here as the root of the four order conditions
//   sum g = 1, sum g^3 = 0, sum g^5 = 0, sum_i g_i^3 (sum_{j<i} g_j + g_i/2)^2 = 0
// nearest to Yoshida's "solution A" (smallest max |w|), by Newton iteration in long double with a
// central-difference Jacobian (ample: the system is polynomial and well conditioned at the root; the
// iteration converges to the long-double root, which is then rounded once to double).
static void y6_conditions(const long double w[4], long double f[4]) {
  const long double g[7] = {w[3], w[2], w[1], w[0], w[1], w[2], w[3]};
  long double e1 = -1.0L, e3 = 0.0L, e5 = 0.0L, e7 = 0.0L, pre = 0.0L;
  for (int i = 0; i < 7; ++i) {
    const long double x = g[i], x3 = x * x * x, mid = pre + x / 2;
    e1 += x;
    e3 += x3;
    e5 += x3 * x * x;
    e7 += x3 * mid * mid;
    pre += x;
  }
  f[0] = e1; f[1] = e3; f[2] = e5; f[3] = e7;
}

static void solve4(long double A[4][4], long double b[4]) {  // Gaussian elimination, partial pivoting
  for (int c = 0; c < 4; ++c) {
    int piv = c;
    for (int r = c + 1; r < 4; ++r)
      if (fabsl(A[r][c]) > fabsl(A[piv][c])) piv = r;
    for (int k = 0; k < 4; ++k) { long double t = A[c][k]; A[c][k] = A[piv][k]; A[piv][k] = t; }
    { long double t = b[c]; b[c] = b[piv]; b[piv] = t; }
    for (int r = c + 1; r < 4; ++r) {
      const long double m = A[r][c] / A[c][c];
      for (int k = c; k < 4; ++k) A[r][k] -= m * A[c][k];
      b[r] -= m * b[c];
    }
  }
  for (int r = 3; r >= 0; --r) {
    for (int k = r + 1; k < 4; ++k) b[r] -= A[r][k] * b[k];
    b[r] /= A[r][r];
  }
}

static const double *yoshida6_weights() {
  static double w6[4];
  static std::once_flag once;
  std::call_once(once, [] {
    long double w[4] = {1.3152L, -1.1777L, 0.2356L, 0.7845L};  // 4-digit neighbourhood of solution A
    for (int it = 0; it < 40; ++it) {
      long double f[4], J[4][4];
      y6_conditions(w, f);
      for (int c = 0; c < 4; ++c) {
        const long double h = 1e-9L;
        long double wp[4], wm[4], fp[4], fm[4];
        for (int k = 0; k < 4; ++k) wp[k] = wm[k] = w[k];
        wp[c] += h; wm[c] -= h;
        y6_conditions(wp, fp);
        y6_conditions(wm, fm);
        for (int r = 0; r < 4; ++r) J[r][c] = (fp[r] - fm[r]) / (2 * h);
      }
      long double rhs[4] = {-f[0], -f[1], -f[2], -f[3]};
      solve4(J, rhs);
      long double step = 0;
      for (int k = 0; k < 4; ++k) { w[k] += rhs[k]; step = fmaxl(step, fabsl(rhs[k])); }
      if (step < 1e-19L) break;
    }
    for (int k = 0; k < 4; ++k) w6[k] = (double)w[k];
  });
  return w6;
}

static int stage_list(int order, double w[kMaxStages]) {
  if (order == 4) {
    const double cbrt2 = std::cbrt(2.0);
    w[0] = 1.0 / (2.0 - cbrt2);
    w[1] = -cbrt2 / (2.0 - cbrt2);
    w[2] = w[0];
    return 3;
  }
  if (order == 6) {
    const double *y = yoshida6_weights();
    w[0] = y[3]; w[1] = y[2]; w[2] = y[1]; w[3] = y[0]; w[4] = y[1]; w[5] = y[2]; w[6] = y[3];
    return 7;
  }
  return 0;
}

// a_s = c_s*dt with c_1 = w_1/2, c_s = (w_{s-1} + w_s)/2, c_{S+1} = w_S/2;  b_s = (eps*w_s)*dt  (R2)
static int stage_constants(int order, double dt, double eps, double a[kMaxStages + 1], double b[kMaxStages]) {
  double w[kMaxStages];
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

// ---- the common tangent vector (R12): host libm, counter k = 2^63 - 1, slots 5..10 -------------------
static void common_tangent(uint64_t seed, double t[6]) {
  const double two_pi_hi = 6.283185307179586;
  const uint64_t k = 0x7FFFFFFFFFFFFFFFull;
  for (int pr = 0; pr < 3; ++pr) {
    const double ua = uniform01(seed, k, 5 + 2 * pr), ub = uniform01(seed, k, 6 + 2 * pr);
    const double rad = std::sqrt(-2.0 * std::log(1.0 - ua));
    const double ang = two_pi_hi * ub;
    t[2 * pr] = rad * std::cos(ang);
    t[2 * pr + 1] = rad * std::sin(ang);
  }
  double s2 = 0.0;
  for (int i = 0; i < 6; ++i) s2 = s2 + t[i] * t[i];
  const double nu = std::sqrt(s2);
  for (int i = 0; i < 6; ++i) t[i] = t[i] / nu;
}

// Coefficients of the drift rotation by the angle d = A p as polynomials in z = p^2 (aw_internal.cuh):
// G[i] = (-1)^i A^(2i+1)/(2i+1)!  (G[0] = A exactly),  M[i] = (-1)^(i+1) A^(2i+2)/(2i+2)!; evaluated in long
// double and rounded once.
static void rotation_coefficients(double A, double G[kTrigTerms + 1], double M[kTrigTerms]) {
  const long double a = (long double)A, a2 = a * a;
  long double pw = a, fact = 1.0L;  // pw = A^(2i+1), fact = (2i+1)!
  for (int i = 0; i <= kTrigTerms; ++i) {
    if (i > 0) { pw *= a2; fact *= (long double)(2 * i) * (long double)(2 * i + 1); }
    G[i] = (double)((i & 1 ? -pw : pw) / fact);
    if (i < kTrigTerms) M[i] = (double)((i & 1 ? pw : -pw) * a / (fact * (long double)(2 * i + 2)));
  }
  G[0] = A;
}

static bool aligned16(const void *p) { return (reinterpret_cast<uintptr_t>(p) & 15u) == 0; }

static int check_planes(const aw_state *s) {
  if (!s) return AW_EINVAL;
  if (s->n < 0 || s->pitch < s->n || (s->pitch & 31) != 0) return AW_EINVAL;
  if (s->n > 0) {
    if (!s->q || !s->acc || !s->status) return AW_EINVAL;
    if (!aligned16(s->q) || !aligned16(s->acc) || (s->w && !aligned16(s->w)) ||
        (s->wind && !aligned16(s->wind)) || (s->qref && !aligned16(s->qref)) ||
        (s->windref && !aligned16(s->windref)))
      return AW_EINVAL;
  }
  return AW_OK;
}

// the marked snapshot is usable: planes present, wind/windref paired
static bool has_ref(const aw_state *s) { return s->qref && ((s->wind == nullptr) == (s->windref == nullptr)); }
// the averaged velocity needs the turn counters too: without them a trajectory that completed a turn inside the
// window would alias silently (the checkpoint wraps the angles whether or not the turns are counted)
static bool has_velocity_ref(const aw_state *s) { return s->qref && s->wind && s->windref; }

static bool aligned(const void *p, uintptr_t a) { return (reinterpret_cast<uintptr_t>(p) & (a - 1)) == 0; }

// energy bound the arithmetic is sized for: max(E, Emax); Emax = 0 / NaN / smaller means "use E"
static double energy_bound(const aw_state *s) { return (s->Emax > s->E) ? s->Emax : s->E; }

static VelocityArgs velocity_args(const aw_state *s) {
  VelocityArgs v;
  v.q = s->q; v.qref = s->qref; v.wind = s->wind; v.windref = s->windref;
  v.pitch = s->pitch;
  v.Dt = s->t - s->tref;
  v.radius = std::sqrt(2.0 * s->E);
  return v;
}

// what aw_integrate checks about its scalar arguments and the struct's switches (shared with the *_map_host calls,
// which must refuse a bad call before the first copy is enqueued)
static int validate_integrate_args(const aw_state *s, int64_t steps, double dt, int64_t stride) {
  if (steps < 0 || stride <= 0 || steps % stride != 0) return AW_EINVAL;
  if (!(dt != 0.0) || !std::isfinite(dt)) return AW_EINVAL;
  if (s->order != 4 && s->order != 6) return AW_ESTATE;
  if (!std::isfinite(s->E) || !std::isfinite(s->eps)) return AW_ESTATE;
  if (stride > 0x7fffffff) return AW_ERANGE;
  if (s->survive != 0 && s->survive != 1) return AW_EINVAL;
  if (s->survive && !(s->surv_hi_x > s->surv_lo_x && s->surv_hi_y > s->surv_lo_y)) return AW_EINVAL;
  if (s->block != 0 && s->block != 32 && s->block != 64 && s->block != 128) return AW_EINVAL;
  if (s->flavour < 0 || s->flavour > 2) return AW_EINVAL;
  return AW_OK;
}

}  // namespace aw

using namespace aw;

extern "C" {

const char *aw_strerror(int code) {
  switch (code) {
    case AW_OK: return "ok";
    case AW_EINVAL: return "invalid argument";
    case AW_ECUDA: return "CUDA runtime error (see aw_last_cuda_error)";
    case AW_ERANGE: return "argument out of the supported range";
    case AW_ESTATE: return "state not usable for this call";
    default: return "unknown aw_status";
  }
}

int aw_last_cuda_error(void) { return g_last_cuda; }
int aw_version(void) { return AW_VERSION; }
uint64_t aw_launch_count(void) { return g_launches.load(std::memory_order_relaxed); }

size_t aw_state_bytes(int64_t n, int with_tangent, int with_wind, int64_t *pitch_out) {
  if (n < 0) n = 0;
  const int64_t pitch = (n + 31) / 32 * 32;
  if (pitch_out) *pitch_out = pitch;
  size_t bytes = (size_t)6 * pitch * 8 + (size_t)4 * pitch * 8 + (size_t)n;
  if (with_tangent) bytes += (size_t)6 * pitch * 8;
  if (with_wind) bytes += (size_t)3 * pitch * 4;
  return bytes;
}

int aw_stage_constants(int order, double dt, double eps, double *a_host, double *b_host) {
  if (!a_host || !b_host) return AW_EINVAL;
  double a[kMaxStages + 1], b[kMaxStages];
  const int S = stage_constants(order, dt, eps, a, b);
  if (S == 0) return AW_EINVAL;
  std::memcpy(a_host, a, sizeof(double) * (S + 1));
  std::memcpy(b_host, b, sizeof(double) * S);
  return S;
}

int aw_trig_level(const aw_state *s, double dt) {
  if (!s || !(dt != 0.0) || !std::isfinite(dt)) return AW_EINVAL;
  if (!std::isfinite(s->E) || !std::isfinite(s->eps) || (s->order != 4 && s->order != 6)) return AW_ESTATE;
  if (s->trig) return 0;
  double a[kMaxStages + 1], b[kMaxStages];
  const int S = stage_constants(s->order, dt, s->eps, a, b);
  double amax = std::fmax(std::fabs(a[0]), std::fmax(std::fabs(a[S]), std::fabs(a[S] + a[0])));
  for (int k = 1; k < S; ++k) amax = std::fmax(amax, std::fabs(a[k]));
  return trig_level_for(amax * std::sqrt(2.0 * (energy_bound(s) + 2.0 * std::fabs(s->eps))));
}

int aw_block_size(const aw_state *s, double dt) {
  if (!s || s->n < 0) return AW_EINVAL;
  if (s->block != 0 && s->block != 32 && s->block != 64 && s->block != 128) return AW_EINVAL;
  const int level = aw_trig_level(s, dt);
  if (level < 0) return level;
  return integrate_block_size(s->n, s->block, kernel_uses_table(s->order, level));
}

int aw_kernel_schedule(const aw_state *s, double dt) {
  if (!s || s->n < 0 || s->flavour < 0 || s->flavour > 2) return AW_EINVAL;
  const int level = aw_trig_level(s, dt);
  if (level < 0) return level;
  return integrate_latency_flavour(s->n, s->flavour) ? 0 : 1;
}

int aw_common_tangent(uint64_t seed, double *t6_host) {
  if (!t6_host) return AW_EINVAL;
  common_tangent(seed, t6_host);
  return AW_OK;
}

int aw_init_shell(aw_state *s, const aw_grid *grid, double E, double eps, uint64_t seed) {
  if (!s || !grid) return AW_EINVAL;
  int rc = check_planes(s);
  if (rc != AW_OK) return rc;
  if (grid->gx <= 0 || grid->gy <= 0) return AW_EINVAL;
  if (grid->k0 < 0 || grid->k0 > (int64_t)grid->gx * grid->gy - s->n) return AW_EINVAL;  // slice inside the ensemble
  if (grid->angle_mode != 0 && grid->angle_mode != 1) return AW_EINVAL;
  if (grid->tangent_mode != 0 && grid->tangent_mode != 1) return AW_EINVAL;
  if (grid->resample < 0 || grid->resample > 1024) return AW_EINVAL;
  if (grid->shape == AW_SHAPE_GRID || grid->shape == AW_SHAPE_RECT) {
    if (!(grid->hi_x > grid->lo_x) || !(grid->hi_y > grid->lo_y)) return AW_EINVAL;
    if (!std::isfinite(grid->lo_x) || !std::isfinite(grid->hi_x) || !std::isfinite(grid->lo_y) ||
        !std::isfinite(grid->hi_y))
      return AW_EINVAL;
  } else if (grid->shape == AW_SHAPE_DISK || grid->shape == AW_SHAPE_GAUSS) {
    if (!(grid->r >= 0.0) || !std::isfinite(grid->r) || !std::isfinite(grid->cx) || !std::isfinite(grid->cy))
      return AW_EINVAL;
  } else if (grid->shape != AW_SHAPE_SPHERE) {
    return AW_EINVAL;
  }
  if (!std::isfinite(E) || !std::isfinite(eps) || !(E - 2.0 * std::fabs(eps) > 0.0)) return AW_ERANGE;

  if (s->n > 0) {
    InitParams p;
    p.q = s->q; p.w = s->w; p.acc = s->acc; p.wind = s->wind; p.status = s->status;
    p.n = s->n; p.pitch = s->pitch;
    p.g = *grid;
    p.E = E; p.eps = eps; p.seed = seed;
    common_tangent(seed, p.tcommon);
    AW_CUDA(launch_init(p, (cudaStream_t)s->stream));
  }
  s->E = E; s->Emax = E; s->eps = eps; s->t = 0.0; s->step = 0; s->ready = 1;
  if (s->order != 4 && s->order != 6) s->order = 4;
  return AW_OK;
}

int aw_integrate(aw_state *s, int64_t n, int64_t steps, double dt, int64_t stride) {
  if (!s) return AW_EINVAL;
  int rc = check_planes(s);
  if (rc != AW_OK) return rc;
  if (n != s->n) return AW_EINVAL;
  if ((rc = validate_integrate_args(s, steps, dt, stride)) != AW_OK) return rc;
  if (!s->ready) return AW_ESTATE;
  const double vmax = std::sqrt(2.0 * (energy_bound(s) + 2.0 * std::fabs(s->eps)));
  if (!((double)stride * std::fabs(dt) * vmax < 1024.0)) return AW_ERANGE;
  if (steps == 0 || n == 0) return AW_OK;

  double a[kMaxStages + 1], b[kMaxStages];
  const int S = stage_constants(s->order, dt, s->eps, a, b);
  IntegrateParams p;
  std::memset(&p, 0, sizeof p);
  p.q = s->q; p.w = s->w; p.acc = s->acc; p.wind = s->wind; p.status = s->status;
  p.n = s->n; p.pitch = s->pitch;
  p.stride = (int32_t)stride;
  // palindromic stage lists (order 4 and 6): a_1 == a_{S+1}, so the merged drift a_{S+1} + a_1 = 2 a_1 exactly
  if (a[0] != a[S]) return AW_ESTATE;
  p.a_open = a[0];
  for (int k = 1; k < S; ++k) p.a_loop[k - 1] = a[k];
  p.a_loop[S - 1] = a[S] + a[0];
  if (b[S - 1] != b[0]) return AW_ESTATE;  // palindromic: the outer stages share the weight the zeta pair is scaled by
  for (int k = 0; k < S; ++k) {
    p.b2[k] = 2.0 * b[k];
    p.rho[k] = (b[0] != 0.0) ? b[k] / b[0] : 0.0;
    p.b4[k] = 4.0 * b[k];
    p.rho2[k] = 2.0 * p.rho[k];
    p.ah_loop[k] = 0.5 * p.a_loop[k];
    rotation_coefficients(p.ah_loop[k], p.grot_uv[k], p.mrot_uv[k]);
    rotation_coefficients(p.a_loop[k], p.grot_z[k], p.mrot_z[k]);
  }
  p.eps = s->eps;
  p.survive = s->survive;
  p.surv[0] = s->surv_lo_x; p.surv[1] = s->surv_hi_x; p.surv[2] = s->surv_lo_y; p.surv[3] = s->surv_hi_y;
  // running-(sin, cos) variant: degree from the largest drift angle, re-synchronisation cadence from stride
  double amax = std::fabs(p.a_open);
  for (int k = 0; k < S; ++k) amax = std::fmax(amax, std::fabs(p.a_loop[k]));
  p.level = s->trig ? 0 : trig_level_for(amax * vmax);
  if (p.level > 0 && (amax != std::fabs(p.a_loop[S - 1]) || !drift_ratios_hold(S, p.a_loop))) p.level = 0;
  // the largest |P| this launch's arithmetic supports: the Taylor degrees of the level (kLevelMaxD / amax) and the
  // exact range of the two-constant argument reduction (R7: stride |dt| |P| < 1024); as an energy, P^2 <= 2(H + 2|eps|)
  {
    const double v_level = trig_level_max_angle(p.level) / amax;
    const double v_range = 1024.0 / ((double)stride * std::fabs(dt));
    const double v = std::fmin(v_level, v_range);
    const double hmax = 0.5 * v * v - 2.0 * std::fabs(s->eps);
    const cudaError_t e = launch_range_check(s->q, s->status, s->n, s->pitch, s->eps, hmax, (cudaStream_t)s->stream);
    if (e != cudaSuccess) return cuda_fail(e);
  }
  p.block = integrate_block_size(s->n, s->block, kernel_uses_table(s->order, p.level));
  const bool latency = integrate_latency_flavour(s->n, s->flavour);
  const int64_t pieces = (stride + kMaxChunk - 1) / kMaxChunk;
  p.chunk = (int32_t)((stride + pieces - 1) / pieces);

  const int64_t total_chk = steps / stride;
  int64_t chk_per_launch = AW_MAX_STEPS_PER_LAUNCH / stride;
  if (chk_per_launch < 1) chk_per_launch = 1;
  const double t0 = s->t;
  const int64_t step0 = s->step;
  for (int64_t done = 0; done < total_chk; done += chk_per_launch) {
    const int64_t now = (total_chk - done < chk_per_launch) ? total_chk - done : chk_per_launch;
    p.nchk = (int32_t)now;
    const cudaError_t e = launch_integrate(p, s->order, s->w != nullptr, latency, (cudaStream_t)s->stream);
    if (e != cudaSuccess) return cuda_fail(e);
    s->step = step0 + (done + now) * stride;
    s->t = t0 + (double)(s->step - step0) * std::fabs(dt);
  }
  return AW_OK;
}

int aw_mark(aw_state *s) {
  if (!s) return AW_EINVAL;
  int rc = check_planes(s);
  if (rc != AW_OK) return rc;
  if (!s->ready) return AW_ESTATE;
  if (s->n > 0 && !has_ref(s)) return AW_ESTATE;
  cudaStream_t st = (cudaStream_t)s->stream;
  if (s->n > 0) {
    AW_CUDA(cudaMemcpyAsync(s->qref, s->q, (size_t)6 * s->pitch * 8, cudaMemcpyDeviceToDevice, st));
    if (s->wind)
      AW_CUDA(cudaMemcpyAsync(s->windref, s->wind, (size_t)3 * s->pitch * 4, cudaMemcpyDeviceToDevice, st));
  }
  s->tref = s->t;
  return AW_OK;
}

int aw_indicator(const aw_state *s, int kind, double thr, void *out_dev) {
  if (!s || !out_dev) return AW_EINVAL;
  int rc = check_planes(s);
  if (rc != AW_OK) return rc;
  if (kind < AW_IND_FLI || kind > AW_IND_DHS) return AW_EINVAL;
  if (!s->ready) return AW_ESTATE;
  if (kind == AW_IND_DHS) {
    if (!aligned16(out_dev)) return AW_EINVAL;
    if (s->n == 0) return AW_OK;
    AW_CUDA(launch_signed_dh(s->q, s->acc, s->status, s->n, s->pitch, s->eps, static_cast<double *>(out_dev),
                             (cudaStream_t)s->stream));
    return AW_OK;
  }
  if (kind >= AW_IND_DP) {
    if (!has_ref(s)) return AW_ESTATE;
    if (kind != AW_IND_DP && (!has_velocity_ref(s) || !(s->t > s->tref))) return AW_ESTATE;
    if (!aligned16(out_dev)) return AW_EINVAL;
    if (s->n == 0) return AW_OK;
    AW_CUDA(launch_indicator_ref(velocity_args(s), s->status, s->n, kind, static_cast<double *>(out_dev),
                                 (cudaStream_t)s->stream));
    return AW_OK;
  }
  if (kind != AW_IND_DH && !s->w) return AW_ESTATE;
  if (kind == AW_IND_FTLE && !(s->t > 0.0)) return AW_ESTATE;
  if (kind == AW_IND_CLASS && thr != thr) return AW_EINVAL;
  if (kind != AW_IND_CLASS && !aligned16(out_dev)) return AW_EINVAL;
  if (s->n == 0) return AW_OK;
  AW_CUDA(launch_indicator(s->acc, s->status, s->n, s->pitch, kind, thr, s->t, out_dev,
                           (cudaStream_t)s->stream));
  return AW_OK;
}

size_t aw_energy_stats_scratch_bytes(int64_t n) {
  if (n < 0) n = 0;
  const int64_t nb = energy_stats_blocks(n);
  return (size_t)(nb > 0 ? nb : 1) * energy_partial_bytes();
}

int aw_energy_stats(const aw_state *s, void *scratch_dev, double *out_dev) {
  if (!s || !scratch_dev || !out_dev) return AW_EINVAL;
  int rc = check_planes(s);
  if (rc != AW_OK) return rc;
  if (!aligned16(scratch_dev) || !aligned16(out_dev)) return AW_EINVAL;
  if (!s->ready) return AW_ESTATE;
  AW_CUDA(launch_energy_stats(s->q, s->acc, s->status, s->n, s->pitch, s->eps, scratch_dev, out_dev,
                              (cudaStream_t)s->stream));
  return AW_OK;
}

int aw_energy_stats_noalloc(const aw_state *s, double *out_dev) {
  if (!s || !out_dev) return AW_EINVAL;
  int rc = check_planes(s);
  if (rc != AW_OK) return rc;
  if (!aligned16(out_dev)) return AW_EINVAL;
  if (s->n > AW_NOALLOC_MAX_N) return AW_ERANGE;   // the static scratch array holds AW_NOALLOC_MAX_N / 2048 partials
  if (!s->ready) return AW_ESTATE;
  AW_CUDA(launch_energy_stats_noalloc(s->q, s->acc, s->status, s->n, s->pitch, s->eps, out_dev,
                                      (cudaStream_t)s->stream));
  return AW_OK;
}

int aw_density(const aw_state *s, uint32_t *hist_dev, int32_t gx, int32_t gy, double lo, double hi,
               int mode, uint64_t *dropped_dev) {
  if (!s || !hist_dev) return AW_EINVAL;
  int rc = check_planes(s);
  if (rc != AW_OK) return rc;
  if (mode < AW_DENS_ACTION || mode > AW_DENS_VEL_BOTH || gx <= 0 || gy <= 0 || !(hi > lo) ||
      !std::isfinite(lo) || !std::isfinite(hi))
    return AW_EINVAL;
  if ((int64_t)gx * gy >= 0xffffffffll) return AW_ERANGE;
  if (!s->ready) return AW_ESTATE;
  if (!aligned(hist_dev, 4) || !aligned(dropped_dev, 8)) return AW_EINVAL;
  if (mode != AW_DENS_ACTION && (!has_velocity_ref(s) || !(s->t > s->tref))) return AW_ESTATE;
  if (s->n == 0) return AW_OK;
  const double fx = (double)gx / (hi - lo), fy = (double)gy / (hi - lo);
  AW_CUDA(launch_density(velocity_args(s), mode, s->status, s->n, hist_dev, gx, gy, lo, fx, fy,
                         reinterpret_cast<unsigned long long *>(dropped_dev), (cudaStream_t)s->stream));
  return AW_OK;
}

int aw_bound_energy(aw_state *s, void *scratch_dev) {
  if (!s || !scratch_dev) return AW_EINVAL;
  int rc = check_planes(s);
  if (rc != AW_OK) return rc;
  if (!aligned(scratch_dev, 8)) return AW_EINVAL;
  if (!s->ready || !std::isfinite(s->eps)) return AW_ESTATE;
  if (s->n == 0) return AW_OK;
  cudaStream_t st = (cudaStream_t)s->stream;
  unsigned long long key = 0ull;
  AW_CUDA(cudaMemsetAsync(scratch_dev, 0, 8, st));
  AW_CUDA(launch_energy_bound(s->q, s->status, s->n, s->pitch, s->eps, static_cast<unsigned long long *>(scratch_dev), st));
  AW_CUDA(cudaMemcpyAsync(&key, scratch_dev, 8, cudaMemcpyDeviceToHost, st));
  AW_CUDA(cudaStreamSynchronize(st));
  bool any = false;
  const double h = energy_key_decode(key, &any);
  if (any) s->Emax = h;
  return AW_OK;
}

}  // extern "C"

// Both *_map_host calls: everything that can be checked without the data is checked before the first copy is
// enqueued; once work is in flight every exit path synchronises the stream first (the header promises that the
// caller's host buffers are free again when the call returns).
namespace {
int synced(cudaStream_t st, int rc) {
  const cudaError_t e = cudaStreamSynchronize(st);
  if (rc == AW_OK && e != cudaSuccess) return ::aw::cuda_fail(e);
  return rc;
}
#define AW_CUDA_SYNCED(call)                                                      \
  do {                                                                            \
    cudaError_t e_ = (call);                                                      \
    if (e_ != cudaSuccess) { cudaStreamSynchronize(st); return ::aw::cuda_fail(e_); } \
  } while (0)

int validate_hist_args(int32_t gx, int32_t gy, double lo, double hi, const void *hist_dev) {
  if (gx <= 0 || gy <= 0 || !(hi > lo) || !std::isfinite(lo) || !std::isfinite(hi)) return AW_EINVAL;
  if ((int64_t)gx * gy >= 0xffffffffll) return AW_ERANGE;
  if (!hist_dev || !aligned(hist_dev, 8)) return AW_EINVAL;
  return AW_OK;
}

int upload_state(aw_state *s, const aw_host_in *in, cudaStream_t st) {
  const size_t P = (size_t)s->pitch;
  if (s->n == 0) return AW_OK;
  AW_CUDA_SYNCED(cudaMemcpyAsync(s->q, in->q, 6 * P * 8, cudaMemcpyHostToDevice, st));
  if (s->w) AW_CUDA_SYNCED(cudaMemcpyAsync(s->w, in->w, 6 * P * 8, cudaMemcpyHostToDevice, st));
  AW_CUDA_SYNCED(cudaMemcpyAsync(s->acc, in->acc, 4 * P * 8, cudaMemcpyHostToDevice, st));
  if (s->wind) AW_CUDA_SYNCED(cudaMemcpyAsync(s->wind, in->wind, 3 * P * 4, cudaMemcpyHostToDevice, st));
  AW_CUDA_SYNCED(cudaMemcpyAsync(s->status, in->status, (size_t)s->n, cudaMemcpyHostToDevice, st));
  return AW_OK;
}

int download_state(const aw_state *s, const aw_host_out *out, cudaStream_t st) {
  const size_t P = (size_t)s->pitch;
  if (s->n == 0) return AW_OK;
  if (out->q) AW_CUDA_SYNCED(cudaMemcpyAsync(out->q, s->q, 6 * P * 8, cudaMemcpyDeviceToHost, st));
  if (out->acc) AW_CUDA_SYNCED(cudaMemcpyAsync(out->acc, s->acc, 4 * P * 8, cudaMemcpyDeviceToHost, st));
  if (out->status) AW_CUDA_SYNCED(cudaMemcpyAsync(out->status, s->status, (size_t)s->n, cudaMemcpyDeviceToHost, st));
  return AW_OK;
}
}  // namespace

extern "C" {

int aw_map_host(aw_state *s, const aw_host_in *in, int64_t steps, double dt, int64_t stride, int kind,
                double thr, int32_t gx, int32_t gy, double lo, double hi, void *ind_dev, void *hist_dev,
                const aw_host_out *out) {
  if (!s || !in || !out) return AW_EINVAL;
  int rc = check_planes(s);
  if (rc != AW_OK) return rc;
  if (!in->q || !in->acc || !in->status || (s->w && !in->w) || (s->wind && !in->wind)) return AW_EINVAL;
  if ((rc = validate_integrate_args(s, steps, dt, stride)) != AW_OK) return rc;
  if (out->image) {  // what aw_indicator would refuse after the integration, refused now
    if (!ind_dev) return AW_EINVAL;
    if (kind < AW_IND_FLI || kind > AW_IND_DHS) return AW_EINVAL;
    if (kind >= AW_IND_DP && kind <= AW_IND_VZ) return AW_ESTATE;  // need a snapshot: aw_velocity_map_host
    if ((kind == AW_IND_FLI || kind == AW_IND_FTLE || kind == AW_IND_CLASS) && !s->w) return AW_ESTATE;
    if (kind == AW_IND_FTLE && !(s->t + (double)steps * std::fabs(dt) > 0.0)) return AW_ESTATE;
    if (kind == AW_IND_CLASS && thr != thr) return AW_EINVAL;
    if (kind != AW_IND_CLASS && !aligned16(ind_dev)) return AW_EINVAL;
  }
  if (out->hist && (rc = validate_hist_args(gx, gy, lo, hi, hist_dev)) != AW_OK) return rc;
  cudaStream_t st = (cudaStream_t)s->stream;
  if ((rc = upload_state(s, in, st)) != AW_OK) return rc;
  s->ready = 1;
  // the trigonometry level from the uploaded data, not from the struct's E
  void *scratch = (out->hist && hist_dev) ? hist_dev : (aligned(ind_dev, 8) ? ind_dev : nullptr);
  if (scratch && (rc = aw_bound_energy(s, scratch)) != AW_OK) return synced(st, rc);
  if ((rc = aw_integrate(s, s->n, steps, dt, stride)) != AW_OK) return synced(st, rc);
  if (out->image) {
    if ((rc = aw_indicator(s, kind, thr, ind_dev)) != AW_OK) return synced(st, rc);
    const size_t bytes = (kind == AW_IND_CLASS) ? (size_t)s->n : (size_t)s->n * 8;
    if (s->n > 0) AW_CUDA_SYNCED(cudaMemcpyAsync(out->image, ind_dev, bytes, cudaMemcpyDeviceToHost, st));
  }
  if (out->hist) {
    const size_t hb = (size_t)gx * gy * 4, off = (hb + 7) / 8 * 8;  // counter 8-byte aligned for any gx*gy
    AW_CUDA_SYNCED(cudaMemsetAsync(hist_dev, 0, off + 8, st));
    uint64_t *drop_dev = reinterpret_cast<uint64_t *>(static_cast<char *>(hist_dev) + off);
    if ((rc = aw_density(s, static_cast<uint32_t *>(hist_dev), gx, gy, lo, hi, 0, drop_dev)) != AW_OK)
      return synced(st, rc);
    AW_CUDA_SYNCED(cudaMemcpyAsync(out->hist, hist_dev, hb, cudaMemcpyDeviceToHost, st));
    if (out->dropped) AW_CUDA_SYNCED(cudaMemcpyAsync(out->dropped, drop_dev, 8, cudaMemcpyDeviceToHost, st));
  }
  if ((rc = download_state(s, out, st)) != AW_OK) return rc;
  return synced(st, AW_OK);
}

int aw_velocity_map_host(aw_state *s, const aw_host_in *in, int64_t steps, double dt, int64_t stride, int mode,
                         int32_t gx, int32_t gy, double lo, double hi, void *hist_dev, const aw_host_out *out) {
  if (!s || !in || !out || !hist_dev || !out->hist) return AW_EINVAL;
  int rc = check_planes(s);
  if (rc != AW_OK) return rc;
  if (!in->q || !in->acc || !in->status || (s->w && !in->w) || (s->wind && !in->wind)) return AW_EINVAL;
  if (mode < AW_DENS_VEL_UPPER || mode > AW_DENS_VEL_BOTH) return AW_EINVAL;
  if ((rc = validate_hist_args(gx, gy, lo, hi, hist_dev)) != AW_OK) return rc;
  if ((rc = validate_integrate_args(s, steps, dt, stride)) != AW_OK) return rc;
  if (s->n > 0 && !has_velocity_ref(s)) return AW_ESTATE;
  if (steps == 0) return AW_ESTATE;  // empty averaging window
  cudaStream_t st = (cudaStream_t)s->stream;
  if ((rc = upload_state(s, in, st)) != AW_OK) return rc;
  s->ready = 1;
  if ((rc = aw_bound_energy(s, hist_dev)) != AW_OK) return synced(st, rc);
  if ((rc = aw_mark(s)) != AW_OK) return synced(st, rc);
  if ((rc = aw_integrate(s, s->n, steps, dt, stride)) != AW_OK) return synced(st, rc);
  const size_t hb = (size_t)gx * gy * 4, off = (hb + 7) / 8 * 8;
  AW_CUDA_SYNCED(cudaMemsetAsync(hist_dev, 0, off + 8, st));
  uint64_t *drop_dev = reinterpret_cast<uint64_t *>(static_cast<char *>(hist_dev) + off);
  if ((rc = aw_density(s, static_cast<uint32_t *>(hist_dev), gx, gy, lo, hi, mode, drop_dev)) != AW_OK)
    return synced(st, rc);
  AW_CUDA_SYNCED(cudaMemcpyAsync(out->hist, hist_dev, hb, cudaMemcpyDeviceToHost, st));
  if (out->dropped) AW_CUDA_SYNCED(cudaMemcpyAsync(out->dropped, drop_dev, 8, cudaMemcpyDeviceToHost, st));
  if ((rc = download_state(s, out, st)) != AW_OK) return rc;
  return synced(st, AW_OK);
}

}  // extern "C"
