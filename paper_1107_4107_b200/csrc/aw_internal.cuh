// aw_internal.cuh — declarations shared by the translation units of libaw (not part of the ABI).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include "../../include/aw.h"

namespace aw {

constexpr int kMaxStages = 7;
constexpr int kTrigTerms = 8;  // largest Taylor degree N of the drift rotations (level 7, 2z pair)

// Kernel parameters of the integrator; lives in the constant bank (__grid_constant__), so the stage
// constants are constant-bank operands of the DFMA instructions and cost no registers.
struct IntegrateParams {
  double *q;
  double *w;
  double *acc;
  int32_t *wind;
  uint8_t *status;
  int64_t n, pitch;
  int32_t nchk;    // checkpoints in this launch
  int32_t stride;  // steps between checkpoints
  int32_t chunk;   // steps between re-synchronisations of the running (sin, cos) pairs; divides the
                   // stride into equal-as-possible pieces of <= kMaxChunk steps (a function of stride only)
  int32_t level;   // trigonometry variant picked on the host from the largest drift angle (aw_integrate.cu)
  double a_open;   // a_1 (= a_{S+1}): angle drift that opens a block of `stride` steps; the block is closed by
                   // the angle drift -a_open, which takes the last merged drift back to the step boundary
  // Drift after kick s (s = 0..S-1): a_2 .. a_S, then a_{S+1} + a_1 (closing drift of one step merged with the
  // opening drift of the next).  The kernel's momentum-like variables are twice the natural ones (aw_integrate.cu,
  // struct Traj), so u, v (and du, dv) advance with a/2 and zeta = 2z (and dzeta) with a.
  double a_loop[kMaxStages];   // a: zeta += a pzeta, dzeta += a Q
  double ah_loop[kMaxStages];  // a / 2 (exact): u += (a/2) pu', du += (a/2) Pu
  // Rotation of the running (sin, cos) pairs through the drift after kick s by the angle d = A p as polynomials in
  // z = p^2 (aw_integrate.cu):   sin d = p (G[0] + G[1] z + ...),  G[i] = (-1)^i A^(2i+1) / (2i+1)!   (G[0] = A exactly)
  //                              cos d - 1 = z (M[0] + M[1] z + ...),  M[i] = (-1)^(i+1) A^(2i+2) / (2i+2)!
  // one set for the u and v pairs (A = a/2, p = pu', pv') and one for the zeta pair (A = a, p = pzeta)
  double grot_uv[kMaxStages][kTrigTerms + 1], mrot_uv[kMaxStages][kTrigTerms];
  double grot_z[kMaxStages][kTrigTerms + 1], mrot_z[kMaxStages][kTrigTerms];
  double b2[kMaxStages];     // 2 b_s
  double rho[kMaxStages];    // b_s / b_0 (0 if b_0 = 0): the zeta pair is carried scaled by 2 b_0 (aw_integrate.cu, kick)
  double b4[kMaxStages];     // 4 b_s  and
  double rho2[kMaxStages];   // 2 b_s / b_0: the same two factors for the 7-stage scheme, whose pzt is 4 pz
  double eps;
  int32_t survive;  // survivor filter (R25): 1 = test (px, py) against surv[] at every checkpoint
  int32_t block;    // threads per block (32, 64 or 128)
  double surv[4];   // lo_x, hi_x, lo_y, hi_y (half-open)
};

struct InitParams {
  double *q;
  double *w;
  double *acc;
  int32_t *wind;
  uint8_t *status;
  int64_t n, pitch;
  aw_grid g;
  double E, eps;
  uint64_t seed;
  double tcommon[6];
};

// host-side launchers (each returns cudaError_t of the launch and bumps the launch counter)
cudaError_t launch_integrate(const IntegrateParams &p, int order, bool tangent, bool latency, cudaStream_t st);
// which of the two ptxas schedules of the same kernel to launch (aw_state.flavour; aw_integrate.cu)
bool integrate_latency_flavour(int64_t n, int forced);
// Trigonometry variant for a largest drift angle max_s |a_s| * max|p| (0 = full sincos every stage).
int trig_level_for(double max_drift_angle);
// largest drift angle max_s |a_s| * max|p| the level supports (infinity for level 0)
double trig_level_max_angle(int level);
int integrate_block_size(int64_t n, int forced, bool uses_table);
bool kernel_uses_table(int order, int level);
// true if |a_loop[s]| / max |a_loop| are within the ratios the per-drift Taylor degrees were derived for
bool drift_ratios_hold(int S, const double *a_loop);
constexpr int kMaxChunk = 128;
cudaError_t launch_init(const InitParams &p, cudaStream_t st);
cudaError_t launch_indicator(const double *acc, const uint8_t *status, int64_t n, int64_t pitch, int kind,
                             double thr, double t, void *out, cudaStream_t st);
// Everything the averaged-velocity front end needs (R26, R27): current and marked planes.
struct VelocityArgs {
  const double *q, *qref;          // 6*pitch each
  const int32_t *wind, *windref;   // 3*pitch each or both NULL
  int64_t pitch;
  double Dt;      // t - tref > 0
  double radius;  // sqrt(2E), rounded once on the host
};
// kinds AW_IND_DP, AW_IND_VX..VZ
cudaError_t launch_indicator_ref(const VelocityArgs &v, const uint8_t *status, int64_t n, int kind, double *out,
                                 cudaStream_t st);
// mode 0: bins (px, py) = planes 3, 4 of v.q; modes 1-3: bins (Vhat_x, Vhat_y) of one / both hemispheres
cudaError_t launch_density(const VelocityArgs &v, int mode, const uint8_t *status, int64_t n,
                           uint32_t *hist, int32_t gx, int32_t gy, double lo, double fx, double fy,
                           unsigned long long *dropped, cudaStream_t st);
int64_t energy_stats_blocks(int64_t n);
size_t energy_partial_bytes();
cudaError_t launch_energy_stats(const double *q, const double *acc, const uint8_t *status, int64_t n, int64_t pitch,
                                double eps, void *scratch, double *out, cudaStream_t st);
// the same two kernels with the block partials in the library's own static device array (aw_energy_stats_noalloc)
int64_t energy_stats_noalloc_max_n();
cudaError_t launch_energy_stats_noalloc(const double *q, const double *acc, const uint8_t *status, int64_t n,
                                        int64_t pitch, double eps, double *out, cudaStream_t st);
cudaError_t launch_signed_dh(const double *q, const double *acc, const uint8_t *status, int64_t n, int64_t pitch,
                             double eps, double *out, cudaStream_t st);
// max over live, finite trajectories of H(X,P), as a monotone 64-bit key (0 = none) in *key_out (aw_bound_energy)
cudaError_t launch_energy_bound(const double *q, const uint8_t *status, int64_t n, int64_t pitch, double eps,
                                unsigned long long *key_out, cudaStream_t st);
double energy_key_decode(unsigned long long key, bool *any);
// status <- AW_ST_RANGE where a live trajectory's H(X,P) exceeds hmax (the precondition of the integrator's arithmetic)
cudaError_t launch_range_check(const double *q, uint8_t *status, int64_t n, int64_t pitch, double eps, double hmax,
                               cudaStream_t st);

void count_launch();

// ---- device helpers shared by kernels --------------------------------------------------------------
#ifdef __CUDACC__
// mix64 / u(seed, k, slot) — the counter-based generator specified in include/aw.h (R11).
__host__ __device__ __forceinline__ uint64_t mix64(uint64_t seed, uint64_t ctr) {
  uint64_t z = seed + ctr * 0x9E3779B97F4A7C15ull;
  z ^= z >> 30;
  z *= 0xBF58476D1CE4E5B9ull;
  z ^= z >> 27;
  z *= 0x94D049BB133111EBull;
  z ^= z >> 31;
  return z;
}
__host__ __device__ __forceinline__ double uniform01(uint64_t seed, uint64_t k, uint64_t slot) {
  return (double)(mix64(seed, 16ull * k + slot) >> 11) * (1.0 / 9007199254740992.0);
}
#endif

}  // namespace aw
