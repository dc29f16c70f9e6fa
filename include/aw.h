/* aw.h — C ABI of libaw: the ensemble hot path of arXiv 1107.4107 ("Mapping the Arnold web with a
 * GPU-supercomputer") as hand-written CUDA for sm_100a (NVIDIA B200).
 *
 * Citations: P:<n> = line n of the paper text; R<n> = reading n in DESIGN.md §3;
 * §8(x) = SURVEY.md hot-path scope table.
 *
 * What the library computes:
 *   model      H(P,X) = P^2/2 + eps * H_p(X)                       P:33 eq.(1)
 *              H_p(x,y,z) = cos x cos y (1 + cos 2z)                P:43 eq.(2)
 *   scheme     fixed-step symplectic composition (Yoshida 1990)     P:55, ref. 25
 *              order 6 (the paper's, 7 stages) or order 4 (BASELINE configs, 3 stages)      R1, R2
 *   ensemble   N independent realisations, one per GPU thread
 *   ICs        on the energy shell H = E, third action from the energy condition
 *   indicator  tangent vector through the exact derivative of the discrete map -> FLI / FTLE   R3, R13
 *   density    histogram of the ensemble over the first two actions, accumulated in time
 *
 * Conventions common to every entry point
 *   - returns an aw_status (0 = AW_OK, negative = error); never throws, never sets errno;
 *   - every argument is validated ON THE HOST before anything is launched;
 *   - all device work is enqueued asynchronously on aw_state.stream; no call synchronises unless its
 *     comment says so (aw_bound_energy and the *_host calls do);
 *   - the library never allocates or frees the caller's planes; pointers marked "device" must be
 *     device-accessible global memory, 16-byte aligned; "host" pointers are ordinary host memory;
 *   - thread-safe for distinct aw_state objects; the only library state is a thread-local
 *     last-CUDA-error code and a process-wide launch counter;
 *   - there is NO CPU fallback: without a CUDA device every compute entry returns AW_ECUDA.
 */
#ifndef AW_H_
#define AW_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define AW_VERSION 210 /* 2.1.0: + aw_energy_stats_noalloc.  2.0.0: aw_grid.k0, aw_state.Emax / block, AW_ST_RANGE, aw_bound_energy; probes out */

#if defined(__GNUC__)
#define AW_API __attribute__((visibility("default")))
#else
#define AW_API
#endif

typedef enum {
  AW_OK = 0,
  AW_EINVAL = -1, /* bad argument: null / misaligned plane, n mismatch, stride <= 0, ...       */
  AW_ECUDA = -2,  /* a CUDA runtime call failed; see aw_last_cuda_error()                       */
  AW_ERANGE = -3, /* argument outside the range the arithmetic supports (see aw_integrate)      */
  AW_ESTATE = -4  /* aw_state not usable for this call (not initialised, no tangent planes ...) */
} aw_status;

/* indicator kinds for aw_indicator (R13, R14; DP: P:37; VX..VZ: P:67 + fn. 26) */
enum { AW_IND_FLI = 0, AW_IND_FTLE = 1, AW_IND_DH = 2, AW_IND_CLASS = 3,
       AW_IND_DP = 4, AW_IND_VX = 5, AW_IND_VY = 6, AW_IND_VZ = 7, AW_IND_DHS = 8 };
/* aw_density modes: instantaneous actions (BASELINE) or the paper's projected averaged velocity (R19, R26) */
enum { AW_DENS_ACTION = 0, AW_DENS_VEL_UPPER = 1, AW_DENS_VEL_LOWER = 2, AW_DENS_VEL_BOTH = 3 };
/* aw_grid.shape */
enum { AW_SHAPE_GRID = 0, AW_SHAPE_DISK = 1, AW_SHAPE_GAUSS = 2, AW_SHAPE_SPHERE = 3, AW_SHAPE_RECT = 4 };
/* per-trajectory status byte */
enum { AW_ST_OFFSHELL = 0, AW_ST_LIVE = 1, AW_ST_NONFINITE = 2, AW_ST_LEFT = 3,
       AW_ST_RANGE = 4 /* energy above the bound aw_integrate was launched for (see aw_state.Emax): not integrated */ };

/* Static, never-freed description of a status code. */
AW_API const char *aw_strerror(int code);
/* cudaError_t (as int) of the last AW_ECUDA returned on the calling thread; 0 if none. */
AW_API int aw_last_cuda_error(void);
/* AW_VERSION the library was built from. */
AW_API int aw_version(void);
/* Number of CUDA kernels this library has launched in this process so far (monotonic). */
AW_API uint64_t aw_launch_count(void);

/* Ensemble state: structure-of-arrays planes in device memory, owned by the caller (§8(b)).
 * Plane c of a buffer starts at element c*pitch; trajectory k is element k of every plane, so a warp
 * reads 32 consecutive doubles per plane (coalesced 256-byte segments).  The struct is plain data. */
typedef struct {
  int64_t n;       /* trajectories                                                            */
  int64_t pitch;   /* elements between planes, >= n, multiple of 32                           */
  double *q;       /* device, 6*pitch: planes x, y, z, px, py, pz  (angles X, actions P)  */
  double *w;       /* device, 6*pitch tangent planes dx,dy,dz,dpx,dpy,dpz; NULL = no tangent  */
  double *acc;     /* device, 4*pitch: logsum, fli_max, H0, dH_max  (R4, R13, R16)            */
  int32_t *wind;   /* device, 3*pitch whole-turn counters of x,y,z (R7); NULL = not tracked   */
  uint8_t *status; /* device, n bytes: AW_ST_*                                                */
  double E, eps;   /* shell energy and perturbation strength (set by aw_init_shell; R5)       */
  double t;        /* elapsed model time, sum of steps*|dt| (advanced by aw_integrate)         */
  int64_t step;    /* elapsed steps                                                           */
  int32_t order;   /* 4 or 6 (R1); set by the caller before aw_integrate; default 4           */
  int32_t ready;   /* set to 1 by aw_init_shell (or by the caller after uploading a state)    */
  int32_t trig;    /* 0 (default): running (sin, cos) pairs advanced by rotations, see aw_integrate;
                      1: evaluate the device sincos at every stage                            */
  int32_t survive; /* 1: survivor filter on (R25), see surv_* below; 0 (default): off    */
  void *stream;    /* cudaStream_t; NULL = legacy default stream                              */
  double *qref;    /* device, 6*pitch: snapshot of q written by aw_mark (start of the averaging
                      window of P:67 / the P(0) of P:37); NULL = no snapshot planes             */
  int32_t *windref; /* device, 3*pitch: snapshot of wind; NULL iff wind is NULL                */
  double tref;     /* model time of the snapshot (set by aw_mark)                             */
  double surv_lo_x, surv_hi_x, surv_lo_y, surv_hi_y; /* launch rectangle of the survivor filter:
                      a trajectory whose (px, py) is outside [lo_x, hi_x) x [lo_y, hi_y) at a
                      checkpoint gets status AW_ST_LEFT and is frozen there                    */
  double Emax;     /* upper bound of H(X,P) over the live trajectories (P^2 <= 2(H + 2|eps|) on the whole orbit).
                      aw_integrate sizes its arithmetic (trigonometry level, angle range) for max(E, Emax) and CHECKS
                      it on the device: a trajectory with H above what the launch supports gets AW_ST_RANGE and is left
                      untouched, never integrated inaccurately.  aw_init_shell sets it to E; aw_bound_energy sets it
                      from the data (uploaded states); 0 / NaN = use E                              */
  int32_t block;   /* threads per block of the integrator: 0 (default) = chosen from n so that small ensembles
                      spread over all SMs; 32, 64 or 128 = forced.  The result does not depend on it    */
  int32_t flavour; /* the integrator kernels exist in two ptxas schedules of the same source and arithmetic: 1 = scheduled
                      for throughput (operand reuse; best with >= 3 warps per sub-partition), 2 = for latency
                      (interleaved chains; best for small ensembles); 0 (default) = chosen from n (latency up to
                      151 552 trajectories on a B200).  The result does not depend on it                 */
} aw_state;

/* Initial-condition family (P:85 whole region, P:87 patch, P:97 cloud; R6, R8, R9, R12, R17, R18). */
typedef struct {
  int32_t gx, gy;               /* the WHOLE ensemble: gx*gy trajectories, trajectory K = j*gx + i; the state
                                   holds the slice K in [k0, k0 + n), element k = K - k0 of its planes    */
  double lo_x, hi_x, lo_y, hi_y; /* action rectangle for shape GRID; samples are cell-centred:
                                    px = lo_x + (i + 1/2)(hi_x - lo_x)/gx, py likewise with j  */
  int32_t angle_mode;           /* 0: all angles 0;  1: angle_a = 2pi * u(seed, k, a), a=0,1,2 */
  int32_t shape;                /* AW_SHAPE_*: DISK  (px,py) = (cx,cy) + r sqrt(u3) (cos,sin)(2pi u4)
                                               GAUSS (px,py) = (cx,cy) + r sqrt(-2 ln(1-u3)) (cos,sin)(2pi u4)
                                               SPHERE (R28) direction uniform on the unit sphere:
                                                 cos(th) = 1 - 2 u3, phi = 2pi u4, |P| = sqrt(2(E - eps H_p(X)))
                                                 P = |P| (sin th cos phi, sin th sin phi, pz_sign cos th);
                                                 never off the shell; lo/hi/cx/cy/r unused
                                               RECT ("a small segment of the sphere"; R33) uniform random
                                                 points of the rectangle: px = lo_x + u3 (hi_x - lo_x),
                                                 py = lo_y + u4 (hi_y - lo_y)                     */
  double cx, cy, r;
  int32_t pz_sign;              /* +1 (default, upper hemisphere; R9) or -1                    */
  int32_t tangent_mode;         /* 0: one common seeded unit vector (R12); 1: per trajectory   */
  int64_t k0;                   /* first trajectory of the slice this state holds (0 for the whole ensemble).  Grid
                                   position and every random draw are functions of the GLOBAL index K, so a slice
                                   is bit-identical to the same rows of the whole (multi-GPU sharding, P:13, P:63;
                                   R30): rank r of a row-sharded job passes k0 = j0*gx, n = rows*gx          */
  int32_t resample;             /* shapes DISK, GAUSS, RECT: a draw (px, py, X) with 2(E - eps H_p(X)) < px^2 + py^2 has no
                                   real third action ("v_z from the fixed energy condition").  0: mask it (status
                                   0, R8).  m > 0: draw the trajectory again, up to m times — attempt a takes ALL its
                                   draws (angles, cloud point) from seed_a = seed + a*0xD1B54A32D192ED03 (mod 2^64) —
                                   until it is on the shell (rejection sampling: the accepted points are distributed
                                   like the unmasked points of the plain ensemble; R31).  Every trajectory is then
                                   live (up to probability P(off shell)^(m+1)), so no warp lane idles            */
  int32_t reserved_;
} aw_grid;

/* Bytes the caller must provide for each buffer.  *pitch_out = n rounded up to a multiple of 32.
 * Returns 6*pitch*8 (+ 6*pitch*8 if with_tangent) + 4*pitch*8 (+ 3*pitch*4 if with_wind) + n, i.e. the
 * total if all planes were packed back to back; the planes may equally be separate allocations. */
AW_API size_t aw_state_bytes(int64_t n, int with_tangent, int with_wind, int64_t *pitch_out);

/* Counter-based randomness (R11): mix64(seed, ctr): z = seed + ctr*0x9E3779B97F4A7C15 (mod 2^64);
 * z ^= z>>30; z *= 0xBF58476D1CE4E5B9; z ^= z>>27; z *= 0x94D049BB133111EB; z ^= z>>31.
 * u(seed, K, slot) = (mix64(seed, 16K + slot) >> 11) * 2^-53 in [0,1), K the global index.  Slots: 0-2 angles, 3-4 cloud,
 * 5-10 tangent normals (Box-Muller pairs (5,6), (7,8), (9,10) on (1 - u_a, u_b)).                 */

/* §8(a) a1 — initial conditions on the energy shell ("v_z from the energy
 * condition").  For every K = k0 + k, k in [0, n): (px,py) from the grid or cloud; angles per angle_mode;
 * R = 2(E - eps H_p(X)) - px^2 - py^2; R < 0 -> status 0 and all six state words NaN (R8);
 * else pz = pz_sign*sqrt(R), status 1.  acc = {0, 0, H(X,P), 0}; wind = 0; tangent = common unit
 * vector (computed on the host, see aw_common_tangent) or the per-trajectory one.  Sets s->E, eps,
 * Emax = E, t = 0, step = 0, ready = 1.  Errors: AW_EINVAL (null s/grid/planes, k0 < 0 or k0 + n > gx*gy, pitch < n or not a
 * multiple of 32, hi <= lo, r < 0, bad modes), AW_ERANGE (E - 2|eps| <= 0 or non-finite). */
AW_API int aw_init_shell(aw_state *s, const aw_grid *grid, double E, double eps, uint64_t seed);

/* §8(a) a2 + a3 + a4 — advance every live trajectory by `steps` steps of size dt.
 * One step = for s in 1..S { X += a_s P; P -= b_s grad H_p(X) } X += a_{S+1} P  with
 * a_s = c_s*dt, b_s = (eps*w_s)*dt (R2; constants from aw_stage_constants).  If s->w != NULL the
 * tangent vector goes through the exact derivative of the same map (R3).  Every `stride` steps the
 * fused checkpoint runs (R4): renormalise the tangent vector, logsum += ln|w|, fli = max(fli, logsum);
 * dH_max = max(dH_max, |H - H0|); wrap the angles to [-pi,pi] counting whole turns into wind (R7);
 * a non-finite state sets status 2 and freezes the trajectory; with s->survive == 1 a trajectory whose
 * (px, py) is outside the launch rectangle s->surv_* at a checkpoint gets status 3 (AW_ST_LEFT) and is
 * frozen at that checkpoint ("tracked only those trajectories which remained within the area during
 * the whole observation time"; R25) — it is then skipped by every later call, image and histogram.
 * n must equal s->n.  steps >= 0, stride > 0, steps % stride == 0; dt != 0 finite (dt < 0 integrates
 * backwards).  steps == 0 or n == 0 is a no-op.  AW_ERANGE if stride*|dt|*sqrt(2(E+2|eps|)) >= 1024
 * (the angle would leave the range the two-constant argument reduction handles exactly, R7).
 * AW_ESTATE if !s->ready or order not in {4, 6}.  Advances s->t and s->step.
 * Trigonometry: the kick needs sin/cos of x + y, x - y and 2z at every stage.  With s->trig == 0 the kernel carries
 * the three (sin, cos) pairs in registers and advances a pair through a drift by a rotation with the drift angle
 * d = A p (Taylor polynomials in p with the powers of A folded into the coefficients) whenever degree <= 5 keeps the
 * truncation below 2^-60; the degree of every drift and pair type is fixed at compile time from the level the host
 * picks (max_s |a_s| sqrt(2(Emax + 2|eps|)); aw_trig_level reports it) and the drift's ratio to the longest one.  A
 * pair every drift rotates is recomputed from the tracked angle with the device sincos at every checkpoint and at
 * least every 128 steps.  After a drift too long to rotate through, the kick evaluates the pair from the angle with
 * a table-driven sincos (512-entry table of the whole circle in shared memory + degree-2 residual rotation; no
 * quadrant logic); from level 5 on the kernels mix the two per drift and per pair, and at level 0 (drift angle
 * beyond 2 rad, or s->trig == 1) every stage uses the table.
 * The bound is max(s->E, s->Emax) and it is ENFORCED: every call first runs one elementwise kernel that
 * evaluates each live trajectory's H(X,P) and compares it with the largest energy the chosen level (and the angle
 * range of R7) supports; above it the trajectory gets AW_ST_RANGE and is not touched (P^2 <= 2(H + 2|eps|)
 * along the whole orbit, so the check before the first step covers every step).  The flag is a status like any other:
 * to integrate such a trajectory after all, set its status byte back to AW_ST_LIVE and raise the bound (aw_bound_energy
 * considers live trajectories only).  Call aw_bound_energy after uploading a state whose energy the struct does not
 * know.
 * The work is split into kernel launches of at most AW_MAX_STEPS_PER_LAUNCH steps (a multiple of
 * stride); the result does not depend on the split. */
#define AW_MAX_STEPS_PER_LAUNCH 20000
AW_API int aw_integrate(aw_state *s, int64_t n, int64_t steps, double dt, int64_t stride);

/* §8(f) 1-2 — snapshot of the state: qref <- q, windref <- wind, tref <- t (device-to-device copies on
 * s->stream).  It is the X(t) of the averaging window [t, t + Dt] of P:67 and the P(0) of the drift
 * detector dP(t) = |P(t) - P(0)| of P:37.  AW_ESTATE if s->qref == NULL, if wind and windref are not
 * both NULL or both non-NULL, or if the state is not ready. */
AW_API int aw_mark(aw_state *s);

/* §8(a) a5 — indicator image.  kind AW_IND_FLI: fli_max; AW_IND_FTLE: logsum / s->t; AW_IND_DH:
 * dH_max -> out_dev = n doubles (device), NaN where status != 1.  AW_IND_CLASS: out_dev = n bytes
 * (device), 1 if fli_max > thr else 0, 255 where status != 1 (R14; pass thr = log(t) + 3 for the
 * default).  AW_ESTATE if a tangent indicator is asked of a state without tangent planes, or FTLE
 * at t == 0.
 * §8(f): AW_IND_DP: |P - Pref| (three rounded squares summed left to right, IEEE sqrt).
 * AW_IND_VX / VY / VZ: component of the projected averaged velocity Vhat (see aw_density), NaN where
 * the trajectory is not live or |V| = 0.  These need s->qref (AW_ESTATE if NULL); VX..VZ also need
 * s->wind, s->windref and s->t > s->tref.
 * AW_IND_DHS: the signed energy error of the CURRENT state, H(X,P) - H0, by the routine the checkpoint uses
 * (BASELINE configs[2] "energy-drift statistics"; R29). */
AW_API int aw_indicator(const aw_state *s, int kind, double thr, void *out_dev);

/* Energy-drift statistics over the live trajectories (BASELINE configs[2]; R29; "no secular growth"):
 * out_dev[0] live count, [1] max dH_max, [2] mean dH_max, [3] rms dH_max, [4] mean and [5] rms of the signed
 * error H(X,P) - H0 of the current state, [6] index of the first trajectory attaining max dH_max (-1 if none),
 * [7] max |signed error|; means are NaN for an empty ensemble.  out_dev: 8 doubles (device); scratch_dev: device,
 * aw_energy_stats_scratch_bytes(n) bytes, 16-byte aligned.  Two kernels, deterministic (fixed reduction order,
 * no floating-point atomics): the same state gives the same bits on every run. */
AW_API size_t aw_energy_stats_scratch_bytes(int64_t n);
AW_API int aw_energy_stats(const aw_state *s, void *scratch_dev, double *out_dev);

/* aw_energy_stats for callers that cannot allocate device memory (under CUDA graph capture, serving loops, harnesses
 * that forbid cudaMalloc): same kernels, same result bit for bit, but the block partials live in a static device
 * array inside the library (AW_NOALLOC_MAX_N / 2048 partials of 64 bytes = 512 KiB, held by every GPU that loads the
 * library until the process exits), so the caller passes only the state and out_dev (8 doubles, device, 16-byte
 * aligned).  The call allocates and frees nothing: no cudaMalloc / cudaFree, no allocating library routine; the first
 * call on a device looks the array's address up once (cudaGetSymbolAddress, with the current device — the one that
 * holds s — current).  AW_ERANGE if s->n > AW_NOALLOC_MAX_N (use aw_energy_stats with caller scratch instead);
 * otherwise the errors of aw_energy_stats.  Nothing in the array has to be cleared between calls (partials [0, nb)
 * are overwritten before they are read) and a call never sees the previous call's contents.  All calls on one device
 * SHARE the array: calls whose kernels can overlap on the GPU (different streams, no ordering between them) race —
 * order them on one stream or with events.  Asynchronous on s->stream like aw_energy_stats. */
#define AW_NOALLOC_MAX_N 16777216 /* 2^24 trajectories */
AW_API int aw_energy_stats_noalloc(const aw_state *s, double *out_dev);

/* §8(a) a6 — visited-cell density over the first two actions (R19, R20).  For each live
 * trajectory ix = floor((px - lo) * (gx/(hi - lo))), iy likewise with gy; inside -> hist[iy*gx + ix]
 * += 1, else *dropped_dev += 1 (dropped_dev may be NULL; 8-byte aligned).  ADDS into hist_dev (device, gx*gy
 * uint32, 4-byte aligned; the caller zeroes it) so repeated calls give the time-accumulated density.
 * mode AW_DENS_ACTION (0): the point binned is the instantaneous (px, py) (BASELINE configs[4]).
 * modes 1-3, §8(f) 1 — the paper's own indicator (P:67, P:171 fn. 26; R26, R27): the point binned is
 * (Vhat_x, Vhat_y) of the averaged finite-time velocity over the window [tref, t] since aw_mark,
 *   dX_a = (double)(wind_a - windref_a) * 2pi_hi + (x_a - xref_a),   V_a = dX_a / (t - tref),
 *   |V| = sqrt((Vx Vx + Vy Vy) + Vz Vz),   Vhat_a = V_a * (sqrt(2E) / |V|)     (central projection on S),
 * every operation rounded separately in this order (no FMA), i.e. the sphere S seen along the third
 * axis: AW_DENS_VEL_UPPER counts the hemisphere Vhat_z >= 0, _LOWER Vhat_z < 0, _BOTH both (folded);
 * the other hemisphere, |V| = 0 or non-finite, and points outside [lo, hi)^2 go to *dropped_dev.
 * AW_ESTATE if s->qref, s->wind or s->windref is NULL (without turn counters a trajectory that completed a turn
 * inside the window would alias silently) or !(s->t > s->tref).  AW_EINVAL for misaligned hist_dev / dropped_dev. */
AW_API int aw_density(const aw_state *s, uint32_t *hist_dev, int32_t gx, int32_t gy, double lo, double hi,
               int mode, uint64_t *dropped_dev);

/* Largest energy among the live trajectories, from the data (SYNCHRONOUS: one reduction kernel, an 8-byte copy
 * and a stream synchronise): s->Emax <- max over live k of H(X_k, P_k) by the routine the checkpoint uses.  For
 * states the library did not initialise (uploaded planes, aw_map_host): afterwards aw_integrate picks the
 * trigonometry level from the data instead of trusting s->E.  scratch_dev: 8 bytes of device memory, 8-byte
 * aligned.  An ensemble without live trajectories leaves Emax unchanged.  Needs s->eps set and ready. */
AW_API int aw_bound_energy(aw_state *s, void *scratch_dev);

/* Host helpers (pure host arithmetic, no device needed) ------------------------------------------ */

/* Stage constants of the scheme (R2): fills a[0..S] and b[0..S-1], returns S (3 for order 4, 7 for
 * order 6) or AW_EINVAL.  Order-6 weights are obtained inside the library by Newton iteration on the
 * four order conditions in extended precision. */
AW_API int aw_stage_constants(int order, double dt, double eps, double *a_host, double *b_host);
/* Trigonometry level aw_integrate would use for this state and dt: the bracket of the largest drift angle
 * d = max_s |a_s| sqrt(2(max(E, Emax) + 2|eps|)): 1..9 <-> d <= 0.0104, 0.0147, 0.0354, 0.05, 0.1166, 0.2192, 0.357,
 * 0.54, 2; 0 = beyond (or s->trig == 1): table-driven sincos at every stage.  Levels 1-4 rotate every pair through
 * every drift; from level 5 on the long drifts go through the table; or a negative aw_status.  Pure host arithmetic. */
AW_API int aw_trig_level(const aw_state *s, double dt);
/* Threads per block aw_integrate launches for this state and dt: s->block if forced, else 128 when ceil(n/128) fills
 * every SM with its 4 resident blocks, else the smallest of 32, 64, 128 whose blocks are all resident at once (16 per
 * SM; 6 per SM for the trigonometry levels that keep the 32 KB sincos table in shared memory), so that a small
 * ensemble's warps spread over all SMs (queries the current device's SM count; 148 if there is none).  The result
 * of aw_integrate does not depend on it.  Negative aw_status as aw_trig_level. */
AW_API int aw_block_size(const aw_state *s, double dt);
/* Which ptxas schedule of the integrator kernel aw_integrate launches for this state and dt (aw_state.flavour): 1 = the
 * throughput flavour, 0 = the latency flavour; or a negative aw_status.  The kernel is integrate_kernel<S, TAN, LEVEL, SCHEDULE> with S = 3 / 7 stages. */
AW_API int aw_kernel_schedule(const aw_state *s, double dt);
/* The common tangent vector of tangent_mode 0: unit vector from u(seed, 2^63-1, 5..10) (R12). */
AW_API int aw_common_tangent(uint64_t seed, double *t6_host);

/* End-to-end call with HOST buffers (synchronous) ------------------------------------------------ *
 * Uploads a host-resident state into the caller-provided device planes of *s (q, w if non-NULL, acc,
 * wind if non-NULL, status; host layouts identical to the device ones), runs aw_integrate(steps, dt,
 * stride), aw_indicator(kind, thr) and aw_density(gx, gy, lo, hi), and downloads the image
 * (n doubles, or n bytes for CLASS) and the histogram (gx*gy uint32, ADDED into hist_host's content
 * is NOT done: the device histogram is zeroed first and hist_host is overwritten) and the final state
 * planes that are non-NULL in the out arguments.  ind_dev / hist_dev are device scratch of n*8 and
 * AW_HIST_SCRATCH_BYTES(gx, gy) = gx*gy*4 rounded up to a multiple of 8, + 8 bytes (histogram, then the 64-bit
 * dropped counter, 8-byte aligned whatever the parity of gx*gy).  Every argument is validated before the first
 * copy is enqueued; the trigonometry level is picked from the uploaded data (aw_bound_energy); on any failure
 * after work was enqueued the stream is synchronised before returning, so the host buffers are always free
 * again when the call returns.  Synchronises s->stream before returning. */
#define AW_HIST_SCRATCH_BYTES(gx, gy) ((((size_t)(gx) * (size_t)(gy) * 4 + 7) / 8) * 8 + 8)
typedef struct {
  const double *q, *w, *acc;  /* host, same pitch as s                                            */
  const int32_t *wind;        /* host or NULL                                                     */
  const uint8_t *status;      /* host                                                             */
} aw_host_in;
typedef struct {
  void *image;        /* host, n doubles (n bytes for CLASS) or NULL                              */
  uint32_t *hist;     /* host, gx*gy or NULL (then no density is computed)                        */
  uint64_t *dropped;  /* host, 1 or NULL                                                          */
  double *q;          /* host, 6*pitch final state or NULL                                        */
  double *acc;        /* host, 4*pitch final accumulators or NULL                                 */
  uint8_t *status;    /* host, n or NULL                                                          */
} aw_host_out;
AW_API int aw_map_host(aw_state *s, const aw_host_in *in, int64_t steps, double dt, int64_t stride, int kind,
                double thr, int32_t gx, int32_t gy, double lo, double hi, void *ind_dev,
                void *hist_dev, const aw_host_out *out);

/* The paper's own pipeline end to end with HOST buffers (synchronous): uploads the host-resident state as
 * aw_map_host does, takes the snapshot (aw_mark: the state is the X(t) of the window), runs aw_integrate(steps, dt,
 * stride) — the averaging window Dt = steps*|dt| — then aw_density(mode 1..3) of the projected averaged velocity into
 * the zeroed device histogram, and downloads it (gx*gy uint32) plus out->dropped / q / acc / status where non-NULL;
 * out->image is ignored.  hist_dev: device scratch of AW_HIST_SCRATCH_BYTES(gx, gy).  s must carry qref, wind and windref. */
AW_API int aw_velocity_map_host(aw_state *s, const aw_host_in *in, int64_t steps, double dt, int64_t stride, int mode,
                                int32_t gx, int32_t gy, double lo, double hi, void *hist_dev,
                                const aw_host_out *out);

#ifdef __cplusplus
}
#endif
#endif /* AW_H_ */
