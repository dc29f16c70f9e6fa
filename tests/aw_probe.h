/* aw_probe.h — TEST AND MEASUREMENT SUPPORT, not part of the product ABI (include/aw.h).
 *
 * libaw_probe.so (tests/aw_probe.cu, built by tests/aw_probe.py) exposes device routines of the library to the
 * tests — the integrator's own sincos, the counter-based generator, the Hamiltonian routine the checkpoint uses —
 * by compiling the same device headers (paper_1107_4107_b200/csrc/aw_trig.cuh, aw_model.cuh, aw_internal.cuh)
 * into small elementwise kernels, plus two fp64 micro-benchmarks bench.py uses to print a measured DFMA peak
 * beside the derived one.  Every call is synchronous.  Return value: 0 ok, -1 bad argument, -2 CUDA error.
 */
#ifndef AW_PROBE_H_
#define AW_PROBE_H_
#include <stdint.h>
#ifdef __cplusplus
extern "C" {
#endif
#if defined(__GNUC__)
#define AWP_API __attribute__((visibility("default")))
#else
#define AWP_API
#endif

/* Device sincos used by the integrator (csrc/aw_trig.cuh, pin P14), on n device doubles. */
AWP_API int awp_sincos(const double *x_dev, int64_t n, double *sin_dev, double *cos_dev, void *stream);
/* Table-driven sincos of the step loop (csrc/aw_tsincos.cuh; DESIGN.md §6.1 (ii)), on n device doubles, |x| < 1024. */
AWP_API int awp_tsincos(const double *x_dev, int64_t n, double *sin_dev, double *cos_dev, void *stream);
/* u(seed, k0 + i, slot) for i in [0, n) written to out_dev (device); include/aw.h, R11. */
AWP_API int awp_uniform(uint64_t seed, uint64_t k0, int64_t n, uint32_t slot, double *out_dev, void *stream);
/* H(X,P) by the device routine the checkpoint uses, for n states in SoA planes q (6*pitch). */
AWP_API int awp_hamiltonian(const double *q_dev, int64_t n, int64_t pitch, double eps, double *out_dev, void *stream);
/* fp64 FMA peak: every thread runs `chains` (1, 2, 4, 8, 16) independent DFMA chains of `iters` links; grid =
 * blocks x threads.  Writes elapsed milliseconds (CUDA events) and the DFMA thread-instruction count to the host
 * outputs; flop/s = 2*dfma/ms*1e3.  sink_dev: >= 8 bytes device. */
AWP_API int awp_dfma_peak(int blocks, int threads, int chains, int64_t iters, double *sink_dev, double *ms_host,
                          double *dfma_host, void *stream);
/* fp64 issue rate by operand shape (the register-operand bandwidth behind DESIGN.md §6.1): 8 independent chains per
 * thread, 32 fp64 instructions per loop trip.  shape 0: fma(v, u0, w0) shared operands; 1: fma(v, u_c, w_c) three
 * distinct registers; 2: fma(v, u_c, immediate); 3: fma(v, v, w_c); 4: v * u_c (DMUL); 5: fma(u_c, w_c', v).
 * work_dev: >= 136 doubles. */
AWP_API int awp_dfma_shape(int blocks, int threads, int shape, int64_t iters, double *work_dev, double *ms_host,
                           double *inst_host, void *stream);
#ifdef __cplusplus
}
#endif
#endif /* AW_PROBE_H_ */
