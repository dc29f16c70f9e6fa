// aw_model.cuh — the Hamiltonian of the paper as ONE device routine (eq. 1, eq. 2), used by
// aw_init_shell for H0 and by the checkpoint for |H - H0| (R4: "the value the same routine returned").
#pragma once
#include "aw_trig.cuh"

namespace aw {

// H_p(X) = cos x cos y (1 + cos 2z) = 2 cos x cos y cos^2 z
__device__ __forceinline__ double hp_dev(double x, double y, double z) {
  double sx, cx, sy, cy, sz, cz;
  sincos(x, sx, cx);
  sincos(y, sy, cy);
  sincos(z, sz, cz);
  return (cx * cy) * (2.0 * (cz * cz));
}

// H(X,P) = P^2/2 + eps H_p(X)
__device__ __forceinline__ double hamiltonian_dev(double x, double y, double z, double px, double py,
                                                  double pz, double eps) {
  const double kin = 0.5 * fma(pz, pz, fma(py, py, px * px));
  return fma(eps, hp_dev(x, y, z), kin);
}

}  // namespace aw
