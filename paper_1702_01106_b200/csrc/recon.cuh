// recon.cuh -- reconstruction operators R: generalised minmod on the 3-point stencil
// (L115, L651) and MP5 (Suresh & Huynh 1997; not in the paper, required by BASELINE.json -- reading C-6).
#pragma once

#include <math.h>

#include "fp64ops.cuh"

namespace grim {

// minmod functions as selects (no branches): the common sign's smallest magnitude, else zero
__device__ __forceinline__ double minmod2(double a, double b) {
  const double lo = fmin(a, b), hi = fmax(a, b);
  return (a > 0.0 && b > 0.0) ? lo : ((a < 0.0 && b < 0.0) ? hi : 0.0);
}

__device__ __forceinline__ double minmod3(double a, double b, double c) {
  const double lo = fmin(a, fmin(b, c)), hi = fmax(a, fmax(b, c));
  return (a > 0.0 && b > 0.0 && c > 0.0) ? lo : ((a < 0.0 && b < 0.0 && c < 0.0) ? hi : 0.0);
}

__device__ __forceinline__ double minmod4(double a, double b, double c, double d) {
  const double lo = fmin(fmin(a, b), fmin(c, d)), hi = fmax(fmax(a, b), fmax(c, d));
  return (a > 0.0 && b > 0.0 && c > 0.0 && d > 0.0) ? lo : ((a < 0.0 && b < 0.0 && c < 0.0 && d < 0.0) ? hi : 0.0);
}

// limited slope of the 3-point stencil: minmod(theta (v0 - vm), (vp - vm)/2, theta (vp - v0))  (L115)
__device__ __forceinline__ double limited_slope(double theta, double vm, double v0, double vp) {
  return minmod3(theta * (v0 - vm), 0.5 * (vp - vm), theta * (vp - v0));
}

// The monotonicity-preserving bounds of MP5, applied only where the unlimited value fails the acceptance test:
// out of line, so that the 2N inlined copies of mp5_face in the flux kernel stay short (the kernel is bound by
// instruction fetch otherwise) -- smooth data never comes here.
__device__ __noinline__ double mp5_limited(double vor, double vm2, double vm1, double v0, double vp1, double vp2) {
  const double alpha = 4.0;
  double dm1 = vm2 - 2.0 * vm1 + v0;
  double d0 = vm1 - 2.0 * v0 + vp1;
  double dp1 = v0 - 2.0 * vp1 + vp2;
  double dM4p = minmod4(4.0 * d0 - dp1, 4.0 * dp1 - d0, d0, dp1);
  double dM4m = minmod4(4.0 * dm1 - d0, 4.0 * d0 - dm1, dm1, d0);
  double vul = v0 + alpha * (v0 - vm1);
  double vav = 0.5 * (v0 + vp1);
  double vmd = vav - 0.5 * dM4p;
  double vlc = v0 + 0.5 * (v0 - vm1) + (4.0 / 3.0) * dM4m;
  double vmin = fmax(fmin(fmin(v0, vp1), vmd), fmin(fmin(v0, vul), vlc));
  double vmax = fmin(fmax(fmax(v0, vp1), vmd), fmax(fmax(v0, vul), vlc));
  return vor + minmod2(vmin - vor, vmax - vor);
}

// MP5 value at the i+1/2 face from v_{i-2..i+2}; alpha = 4, eps = 1e-10 (C-6)
template <class A>
__device__ __forceinline__ double mp5_face(A &ar, double vm2, double vm1, double v0, double vp1, double vp2) {
  const double alpha = 4.0, eps = 1e-10;
  double vor = div60(ar, 2.0 * vm2 - 13.0 * vm1 + 47.0 * v0 + 27.0 * vp1 - 3.0 * vp2);
  double vmp = v0 + minmod2(vp1 - v0, alpha * (v0 - vm1));
  if ((vor - v0) * (vor - vmp) <= eps) return vor;
  return mp5_limited(vor, vm2, vm1, v0, vp1, vp2);
}

// v[0..4] = P_{i-2..i+2}.  hi = P^-_{i+1/2} (left state of the upper face), lo = P^+_{i-1/2} (right state of
// the lower face) (L158-160)
template <int RECON, class A>
__device__ __forceinline__ void reconstruct(A &ar, double theta, double vm2, double vm1, double v0, double vp1, double vp2,
                                            double &hi, double &lo) {
  if constexpr (RECON == 1) {
    hi = mp5_face(ar, vm2, vm1, v0, vp1, vp2);
    lo = mp5_face(ar, vp2, vp1, v0, vm1, vm2);
  } else {
    double s = limited_slope(theta, vm1, v0, vp1);
    hi = v0 + 0.5 * s;
    lo = v0 - 0.5 * s;
  }
}

}  // namespace grim
