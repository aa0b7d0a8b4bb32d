// Branch-free fp64 reciprocal / reciprocal square root for the hot kernels (sm_100a).
// The FP64 pipe is the binding roofline of this path: an IEEE division costs ~10 pipe
// instructions plus a slow-path branch, MUFU.RCP64H + one cubic Newton step costs 3, MUFU.RSQ64H + one
// cubic step costs 5.  Both return the result to within ~1 ulp for normal, positive-range arguments
// (seed error e0 <= 2^-20 -> e0^3 <= 2^-60); arguments on this path (rho, c^2, |khat|^2, WENO
// denominators >= (4 eps)^8) are always normal.  tests/test_gpu_parity.py::test_fastmath_accuracy
// measures the error against correctly rounded results on the device.
#pragma once

__device__ __forceinline__ double frcp(double x) {
  double y;
  asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(x));
  const double e = fma(-x, y, 1.0);
  const double t = fma(e, e, e);
  return fma(y, t, y);
}

__device__ __forceinline__ double frsqrt(double x) {
  double y;
  asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(x));
  const double t = x * y;
  const double e = fma(-t, y, 1.0);
  const double p = fma(0.375, e, 0.5);
  return fma(y, p * e, y);
}

// Sutherland's law in the reference scales (U11): mu(T)/mu(1) = T^(3/2) (1 + S) / (T + S), S > 0.
__device__ __forceinline__ double sutherland_factor(double T, double S) {
  return (T * (T * frsqrt(T))) * ((1.0 + S) * frcp(T + S));
}
