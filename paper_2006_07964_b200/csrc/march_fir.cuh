// Eq. 19's central correction and the 6th-order central viscous derivative in flux form, evaluated as one transposed
// 6-tap FIR over the point fluxes (shared by the marching sweep kernels).  sm_100a, fp64.
//   D_j = Phi_{j+1/2} - Phi_{j-1/2},   Phi_{j+1/2} = F+_{j+1/2} + F-_{j+1/2} + sum_t a_t F_{j-2+t} - sum_t b_t Fv_{j-2+t}
// with a = (c3, c2+c3, c1+c2+c3, mirrored), c = (17/256, -13/320, 19/3840) (Eq. 19) and b likewise from
// (3/4, -3/20, 1/60).  Exact identity; only the summation order differs from Eq. 19 as printed.
#pragma once

// flux-form coefficients: a_t for Eq. 19's central part, b_t for the 6th-order central difference
#define A3 (19.0 / 3840.0)
#define A2 (-13.0 / 320.0 + 19.0 / 3840.0)
#define A1 (17.0 / 256.0 - 13.0 / 320.0 + 19.0 / 3840.0)
#define B3 (1.0 / 60.0)
#define B2 (-3.0 / 20.0 + 1.0 / 60.0)
#define B1 (3.0 / 4.0 - 3.0 / 20.0 + 1.0 / 60.0)

// one transposed-FIR update with the newest point flux x (and viscous xv); returns the filter output
__device__ __forceinline__ double fir_push(double acc[5], double x) {
  const double out = fma(A3, x, acc[0]);
  acc[0] = fma(A2, x, acc[1]);
  acc[1] = fma(A1, x, acc[2]);
  acc[2] = fma(A1, x, acc[3]);
  acc[3] = fma(A2, x, acc[4]);
  acc[4] = A3 * x;
  return out;
}
__device__ __forceinline__ double fir_push2(double acc[5], double x, double xv) {
  const double out = fma(-B3, xv, fma(A3, x, acc[0]));
  acc[0] = fma(-B2, xv, fma(A2, x, acc[1]));
  acc[1] = fma(-B1, xv, fma(A1, x, acc[2]));
  acc[2] = fma(-B1, xv, fma(A1, x, acc[3]));
  acc[3] = fma(-B2, xv, fma(A2, x, acc[4]));
  acc[4] = fma(-B3, xv, A3 * x);
  return out;
}

