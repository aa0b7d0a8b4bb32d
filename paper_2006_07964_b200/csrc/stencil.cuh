// Small device helpers shared by the kernels of csrc/ (sm_100a, fp64): the 6th-order central difference the paper names
// for metrics and viscous terms (coefficients 3/4, -3/20, 1/60) and the cp.async (LDGSTS) wrappers.
// Shares no code with oracle/.
#pragma once

// delta a = 3/4 (a_{+1} - a_{-1}) - 3/20 (a_{+2} - a_{-2}) + 1/60 (a_{+3} - a_{-3}),  unit spacing
__device__ __forceinline__ double d6c(double m3, double m2, double m1, double p1, double p2, double p3) {
  return (3.0 / 4.0) * (p1 - m1) - (3.0 / 20.0) * (p2 - m2) + (1.0 / 60.0) * (p3 - m3);
}

// 8-byte cp.async into shared memory (thread-private staging columns)
__device__ __forceinline__ void cp8(double* dst, const double* src) {
  const unsigned d = (unsigned)__cvta_generic_to_shared(dst);
  asm volatile("cp.async.ca.shared.global [%0], [%1], 8;" ::"r"(d), "l"(src) : "memory");
}
__device__ __forceinline__ void cp_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
template <int N>
__device__ __forceinline__ void cp_wait() { asm volatile("cp.async.wait_group %0;" ::"n"(N) : "memory"); }
