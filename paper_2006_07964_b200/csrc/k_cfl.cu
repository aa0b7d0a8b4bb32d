// On-device CFL time step ("time step dt" stored per point, "reduced-dimensional operation", Fig. 2
// timestep_gpu; reading U16): per interior point the spectral-radius sum  s = sum_d ( |k_d . u| + c |k_d| ),  k_d = J khat^d,
// reduced with MAX over all interior points of all blocks (order-independent: deterministic), dt = CFL / max s.
// Optionally the local time step CFL / s is written per point.  sm_100a, fp64.  Shares no code with oracle/.
// One pass over Q (5), khat (9), J (1): 120 bytes per point, bandwidth-bound; plain IEEE division and square root (not on
// the FP64-bound path, and the result feeds every later step: correctly rounded operations keep it within an ulp or two
// of the oracle's).
#include "cfd_internal.cuh"

namespace {

constexpr int CT = 256;

// max that KEEPS a NaN (fmax drops it): a point with rho <= 0 or p < 0 gives s = NaN (or Inf), and the reduction must carry
// that to the host so that cfd_cfl_dt can refuse the state instead of returning a dt from the remaining points.
__device__ __forceinline__ double max_nan(double a, double b) { return (b > a || b != b) ? b : a; }

__global__ void __launch_bounds__(CT) k_cfl(BlockDev B, double gamma, double cfl, double* __restrict__ partials,
                                            double* __restrict__ dt_local) {
  const int ni = B.n[0], nj = B.n[1];
  const long long N = (long long)ni * nj * B.n[2];
  const long long M = B.M;
  double mx = 0.0;
  for (long long t = (long long)blockIdx.x * CT + threadIdx.x; t < N; t += (long long)gridDim.x * CT) {
    const int i = (int)(t % ni);
    const long long u_ = t / ni;
    const int j = (int)(u_ % nj);
    const int k = (int)(u_ / nj);
    const long long p = B.idx(i, j, k);
    const double rho = B.q[p];
    const double u = B.q[M + p] / rho, v = B.q[2 * M + p] / rho, w = B.q[3 * M + p] / rho;
    const double pr = (gamma - 1.0) * (B.q[4 * M + p] - 0.5 * rho * (u * u + v * v + w * w));
    const double c = sqrt(gamma * pr / rho);
    const double J = B.jac[p];
    double s = 0.0;
#pragma unroll
    for (int d = 0; d < 3; ++d) {
      const double kx = J * B.khat[(d * 3 + 0) * M + p], ky = J * B.khat[(d * 3 + 1) * M + p], kz = J * B.khat[(d * 3 + 2) * M + p];
      s += fabs(kx * u + ky * v + kz * w) + c * sqrt(kx * kx + ky * ky + kz * kz);
    }
    if (!(rho > 0.0) || !(pr >= 0.0)) s = __longlong_as_double(0x7ff8000000000000LL);  // rho <= 0 with p < 0 would give a real c
    if (dt_local) dt_local[p] = cfl / s;
    mx = max_nan(mx, s);
  }
  __shared__ double sm[CT / 32];
  for (int o = 16; o > 0; o >>= 1) mx = max_nan(mx, __shfl_down_sync(0xffffffffu, mx, o));
  if ((threadIdx.x & 31) == 0) sm[threadIdx.x >> 5] = mx;
  __syncthreads();
  if (threadIdx.x == 0) {
    double v = sm[0];
    for (int w = 1; w < CT / 32; ++w) v = max_nan(v, sm[w]);
    partials[blockIdx.x] = v;
  }
}

__global__ void k_cfl_final(const double* __restrict__ partials, int n, double* __restrict__ out) {
  double v = 0.0;
  for (int t = threadIdx.x; t < n; t += 32) v = max_nan(v, partials[t]);
  for (int o = 16; o > 0; o >>= 1) v = max_nan(v, __shfl_down_sync(0xffffffffu, v, o));
  if (threadIdx.x == 0) *out = v;
}

}  // namespace

// Enqueues the reduction; the maximum of s lands in c->d_res[5].  dt_local: per-block device arrays [M] or null.
int launch_cfl(cfd_ctx* c, double cfl, double* const* dt_local) {
  double* partials = c->ws + ws_partials_offset_doubles(c);
  int used = 0;
  const int cap = rk_max_partial_blocks();
  for (size_t b = 0; b < c->blk.size(); ++b) {
    if (!c->is_local(b)) continue;
    const BlockDev& B = c->blk[b];
    const long long N = (long long)B.n[0] * B.n[1] * B.n[2];
    long long g = (N + CT - 1) / CT;
    if (g > 148 * 8) g = 148 * 8;  // grid-stride: 8 CTAs per SM
    if (g > cap) g = cap;
    ProfScope ps(c, PK_OTHER);
    k_cfl<<<(unsigned)g, CT, 0, c->stream>>>(B, c->pd.gamma, cfl, partials + used, dt_local ? dt_local[b] : nullptr);
    used += (int)g;
    c->launches++;
  }
  {
    ProfScope ps(c, PK_OTHER);
    k_cfl_final<<<1, 32, 0, c->stream>>>(partials, used, c->d_res + 5);
    c->launches++;
  }
  CUDA_TRY(c, cudaGetLastError());
  return CFD_OK;
}
