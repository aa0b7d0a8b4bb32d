// S3 (viscous point fluxes, Eqs. 5, 6, 21) and the launch sequence of cfd_rhs.   sm_100a, fp64.
// P:L<n> = PAPER.md line; U<k> = DESIGN.md reading.  Shares no code with oracle/.
//
// cfd_rhs = [k_phi -> k_visc_flux] (Navier–Stokes only) -> k_sweep<xi> -> k_sweep<eta> -> k_sweep<zeta>.
// The viscous fluxes are stored once per point and direction (12 doubles) and differentiated inside the sweep
// of their direction (k_sweep.cu), so there is no separate divergence pass and r is written once per sweep.
#include "cfd_internal.cuh"
#include "fastmath.cuh"

int launch_sweeps(cfd_ctx* c, const BlockDev& B);

// phi = (u, v, w, T = gamma p / rho) at every stored point, ghosts included (unfilled corner ghosts give
// values nobody reads).
__global__ void __launch_bounds__(256) k_phi(BlockDev B, double gamma, double* __restrict__ phi) {
  const long long M = B.M;
  const long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (t >= M) return;
  const double* __restrict__ q = B.q;
  const double rho = q[t], ir = frcp(rho);
  const double u = q[M + t] * ir, v = q[2 * M + t] * ir, w = q[3 * M + t] * ir;
  const double pr = (gamma - 1.0) * fma(-0.5 * rho, fma(u, u, fma(v, v, w * w)), q[4 * M + t]);
  phi[t] = u; phi[M + t] = v; phi[2 * M + t] = w; phi[3 * M + t] = (gamma * pr) * ir;
}

__device__ __forceinline__ double d6c(double m3, double m2, double m1, double p1, double p2, double p3) {
  return (3.0 / 4.0) * (p1 - m1) - (3.0 / 20.0) * (p2 - m2) + (1.0 / 60.0) * (p3 - m3);
}

// Point viscous fluxes at every point with at most one index out of range (by <= 3): gradients of phi by 6th-order
// central differences + chain rule (Eq. 21), tau and beta (Eq. 6), then the three directional fluxes (Eq. 5; rows
// 2..5, row 1 is identically zero) into W[d*4 + (m-1)][M].  Ghost points only get the flux of their own
// direction (the only one ever differentiated there).
__global__ void __launch_bounds__(128) k_visc_flux(BlockDev B, ParamsDev P, const double* __restrict__ phi, double* __restrict__ W) {
  const int e0 = B.n[0] + 6;
  const int i = blockIdx.x * blockDim.x + threadIdx.x - 3;
  const int j = blockIdx.y - 3, k = blockIdx.z - 3;
  if (i >= e0 - 3) return;
  const int oi = (i < 0 || i >= B.n[0]), oj = (j < 0 || j >= B.n[1]), ok = (k < 0 || k >= B.n[2]);
  if (oi + oj + ok > 1) return;
  const long long M = B.M, p = B.idx(i, j, k);
  double dphi[3][4];
#pragma unroll
  for (int d = 0; d < 3; ++d) {
    const long long st = B.s[d];
#pragma unroll
    for (int f = 0; f < 4; ++f) {
      const double* a = phi + f * M + p;
      dphi[d][f] = d6c(a[-3 * st], a[-2 * st], a[-st], a[st], a[2 * st], a[3 * st]);
    }
  }
  double kh[3][3];
#pragma unroll
  for (int d = 0; d < 3; ++d)
#pragma unroll
    for (int c = 0; c < 3; ++c) kh[d][c] = B.khat[(d * 3 + c) * M + p];
  const double J = B.jac[p];
  double g[3][4];
#pragma unroll
  for (int c = 0; c < 3; ++c)
#pragma unroll
    for (int f = 0; f < 4; ++f) g[c][f] = J * ((kh[0][c] * dphi[0][f] + kh[1][c] * dphi[1][f]) + kh[2][c] * dphi[2][f]);
  const double u = phi[p], v = phi[M + p], w = phi[2 * M + p];
  const double mu = P.mu, kap = P.kappa;
  const double div = g[0][0] + g[1][1] + g[2][2];
  const double lam = -(2.0 / 3.0) * mu;
  const double txx = lam * div + 2.0 * mu * g[0][0];
  const double tyy = lam * div + 2.0 * mu * g[1][1];
  const double tzz = lam * div + 2.0 * mu * g[2][2];
  const double txy = mu * (g[1][0] + g[0][1]);
  const double txz = mu * (g[2][0] + g[0][2]);
  const double tyz = mu * (g[2][1] + g[1][2]);
  const double bx = u * txx + v * txy + w * txz + kap * g[0][3];
  const double by = u * txy + v * tyy + w * tyz + kap * g[1][3];
  const double bz = u * txz + v * tyz + w * tzz + kap * g[2][3];
#pragma unroll
  for (int d = 0; d < 3; ++d) {
    if ((oi && d != 0) || (oj && d != 1) || (ok && d != 2)) continue;
    const double a = kh[d][0], b = kh[d][1], c = kh[d][2];
    W[(d * 4 + 0) * M + p] = a * txx + b * txy + c * txz;
    W[(d * 4 + 1) * M + p] = a * txy + b * tyy + c * tyz;
    W[(d * 4 + 2) * M + p] = a * txz + b * tyz + c * tzz;
    W[(d * 4 + 3) * M + p] = a * bx + b * by + c * bz;
  }
}

int launch_rhs(cfd_ctx* c) {
  if (c->prm.scheme != 0) { c->err = "cfd_rhs: scheme 1 (original AFWENO) is not built yet"; return CFD_E_ARG; }
  for (const BlockDev& B : c->blk) {
    if (c->pd.viscous) {
      double* phi = c->ws + 12 * c->max_M;
      { ProfScope ps(c, PK_VISC_PHI); k_phi<<<(unsigned)((B.M + 255) / 256), 256, 0, c->stream>>>(B, c->pd.gamma, phi); }
      dim3 g1((B.n[0] + 6 + 127) / 128, B.n[1] + 6, B.n[2] + 6);
      { ProfScope ps(c, PK_VISC_FLUX); k_visc_flux<<<g1, 128, 0, c->stream>>>(B, c->pd, phi, c->ws); }
      c->launches += 2;
    }
    launch_sweeps(c, B);
  }
  CUDA_TRY(c, cudaGetLastError());
  return CFD_OK;
}
