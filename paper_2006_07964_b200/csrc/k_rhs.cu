// S3 (viscous point fluxes, Eqs. 5, 6, 21) and the launch sequence of cfd_rhs.   sm_100a, fp64.
// P:L<n> = PAPER.md line; U<k> = DESIGN.md reading.  Shares no code with oracle/.
//
// cfd_rhs = [k_phi -> k_visc_flux] (Navier–Stokes only) -> k_sweep<xi> -> k_sweep<eta> -> k_sweep<zeta>.
// The viscous fluxes are stored once per point and direction (12 doubles) and differentiated inside the sweep
// of their direction (k_sweep.cu), so there is no separate divergence pass and r is written once per sweep.
#include "cfd_internal.cuh"
#include "fastmath.cuh"

int launch_sweeps(cfd_ctx* c, const BlockDev& B, const RkFuse* rk, int* rk_ctas);
__global__ void k_res_final(const double* __restrict__ partials, int n, double* __restrict__ res);

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
// One CTA = one run of T points along i (plus 3 on either side) at fixed (j, k).  SXI: the xi flux rows stay in
// shared memory and the CTA writes their 6th-order central xi-derivative S = d(Fv^xi)/d(xi) on interior
// points instead of the rows themselves (rows W[0..3]); the eta sweep adds S to r (the xi marching sweep then needs
// no viscous input).  !SXI: the xi rows are written as they are (sweep plans 1-3 differentiate them in the xi sweep).
template <bool SXI>
__global__ void __launch_bounds__(256) k_visc_flux(BlockDev B, ParamsDev P, const double* __restrict__ phi, double* __restrict__ W,
                                                   int T) {
  __shared__ double sW[4][256];
  const int i0 = blockIdx.x * T;
  const int t = threadIdx.x;           // point i = i0 - 3 + t,  t in [0, T + 6)
  const int i = i0 - 3 + t;
  const int j = blockIdx.y - 3, k = blockIdx.z - 3;
  const int iend = min(i0 + T, B.n[0]);  // SXI: this CTA's outputs are [i0, iend), read with a halo of 3
  const int oi = (i < 0 || i >= B.n[0]), oj = (j < 0 || j >= B.n[1]), ok = (k < 0 || k >= B.n[2]);
  // own: point this CTA writes point-wise results for;  halo: only its xi rows are needed (for the xi derivative)
  const bool own = SXI ? (i >= i0 && i < iend) : (t < T && i < B.n[0] + 3);
  const bool halo = SXI && !own && t < (iend - i0) + 6;
  const bool row_in = (oj + ok) == 0;
  const bool need_xi = row_in && (own || halo);
  const bool need_other = own && !oi;
  const bool work = (need_xi || need_other) && (oi + oj + ok) <= 1 && i >= -3 && i < B.n[0] + 3;
  const long long M = B.M;
  if (work) {
    const long long p = B.idx(i, j, k);
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
    double mu = P.mu, kap = P.kappa;
    if (P.suth > 0.0) {  // mu(T) by Sutherland's law (U11)
      const double f = sutherland_factor(phi[3 * M + p], P.suth);
      mu *= f; kap *= f;
    }
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
      const double w0 = a * txx + b * txy + c * txz;
      const double w1 = a * txy + b * tyy + c * tyz;
      const double w2 = a * txz + b * tyz + c * tzz;
      const double w3 = a * bx + b * by + c * bz;
      if (d == 0 && SXI) {
        sW[0][t] = w0; sW[1][t] = w1; sW[2][t] = w2; sW[3][t] = w3;
      } else if (own) {
        W[(d * 4 + 0) * M + p] = w0;
        W[(d * 4 + 1) * M + p] = w1;
        W[(d * 4 + 2) * M + p] = w2;
        W[(d * 4 + 3) * M + p] = w3;
      }
    }
  }
  if (SXI) {
    __syncthreads();
    if (own && row_in && !oi) {
      const long long p = B.idx(i, j, k);
#pragma unroll
      for (int m = 0; m < 4; ++m)
        W[(long long)m * M + p] = d6c(sW[m][t - 3], sW[m][t - 2], sW[m][t - 1], sW[m][t + 1], sW[m][t + 2], sW[m][t + 3]);
    }
  }
}

// launch geometry of k_visc_flux: runs of T points along i, T + 6 <= 256 threads, all runs equally long
static void visc_geometry(const BlockDev& B, bool sxi, int* T, dim3* grid, int* threads) {
  const int span = sxi ? B.n[0] : B.n[0] + 6;  // !SXI: the i-ghost points are "own" points of the first / last run
  const int nrun = (span + 249) / 250;
  *T = (span + nrun - 1) / nrun;
  *threads = ((*T + 6 + 31) / 32) * 32;
  *grid = dim3(nrun, B.n[1] + 6, B.n[2] + 6);
}

// cfd_rhs (fused_stage 0) or, with fused_stage 1..3 (default sweep plan only), the RHS with the RK stage fused into
// the last sweep (cfd_stage_fused): the new state lands in the r buffers and the caller exchanges the buffer roles.
int launch_rhs(cfd_ctx* c, int fused_stage, double dt) {
  RkFuse rk;
  rk.stage = fused_stage;
  rk.dt = dt;
  rk.a = fused_stage == 2 ? 3.0 / 4.0 : (fused_stage == 3 ? 1.0 / 3.0 : 0.0);
  rk.b = fused_stage == 2 ? 1.0 / 4.0 : (fused_stage == 3 ? 2.0 / 3.0 : 1.0);
  double* const partials = c->ws + ws_partials_offset_doubles(c);
  const long long cap = (long long)rk_max_partial_blocks() * (long long)c->blk.size();
  long long used = 0;
  // Blocks are independent until the ghost fill: with several blocks (and no per-kernel timing) each block's chain of
  // kernels goes to one of the side streams, forked from and joined back into the context's stream, so that small
  // blocks (C4: 8 x 96^3, about one wave of CTAs per kernel) fill the GPU together.  Every block has its own scratch.
  cudaStream_t const main_stream = c->stream;
  const bool fork = c->blk.size() > 1 && !c->prof_on && c->side[0] != nullptr;
  if (fork) {
    CUDA_TRY(c, cudaEventRecord(c->ev_fork, main_stream));
    for (int t = 0; t < cfd_ctx::NSIDE; ++t) CUDA_TRY(c, cudaStreamWaitEvent(c->side[t], c->ev_fork, 0));
  }
  int bi = 0;
  for (const BlockDev& B : c->blk) {
    if (fork) c->stream = c->side[bi++ % cfd_ctx::NSIDE];
    if (c->pd.viscous && c->sweep_plan == 0 && !c->visc_tiled) {
      ProfScope ps(c, PK_VISC_FLUX);
      launch_visc_march(c, B);
    } else if (c->pd.viscous) {
      double* phi = B.ws + 12 * B.M;
      { ProfScope ps(c, PK_VISC_PHI); k_phi<<<(unsigned)((B.M + 255) / 256), 256, 0, c->stream>>>(B, c->pd.gamma, phi); }
      const bool sxi = c->sweep_plan == 0;
      int T, threads;
      dim3 g1;
      visc_geometry(B, sxi, &T, &g1, &threads);
      {
        ProfScope ps(c, PK_VISC_FLUX);
        if (sxi) k_visc_flux<true><<<g1, threads, 0, c->stream>>>(B, c->pd, phi, B.ws, T);
        else k_visc_flux<false><<<g1, threads, 0, c->stream>>>(B, c->pd, phi, B.ws, T);
      }
      c->launches += 2;
    }
    rk.partials = partials + used * 5;
    rk.max_ctas = cap - used < rk_max_partial_blocks() ? cap - used : rk_max_partial_blocks();
    int ctas = 0;
    const int rc = launch_sweeps(c, B, fused_stage ? &rk : nullptr, &ctas);
    if (rc != 0) { c->stream = main_stream; return rc; }
    if (fused_stage == 1) used += ctas;
  }
  c->stream = main_stream;
  if (fork) {
    for (int t = 0; t < cfd_ctx::NSIDE; ++t) {
      CUDA_TRY(c, cudaEventRecord(c->ev_join[t], c->side[t]));
      CUDA_TRY(c, cudaStreamWaitEvent(main_stream, c->ev_join[t], 0));
    }
  }
  if (fused_stage == 1) {
    ProfScope ps(c, PK_RES);
    k_res_final<<<1, 160, 0, c->stream>>>(partials, (int)used, c->d_res);
    c->launches++;
  }
  CUDA_TRY(c, cudaGetLastError());
  return CFD_OK;
}
