// S2 (inviscid sweeps: modified AFWENO + Steger–Warming + Eq. 19) and S3 (viscous terms) for sm_100a.
// fp64 throughout; no tensor cores (this is stencil + per-point algebra, not a contraction).
// P:L<n> = PAPER.md line; U<k> = DESIGN.md reading.  Shares no code with oracle/.
//
// Algebra notes (what differs from a literal transcription; all exact identities):
//  * L_i Q_s is evaluated without forming L: with dm = m_s - rho_s u_i, E = q2/2 rho_s - u_i.m_s + e_s,
//    A = rho_s - (g-1)/c^2 E:  V_{1..3} = n A - n x dm,  V_{4,5} = ((g-1) E +- c n.dm) / (2 c^2)      (U4)
//  * R_i v likewise: a = n.v_{123}, s = v4+v5, t = c (v4-v5), w = n x v_{123}:
//    U = (a+s, u (a+s) + w + n t, q2/2 a + u.w + H s + theta t)
//  * WENO weights with a common denominator: alpha_k = 1/(eps+beta_k)^2 is replaced by the product of the
//    other two (eps+beta)^2, and both normalisations share one reciprocal (Eq. 15 up to rounding).
#include "cfd_internal.cuh"

__device__ __forceinline__ double rcp(double x) { return __drcp_rn(x); }

__device__ __forceinline__ double khalf(double m2, double m1, double z0, double p1, double p2, double p3) {
  // U5: symmetric 6-point Lagrange; explicit intrinsics so that both users of one interface get the same bits
  const double a = __dadd_rn(z0, p1), b = __dadd_rn(m1, p2), c = __dadd_rn(m2, p3);
  return __dmul_rn(__fma_rn(150.0, a, __fma_rn(-25.0, b, __dmul_rn(3.0, c))), 1.0 / 256.0);
}

// Eq. 17 (Jiang–Shu form) + Eq. 14 interpolants paired by stencil (U1) + Eq. 15/16 weights;
// vL = state at i+1/2 from the left-biased stencil, vR = state at i-1/2 (same beta).
__device__ __forceinline__ void weno5_lr(double a, double b, double c, double d, double e, double eps, double& vL, double& vR) {
  const double t1 = a - 2.0 * b + c, t2 = a - 4.0 * b + 3.0 * c;
  const double t3 = b - 2.0 * c + d, t4 = b - d;
  const double t5 = c - 2.0 * d + e, t6 = 3.0 * c - 4.0 * d + e;
  const double dA = eps + ((13.0 / 12.0) * t1 * t1 + 0.25 * t2 * t2);
  const double dB = eps + ((13.0 / 12.0) * t3 * t3 + 0.25 * t4 * t4);
  const double dC = eps + ((13.0 / 12.0) * t5 * t5 + 0.25 * t6 * t6);
  const double pA = dB * dC, pB = dA * dC, pC = dA * dB;
  const double sA = pA * pA, sB = 10.0 * (pB * pB), sC = pC * pC;  // 16 * gamma_k * alpha_k * (dA dB dC)^2
  const double qLA = 0.375 * a - 1.25 * b + 1.875 * c;
  const double qLB = -0.125 * b + 0.75 * c + 0.375 * d;
  const double qLC = 0.375 * c + 0.75 * d - 0.125 * e;
  const double qRA = -0.125 * a + 0.75 * b + 0.375 * c;
  const double qRB = 0.375 * b + 0.75 * c - 0.125 * d;
  const double qRC = 1.875 * c - 1.25 * d + 0.375 * e;
  const double denL = sA + sB + 5.0 * sC;
  const double denR = 5.0 * sA + sB + sC;
  const double numL = sA * qLA + sB * qLB + 5.0 * sC * qLC;
  const double numR = 5.0 * sA * qRA + sB * qRB + sC * qRC;
  const double inv = rcp(denL * denR);
  vL = numL * denR * inv;
  vR = numR * denL * inv;
}

// Steger–Warming split flux (U3), SGN = +1 / -1.
template <int SGN>
__device__ __forceinline__ void sw_flux(const double U[5], double kx, double ky, double kz, double gamma, double F[5]) {
  const double g1 = gamma - 1.0;
  const double ir = rcp(U[0]);
  const double u = U[1] * ir, v = U[2] * ir, w = U[3] * ir;
  const double q2 = u * u + v * v + w * w;
  const double p = g1 * (U[4] - 0.5 * U[0] * q2);
  const double c2 = gamma * p * ir;
  const double c = sqrt(c2);
  const double kn = sqrt(kx * kx + ky * ky + kz * kz);
  const double th = kx * u + ky * v + kz * w;
  double l1 = th, l4 = th + c * kn, l5 = th - c * kn;
  if (SGN > 0) { l1 = 0.5 * (l1 + fabs(l1)); l4 = 0.5 * (l4 + fabs(l4)); l5 = 0.5 * (l5 + fabs(l5)); }
  else { l1 = 0.5 * (l1 - fabs(l1)); l4 = 0.5 * (l4 - fabs(l4)); l5 = 0.5 * (l5 - fabs(l5)); }
  const double a1 = 2.0 * g1 * l1, s45 = l4 + l5, d45 = l4 - l5;
  const double f = U[0] * (0.5 / gamma);
  const double cn = c * rcp(kn) * d45;
  const double A0 = a1 + s45;
  F[0] = f * A0;
  F[1] = f * (A0 * u + cn * kx);
  F[2] = f * (A0 * v + cn * ky);
  F[3] = f * (A0 * w + cn * kz);
  F[4] = f * (0.5 * a1 * q2 + 0.5 * s45 * (q2 + c2) + cn * th + ((3.0 - gamma) / (2.0 * g1)) * s45 * c2);
}

// Eq. 4
__device__ __forceinline__ void point_flux(const double Q[5], double kx, double ky, double kz, double gamma, double F[5]) {
  const double ir = rcp(Q[0]);
  const double u = Q[1] * ir, v = Q[2] * ir, w = Q[3] * ir;
  const double p = (gamma - 1.0) * (Q[4] - 0.5 * Q[0] * (u * u + v * v + w * w));
  const double th = kx * u + ky * v + kz * w;
  F[0] = Q[0] * th;
  F[1] = Q[1] * th + kx * p;
  F[2] = Q[2] * th + ky * p;
  F[3] = Q[3] * th + kz * p;
  F[4] = (Q[4] + p) * th;
}

// Steps 1–7 of O2 at one point: Qs[s][m] = Q_{i-2+s}, ks[s][c] = khat^d_{i-3+s} (s = 0..6).
// Fp = F+ at i+1/2, Fm = F- at i-1/2.
__device__ __forceinline__ void afweno_point(const double Qs[5][5], const double ks[7][3], double gamma, double eps,
                                             double Fp[5], double Fm[5]) {
  const double g1 = gamma - 1.0;
  const double rho = Qs[2][0], e = Qs[2][4];
  const double ir = rcp(rho);
  const double u = Qs[2][1] * ir, v = Qs[2][2] * ir, w = Qs[2][3] * ir;
  const double q2 = u * u + v * v + w * w, hq = 0.5 * q2;
  const double p = g1 * (e - rho * hq);
  const double c2 = gamma * p * ir;
  const double c = sqrt(c2);
  const double rc2 = rcp(c2);
  const double H = (e + p) * ir;
  const double kx = ks[3][0], ky = ks[3][1], kz = ks[3][2];
  const double ikn = rcp(sqrt(kx * kx + ky * ky + kz * kz));
  const double nx = kx * ikn, ny = ky * ikn, nz = kz * ikn;
  const double th = nx * u + ny * v + nz * w;
  const double b1 = g1 * rc2, h = 0.5 * rc2;
  double V[5][5];  // [field][stencil]
#pragma unroll
  for (int s = 0; s < 5; ++s) {
    const double rs = Qs[s][0];
    const double dx = Qs[s][1] - rs * u, dy = Qs[s][2] - rs * v, dz = Qs[s][3] - rs * w;
    const double E = hq * rs - (u * Qs[s][1] + v * Qs[s][2] + w * Qs[s][3]) + Qs[s][4];
    const double A = rs - b1 * E;
    const double nd = nx * dx + ny * dy + nz * dz;
    V[0][s] = nx * A - (ny * dz - nz * dy);
    V[1][s] = ny * A - (nz * dx - nx * dz);
    V[2][s] = nz * A - (nx * dy - ny * dx);
    V[3][s] = h * (g1 * E + c * nd);
    V[4][s] = h * (g1 * E - c * nd);
  }
  double vL[5], vR[5];
#pragma unroll
  for (int f = 0; f < 5; ++f) weno5_lr(V[f][0], V[f][1], V[f][2], V[f][3], V[f][4], eps, vL[f], vR[f]);
  double UL[5], UR[5];
  {
    const double a = nx * vL[0] + ny * vL[1] + nz * vL[2], s = vL[3] + vL[4], t = c * (vL[3] - vL[4]);
    const double wx = ny * vL[2] - nz * vL[1], wy = nz * vL[0] - nx * vL[2], wz = nx * vL[1] - ny * vL[0];
    UL[0] = a + s;
    UL[1] = u * UL[0] + wx + nx * t;
    UL[2] = v * UL[0] + wy + ny * t;
    UL[3] = w * UL[0] + wz + nz * t;
    UL[4] = hq * a + (u * wx + v * wy + w * wz) + H * s + th * t;
  }
  {
    const double a = nx * vR[0] + ny * vR[1] + nz * vR[2], s = vR[3] + vR[4], t = c * (vR[3] - vR[4]);
    const double wx = ny * vR[2] - nz * vR[1], wy = nz * vR[0] - nx * vR[2], wz = nx * vR[1] - ny * vR[0];
    UR[0] = a + s;
    UR[1] = u * UR[0] + wx + nx * t;
    UR[2] = v * UR[0] + wy + ny * t;
    UR[3] = w * UR[0] + wz + nz * t;
    UR[4] = hq * a + (u * wx + v * wy + w * wz) + H * s + th * t;
  }
  // half-point metrics: k_{i+1/2} from ks[1..6], k_{i-1/2} from ks[0..5]
  const double kpx = khalf(ks[1][0], ks[2][0], ks[3][0], ks[4][0], ks[5][0], ks[6][0]);
  const double kpy = khalf(ks[1][1], ks[2][1], ks[3][1], ks[4][1], ks[5][1], ks[6][1]);
  const double kpz = khalf(ks[1][2], ks[2][2], ks[3][2], ks[4][2], ks[5][2], ks[6][2]);
  const double kmx = khalf(ks[0][0], ks[1][0], ks[2][0], ks[3][0], ks[4][0], ks[5][0]);
  const double kmy = khalf(ks[0][1], ks[1][1], ks[2][1], ks[3][1], ks[4][1], ks[5][1]);
  const double kmz = khalf(ks[0][2], ks[1][2], ks[2][2], ks[3][2], ks[4][2], ks[5][2]);
  sw_flux<+1>(UL, kpx, kpy, kpz, gamma, Fp);
  sw_flux<-1>(UR, kmx, kmy, kmz, gamma, Fm);
}

// -------------------------------------------------------------------------------------------------
// Inviscid sweep along DIR.  Tile: TS positions along the sweep (TS-2 outputs + one extra WENO point at
// each end) x NL lines.  DIR 0: 64 x 4 (sweep = i, contiguous);  DIR 1, 2: 8 x 32 (i stays the
// coalesced thread dimension).  MODE 0: r = D; 1: r += D; 2: r = -J (r + D) [Euler]; 3: r = r + D.
// -------------------------------------------------------------------------------------------------
template <int DIR>
struct TileCfg {
  static constexpr int TS = DIR == 0 ? 64 : 8;
  static constexpr int NL = DIR == 0 ? 4 : 32;
};

template <int DIR>
__global__ void __launch_bounds__(256) k_inviscid(BlockDev B, ParamsDev P, int mode) {
  constexpr int TS = TileCfg<DIR>::TS, NL = TileCfg<DIR>::NL, T = TS - 2;
  __shared__ double sFp[5][TS * NL], sFm[5][TS * NL], sFt[5][(TS + 4) * NL];
  const int sp = DIR == 0 ? threadIdx.x : threadIdx.y;
  const int ln = DIR == 0 ? threadIdx.y : threadIdx.x;
  int i, j, k, s0;
  if (DIR == 0) { s0 = blockIdx.x * T; i = s0 - 1 + sp; j = blockIdx.y * NL + ln; k = blockIdx.z; }
  else if (DIR == 1) { s0 = blockIdx.y * T; i = blockIdx.x * NL + ln; j = s0 - 1 + sp; k = blockIdx.z; }
  else { s0 = blockIdx.z * T; i = blockIdx.x * NL + ln; j = blockIdx.y; k = s0 - 1 + sp; }
  const int n = B.n[DIR];
  const int pos = s0 - 1 + sp;  // position along the sweep
  const bool lane_ok = DIR == 0 ? (j < B.n[1]) : (i < B.n[0]);
  const bool active = lane_ok && pos <= n;
  const long long M = B.M, sd = B.s[DIR];
  const long long pidx = B.idx(i, j, k);
  const double* __restrict__ q = B.q;
  const double* __restrict__ kh = B.khat + (long long)(DIR * 3) * M;
  auto SIDX = [&](int spx) { return DIR == 0 ? (ln * TS + spx) : (spx * NL + ln); };
  auto TIDX = [&](int slot) { return DIR == 0 ? (ln * (TS + 4) + slot) : (slot * NL + ln); };
  if (active) {
    double Qs[5][5], ks[7][3];
#pragma unroll
    for (int s = 0; s < 5; ++s)
#pragma unroll
      for (int m = 0; m < 5; ++m) Qs[s][m] = q[m * M + pidx + (s - 2) * sd];
#pragma unroll
    for (int s = 0; s < 7; ++s)
#pragma unroll
      for (int c = 0; c < 3; ++c) ks[s][c] = kh[c * M + pidx + (s - 3) * sd];
    double Fp[5], Fm[5], Ft[5];
    afweno_point(Qs, ks, P.gamma, P.eps, Fp, Fm);
    point_flux(Qs[2], ks[3][0], ks[3][1], ks[3][2], P.gamma, Ft);
#pragma unroll
    for (int m = 0; m < 5; ++m) {
      sFp[m][SIDX(sp)] = Fp[m];
      sFm[m][SIDX(sp)] = Fm[m];
      sFt[m][TIDX(sp + 2)] = Ft[m];
    }
    // the four extra point fluxes of the tile: pos-2 (first two positions), pos+2 (last two valid positions)
    if (sp < 2) {
      point_flux(Qs[0], ks[1][0], ks[1][1], ks[1][2], P.gamma, Ft);
#pragma unroll
      for (int m = 0; m < 5; ++m) sFt[m][TIDX(sp)] = Ft[m];
    }
    if (sp >= TS - 2 || pos >= n - 1) {
      point_flux(Qs[4], ks[5][0], ks[5][1], ks[5][2], P.gamma, Ft);
#pragma unroll
      for (int m = 0; m < 5; ++m) sFt[m][TIDX(sp + 4)] = Ft[m];
    }
  }
  __syncthreads();
  if (active && sp >= 1 && sp <= TS - 2 && pos < n) {
    const double jac = B.jac[pidx];
#pragma unroll
    for (int m = 0; m < 5; ++m) {
      const double fph = sFp[m][SIDX(sp)] + sFm[m][SIDX(sp + 1)];
      const double fmh = sFp[m][SIDX(sp - 1)] + sFm[m][SIDX(sp)];
      const double D = (fph - fmh) + (17.0 / 256.0) * (sFt[m][TIDX(sp + 3)] - sFt[m][TIDX(sp + 1)]) -
                       (13.0 / 320.0) * (sFt[m][TIDX(sp + 4)] - sFt[m][TIDX(sp)]) +
                       (19.0 / 3840.0) * (sFt[m][TIDX(sp + 5)] - sFt[m][TIDX(sp - 1)]);
      double* r = B.r + m * M + pidx;
      if (mode == 0) *r = D;
      else if (mode == 1 || mode == 3) *r = *r + D;
      else *r = jac * (0.0 - (*r + D));
    }
  }
}

// -------------------------------------------------------------------------------------------------
// S3 pass A: point viscous fluxes (Eqs. 5, 6, 21) at every point with at most one index out of range
// (by <= 3): gradients of (u,v,w,T) by 6th-order central differences + chain rule, then the three
// directional fluxes (rows 2..5; row 1 is identically zero) into the workspace W[d*4 + (m-1)][M].
// Ghost points only get the flux of their own direction (the only one ever differentiated there).
// -------------------------------------------------------------------------------------------------
__device__ __forceinline__ void phi_of(const double* __restrict__ q, long long M, long long p, double gamma, double ph[4]) {
  const double rho = q[p], ir = rcp(rho);
  const double u = q[M + p] * ir, v = q[2 * M + p] * ir, w = q[3 * M + p] * ir;
  const double pr = (gamma - 1.0) * (q[4 * M + p] - 0.5 * rho * (u * u + v * v + w * w));
  ph[0] = u; ph[1] = v; ph[2] = w; ph[3] = gamma * pr * ir;
}

__device__ __forceinline__ double d6c(double m3, double m2, double m1, double p1, double p2, double p3) {
  return (3.0 / 4.0) * (p1 - m1) - (3.0 / 20.0) * (p2 - m2) + (1.0 / 60.0) * (p3 - m3);
}

__global__ void __launch_bounds__(128) k_visc_flux(BlockDev B, ParamsDev P, double* __restrict__ W) {
  const int e0 = B.n[0] + 6;
  const int i = blockIdx.x * blockDim.x + threadIdx.x - 3;
  const int j = blockIdx.y - 3, k = blockIdx.z - 3;
  if (i >= e0 - 3) return;
  const int oi = (i < 0 || i >= B.n[0]), oj = (j < 0 || j >= B.n[1]), ok = (k < 0 || k >= B.n[2]);
  if (oi + oj + ok > 1) return;
  const long long M = B.M, p = B.idx(i, j, k);
  const double* __restrict__ q = B.q;
  double dphi[3][4];
#pragma unroll
  for (int d = 0; d < 3; ++d) {
    const long long st = B.s[d];
    double a[7][4];
#pragma unroll
    for (int s = 0; s < 7; ++s)
      if (s != 3) phi_of(q, M, p + (s - 3) * st, P.gamma, a[s]);
#pragma unroll
    for (int f = 0; f < 4; ++f) dphi[d][f] = d6c(a[0][f], a[1][f], a[2][f], a[4][f], a[5][f], a[6][f]);
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
  double ph[4];
  phi_of(q, M, p, P.gamma, ph);
  const double mu = P.mu, kap = P.kappa;
  const double div = g[0][0] + g[1][1] + g[2][2];
  const double lam = -(2.0 / 3.0) * mu;
  const double txx = lam * div + 2.0 * mu * g[0][0];
  const double tyy = lam * div + 2.0 * mu * g[1][1];
  const double tzz = lam * div + 2.0 * mu * g[2][2];
  const double txy = mu * (g[1][0] + g[0][1]);
  const double txz = mu * (g[2][0] + g[0][2]);
  const double tyz = mu * (g[2][1] + g[1][2]);
  const double bx = ph[0] * txx + ph[1] * txy + ph[2] * txz + kap * g[0][3];
  const double by = ph[0] * txy + ph[1] * tyy + ph[2] * tyz + kap * g[1][3];
  const double bz = ph[0] * txz + ph[1] * tyz + ph[2] * tzz + kap * g[2][3];
#pragma unroll
  for (int d = 0; d < 3; ++d) {
    // ghost points: only the flux of the out-of-range direction is needed
    if ((oi && d != 0) || (oj && d != 1) || (ok && d != 2)) continue;
    const double a = kh[d][0], b = kh[d][1], c = kh[d][2];
    W[(d * 4 + 0) * M + p] = a * txx + b * txy + c * txz;
    W[(d * 4 + 1) * M + p] = a * txy + b * tyy + c * tyz;
    W[(d * 4 + 2) * M + p] = a * txz + b * tyz + c * tzz;
    W[(d * 4 + 3) * M + p] = a * bx + b * by + c * bz;
  }
}

// S3 pass B: r := J [ (V^xi + V^eta + V^zeta) - r ] with V^d = 6th-order central derivative of the
// stored point fluxes (U18 accumulation order); row 1 has no viscous flux.
__global__ void __launch_bounds__(256) k_visc_div(BlockDev B, const double* __restrict__ W) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  const int j = blockIdx.y, k = blockIdx.z;
  if (i >= B.n[0]) return;
  const long long M = B.M, p = B.idx(i, j, k);
  const double J = B.jac[p];
  B.r[p] = J * (0.0 - B.r[p]);
#pragma unroll
  for (int m = 1; m < 5; ++m) {
    double V[3];
#pragma unroll
    for (int d = 0; d < 3; ++d) {
      const double* f = W + (d * 4 + (m - 1)) * M + p;
      const long long st = B.s[d];
      V[d] = d6c(f[-3 * st], f[-2 * st], f[-st], f[st], f[2 * st], f[3 * st]);
    }
    double* r = B.r + m * M + p;
    *r = J * (((V[0] + V[1]) + V[2]) - *r);
  }
}

int launch_rhs(cfd_ctx* c) {
  if (c->prm.scheme != 0) { c->err = "cfd_rhs: scheme 1 (original AFWENO) is not built yet"; return CFD_E_ARG; }
  for (const BlockDev& B : c->blk) {
    const int visc = c->pd.viscous;
    {
      constexpr int T = TileCfg<0>::TS - 2, NL = TileCfg<0>::NL;
      dim3 grid((B.n[0] + T - 1) / T, (B.n[1] + NL - 1) / NL, B.n[2]);
      ProfScope ps(c, PK_INV_XI);
      k_inviscid<0><<<grid, dim3(TileCfg<0>::TS, NL), 0, c->stream>>>(B, c->pd, 0);
    }
    {
      constexpr int T = TileCfg<1>::TS - 2, NL = TileCfg<1>::NL;
      dim3 grid((B.n[0] + NL - 1) / NL, (B.n[1] + T - 1) / T, B.n[2]);
      ProfScope ps(c, PK_INV_ETA);
      k_inviscid<1><<<grid, dim3(NL, TileCfg<1>::TS), 0, c->stream>>>(B, c->pd, 1);
    }
    {
      constexpr int T = TileCfg<2>::TS - 2, NL = TileCfg<2>::NL;
      dim3 grid((B.n[0] + NL - 1) / NL, B.n[1], (B.n[2] + T - 1) / T);
      ProfScope ps(c, PK_INV_ZETA);
      k_inviscid<2><<<grid, dim3(NL, TileCfg<2>::TS), 0, c->stream>>>(B, c->pd, visc ? 3 : 2);
    }
    c->launches += 3;
    if (visc) {
      dim3 g1((B.n[0] + 6 + 127) / 128, B.n[1] + 6, B.n[2] + 6);
      { ProfScope ps(c, PK_VISC_FLUX); k_visc_flux<<<g1, 128, 0, c->stream>>>(B, c->pd, c->ws); }
      dim3 g2((B.n[0] + 255) / 256, B.n[1], B.n[2]);
      { ProfScope ps(c, PK_VISC_DIV); k_visc_div<<<g2, 256, 0, c->stream>>>(B, c->ws); }
      c->launches += 2;
    }
  }
  CUDA_TRY(c, cudaGetLastError());
  return CFD_OK;
}
