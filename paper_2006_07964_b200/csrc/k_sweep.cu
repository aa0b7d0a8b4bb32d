// S2 (+ the derivative half of S3): one inviscid sweep along xi, eta or zeta — modified AFWENO (Fig. 11,
// P:L509-535) with Steger–Warming splitting (U3), Eq. 19, plus the 6th-order central derivative of the
// point viscous flux of the same direction, accumulated into r.   sm_100a, fp64, no tensor cores
// (stencil + per-point algebra; the FP64 ALUs are the binding roofline).
// P:L<n> = PAPER.md line; U<k> = DESIGN.md reading.  Shares no code with oracle/.
//
// One thread per point of a tile of TS positions along the sweep x NL lines (TS-2 outputs; the two end
// positions only supply F+ / F- to their neighbours).  Phases:
//   1  setup at i (prims, n = khat/|khat|, eigen system), projected differences, WENO corrections,
//      U^L_{i+1/2}, U^R_{i-1/2}; half-point metric khat_{i+1/2} with |khat| and 1/|khat| -> smem (computed ONCE
//      per interface, so both users see the same bits: free-stream preservation, U5); point flux -> smem
//   2  F+_{i+1/2} = SW+(U^L, khat_{i+1/2}),  F-_{i-1/2} = SW-(U^R, khat_{i-1/2}) -> smem
//   3  Eq. 19 + viscous central derivative, r update.
//
// Algebra (exact identities; what differs from a literal transcription):
//  * L_i is applied to the four differences dQ_s = Q_{s+1}-Q_s, never to Q: every quantity of Eqs. 14-17 is
//    a linear combination of differences except the central candidate, and R_i L_i = I turns that one into
//    a plain interpolation of Q:   U^L = Q_i + dQ_1/8 + 3 dQ_2/8 + R_i cL,   U^R = Q_i - 3 dQ_1/8 - dQ_2/8 + R_i cR
//    with cL = (3 sA g1 - 5 sC g2) / (8 denL), cR = (3 sC g2 - 5 sA g1) / (8 denR), g1 = t1 - t3, g2 = t5 - t3.
//  * L_i d without forming L (U4): dm = d_m - d_rho u, E = q2/2 d_rho - u.d_m + d_e, A = d_rho - (g-1)/c^2 E:
//    V_{1..3} = n A - n x dm,  V_{4,5} = ((g-1) E +- c n.dm) / (2 c^2);  R_i v likewise.
//  * alpha_k = 1/(eps+beta_k)^2 replaced by the product of the other two (eps+beta)^2 (common denominator),
//    all three scaled by 4 (cancels in the ratio), one reciprocal for both normalisations.
#include "cfd_internal.cuh"
#include "sweep_math.cuh"

namespace {

template <int DIR>
struct SweepCfg {
  static constexpr int TS = DIR == 0 ? 64 : 32;  // positions along the sweep (TS-2 outputs)
  static constexpr int NL = DIR == 0 ? 4 : 8;    // lines; for DIR 1,2 the lines run along i (coalesced)
  static constexpr int TE = TS + 4;              // point-flux slots: positions -3 .. TS relative to the first output
  static constexpr size_t smem_doubles(bool visc) { return (size_t)15 * TS * NL + (size_t)(visc ? 9 : 5) * TE * NL; }
};

// ACC 0: r = X;  1: r += X;  2: r = J (r + X)   with X = dFv/dxi^d - D^d   (U18 up to summation order)
template <int DIR, int ACC, bool VISC>
__global__ void __launch_bounds__(256, 2) k_sweep(BlockDev B, ParamsDev P, const double* __restrict__ W) {
  constexpr int TS = SweepCfg<DIR>::TS, NL = SweepCfg<DIR>::NL, T = TS - 2, TE = SweepCfg<DIR>::TE;
  extern __shared__ double smem[];
  double* const sFp = smem;                // [5][TS*NL]  F+ at pos+1/2
  double* const sFm = sFp + 5 * TS * NL;   // [5][TS*NL]  F- at pos-1/2
  double* const sK = sFm + 5 * TS * NL;    // [5][TS*NL]  khat_{pos+1/2} (3), |k|, 1/|k|
  double* const sT = sK + 5 * TS * NL;     // [5][TE*NL]  point inviscid flux, slot = sp + 2
  double* const sV = sT + 5 * TE * NL;     // [4][TE*NL]  point viscous flux rows 2..5 (VISC only)

  const int sp = DIR == 0 ? threadIdx.x : threadIdx.y;
  const int ln = DIR == 0 ? threadIdx.y : threadIdx.x;
  int i, j, k, s0;
  if (DIR == 0) { s0 = blockIdx.x * T; i = s0 - 1 + sp; j = blockIdx.y * NL + ln; k = blockIdx.z; }
  else if (DIR == 1) { s0 = blockIdx.y * T; i = blockIdx.x * NL + ln; j = s0 - 1 + sp; k = blockIdx.z; }
  else { s0 = blockIdx.z * T; i = blockIdx.x * NL + ln; j = blockIdx.y; k = s0 - 1 + sp; }
  const int n = B.n[DIR];
  const int pos = s0 - 1 + sp;
  const bool lane_ok = DIR == 0 ? (j < B.n[1]) : (i < B.n[0]);
  const bool active = lane_ok && pos <= n;
  const long long M = B.M, sd = B.s[DIR];
  const long long pidx = B.idx(i, j, k);
  const int SI = DIR == 0 ? ln * TS + sp : sp * NL + ln;            // index of (sp, ln) in a [TS*NL] plane
  const int TI = DIR == 0 ? ln * TE + sp + 2 : (sp + 2) * NL + ln;  // index of slot sp+2 in a [TE*NL] plane
  constexpr int SS = DIR == 0 ? 1 : NL;                             // smem stride of one step along the sweep
  const double gamma = P.gamma;

  double UL[5], UR[5];
  if (active) {
    const double* __restrict__ q = B.q + pidx;
    const double* __restrict__ kh = B.khat + (long long)(DIR * 3) * M + pidx;
    // ---- half-point metric of interface pos+1/2, once per interface (U5) ----
    {
      const double kx = khalf(kh[-2 * sd], kh[-sd], kh[0], kh[sd], kh[2 * sd], kh[3 * sd]);
      const double ky = khalf(kh[M - 2 * sd], kh[M - sd], kh[M], kh[M + sd], kh[M + 2 * sd], kh[M + 3 * sd]);
      const double kz = khalf(kh[2 * M - 2 * sd], kh[2 * M - sd], kh[2 * M], kh[2 * M + sd], kh[2 * M + 2 * sd], kh[2 * M + 3 * sd]);
      const double kk = fma(kx, kx, fma(ky, ky, kz * kz));
      const double ikn = frsqrt(kk);
      sK[SI] = kx; sK[TS * NL + SI] = ky; sK[2 * TS * NL + SI] = kz;
      sK[3 * TS * NL + SI] = kk * ikn; sK[4 * TS * NL + SI] = ikn;
    }
    // ---- state at i, eigen system of n = khat_i / |khat_i| ----
    const double g1 = gamma - 1.0;
    const double Q0 = q[0], Q1 = q[M], Q2 = q[2 * M], Q3 = q[3 * M], Q4 = q[4 * M];
    const double kx = kh[0], ky = kh[M], kz = kh[2 * M];
    const double ir = frcp(Q0);
    const double u = Q1 * ir, v = Q2 * ir, w = Q3 * ir;
    const double hq = 0.5 * fma(u, u, fma(v, v, w * w));
    const double p = g1 * fma(-Q0, hq, Q4);
    const double c2 = (gamma * p) * ir;
    const double rsc = frsqrt(c2);
    const double c = c2 * rsc, rc2 = rsc * rsc;
    const double H = (Q4 + p) * ir;
    const double kk = fma(kx, kx, fma(ky, ky, kz * kz));
    const double ikn = frsqrt(kk);
    const double nx = kx * ikn, ny = ky * ikn, nz = kz * ikn;
    const double th = fma(nx, u, fma(ny, v, nz * w));
    const double b1 = g1 * rc2, hg = (0.5 * g1) * rc2, hc = 0.5 * rsc;
    // ---- point flux at i (Eq. 4), khat . u = |k| th ----
    {
      const double tk = th * (kk * ikn);
      sT[TI] = Q0 * tk;
      sT[TE * NL + TI] = fma(Q1, tk, kx * p);
      sT[2 * TE * NL + TI] = fma(Q2, tk, ky * p);
      sT[3 * TE * NL + TI] = fma(Q3, tk, kz * p);
      sT[4 * TE * NL + TI] = (Q4 + p) * tk;
    }
    // ---- differences dQ_s = Q_{i-1+s} - Q_{i-2+s}, s = 0..3, projected with L_i ----
    double V[5][4];
    double lin[5][2];  // dQ_1, dQ_2 kept for the linear part
    {
      double a0 = q[-2 * sd], a1 = q[M - 2 * sd], a2 = q[2 * M - 2 * sd], a3 = q[3 * M - 2 * sd], a4 = q[4 * M - 2 * sd];
#pragma unroll
      for (int s = 0; s < 4; ++s) {
        const long long o = (long long)(s - 1) * sd;
        double b0, b1_, b2, b3, b4;
        if (s == 1) { b0 = Q0; b1_ = Q1; b2 = Q2; b3 = Q3; b4 = Q4; }
        else { b0 = q[o]; b1_ = q[M + o]; b2 = q[2 * M + o]; b3 = q[3 * M + o]; b4 = q[4 * M + o]; }
        const double d0 = b0 - a0, d1 = b1_ - a1, d2 = b2 - a2, d3 = b3 - a3, d4 = b4 - a4;
        a0 = b0; a1 = b1_; a2 = b2; a3 = b3; a4 = b4;
        if (s == 1 || s == 2) { lin[0][s - 1] = d0; lin[1][s - 1] = d1; lin[2][s - 1] = d2; lin[3][s - 1] = d3; lin[4][s - 1] = d4; }
        const double dx = fma(-d0, u, d1), dy = fma(-d0, v, d2), dz = fma(-d0, w, d3);
        const double E = fma(hq, d0, d4) - fma(u, d1, fma(v, d2, w * d3));
        const double A = fma(-b1, E, d0);
        const double nd = fma(nx, dx, fma(ny, dy, nz * dz));
        V[0][s] = fma(nx, A, fma(nz, dy, -ny * dz));
        V[1][s] = fma(ny, A, fma(nx, dz, -nz * dx));
        V[2][s] = fma(nz, A, fma(ny, dx, -nx * dy));
        const double x = hg * E, y = hc * nd;  // (g-1) E / (2 c^2),  c n.dm / (2 c^2)
        V[3][s] = x + y;
        V[4][s] = x - y;
      }
    }
    // ---- WENO corrections per characteristic field (shared beta: P:L488-496) ----
    double cL[5], cR[5];
    const double eps4 = 4.0 * P.eps;
#pragma unroll
    for (int f = 0; f < 5; ++f) weno_corr(V[f][0], V[f][1], V[f][2], V[f][3], eps4, cL[f], cR[f]);
    // ---- back-projection with R_i plus the linear interpolation of Q ----
#pragma unroll
    for (int side = 0; side < 2; ++side) {
      const double* cc = side == 0 ? cL : cR;
      double* U = side == 0 ? UL : UR;
      const double w1 = side == 0 ? 0.125 : -0.375, w2 = side == 0 ? 0.375 : -0.125;
      const double a = fma(nx, cc[0], fma(ny, cc[1], nz * cc[2])), s = cc[3] + cc[4], t = c * (cc[3] - cc[4]);
      const double wx = fma(ny, cc[2], -nz * cc[1]), wy = fma(nz, cc[0], -nx * cc[2]), wz = fma(nx, cc[1], -ny * cc[0]);
      const double r0 = a + s;
      U[0] = fma(w1, lin[0][0], fma(w2, lin[0][1], Q0)) + r0;
      U[1] = fma(w1, lin[1][0], fma(w2, lin[1][1], Q1)) + fma(u, r0, fma(nx, t, wx));
      U[2] = fma(w1, lin[2][0], fma(w2, lin[2][1], Q2)) + fma(v, r0, fma(ny, t, wy));
      U[3] = fma(w1, lin[3][0], fma(w2, lin[3][1], Q3)) + fma(w, r0, fma(nz, t, wz));
      U[4] = fma(w1, lin[4][0], fma(w2, lin[4][1], Q4)) + fma(hq, a, fma(u, wx, fma(v, wy, fma(w, wz, fma(H, s, th * t)))));
    }
    // ---- the four extra point fluxes of the tile (slots -2,-1 and TS, TS+1 relative to sp) and viscous rows ----
    if (sp < 2) {
      double F[5];
      const long long o = -2 * sd;
      point_flux(q[o], q[M + o], q[2 * M + o], q[3 * M + o], q[4 * M + o], kh[o], kh[M + o], kh[2 * M + o], gamma, F);
#pragma unroll
      for (int m = 0; m < 5; ++m) sT[m * TE * NL + TI - 2 * SS] = F[m];
      if (VISC) {
#pragma unroll
        for (int m = 0; m < 4; ++m) sV[m * TE * NL + TI - 2 * SS] = W[(long long)(DIR * 4 + m) * M + pidx + o];
      }
    }
    if (sp >= TS - 2 || pos >= n - 1) {
      double F[5];
      const long long o = 2 * sd;
      point_flux(q[o], q[M + o], q[2 * M + o], q[3 * M + o], q[4 * M + o], kh[o], kh[M + o], kh[2 * M + o], gamma, F);
#pragma unroll
      for (int m = 0; m < 5; ++m) sT[m * TE * NL + TI + 2 * SS] = F[m];
      if (VISC) {
#pragma unroll
        for (int m = 0; m < 4; ++m) sV[m * TE * NL + TI + 2 * SS] = W[(long long)(DIR * 4 + m) * M + pidx + o];
      }
    }
    if (VISC) {
#pragma unroll
      for (int m = 0; m < 4; ++m) sV[m * TE * NL + TI] = W[(long long)(DIR * 4 + m) * M + pidx];
    }
  }
  __syncthreads();
  if (active) {
    double F[5];
    {
      sw_flux<+1>(UL, sK[SI], sK[TS * NL + SI], sK[2 * TS * NL + SI], sK[3 * TS * NL + SI], sK[4 * TS * NL + SI], gamma, F);
#pragma unroll
      for (int m = 0; m < 5; ++m) sFp[m * TS * NL + SI] = F[m];
    }
    if (sp > 0) {
      const int SM1 = SI - SS;
      sw_flux<-1>(UR, sK[SM1], sK[TS * NL + SM1], sK[2 * TS * NL + SM1], sK[3 * TS * NL + SM1], sK[4 * TS * NL + SM1], gamma, F);
#pragma unroll
      for (int m = 0; m < 5; ++m) sFm[m * TS * NL + SI] = F[m];
    }
  }
  __syncthreads();
  if (active && sp >= 1 && sp <= TS - 2 && pos < n) {
    double jac = 0.0;
    if (ACC == 2) jac = B.jac[pidx];
#pragma unroll
    for (int m = 0; m < 5; ++m) {
      const double* fp = sFp + m * TS * NL + SI;
      const double* fm = sFm + m * TS * NL + SI;
      const double* ft = sT + m * TE * NL + TI;
      const double fph = fp[0] + fm[SS];
      const double fmh = fp[-SS] + fm[0];
      // Eq. 19
      const double D = (fph - fmh) + (17.0 / 256.0) * (ft[SS] - ft[-SS]) - (13.0 / 320.0) * (ft[2 * SS] - ft[-2 * SS]) +
                       (19.0 / 3840.0) * (ft[3 * SS] - ft[-3 * SS]);
      double X = -D;
      if (VISC && m > 0) {
        const double* fv = sV + (m - 1) * TE * NL + TI;
        const double dv = (3.0 / 4.0) * (fv[SS] - fv[-SS]) - (3.0 / 20.0) * (fv[2 * SS] - fv[-2 * SS]) +
                          (1.0 / 60.0) * (fv[3 * SS] - fv[-3 * SS]);
        X = dv - D;
      }
      double* r = B.r + m * M + pidx;
      if (ACC == 0) *r = X;
      else if (ACC == 1) *r = *r + X;
      else *r = jac * (*r + X);
    }
  }
}

template <int DIR, int ACC>
void launch_one(cfd_ctx* c, const BlockDev& B, bool visc) {
  constexpr int TS = SweepCfg<DIR>::TS, NL = SweepCfg<DIR>::NL, T = TS - 2;
  dim3 grid, block;
  if (DIR == 0) { grid = dim3((B.n[0] + T - 1) / T, (B.n[1] + NL - 1) / NL, B.n[2]); block = dim3(TS, NL); }
  else if (DIR == 1) { grid = dim3((B.n[0] + NL - 1) / NL, (B.n[1] + T - 1) / T, B.n[2]); block = dim3(NL, TS); }
  else { grid = dim3((B.n[0] + NL - 1) / NL, B.n[1], (B.n[2] + T - 1) / T); block = dim3(NL, TS); }
  const size_t sm = SweepCfg<DIR>::smem_doubles(visc) * sizeof(double);
  if (visc) k_sweep<DIR, ACC, true><<<grid, block, sm, c->stream>>>(B, c->pd, B.ws);
  else k_sweep<DIR, ACC, false><<<grid, block, sm, c->stream>>>(B, c->pd, B.ws);
}

}  // namespace

int march_init();
int launch_march(cfd_ctx* c, const BlockDev& B, int dir, int acc, const RkFuse* rk, int* rk_ctas, bool sx = false, bool no_rows = false);
int launch_march_xi(cfd_ctx* c, const BlockDev& B, int acc);

int sweep_init() {
  // opt in to > 48 KB of dynamic shared memory
  cudaError_t e = cudaSuccess;
#define OPT(D, A)                                                                                                               \
  if (e == cudaSuccess) e = cudaFuncSetAttribute(k_sweep<D, A, true>, cudaFuncAttributeMaxDynamicSharedMemorySize,              \
                                                 (int)(SweepCfg<D>::smem_doubles(true) * sizeof(double)));                      \
  if (e == cudaSuccess) e = cudaFuncSetAttribute(k_sweep<D, A, false>, cudaFuncAttributeMaxDynamicSharedMemorySize,             \
                                                 (int)(SweepCfg<D>::smem_doubles(false) * sizeof(double)));
  OPT(0, 0) OPT(1, 1) OPT(2, 2)
#undef OPT
  if (e != cudaSuccess) return -1;
  return march_init();
}

// Sweep plans (cfd_set_sweep_plan): 0 = all three marching, xi through warp-private transposed staging (k_march_xi);
// 1 = all three tiled (one thread per point);  2 = all three k_march (xi lanes run along j: uncoalesced loads);
// 3 = xi tiled and first (plain store), eta and zeta marching (zeta applies J).
int launch_sweeps(cfd_ctx* c, const BlockDev& B, const RkFuse* rk, int* rk_ctas) {
  if (rk && c->sweep_plan != 0) { c->err = "fused RK stage needs sweep plan 0"; return CFD_E_ARG; }
  if (c->prm.scheme == 1 && c->sweep_plan != 0) { c->err = "scheme 1 (original AFWENO) runs on the default sweep plan only"; return CFD_E_ARG; }
  const bool visc = c->pd.viscous != 0;
  if (c->sweep_plan == 1) {
    { ProfScope ps(c, PK_INV_XI); launch_one<0, 0>(c, B, visc); }
    { ProfScope ps(c, PK_INV_ETA); launch_one<1, 1>(c, B, visc); }
    { ProfScope ps(c, PK_INV_ZETA); launch_one<2, 2>(c, B, visc); }
    c->launches += 3;
  } else if (c->sweep_plan == 2) {
    { ProfScope ps(c, PK_INV_ETA); launch_march(c, B, 1, 0, nullptr, nullptr); }
    { ProfScope ps(c, PK_INV_ZETA); launch_march(c, B, 2, 1, nullptr, nullptr); }
    { ProfScope ps(c, PK_INV_XI); launch_march(c, B, 0, 2, nullptr, nullptr); }
  } else if (c->sweep_plan == 0) {
    {
      ProfScope ps(c, PK_INV_XI);
      const int b = (int)(&B - c->blk.data());
      const bool orig = c->prm.scheme == 1;  // original AFWENO: the chunk-ring kernel or, for odd ni, the plain march
      if (!orig && c->xi_mode == 1 && xi_tma_ok(c, b)) launch_xi_tma(c, b, true);
      else if ((orig || c->xi_mode != 2) && xi_ldg_ok(c, b)) launch_xi_tma(c, b, false);
      else if (orig) launch_march(c, B, 0, 0, nullptr, nullptr, false, true);
      else launch_march_xi(c, B, 0);
    }
    { ProfScope ps(c, PK_INV_ETA); launch_march(c, B, 1, 1, nullptr, nullptr, true); }
    {
      ProfScope ps(c, PK_INV_ZETA);
      const int rc = launch_march(c, B, 2, 2, rk, rk_ctas);
      if (rc != 0) return rc;
    }
  } else {
    { ProfScope ps(c, PK_INV_XI); launch_one<0, 0>(c, B, visc); c->launches++; }
    { ProfScope ps(c, PK_INV_ETA); launch_march(c, B, 1, 1, nullptr, nullptr); }
    { ProfScope ps(c, PK_INV_ZETA); launch_march(c, B, 2, 2, nullptr, nullptr); }
  }
  return 0;
}
