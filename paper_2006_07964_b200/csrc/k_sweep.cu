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
#include "fastmath.cuh"

namespace {

template <int DIR>
struct SweepCfg {
  static constexpr int TS = DIR == 0 ? 64 : 32;  // positions along the sweep (TS-2 outputs)
  static constexpr int NL = DIR == 0 ? 4 : 8;    // lines; for DIR 1,2 the lines run along i (coalesced)
  static constexpr int TE = TS + 4;              // point-flux slots: positions -3 .. TS relative to the first output
  static constexpr size_t smem_doubles(bool visc) { return (size_t)15 * TS * NL + (size_t)(visc ? 9 : 5) * TE * NL; }
};

// Eqs. 14-17 on the projected differences D1..D4 of one characteristic field; eps4 = 4 eps.
__device__ __forceinline__ void weno_corr(double D1, double D2, double D3, double D4, double eps4, double& cL, double& cR) {
  const double t1 = D2 - D1, t3 = D3 - D2, t5 = D4 - D3;
  const double t2 = fma(3.0, D2, -D1), t4 = D2 + D3, t6 = fma(-3.0, D3, D4);
  const double dA = fma((13.0 / 3.0) * t1, t1, fma(t2, t2, eps4));  // 4 (eps + beta_1)
  const double dB = fma((13.0 / 3.0) * t3, t3, fma(t4, t4, eps4));
  const double dC = fma((13.0 / 3.0) * t5, t5, fma(t6, t6, eps4));
  const double pA = dB * dC, pB = dA * dC, pC = dA * dB;
  const double sA = pA * pA, sB = (10.0 * pB) * pB, sC = pC * pC;  // 16 gamma_k alpha_k (dA dB dC)^2
  const double g1 = t1 - t3, g2 = t5 - t3;
  const double x = sA * g1, y = sC * g2;
  const double denL = fma(5.0, sC, sA + sB), denR = fma(5.0, sA, sB + sC);
  const double numL = fma(0.375, x, -0.625 * y), numR = fma(0.375, y, -0.625 * x);
  const double inv = frcp(denL * denR);
  cL = (numL * denR) * inv;
  cR = (numR * denL) * inv;
}

// Steger–Warming split flux (U3) of state U through the interface metric (kx,ky,kz), kn = |k|, ikn = 1/|k|.
template <int SGN>
__device__ __forceinline__ void sw_flux(const double U[5], double kx, double ky, double kz, double kn, double ikn,
                                        double gamma, double F[5]) {
  const double g1 = gamma - 1.0;
  const double ir = frcp(U[0]);
  const double u = U[1] * ir, v = U[2] * ir, w = U[3] * ir;
  const double q2 = fma(u, u, fma(v, v, w * w));
  const double p = g1 * fma(-0.5 * U[0], q2, U[4]);
  const double c2 = (gamma * p) * ir;
  const double c = c2 * frsqrt(c2);
  const double th = fma(kx, u, fma(ky, v, kz * w));
  const double ck = c * kn;
  double l1 = th, l4 = th + ck, l5 = th - ck;
  if (SGN > 0) { l1 = fmax(l1, 0.0); l4 = fmax(l4, 0.0); l5 = fmax(l5, 0.0); }  // (l + |l|)/2 exactly
  else { l1 = fmin(l1, 0.0); l4 = fmin(l4, 0.0); l5 = fmin(l5, 0.0); }
  const double a1 = (2.0 * g1) * l1, s45 = l4 + l5, d45 = l4 - l5;
  const double f = U[0] * (0.5 / gamma);
  const double fA = f * (a1 + s45), fc = f * ((c * ikn) * d45);
  F[0] = fA;
  F[1] = fma(fA, u, fc * kx);
  F[2] = fma(fA, v, fc * ky);
  F[3] = fma(fA, w, fc * kz);
  // 0.5 a1 q2 + 0.5 s45 (q2 + c2) + cn th + (3-g)/(2(g-1)) s45 c2  =  q2/2 (a1+s45) + cn th + s45 c2/(g-1)
  F[4] = fma(0.5 * q2, fA, fma(fc, th, ((f * s45) * c2) * (1.0 / g1)));
}

__device__ __forceinline__ double khalf(double m2, double m1, double z0, double p1, double p2, double p3) {
  // U5: symmetric 6-point Lagrange (150, -25, 3)/256
  return fma(150.0 / 256.0, z0 + p1, fma(-25.0 / 256.0, m1 + p2, (3.0 / 256.0) * (m2 + p3)));
}

// Eq. 4 from conservative state
__device__ __forceinline__ void point_flux(double r, double m1, double m2, double m3, double e, double kx, double ky, double kz,
                                           double gamma, double F[5]) {
  const double ir = frcp(r);
  const double u = m1 * ir, v = m2 * ir, w = m3 * ir;
  const double p = (gamma - 1.0) * fma(-0.5 * r, fma(u, u, fma(v, v, w * w)), e);
  const double th = fma(kx, u, fma(ky, v, kz * w));
  F[0] = r * th;
  F[1] = fma(m1, th, kx * p);
  F[2] = fma(m2, th, ky * p);
  F[3] = fma(m3, th, kz * p);
  F[4] = (e + p) * th;
}

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
  if (visc) k_sweep<DIR, ACC, true><<<grid, block, sm, c->stream>>>(B, c->pd, c->ws);
  else k_sweep<DIR, ACC, false><<<grid, block, sm, c->stream>>>(B, c->pd, c->ws);
}

}  // namespace

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
  return e == cudaSuccess ? 0 : -1;
}

int launch_sweeps(cfd_ctx* c, const BlockDev& B) {
  const bool visc = c->pd.viscous != 0;
  { ProfScope ps(c, PK_INV_XI); launch_one<0, 0>(c, B, visc); }
  { ProfScope ps(c, PK_INV_ETA); launch_one<1, 1>(c, B, visc); }
  { ProfScope ps(c, PK_INV_ZETA); launch_one<2, 2>(c, B, visc); }
  c->launches += 3;
  return 0;
}
