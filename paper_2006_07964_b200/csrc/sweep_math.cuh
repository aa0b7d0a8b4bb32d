// Per-point arithmetic shared by the sweep kernels (k_march.cu: one thread marching along a pencil in eta / zeta;
// k_xi_tma.cu: the xi sweep out of a per-warp chunk ring).  sm_100a, fp64.  P:L<n> = PAPER.md line; U<k> = DESIGN.md reading.
// Shares no code with oracle/.
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
#pragma once
#include "fastmath.cuh"

// Eqs. 14-17 on the projected differences D1..D4 of one characteristic field; eps4 = 4 eps.
__device__ __forceinline__ void weno_corr(double D1, double D2, double D3, double D4, double eps4, double& cL, double& cR) {
  const double t1 = D2 - D1, t3 = D3 - D2, t5 = D4 - D3;
  const double t2 = fma(3.0, D2, -D1), t4 = D2 + D3, t6 = fma(-3.0, D3, D4);
  const double dA = fma((13.0 / 3.0) * t1, t1, fma(t2, t2, eps4));  // 4 (eps + beta_1)
  const double dB = fma((13.0 / 3.0) * t3, t3, fma(t4, t4, eps4));
  const double dC = fma((13.0 / 3.0) * t5, t5, fma(t6, t6, eps4));
  const double pA = dB * dC, pB = dA * dC, pC = dA * dB;
  const double sA = pA * pA, sC = pC * pC, pB10 = 10.0 * pB;  // 16 gamma_k alpha_k (dA dB dC)^2; sB = pB10 pB only inside the sums
  const double g1 = t1 - t3, g2 = t5 - t3;
  const double x = sA * g1, y = sC * g2;
  const double denL = fma(pB10, pB, fma(5.0, sC, sA)), denR = fma(pB10, pB, fma(5.0, sA, sC));
  const double numL = fma(0.375, x, -0.625 * y), numR = fma(0.375, y, -0.625 * x);
  const double inv = frcp(denL * denR);
  cL = (numL * denR) * inv;
  cR = (numR * denL) * inv;
}

__device__ __forceinline__ double pos_part(double x) { return __double2hiint(x) < 0 ? 0.0 : x; }   // max(x, 0)
__device__ __forceinline__ double neg_part(double x) { return __double2hiint(x) < 0 ? x : 0.0; }   // min(x, 0)

// Steger–Warming split flux (U3) of state U through the interface metric (kx,ky,kz), kn = |k|, ikn = 1/|k|, ADDED to F.
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
  // (l +- |l|)/2 exactly = max / min(l, 0); decided on the sign bit with integer instructions (a DSETP would take an
  // FP64-pipe slot, and that pipe is what bounds the sweeps)
  if (SGN > 0) { l1 = pos_part(l1); l4 = pos_part(l4); l5 = pos_part(l5); }
  else { l1 = neg_part(l1); l4 = neg_part(l4); l5 = neg_part(l5); }
  const double a1 = (2.0 * g1) * l1, s45 = l4 + l5, d45 = l4 - l5;
  const double f = U[0] * (0.5 / gamma);
  const double fs = f * s45;
  const double fA = fma(f, a1, fs), fc = f * ((c * ikn) * d45);
  // F is IN/OUT: the split flux is ADDED to what F holds (the caller seeds it with the central part of Phi and chains the
  // two split fluxes), so that the sums Phi = F+ + F- + G ride in the FMAs of the flux rows instead of separate DADDs
  F[0] += fA;
  F[1] = fma(fA, u, fma(fc, kx, F[1]));
  F[2] = fma(fA, v, fma(fc, ky, F[2]));
  F[3] = fma(fA, w, fma(fc, kz, F[3]));
  // 0.5 a1 q2 + 0.5 s45 (q2 + c2) + cn th + (3-g)/(2(g-1)) s45 c2  =  q2/2 (a1+s45) + cn th + s45 c2/(g-1)
  F[4] = fma(0.5 * q2, fA, fma(fc, th, fma(fs * c2, 1.0 / g1, F[4])));
}

// U5: symmetric 6-point Lagrange (150, -25, 3)/256
__device__ __forceinline__ double khalf(double m2, double m1, double z0, double p1, double p2, double p3) {
  return fma(150.0 / 256.0, z0 + p1, fma(-25.0 / 256.0, m1 + p2, (3.0 / 256.0) * (m2 + p3)));
}

// Eq. 4 from the conservative state
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

// O2 steps 1-5 at one point: Qs[s] = Q_{i-2+s} (s = 0..4), k = khat^d_i  ->  U^L_{i+1/2}, U^R_{i-1/2} and the
// point flux F_i (Eq. 4).
__device__ __forceinline__ void afweno_states(const double Qs[5][5], double kx, double ky, double kz, double gamma, double eps4,
                                              double UL[5], double UR[5], double Ft[5]) {
  const double g1 = gamma - 1.0;
  const double Q0 = Qs[2][0], Q1 = Qs[2][1], Q2 = Qs[2][2], Q3 = Qs[2][3], Q4 = Qs[2][4];
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
  {
    const double tk = th * (kk * ikn);  // khat . u
    Ft[0] = Q0 * tk;
    Ft[1] = fma(Q1, tk, kx * p);
    Ft[2] = fma(Q2, tk, ky * p);
    Ft[3] = fma(Q3, tk, kz * p);
    Ft[4] = (Q4 + p) * tk;
  }
  double V[5][4];
#pragma unroll
  for (int s = 0; s < 4; ++s) {
    const double d0 = Qs[s + 1][0] - Qs[s][0], d1 = Qs[s + 1][1] - Qs[s][1], d2 = Qs[s + 1][2] - Qs[s][2],
                 d3 = Qs[s + 1][3] - Qs[s][3], d4 = Qs[s + 1][4] - Qs[s][4];
    const double dx = fma(-d0, u, d1), dy = fma(-d0, v, d2), dz = fma(-d0, w, d3);
    const double E = fma(-w, d3, fma(-v, d2, fma(-u, d1, fma(hq, d0, d4))));
    const double A = fma(-b1, E, d0);
    const double nd = fma(nx, dx, fma(ny, dy, nz * dz));
    V[0][s] = fma(nx, A, fma(nz, dy, -ny * dz));
    V[1][s] = fma(ny, A, fma(nx, dz, -nz * dx));
    V[2][s] = fma(nz, A, fma(ny, dx, -nx * dy));
    const double y = hc * nd;  // c n.dm / (2 c^2);  hg E = (g-1) E / (2 c^2)
    V[3][s] = fma(hg, E, y);
    V[4][s] = fma(hg, E, -y);
  }
  double cL[5], cR[5];
#pragma unroll
  for (int f = 0; f < 5; ++f) weno_corr(V[f][0], V[f][1], V[f][2], V[f][3], eps4, cL[f], cR[f]);
#pragma unroll
  for (int side = 0; side < 2; ++side) {
    const double* cc = side == 0 ? cL : cR;
    double* U = side == 0 ? UL : UR;
    const double w1 = side == 0 ? 0.125 : -0.375, w2 = side == 0 ? 0.375 : -0.125;
    const double a = fma(nx, cc[0], fma(ny, cc[1], nz * cc[2])), s = cc[3] + cc[4], t = c * (cc[3] - cc[4]);
    const double wx = fma(ny, cc[2], -nz * cc[1]), wy = fma(nz, cc[0], -nx * cc[2]), wz = fma(nx, cc[1], -ny * cc[0]);
    const double r0 = a + s;
    U[0] = fma(w1, Qs[2][0] - Qs[1][0], fma(w2, Qs[3][0] - Qs[2][0], Q0)) + r0;
    U[1] = fma(w1, Qs[2][1] - Qs[1][1], fma(w2, Qs[3][1] - Qs[2][1], Q1)) + fma(u, r0, fma(nx, t, wx));
    U[2] = fma(w1, Qs[2][2] - Qs[1][2], fma(w2, Qs[3][2] - Qs[2][2], Q2)) + fma(v, r0, fma(ny, t, wy));
    U[3] = fma(w1, Qs[2][3] - Qs[1][3], fma(w2, Qs[3][3] - Qs[2][3], Q3)) + fma(w, r0, fma(nz, t, wz));
    U[4] = fma(w1, Qs[2][4] - Qs[1][4], fma(w2, Qs[3][4] - Qs[2][4], Q4)) +
           fma(hq, a, fma(u, wx, fma(v, wy, fma(w, wz, fma(H, s, th * t)))));
  }
}

// ---------------------------------------------------------------------------------------------------------
// NEXT-1: the ORIGINAL AFWENO ordering (Fig. 9; reading U7) at one interface i+1/2:
// Q6[s] = Q_{i-2+s} (s = 0..5), (kx,ky,kz) = khat_{i+1/2} (U5) with ikn = 1/|khat_{i+1/2}|.  The eigen-system is built at
// the interface from the arithmetic mean of (rho, u, v, w, p) at i and i+1; the left state U^L_{i+1/2} comes from a
// complete WENO interpolation on i-2..i+2, the right state U^R_{i+1/2} from another one on i-1..i+3 (nothing shared:
// that is what the modified scheme of Fig. 11 saves).  Same algebra as afweno_states (L applied to
// differences, R L = I for the central candidate, common-denominator weights), one side per stencil.
// ---------------------------------------------------------------------------------------------------------
__device__ __forceinline__ double weno_corr_left(double D1, double D2, double D3, double D4, double eps4) {
  const double t1 = D2 - D1, t3 = D3 - D2, t5 = D4 - D3;
  const double t2 = fma(3.0, D2, -D1), t4 = D2 + D3, t6 = fma(-3.0, D3, D4);
  const double dA = fma((13.0 / 3.0) * t1, t1, fma(t2, t2, eps4));
  const double dB = fma((13.0 / 3.0) * t3, t3, fma(t4, t4, eps4));
  const double dC = fma((13.0 / 3.0) * t5, t5, fma(t6, t6, eps4));
  const double pA = dB * dC, pB = dA * dC, pC = dA * dB;
  const double sA = pA * pA, sC = pC * pC;
  const double x = sA * (t1 - t3), y = sC * (t5 - t3);
  return fma(0.375, x, -0.625 * y) * frcp(fma(10.0 * pB, pB, fma(5.0, sC, sA)));
}
__device__ __forceinline__ double weno_corr_right(double D1, double D2, double D3, double D4, double eps4) {
  const double t1 = D2 - D1, t3 = D3 - D2, t5 = D4 - D3;
  const double t2 = fma(3.0, D2, -D1), t4 = D2 + D3, t6 = fma(-3.0, D3, D4);
  const double dA = fma((13.0 / 3.0) * t1, t1, fma(t2, t2, eps4));
  const double dB = fma((13.0 / 3.0) * t3, t3, fma(t4, t4, eps4));
  const double dC = fma((13.0 / 3.0) * t5, t5, fma(t6, t6, eps4));
  const double pA = dB * dC, pB = dA * dC, pC = dA * dB;
  const double sA = pA * pA, sC = pC * pC;
  const double x = sA * (t1 - t3), y = sC * (t5 - t3);
  return fma(0.375, y, -0.625 * x) * frcp(fma(10.0 * pB, pB, fma(5.0, sA, sC)));
}

__device__ __forceinline__ void afweno_iface_orig(const double Q6[6][5], double kx, double ky, double kz, double ikn, double gamma,
                                                  double eps4, double UL[5], double UR[5]) {
  const double g1 = gamma - 1.0;
  // U7: arithmetic mean of the primitives at i (s = 2) and i+1 (s = 3)
  double rho, u, v, w, p;
  {
    const double ia = frcp(Q6[2][0]), ib = frcp(Q6[3][0]);
    const double ua = Q6[2][1] * ia, va = Q6[2][2] * ia, wa = Q6[2][3] * ia;
    const double ub = Q6[3][1] * ib, vb = Q6[3][2] * ib, wb = Q6[3][3] * ib;
    const double pa = g1 * fma(-0.5 * Q6[2][0], fma(ua, ua, fma(va, va, wa * wa)), Q6[2][4]);
    const double pb = g1 * fma(-0.5 * Q6[3][0], fma(ub, ub, fma(vb, vb, wb * wb)), Q6[3][4]);
    rho = 0.5 * (Q6[2][0] + Q6[3][0]); u = 0.5 * (ua + ub); v = 0.5 * (va + vb); w = 0.5 * (wa + wb); p = 0.5 * (pa + pb);
  }
  const double hq = 0.5 * fma(u, u, fma(v, v, w * w));
  const double c2 = (gamma * p) * frcp(rho);
  const double rsc = frsqrt(c2);
  const double c = c2 * rsc, rc2 = rsc * rsc;
  const double H = fma(c2, 1.0 / g1, hq);  // (e + p)/rho of the mean state
  const double nx = kx * ikn, ny = ky * ikn, nz = kz * ikn;
  const double th = fma(nx, u, fma(ny, v, nz * w));
  const double b1 = g1 * rc2, hg = (0.5 * g1) * rc2, hc = 0.5 * rsc;
  double V[5][5];  // [field][difference s: Q_{i-1+s} - Q_{i-2+s}]
#pragma unroll
  for (int s = 0; s < 5; ++s) {
    const double d0 = Q6[s + 1][0] - Q6[s][0], d1 = Q6[s + 1][1] - Q6[s][1], d2 = Q6[s + 1][2] - Q6[s][2],
                 d3 = Q6[s + 1][3] - Q6[s][3], d4 = Q6[s + 1][4] - Q6[s][4];
    const double dx = fma(-d0, u, d1), dy = fma(-d0, v, d2), dz = fma(-d0, w, d3);
    const double E = fma(-w, d3, fma(-v, d2, fma(-u, d1, fma(hq, d0, d4))));
    const double A = fma(-b1, E, d0);
    const double nd = fma(nx, dx, fma(ny, dy, nz * dz));
    V[0][s] = fma(nx, A, fma(nz, dy, -ny * dz));
    V[1][s] = fma(ny, A, fma(nx, dz, -nz * dx));
    V[2][s] = fma(nz, A, fma(ny, dx, -nx * dy));
    const double y = hc * nd;
    V[3][s] = fma(hg, E, y);
    V[4][s] = fma(hg, E, -y);
  }
  double cL[5], cR[5];
#pragma unroll
  for (int f = 0; f < 5; ++f) {
    cL[f] = weno_corr_left(V[f][0], V[f][1], V[f][2], V[f][3], eps4);    // stencil i-2..i+2, left state at i+1/2
    cR[f] = weno_corr_right(V[f][1], V[f][2], V[f][3], V[f][4], eps4);   // stencil i-1..i+3, right state at i+1/2
  }
#pragma unroll
  for (int side = 0; side < 2; ++side) {
    const double* cc = side == 0 ? cL : cR;
    double* U = side == 0 ? UL : UR;
    const int ctr = side == 0 ? 2 : 3;  // the stencil's centre point
    const double w1 = side == 0 ? 0.125 : -0.375, w2 = side == 0 ? 0.375 : -0.125;
    const double a = fma(nx, cc[0], fma(ny, cc[1], nz * cc[2])), s = cc[3] + cc[4], t = c * (cc[3] - cc[4]);
    const double wx = fma(ny, cc[2], -nz * cc[1]), wy = fma(nz, cc[0], -nx * cc[2]), wz = fma(nx, cc[1], -ny * cc[0]);
    const double r0 = a + s;
    double lin[5];
#pragma unroll
    for (int m = 0; m < 5; ++m)
      lin[m] = fma(w1, Q6[ctr][m] - Q6[ctr - 1][m], fma(w2, Q6[ctr + 1][m] - Q6[ctr][m], Q6[ctr][m]));
    U[0] = lin[0] + r0;
    U[1] = lin[1] + fma(u, r0, fma(nx, t, wx));
    U[2] = lin[2] + fma(v, r0, fma(ny, t, wy));
    U[3] = lin[3] + fma(w, r0, fma(nz, t, wz));
    U[4] = lin[4] + fma(hq, a, fma(u, wx, fma(v, wy, fma(w, wz, fma(H, s, th * t)))));
  }
}
