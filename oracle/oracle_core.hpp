// =====================================================================================
// ORACLE — TEST INFRASTRUCTURE, NOT PRODUCT CODE.
//
// Plain, slow, obviously-correct CPU statement of the hot path of
//   Ye, Zhang, Wan, Yan, Sun, "Accelerating CFD simulation with high order finite
//   difference method on curvilinear coordinates for modern GPU clusters",
//   Adv. Aerodyn. 4:7 (2022)  [/root/reference/PAPER.md, cited below as P:L<line>].
//
// It follows the paper step by step, in the paper's order and notation (SURVEY.md §8(c),
// steps O0–O4, readings U1–U18 which are restated in DESIGN.md).  No blocking, fusion or
// re-ordering beyond what the equations state.  It shares NO code with the CUDA path
// (paper_2006_07964_b200/csrc) and neither includes the other's headers.
//
// Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs
// may build, load or call anything in this directory.
//
// Parity status: pinned against the paper's printed constants, exactness properties,
// split-flux identities, free-stream preservation, discrete conservation, formal orders
// 5/6/3, decomposition/permutation equivalence and brute force (tests/test_oracle_*.py).
// "parity unpinned" items (vs. the AUTHORS' closed code): the eigenvector scaling (U4),
// the half-point metric interpolation (U5), ghost-layer closure (U12) and the wall /
// far-field formulas (U13, U14), which the paper does not print.  The readings themselves
// are pinned against mathematics in tests/test_oracle_bc_pins.py: the wall closure by
// polynomial exactness (quartics with zero slope return a(0)), the subsonic far field by
// its Riemann invariants and the upwind side's entropy / tangential velocity with distinct
// interior and far-field states, cfl_dt (U16) by a hand formula on a Cartesian grid, the
// stage-1 residual (U17) by the plain sum of squares of the R field.
//
// Everything is templated on the scalar type T so that oracle/flopcount.cpp can run the
// same per-point routines with a counting type (the contract flop count).
// =====================================================================================
#pragma once
#include <cmath>
#include <cstddef>
#include <cstdint>
#include <vector>
#include <string>

namespace orc {

constexpr int NG = 6;  // ghost layers per face (reading U12; the paper does not state it)

enum FaceType { FT_NONE = 0, FT_PERIODIC = 1, FT_INTERFACE = 2, FT_WALL = 3, FT_FARFIELD = 4 };

struct Params {
  double gamma, mach, reynolds, prandtl, weno_eps;
  int viscous;  // 0 Euler, 1 Navier–Stokes
  int scheme;   // 0 modified AFWENO (Fig. 11), 1 original (Fig. 9)
  double q_inf[5];
  double sutherland;  // S / T_inf of Sutherland's law (U11); <= 0: constant mu = 1
};

struct Face {
  int block, face;  // face: 0 -xi, 1 +xi, 2 -eta, 3 +eta, 4 -zeta, 5 +zeta
  int type;
  int nbr_block, nbr_face;
  int perm[3], sign[3];  // neighbour axis of my axis a is perm[a]; direction sign[a] = +-1
  double shift[3];       // added to the neighbour's coordinates when they become my ghosts
};

// ---- scalar helpers usable with double and with the counting type -------------------
using std::sqrt;
using std::fabs;

// 6th-order central first derivative, unit spacing (P:L105 names the scheme; these are its
// unique coefficients 3/4, -3/20, 1/60).
template <class T>
inline T d6(const T& m3, const T& m2, const T& m1, const T& p1, const T& p2, const T& p3) {
  return T(3.0 / 4.0) * (p1 - m1) - T(3.0 / 20.0) * (p2 - m2) + T(1.0 / 60.0) * (p3 - m3);
}

// O0: primitive variables from Q = (rho, rho u, rho v, rho w, e); p = (g-1)(e - rho|u|^2/2),
// T = gamma p / rho = c^2.
template <class T>
struct Prim {
  T rho, u, v, w, p, c, H, q2;
};
template <class T>
inline Prim<T> prims(const T Q[5], const T& gamma) {
  Prim<T> s;
  s.rho = Q[0];
  s.u = Q[1] / s.rho;
  s.v = Q[2] / s.rho;
  s.w = Q[3] / s.rho;
  s.q2 = s.u * s.u + s.v * s.v + s.w * s.w;
  s.p = (gamma - T(1.0)) * (Q[4] - T(0.5) * s.rho * s.q2);
  s.c = sqrt(gamma * s.p / s.rho);
  s.H = (Q[4] + s.p) / s.rho;
  return s;
}

// Eq. 4: point inviscid flux along the direction with hatted metrics k = grad(xi^d)/J.
template <class T>
inline void point_flux(const T Q[5], const T k[3], const T& gamma, T F[5]) {
  Prim<T> s = prims(Q, gamma);
  T th = k[0] * s.u + k[1] * s.v + k[2] * s.w;  // U/J of Eq. 4 (reading U9)
  F[0] = s.rho * th;
  F[1] = Q[1] * th + k[0] * s.p;
  F[2] = Q[2] * th + k[1] * s.p;
  F[3] = Q[3] * th + k[2] * s.p;
  F[4] = (Q[4] + s.p) * th;
}

// Steger–Warming split flux (P:L159 names it; formula = reading U3).  sgn = +1 -> F+, -1 -> F-.
template <class T>
inline void sw_flux(const T Q[5], const T k[3], const T& gamma, int sgn, T F[5]) {
  Prim<T> s = prims(Q, gamma);
  T kn = sqrt(k[0] * k[0] + k[1] * k[1] + k[2] * k[2]);
  T nx = k[0] / kn, ny = k[1] / kn, nz = k[2] / kn;
  T th = k[0] * s.u + k[1] * s.v + k[2] * s.w;
  T l1 = th, l4 = th + s.c * kn, l5 = th - s.c * kn;
  T sg = T(double(sgn));
  l1 = T(0.5) * (l1 + sg * fabs(l1));
  l4 = T(0.5) * (l4 + sg * fabs(l4));
  l5 = T(0.5) * (l5 + sg * fabs(l5));
  T g1 = gamma - T(1.0);
  T up = s.u + s.c * nx, vp = s.v + s.c * ny, wp = s.w + s.c * nz;
  T um = s.u - s.c * nx, vm = s.v - s.c * ny, wm = s.w - s.c * nz;
  T f = s.rho / (T(2.0) * gamma);
  F[0] = f * (T(2.0) * g1 * l1 + l4 + l5);
  F[1] = f * (T(2.0) * g1 * l1 * s.u + l4 * up + l5 * um);
  F[2] = f * (T(2.0) * g1 * l1 * s.v + l4 * vp + l5 * vm);
  F[3] = f * (T(2.0) * g1 * l1 * s.w + l4 * wp + l5 * wm);
  F[4] = f * (g1 * l1 * s.q2 + T(0.5) * l4 * (up * up + vp * vp + wp * wp) +
              T(0.5) * l5 * (um * um + vm * vm + wm * wm) +
              (T(3.0) - gamma) * (l4 + l5) * s.c * s.c / (T(2.0) * g1));
}

// Left / right eigenvector matrices of d(n.F)/dQ at state Q with unit normal n (reading U4:
// the paper does not print them; this is the branch-free Pulliam–Chaussee /
// Warming–Beam–Hyett form with the rho factors removed).  L[row][col], R[row][col];
// eigenvalues (th, th, th, th+c, th-c).
template <class T>
inline void eig_LR(const T Q[5], const T n[3], const T& gamma, T L[5][5], T R[5][5]) {
  Prim<T> s = prims(Q, gamma);
  const T nx = n[0], ny = n[1], nz = n[2];
  const T u = s.u, v = s.v, w = s.w, c = s.c, H = s.H;
  T g = gamma - T(1.0);
  T c2 = c * c;
  T b1 = g / c2;
  T b2 = b1 * s.q2 / T(2.0);
  T ph = g * s.q2 / T(2.0);
  T th = nx * u + ny * v + nz * w;
  T hq = s.q2 / T(2.0);
  // columns of R
  R[0][0] = nx;           R[0][1] = ny;           R[0][2] = nz;           R[0][3] = T(1.0);   R[0][4] = T(1.0);
  R[1][0] = nx * u;       R[1][1] = ny * u - nz;  R[1][2] = nz * u + ny;  R[1][3] = u + nx * c; R[1][4] = u - nx * c;
  R[2][0] = nx * v + nz;  R[2][1] = ny * v;       R[2][2] = nz * v - nx;  R[2][3] = v + ny * c; R[2][4] = v - ny * c;
  R[3][0] = nx * w - ny;  R[3][1] = ny * w + nx;  R[3][2] = nz * w;       R[3][3] = w + nz * c; R[3][4] = w - nz * c;
  R[4][0] = nx * hq + nz * v - ny * w;
  R[4][1] = ny * hq + nx * w - nz * u;
  R[4][2] = nz * hq + ny * u - nx * v;
  R[4][3] = H + c * th;
  R[4][4] = H - c * th;
  // rows of L
  L[0][0] = nx * (T(1.0) - b2) - (nz * v - ny * w);
  L[0][1] = nx * b1 * u;        L[0][2] = nz + nx * b1 * v;   L[0][3] = -ny + nx * b1 * w;  L[0][4] = -nx * b1;
  L[1][0] = ny * (T(1.0) - b2) - (nx * w - nz * u);
  L[1][1] = -nz + ny * b1 * u;  L[1][2] = ny * b1 * v;        L[1][3] = nx + ny * b1 * w;   L[1][4] = -ny * b1;
  L[2][0] = nz * (T(1.0) - b2) - (ny * u - nx * v);
  L[2][1] = ny + nz * b1 * u;   L[2][2] = -nx + nz * b1 * v;  L[2][3] = nz * b1 * w;        L[2][4] = -nz * b1;
  T h = T(1.0) / (T(2.0) * c2);
  L[3][0] = (ph - c * th) * h;  L[3][1] = (nx * c - g * u) * h;    L[3][2] = (ny * c - g * v) * h;
  L[3][3] = (nz * c - g * w) * h;  L[3][4] = g * h;
  L[4][0] = (ph + c * th) * h;  L[4][1] = -(nx * c + g * u) * h;   L[4][2] = -(ny * c + g * v) * h;
  L[4][3] = -(nz * c + g * w) * h; L[4][4] = g * h;
}

// Eq. 14 interpolants paired BY STENCIL with the Eq. 16 linear weights (reading U1), Eq. 15 non-linear weights, Eq. 13 combination.
// Stencil values (a,b,c,d,e) = u_{i-2..i+2}.
//   vL = value at i+1/2 from the left-biased stencil  (feeds F+ at i+1/2)
//   vR = value at i-1/2 from the right-biased stencil (feeds F- at i-1/2), same beta
// Eq. 17 smoothness indicators in the equivalent Jiang–Shu form
//   beta = 13/12 (second difference)^2 + 1/4 (first-difference form)^2 ;
// bA on {i-2,i-1,i} (= beta_1), bB on {i-1,i,i+1} (= beta_2), bC on {i,i+1,i+2} (= beta_3).
template <class T>
inline void weno5_beta(const T& a, const T& b, const T& c, const T& d, const T& e, T& bA, T& bB, T& bC) {
  T t1 = a - T(2.0) * b + c, t2 = a - T(4.0) * b + T(3.0) * c;
  bA = T(13.0 / 12.0) * t1 * t1 + T(0.25) * t2 * t2;
  T t3 = b - T(2.0) * c + d, t4 = b - d;
  bB = T(13.0 / 12.0) * t3 * t3 + T(0.25) * t4 * t4;
  T t5 = c - T(2.0) * d + e, t6 = T(3.0) * c - T(4.0) * d + e;
  bC = T(13.0 / 12.0) * t5 * t5 + T(0.25) * t6 * t6;
}

template <class T>
inline void weno5_LR(const T& a, const T& b, const T& c, const T& d, const T& e, const T& eps,
                     T& vL, T& vR) {
  T bA, bB, bC;
  weno5_beta(a, b, c, d, e, bA, bB, bC);
  T aA = T(1.0) / ((eps + bA) * (eps + bA));
  T aB = T(1.0) / ((eps + bB) * (eps + bB));
  T aC = T(1.0) / ((eps + bC) * (eps + bC));
  // left state at i+1/2: gamma = (1/16, 5/8, 5/16) on {i-2,i-1,i}, {i-1,i,i+1}, {i,i+1,i+2}
  {
    T wA = T(1.0 / 16.0) * aA, wB = T(5.0 / 8.0) * aB, wC = T(5.0 / 16.0) * aC;
    T pA = T(3.0 / 8.0) * a - T(5.0 / 4.0) * b + T(15.0 / 8.0) * c;
    T pB = -T(1.0 / 8.0) * b + T(3.0 / 4.0) * c + T(3.0 / 8.0) * d;
    T pC = T(3.0 / 8.0) * c + T(3.0 / 4.0) * d - T(1.0 / 8.0) * e;
    vL = (wA * pA + wB * pB + wC * pC) / (wA + wB + wC);
  }
  // right state at i-1/2: mirror image
  {
    T wA = T(5.0 / 16.0) * aA, wB = T(5.0 / 8.0) * aB, wC = T(1.0 / 16.0) * aC;
    T pA = -T(1.0 / 8.0) * a + T(3.0 / 4.0) * b + T(3.0 / 8.0) * c;
    T pB = T(3.0 / 8.0) * b + T(3.0 / 4.0) * c - T(1.0 / 8.0) * d;
    T pC = T(15.0 / 8.0) * c - T(5.0 / 4.0) * d + T(3.0 / 8.0) * e;
    vR = (wA * pA + wB * pB + wC * pC) / (wA + wB + wC);
  }
}

// Half-point hatted metric (reading U5; the paper only says "interpolated from point values
// directly"): symmetric 6-point Lagrange, k_{i+1/2} from k_{i-2..i+3}.
template <class T>
inline T khat_half(const T& m2, const T& m1, const T& z0, const T& p1, const T& p2, const T& p3) {
  return (T(150.0) * (z0 + p1) - T(25.0) * (m1 + p2) + T(3.0) * (m2 + p3)) / T(256.0);
}

// O2: inviscid derivative D_i, i = 0..n-1, along one grid line (modified AFWENO, Fig. 11
// P:L509–535, Eqs. 9–19).  Line arrays carry NG ghost points on each side:
//   Ql[m][NG + i], kl[c][NG + i] for i = -NG .. n+NG-1.   D[m][i] for i = 0..n-1.
// scheme 0 = modified (eigen-system at i), scheme 1 = original (eigen-system at i+1/2, Fig. 9).
template <class T>
void inviscid_line(int n, const T* const Ql[5], const T* const kl[3], const T& gamma, const T& eps,
                   int scheme, T* const D[5]) {
  const int o = NG;
  std::vector<T> Fp(5 * (n + 2)), Fm(5 * (n + 2)), Fpt(5 * (n + 6));
  // helper lambdas for indexing: Fp(m, i) for i in [-1, n], Fpt(m,i) for i in [-3, n+2]
  auto fp = [&](int m, int i) -> T& { return Fp[m * (n + 2) + (i + 1)]; };
  auto fm = [&](int m, int i) -> T& { return Fm[m * (n + 2) + (i + 1)]; };
  auto ft = [&](int m, int i) -> T& { return Fpt[m * (n + 6) + (i + 3)]; };

  if (scheme == 0) {
    for (int i = -1; i <= n; ++i) {
      // step 1–2: eigen-system at point i with n = k_i/|k_i|
      T Qi[5], ki[3], nn[3];
      for (int m = 0; m < 5; ++m) Qi[m] = Ql[m][o + i];
      for (int c = 0; c < 3; ++c) ki[c] = kl[c][o + i];
      T kn = sqrt(ki[0] * ki[0] + ki[1] * ki[1] + ki[2] * ki[2]);
      for (int c = 0; c < 3; ++c) nn[c] = ki[c] / kn;
      T L[5][5], R[5][5];
      eig_LR(Qi, nn, gamma, L, R);
      // step 3: V_m = L_i Q_{i+m}
      T V[5][5];  // V[s][field], s = 0..4 <-> i-2..i+2
      for (int s = 0; s < 5; ++s)
        for (int f = 0; f < 5; ++f) {
          T acc = T(0.0);
          for (int m = 0; m < 5; ++m) acc = acc + L[f][m] * Ql[m][o + i - 2 + s];
          V[s][f] = acc;
        }
      // step 4: WENO in characteristic space
      T vL[5], vR[5];
      for (int f = 0; f < 5; ++f) weno5_LR(V[0][f], V[1][f], V[2][f], V[3][f], V[4][f], eps, vL[f], vR[f]);
      // step 5: back to conservative variables
      T UL[5], UR[5];
      for (int m = 0; m < 5; ++m) {
        T aL = T(0.0), aR = T(0.0);
        for (int f = 0; f < 5; ++f) {
          aL = aL + R[m][f] * vL[f];
          aR = aR + R[m][f] * vR[f];
        }
        UL[m] = aL;
        UR[m] = aR;
      }
      // steps 6–7: half-point metrics and split fluxes
      if (i <= n - 1) {  // F+ at i+1/2, needed for i = -1 .. n-1
        T kh[3];
        for (int c = 0; c < 3; ++c)
          kh[c] = khat_half(kl[c][o + i - 2], kl[c][o + i - 1], kl[c][o + i], kl[c][o + i + 1],
                            kl[c][o + i + 2], kl[c][o + i + 3]);
        T F[5];
        sw_flux(UL, kh, gamma, +1, F);
        for (int m = 0; m < 5; ++m) fp(m, i) = F[m];
      }
      if (i >= 0) {  // F- at i-1/2, needed for i = 0 .. n
        T kh[3];
        for (int c = 0; c < 3; ++c)
          kh[c] = khat_half(kl[c][o + i - 3], kl[c][o + i - 2], kl[c][o + i - 1], kl[c][o + i],
                            kl[c][o + i + 1], kl[c][o + i + 2]);
        T F[5];
        sw_flux(UR, kh, gamma, -1, F);
        for (int m = 0; m < 5; ++m) fm(m, i) = F[m];
      }
    }
  } else {
    // Original AFWENO ordering (Fig. 9): characteristic space at i+1/2 (reading U7:
    // arithmetic mean of (rho,u,v,w,p) at i and i+1, normal from k_{i+1/2}); two complete
    // interpolations, left-biased (i-2..i+2) and right-biased (i-1..i+3).
    for (int i = -1; i <= n - 1; ++i) {
      T kh[3];
      for (int c = 0; c < 3; ++c)
        kh[c] = khat_half(kl[c][o + i - 2], kl[c][o + i - 1], kl[c][o + i], kl[c][o + i + 1],
                          kl[c][o + i + 2], kl[c][o + i + 3]);
      T Q0[5], Q1[5];
      for (int m = 0; m < 5; ++m) { Q0[m] = Ql[m][o + i]; Q1[m] = Ql[m][o + i + 1]; }
      Prim<T> s0 = prims(Q0, gamma), s1 = prims(Q1, gamma);
      T rho = T(0.5) * (s0.rho + s1.rho), u = T(0.5) * (s0.u + s1.u), v = T(0.5) * (s0.v + s1.v);
      T w = T(0.5) * (s0.w + s1.w), p = T(0.5) * (s0.p + s1.p);
      T Qa[5] = {rho, rho * u, rho * v, rho * w, p / (gamma - T(1.0)) + T(0.5) * rho * (u * u + v * v + w * w)};
      T kn = sqrt(kh[0] * kh[0] + kh[1] * kh[1] + kh[2] * kh[2]);
      T nn[3] = {kh[0] / kn, kh[1] / kn, kh[2] / kn};
      T L[5][5], R[5][5];
      eig_LR(Qa, nn, gamma, L, R);
      T V[6][5];  // i-2 .. i+3
      for (int s = 0; s < 6; ++s)
        for (int f = 0; f < 5; ++f) {
          T acc = T(0.0);
          for (int m = 0; m < 5; ++m) acc = acc + L[f][m] * Ql[m][o + i - 2 + s];
          V[s][f] = acc;
        }
      T vL[5], vR[5], dum;
      for (int f = 0; f < 5; ++f) {
        weno5_LR(V[0][f], V[1][f], V[2][f], V[3][f], V[4][f], eps, vL[f], dum);   // left state at i+1/2
        weno5_LR(V[1][f], V[2][f], V[3][f], V[4][f], V[5][f], eps, dum, vR[f]);   // right state at (i+1)-1/2
      }
      T UL[5], UR[5];
      for (int m = 0; m < 5; ++m) {
        T aL = T(0.0), aR = T(0.0);
        for (int f = 0; f < 5; ++f) { aL = aL + R[m][f] * vL[f]; aR = aR + R[m][f] * vR[f]; }
        UL[m] = aL; UR[m] = aR;
      }
      T Fa[5], Fb[5];
      sw_flux(UL, kh, gamma, +1, Fa);
      sw_flux(UR, kh, gamma, -1, Fb);
      for (int m = 0; m < 5; ++m) { fp(m, i) = Fa[m]; fm(m, i + 1) = Fb[m]; }
    }
  }
  // step 8: point fluxes F_i (Eq. 4) for i = -3 .. n+2
  for (int i = -3; i <= n + 2; ++i) {
    T Qi[5], ki[3], F[5];
    for (int m = 0; m < 5; ++m) Qi[m] = Ql[m][o + i];
    for (int c = 0; c < 3; ++c) ki[c] = kl[c][o + i];
    point_flux(Qi, ki, gamma, F);
    for (int m = 0; m < 5; ++m) ft(m, i) = F[m];
  }
  // steps 7 (sum, cuda_sum_split_flux of Fig. 11) and 9 (Eq. 19)
  for (int i = 0; i < n; ++i)
    for (int m = 0; m < 5; ++m) {
      T fph = fp(m, i) + fm(m, i + 1);      // f_{i+1/2}
      T fmh = fp(m, i - 1) + fm(m, i);      // f_{i-1/2}
      D[m][i] = (fph - fmh) + T(17.0 / 256.0) * (ft(m, i + 1) - ft(m, i - 1)) -
                T(13.0 / 320.0) * (ft(m, i + 2) - ft(m, i - 2)) +
                T(19.0 / 3840.0) * (ft(m, i + 3) - ft(m, i - 3));
    }
}

// O3 (first half): Cartesian gradients of phi = (u,v,w,T) by the chain rule Eq. 21
// with xi_x = J * xihat_x.  dphi[d][f] = d phi_f / d xi^d; kh[d][c] = hatted metric; out g[c][f].
template <class T>
inline void grad_point(const T dphi[3][4], const T kh[3][3], const T& J, T g[3][4]) {
  for (int c = 0; c < 3; ++c)
    for (int f = 0; f < 4; ++f)
      g[c][f] = J * ((kh[0][c] * dphi[0][f] + kh[1][c] * dphi[1][f]) + kh[2][c] * dphi[2][f]);
}

// Molecular viscosity mu(T) ("molecular viscosity mu" stored per point; reading U11, NEXT-3): Sutherland's law in
// the reference scales (T_inf = 1, mu(1) = 1):  mu = T^(3/2) (1 + S) / (T + S),  S = 110.4 K / T_inf;  S <= 0: mu = 1.
template <class T>
inline T sutherland_mu(const T& Tt, double S) {
  if (!(S > 0.0)) return T(1.0);
  return Tt * sqrt(Tt) * T(1.0 + S) / (Tt + T(S));
}

// O3 (second half): point viscous flux along direction with hatted metrics k (Eqs. 5–6,
// P:L83–93; readings U8, U9).  g[c][f] = d phi_f / d x_c, phi = (u,v,w,T); mu_eff = (Ma/Re) mu,
// lambda = -2/3 mu_eff; qdot_c = kappa dT/dx_c with kappa = mu_eff / (Pr (gamma-1)).
template <class T>
inline void visc_flux_point(const T vel[3], const T g[3][4], const T k[3], const T& mu, const T& kappa,
                            T Fv[5]) {
  T div = g[0][0] + g[1][1] + g[2][2];
  T lam = -T(2.0 / 3.0) * mu;
  T txx = lam * div + T(2.0) * mu * g[0][0];
  T tyy = lam * div + T(2.0) * mu * g[1][1];
  T tzz = lam * div + T(2.0) * mu * g[2][2];
  T txy = mu * (g[1][0] + g[0][1]);
  T txz = mu * (g[2][0] + g[0][2]);
  T tyz = mu * (g[2][1] + g[1][2]);
  T bx = vel[0] * txx + vel[1] * txy + vel[2] * txz + kappa * g[0][3];
  T by = vel[0] * txy + vel[1] * tyy + vel[2] * tyz + kappa * g[1][3];
  T bz = vel[0] * txz + vel[1] * tyz + vel[2] * tzz + kappa * g[2][3];
  Fv[0] = T(0.0);
  Fv[1] = k[0] * txx + k[1] * txy + k[2] * txz;
  Fv[2] = k[0] * txy + k[1] * tyy + k[2] * tyz;
  Fv[3] = k[0] * txz + k[1] * tyz + k[2] * tzz;
  Fv[4] = k[0] * bx + k[1] * by + k[2] * bz;
}

// phi = (u, v, w, T = gamma p / rho) at a point.
template <class T>
inline void phi_point(const T Q[5], const T& gamma, T phi[4]) {
  Prim<T> s = prims(Q, gamma);
  phi[0] = s.u; phi[1] = s.v; phi[2] = s.w; phi[3] = gamma * s.p / s.rho;
}

// ---- Eq. 7 / Eq. 8: one metric from products of first derivatives --------
// Implemented at block level below (needs 3-D arrays).

// =====================================================================================
// Block-level solver (double only)
// =====================================================================================
struct Block {
  int n[3];        // interior sizes ni, nj, nk
  int m[3];        // with ghosts
  size_t M;        // m0*m1*m2
  std::vector<double> q, qn, r, xyz, khat, jac;
  int ftype[6];    // face types, FT_NONE if no descriptor
  int fidx[6];     // index into faces, -1 if none
  inline size_t idx(int i, int j, int k) const {
    return (size_t(k + NG) * m[1] + size_t(j + NG)) * m[0] + size_t(i + NG);
  }
  inline size_t stride(int axis) const { return axis == 0 ? 1 : (axis == 1 ? size_t(m[0]) : size_t(m[0]) * m[1]); }
};

struct Solver {
  Params prm;
  std::vector<Block> blk;
  std::vector<Face> faces;
  std::string err;
  int nthreads = 1;

  int create(int nblocks, const int* dims, int nfaces, const Face* f, const Params* p);
  int compute_metrics();
  int rhs();
  int rk_stage(int stage, double dt, double* res5);
  int exchange_interfaces();
  int apply_bc();
  double cfl_dt(double cfl) const;

  // pieces (public for the pins)
  void fill_connect(int field /*0 q, 1 xyz*/);
  void bc_xyz();
  int map_index(const Face& f, const int me[3], int nb[3]) const;
};

}  // namespace orc
