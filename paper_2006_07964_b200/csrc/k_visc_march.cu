// S3 up to the point fluxes as ONE k-marching kernel (replaces k_phi + k_visc_flux<true> on the default plan).
// sm_100a, fp64.  P:L<n> = PAPER.md line; U<k> = DESIGN.md reading.  Shares no code with oracle/.
//
// k_visc_flux reads 72 neighbour values of phi per point through L1 (latency-bound: DRAM 44 %, LSU wavefronts 62 %) and
// needs phi stored by a separate pass.  Here a CTA owns a tile of (i, j) columns and marches along k:
//   * phi = (u, v, w, T) is computed from Q on the fly and never stored;
//   * the zeta stencil lives in REGISTERS: each thread keeps phi of its own column at k-3 .. k+3 (28 doubles);
//   * the (i, j) plane of phi at k (tile + halo of 3 in j, 6 in i) lives in SHARED memory, double buffered: the xi and
//     eta stencils read it with LDS;
//   * Q of plane k+4 and the halo cells of plane k+1 arrive by cp.async in thread-private shared-memory slots one step
//     ahead (no registers held across a step); the ten metric values of plane k+1 are loaded at the end of step k, when few
//     registers are live (staging them through shared memory cost more shared-memory instructions than it hid latency);
//   * the xi rows of the flux go to shared memory and come back as S = d(Fv^xi)/d(xi), as in k_visc_flux<true>.
// Output (workspace rows): W[0..3] = S on interior points; W[4..7] = Fv^eta rows 2..5 on (i, k) interior, j in [-3, nj+3);
// W[8..11] = Fv^zeta rows 2..5 on (i, j) interior, k in [-3, nk+3).  Same arithmetic per point as k_phi + k_visc_flux.
#include "cfd_internal.cuh"
#include "fastmath.cuh"
#include "stencil.cuh"
#include <cmath>

namespace {

// Tile geometry: VX x VY threads own the columns i0-3 .. i0+VX-4 of the rows j0 .. j0+VY-1; VX-6 of them are output columns.
// The plane row pitch PC is congruent to VX modulo 16 doubles, so that consecutive threads (also across a row change
// inside a warp when VX is not a multiple of 32) hit consecutive banks.  Every thread stages HPT halo cells of the plane.
template <int VX_, int VY_>
struct VG {
  static constexpr int VX = VX_, VY = VY_;
  static constexpr int PC = VX + 16;          // plane columns i0-6 .. i0+VX-1 (VX + 6), padded
  static constexpr int PR = VY + 6;           // plane rows j0-3 .. j0+VY+2
  static constexpr int NHALO = 2 * 3 * VX + 2 * 3 * VY;
  static constexpr int NT = VX * VY;
  static constexpr int HPT = (NHALO + NT - 1) / NT;   // halo cells staged per thread
  static constexpr int MINB = NT <= 256 ? 2 : 1;      // CTAs per SM (128 registers per thread either way)
  static_assert(NT <= 512, "k_visc_march: tile geometry");
  // shared memory (doubles): phi planes [2][4][PR][PC] | xi rows [2][4][VY][VX] | Q stage [5][NT] | halo stage [5][HPT NT]
  static constexpr int SM_PHI = 2 * 4 * PR * PC, SM_WX = 2 * 4 * NT, SM_Q = 5 * NT, SM_H = 5 * HPT * NT;
  static constexpr int SMEM = (SM_PHI + SM_WX + SM_Q + SM_H) * 8;
};

// phi = (u, v, w, T = gamma p / rho) from the conservative state: the arithmetic of k_phi
__device__ __forceinline__ void phi_of(double r, double m1, double m2, double m3, double e, double gamma, double f[4]) {
  const double ir = frcp(r);
  const double u = m1 * ir, v = m2 * ir, w = m3 * ir;
  const double pr = (gamma - 1.0) * fma(-0.5 * r, fma(u, u, fma(v, v, w * w)), e);
  f[0] = u; f[1] = v; f[2] = w; f[3] = (gamma * pr) * ir;
}

template <class G>
__global__ void __launch_bounds__(G::NT, G::MINB) k_visc_march(BlockDev B, ParamsDev P, double* __restrict__ W, int TI, int KS) {
  constexpr int VX = G::VX, VY = G::VY, PC = G::PC, PR = G::PR, NHALO = G::NHALO, NT = G::NT, HPT = G::HPT;
  constexpr int SM_PHI = G::SM_PHI, SM_WX = G::SM_WX, SM_Q = G::SM_Q;
  extern __shared__ double vsm[];
  double* const sphi = vsm;               // [2][4][PR][PC]
  double* const swx = sphi + SM_PHI;      // [2][4][VY][VX]
  double* const sq = swx + SM_WX;         // [5][NT]
  double* const sh = sq + SM_Q;           // [5][HPT NT]
  const int tx = threadIdx.x, ty = threadIdx.y, tid = ty * VX + tx;
  const int i0 = blockIdx.x * TI, j0 = -3 + (int)blockIdx.y * VY;
  const int kb = -3 + (int)blockIdx.z * KS, ke = min(kb + KS, B.n[2] + 3);
  const int i = i0 - 3 + tx, j = j0 + ty;
  const long long M = B.M, s1 = B.s[1], s2 = B.s[2];
  const double gamma = P.gamma;
  // my column: inside the array?  (plane filler)   which results are wanted from it?
  const bool col_in = (i + NG < B.m[0]) && (j + NG < B.m[1]);
  const bool oi = i < 0 || i >= B.n[0], oj = j < 0 || j >= B.n[1];
  const bool own = tx >= 3 && tx < TI + 3 && i < B.n[0];                       // point-wise outputs are mine
  const bool want_xi = tx < TI + 6 && i < B.n[0] + 3 && !oj;                    // xi rows (k interior)
  const bool want_eta = own && j < B.n[1] + 3;                                  // eta rows (k interior)
  const bool want_zeta = own && !oj;                                            // zeta rows (all k of the march)
  const bool any = col_in && (want_xi || want_eta || want_zeta) && !(oi && oj);
  const long long pcol = (long long)(j + NG) * s1 + (i + NG);                  // array offset of (i, j, k = -NG)
  // my halo cells of the plane (if any): top band, bottom band, left columns, right columns
  int hpl[HPT];           // offset of the cell inside one field of the plane (hr * PC + hc)
  bool halo_in[HPT];
  long long phal[HPT];
#pragma unroll
  for (int h = 0; h < HPT; ++h) {
    const int t = tid + h * NT;
    int hc = -1, hr = -1;  // plane column / row
    if (t < 3 * VX) { hr = t / VX; hc = 3 + t % VX; }
    else if (t < 6 * VX) { hr = VY + 3 + (t - 3 * VX) / VX; hc = 3 + t % VX; }
    else if (t < 6 * VX + 3 * VY) { hr = 3 + (t - 6 * VX) / 3; hc = (t - 6 * VX) % 3; }
    else if (t < NHALO) { hr = 3 + (t - 6 * VX - 3 * VY) / 3; hc = VX + 3 + (t - 6 * VX - 3 * VY) % 3; }
    const int hi = i0 - 6 + hc, hj = j0 - 3 + hr;
    halo_in[h] = hc >= 0 && hi + NG >= 0 && hi + NG < B.m[0] && hj + NG >= 0 && hj + NG < B.m[1];
    phal[h] = (long long)(hj + NG) * s1 + (hi + NG);
    hpl[h] = hr * PC + hc;
  }

  auto stage = [&](int k) {  // cp.async for the step of plane k: Q(k+3) of my column, my halo cell at k, metrics at k
    if (col_in && k + 3 + NG < B.m[2]) {
      const long long o = pcol + (long long)(k + 3 + NG) * s2;
#pragma unroll
      for (int m = 0; m < 5; ++m) cp8(sq + m * NT + tid, B.q + m * M + o);
    }
#pragma unroll
    for (int h = 0; h < HPT; ++h) {
      if (halo_in[h]) {
        const long long o = phal[h] + (long long)(k + NG) * s2;
#pragma unroll
        for (int m = 0; m < 5; ++m) cp8(sh + (m * HPT + h) * NT + tid, B.q + m * M + o);
      }
    }
    cp_commit();
  };

  // ---- prologue: phi of my column at kb-3 .. kb+2 ----
  double ph[7][4];
#pragma unroll
  for (int t = 0; t < 7; ++t)
#pragma unroll
    for (int f = 0; f < 4; ++f) ph[t][f] = 0.0;
  if (col_in) {
#pragma unroll
    for (int t = 0; t < 6; ++t) {
      const long long o = pcol + (long long)(kb - 3 + t + NG) * s2;
      phi_of(B.q[o], B.q[M + o], B.q[2 * M + o], B.q[3 * M + o], B.q[4 * M + o], gamma, ph[t]);
    }
  }
  stage(kb);
  // the ten metric values of plane k are loaded at the END of step k-1 (after its flux arithmetic, when few registers are
  // live) and used in the second half of step k: half a step of distance covers the DRAM latency of these streaming loads
  double kh[3][3], J = 0.0;
#pragma unroll
  for (int d = 0; d < 3; ++d)
#pragma unroll
    for (int c = 0; c < 3; ++c) kh[d][c] = 0.0;
  auto load_metrics = [&](int k) {
    if (any) {
      const long long o = pcol + (long long)(k + NG) * s2;
#pragma unroll
      for (int d = 0; d < 3; ++d)
#pragma unroll
        for (int c = 0; c < 3; ++c) kh[d][c] = __ldg(B.khat + (d * 3 + c) * M + o);
      J = __ldg(B.jac + o);
    }
  };
  load_metrics(kb);
  const double mu0 = P.mu, kap0 = P.kappa, suth = P.suth;
  auto s_of_plane = [&](int kk) {
    if (own && !oj && col_in && kk >= 0 && kk < B.n[2]) {
      const long long p = pcol + (long long)(kk + NG) * s2;
      const double* const sx = swx + (kk & 1) * (4 * NT);
#pragma unroll
      for (int m = 0; m < 4; ++m) {
        const double* a = sx + (m * VY + ty) * VX + tx;
        W[(long long)m * M + p] = d6c(a[-3], a[-2], a[-1], a[1], a[2], a[3]);
      }
    }
  };
  for (int k = kb; k < ke; ++k) {
    cp_wait<0>();
    const bool ok = k < 0 || k >= B.n[2];
    double* const pl = sphi + (k & 1) * (4 * PR * PC);
    // ---- newest plane of my column into the register pipeline; plane k (my own phi and my halo cell) into shared memory ----
    if (col_in && k + 3 + NG < B.m[2])
      phi_of(sq[tid], sq[NT + tid], sq[2 * NT + tid], sq[3 * NT + tid], sq[4 * NT + tid], gamma, ph[6]);
#pragma unroll
    for (int f = 0; f < 4; ++f) pl[(f * PR + ty + 3) * PC + tx + 3] = ph[3][f];
#pragma unroll
    for (int h = 0; h < HPT; ++h) {
      if (halo_in[h]) {
        double hf[4];
        const double* a = sh + h * NT + tid;
        phi_of(a[0], a[HPT * NT], a[2 * HPT * NT], a[3 * HPT * NT], a[4 * HPT * NT], gamma, hf);
#pragma unroll
        for (int f = 0; f < 4; ++f) pl[f * PR * PC + hpl[h]] = hf[f];
      }
    }
    if (k + 1 < ke) stage(k + 1);
    __syncthreads();
    // S = d(Fv^xi)/d(xi) of the PREVIOUS plane: its xi rows were written before this barrier (one barrier per step)
    if (k > kb) s_of_plane(k - 1);
    const bool do_xi = want_xi && !ok && col_in;
    const bool do_eta = want_eta && !ok && !oi && col_in;
    const bool do_zeta = want_zeta && !oi && col_in;
    if (do_xi || do_eta || do_zeta) {
      double g[3][4];
#pragma unroll
      for (int f = 0; f < 4; ++f) {
        const double* a = pl + (f * PR + ty + 3) * PC + tx + 3;
        const double dx = d6c(a[-3], a[-2], a[-1], a[1], a[2], a[3]);
        const double dy = d6c(a[-3 * PC], a[-2 * PC], a[-PC], a[PC], a[2 * PC], a[3 * PC]);
        const double dz = d6c(ph[0][f], ph[1][f], ph[2][f], ph[4][f], ph[5][f], ph[6][f]);
#pragma unroll
        for (int c = 0; c < 3; ++c) g[c][f] = J * ((kh[0][c] * dx + kh[1][c] * dy) + kh[2][c] * dz);
      }
      const double u = ph[3][0], v = ph[3][1], w = ph[3][2];
      double mu = mu0, kap = kap0;
      if (suth > 0.0) {  // mu(T) by Sutherland's law (U11): uniform branch
        const double f = sutherland_factor(ph[3][3], suth);
        mu *= f; kap *= f;
      }
      const double lam = -(2.0 / 3.0) * mu;
      const double div = g[0][0] + g[1][1] + g[2][2];
      const double txx = lam * div + 2.0 * mu * g[0][0];
      const double tyy = lam * div + 2.0 * mu * g[1][1];
      const double tzz = lam * div + 2.0 * mu * g[2][2];
      const double txy = mu * (g[1][0] + g[0][1]);
      const double txz = mu * (g[2][0] + g[0][2]);
      const double tyz = mu * (g[2][1] + g[1][2]);
      const double bx = u * txx + v * txy + w * txz + kap * g[0][3];
      const double by = u * txy + v * tyy + w * tyz + kap * g[1][3];
      const double bz = u * txz + v * tyz + w * tzz + kap * g[2][3];
      const long long p = pcol + (long long)(k + NG) * s2;
#pragma unroll
      for (int d = 0; d < 3; ++d) {
        if ((d == 0 && !do_xi) || (d == 1 && !do_eta) || (d == 2 && !do_zeta)) continue;
        const double a = kh[d][0], b = kh[d][1], c = kh[d][2];
        const double w0 = a * txx + b * txy + c * txz;
        const double w1 = a * txy + b * tyy + c * tyz;
        const double w2 = a * txz + b * tyz + c * tzz;
        const double w3 = a * bx + b * by + c * bz;
        if (d == 0) {
          double* const sx = swx + (k & 1) * (4 * NT);
          sx[(0 * VY + ty) * VX + tx] = w0; sx[(1 * VY + ty) * VX + tx] = w1;
          sx[(2 * VY + ty) * VX + tx] = w2; sx[(3 * VY + ty) * VX + tx] = w3;
        } else {
          W[(d * 4 + 0) * M + p] = w0; W[(d * 4 + 1) * M + p] = w1;
          W[(d * 4 + 2) * M + p] = w2; W[(d * 4 + 3) * M + p] = w3;
        }
      }
    }
    if (k + 1 < ke) load_metrics(k + 1);
#pragma unroll
    for (int t = 0; t < 6; ++t)
#pragma unroll
      for (int f = 0; f < 4; ++f) ph[t][f] = ph[t + 1][f];
  }
  __syncthreads();
  s_of_plane(ke - 1);
}

using G0 = VG<64, 8>;

}  // namespace

int visc_march_init() {
  return cudaFuncSetAttribute(k_visc_march<G0>, cudaFuncAttributeMaxDynamicSharedMemorySize, G0::SMEM) == cudaSuccess ? 0 : -1;
}

// S3 point fluxes of block B (default plan): S, Fv^eta rows, Fv^zeta rows into the workspace.
// Tile geometry: 64 x 8 threads.  Measured on B200 (256^3, 128^3, 8 x 96^3): 70 x 7 (12 % fewer thread-planes at 256^3),
// 54 x 9 and two 64 x 4 CTAs per SM all land within +-5 % of it -- the kernel is bound by the shared-memory pipe and the
// per-plane barrier, not by the tile's halo overhead -- so only this one is instantiated.
int launch_visc_march(cfd_ctx* c, const BlockDev& B) {
  using G = G0;
  const int TImax = G::VX - 6;
  const int ntile = (B.n[0] + TImax - 1) / TImax;
  const int TI = (B.n[0] + ntile - 1) / ntile;
  const int nk = B.n[2] + 6;
  const int rows = (B.n[1] + 6 + G::VY - 1) / G::VY;
  const int cols = ntile * rows;
  // k segments: each repeats 6 planes of priming (~3 planes' worth of time); whole waves of 148 CTAs (one CTA per SM)
  int nseg = 1;
  double best = -1.0;
  const int maxseg = nk / 24 > 0 ? nk / 24 : 1;
  for (int ns = 1; ns <= maxseg; ++ns) {
    const int ks = (nk + ns - 1) / ns, n2 = (nk + ks - 1) / ks;
    const double waves = (double)cols * n2 / (148.0 * G::MINB);
    const double eff = waves / ceil(waves) * ks / (ks + 3.0);
    if (eff > best + 1e-9) { best = eff; nseg = ns; }
  }
  const int KS = (nk + nseg - 1) / nseg;
  dim3 grid(ntile, rows, (nk + KS - 1) / KS);
  k_visc_march<G><<<grid, dim3(G::VX, G::VY), G::SMEM, c->stream>>>(B, c->pd, B.ws, TI, KS);
  c->launches++;
  return 0;
}
