// S3 up to the point fluxes as ONE k-marching kernel.   sm_100a, fp64.
// P:L<n> = PAPER.md line; U<k> = DESIGN.md reading.  Shares no code with oracle/.
//
// A CTA owns a tile of (i, j) columns and marches along k:
//   * phi = (u, v, w, T) is computed from Q on the fly and never stored;
//   * the zeta stencil lives in REGISTERS: each thread keeps phi of its own column at k-3 .. k+3 (28 doubles).  The k loop
//     is unrolled SEVEN times with the register names rotating, so the pipeline is never shifted (the shifts were 36 of the
//     ~735 instructions of a step);
//   * the (i, j) plane of phi at k (tile + halo of 3 in j, 6 in i) lives in SHARED memory, double buffered: the xi and
//     eta stencils read it with LDS;
//   * Q of plane k+4 and the halo cells of plane k+1 arrive by cp.async in thread-private shared-memory slots one step
//     ahead (no registers held across a step); the ten metric values of plane k+1 are loaded at the end of step k, when few
//     registers are live;
//   * the xi rows of the flux go to shared memory and come back as S = d(Fv^xi)/d(xi).
// Addressing: one 32-bit element offset per thread (its column at the current plane) on top of per-row base pointers that
// arrive as kernel parameters: one IMAD.WIDE per global access.  (With 64-bit offsets recomputed from the block
// descriptor the compiler, capped at 128 registers, rematerialised ~200 integer instructions per step.)  Columns that
// stick out of the array are clamped onto its last column instead of predicated: they compute and never store.
// Output (workspace rows): W[0..3] = S on interior points; W[4..7] = Fv^eta rows 2..5 on (i, k) interior, j in [-3, nj+3);
// W[8..11] = Fv^zeta rows 2..5 on (i, j) interior, k in [-3, nk+3).
#include "cfd_internal.cuh"
#include "fastmath.cuh"
#include "stencil.cuh"
#include <cmath>
#include <type_traits>

namespace {

// Tile geometry: VX x VY threads own the columns i0-3 .. i0+VX-4 of the rows j0 .. j0+VY-1; VX-6 of them are output columns.
// The plane row pitch PC is congruent to VX modulo 16 doubles, so that consecutive threads (also across a row change
// inside a warp when VX is not a multiple of 32) hit consecutive banks.  Every thread stages at most one halo cell.
template <int VX_, int VY_>
struct VG {
  static constexpr int VX = VX_, VY = VY_;
  static constexpr int PC = VX + 16;          // plane columns i0-6 .. i0+VX-1 (VX + 6), padded
  static constexpr int PR = VY + 6;           // plane rows j0-3 .. j0+VY+2
  static constexpr int NHALO = 2 * 3 * VX + 2 * 3 * VY;
  static constexpr int NT = VX * VY;
  static constexpr int MINB = NT <= 256 ? 2 : 1;      // CTAs per SM (128 registers per thread either way)
  static_assert(NT <= 512 && NHALO <= NT, "k_visc_march: tile geometry");
  // shared memory (doubles): phi planes [2][4][PR][PC] | xi rows [2][4][VY][VX] | Q stage [5][NT] | halo stage [5][NT]
  static constexpr int SM_PLANE = 4 * PR * PC, SM_WXB = 4 * NT;
  static constexpr int SM_PHI = 2 * SM_PLANE, SM_WX = 2 * SM_WXB, SM_Q = 5 * NT, SM_H = 5 * NT;
  static constexpr int SMEM = (SM_PHI + SM_WX + SM_Q + SM_H) * 8;
};

// Row base pointers (array origin) and sizes: everything the kernel reads from its parameters
struct ViscArgs {
  const double* q[5];
  const double* kh[9];
  const double* jac;
  double* w[12];
  int n[3], m[3];
  unsigned s1, s2;    // row and plane pitch in doubles
  int TI, KS;
  double gamma, mu, kappa, suth;
};

// thread roles, packed in one register
constexpr unsigned F_XI = 1u, F_ETA = 2u, F_ZETA = 4u, F_S = 8u, F_ANY = 16u, F_HALO = 32u;

// phi = (u, v, w, T = gamma p / rho) from the conservative state
__device__ __forceinline__ void phi_of(double r, double m1, double m2, double m3, double e, double gamma, double f[4]) {
  const double ir = frcp(r);
  const double u = m1 * ir, v = m2 * ir, w = m3 * ir;
  const double pr = (gamma - 1.0) * fma(-0.5 * r, fma(u, u, fma(v, v, w * w)), e);
  f[0] = u; f[1] = v; f[2] = w; f[3] = (gamma * pr) * ir;
}

template <class G>
__global__ void __launch_bounds__(G::NT, G::MINB) k_visc_march(const __grid_constant__ ViscArgs A) {
  constexpr int VX = G::VX, VY = G::VY, PC = G::PC, PR = G::PR, NHALO = G::NHALO, NT = G::NT;
  extern __shared__ double vsm[];
  double* const sphi = vsm;                 // [2][4][PR][PC]
  double* const swx = sphi + G::SM_PHI;     // [2][4][VY][VX]
  double* const sq = swx + G::SM_WX;        // [5][NT]
  double* const sh = sq + G::SM_Q;          // [5][NT]
  const int tx = threadIdx.x, ty = threadIdx.y, tid = ty * VX + tx;
  const int i0 = blockIdx.x * A.TI, j0 = -3 + (int)blockIdx.y * VY;
  const int kb = -3 + (int)blockIdx.z * A.KS, ke = min(kb + A.KS, A.n[2] + 3);
  const int i = i0 - 3 + tx, j = j0 + ty;
  const unsigned s2 = A.s2;
  const double gamma = A.gamma;
  unsigned flags = 0;
  unsigned p;      // element offset of my column at the current plane
  int dh = 0;      // my halo cell's column minus my own (elements)
  int hpl = 0;     // my halo cell inside one field of the plane
  {
    const bool col_in = (i + NG < A.m[0]) && (j + NG < A.m[1]);
    const bool oi = i < 0 || i >= A.n[0], oj = j < 0 || j >= A.n[1];
    const bool own = tx >= 3 && tx < A.TI + 3 && i < A.n[0];                     // point-wise outputs are mine
    const bool want_xi = tx < A.TI + 6 && i < A.n[0] + 3 && !oj;                  // xi rows (k interior)
    const bool want_eta = own && j < A.n[1] + 3;                                  // eta rows (k interior)
    const bool want_zeta = own && !oj;                                            // zeta rows (all k of the march)
    if (col_in && want_xi) flags |= F_XI;
    if (col_in && want_eta) flags |= F_ETA;
    if (col_in && want_zeta) flags |= F_ZETA | F_S;
    if (col_in && (want_xi || want_eta || want_zeta) && !(oi && oj)) flags |= F_ANY;
    const int ic = min(i, A.m[0] - NG - 1), jc = min(j, A.m[1] - NG - 1);         // clamped onto the array
    const unsigned pc = (unsigned)(jc + NG) * A.s1 + (unsigned)(ic + NG);
    p = pc + (unsigned)(kb + NG) * s2;
    // my halo cell of the plane (if any): top band, bottom band, left columns, right columns
    int hc = -1, hr = 0;
    if (tid < 3 * VX) { hr = tid / VX; hc = 3 + tid % VX; }
    else if (tid < 6 * VX) { hr = VY + 3 + (tid - 3 * VX) / VX; hc = 3 + tid % VX; }
    else if (tid < 6 * VX + 3 * VY) { hr = 3 + (tid - 6 * VX) / 3; hc = (tid - 6 * VX) % 3; }
    else if (tid < NHALO) { hr = 3 + (tid - 6 * VX - 3 * VY) / 3; hc = VX + 3 + (tid - 6 * VX - 3 * VY) % 3; }
    const int hi = i0 - 6 + hc, hj = j0 - 3 + hr;
    if (hc >= 0 && hi + NG >= 0 && hi + NG < A.m[0] && hj + NG >= 0 && hj + NG < A.m[1]) {
      flags |= F_HALO;
      dh = (int)((unsigned)(hj + NG) * A.s1 + (unsigned)(hi + NG)) - (int)pc;
      hpl = hr * PC + hc;
    }
  }
  double* const myq = sq + tid;
  double* const myh = sh + tid;
  double* const mypl = sphi + (ty + 3) * PC + tx + 3;   // my own cell in field 0 of plane buffer 0
  double* const mywx = swx + ty * VX + tx;              // my xi-row cell, row 0 of buffer 0

  // cp.async for the step of the plane at offset pp: Q three planes further of my column, my halo cell of that plane
  auto stage = [&](unsigned pp) {
    const unsigned o = pp + 3u * s2;
#pragma unroll
    for (int m = 0; m < 5; ++m) cp8(myq + m * NT, A.q[m] + o);
    if (flags & F_HALO) {
      const unsigned oh = pp + (unsigned)dh;
#pragma unroll
      for (int m = 0; m < 5; ++m) cp8(myh + m * NT, A.q[m] + oh);
    }
    cp_commit();
  };
  double kh[3][3], J = 0.0;
#pragma unroll
  for (int d = 0; d < 3; ++d)
#pragma unroll
    for (int c = 0; c < 3; ++c) kh[d][c] = 0.0;
  auto load_metrics = [&](unsigned pp) {
    if (flags & F_ANY) {
#pragma unroll
      for (int d = 0; d < 3; ++d)
#pragma unroll
        for (int c = 0; c < 3; ++c) kh[d][c] = __ldg(A.kh[d * 3 + c] + pp);
      J = __ldg(A.jac + pp);
    }
  };

  // ---- prologue: phi of my column at kb-3 .. kb+2 (pipeline slots 0 .. 5 of rotation 0) ----
  double ph[7][4];
#pragma unroll
  for (int t = 0; t < 6; ++t) {
    const unsigned o = p + (unsigned)(t - 3) * s2;
    phi_of(A.q[0][o], A.q[1][o], A.q[2][o], A.q[3][o], A.q[4][o], gamma, ph[t]);
  }
#pragma unroll
  for (int f = 0; f < 4; ++f) ph[6][f] = 0.0;
  stage(p);
  load_metrics(p);
  const double mu0 = A.mu, kap0 = A.kappa, suth = A.suth;
  unsigned par = 0;   // plane / xi-row buffer of the current step

  // S = d(Fv^xi)/d(xi) of the plane whose xi rows sit in buffer b, stored at offset pp
  auto s_of_plane = [&](unsigned b, unsigned pp) {
    const double* a = mywx + b * G::SM_WXB;
#pragma unroll
    for (int m = 0; m < 4; ++m, a += NT) A.w[m][pp] = d6c(a[-3], a[-2], a[-1], a[1], a[2], a[3]);
  };

  // One plane step; R = rotation of the register pipeline: plane k-3+t lives in ph[(t + R) % 7].
  // prev_in / cur_in: plane k-1 / k is an interior plane (uniform).
  auto step = [&](auto Rc, bool prev_in, bool cur_in, bool more) {
    constexpr int R = decltype(Rc)::value;
    double(&c0)[4] = ph[(0 + R) % 7]; double(&c1)[4] = ph[(1 + R) % 7]; double(&c2)[4] = ph[(2 + R) % 7];
    double(&c3)[4] = ph[(3 + R) % 7]; double(&c4)[4] = ph[(4 + R) % 7]; double(&c5)[4] = ph[(5 + R) % 7];
    double(&c6)[4] = ph[(6 + R) % 7];
    cp_wait<0>();
    double* const pl = mypl + par * G::SM_PLANE;
    // ---- newest plane of my column into the register pipeline; plane k (my own phi and my halo cell) into shared memory ----
    phi_of(myq[0], myq[NT], myq[2 * NT], myq[3 * NT], myq[4 * NT], gamma, c6);
#pragma unroll
    for (int f = 0; f < 4; ++f) pl[f * PR * PC] = c3[f];
    if (flags & F_HALO) {
      double hf[4];
      phi_of(myh[0], myh[NT], myh[2 * NT], myh[3 * NT], myh[4 * NT], gamma, hf);
      double* const hp = sphi + par * G::SM_PLANE + hpl;
#pragma unroll
      for (int f = 0; f < 4; ++f) hp[f * PR * PC] = hf[f];
    }
    if (more) stage(p + s2);
    __syncthreads();
    // S of the PREVIOUS plane: its xi rows were written before this barrier (one barrier per step)
    if (prev_in && (flags & F_S)) s_of_plane(par ^ 1u, p - s2);
    const bool do_xi = cur_in && (flags & F_XI);
    const bool do_eta = cur_in && (flags & F_ETA);
    const bool do_zeta = (flags & F_ZETA) != 0;
    if (do_xi || do_eta || do_zeta) {
      double g[3][4];
#pragma unroll
      for (int f = 0; f < 4; ++f) {
        const double* a = pl + f * PR * PC;
        const double dx = d6c(a[-3], a[-2], a[-1], a[1], a[2], a[3]);
        const double dy = d6c(a[-3 * PC], a[-2 * PC], a[-PC], a[PC], a[2 * PC], a[3 * PC]);
        const double dz = d6c(c0[f], c1[f], c2[f], c4[f], c5[f], c6[f]);
#pragma unroll
        for (int c = 0; c < 3; ++c) g[c][f] = J * ((kh[0][c] * dx + kh[1][c] * dy) + kh[2][c] * dz);
      }
      const double u = c3[0], v = c3[1], w = c3[2];
      double mu = mu0, kap = kap0;
      if (suth > 0.0) {  // mu(T) by Sutherland's law (U11): uniform branch
        const double f = sutherland_factor(c3[3], suth);
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
#pragma unroll
      for (int d = 0; d < 3; ++d) {
        if ((d == 0 && !do_xi) || (d == 1 && !do_eta) || (d == 2 && !do_zeta)) continue;
        const double a = kh[d][0], b = kh[d][1], c = kh[d][2];
        const double w0 = a * txx + b * txy + c * txz;
        const double w1 = a * txy + b * tyy + c * tyz;
        const double w2 = a * txz + b * tyz + c * tzz;
        const double w3 = a * bx + b * by + c * bz;
        if (d == 0) {
          double* const sx = mywx + par * G::SM_WXB;
          sx[0] = w0; sx[NT] = w1; sx[2 * NT] = w2; sx[3 * NT] = w3;
        } else {
          A.w[d * 4 + 0][p] = w0; A.w[d * 4 + 1][p] = w1;
          A.w[d * 4 + 2][p] = w2; A.w[d * 4 + 3][p] = w3;
        }
      }
    }
    if (more) load_metrics(p + s2);
    p += s2;
    par ^= 1u;
  };

  const int n2 = A.n[2];
  int k = kb;
#define VSTEP(R)                                                                                                    \
  step(std::integral_constant<int, R>{}, (unsigned)(k - 1) < (unsigned)n2 && k > kb, (unsigned)k < (unsigned)n2, k + 1 < ke); \
  ++k;
  while (true) {
    VSTEP(0) if (k >= ke) break;
    VSTEP(1) if (k >= ke) break;
    VSTEP(2) if (k >= ke) break;
    VSTEP(3) if (k >= ke) break;
    VSTEP(4) if (k >= ke) break;
    VSTEP(5) if (k >= ke) break;
    VSTEP(6) if (k >= ke) break;
  }
#undef VSTEP
  __syncthreads();
  if ((unsigned)(ke - 1) < (unsigned)n2 && (flags & F_S)) s_of_plane(par ^ 1u, p - s2);
}

using G0 = VG<64, 8>;
using G1 = VG<70, 7>;
using G2 = VG<54, 9>;

}  // namespace

int visc_march_init() {
  if (cudaFuncSetAttribute(k_visc_march<G1>, cudaFuncAttributeMaxDynamicSharedMemorySize, G1::SMEM) != cudaSuccess) return -1;
  if (cudaFuncSetAttribute(k_visc_march<G2>, cudaFuncAttributeMaxDynamicSharedMemorySize, G2::SMEM) != cudaSuccess) return -1;
  return cudaFuncSetAttribute(k_visc_march<G0>, cudaFuncAttributeMaxDynamicSharedMemorySize, G0::SMEM) == cudaSuccess ? 0 : -1;
}

// S3 point fluxes of block B (default plan): S, Fv^eta rows, Fv^zeta rows into the workspace.
// Three tile geometries are instantiated (G0 = 64 x 8, G1 = 70 x 7, G2 = 54 x 9 threads; bit-equal results).  They land
// within +-5 % of each other on B200 (256^3, 128^3, 8 x 96^3) -- the kernel is bound by the shared-memory pipe and the
// per-plane barrier, not by the tile's halo overhead -- so launch_visc_march picks, per block, the one with the fewest
// thread-planes (visc_thread_planes below) unless cfd_set_visc_tile fixes it.
template <class G>
static long long visc_thread_planes(const BlockDev& B) {
  const int TImax = G::VX - 6;
  const long long ntile = (B.n[0] + TImax - 1) / TImax, rows = (B.n[1] + 6 + G::VY - 1) / G::VY;
  return ntile * rows * G::NT;
}
template <class G>
static int launch_visc_march_g(cfd_ctx* c, const BlockDev& B);

// Tile geometry: the one with the fewest thread-planes for this block (64 x 8, 70 x 7 or 54 x 9 threads: 58, 64 or 48
// output columns per tile row; measured at 256^3: 1.005 / 1.031 / 1.103 ms, at 128^3: 0.166 / 0.180 / 0.159 ms);
// cfd_set_visc_tile forces one (tests, measurements).
int launch_visc_march(cfd_ctx* c, const BlockDev& B) {
  const int force = c->visc_tile;
  const long long t0 = visc_thread_planes<G0>(B), t1 = visc_thread_planes<G1>(B), t2 = visc_thread_planes<G2>(B);
  int g = 0;
  if (t1 < t0 && t1 <= t2) g = 1;
  else if (t2 < t0 && t2 < t1) g = 2;
  if (force >= 0) g = force;
  return g == 1 ? launch_visc_march_g<G1>(c, B) : (g == 2 ? launch_visc_march_g<G2>(c, B) : launch_visc_march_g<G0>(c, B));
}

template <class G>
static int launch_visc_march_g(cfd_ctx* c, const BlockDev& B) {
  if (B.M + 2 >= (1LL << 32)) { c->err = "k_visc_march: block too large for 32-bit element offsets"; return CFD_E_ARG; }
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
  ViscArgs A;
  for (int m = 0; m < 5; ++m) A.q[m] = B.q + (long long)m * B.M;
  for (int m = 0; m < 9; ++m) A.kh[m] = B.khat + (long long)m * B.M;
  A.jac = B.jac;
  for (int m = 0; m < 12; ++m) A.w[m] = B.ws + (long long)m * B.M;
  for (int a = 0; a < 3; ++a) { A.n[a] = B.n[a]; A.m[a] = B.m[a]; }
  A.s1 = (unsigned)B.s[1]; A.s2 = (unsigned)B.s[2];
  A.TI = TI; A.KS = KS;
  A.gamma = c->pd.gamma; A.mu = c->pd.mu; A.kappa = c->pd.kappa; A.suth = c->pd.suth;
  dim3 grid(ntile, rows, (nk + KS - 1) / KS);
  k_visc_march<G><<<grid, dim3(G::VX, G::VY), G::SMEM, c->stream>>>(A);
  c->launches++;
  return 0;
}
