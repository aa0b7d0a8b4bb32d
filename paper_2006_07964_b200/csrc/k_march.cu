// S2 (+ the derivative half of S3) as a MARCHING sweep: one thread owns one grid line segment and walks along the
// sweep direction; lanes of a warp are neighbouring lines (coalesced when the lanes run along i: eta and zeta sweeps).
// sm_100a, fp64.  P:L<n> = PAPER.md line; U<k> = DESIGN.md reading.  Shares no code with oracle/.
//
// Why marching: with one thread per point every thread re-reads a 5-point Q stencil, a 7-point khat
// stencil and 12 neighbour fluxes -- ~170 L1/shared accesses per point against a budget of ~175 at full FP64 rate, so
// the data pipe, the issue slots and the FP64 pipe were co-limiters.  A marching thread loads each value ONCE:
//  * Q and khat of position j+3 arrive by cp.async into a thread-private 8-slot shared-memory ring while the thread
//    computes position j (no registers held, no barrier: nobody else reads the column);
//  * the interface metric khat_{j-1/2} (U5), both split fluxes of that interface and the numerical flux are formed
//    once per interface in registers;
//  * Eq. 19's central correction and the 6th-order central viscous derivative are written in flux form and evaluated
//    as ONE transposed 6-tap FIR over the point fluxes (5 running accumulators per equation in registers):
//       D_j = Phi_{j+1/2} - Phi_{j-1/2},   Phi_{j+1/2} = F+_{j+1/2} + F-_{j+1/2} + sum_t a_t F_{j-2+t} - sum_t b_t Fv_{j-2+t}
//    with a = (c3, c2+c3, c1+c2+c3, mirrored), c = (17/256, -13/320, 19/3840) (Eq. 19) and b likewise from
//    (3/4, -3/20, 1/60).  Exact identity; only the summation order differs from Eq. 19 as printed.
#include "cfd_internal.cuh"
#include "sweep_math.cuh"

namespace {

constexpr int MT = 128;     // threads per CTA
constexpr int RING = 8;     // ring slots (positions j-3 .. j+3 live, one spare)
constexpr int RV = 8;       // doubles per slot: Q (5) + khat^d (3)

struct MarchArgs {
  const double* q;      // + interior origin
  const double* kh;     // khat^d, + interior origin
  const double* W;      // viscous flux rows of direction d, + interior origin (VISC)
  const double* jac;    // + interior origin (ACC 2)
  double* r;            // + interior origin
  long long M;          // plane stride between variables
  long long sl, sm, st; // strides: neighbouring lane, one step along the sweep, third index
  int nl, nt, n, S;     // lanes, third extent, sweep length, segment length
  double gamma, eps4;
};

__device__ __forceinline__ void cp8(double* dst, const double* src) {
  const unsigned d = (unsigned)__cvta_generic_to_shared(dst);
  asm volatile("cp.async.ca.shared.global [%0], [%1], 8;" ::"r"(d), "l"(src) : "memory");
}
__device__ __forceinline__ void cp_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
template <int N>
__device__ __forceinline__ void cp_wait() { asm volatile("cp.async.wait_group %0;" ::"n"(N) : "memory"); }

// flux-form coefficients: a_t for Eq. 19's central part, b_t for the 6th-order central difference
#define A3 (19.0 / 3840.0)
#define A2 (-13.0 / 320.0 + 19.0 / 3840.0)
#define A1 (17.0 / 256.0 - 13.0 / 320.0 + 19.0 / 3840.0)
#define B3 (1.0 / 60.0)
#define B2 (-3.0 / 20.0 + 1.0 / 60.0)
#define B1 (3.0 / 4.0 - 3.0 / 20.0 + 1.0 / 60.0)

// one transposed-FIR update with the newest point flux x (and viscous xv); returns the filter output
__device__ __forceinline__ double fir_push(double acc[5], double x) {
  const double out = fma(A3, x, acc[0]);
  acc[0] = fma(A2, x, acc[1]);
  acc[1] = fma(A1, x, acc[2]);
  acc[2] = fma(A1, x, acc[3]);
  acc[3] = fma(A2, x, acc[4]);
  acc[4] = A3 * x;
  return out;
}
__device__ __forceinline__ double fir_push2(double acc[5], double x, double xv) {
  const double out = fma(-B3, xv, fma(A3, x, acc[0]));
  acc[0] = fma(-B2, xv, fma(A2, x, acc[1]));
  acc[1] = fma(-B1, xv, fma(A1, x, acc[2]));
  acc[2] = fma(-B1, xv, fma(A1, x, acc[3]));
  acc[3] = fma(-B2, xv, fma(A2, x, acc[4]));
  acc[4] = fma(-B3, xv, A3 * x);
  return out;
}

// ACC 0: r = X;  1: r += X;  2: r = J (r + X)   with X = dFv/dxi^d - D^d = -(Phi_{j+1/2} - Phi_{j-1/2})
template <int ACC, bool VISC>
__global__ void __launch_bounds__(MT, 2) k_march(MarchArgs A) {
  extern __shared__ double ring[];  // [RING][RV][MT], thread-private columns
  const int tid = threadIdx.x;
  const long long L = (long long)blockIdx.x * MT + tid;
  if (L >= (long long)A.nl * A.nt) return;  // no barriers in this kernel
  const int il = (int)(L % A.nl), it = (int)(L / A.nl);
  const int p0 = blockIdx.y * A.S;
  const int p1 = min(A.n, p0 + A.S);
  const long long base = il * A.sl + it * A.st;
  const double* __restrict__ q = A.q + base;
  const double* __restrict__ kh = A.kh + base;
  const double* __restrict__ W = VISC ? A.W + base : nullptr;
  double* __restrict__ r = A.r + base;
  const long long M = A.M, sm = A.sm;
  const double gamma = A.gamma, eps4 = A.eps4;
  double* const col = ring + tid;
#define SLOT(p) (col + (((p) + 8) & 7) * (RV * MT))
  auto fetch = [&](int p) {
    double* s = SLOT(p);
    const long long o = p * sm;
#pragma unroll
    for (int m = 0; m < 5; ++m) cp8(s + m * MT, q + m * M + o);
#pragma unroll
    for (int c = 0; c < 3; ++c) cp8(s + (5 + c) * MT, kh + c * M + o);
  };
  // ---- prologue: positions p0-4 .. p0+1 (first step j = p0-1 reads Q j-2..j+2 and khat j-3..j+2) ----
  for (int p = p0 - 4; p <= p0 + 1; ++p) fetch(p);
  cp_commit();
  double acc[5][5];
#pragma unroll
  for (int m = 0; m < 5; ++m)
#pragma unroll
    for (int t = 0; t < 5; ++t) acc[m][t] = 0.0;
  cp_wait<0>();
  // prime the FIR with the point fluxes of p0-3 .. p0 (the loop then pushes F_{j+2} at step j)
  for (int p = p0 - 3; p <= p0; ++p) {
    const double* s = SLOT(p);
    double F[5];
    point_flux(s[0], s[MT], s[2 * MT], s[3 * MT], s[4 * MT], s[5 * MT], s[6 * MT], s[7 * MT], gamma, F);
    fir_push(acc[0], F[0]);
#pragma unroll
    for (int m = 1; m < 5; ++m) {
      if (VISC) fir_push2(acc[m], F[m], W[(long long)(m - 1) * M + p * sm]);
      else fir_push(acc[m], F[m]);
    }
  }
  double ULc[5] = {0, 0, 0, 0, 0}, Phip[5] = {0, 0, 0, 0, 0};
  double wv[4] = {0, 0, 0, 0};
  if (VISC) {
#pragma unroll
    for (int m = 0; m < 4; ++m) wv[m] = W[(long long)m * M + (p0 + 1) * sm];
  }
  for (int j = p0 - 1; j <= p1; ++j) {
    // ---- prefetch position j+3 for the next step ----
    if (j < p1) fetch(j + 3);
    cp_commit();
    double wn[4] = {0, 0, 0, 0};
    if (VISC && j < p1) {
#pragma unroll
      for (int m = 0; m < 4; ++m) wn[m] = W[(long long)m * M + (long long)(j + 3) * sm];
    }
    double rold[5] = {0, 0, 0, 0, 0}, jac = 0.0;
    if (ACC >= 1 && j > p0) {
#pragma unroll
      for (int m = 0; m < 5; ++m) rold[m] = r[m * M + (long long)(j - 1) * sm];
      if (ACC == 2) jac = A.jac[base + (long long)(j - 1) * sm];
    }
    cp_wait<1>();
    // ---- point j: U^L_{j+1/2}, U^R_{j-1/2} ----
    double Qs[5][5], UL[5], UR[5], Fc[5];
#pragma unroll
    for (int s = 0; s < 5; ++s) {
      const double* sl = SLOT(j - 2 + s);
#pragma unroll
      for (int m = 0; m < 5; ++m) Qs[s][m] = sl[m * MT];
    }
    const double* sc = SLOT(j);
    afweno_states(Qs, sc[5 * MT], sc[6 * MT], sc[7 * MT], gamma, eps4, UL, UR, Fc);
    // ---- FIR: push the point flux of j+2; output = central + viscous part of Phi_{j-1/2} ----
    double G[5];
    {
      const double* s2 = SLOT(j + 2);
      double F[5];
      point_flux(Qs[4][0], Qs[4][1], Qs[4][2], Qs[4][3], Qs[4][4], s2[5 * MT], s2[6 * MT], s2[7 * MT], gamma, F);
      G[0] = fir_push(acc[0], F[0]);
#pragma unroll
      for (int m = 1; m < 5; ++m) G[m] = VISC ? fir_push2(acc[m], F[m], wv[m - 1]) : fir_push(acc[m], F[m]);
    }
    if (j >= p0) {
      // ---- interface j-1/2: metric (U5), both split fluxes, numerical flux ----
      const double *k0 = SLOT(j - 3), *k1 = SLOT(j - 2), *k2 = SLOT(j - 1), *k4 = SLOT(j + 1), *k5 = SLOT(j + 2);
      const double kx = khalf(k0[5 * MT], k1[5 * MT], k2[5 * MT], sc[5 * MT], k4[5 * MT], k5[5 * MT]);
      const double ky = khalf(k0[6 * MT], k1[6 * MT], k2[6 * MT], sc[6 * MT], k4[6 * MT], k5[6 * MT]);
      const double kz = khalf(k0[7 * MT], k1[7 * MT], k2[7 * MT], sc[7 * MT], k4[7 * MT], k5[7 * MT]);
      const double kk = fma(kx, kx, fma(ky, ky, kz * kz));
      const double ikn = frsqrt(kk), kn = kk * ikn;
      double Fp[5], Fm[5];
      sw_flux<+1>(ULc, kx, ky, kz, kn, ikn, gamma, Fp);
      sw_flux<-1>(UR, kx, ky, kz, kn, ikn, gamma, Fm);
#pragma unroll
      for (int m = 0; m < 5; ++m) {
        const double Phi = (Fp[m] + Fm[m]) + G[m];
        if (j > p0) {
          const double X = Phip[m] - Phi;
          double* rp = r + m * M + (long long)(j - 1) * sm;
          if (ACC == 0) *rp = X;
          else if (ACC == 1) *rp = rold[m] + X;
          else *rp = jac * (rold[m] + X);
        }
        Phip[m] = Phi;
      }
    }
#pragma unroll
    for (int m = 0; m < 5; ++m) ULc[m] = UL[m];
    if (VISC) {
#pragma unroll
      for (int m = 0; m < 4; ++m) wv[m] = wn[m];
    }
  }
#undef SLOT
}


template <int ACC>
void launch_march_t(cfd_ctx* c, const MarchArgs& A, bool visc) {
  const long long lanes = (long long)A.nl * A.nt;
  dim3 grid((unsigned)((lanes + MT - 1) / MT), (unsigned)((A.n + A.S - 1) / A.S));
  const size_t smem = sizeof(double) * RING * RV * MT;
  if (visc) k_march<ACC, true><<<grid, MT, smem, c->stream>>>(A);
  else k_march<ACC, false><<<grid, MT, smem, c->stream>>>(A);
}

}  // namespace

int march_init() {
  cudaError_t e = cudaSuccess;
  const int smem = (int)(sizeof(double) * RING * RV * MT);
#define OPT(A)                                                                                                      \
  if (e == cudaSuccess) e = cudaFuncSetAttribute(k_march<A, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem); \
  if (e == cudaSuccess) e = cudaFuncSetAttribute(k_march<A, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem);
  OPT(0) OPT(1) OPT(2)
#undef OPT
  return e == cudaSuccess ? 0 : -1;
}

// One marching sweep of block B along dir (0 xi, 1 eta, 2 zeta) with accumulation mode acc.
int launch_march(cfd_ctx* c, const BlockDev& B, int dir, int acc) {
  const bool visc = c->pd.viscous != 0;
  const long long o0 = B.idx(0, 0, 0);
  MarchArgs A;
  A.q = B.q + o0;
  A.kh = B.khat + (long long)(dir * 3) * B.M + o0;
  A.W = visc ? c->ws + (long long)(dir * 4) * B.M + o0 : nullptr;
  A.jac = B.jac + o0;
  A.r = B.r + o0;
  A.M = B.M;
  const int la = dir == 0 ? 1 : 0;                   // lane axis: i, except for the xi sweep (j)
  const int ta = dir == 2 ? 1 : 2;                   // third axis
  A.sl = B.s[la]; A.sm = B.s[dir]; A.st = B.s[ta];
  A.nl = B.n[la]; A.nt = B.n[ta]; A.n = B.n[dir];
  // segment length: enough CTAs for ~4 waves of 148 SMs x 2 CTAs, segments of at least 16 points
  const long long lanes = (long long)A.nl * A.nt;
  const long long ctas_per_seg = (lanes + MT - 1) / MT;
  long long nseg = (148LL * 2 * 4 + ctas_per_seg - 1) / ctas_per_seg;
  const long long maxseg = A.n / 16 > 0 ? A.n / 16 : 1;
  if (nseg > maxseg) nseg = maxseg;
  if (nseg < 1) nseg = 1;
  A.S = (int)((A.n + nseg - 1) / nseg);
  A.gamma = c->pd.gamma;
  A.eps4 = 4.0 * c->pd.eps;
  if (acc == 0) launch_march_t<0>(c, A, visc);
  else if (acc == 1) launch_march_t<1>(c, A, visc);
  else launch_march_t<2>(c, A, visc);
  c->launches++;
  return 0;
}
