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
#include "march_fir.cuh"
#include "stencil.cuh"
#include <cmath>

namespace {

constexpr int MT = 128;     // threads per CTA
#ifndef MINB
#define MINB 2
#endif
constexpr int RING = 8;     // ring slots (positions j-3 .. j+3 live, one spare)
constexpr int RV = 8;       // doubles per slot: Q (5) + khat^d (3)

struct MarchArgs {
  const double* q;      // + interior origin
  const double* kh;     // khat^d, + interior origin
  const double* W;      // viscous flux rows of direction d, + interior origin (VISC)
  const double* jac;    // + interior origin (ACC 2)
  const double* qn;     // q^n + interior origin (ACC 3, stages 2 and 3)
  const double* Sx;     // SX: S = d(Fv^xi)/d(xi) rows 2..5 (k_visc_march), + interior origin
  double* r;            // + interior origin
  double* partials;     // ACC 3 stage 1: 5 partial sums of R_m^2 per CTA
  long long M;          // plane stride between variables
  long long sl, sm, st; // strides: neighbouring lane, one step along the sweep, third index
  int nl, nt, n, S;     // lanes, third extent, sweep length, segment length
  double gamma, eps4;
  double dt, rk_a, rk_b; // ACC 3 (Eq. 20)
  int bcm;              // ACC 3 stage 1 (U17a): node planes owned by a physical BC, left out of the residual sum: bit 0 / 1 lane index
                        // 0 / nl-1, bit 2 / 3 third index 0 / nt-1, bit 4 / 5 sweep position 0 / n-1
};

// ACC 0: r = X;  1: r += X;  2: r = J (r + X);  3: the RK stage fused into the last sweep (Eq. 20):
//   with R = J (r + X):  out = a q^n + b (q + dt R)  written to the r buffer (the caller then exchanges the roles of the
//   q and r buffers; q itself cannot be overwritten while neighbouring threads still read it).  ST1 (stage 1):
//   a = 0, b = 1, q^n is not read (the old q buffer becomes q^n by the same exchange) and the CTA writes its
//   partial sums of R_m^2 (U17; fixed order: run-to-run deterministic).
//   X = dFv/dxi^d - D^d = -(Phi_{j+1/2} - Phi_{j-1/2}).
// Every operand arrives through thread-private shared-memory columns filled by cp.async one step ahead (Q, khat of
// position j+3; the viscous rows of j+3; old r, J, q^n of the output position): nothing is held in registers across
// a step, which is what the register allocation of this kernel (~250 registers, 2 CTAs per SM) needs.
template <int ACC, bool ST1, bool SX>
struct OutCfg {
  static constexpr int O_R = 0;                                  // old r (5), ACC >= 1
  static constexpr int O_J = ACC >= 1 ? 5 : 0;                   // J (1), ACC >= 2
  static constexpr int O_QN = O_J + (ACC >= 2 ? 1 : 0);          // q^n (5), ACC 3 stages 2, 3
  static constexpr int O_S = O_QN + ((ACC == 3 && !ST1) ? 5 : 0);  // S = d(Fv^xi)/d(xi) rows 2..5 (4), SX
  static constexpr int NOUT = O_S + (SX ? 4 : 0);
};
template <int ACC, bool VISC, bool ST1, bool SX>
constexpr int march_smem_doubles() {
  return (RING * RV + (VISC ? 8 : 0) + 2 * OutCfg<ACC, ST1, SX>::NOUT + ((ACC == 3 && ST1) ? 5 : 0)) * MT;
}

// SX (with ACC >= 1): the viscous xi term S written by k_visc_march is added to r here (the xi sweep runs first
// and knows nothing about viscosity).
// SCH: 0 = modified AFWENO (Fig. 11: eigen-system at the point, shared beta), 1 = original AFWENO (Fig. 9, NEXT-1:
// eigen-system at the interface, two complete interpolations over j-3 .. j+2; sweep_math.cuh afweno_iface_orig).
template <int ACC, bool VISC, bool ST1, bool SX, int SCH>
__global__ void __launch_bounds__(MT, MINB) k_march(MarchArgs A) {
  extern __shared__ double ring[];  // thread-private columns: [RING][RV][MT] | W [2][4][MT] | out operands [2][NOUT][MT] | res [5][MT]
  using OC = OutCfg<ACC, ST1, SX>;
  constexpr int NOUT = OC::NOUT;
  const int tid = threadIdx.x;
  const long long L = (long long)blockIdx.x * MT + tid;
  const bool live = L < (long long)A.nl * A.nt;
  double* const col = ring + tid;
  double* const wcol = col + RING * RV * MT;
  double* const ocol = wcol + (VISC ? 8 : 0) * MT;
  double* const rcol = ocol + 2 * NOUT * MT;
  if (ACC == 3 && ST1) {
#pragma unroll
    for (int m = 0; m < 5; ++m) rcol[m * MT] = 0.0;
  }
  if (live) {
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
#define SLOT(p) (col + (((p) + 8) & 7) * (RV * MT))
    auto fetch = [&](int p) {
      double* s = SLOT(p);
      const long long o = p * sm;
#pragma unroll
      for (int m = 0; m < 5; ++m) cp8(s + m * MT, q + m * M + o);
#pragma unroll
      for (int c = 0; c < 3; ++c) cp8(s + (5 + c) * MT, kh + c * M + o);
    };
    auto fetch_w = [&](int p) {
      double* s = wcol + (p & 1) * (4 * MT);
      const long long o = p * sm;
#pragma unroll
      for (int m = 0; m < 4; ++m) cp8(s + m * MT, W + m * M + o);
    };
    auto fetch_out = [&](int p) {  // operands of the output at position p
      double* s = ocol + (p & 1) * (NOUT * MT);
      const long long o = p * sm;
      if (ACC >= 1) {
#pragma unroll
        for (int m = 0; m < 5; ++m) cp8(s + (OC::O_R + m) * MT, r + m * M + o);
      }
      if (ACC >= 2) cp8(s + OC::O_J * MT, A.jac + base + o);
      if (ACC == 3 && !ST1) {
#pragma unroll
        for (int m = 0; m < 5; ++m) cp8(s + (OC::O_QN + m) * MT, A.qn + base + m * M + o);
      }
      if (SX) {
#pragma unroll
        for (int m = 0; m < 4; ++m) cp8(s + (OC::O_S + m) * MT, A.Sx + base + m * M + o);
      }
    };
    // ---- prologue: positions p0-4 .. p0+1 (first step j = p0-1 reads Q j-2..j+2 and khat j-3..j+2) ----
    for (int p = p0 - 4; p <= p0 + 1; ++p) fetch(p);
    if (VISC) fetch_w(p0 + 1);
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
#pragma unroll 2
    for (int j = p0 - 1; j <= p1; ++j) {
      // ---- prefetch for the next step: Q, khat, W of position j+3; operands of the output at position j ----
      if (j < p1) {
        fetch(j + 3);
        if (VISC) fetch_w(j + 3);
        if (NOUT > 0 && j >= p0) fetch_out(j);
      }
      cp_commit();
      cp_wait<1>();
      // ---- point j: U^L_{j+1/2}, U^R_{j-1/2} (SCH 0); SCH 1 forms both states of interface j-1/2 further down ----
      double Qs[5][5], UL[5], UR[5], Fc[5];
#pragma unroll
      for (int s = 0; s < 5; ++s) {
        const double* sl = SLOT(j - 2 + s);
#pragma unroll
        for (int m = 0; m < 5; ++m) Qs[s][m] = sl[m * MT];
      }
      const double* sc = SLOT(j);
      if (SCH == 0) afweno_states(Qs, sc[5 * MT], sc[6 * MT], sc[7 * MT], gamma, eps4, UL, UR, Fc);
      // ---- FIR: push the point flux of j+2; output = central + viscous part of Phi_{j-1/2} ----
      double G[5];
      {
        const double* s2 = SLOT(j + 2);
        const double* sw = wcol + ((j + 2) & 1) * (4 * MT);
        double F[5];
        point_flux(Qs[4][0], Qs[4][1], Qs[4][2], Qs[4][3], Qs[4][4], s2[5 * MT], s2[6 * MT], s2[7 * MT], gamma, F);
        G[0] = fir_push(acc[0], F[0]);
#pragma unroll
        for (int m = 1; m < 5; ++m) G[m] = VISC ? fir_push2(acc[m], F[m], sw[(m - 1) * MT]) : fir_push(acc[m], F[m]);
      }
      if (j >= p0) {
        // ---- interface j-1/2: metric (U5), both split fluxes, numerical flux ----
        const double *k0 = SLOT(j - 3), *k1 = SLOT(j - 2), *k2 = SLOT(j - 1), *k4 = SLOT(j + 1), *k5 = SLOT(j + 2);
        const double kx = khalf(k0[5 * MT], k1[5 * MT], k2[5 * MT], sc[5 * MT], k4[5 * MT], k5[5 * MT]);
        const double ky = khalf(k0[6 * MT], k1[6 * MT], k2[6 * MT], sc[6 * MT], k4[6 * MT], k5[6 * MT]);
        const double kz = khalf(k0[7 * MT], k1[7 * MT], k2[7 * MT], sc[7 * MT], k4[7 * MT], k5[7 * MT]);
        const double kk = fma(kx, kx, fma(ky, ky, kz * kz));
        const double ikn = frsqrt(kk), kn = kk * ikn;
        double Ph[5];   // Phi_{j-1/2} = G + F+ + F-: the split fluxes are accumulated onto the FIR output
#pragma unroll
        for (int m = 0; m < 5; ++m) Ph[m] = G[m];
        if (SCH == 0) {
          sw_flux<+1>(ULc, kx, ky, kz, kn, ikn, gamma, Ph);
          sw_flux<-1>(UR, kx, ky, kz, kn, ikn, gamma, Ph);
        } else {
          double Q6[6][5];
#pragma unroll
          for (int m = 0; m < 5; ++m) {
            Q6[0][m] = k0[m * MT];
#pragma unroll
            for (int s = 0; s < 5; ++s) Q6[s + 1][m] = Qs[s][m];
          }
          afweno_iface_orig(Q6, kx, ky, kz, ikn, gamma, eps4, UL, UR);
          sw_flux<+1>(UL, kx, ky, kz, kn, ikn, gamma, Ph);
          sw_flux<-1>(UR, kx, ky, kz, kn, ikn, gamma, Ph);
        }
        const double* so = ocol + ((j - 1) & 1) * (NOUT * MT);
        double jac = 0.0;
        if (ACC >= 2 && j > p0) jac = so[OC::O_J * MT];
        // U17a: output position j-1 on a node plane a zeta-face BC owns (A.bcm sits in the constant bank: no register)
        const bool bc_pos = ACC == 3 && ST1 && (((A.bcm & 16) && j - 1 == 0) || ((A.bcm & 32) && j - 1 == A.n - 1));
#pragma unroll
        for (int m = 0; m < 5; ++m) {
          const double Phi = Ph[m];
          if (j > p0) {
            const double X = Phip[m] - Phi;
            double* rp = r + m * M + (long long)(j - 1) * sm;
            if (ACC == 0) *rp = X;
            else if (ACC == 1) *rp = (SX && m > 0) ? (so[(OC::O_R + m) * MT] + so[(OC::O_S + m - 1) * MT]) + X : so[(OC::O_R + m) * MT] + X;
            else if (ACC == 2) *rp = jac * (so[(OC::O_R + m) * MT] + X);
            else {
              const double R = jac * (so[(OC::O_R + m) * MT] + X);
              const double qc = k2[m * MT];  // Q_m at position j-1
              if (ST1) {
                if (!bc_pos) rcol[m * MT] += R * R;
                *rp = qc + A.dt * R;
              } else {
                *rp = A.rk_a * so[(OC::O_QN + m) * MT] + A.rk_b * (qc + A.dt * R);
              }
            }
          }
          Phip[m] = Phi;
        }
      }
      if (SCH == 0) {
#pragma unroll
        for (int m = 0; m < 5; ++m) ULc[m] = UL[m];
      }
    }
#undef SLOT
  }
  if (ACC == 3 && ST1) {
    // U17a: a whole line on a node plane that a physical BC owns (lane / third index at a WALL / FARFIELD face) contributes
    // nothing; decided here, after the march, so that no flag lives in a register across the loop
    if (live && (A.bcm & 15)) {
      const int il = (int)(L % A.nl), it = (int)(L / A.nl);
      if (((A.bcm & 1) && il == 0) || ((A.bcm & 2) && il == A.nl - 1) || ((A.bcm & 4) && it == 0) || ((A.bcm & 8) && it == A.nt - 1)) {
#pragma unroll
        for (int m = 0; m < 5; ++m) rcol[m * MT] = 0.0;
      }
    }
    // fixed-order partial sums of R_m^2 over this CTA's points
    __shared__ double swr[5][MT / 32];
    const int lane = tid & 31, wid = tid >> 5;
#pragma unroll
    for (int m = 0; m < 5; ++m) {
      double v = rcol[m * MT];
      for (int o = 16; o > 0; o >>= 1) v += __shfl_down_sync(0xffffffffu, v, o);
      if (lane == 0) swr[m][wid] = v;
    }
    __syncthreads();
    if (tid < 5) {
      double v = 0.0;
      for (int w = 0; w < MT / 32; ++w) v += swr[tid][w];
      A.partials[((long long)blockIdx.y * gridDim.x + blockIdx.x) * 5 + tid] = v;
    }
  }
}

// ---------------------------------------------------------------------------------------------------------
// The xi sweep as a marching sweep with WARP-PRIVATE TRANSPOSED STAGING.  Marching along i puts the lanes of a warp
// on neighbouring j lines (stride m0 doubles): a per-lane load would use 8 of every 32-byte sector.  Instead the warp
// loads, for its 32 lines, aligned chunks of 4 consecutive i positions (one full 32-byte sector per line and
// variable; lane -> (line l/4 + 8t, position l%4)) with cp.async into a per-line ring in shared memory (line stride
// odd: the consumer's reads, all lanes at the same offset, are conflict-free), and every lane then marches along its
// own line out of shared memory exactly like k_march.  Nothing crosses warps: only __syncwarp.
//   ring per line: Q (5) + khat^xi (3) x XR = 10 positions, viscous rows (4) x XW = 5 positions -> 100 doubles (+1 pad);
//   chunk [c, c+4) is issued at step j = c-3 (its slots, positions c-10..c-7, died at step c-4) and awaited at c-2.
// The output of step j (r at position j-1) is parked in the Q slots of position j-3 (dead: Q is read at j-2..j+2 only)
// and written out by the same lane mapping as the loads, four positions = one full sector per line at a time, just
// before those slots are refilled; the flush applies the accumulation mode (r = X, r += X, r = J (r + X)).
constexpr int XR = 10;
constexpr int XLS = 8 * XR + 1;  // 81 doubles per line
constexpr int XWARPS = 4;

struct XiArgs {
  const double* q;      // + interior origin
  const double* kh;
  double* r;
  long long M;          // plane stride between variables
  long long sl, st;     // strides: neighbouring line (lane axis), third index; the sweep runs along stride 1
  int nl, nt, n, S;     // lines, third extent, sweep length, segment length
  int nlb;              // number of 32-line groups per third index
  int ph;               // chunk phase: chunk starts c = ph (mod 4) are 32-byte aligned in memory
  double gamma, eps4;
};

__device__ __forceinline__ int wrap10(int s) { return s >= XR ? s - XR : s; }

__global__ void __launch_bounds__(32 * XWARPS, 2) k_march_xi(XiArgs A) {
  extern __shared__ double ring[];
  const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
  const long long unit = (long long)blockIdx.x * XWARPS + wid;
  const int lb = (int)(unit % A.nlb);
  const long long it = unit / A.nlb;
  if (it >= A.nt) return;  // warp-uniform; no CTA barriers in this kernel
  const int p0 = blockIdx.y * A.S;
  const int p1 = min(A.n, p0 + A.S);
  double* const wbase = ring + wid * (32 * XLS);
  double* const my = wbase + lane * XLS;
  const int l0 = lb * 32;
  const long long M = A.M;
  const double gamma = A.gamma, eps4 = A.eps4;
  // loader / flusher role of this lane: lines l0 + lsub + 8t (t = 0..3), position (chunk start) + lpos
  const int lsub = lane >> 2, lpos = lane & 3;
  const long long tbase = it * A.st;
  long long goff[4];
  bool lok[4];
#pragma unroll
  for (int t = 0; t < 4; ++t) {
    const int ln = l0 + lsub + 8 * t;
    lok[t] = ln < A.nl;
    goff[t] = tbase + (long long)min(ln, A.nl - 1) * A.sl;
  }
  double* const lbase = wbase + lsub * XLS;  // + t * 8 * XLS
  const int qlo = p0 - 4, qhi = p1 + 2;

  auto load_chunk = [&](int c) {
    const int pos = c + lpos;
    if (pos >= qlo && pos <= qhi) {
      const int s = (pos + 2 * XR) % XR;
#pragma unroll
      for (int t = 0; t < 4; ++t) {
        double* d = lbase + t * 8 * XLS + s;
        const double* gq = A.q + goff[t] + pos;
        const double* gk = A.kh + goff[t] + pos;
#pragma unroll
        for (int m = 0; m < 5; ++m) cp8(d + m * XR, gq + m * M);
#pragma unroll
        for (int cc = 0; cc < 3; ++cc) cp8(d + (5 + cc) * XR, gk + cc * M);
      }
    }
  };
  // write out the parked outputs of r positions g .. g+3 (parked in the Q slots of positions g-2 .. g+1)
  auto flush = [&](int g) {
    const int pos = g + lpos;
    if (pos >= p0 && pos < p1) {
      const int s = (pos - 2 + 2 * XR) % XR;
#pragma unroll
      for (int t = 0; t < 4; ++t) {
        if (!lok[t]) continue;
        const double* sX = lbase + t * 8 * XLS + s;
        double* gr = A.r + goff[t] + pos;
#pragma unroll
        for (int m = 0; m < 5; ++m) gr[m * M] = sX[m * XR];
      }
    }
  };

  // ---- prologue: every chunk that starts at or before p0+1 (positions < p0-4 masked out) ----
  {
    int c = p0 - 4;
    c -= ((c - A.ph) & 3);  // align down to the chunk phase
    for (; c <= p0 + 1; c += 4) load_chunk(c);
    cp_commit();
  }
  double acc[5][5];
#pragma unroll
  for (int m = 0; m < 5; ++m)
#pragma unroll
    for (int t = 0; t < 5; ++t) acc[m][t] = 0.0;
  cp_wait<0>();
  __syncwarp();
  int s0 = (p0 - 1 - 3 + 2 * XR) % XR;  // slot of position j-3 at the first step j = p0-1
  // prime the FIR with the point fluxes of p0-3 .. p0 (slots s0+1 .. s0+4)
#pragma unroll
  for (int t = 0; t < 4; ++t) {
    const double* s = my + wrap10(s0 + 1 + t);
    double F[5];
    point_flux(s[0], s[XR], s[2 * XR], s[3 * XR], s[4 * XR], s[5 * XR], s[6 * XR], s[7 * XR], gamma, F);
    fir_push(acc[0], F[0]);
#pragma unroll
    for (int m = 1; m < 5; ++m) fir_push(acc[m], F[m]);
  }
  double ULc[5] = {0, 0, 0, 0, 0}, Phip[5] = {0, 0, 0, 0, 0};
  for (int j = p0 - 1; j <= p1; ++j) {
    if (((j + 3 - A.ph) & 3) == 0) {  // chunk c = j+3: flush the outputs parked in its slots, then refill them
      __syncwarp();
      flush(j + 3 - 8);
      load_chunk(j + 3);
      cp_commit();
    } else if (((j + 2 - A.ph) & 3) == 0) {
      cp_wait<0>();
      __syncwarp();
    }
    const double* sl0 = my + s0;
    const double* sl1 = my + wrap10(s0 + 1);
    const double* sl2 = my + wrap10(s0 + 2);
    const double* sl3 = my + wrap10(s0 + 3);
    const double* sl4 = my + wrap10(s0 + 4);
    const double* sl5 = my + wrap10(s0 + 5);
    // ---- point j: U^L_{j+1/2}, U^R_{j-1/2} ----
    double Qs[5][5], UL[5], UR[5], Fc[5];
#pragma unroll
    for (int m = 0; m < 5; ++m) {
      Qs[0][m] = sl1[m * XR]; Qs[1][m] = sl2[m * XR]; Qs[2][m] = sl3[m * XR]; Qs[3][m] = sl4[m * XR]; Qs[4][m] = sl5[m * XR];
    }
    afweno_states(Qs, sl3[5 * XR], sl3[6 * XR], sl3[7 * XR], gamma, eps4, UL, UR, Fc);
    // ---- FIR: push the point flux of j+2; output = central + viscous part of Phi_{j-1/2} ----
    double G[5];
    {
      double F[5];
      point_flux(Qs[4][0], Qs[4][1], Qs[4][2], Qs[4][3], Qs[4][4], sl5[5 * XR], sl5[6 * XR], sl5[7 * XR], gamma, F);
      G[0] = fir_push(acc[0], F[0]);
#pragma unroll
      for (int m = 1; m < 5; ++m) G[m] = fir_push(acc[m], F[m]);
    }
    if (j >= p0) {
      // ---- interface j-1/2: metric (U5), both split fluxes, numerical flux ----
      const double kx = khalf(sl0[5 * XR], sl1[5 * XR], sl2[5 * XR], sl3[5 * XR], sl4[5 * XR], sl5[5 * XR]);
      const double ky = khalf(sl0[6 * XR], sl1[6 * XR], sl2[6 * XR], sl3[6 * XR], sl4[6 * XR], sl5[6 * XR]);
      const double kz = khalf(sl0[7 * XR], sl1[7 * XR], sl2[7 * XR], sl3[7 * XR], sl4[7 * XR], sl5[7 * XR]);
      const double kk = fma(kx, kx, fma(ky, ky, kz * kz));
      const double ikn = frsqrt(kk), kn = kk * ikn;
      double Ph[5];
#pragma unroll
      for (int m = 0; m < 5; ++m) Ph[m] = G[m];
      sw_flux<+1>(ULc, kx, ky, kz, kn, ikn, gamma, Ph);
      sw_flux<-1>(UR, kx, ky, kz, kn, ikn, gamma, Ph);
      double* park = my + s0;  // Q slots of position j-3
#pragma unroll
      for (int m = 0; m < 5; ++m) {
        const double Phi = Ph[m];
        if (j > p0) park[m * XR] = Phip[m] - Phi;
        Phip[m] = Phi;
      }
    }
#pragma unroll
    for (int m = 0; m < 5; ++m) ULc[m] = UL[m];
    s0 = wrap10(s0 + 1);
  }
  // ---- flush what is still parked: groups after the last one flushed in the loop ----
  __syncwarp();
  {
    // in-loop flushes covered groups g = j+3-8 for the issue steps j <= p1, i.e. g <= p1-5 on the chunk phase
    int g = p1 - 5;
    g -= ((g - A.ph) & 3);  // last group flushed in the loop (or earlier than any output)
    for (g += 4; g < p1; g += 4) flush(g);
  }
}

}  // namespace

// Segment count along the sweep: enough CTAs to fill 148 SMs x 2 resident CTAs, as few partial waves as possible,
// segments of at least 16 points (each segment repeats ~1.5 steps of prologue work), lengths a multiple of quantum.
int pick_segments(long long ctas_per_seg, int n, int quantum) {
  const int maxseg = n / 16 > 0 ? n / 16 : 1;
  const double slots = 148.0 * 2.0;
  int best = 1;
  double best_eff = -1.0;
  for (int ns = 1; ns <= maxseg; ++ns) {
    int S = (n + ns - 1) / ns;
    S = ((S + quantum - 1) / quantum) * quantum;
    const int nseg = (n + S - 1) / S;
    const double waves = (double)(ctas_per_seg * nseg) / slots;
    const double eff = waves / ceil(waves) * ((double)n / (double)(nseg * (S + 1.5)));
    if (eff > best_eff + 1e-9) { best_eff = eff; best = ns; }
  }
  return best;
}

namespace {

template <int ACC, bool VISC, bool ST1, bool SX = false, int SCH = 0>
void launch_march_k(cfd_ctx* c, const MarchArgs& A) {
  const long long lanes = (long long)A.nl * A.nt;
  dim3 grid((unsigned)((lanes + MT - 1) / MT), (unsigned)((A.n + A.S - 1) / A.S));
  const size_t smem = sizeof(double) * march_smem_doubles<ACC, VISC, ST1, SX>();
  k_march<ACC, VISC, ST1, SX, SCH><<<grid, MT, smem, c->stream>>>(A);
}

template <int ACC, bool VISC, bool ST1, bool SX = false, int SCH = 0>
cudaError_t march_attr() {
  return cudaFuncSetAttribute(k_march<ACC, VISC, ST1, SX, SCH>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                              (int)(sizeof(double) * march_smem_doubles<ACC, VISC, ST1, SX>()));
}

}  // namespace

int march_init() {
  cudaError_t e = cudaSuccess;
#define OPT(A, S)                                          \
  if (e == cudaSuccess) e = march_attr<A, true, S>();      \
  if (e == cudaSuccess) e = march_attr<A, false, S>();
  OPT(2, false) OPT(3, false) OPT(3, true)
#undef OPT
  if (e == cudaSuccess) e = march_attr<1, true, false, true>();
  if (e == cudaSuccess) e = march_attr<1, false, false, false>();
  // scheme 1 (original AFWENO): the kernels of the default plan only
  if (e == cudaSuccess) e = march_attr<0, false, false, false, 1>();
  if (e == cudaSuccess) e = march_attr<1, true, false, true, 1>();
  if (e == cudaSuccess) e = march_attr<1, false, false, false, 1>();
#define OPT1(A, S)                                                      \
  if (e == cudaSuccess) e = march_attr<A, true, S, false, 1>();         \
  if (e == cudaSuccess) e = march_attr<A, false, S, false, 1>();
  OPT1(2, false) OPT1(3, false) OPT1(3, true)
#undef OPT1
  const int smx = (int)(sizeof(double) * XWARPS * 32 * XLS);
  if (e == cudaSuccess) e = cudaFuncSetAttribute(k_march_xi, cudaFuncAttributeMaxDynamicSharedMemorySize, smx);
  return e == cudaSuccess ? 0 : -1;
}

// One marching sweep of block B along dir (0 xi, 1 eta, 2 zeta) with accumulation mode acc (0..2), or, with rk != null,
// the last sweep fused with the RK stage (acc 3): the new state goes to B.r; *rk_ctas receives the number of CTAs
// (= partial-sum groups written to rk->partials at stage 1).
// no_rows: the sweep differentiates no viscous flux rows even in a viscous run (the xi sweep of the default plan).
int launch_march(cfd_ctx* c, const BlockDev& B, int dir, int acc, const RkFuse* rk, int* rk_ctas, bool sx, bool no_rows) {
  const bool visc = c->pd.viscous != 0 && !no_rows;
  const long long o0 = B.idx(0, 0, 0);
  MarchArgs A;
  A.q = B.q + o0;
  A.kh = B.khat + (long long)(dir * 3) * B.M + o0;
  A.W = visc ? B.ws + (long long)(dir * 4) * B.M + o0 : nullptr;
  A.jac = B.jac + o0;
  A.qn = B.qn + o0;
  A.Sx = B.ws + o0;
  A.r = B.r + o0;
  A.partials = rk ? rk->partials : nullptr;
  A.dt = rk ? rk->dt : 0.0; A.rk_a = rk ? rk->a : 0.0; A.rk_b = rk ? rk->b : 0.0;
  A.M = B.M;
  const int la = dir == 0 ? 1 : 0;                   // lane axis: i, except for the xi sweep (j)
  const int ta = dir == 2 ? 1 : 2;                   // third axis
  A.sl = B.s[la]; A.sm = B.s[dir]; A.st = B.s[ta];
  A.nl = B.n[la]; A.nt = B.n[ta]; A.n = B.n[dir];
  A.bcm = ((B.bcmask >> (2 * la)) & 3) | (((B.bcmask >> (2 * ta)) & 3) << 2) | (((B.bcmask >> (2 * dir)) & 3) << 4);
  const long long lanes = (long long)A.nl * A.nt;
  const long long ctas_per_seg = (lanes + MT - 1) / MT;
  int nseg = pick_segments(ctas_per_seg * c->conc, A.n, 1);
  if (rk && rk->stage == 1) {
    while (nseg > 1 && ctas_per_seg * nseg > rk->max_ctas) --nseg;
    if (ctas_per_seg * nseg > rk->max_ctas) { c->err = "fused RK stage: block too large for the residual partials"; return CFD_E_WORKSPACE; }
  }
  A.S = (A.n + nseg - 1) / nseg;
  A.gamma = c->pd.gamma;
  A.eps4 = 4.0 * c->pd.eps;
  if (rk_ctas) *rk_ctas = (int)(ctas_per_seg * ((A.n + A.S - 1) / A.S));
#define GO(AC, ST)                                           \
  do {                                                       \
    if (visc) launch_march_k<AC, true, ST>(c, A);            \
    else launch_march_k<AC, false, ST>(c, A);                \
  } while (0)
#define GO1(AC, ST)                                          \
  do {                                                       \
    if (visc) launch_march_k<AC, true, ST, false, 1>(c, A);  \
    else launch_march_k<AC, false, ST, false, 1>(c, A);      \
  } while (0)
  if (c->prm.scheme == 1) {  // original AFWENO (NEXT-1): default plan only (launch_rhs checks)
    if (rk) { if (rk->stage == 1) GO1(3, true); else GO1(3, false); }
    else if (acc == 0) launch_march_k<0, false, false, false, 1>(c, A);
    else if (acc == 1 && sx && visc) launch_march_k<1, true, false, true, 1>(c, A);
    else if (acc == 1) launch_march_k<1, false, false, false, 1>(c, A);
    else GO1(2, false);
  }
  else if (rk) { if (rk->stage == 1) GO(3, true); else GO(3, false); }
  else if (acc == 1 && sx && visc) launch_march_k<1, true, false, true>(c, A);
  else if (acc == 1 && !visc) launch_march_k<1, false, false, false>(c, A);
  else if (acc == 2) GO(2, false);
  else { c->err = "launch_march: this accumulation mode is not instantiated"; return CFD_E_ARG; }
#undef GO
#undef GO1
  c->launches++;
  return 0;
}

// The xi sweep of block B (r = X^xi) as a staged marching sweep (k_march_xi): blocks with odd ni and plan 4.
int launch_march_xi(cfd_ctx* c, const BlockDev& B) {
  const long long o0 = B.idx(0, 0, 0);
  XiArgs A;
  A.q = B.q + o0;
  A.kh = B.khat + o0;
  A.r = B.r + o0;
  A.M = B.M;
  A.sl = B.s[1]; A.st = B.s[2];
  A.nl = B.n[1]; A.nt = B.n[2]; A.n = B.n[0];
  A.nlb = (A.nl + 31) / 32;
  A.ph = (4 - (NG & 3)) & 3;
  const long long units = (long long)A.nlb * A.nt;
  const int nseg = pick_segments((units + XWARPS - 1) / XWARPS * c->conc, A.n, 1);
  A.S = (A.n + nseg - 1) / nseg;
  A.gamma = c->pd.gamma;
  A.eps4 = 4.0 * c->pd.eps;
  dim3 grid((unsigned)((units + XWARPS - 1) / XWARPS), (unsigned)((A.n + A.S - 1) / A.S));
  k_march_xi<<<grid, 32 * XWARPS, sizeof(double) * XWARPS * 32 * XLS, c->stream>>>(A);
  c->launches++;
  return 0;
}
