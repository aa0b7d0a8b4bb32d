// S2 along xi as a marching sweep out of a per-warp CHUNK RING in shared memory (sm_100a, fp64).
// P:L<n> = PAPER.md line; U<k> = DESIGN.md reading.  Shares no code with oracle/.
//
// Marching along i puts the 32 lanes of a warp on 32 neighbouring j lines (stride m0 doubles), so per-lane loads would
// use 8 bytes of every 32-byte sector.  Here each warp owns a ring of three chunks; a chunk is 4 consecutive i positions
// (one aligned 32-byte sector per line) x 32 lines x 8 variables (Q and khat^xi), laid out densely
// ([var][line][4 positions], 32 B per line) with a 32-byte XOR swizzle (address bit 4 ^= bit 7), so that the 16-byte
// reads "my line, positions (2h, 2h+1)" of a quarter warp hit 8 distinct bank groups: conflict-free LDS.128.
// Nothing crosses warps: __syncwarp (and warp-private mbarriers in the TMA variant) only.
//   * step j reads Q at j-2..j+2 and khat at j-3..j+2 as 3-4 position pairs and computes exactly what k_march does;
//   * the output of step j (r at position j-1, array index x = j+5) is parked in shared memory and leaves in groups of
//     four positions per line.  k_xi_ldg writes SECTOR-ALIGNED groups (array indices 4c..4c+3: x = 4c, 4c+1 wait in a
//     2.5 KB side buffer, x = 4c+2, 4c+3 in the dead Q words of positions 4c, 4c+1); k_xi_tma stores the box of a whole
//     chunk (x = 4c+2..4c+5 parked in the Q words of chunk c), which straddles two half sectors per line because
//     interior position 0 sits at array index NG = 6, 16 bytes into a sector.  When a chunk's khat has been read for
//     the last time its slot is refilled with the chunk two ahead.
// Two ways to fill the ring and to write r:
//   k_xi_ldg (default)  warp-cooperative 16-byte cp.async (lane -> line l/2 + 16t, half l%2), swizzle by hand, STG.128 of
//                       full sectors;
//   k_xi_tma (plan 5)   cp.async.bulk.tensor boxes 4 x 32 x 1 x nvar with SWIZZLE_32B, TMA store; correct, but the TMA
//                       unit needs ~5 cycles per 32-byte box row on B200, which makes this variant TMA-bound.
// Array index along i: a = position + NG; chunks are a/4; segments start at multiples of 4 (interior), so a segment's
// first and last output group are half groups (masked stores).  The xi sweep runs first (r = X); the viscous xi term S is added by the eta sweep.
#include <cuda.h>

#include "cfd_internal.cuh"
#include "march_fir.cuh"
#include "sweep_math.cuh"

static_assert((NG - 2) % 4 == 0, "k_xi_tma: r groups must coincide with 32-byte chunks");

namespace {

constexpr int TW = 4;                       // warps per CTA
constexpr int PLANE = 32 * 32;              // bytes of one variable of one chunk: 32 lines x 32 B
constexpr int SLOT = 8 * PLANE;             // Q (5) + khat (3)
constexpr int WARP_BYTES = 3 * SLOT;         // ring of 3 chunks = 24 KB
constexpr int XT_SMEM = TW * WARP_BYTES + 256 /*alignment slack*/ + TW * 4 * 8 /*mbarriers*/;
constexpr int XL_WARP_BYTES = 3 * SLOT + 5 * 512;   // k_xi_ldg: ring + side buffer of parked outputs (2.5 KB)
constexpr int XL_SMEM = TW * XL_WARP_BYTES + 256;

struct XiTArgs {
  int nl, nt, n, S;     // lines (j), third extent (k), sweep length, segment length (multiple of 4)
  int nlb;              // 32-line groups per k
  double gamma, eps4;
};

__device__ __forceinline__ unsigned smem_u32(const void* p) { return (unsigned)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void mbar_init(unsigned bar, unsigned count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(unsigned bar, unsigned bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(unsigned bar, unsigned parity) {
  asm volatile(
      "{\n"
      ".reg .pred p;\n"
      "WAIT_%=:\n"
      "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
      "@p bra DONE_%=;\n"
      "bra WAIT_%=;\n"
      "DONE_%=:\n"
      "}\n" ::"r"(bar), "r"(parity)
      : "memory");
}
__device__ __forceinline__ void tma_load4(unsigned dst, const CUtensorMap* tm, unsigned bar, int c0, int c1, int c2, int c3) {
  asm volatile("cp.async.bulk.tensor.4d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%3, %4, %5, %6}], [%2];" ::"r"(dst),
               "l"(tm), "r"(bar), "r"(c0), "r"(c1), "r"(c2), "r"(c3)
               : "memory");
}
__device__ __forceinline__ void tma_store4(const CUtensorMap* tm, unsigned src, int c0, int c1, int c2, int c3) {
  asm volatile("cp.async.bulk.tensor.4d.global.shared::cta.bulk_group [%0, {%2, %3, %4, %5}], [%1];" ::"l"(tm), "r"(src), "r"(c0),
               "r"(c1), "r"(c2), "r"(c3)
               : "memory");
}
__device__ __forceinline__ void tma_commit() { asm volatile("cp.async.bulk.commit_group;" ::: "memory"); }
__device__ __forceinline__ void tma_wait_read0() { asm volatile("cp.async.bulk.wait_group.read 0;" ::: "memory"); }
__device__ __forceinline__ void tma_wait0() { asm volatile("cp.async.bulk.wait_group 0;" ::: "memory"); }
__device__ __forceinline__ void fence_async() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }

// per-warp state that survives a step (all in registers)
struct XiState {
  double acc[5][5];   // transposed-FIR accumulators (march_fir.cuh)
  double ULc[5];      // U^L_{j-1/2} from the previous step
  double Phip[5];     // Phi_{j-1/2} of the previous step
};

// One marching step at position j (array index a = j + NG, PAR = a & 1).  P0..P3: this lane's position pairs in the
// ring (16 bytes each, variable v at + v * PLANE):
//   PAR 1 (a odd):  P0 = (a-3, a-2), P1 = (a-1, a), P2 = (a+1, a+2)
//   PAR 0 (a even): P0 = (a-4, a-3), P1 = (a-2, a-1), P2 = (a, a+1), P3 = (a+2, a+3)
#define LD2(P, v) (*reinterpret_cast<const double2*>((P) + (v) * PLANE))
// SCH 0: modified AFWENO (eigen-system at point a, Fig. 11); SCH 1: original AFWENO (eigen-system at interface a-1/2,
// two complete interpolations over a-3 .. a+2, Fig. 9; NEXT-1).
// park / pstr: where the output of this step (r at array index a-1) is parked: park[m * pstr], m = 0..4.
template <int PAR, int SCH = 0>
__device__ __forceinline__ void xi_step(XiState& st, char* P0, const char* P1, const char* P2, const char* P3, bool iface, bool store,
                                        double gamma, double eps4, double* park, int pstr) {
  double Qs[5][5], UL[5], UR[5], Fc[5];
#pragma unroll
  for (int m = 0; m < 5; ++m) {
    const double2 v1 = LD2(P1, m), v2 = LD2(P2, m);
    if (PAR) {
      const double2 v0 = LD2(P0, m);
      Qs[0][m] = v0.y; Qs[1][m] = v1.x; Qs[2][m] = v1.y; Qs[3][m] = v2.x; Qs[4][m] = v2.y;
    } else {
      const double2 v3 = LD2(P3, m);
      Qs[0][m] = v1.x; Qs[1][m] = v1.y; Qs[2][m] = v2.x; Qs[3][m] = v2.y; Qs[4][m] = v3.x;
    }
  }
  if (SCH == 0) {
    double kc[3];  // khat^xi at a
#pragma unroll
    for (int c = 0; c < 3; ++c) kc[c] = PAR ? LD2(P1, 5 + c).y : LD2(P2, 5 + c).x;
    afweno_states(Qs, kc[0], kc[1], kc[2], gamma, eps4, UL, UR, Fc);
  }
  // FIR: push the point flux of a+2; output = central part of Phi_{j-1/2}
  double G[5];
  {
    double F[5], k2[3];
#pragma unroll
    for (int c = 0; c < 3; ++c) k2[c] = PAR ? LD2(P2, 5 + c).y : LD2(P3, 5 + c).x;
    point_flux(Qs[4][0], Qs[4][1], Qs[4][2], Qs[4][3], Qs[4][4], k2[0], k2[1], k2[2], gamma, F);
#pragma unroll
    for (int m = 0; m < 5; ++m) G[m] = fir_push(st.acc[m], F[m]);
  }
  if (iface) {
    // interface j-1/2: metric (U5) from khat^xi at a-3 .. a+2, both split fluxes, numerical flux
    double kh[3];
#pragma unroll
    for (int c = 0; c < 3; ++c) {
      const double2 v0 = LD2(P0, 5 + c), v1 = LD2(P1, 5 + c), v2 = LD2(P2, 5 + c);
      if (PAR) kh[c] = khalf(v0.x, v0.y, v1.x, v1.y, v2.x, v2.y);
      else kh[c] = khalf(v0.y, v1.x, v1.y, v2.x, v2.y, LD2(P3, 5 + c).x);
    }
    const double kk = fma(kh[0], kh[0], fma(kh[1], kh[1], kh[2] * kh[2]));
    const double ikn = frsqrt(kk), kn = kk * ikn;
    double Ph[5];   // Phi_{j-1/2} = G + F+ + F-: the split fluxes are accumulated onto the FIR output
#pragma unroll
    for (int m = 0; m < 5; ++m) Ph[m] = G[m];
    if (SCH == 0) {
      sw_flux<+1>(st.ULc, kh[0], kh[1], kh[2], kn, ikn, gamma, Ph);
      sw_flux<-1>(UR, kh[0], kh[1], kh[2], kn, ikn, gamma, Ph);
    } else {
      double Q6[6][5];
#pragma unroll
      for (int m = 0; m < 5; ++m) {
        Q6[0][m] = PAR ? LD2(P0, m).x : LD2(P0, m).y;  // Q at a-3
#pragma unroll
        for (int t = 0; t < 5; ++t) Q6[t + 1][m] = Qs[t][m];
      }
      afweno_iface_orig(Q6, kh[0], kh[1], kh[2], ikn, gamma, eps4, UL, UR);
      sw_flux<+1>(UL, kh[0], kh[1], kh[2], kn, ikn, gamma, Ph);
      sw_flux<-1>(UR, kh[0], kh[1], kh[2], kn, ikn, gamma, Ph);
    }
#pragma unroll
    for (int m = 0; m < 5; ++m) {
      const double Phi = Ph[m];
      if (store) park[m * pstr] = st.Phip[m] - Phi;
      st.Phip[m] = Phi;
    }
  }
  if (SCH == 0) {
#pragma unroll
    for (int m = 0; m < 5; ++m) st.ULc[m] = UL[m];
  }
}

// r = X^xi; the xi sweep runs first and carries no viscous data (the eta sweep adds S = d(Fv^xi)/d(xi)).
__global__ void __launch_bounds__(32 * TW, 2)
k_xi_tma(const __grid_constant__ CUtensorMap tq, const __grid_constant__ CUtensorMap tk, const __grid_constant__ CUtensorMap tr,
         XiTArgs A) {
  extern __shared__ char smem_raw[];
  const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
  const long long unit = (long long)blockIdx.x * TW + wid;
  const int lb = (int)(unit % A.nlb);
  const int it = (int)(unit / A.nlb);
  if (it >= A.nt) return;  // warp-uniform; the kernel has no CTA-wide barrier
  const int p0 = blockIdx.y * A.S;  // multiple of 4
  const int p1 = min(A.n, p0 + A.S);
  // shared memory: [TW] x 3 chunk slots, 256-byte aligned (the swizzle uses address bits 4 and 7)
  char* const base = smem_raw + ((256u - (smem_u32(smem_raw) & 255u)) & 255u);
  char* const ring = base + wid * WARP_BYTES;
  const unsigned bars = smem_u32(base + TW * WARP_BYTES) + wid * 32;  // full[0..2]
  const int c1 = lb * 32 + NG, c2 = it + NG;  // TMA coordinates of this warp's first line
  const int swz = (lane >> 2) & 1;
  const int off0 = lane * 32 + (swz << 4), off1 = lane * 32 + ((swz ^ 1) << 4);  // pair 0 / 1 of my line inside a plane
  auto pair_ptr = [&](int pn) -> char* {  // pn = array index >> 1
    const int ch = pn >> 1;
    return ring + (ch % 3) * SLOT + ((pn & 1) ? off1 : off0);
  };
  auto load_chunk = [&](int ch) {  // lane 0 only
    const unsigned bar = bars + (ch % 3) * 8;
    const unsigned dst = smem_u32(ring + (ch % 3) * SLOT);
    mbar_expect_tx(bar, SLOT);
    tma_load4(dst, &tq, bar, ch * 4, c1, c2, 0);
    tma_load4(dst + 5 * PLANE, &tk, bar, ch * 4, c1, c2, 0);
  };
  unsigned par_full = 0;  // phase parity to wait for, per barrier
  auto wait_chunk = [&](int ch) {
    const int s = ch % 3;
    mbar_wait(bars + s * 8, (par_full >> s) & 1u);
    par_full ^= 1u << s;
  };
  // r positions 4(ch-1) .. 4(ch-1)+3 are parked in the Q planes of chunk ch: store the box, free the slot
  auto flush = [&](int ch) {
    char* const slot = ring + (ch % 3) * SLOT;
    fence_async();
    __syncwarp();
    if (lane == 0) {
      tma_store4(&tr, smem_u32(slot), ch * 4 + 2, c1, c2, 0);
      tma_commit();
    }
  };

  if (lane == 0) {
    for (int b = 0; b < 3; ++b) mbar_init(bars + b * 8, 1);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    fence_async();
  }
  __syncwarp();
  const int a0 = p0 - 1 + NG;     // array index of the first step; a0 & 3 == 1
  const int ch0 = a0 >> 2;        // its chunk
  if (lane == 0) { load_chunk(ch0 - 1); load_chunk(ch0); load_chunk(ch0 + 1); }
  XiState st;
#pragma unroll
  for (int m = 0; m < 5; ++m) {
#pragma unroll
    for (int t = 0; t < 5; ++t) st.acc[m][t] = 0.0;
    st.ULc[m] = 0.0; st.Phip[m] = 0.0;
  }
  wait_chunk(ch0 - 1);
  wait_chunk(ch0);
  // pairs of the first step (a0 odd): P0 = (a0-3, a0-2), P1 = (a0-1, a0), P2 = (a0+1, a0+2)
  const int pb0 = (a0 - 3) >> 1;
  char* P0 = pair_ptr(pb0);
  char* P1 = pair_ptr(pb0 + 1);
  char* P2 = pair_ptr(pb0 + 2);
  char* P3 = P2;
  // prime the FIR with the point fluxes of positions p0-3 .. p0 (array a0-2 .. a0+1)
#pragma unroll
  for (int t = 0; t < 4; ++t) {
    const char* P = t == 0 ? P0 : (t == 3 ? P2 : P1);
    double v[8];
#pragma unroll
    for (int x = 0; x < 8; ++x) v[x] = (t == 0 || t == 2) ? LD2(P, x).y : LD2(P, x).x;
    double F[5];
    point_flux(v[0], v[1], v[2], v[3], v[4], v[5], v[6], v[7], A.gamma, F);
#pragma unroll
    for (int m = 0; m < 5; ++m) fir_push(st.acc[m], F[m]);
  }
  const double gamma = A.gamma, eps4 = A.eps4;
  int last3 = -1;  // last step with (a & 3) == 3
  for (int j = p0 - 1; j <= p1; j += 2) {
    const int a = j + NG;  // odd
    // ---------------- step A (a odd) ----------------
    const bool ev = (a & 3) == 3;
    if (ev) {
      // the chunk before chunk(a) holds the parked r positions j-5 .. j-2: flush it (not the first time: those
      // positions belong to the previous segment and nothing was parked)
      if (j >= p0 + 5) flush((a >> 2) - 1);
      last3 = j;
    }
    xi_step<1>(st, P0, P1, P2, P3, j >= p0, j > p0, gamma, eps4, reinterpret_cast<double*>(P0), PLANE / 8);  // parked in the Q words of position a-3
    if (ev) {
      // refill the freed slot with the chunk two ahead (if any step will read it); the TMA store issued by flush() must
      // have finished reading the slot first
      __syncwarp();
      if (lane == 0) {
        tma_wait_read0();
        const int cn = (a >> 2) + 2;
        if (cn * 4 <= p1 + NG + 2) load_chunk(cn);
      }
    }
    // ---------------- step B (a + 1 even) ----------------
    if (j + 1 <= p1) {
      const int a1 = a + 1;
      if ((a1 & 3) == 2) wait_chunk((a1 >> 2) + 1);  // position a1+2 opens the next chunk
      P3 = pair_ptr(pb0 + ((j - (p0 - 1)) >> 1) + 3);
      xi_step<0>(st, P0, P1, P2, P3, true, j + 1 > p0, gamma, eps4, reinterpret_cast<double*>(P0) + 1, PLANE / 8);
      P0 = P1; P1 = P2; P2 = P3;
    }
  }
  // ---- the last group of parked outputs: the chunk of the last (a & 3) == 3 step ----
  __syncwarp();
  flush((last3 + NG) >> 2);
  if (lane == 0) tma_wait0();
}

// ---------------------------------------------------------------------------------------------------------
// The same sweep with the ring filled by warp-cooperative 16-byte cp.async instead of TMA.  Measured on B200 the TMA
// unit spends ~5 cycles per 32-byte box row (6 B/cycle/SM), which makes the TMA variant TMA-bound (1.41 ms at 256^3);
// 16-byte LDGSTS with lane -> (line l/2 + 16t, half l%2) writes the same swizzled layout (the XOR done by hand), two
// lanes cover one sector of a line and a quarter warp writes 128 contiguous bytes.  The flush uses the same lane
// mapping: LDS.128 of the parked outputs, STG.128 to r.
struct XiLArgs {
  const double* q;    // array origin (ghosts included) of the current q
  const double* kh;   // khat^xi rows
  double* r;
  long long M, s1, s2;  // variable, j, k strides (doubles)
  XiTArgs g;
};

__device__ __forceinline__ void cp16(char* dst, const double* src) {
  asm volatile("cp.async.cg.shared.global.L2::128B [%0], [%1], 16;" ::"r"(smem_u32(dst)), "l"(src) : "memory");
}

template <int SCH>
__global__ void __launch_bounds__(32 * TW, 2) k_xi_ldg(XiLArgs L) {
  extern __shared__ char smem_raw[];
  const XiTArgs& A = L.g;
  const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
  const long long unit = (long long)blockIdx.x * TW + wid;
  const int lb = (int)(unit % A.nlb);
  const int it = (int)(unit / A.nlb);
  if (it >= A.nt) return;  // warp-uniform; the kernel has no CTA-wide barrier
  const int p0 = blockIdx.y * A.S;  // multiple of 4
  const int p1 = min(A.n, p0 + A.S);
  char* const base = smem_raw + ((256u - (smem_u32(smem_raw) & 255u)) & 255u);
  char* const ring = base + wid * XL_WARP_BYTES;
  char* const obuf = ring + 3 * SLOT;  // side buffer: the first two outputs of a sector group, [5 vars][32 lines][2 positions]
  const int swz = (lane >> 2) & 1;
  const int off0 = lane * 32 + (swz << 4), off1 = lane * 32 + ((swz ^ 1) << 4);
  auto pair_ptr = [&](int pn) -> char* { return ring + ((pn >> 1) % 3) * SLOT + ((pn & 1) ? off1 : off0); };
  // loader / flusher role: lines lsub + 16 t (t = 0, 1), half lh of the chunk
  const int lsub = lane >> 1, lh = lane & 1;
  long long goff[2];
  bool lok[2];
  int soff[2];
#pragma unroll
  for (int t = 0; t < 2; ++t) {
    const int ln = lsub + 16 * t;                     // line within the warp's group
    const int jl = lb * 32 + ln;                      // interior j of that line
    lok[t] = jl < A.nl;
    goff[t] = (long long)(it + NG) * L.s2 + (long long)(min(jl, A.nl - 1) + NG) * L.s1 + 2 * lh;
    soff[t] = ln * 32 + ((lh ^ ((ln >> 2) & 1)) << 4);
  }
  const long long M = L.M;
  auto load_chunk = [&](int ch) {
    char* const slot = ring + (ch % 3) * SLOT;
#pragma unroll
    for (int t = 0; t < 2; ++t) {
      const long long g = goff[t] + ch * 4;
#pragma unroll
      for (int m = 0; m < 5; ++m) cp16(slot + m * PLANE + soff[t], L.q + m * M + g);
#pragma unroll
      for (int cc = 0; cc < 3; ++cc) cp16(slot + (5 + cc) * PLANE + soff[t], L.kh + cc * M + g);
    }
  };
  // Outputs leave in SECTOR-ALIGNED groups: group c = r at array indices 4c .. 4c+3 (one full 32-byte sector per line).
  // Step a produces r at array index x = a-1.  x = 4c, 4c+1 are parked in the side buffer; x = 4c+2, 4c+3 in the Q words of
  // positions 4c, 4c+1 (pair 0 of chunk c: position x-2 = a-3 is dead for Q).  (Interior position 0 sits at array index
  // NG = 6, i.e. 16 bytes into a sector: writing the four outputs of a CHUNK, 4c+2 .. 4c+5, would touch two half sectors
  // per line; measured 1.13 ms against 0.81 ms for this kernel at 256^3.)
  auto flush = [&](int c, int rlo, int rhi) {  // only r positions in [rlo, rhi) are written
    const char* const slot = ring + (c % 3) * SLOT;
    const int rp = c * 4 + 2 * lh - NG;  // first of my two r positions
#pragma unroll
    for (int t = 0; t < 2; ++t) {
      if (!lok[t]) continue;
      double* const gr = L.r + goff[t] + c * 4;   // goff holds + 2 lh
      const int ln = lsub + 16 * t;
#pragma unroll
      for (int m = 0; m < 5; ++m) {
        const double2 v = lh == 0 ? *reinterpret_cast<const double2*>(obuf + m * 512 + ln * 16)
                                  : *reinterpret_cast<const double2*>(slot + m * PLANE + ln * 32 + (((ln >> 2) & 1) << 4));
        if (rp >= rlo && rp + 1 < rhi) *reinterpret_cast<double2*>(gr + m * M) = v;
        else {
          if (rp >= rlo && rp < rhi) gr[m * M] = v.x;
          if (rp + 1 >= rlo && rp + 1 < rhi) gr[m * M + 1] = v.y;
        }
      }
    }
  };
  double* const opark = reinterpret_cast<double*>(obuf + lane * 16);  // my line's two side-buffer words of variable 0

  const int a0 = p0 - 1 + NG;
  const int ch0 = a0 >> 2;
  load_chunk(ch0 - 1); load_chunk(ch0);
  asm volatile("cp.async.commit_group;" ::: "memory");
  load_chunk(ch0 + 1);
  asm volatile("cp.async.commit_group;" ::: "memory");
  XiState st;
#pragma unroll
  for (int m = 0; m < 5; ++m) {
#pragma unroll
    for (int t = 0; t < 5; ++t) st.acc[m][t] = 0.0;
    st.ULc[m] = 0.0; st.Phip[m] = 0.0;
  }
  asm volatile("cp.async.wait_group 1;" ::: "memory");
  __syncwarp();
  const int pb0 = (a0 - 3) >> 1;
  char* P0 = pair_ptr(pb0);
  char* P1 = pair_ptr(pb0 + 1);
  char* P2 = pair_ptr(pb0 + 2);
  char* P3 = P2;
#pragma unroll
  for (int t = 0; t < 4; ++t) {
    const char* P = t == 0 ? P0 : (t == 3 ? P2 : P1);
    double v[8];
#pragma unroll
    for (int x = 0; x < 8; ++x) v[x] = (t == 0 || t == 2) ? LD2(P, x).y : LD2(P, x).x;
    double F[5];
    point_flux(v[0], v[1], v[2], v[3], v[4], v[5], v[6], v[7], A.gamma, F);
#pragma unroll
    for (int m = 0; m < 5; ++m) fir_push(st.acc[m], F[m]);
  }
  const double gamma = A.gamma, eps4 = A.eps4;
  for (int j = p0 - 1; j <= p1; j += 2) {
    const int a = j + NG;  // odd
    const bool q3 = (a & 3) == 3;
    if (q3) {
      // every lane has read the last khat of the chunk before chunk(a): refill its slot with the chunk two ahead
      __syncwarp();
      const int cn = (a >> 2) + 2;
      if (cn * 4 <= p1 + NG + 2) load_chunk(cn);
      asm volatile("cp.async.commit_group;" ::: "memory");
    } else if (j >= p0 + 3) {
      // a = 4c+5: group c is complete (x = 4c+3 was parked by the previous step): write it, then the side buffer is free
      __syncwarp();
      flush((a >> 2) - 1, p0, p1);
      __syncwarp();
    }
    // this step's output x = a-1: side buffer word 0 (a = 1 mod 4) or the Q words of position a-3 (a = 3 mod 4)
    xi_step<1, SCH>(st, P0, P1, P2, P3, j >= p0, j > p0, gamma, eps4, q3 ? reinterpret_cast<double*>(P0) : opark,
                    q3 ? PLANE / 8 : 64);
    if (j + 1 <= p1) {
      const int a1 = a + 1;
      if ((a1 & 3) == 2) {  // position a1+2 opens the next chunk
        asm volatile("cp.async.wait_group 0;" ::: "memory");
        __syncwarp();
      }
      P3 = pair_ptr(pb0 + ((j - (p0 - 1)) >> 1) + 3);
      // output x = a: side buffer word 1, or the Q words of position a1-3 = a-2 (second word of pair P0)
      xi_step<0, SCH>(st, P0, P1, P2, P3, true, j + 1 > p0, gamma, eps4, q3 ? reinterpret_cast<double*>(P0) + 1 : opark + 1,
                      q3 ? PLANE / 8 : 64);
      P0 = P1; P1 = P2; P2 = P3;
    }
  }
  // ---- the last group: complete (p1 = 2 mod 4) or its first half only (p1 = 0 mod 4; the rest belongs to the next segment) ----
  asm volatile("cp.async.wait_group 0;" ::: "memory");
  __syncwarp();
  flush((p1 + NG - 1) >> 2, p0, p1);
}

#undef LD2

// ---- host side: tensor maps (one per state buffer and block, plus khat^xi and S) and the launcher ----
struct XiMaps {
  bool ok = false;
  CUtensorMap st[3];  // the caller's q, qn, r buffers (cfd_ctx::base): 4-D (i, j, k, var), box 4 x 32 x 1 x 5
  CUtensorMap kh;     // khat^xi rows: box 4 x 32 x 1 x 3
};
struct XiTmaState {
  std::vector<XiMaps> maps;
  bool ldg_ok = false;
};

typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*, const cuuint64_t*,
                                  const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave, CUtensorMapSwizzle,
                                  CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

bool encode(EncodeTiledFn fn, CUtensorMap* tm, const BlockDev& B, double* basep, int nvar) {
  const cuuint64_t dims[4] = {(cuuint64_t)B.m[0], (cuuint64_t)B.m[1], (cuuint64_t)B.m[2], (cuuint64_t)nvar};
  const cuuint64_t strides[3] = {(cuuint64_t)B.m[0] * 8, (cuuint64_t)B.m[0] * B.m[1] * 8, (cuuint64_t)B.M * 8};
  const cuuint32_t box[4] = {4, 32, 1, (cuuint32_t)nvar};
  const cuuint32_t es[4] = {1, 1, 1, 1};
  return fn(tm, CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 4, basep, dims, strides, box, es, CU_TENSOR_MAP_INTERLEAVE_NONE,
            CU_TENSOR_MAP_SWIZZLE_32B, CU_TENSOR_MAP_L2_PROMOTION_L2_128B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS;
}

}  // namespace

// Builds the tensor maps of every block whose layout TMA accepts (row pitch a multiple of 16 bytes, i.e. ni even).
// Blocks without maps use the 16-byte cp.async ring kernel (k_xi_ldg) or, for odd ni, k_march_xi instead.  Never fails: "no TMA" is a valid outcome.
void xi_tma_setup(cfd_ctx* c) {
  XiTmaState* S = new XiTmaState;
  S->maps.resize(c->blk.size());
  c->xi_tma = S;
  if (cudaFuncSetAttribute(k_xi_ldg<0>, cudaFuncAttributeMaxDynamicSharedMemorySize, XL_SMEM) != cudaSuccess ||
      cudaFuncSetAttribute(k_xi_ldg<1>, cudaFuncAttributeMaxDynamicSharedMemorySize, XL_SMEM) != cudaSuccess) {
    cudaGetLastError();
    return;
  }
  S->ldg_ok = true;
  EncodeTiledFn fn = nullptr;
  cudaDriverEntryPointQueryResult qr;
  if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", (void**)&fn, cudaEnableDefault, &qr) != cudaSuccess || !fn ||
      qr != cudaDriverEntryPointSuccess) {
    cudaGetLastError();
    return;
  }
  if (cudaFuncSetAttribute(k_xi_tma, cudaFuncAttributeMaxDynamicSharedMemorySize, XT_SMEM) != cudaSuccess) {
    cudaGetLastError();
    return;
  }
  for (size_t b = 0; b < c->blk.size(); ++b) {
    const BlockDev& B = c->blk[b];
    XiMaps& X = S->maps[b];
    if ((B.m[0] & 1) || B.n[0] < 8 || !c->is_local(b)) continue;
    bool ok = true;
    for (int t = 0; t < 3; ++t) ok = ok && encode(fn, &X.st[t], B, c->base[t][b], 5);
    ok = ok && encode(fn, &X.kh, B, B.khat, 3);
    X.ok = ok;
  }
}

void xi_tma_free(cfd_ctx* c) {
  delete static_cast<XiTmaState*>(c->xi_tma);
  c->xi_tma = nullptr;
}

bool xi_tma_ok(const cfd_ctx* c, int b) {
  const XiTmaState* S = static_cast<const XiTmaState*>(c->xi_tma);
  return S && S->maps[b].ok;
}
// the 16-byte cp.async variant needs an even row pitch (16-byte aligned position pairs) and ni >= 8
bool xi_ldg_ok(const cfd_ctx* c, int b) {
  const XiTmaState* S = static_cast<const XiTmaState*>(c->xi_tma);
  return S && S->ldg_ok && !(c->blk[b].m[0] & 1) && c->blk[b].n[0] >= 8;
}

int pick_segments(long long ctas_per_seg, int n, int quantum);

// The xi sweep of block b (r = X^xi) with the chunk-ring marching kernel; tma: fill the ring by TMA (k_xi_tma),
// else by 16-byte cp.async (k_xi_ldg, the default: the TMA unit is the bottleneck for 32-byte box rows).
int launch_xi_tma(cfd_ctx* c, int b, bool tma) {
  const XiTmaState* S = static_cast<const XiTmaState*>(c->xi_tma);
  const XiMaps& X = S->maps[b];
  const BlockDev& B = c->blk[b];
  XiTArgs A;
  A.nl = B.n[1]; A.nt = B.n[2]; A.n = B.n[0];
  A.nlb = (A.nl + 31) / 32;
  const long long units = (long long)A.nlb * A.nt;
  const long long ctas = (units + TW - 1) / TW;
  const int nseg = pick_segments(ctas * c->conc, A.n, 4);
  A.S = (((A.n + nseg - 1) / nseg) + 3) & ~3;
  A.gamma = c->pd.gamma;
  A.eps4 = 4.0 * c->pd.eps;
  dim3 grid((unsigned)ctas, (unsigned)((A.n + A.S - 1) / A.S));
  if (!tma) {
    XiLArgs L;
    L.q = B.q; L.kh = B.khat; L.r = B.r;
    L.M = B.M; L.s1 = B.s[1]; L.s2 = B.s[2];
    L.g = A;
    if (c->prm.scheme == 1) k_xi_ldg<1><<<grid, 32 * TW, XL_SMEM, c->stream>>>(L);
    else k_xi_ldg<0><<<grid, 32 * TW, XL_SMEM, c->stream>>>(L);  // the viscous xi term S is added by the eta sweep
    c->launches++;
    return 0;
  }
  const CUtensorMap& tq = X.st[c->role[0]];
  const CUtensorMap& tr = X.st[c->role[2]];
  k_xi_tma<<<grid, 32 * TW, XT_SMEM, c->stream>>>(tq, X.kh, tr, A);
  c->launches++;
  return 0;
}
