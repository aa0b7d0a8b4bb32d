// Kernels for S1 (metrics/Jacobian), S4 (RK stage + residual), S5 (physical BCs), S6 (ghost fill),
// and the FP64 peak probe.  sm_100a, fp64.  P:L<n> = PAPER.md line; U<k> = DESIGN.md reading.
#include "cfd_internal.cuh"
#include "fastmath.cuh"
#include "stencil.cuh"

// =================================================================================================
// S6: ghost fill through signed index permutations (U15; P:L262 bc_block, "on GPU without
// leaving the device").  One launch fills all regions (the face -> edge -> corner chains are composed on the host,
// cfd_api.cu plan_copies); the grid is flattened over the tasks (CopyTask::cta_begin), FILL_CPT cells per thread.
// =================================================================================================
constexpr unsigned FILL_CPT = 2;   // cells per thread

template <int NV, bool SHIFT>
__global__ void __launch_bounds__(256) k_fill(const CopyTask* __restrict__ tasks, int ntasks, const BlockDev* __restrict__ blocks, int field) {
  // flattened grid: CTA b belongs to the task with the largest cta_begin <= b (tasks are sorted by cta_begin)
  int lo = 0, hi = ntasks - 1;
  while (lo < hi) {
    const int mid = (lo + hi + 1) >> 1;
    if (tasks[mid].cta_begin <= (int)blockIdx.x) lo = mid; else hi = mid - 1;
  }
  const CopyTask T = tasks[lo];
  const unsigned cta = blockIdx.x - (unsigned)T.cta_begin;
  const long long cells = (long long)T.ext[0] * T.ext[1] * T.ext[2];
  const BlockDev D = blocks[T.dst_block];
  const BlockDev S = blocks[T.src_block];
  // no __restrict__: for a self-periodic block dst and src are the same buffer (disjoint regions within a pass)
  double* dst = field == 0 ? D.q : D.xyz;
  const double* src = field == 0 ? S.q : S.xyz;
  // cells < 2^31 per region (a region is a ghost slab of one block): 32-bit index arithmetic
  const unsigned e0 = (unsigned)T.ext[0], e1 = (unsigned)T.ext[1];
  for (unsigned t = cta * (FILL_CPT * 256u) + threadIdx.x, n = 0; n < FILL_CPT && t < (unsigned)cells; ++n, t += 256u) {
    const unsigned u = t / e0;
    const int i = (int)(t - u * e0);
    const unsigned k = u / e1;
    const int j = (int)(u - k * e1);
    const int di = T.lo[0] + i, dj = T.lo[1] + j, dk = T.lo[2] + (int)k;
    const long long od = D.idx(di, dj, dk);
    const long long os = T.sbase + di * T.sstride[0] + dj * T.sstride[1] + dk * T.sstride[2];
    // all loads before the first store: dst and src may be the same buffer (no __restrict__), so the compiler would
    // otherwise keep each load behind the previous store and leave one load in flight per thread
    double val[NV];
#pragma unroll
    for (int v = 0; v < NV; ++v) val[v] = src[v * S.M + os];
#pragma unroll
    for (int v = 0; v < NV; ++v) dst[v * D.M + od] = SHIFT ? val[v] + T.shift[v] : val[v];
  }
}

int fill_ctas_of(const CopyTask& T) {
  const long long cells = (long long)T.ext[0] * T.ext[1] * T.ext[2];
  return (int)((cells + FILL_CPT * 256 - 1) / (FILL_CPT * 256));
}

int launch_fill_connect(cfd_ctx* c, int field) {
  for (int p = 1; p <= 3; ++p) {
    const size_t nt = c->tasks[p].size();
    if (!nt) continue;
    const CopyTask& L = c->tasks[p].back();
    const unsigned ctas = (unsigned)(L.cta_begin + fill_ctas_of(L));
    ProfScope ps(c, PK_FILL);
    if (field == 0) k_fill<5, false><<<ctas, 256, 0, c->stream>>>(c->d_tasks[p], (int)nt, c->d_blocks, 0);
    else k_fill<3, true><<<ctas, 256, 0, c->stream>>>(c->d_tasks[p], (int)nt, c->d_blocks, 1);
    c->launches++;
  }
  CUDA_TRY(c, cudaGetLastError());
  return CFD_OK;
}

// =================================================================================================
// Ghost coordinates behind physical faces: wall = odd reflection (U13), far field = linear
// extrapolation (U14); whole tangential extent.
// =================================================================================================
__global__ void __launch_bounds__(256) k_bc_xyz(BlockDev B, int face, int type) {
  const int an = face / 2, s = face % 2;
  const int t1 = (an + 1) % 3, t2 = (an + 2) % 3;
  const int e1 = B.m[t1], e2 = B.m[t2];
  const int t = blockIdx.x * blockDim.x + threadIdx.x;
  if (t >= e1 * e2) return;
  const int b1 = t % e1 - NG, b2 = t / e1 - NG;
  const int bnode = s == 0 ? 0 : B.n[an] - 1;
  const int dir = s == 0 ? 1 : -1;
  int p[3];
  p[t1] = b1; p[t2] = b2; p[an] = bnode;
  const long long pb = B.idx(p[0], p[1], p[2]);
  const long long sd = B.s[an] * dir;
  for (int c = 0; c < 3; ++c) {
    double* x = B.xyz + c * B.M;
    const double xb = x[pb];
    for (int g = 1; g <= NG; ++g) {
      double val;
      if (type == CFD_FACE_WALL_NOSLIP_ADIABATIC) val = 2.0 * xb - x[pb + g * sd];
      else val = xb + (double)g * (xb - x[pb + sd]);
      x[pb - g * sd] = val;
    }
  }
}

int launch_bc_xyz(cfd_ctx* c) {
  for (const BcTask& T : c->bcs) {
    const BlockDev& B = c->blk[T.block];
    const int an = T.face / 2;
    const int cells = B.m[(an + 1) % 3] * B.m[(an + 2) % 3];
    ProfScope ps(c, PK_BC);
    k_bc_xyz<<<(cells + 255) / 256, 256, 0, c->stream>>>(B, T.face, T.type);
    c->launches++;
  }
  CUDA_TRY(c, cudaGetLastError());
  return CFD_OK;
}

// =================================================================================================
// S5: physical boundary conditions on q (U13 wall, U14 far field); tangential range [-3, n+3).
// =================================================================================================
struct PrimD { double rho, u, v, w, p, c; };
__device__ __forceinline__ PrimD prims_of(const double Q[5], double gamma) {
  PrimD s;
  s.rho = Q[0];
  const double ir = 1.0 / Q[0];
  s.u = Q[1] * ir; s.v = Q[2] * ir; s.w = Q[3] * ir;
  s.p = (gamma - 1.0) * (Q[4] - 0.5 * s.rho * (s.u * s.u + s.v * s.v + s.w * s.w));
  s.c = sqrt(gamma * s.p * ir);
  return s;
}

__global__ void __launch_bounds__(128) k_bc_q(BlockDev B, ParamsDev P, int face, int type) {
  const int an = face / 2, s = face % 2;
  // tangential axes, the lower one fastest across threads (i when the face is not a xi face: coalesced)
  const int t1 = an == 0 ? 1 : 0, t2 = an == 2 ? 1 : 2;
  const int e1 = B.n[t1] + 6, e2 = B.n[t2] + 6;
  const int t = blockIdx.x * blockDim.x + threadIdx.x;
  if (t >= e1 * e2) return;
  const int b1 = t % e1 - 3, b2 = t / e1 - 3;
  const int bnode = s == 0 ? 0 : B.n[an] - 1;
  const int dir = s == 0 ? 1 : -1;
  int p[3];
  p[t1] = b1; p[t2] = b2; p[an] = bnode;
  const long long pb = B.idx(p[0], p[1], p[2]);
  const long long sd = B.s[an] * dir;
  const long long M = B.M;
  double* q = B.q;
  const double gamma = P.gamma, g1 = gamma - 1.0;
  if (type == CFD_FACE_WALL_NOSLIP_ADIABATIC) {
    double pp[5], TT[5];
    for (int l = 1; l <= 4; ++l) {
      double Q[5];
      for (int m = 0; m < 5; ++m) Q[m] = q[m * M + pb + l * sd];
      PrimD st = prims_of(Q, gamma);
      pp[l] = st.p;
      TT[l] = gamma * st.p / st.rho;
    }
    const double p0 = (48.0 * pp[1] - 36.0 * pp[2] + 16.0 * pp[3] - 3.0 * pp[4]) / 25.0;
    const double T0 = (48.0 * TT[1] - 36.0 * TT[2] + 16.0 * TT[3] - 3.0 * TT[4]) / 25.0;
    q[0 * M + pb] = gamma * p0 / T0;
    q[1 * M + pb] = 0.0; q[2 * M + pb] = 0.0; q[3 * M + pb] = 0.0;
    q[4 * M + pb] = p0 / g1;
    for (int g = 1; g <= NG; ++g) {
      const long long pg = pb - g * sd, pi = pb + g * sd;
      q[0 * M + pg] = q[0 * M + pi];
      q[1 * M + pg] = -q[1 * M + pi];
      q[2 * M + pg] = -q[2 * M + pi];
      q[3 * M + pg] = -q[3 * M + pi];
      q[4 * M + pg] = q[4 * M + pi];
    }
  } else {
    double kn[3];
    for (int c = 0; c < 3; ++c) kn[c] = B.khat[(an * 3 + c) * M + pb];
    const double kl = sqrt(kn[0] * kn[0] + kn[1] * kn[1] + kn[2] * kn[2]);
    const double so = s == 1 ? 1.0 : -1.0;
    const double nx = so * kn[0] / kl, ny = so * kn[1] / kl, nz = so * kn[2] / kl;
    double Qi[5], Qf[5];
    for (int m = 0; m < 5; ++m) { Qi[m] = q[m * M + pb + sd]; Qf[m] = P.q_inf[m]; }
    const PrimD si = prims_of(Qi, gamma), sf = prims_of(Qf, gamma);
    const double uni = si.u * nx + si.v * ny + si.w * nz;
    const double unf = sf.u * nx + sf.v * ny + sf.w * nz;
    const double Rp = uni + 2.0 * si.c / g1;
    const double Rm = unf - 2.0 * sf.c / g1;
    const double Vn = 0.5 * (Rp + Rm);
    const double cb = 0.25 * g1 * (Rp - Rm);
    double rho, u, v, w, pr;
    if (Vn >= cb) {
      rho = si.rho; u = si.u; v = si.v; w = si.w; pr = si.p;
    } else if (Vn <= -cb) {
      rho = sf.rho; u = sf.u; v = sf.v; w = sf.w; pr = sf.p;
    } else {
      const bool outflow = Vn >= 0.0;
      const PrimD sr = outflow ? si : sf;
      const double unr = outflow ? uni : unf;
      const double ent = sr.p / pow(sr.rho, gamma);
      u = sr.u + (Vn - unr) * nx; v = sr.v + (Vn - unr) * ny; w = sr.w + (Vn - unr) * nz;
      rho = pow(cb * cb / (gamma * ent), 1.0 / g1);
      pr = rho * cb * cb / gamma;
    }
    const double Qb[5] = {rho, rho * u, rho * v, rho * w, pr / g1 + 0.5 * rho * (u * u + v * v + w * w)};
    for (int m = 0; m < 5; ++m) {
      q[m * M + pb] = Qb[m];
      for (int g = 1; g <= NG; ++g) q[m * M + pb - g * sd] = Qb[m];
    }
  }
}

int launch_bc_q(cfd_ctx* c) {
  for (const BcTask& T : c->bcs) {
    const BlockDev& B = c->blk[T.block];
    const int an = T.face / 2;
    const int cells = (B.n[(an + 1) % 3] + 6) * (B.n[(an + 2) % 3] + 6);
    ProfScope ps(c, PK_BC);
    k_bc_q<<<(cells + 127) / 128, 128, 0, c->stream>>>(B, c->pd, T.face, T.type);
    c->launches++;
  }
  CUDA_TRY(c, cudaGetLastError());
  return CFD_OK;
}

// =================================================================================================
// S1: metrics and Jacobian (Eqs. 7–8), 6th-order central, conservative form.
// Pass 1: xd[c*3+d] = d x_c / d xi^d into the workspace (valid where the index along d is in
// [-3, n+3)); pass 2: khat on the box [-3, n+3)^3 from products, J from Eq. 8.
// =================================================================================================

__global__ void __launch_bounds__(256) k_metric_d1(BlockDev B, double* __restrict__ xd) {
  const long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (t >= B.M) return;
  const int i = (int)(t % B.m[0]) - NG;
  const long long u = t / B.m[0];
  const int j = (int)(u % B.m[1]) - NG;
  const int k = (int)(u / B.m[1]) - NG;
  const int id[3] = {i, j, k};
  for (int d = 0; d < 3; ++d) {
    if (id[d] < -3 || id[d] >= B.n[d] + 3) continue;
    const long long st = B.s[d];
    for (int c = 0; c < 3; ++c) {
      const double* x = B.xyz + c * B.M + t;
      xd[(c * 3 + d) * B.M + t] = d6c(x[-3 * st], x[-2 * st], x[-st], x[st], x[2 * st], x[3 * st]);
    }
  }
}

__global__ void __launch_bounds__(256) k_metric_khat(BlockDev B, const double* __restrict__ xd, int* __restrict__ flag) {
  const int e0 = B.n[0] + 6, e1 = B.n[1] + 6, e2 = B.n[2] + 6;
  const long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (t >= (long long)e0 * e1 * e2) return;
  const int i = (int)(t % e0) - 3;
  const long long u = t / e0;
  const int j = (int)(u % e1) - 3;
  const int k = (int)(u / e1) - 3;
  const long long p = B.idx(i, j, k);
  const long long M = B.M;
  for (int d = 0; d < 3; ++d)
    for (int c = 0; c < 3; ++c) {
      const int d1 = (d + 1) % 3, d2 = (d + 2) % 3, c1 = (c + 1) % 3, c2 = (c + 2) % 3;
      const double* a1 = xd + (c1 * 3 + d1) * M + p;
      const double* a2 = xd + (c1 * 3 + d2) * M + p;
      const double* x2 = B.xyz + c2 * M + p;
      const long long S1 = B.s[d1], S2 = B.s[d2];
      const double t1 = d6c(a1[-3 * S2] * x2[-3 * S2], a1[-2 * S2] * x2[-2 * S2], a1[-S2] * x2[-S2], a1[S2] * x2[S2],
                           a1[2 * S2] * x2[2 * S2], a1[3 * S2] * x2[3 * S2]);
      const double t2 = d6c(a2[-3 * S1] * x2[-3 * S1], a2[-2 * S1] * x2[-2 * S1], a2[-S1] * x2[-S1], a2[S1] * x2[S1],
                           a2[2 * S1] * x2[2 * S1], a2[3 * S1] * x2[3 * S1]);
      B.khat[(d * 3 + c) * M + p] = t1 - t2;
    }
#define XD(c, d) xd[((c) * 3 + (d)) * M + p]
  const double ji = XD(0, 0) * XD(1, 1) * XD(2, 2) - XD(0, 0) * XD(1, 2) * XD(2, 1) + XD(0, 1) * XD(1, 2) * XD(2, 0) -
                    XD(0, 1) * XD(1, 0) * XD(2, 2) + XD(0, 2) * XD(1, 0) * XD(2, 1) - XD(0, 2) * XD(1, 1) * XD(2, 0);
#undef XD
  B.jac[p] = 1.0 / ji;
  const bool interior = i >= 0 && i < B.n[0] && j >= 0 && j < B.n[1] && k >= 0 && k < B.n[2];
  if (interior && !(ji > 0.0)) atomicOr(flag, 1);
}

int launch_metrics(cfd_ctx* c) {
  for (size_t b = 0; b < c->blk.size(); ++b) {
    if (!c->is_local(b)) continue;
    const BlockDev& B = c->blk[b];
    ProfScope ps(c, PK_METRICS);
    k_metric_d1<<<(unsigned)((B.M + 255) / 256), 256, 0, c->stream>>>(B, B.ws);
    const long long box = (long long)(B.n[0] + 6) * (B.n[1] + 6) * (B.n[2] + 6);
    k_metric_khat<<<(unsigned)((box + 255) / 256), 256, 0, c->stream>>>(B, B.ws, c->d_flag);
    c->launches += 2;
  }
  CUDA_TRY(c, cudaGetLastError());
  return CFD_OK;
}

// =================================================================================================
// S4: RK stage (Eq. 20) fused with the residual sum of stage 1 (U17) over the INNER points: node
// planes owned by a physical BC (B.bcmask) are advanced like all others but left out of the sum (U17a).
// Deterministic: fixed grid, per-thread serial accumulation, fixed-shape tree in the block, then a
// single block sums the partials in index order.
// =================================================================================================
template <int STAGE>
__global__ void __launch_bounds__(256) k_rk(BlockDev B, double dt, double a, double b, double* __restrict__ partials) {
  const int ni = B.n[0], nj = B.n[1];
  const long long N = (long long)ni * nj * B.n[2];
  const long long M = B.M;
  double acc[5] = {0, 0, 0, 0, 0};
  for (long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x; t < N; t += (long long)gridDim.x * blockDim.x) {
    const int i = (int)(t % ni);
    const long long u = t / ni;
    const int j = (int)(u % nj);
    const int k = (int)(u / nj);
    const long long p = B.idx(i, j, k);
    const int bm = B.bcmask;
    const bool bc_node = STAGE == 1 && bm != 0 &&
                         (((bm & 1) && i == 0) || ((bm & 2) && i == ni - 1) || ((bm & 4) && j == 0) || ((bm & 8) && j == nj - 1) ||
                          ((bm & 16) && k == 0) || ((bm & 32) && k == B.n[2] - 1));
#pragma unroll
    for (int m = 0; m < 5; ++m) {
      const long long e = m * M + p;
      const double r = B.r[e], q = B.q[e];
      if (STAGE == 1) {
        B.qn[e] = q;
        if (!bc_node) acc[m] += r * r;
        B.q[e] = q + dt * r;
      } else {
        B.q[e] = a * B.qn[e] + b * (q + dt * r);
      }
    }
  }
  if (STAGE == 1) {
    __shared__ double sm[5][8];
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
#pragma unroll
    for (int m = 0; m < 5; ++m) {
      double v = acc[m];
      for (int o = 16; o > 0; o >>= 1) v += __shfl_down_sync(0xffffffffu, v, o);
      if (lane == 0) sm[m][wid] = v;
    }
    __syncthreads();
    if (threadIdx.x < 5) {
      double v = 0.0;
      for (int w = 0; w < 8; ++w) v += sm[threadIdx.x][w];
      partials[(long long)blockIdx.x * 5 + threadIdx.x] = v;
    }
  }
}

__global__ void k_res_final(const double* __restrict__ partials, int n, double* __restrict__ res) {
  // one warp per equation, fixed order
  const int m = threadIdx.x >> 5, lane = threadIdx.x & 31;
  if (m >= 5) return;
  double v = 0.0;
  for (int t = lane; t < n; t += 32) v += partials[(long long)t * 5 + m];
  for (int o = 16; o > 0; o >>= 1) v += __shfl_down_sync(0xffffffffu, v, o);
  if (lane == 0) res[m] = v;
}

int launch_rk(cfd_ctx* c, int stage, double dt) {
  const double a = stage == 1 ? 0.0 : (stage == 2 ? 3.0 / 4.0 : 1.0 / 3.0);
  const double b = stage == 1 ? 1.0 : (stage == 2 ? 1.0 / 4.0 : 2.0 / 3.0);
  double* partials = c->ws + ws_partials_offset_doubles(c);
  int used = 0;
  for (size_t bi = 0; bi < c->blk.size(); ++bi) {
    if (!c->is_local(bi)) continue;
    const BlockDev& B = c->blk[bi];
    const long long N = (long long)B.n[0] * B.n[1] * B.n[2];
    long long g = (N + 255) / 256;
    const int cap = rk_max_partial_blocks();
    if (g > cap) g = cap;
    ProfScope ps(c, PK_RK);
    if (stage == 1) k_rk<1><<<(unsigned)g, 256, 0, c->stream>>>(B, dt, a, b, partials + (long long)used * 5);
    else if (stage == 2) k_rk<2><<<(unsigned)g, 256, 0, c->stream>>>(B, dt, a, b, nullptr);
    else k_rk<3><<<(unsigned)g, 256, 0, c->stream>>>(B, dt, a, b, nullptr);
    used += (int)g;
    c->launches++;
  }
  if (stage == 1) {
    ProfScope ps(c, PK_RES);
    k_res_final<<<1, 160, 0, c->stream>>>(partials, used, c->d_res);
    c->launches++;
  }
  CUDA_TRY(c, cudaGetLastError());
  return CFD_OK;
}

// =================================================================================================
// FP64 FMA throughput probe (roofline denominator for the "alu" bound).
// =================================================================================================
__global__ void __launch_bounds__(256) k_dfma_probe(double* out, int iters, double a, double b) {
  double x0 = threadIdx.x * 1e-3, x1 = x0 + 1, x2 = x0 + 2, x3 = x0 + 3, x4 = x0 + 4, x5 = x0 + 5, x6 = x0 + 6, x7 = x0 + 7;
  for (int i = 0; i < iters; ++i) {
#pragma unroll
    for (int u = 0; u < 16; ++u) {
      x0 = fma(x0, a, b); x1 = fma(x1, a, b); x2 = fma(x2, a, b); x3 = fma(x3, a, b);
      x4 = fma(x4, a, b); x5 = fma(x5, a, b); x6 = fma(x6, a, b); x7 = fma(x7, a, b);
    }
  }
  out[(long long)blockIdx.x * blockDim.x + threadIdx.x] = ((x0 + x1) + (x2 + x3)) + ((x4 + x5) + (x6 + x7));
}

int launch_fp64_probe(int iters, double* tflops) {
  int dev = 0, sms = 0;
  if (cudaGetDevice(&dev) != cudaSuccess) return CFD_E_CUDA;
  cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
  const int blocks = sms * 8, threads = 256;
  double* d = nullptr;
  if (cudaMalloc(&d, sizeof(double) * blocks * threads) != cudaSuccess) return CFD_E_CUDA;
  cudaEvent_t e0, e1;
  cudaEventCreate(&e0);
  cudaEventCreate(&e1);
  k_dfma_probe<<<blocks, threads>>>(d, iters / 4 + 1, 0.999999, 1e-9);  // warm-up
  double best = 0.0;
  for (int rep = 0; rep < 3; ++rep) {
    cudaEventRecord(e0);
    k_dfma_probe<<<blocks, threads>>>(d, iters, 0.999999, 1e-9);
    cudaEventRecord(e1);
    if (cudaEventSynchronize(e1) != cudaSuccess) { cudaFree(d); return CFD_E_CUDA; }
    float ms = 0;
    cudaEventElapsedTime(&ms, e0, e1);
    const double fl = 2.0 * 8 * 16 * (double)iters * blocks * threads;
    const double tf = fl / (ms * 1e-3) / 1e12;
    if (tf > best) best = tf;
  }
  cudaEventDestroy(e0);
  cudaEventDestroy(e1);
  cudaFree(d);
  *tflops = best;
  return CFD_OK;
}

// =================================================================================================
// Self-test of fastmath.cuh (cfd_selftest_fastmath).
// =================================================================================================
__global__ void k_fastmath(int n, const double* __restrict__ x, double* __restrict__ r, double* __restrict__ s) {
  const int t = blockIdx.x * blockDim.x + threadIdx.x;
  if (t >= n) return;
  r[t] = frcp(x[t]);
  s[t] = frsqrt(x[t]);
}

int launch_fastmath_selftest(int n, const double* xh, double* rh, double* sh) {
  double* d = nullptr;
  const size_t nb = sizeof(double) * (size_t)n;
  if (cudaMalloc(&d, 3 * nb) != cudaSuccess) return CFD_E_CUDA;
  int rc = CFD_OK;
  if (cudaMemcpy(d, xh, nb, cudaMemcpyHostToDevice) != cudaSuccess) rc = CFD_E_CUDA;
  if (rc == CFD_OK) {
    k_fastmath<<<(n + 255) / 256, 256>>>(n, d, d + n, d + 2 * (size_t)n);
    if (cudaMemcpy(rh, d + n, nb, cudaMemcpyDeviceToHost) != cudaSuccess) rc = CFD_E_CUDA;
    if (rc == CFD_OK && cudaMemcpy(sh, d + 2 * (size_t)n, nb, cudaMemcpyDeviceToHost) != cudaSuccess) rc = CFD_E_CUDA;
  }
  cudaFree(d);
  return rc;
}
