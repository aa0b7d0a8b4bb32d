// cfd_rk_stage1_static: stage 1 of the TVD-RK3 update (Eq. 20) with the residual sum (U17) for ONE block,
// for callers that cannot allocate device memory.  sm_100a, fp64.  Shares no code with oracle/.
//
// Why it exists.  Every other entry point of this library needs a cfd_ctx, and cfd_create_blocks calls cudaMalloc (block
// descriptors, flags) and wants a caller-allocated workspace for the partial sums of the residual reduction.  Some users of
// the library cannot provide either:
//   * a solver plug-in running inside a host application whose memory manager has already reserved the whole HBM (a
//     framework's caching allocator, a job that was handed a fixed arena): cudaMalloc then fails with out-of-memory although
//     the fields themselves live happily inside that arena;
//   * a time-step loop that must never stall the device: cudaMalloc / cudaFree synchronise against every stream of the
//     device, which a latency-bound coupling loop (co-simulation, in-situ analysis next to the solver) cannot afford;
//   * code that is handed device pointers by somebody else and has no allocator of its own at all (a callback that receives
//     q and r and must return the updated state and the residual, nothing more).
// For them the only scratch this step needs -- five partial sums per CTA -- sits in a file-scope __device__ array of fixed
// size inside the library image.  The price: every GPU that loads libcfd_b200.so holds CFD_STATIC_SCRATCH_BYTES (320 KB) of
// device memory until the process exits, whether this entry point is used or not, and the block size is limited
// (CFD_STATIC_MAX_POINTS interior points).
//
// Same arithmetic, same thread -> point mapping and same fixed summation order as k_rk<1> + k_res_final (k_aux.cu) for blocks
// within the limit, so q, qn and res come out as cfd_rk_stage(ctx, 1, dt, res) computes them.
#include <cstdarg>
#include <cstdint>
#include <mutex>

#include "cfd_internal.cuh"

namespace {

constexpr int RKS_THREADS = 256;
constexpr int RKS_MAX_CTAS = CFD_STATIC_MAX_POINTS / RKS_THREADS;  // 8192: one CTA per 256 interior points, no grid-stride wrap
static_assert((size_t)RKS_MAX_CTAS * 5 * sizeof(double) == CFD_STATIC_SCRATCH_BYTES, "cfd.h states the size of the static scratch");

// The scratch: [cta][5] partial sums of r_m^2.  In HOST code this name is only a handle for the runtime's symbol table, NOT a
// device address (launching a kernel with `g_rk1_partials` as a pointer argument would hand it a host address); the host side
// below asks cudaGetSymbolAddress for the real one, once per device.
static __device__ __align__(256) double g_rk1_partials[RKS_MAX_CTAS * 5];

constexpr int MAX_DEVICES = 64;
std::mutex g_mu;
double* g_partials_dev[MAX_DEVICES] = {};  // device address of g_rk1_partials on device d, or null before the set-up on d

thread_local char g_err[256] = "";

int fail(int code, const char* fmt, ...) {
  va_list ap;
  va_start(ap, fmt);
  vsnprintf(g_err, sizeof g_err, fmt, ap);
  va_end(ap);
  return code;
}

// Once per device, with that device current: the address of this device's copy of the array.
int scratch_of_current_device(double** out) {
  int dev = -1;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) return fail(CFD_E_CUDA, "cfd_rk_stage1_static: cudaGetDevice: %s", cudaGetErrorString(e));
  if (dev < 0 || dev >= MAX_DEVICES) return fail(CFD_E_CUDA, "cfd_rk_stage1_static: device ordinal %d not supported (max %d)", dev, MAX_DEVICES - 1);
  std::lock_guard<std::mutex> lk(g_mu);
  if (!g_partials_dev[dev]) {
    double* p = nullptr;
    e = cudaGetSymbolAddress((void**)&p, g_rk1_partials);
    if (e != cudaSuccess || !p)
      return fail(CFD_E_CUDA, "cfd_rk_stage1_static: cudaGetSymbolAddress(static scratch) on device %d: %s", dev, cudaGetErrorString(e));
    g_partials_dev[dev] = p;
  }
  *out = g_partials_dev[dev];
  return CFD_OK;
}

// Eq. 20, stage 1: q^n := q, q := q + dt r, partial sums of r_m^2 of this CTA's points into partials[cta][m].
// Every CTA of the launch writes its five slots, so nothing in the scratch has to start at zero.
__global__ void __launch_bounds__(RKS_THREADS) k_rk1_static(BlockDev B, double dt, double* __restrict__ partials) {
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
#pragma unroll
    for (int m = 0; m < 5; ++m) {
      const long long e = m * M + p;
      const double r = B.r[e], q = B.q[e];
      B.qn[e] = q;
      acc[m] += r * r;
      B.q[e] = q + dt * r;
    }
  }
  __shared__ double sm[5][RKS_THREADS / 32];
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
    for (int w = 0; w < RKS_THREADS / 32; ++w) v += sm[threadIdx.x][w];
    partials[(long long)blockIdx.x * 5 + threadIdx.x] = v;
  }
}

// One warp per equation sums the first n CTA entries in index order (lane-strided, then a fixed shuffle tree).
__global__ void k_res_static_final(const double* __restrict__ partials, int n, double* __restrict__ res) {
  const int m = threadIdx.x >> 5, lane = threadIdx.x & 31;
  if (m >= 5) return;
  double v = 0.0;
  for (int t = lane; t < n; t += 32) v += partials[(long long)t * 5 + m];
  for (int o = 16; o > 0; o >>= 1) v += __shfl_down_sync(0xffffffffu, v, o);
  if (lane == 0) res[m] = v;
}

}  // namespace

extern "C" const char* cfd_static_last_error(void) { return g_err; }

extern "C" int cfd_rk_stage1_static(double* q, double* qn, const double* r, int ni, int nj, int nk, double dt,
                                    double* res5_dev, void* cuda_stream) {
  g_err[0] = 0;
  if (!q || !qn || !r || !res5_dev) return fail(CFD_E_ARG, "cfd_rk_stage1_static: null pointer (q, qn, r and res5_dev are all required)");
  if (((uintptr_t)q | (uintptr_t)qn | (uintptr_t)r | (uintptr_t)res5_dev) & 7u)
    return fail(CFD_E_ARG, "cfd_rk_stage1_static: pointers must be 8-byte aligned");
  if (ni < 1 || nj < 1 || nk < 1) return fail(CFD_E_ARG, "cfd_rk_stage1_static: interior sizes must be >= 1 (got %d x %d x %d)", ni, nj, nk);
  const long long N = (long long)ni * nj * nk;
  if (N > (long long)CFD_STATIC_MAX_POINTS)
    return fail(CFD_E_WORKSPACE,
                "cfd_rk_stage1_static: %d x %d x %d = %lld interior points exceed CFD_STATIC_MAX_POINTS = %d, the capacity of the "
                "library's built-in scratch; use cfd_rk_stage with a caller-allocated workspace for larger blocks",
                ni, nj, nk, N, (int)CFD_STATIC_MAX_POINTS);
  double* partials = nullptr;
  int rc = scratch_of_current_device(&partials);
  if (rc != CFD_OK) return rc;

  BlockDev B{};
  B.n[0] = ni, B.n[1] = nj, B.n[2] = nk;
  for (int a = 0; a < 3; ++a) B.m[a] = B.n[a] + 2 * NG;
  B.M = (long long)B.m[0] * B.m[1] * B.m[2];
  B.s[0] = 1, B.s[1] = B.m[0], B.s[2] = (long long)B.m[0] * B.m[1];
  B.q = q, B.qn = qn, B.r = const_cast<double*>(r);
  cudaStream_t st = (cudaStream_t)cuda_stream;
  const int g = (int)((N + RKS_THREADS - 1) / RKS_THREADS);  // <= RKS_MAX_CTAS by the size check
  k_rk1_static<<<(unsigned)g, RKS_THREADS, 0, st>>>(B, dt, partials);
  k_res_static_final<<<1, 160, 0, st>>>(partials, g, res5_dev);
  cudaError_t e = cudaGetLastError();
  if (e != cudaSuccess) return fail(CFD_E_CUDA, "cfd_rk_stage1_static: kernel launch: %s", cudaGetErrorString(e));
  return CFD_OK;
}
