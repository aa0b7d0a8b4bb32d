// Internal declarations of the sm_100a CUDA path (not part of the C ABI; see include/cfd.h).
// Shares no code with oracle/.  P:L<n> = /root/reference/PAPER.md line n; U<k> = DESIGN.md reading k.
#pragma once
#include <cuda_runtime.h>

#include <cstdio>
#include <string>
#include <vector>

#include "cfd.h"

#define NG CFD_NG

// Scratch rows (doubles per stored point) of every block inside the caller's workspace: the viscous rows S (4), Fv^eta (4),
// Fv^zeta (4); cfd_compute_metrics reuses them for the 9 first derivatives of the coordinates.
constexpr int WS_ROWS = 12;

// Device view of one block.  Strides in doubles: s[0] = 1, s[1] = m0, s[2] = m0*m1.
struct BlockDev {
  int n[3];
  int m[3];
  long long M;
  long long s[3];
  double *q, *qn, *r, *xyz, *khat, *jac;
  double* ws;  // this block's WS_ROWS M doubles of scratch inside the caller's workspace (viscous rows / metric derivatives)
  int bcmask = 0;  // bit f set: face f carries a physical BC (WALL / FARFIELD): its node plane is not an inner point of the residual sum (U17a)
  // offset of interior node (0,0,0)
  __host__ __device__ inline long long idx(int i, int j, int k) const {
    return ((long long)(k + NG) * m[1] + (j + NG)) * m[0] + (i + NG);
  }
};

struct ParamsDev {
  double gamma, eps, mu, kappa;  // mu = Ma/Re (U9), kappa = mu / (Pr (gamma-1)); both times mu(T) when suth > 0
  double suth;                   // Sutherland's S / T_inf (U11); <= 0: constant mu = 1
  double q_inf[5];
  int viscous;
};

// One rectangular ghost region of one block, filled from a neighbour through an affine index map
// (U15): src index along neighbour axis perm[a] = sgn[a] * (dst index along a) + off[a].
struct CopyTask {
  int dst_block, src_block;
  int lo[3], ext[3];       // destination box: lo .. lo+ext-1 (interior-relative indices)
  long long sstride[3];    // stride (in doubles) in the SOURCE array when the dst index a increases by one (signed)
  long long sbase;         // source offset (doubles) of dst index (0,0,0) mapped
  double shift[3];         // coordinate shift (xyz fill only)
  int pass;                // 1: all regions are filled by one launch (the chains are composed on the host)
  int cta_begin;           // first CTA of this task in the flattened grid of the launch (prefix sum of the tasks' CTA counts)
};

struct BcTask {
  int block, face, type;   // CFD_FACE_WALL_NOSLIP_ADIABATIC or CFD_FACE_FARFIELD_CHAR
};

struct cfd_ctx {
  cfd_params prm;
  ParamsDev pd;
  std::vector<BlockDev> blk;
  std::vector<char> local;            // NEXT-4: local[b] = 0 for a block owned by a peer GPU (its pointers are peer-mapped; only the ghost fill reads them)
  bool is_local(size_t b) const { return local.empty() || local[b] != 0; }
  bool has_remote() const { for (char l : local) if (!l) return true; return false; }  // some block is advanced by a peer process
  std::vector<cfd_face> faces;
  std::vector<CopyTask> tasks[4];     // per pass 1..3
  std::vector<BcTask> bcs;
  CopyTask* d_tasks[4] = {nullptr, nullptr, nullptr, nullptr};
  BlockDev* d_blocks = nullptr;       // the descriptor array of the current buffer roles (points into d_blocks_all)
  BlockDev* d_blocks_all = nullptr;   // [6][nblocks]: one array per assignment of the three state buffers to (q, qn, r)
  std::vector<double*> base[3];       // per block: the caller's q, qn, r buffers as given to cfd_create_blocks
  void* xi_tma = nullptr;             // tensor maps of the TMA xi sweep (k_xi_tma.cu), or null
  int role[3] = {0, 1, 2};            // role[x] = which base buffer currently serves as q (x=0), qn (1), r (2)
  int* d_flag = nullptr;              // J <= 0 flag
  double* d_res = nullptr;            // 5 residual sums
  cudaStream_t stream = nullptr;
  double* ws = nullptr;
  size_t ws_bytes = 0;
  long long max_M = 0;
  long long sum_M = 0;                // sum of M over the blocks: the per-block scratch areas are WS_ROWS M doubles each
  static constexpr int NSIDE = 8;     // side streams: the blocks of a multi-block case run their per-block kernels concurrently
  cudaStream_t side[NSIDE] = {};
  cudaEvent_t ev_fork = nullptr, ev_join[NSIDE] = {};
  int conc = 1;                       // blocks whose kernel chains run concurrently (side streams): the sweeps size their segments for conc x their own CTAs
  long long launches = 0;
  int visc_tile = -1;                 // cfd_set_visc_tile: -1 = by block size, 0 / 1 / 2 = 64 x 8 / 70 x 7 / 54 x 9 threads
  unsigned only_mask = 0xffffffffu;  // cfd_profile_only: kernel classes (bit = ProfClass id) that launch_rhs still launches
  int xi_mode = 0;                    // xi kernel (cfd_set_sweep_plan): 0 chunk ring + 16-byte cp.async, 1 (plan 5) chunk ring + TMA, 2 (plan 4) 8-byte cp.async staging
  std::string err;
  // per-kernel event timing (cfd_profile_*): event pairs in launch order, reused after each read
  bool prof_on = false;
  std::vector<cudaEvent_t> prof_ev;
  std::vector<int> prof_id;
  size_t prof_used = 0;
};

// kernel classes of cfd_profile_read
enum ProfClass { PK_INV_XI = 0, PK_INV_ETA, PK_INV_ZETA, PK_VISC_FLUX, PK_VISC_PHI, PK_RK, PK_RES, PK_FILL, PK_BC, PK_METRICS, PK_COPY, PK_OTHER };

// Brackets the launches enqueued during its lifetime with two events when profiling is on.
struct ProfScope {
  cfd_ctx* c;
  cudaEvent_t stop = nullptr;
  ProfScope(cfd_ctx* ctx, int id) : c(ctx) {
    if (!c->prof_on) return;
    if (c->prof_used + 2 > c->prof_ev.size()) {
      cudaEvent_t a, b;
      if (cudaEventCreate(&a) != cudaSuccess || cudaEventCreate(&b) != cudaSuccess) return;
      c->prof_ev.push_back(a);
      c->prof_ev.push_back(b);
    }
    cudaEventRecord(c->prof_ev[c->prof_used], c->stream);
    stop = c->prof_ev[c->prof_used + 1];
    c->prof_id.resize(c->prof_ev.size() / 2);
    c->prof_id[c->prof_used / 2] = id;
    c->prof_used += 2;
  }
  ~ProfScope() {
    if (stop) cudaEventRecord(stop, c->stream);
  }
};

// RK stage fused into the last marching sweep (k_march ACC 3)
struct RkFuse {
  int stage;          // 1..3
  double dt, a, b;    // Eq. 20: out = a q^n + b (q + dt R)
  double* partials;   // stage 1: where this launch writes its per-CTA partial sums of R_m^2 (5 per CTA)
  long long max_ctas; // capacity of partials / 5
};

// ---- kernel launchers (each enqueues on ctx->stream and bumps ctx->launches) --------------------
int launch_fill_connect(cfd_ctx* c, int field /*0 q, 1 xyz*/);
int fill_ctas_of(const CopyTask& T);   // CTAs of one ghost-fill task in the flattened grid
int launch_bc_xyz(cfd_ctx* c);
int launch_bc_q(cfd_ctx* c);
int launch_metrics(cfd_ctx* c);
int launch_rhs(cfd_ctx* c, int fused_stage /*0 = plain rhs*/, double dt);
void set_roles(cfd_ctx* c, int iq, int iqn, int ir);
int launch_rk(cfd_ctx* c, int stage, double dt);
int launch_cfl(cfd_ctx* c, double cfl, double* const* dt_local);
int launch_fp64_probe(int iters, double* tflops);
int launch_fastmath_selftest(int n, const double* x_host, double* rcp_host, double* rsqrt_host);
int sweep_init();
int visc_march_init();
int launch_visc_march(cfd_ctx* c, const BlockDev& B);
void xi_tma_setup(cfd_ctx* c);
void xi_tma_free(cfd_ctx* c);
bool xi_tma_ok(const cfd_ctx* c, int b);
bool xi_ldg_ok(const cfd_ctx* c, int b);
int launch_xi_tma(cfd_ctx* c, int b, bool tma);

size_t ws_partials_offset_doubles(const cfd_ctx* c);
int rk_max_partial_blocks();

#define CUDA_TRY(ctx, expr)                                                      \
  do {                                                                           \
    cudaError_t _e = (expr);                                                     \
    if (_e != cudaSuccess) {                                                     \
      (ctx)->err = std::string(#expr) + ": " + cudaGetErrorString(_e);           \
      return CFD_E_CUDA;                                                         \
    }                                                                            \
  } while (0)
