// C-ABI entry points (include/cfd.h): validation, host-side topology planning, launch sequencing.
// Every step of the path itself runs in the kernels of k_*.cu.
#include <cstdint>
#include <cstring>

#include "cfd_internal.cuh"

static thread_local std::string g_create_err;

static inline bool is_connect(int t) { return t == CFD_FACE_PERIODIC || t == CFD_FACE_INTERFACE; }

size_t ws_partials_offset_doubles(const cfd_ctx* c) { return (size_t)WS_ROWS * (size_t)c->sum_M + 8; }  // + 8: past the shifted scratch rows
int rk_max_partial_blocks() { return 16384; }

extern "C" size_t cfd_workspace_bytes_sharded(int nblocks, const cfd_dims* dims, const int* local, const cfd_params*) {
  long long sum = 0;  // every LOCAL block has its own WS_ROWS M doubles (the blocks' kernels run concurrently on side streams)
  for (int b = 0; b < nblocks; ++b)
    if (!local || local[b]) sum += (long long)(dims[b].ni + 2 * NG) * (dims[b].nj + 2 * NG) * (dims[b].nk + 2 * NG);
  return ((size_t)WS_ROWS * (size_t)sum + (size_t)rk_max_partial_blocks() * 5 * (size_t)(nblocks > 0 ? nblocks : 1) + 64) * sizeof(double);
}
extern "C" size_t cfd_workspace_bytes(int nblocks, const cfd_dims* dims, const cfd_params* prm) {
  return cfd_workspace_bytes_sharded(nblocks, dims, nullptr, prm);
}

// the six assignments of three buffers to the roles (q, qn, r): id -> role[]
static void roles_of(int id, int r[3]) {
  static const int P[6][3] = {{0, 1, 2}, {0, 2, 1}, {1, 0, 2}, {1, 2, 0}, {2, 0, 1}, {2, 1, 0}};
  for (int x = 0; x < 3; ++x) r[x] = P[id][x];
}
void set_roles(cfd_ctx* c, int iq, int iqn, int ir) {
  c->role[0] = iq; c->role[1] = iqn; c->role[2] = ir;
  int id = 0;
  for (; id < 6; ++id) {
    int r[3];
    roles_of(id, r);
    if (r[0] == iq && r[1] == iqn && r[2] == ir) break;
  }
  const size_t nb = c->blk.size();
  for (size_t b = 0; b < nb; ++b) { c->blk[b].q = c->base[iq][b]; c->blk[b].qn = c->base[iqn][b]; c->blk[b].r = c->base[ir][b]; }
  c->d_blocks = c->d_blocks_all + (size_t)id * nb;
}

static int fail_create(int code, const std::string& msg) {
  g_create_err = msg;
  return code;
}

// Host-side plan of the ghost fill (U15).  The fill is defined as three sequential passes (faces, then edges, then corners:
// the 26 ghost regions of a block, each filled through the lowest out-of-range axis whose face is PERIODIC / INTERFACE,
// from the neighbour's cells -- which for edges and corners are themselves ghost cells filled by the previous pass).
// Every such chain ends at cells that no pass writes (interior cells, or ghost cells behind a physical face), and every hop
// is a signed permutation plus an offset, so the chain is composed HERE into one affine map per region: all regions are
// filled by ONE launch that reads final sources only (same values, bit for bit, as the three passes).
struct IdxMap {       // index vector in block `blk` = P x + o for the destination index vector x
  int blk;
  int P[3][3];
  int o[3];
  double shift[3];    // accumulated coordinate translation (xyz fill)
};

static bool hop(const cfd_ctx* c, const int ftype[], const int fidx[], IdxMap& m, const int probe[3]) {
  // where does the probe point sit in the current block?  pick the lowest out-of-range axis behind a connecting face
  const BlockDev& B = c->blk[m.blk];
  int y[3];
  for (int a = 0; a < 3; ++a) y[a] = m.P[a][0] * probe[0] + m.P[a][1] * probe[1] + m.P[a][2] * probe[2] + m.o[a];
  int an = -1, s = 0;
  for (int a = 0; a < 3 && an < 0; ++a) {
    if (y[a] >= 0 && y[a] < B.n[a]) continue;
    const int fc = 2 * a + (y[a] < 0 ? 0 : 1);
    if (is_connect(ftype[m.blk * 6 + fc])) { an = a; s = fc % 2; }
  }
  if (an < 0) return false;
  const cfd_face& F = c->faces[fidx[m.blk * 6 + 2 * an + s]];
  const BlockDev& N = c->blk[F.nbr_block];
  const int sp = F.nbr_face % 2;
  IdxMap r;
  r.blk = F.nbr_block;
  for (int a = 0; a < 3; ++a) {
    const int ap = F.perm[a];
    int sgn, off;
    if (a == an) {
      if (s == 0 && sp == 1) { sgn = 1; off = N.n[ap]; }
      else if (s == 0 && sp == 0) { sgn = -1; off = -1; }
      else if (s == 1 && sp == 0) { sgn = 1; off = -B.n[a]; }
      else { sgn = -1; off = N.n[ap] + B.n[a] - 1; }
    } else {
      sgn = F.sign[a] > 0 ? 1 : -1;
      off = F.sign[a] > 0 ? 0 : B.n[a] - 1;
    }
    // neighbour index along ap = sgn * (my index along a) + off, my index = row a of (P x + o)
    for (int t = 0; t < 3; ++t) r.P[ap][t] = sgn * m.P[a][t];
    r.o[ap] = sgn * m.o[a] + off;
  }
  for (int t = 0; t < 3; ++t) r.shift[t] = m.shift[t] + F.shift[t];
  m = r;
  return true;
}

static void plan_copies(cfd_ctx* c) {
  const size_t nb = c->blk.size();
  std::vector<int> ftype(nb * 6, 0), fidx(nb * 6, -1);
  for (size_t t = 0; t < c->faces.size(); ++t) {
    ftype[(size_t)c->faces[t].block * 6 + c->faces[t].face] = c->faces[t].type;
    fidx[(size_t)c->faces[t].block * 6 + c->faces[t].face] = (int)t;
  }
  for (size_t b = 0; b < nb; ++b) {
    if (!c->is_local(b)) continue;  // a peer GPU fills the ghost layers of its own blocks
    const BlockDev& B = c->blk[b];
    for (int code = 0; code < 27; ++code) {
      int side[3] = {code % 3, (code / 3) % 3, code / 9};  // 0 below, 1 inside, 2 above
      if (code == 13) continue;
      CopyTask T;
      T.dst_block = (int)b;
      int probe[3];
      for (int a = 0; a < 3; ++a) {
        T.lo[a] = side[a] == 0 ? -NG : (side[a] == 1 ? 0 : B.n[a]);
        T.ext[a] = side[a] == 1 ? B.n[a] : NG;
        probe[a] = T.lo[a];
      }
      IdxMap m;
      m.blk = (int)b;
      for (int a = 0; a < 3; ++a) {
        for (int t = 0; t < 3; ++t) m.P[a][t] = a == t ? 1 : 0;
        m.o[a] = 0;
        m.shift[a] = 0.0;
      }
      int hops = 0;
      while (hops < 3 && hop(c, ftype.data(), fidx.data(), m, probe)) ++hops;
      if (hops == 0) continue;  // no connecting face behind this region: the physical boundary conditions own it
      const BlockDev& S = c->blk[m.blk];
      T.src_block = m.blk;
      long long base = 0;
      for (int t = 0; t < 3; ++t) T.sstride[t] = 0;
      for (int a = 0; a < 3; ++a) {
        for (int t = 0; t < 3; ++t) T.sstride[t] += (long long)m.P[a][t] * S.s[a];
        base += (long long)(m.o[a] + NG) * S.s[a];
        T.shift[a] = m.shift[a];
      }
      T.sbase = base;
      T.pass = 1;
      T.cta_begin = c->tasks[1].empty() ? 0 : c->tasks[1].back().cta_begin + fill_ctas_of(c->tasks[1].back());
      c->tasks[1].push_back(T);
    }
  }
}

extern "C" int cfd_create_blocks(cfd_ctx** out, int nblocks, const cfd_dims* dims, const cfd_block_ptrs* ptrs, int nfaces,
                                 const cfd_face* faces, const cfd_params* params, void* workspace, size_t workspace_bytes,
                                 void* cuda_stream) {
  return cfd_create_blocks_sharded(out, nblocks, dims, ptrs, nullptr, nfaces, faces, params, workspace, workspace_bytes, cuda_stream);
}

extern "C" int cfd_create_blocks_sharded(cfd_ctx** out, int nblocks, const cfd_dims* dims, const cfd_block_ptrs* ptrs, const int* local,
                                         int nfaces, const cfd_face* faces, const cfd_params* params, void* workspace,
                                         size_t workspace_bytes, void* cuda_stream) {
  if (!out || nblocks < 1 || !dims || !ptrs || !params || nfaces < 0 || (nfaces > 0 && !faces))
    return fail_create(CFD_E_ARG, "cfd_create_blocks: null argument or nblocks < 1");
  *out = nullptr;
  if (!(params->gamma > 1.0) || !(params->weno_eps > 0.0) || !(params->weno_eps < 1e3))
    return fail_create(CFD_E_ARG, "cfd_create_blocks: need gamma > 1 and 0 < weno_eps < 1e3");
  if (params->viscous && (!(params->reynolds > 0.0) || !(params->prandtl > 0.0) || !(params->mach >= 0.0)))
    return fail_create(CFD_E_ARG, "cfd_create_blocks: viscous run needs reynolds > 0, prandtl > 0, mach >= 0");
  if (params->scheme != 0 && params->scheme != 1) return fail_create(CFD_E_ARG, "cfd_create_blocks: scheme must be 0 or 1");
  int ndev = 0;
  if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev < 1)
    return fail_create(CFD_E_CUDA, "cfd_create_blocks: no CUDA device (there is no CPU fallback)");

  cfd_ctx* c = new cfd_ctx();
  c->prm = *params;
  c->pd.gamma = params->gamma;
  c->pd.eps = params->weno_eps;
  c->pd.viscous = params->viscous;
  c->pd.mu = params->viscous ? params->mach / params->reynolds : 0.0;
  c->pd.kappa = params->viscous ? c->pd.mu / (params->prandtl * (params->gamma - 1.0)) : 0.0;
  c->pd.suth = params->sutherland > 0.0 ? params->sutherland : 0.0;
  for (int m = 0; m < 5; ++m) c->pd.q_inf[m] = params->q_inf[m];
  c->stream = (cudaStream_t)cuda_stream;
  c->blk.resize(nblocks);
  if (local) {
    c->local.assign(local, local + nblocks);
    bool any = false;
    for (int b = 0; b < nblocks; ++b) any = any || local[b];
    if (!any) { delete c; return fail_create(CFD_E_ARG, "cfd_create_blocks_sharded: this context owns no block"); }
  }
  for (int b = 0; b < nblocks; ++b) {
    BlockDev& B = c->blk[b];
    B.n[0] = dims[b].ni; B.n[1] = dims[b].nj; B.n[2] = dims[b].nk;
    for (int a = 0; a < 3; ++a) {
      if (B.n[a] < NG) { delete c; return fail_create(CFD_E_ARG, "cfd_create_blocks: interior size must be >= 6 on every axis"); }
      B.m[a] = B.n[a] + 2 * NG;
    }
    B.M = (long long)B.m[0] * B.m[1] * B.m[2];
    B.s[0] = 1; B.s[1] = B.m[0]; B.s[2] = (long long)B.m[0] * B.m[1];
    B.q = ptrs[b].q; B.qn = ptrs[b].qn; B.r = ptrs[b].r; B.xyz = ptrs[b].xyz; B.khat = ptrs[b].khat; B.jac = ptrs[b].jac;
    const void* pp[6] = {B.q, B.qn, B.r, B.xyz, B.khat, B.jac};
    for (int t = 0; t < (c->is_local(b) ? 6 : 4); ++t)  // a peer's block: q, qn, r, xyz (peer-mapped) only
      if (!pp[t] || ((uintptr_t)pp[t] & 15u)) { delete c; return fail_create(CFD_E_ARG, "cfd_create_blocks: null or misaligned (16 B) field pointer"); }
    if (!c->is_local(b)) continue;
    if (B.M > c->max_M) c->max_M = B.M;
    c->sum_M += B.M;
  }
  // ---- faces ----
  c->faces.assign(faces, faces + nfaces);
  std::vector<int> seen((size_t)nblocks * 6, 0);
  for (int t = 0; t < nfaces; ++t) {
    const cfd_face& F = c->faces[t];
    auto bad = [&](const char* m) { delete c; return fail_create(CFD_E_TOPOLOGY, std::string("cfd_create_blocks: face ") + std::to_string(t) + ": " + m); };
    if (F.block < 0 || F.block >= nblocks || F.face < 0 || F.face > 5) return bad("bad block/face id");
    if (seen[(size_t)F.block * 6 + F.face]++) return bad("described twice");
    if (is_connect(F.type)) {
      if (F.nbr_block < 0 || F.nbr_block >= nblocks || F.nbr_face < 0 || F.nbr_face > 5) return bad("bad neighbour");
      int cnt[3] = {0, 0, 0};
      for (int a = 0; a < 3; ++a) {
        if (F.perm[a] < 0 || F.perm[a] > 2 || (F.sign[a] != 1 && F.sign[a] != -1)) return bad("bad perm/sign");
        cnt[F.perm[a]]++;
      }
      if (cnt[0] != 1 || cnt[1] != 1 || cnt[2] != 1) return bad("perm is not a permutation");
      const bool even = (F.perm[0] == 0 && F.perm[1] == 1) || (F.perm[0] == 1 && F.perm[1] == 2) || (F.perm[0] == 2 && F.perm[1] == 0);
      if ((even ? 1 : -1) * F.sign[0] * F.sign[1] * F.sign[2] != 1) return bad("not a proper rotation");
      const int an = F.face / 2;
      if (F.perm[an] != F.nbr_face / 2) return bad("nbr_face axis != perm[normal axis]");
      if (F.sign[an] != ((F.face % 2) != (F.nbr_face % 2) ? 1 : -1)) return bad("normal-axis sign inconsistent with the face pair");
      for (int a = 0; a < 3; ++a)
        if (a != an && c->blk[F.nbr_block].n[F.perm[a]] != c->blk[F.block].n[a]) return bad("interface extents do not match");
    } else if (F.type == CFD_FACE_WALL_NOSLIP_ADIABATIC || F.type == CFD_FACE_FARFIELD_CHAR) {
      // the wall closure reads the nodes 1..4 and mirrors the nodes 1..6 behind the wall: they must be interior nodes
      if (F.type == CFD_FACE_WALL_NOSLIP_ADIABATIC && c->blk[F.block].n[F.face / 2] < NG + 1)
        return bad("a wall needs at least 7 interior nodes along its normal");
      BcTask T{F.block, F.face, F.type};
      c->blk[F.block].bcmask |= 1 << F.face;
      if (c->is_local(F.block)) c->bcs.push_back(T);
    } else {
      return bad("unknown face type");
    }
  }
  // every face of every block must be described (an undescribed face would leave its ghost layers unfilled), and
  // the two sides of a connection must describe each other (U15)
  for (int b = 0; b < nblocks; ++b)
    for (int f = 0; f < 6; ++f)
      if (!seen[(size_t)b * 6 + f]) {
        delete c;
        return fail_create(CFD_E_TOPOLOGY, "cfd_create_blocks: block " + std::to_string(b) + " face " + std::to_string(f) +
                                               " has no face descriptor");
      }
  for (int t = 0; t < nfaces; ++t) {
    const cfd_face& F = c->faces[t];
    if (!is_connect(F.type)) continue;
    const cfd_face* N = nullptr;
    for (int u = 0; u < nfaces; ++u)
      if (c->faces[u].block == F.nbr_block && c->faces[u].face == F.nbr_face) N = &c->faces[u];
    bool ok = N && is_connect(N->type) && N->nbr_block == F.block && N->nbr_face == F.face;
    for (int a = 0; ok && a < 3; ++a) ok = N->perm[F.perm[a]] == a && N->sign[F.perm[a]] == F.sign[a];  // inverse rotation
    if (!ok) {
      delete c;
      return fail_create(CFD_E_TOPOLOGY, "cfd_create_blocks: face " + std::to_string(t) +
                                             ": the neighbour's descriptor does not point back with the inverse permutation");
    }
  }
  // ---- workspace ----
  size_t need = cfd_workspace_bytes_sharded(nblocks, dims, local, params);
  if (!workspace || workspace_bytes < need || ((uintptr_t)workspace & 15u)) {
    delete c;
    return fail_create(CFD_E_WORKSPACE, "cfd_create_blocks: workspace null, misaligned or smaller than cfd_workspace_bytes()");
  }
  c->ws = (double*)workspace;
  c->ws_bytes = workspace_bytes;
  {
    long long off = 0;
    // + 2: the scratch rows are indexed like the fields but shifted by two doubles, so that interior i = 0 (array index NG = 6)
    // starts a 32-byte sector: the rows are written in interior runs, and half-sector writes cost a read-modify-write
    for (size_t b = 0; b < c->blk.size(); ++b) {
      BlockDev& B = c->blk[b];
      if (!c->is_local(b)) { B.ws = nullptr; continue; }
      B.ws = c->ws + (long long)WS_ROWS * off + 2;
      off += B.M;
    }
  }
  plan_copies(c);
  // ---- small device-side descriptor arrays (a few KB; the only allocations the library makes) ----
  auto cuda_fail = [&](cudaError_t e, const char* what) {
    std::string m = std::string("cfd_create_blocks: ") + what + ": " + cudaGetErrorString(e);
    cfd_destroy(c);
    return fail_create(CFD_E_CUDA, m);
  };
  cudaError_t e;
  // one descriptor array per assignment of the caller's (q, qn, r) buffers to the three roles: the fused stage
  // (cfd_stage_fused) exchanges roles instead of copying
  for (int b = 0; b < nblocks; ++b) { c->base[0].push_back(ptrs[b].q); c->base[1].push_back(ptrs[b].qn); c->base[2].push_back(ptrs[b].r); }
  if ((e = cudaMalloc(&c->d_blocks_all, sizeof(BlockDev) * nblocks * 6)) != cudaSuccess) return cuda_fail(e, "cudaMalloc blocks");
  {
    std::vector<BlockDev> all((size_t)nblocks * 6);
    for (int id = 0; id < 6; ++id) {
      int r[3];
      roles_of(id, r);
      for (int b = 0; b < nblocks; ++b) {
        BlockDev B = c->blk[b];
        B.q = c->base[r[0]][b]; B.qn = c->base[r[1]][b]; B.r = c->base[r[2]][b];
        all[(size_t)id * nblocks + b] = B;
      }
    }
    if ((e = cudaMemcpy(c->d_blocks_all, all.data(), sizeof(BlockDev) * all.size(), cudaMemcpyHostToDevice)) != cudaSuccess) return cuda_fail(e, "cudaMemcpy blocks");
  }
  set_roles(c, 0, 1, 2);
  xi_tma_setup(c);
  if (nblocks > 1) {
    for (int t = 0; t < cfd_ctx::NSIDE; ++t) {
      if ((e = cudaStreamCreateWithFlags(&c->side[t], cudaStreamNonBlocking)) != cudaSuccess) return cuda_fail(e, "cudaStreamCreate");
      if ((e = cudaEventCreateWithFlags(&c->ev_join[t], cudaEventDisableTiming)) != cudaSuccess) return cuda_fail(e, "cudaEventCreate");
    }
    if ((e = cudaEventCreateWithFlags(&c->ev_fork, cudaEventDisableTiming)) != cudaSuccess) return cuda_fail(e, "cudaEventCreate");
  }
  for (int p = 1; p <= 3; ++p) {
    if (c->tasks[p].empty()) continue;
    if ((e = cudaMalloc(&c->d_tasks[p], sizeof(CopyTask) * c->tasks[p].size())) != cudaSuccess) return cuda_fail(e, "cudaMalloc tasks");
    if ((e = cudaMemcpy(c->d_tasks[p], c->tasks[p].data(), sizeof(CopyTask) * c->tasks[p].size(), cudaMemcpyHostToDevice)) != cudaSuccess)
      return cuda_fail(e, "cudaMemcpy tasks");
  }
  if ((e = cudaMalloc(&c->d_flag, sizeof(int))) != cudaSuccess) return cuda_fail(e, "cudaMalloc flag");
  if ((e = cudaMalloc(&c->d_res, sizeof(double) * 8)) != cudaSuccess) return cuda_fail(e, "cudaMalloc res");
  if (sweep_init() != 0 || visc_march_init() != 0) return cuda_fail(cudaGetLastError(), "cudaFuncSetAttribute (dynamic shared memory of the sweep kernels)");
  *out = c;
  return CFD_OK;
}

extern "C" int cfd_destroy(cfd_ctx* c) {
  if (!c) return CFD_OK;
  if (c->d_blocks_all) cudaFree(c->d_blocks_all);
  xi_tma_free(c);
  for (int t = 0; t < cfd_ctx::NSIDE; ++t) {
    if (c->side[t]) cudaStreamDestroy(c->side[t]);
    if (c->ev_join[t]) cudaEventDestroy(c->ev_join[t]);
  }
  if (c->ev_fork) cudaEventDestroy(c->ev_fork);
  for (int p = 1; p <= 3; ++p)
    if (c->d_tasks[p]) cudaFree(c->d_tasks[p]);
  if (c->d_flag) cudaFree(c->d_flag);
  if (c->d_res) cudaFree(c->d_res);
  for (cudaEvent_t e : c->prof_ev) cudaEventDestroy(e);
  delete c;
  return CFD_OK;
}

extern "C" const char* cfd_last_error(const cfd_ctx* c) { return c ? c->err.c_str() : g_create_err.c_str(); }
extern "C" long long cfd_launch_count(const cfd_ctx* c) { return c ? c->launches : 0; }

extern "C" int cfd_compute_metrics(cfd_ctx* c) {
  if (!c) return CFD_E_ARG;
  int rc;
  if ((rc = launch_fill_connect(c, 1)) != 0) return rc;
  if ((rc = launch_bc_xyz(c)) != 0) return rc;
  CUDA_TRY(c, cudaMemsetAsync(c->d_flag, 0, sizeof(int), c->stream));
  if ((rc = launch_metrics(c)) != 0) return rc;
  int flag = 0;
  CUDA_TRY(c, cudaMemcpyAsync(&flag, c->d_flag, sizeof(int), cudaMemcpyDeviceToHost, c->stream));
  CUDA_TRY(c, cudaStreamSynchronize(c->stream));
  if (flag) { c->err = "cfd_compute_metrics: J <= 0 at an interior node"; return CFD_E_JACOBIAN; }
  return CFD_OK;
}

extern "C" int cfd_rhs(cfd_ctx* c) {
  if (!c) return CFD_E_ARG;
  return launch_rhs(c, 0, 0.0);
}

extern "C" int cfd_rk_stage(cfd_ctx* c, int stage, double dt, double* res5) {
  if (!c) return CFD_E_ARG;
  if (stage < 1 || stage > 3) { c->err = "cfd_rk_stage: stage must be 1..3"; return CFD_E_STAGE; }
  int rc = launch_rk(c, stage, dt);
  if (rc != 0) return rc;
  if (res5 && stage == 1) {
    CUDA_TRY(c, cudaMemcpyAsync(res5, c->d_res, 5 * sizeof(double), cudaMemcpyDeviceToHost, c->stream));
    CUDA_TRY(c, cudaStreamSynchronize(c->stream));
  }
  return CFD_OK;
}

extern "C" int cfd_cfl_dt(cfd_ctx* c, double cfl, double* dt_host, double* const* dt_local) {
  if (!c || !dt_host) return CFD_E_ARG;
  if (!(cfl > 0.0)) { c->err = "cfd_cfl_dt: cfl must be > 0"; return CFD_E_ARG; }
  if (dt_local)
    for (size_t b = 0; b < c->blk.size(); ++b)
      if (c->is_local(b) && (!dt_local[b] || ((uintptr_t)dt_local[b] & 7u))) { c->err = "cfd_cfl_dt: null or misaligned dt_local pointer"; return CFD_E_ARG; }
  int rc = launch_cfl(c, cfl, dt_local);
  if (rc != 0) return rc;
  double smax = 0.0;
  CUDA_TRY(c, cudaMemcpyAsync(&smax, c->d_res + 5, sizeof(double), cudaMemcpyDeviceToHost, c->stream));
  CUDA_TRY(c, cudaStreamSynchronize(c->stream));
  if (!(smax > 0.0) || smax != smax || smax > 1.7976931348623157e308) {
    c->err = "cfd_cfl_dt: non-positive, infinite or NaN spectral radius (state not physical: rho <= 0 or p < 0 at an interior point)";
    return CFD_E_ARG;
  }
  *dt_host = cfl / smax;
  return CFD_OK;
}

extern "C" int cfd_exchange_interfaces(cfd_ctx* c) {
  if (!c) return CFD_E_ARG;
  return launch_fill_connect(c, 0);
}

extern "C" int cfd_apply_bc(cfd_ctx* c) {
  if (!c) return CFD_E_ARG;
  return launch_bc_q(c);
}

// The single-call stages run the ghost fill right behind the local sweeps.  On a context with peer-owned blocks that fill
// reads the peers' interiors over P2P, and nothing in this process can know whether the peers have finished writing their
// new state (or have rotated their buffer roles): the caller must put a cross-process barrier in between, which only the
// split sequence cfd_stage_fused_local -> barrier -> cfd_exchange_interfaces -> barrier -> cfd_apply_bc allows.
static int refuse_if_sharded(cfd_ctx* c, const char* fn) {
  if (!c->has_remote()) return CFD_OK;
  c->err = std::string(fn) + ": this context has blocks owned by peer processes (cfd_create_blocks_sharded); the ghost fill must "
           "be separated from the sweeps by a cross-process barrier: call cfd_stage_fused_local, synchronise the processes, then "
           "cfd_exchange_interfaces and cfd_apply_bc";
  return CFD_E_ARG;
}

extern "C" int cfd_stage(cfd_ctx* c, int stage, double dt, double* res5) {
  int rc;
  if (!c) return CFD_E_ARG;
  if ((rc = refuse_if_sharded(c, "cfd_stage")) != 0) return rc;
  if ((rc = cfd_rhs(c)) != 0) return rc;
  if ((rc = cfd_rk_stage(c, stage, dt, res5)) != 0) return rc;
  if ((rc = cfd_exchange_interfaces(c)) != 0) return rc;
  return cfd_apply_bc(c);
}

extern "C" int cfd_stage_fused_local(cfd_ctx* c, int stage, double dt, double* res5) {
  if (!c) return CFD_E_ARG;
  if (stage < 1 || stage > 3) { c->err = "cfd_stage_fused: stage must be 1..3"; return CFD_E_STAGE; }
  int rc = launch_rhs(c, stage, dt);
  if (rc != 0) return rc;
  // the new state was written to the r buffers: exchange the roles (stage 1: the old q becomes q^n, Eq. 20)
  if (stage == 1) set_roles(c, c->role[2], c->role[0], c->role[1]);
  else set_roles(c, c->role[2], c->role[1], c->role[0]);
  if (res5 && stage == 1) {
    CUDA_TRY(c, cudaMemcpyAsync(res5, c->d_res, 5 * sizeof(double), cudaMemcpyDeviceToHost, c->stream));
    CUDA_TRY(c, cudaStreamSynchronize(c->stream));
  }
  return CFD_OK;
}

extern "C" int cfd_stage_fused(cfd_ctx* c, int stage, double dt, double* res5) {
  if (!c) return CFD_E_ARG;
  int rc = refuse_if_sharded(c, "cfd_stage_fused");
  if (rc != 0) return rc;
  rc = cfd_stage_fused_local(c, stage, dt, res5);
  if (rc != 0) return rc;
  if ((rc = cfd_exchange_interfaces(c)) != 0) return rc;
  return cfd_apply_bc(c);
}

extern "C" int cfd_buffer_roles(const cfd_ctx* c, int roles[3]) {
  if (!c || !roles) return CFD_E_ARG;
  for (int x = 0; x < 3; ++x) roles[x] = c->role[x];
  return CFD_OK;
}

extern "C" int cfd_step_host(cfd_ctx* c, const double* const* qin, double* const* qout, double dt, double* res5) {
  if (!c || !qin || !qout) return CFD_E_ARG;
  if (int rs = refuse_if_sharded(c, "cfd_step_host")) return rs;
  auto copy3d = [&](const BlockDev& B, double* dev, double* host, bool to_dev) {
    cudaMemcpy3DParms p;
    memset(&p, 0, sizeof(p));
    cudaPitchedPtr d = make_cudaPitchedPtr(dev, (size_t)B.m[0] * 8, (size_t)B.m[0] * 8, (size_t)B.m[1]);
    cudaPitchedPtr h = make_cudaPitchedPtr(host, (size_t)B.n[0] * 8, (size_t)B.n[0] * 8, (size_t)B.n[1]);
    const cudaPos dpos = make_cudaPos((size_t)NG * 8, NG, NG), hpos = make_cudaPos(0, 0, 0);
    p.srcPtr = to_dev ? h : d; p.srcPos = to_dev ? hpos : dpos;
    p.dstPtr = to_dev ? d : h; p.dstPos = to_dev ? dpos : hpos;
    p.extent = make_cudaExtent((size_t)B.n[0] * 8, (size_t)B.n[1], (size_t)B.n[2]);
    p.kind = to_dev ? cudaMemcpyHostToDevice : cudaMemcpyDeviceToHost;
    return cudaMemcpy3DAsync(&p, c->stream);
  };
  for (size_t b = 0; b < c->blk.size(); ++b) {
    if (!c->is_local(b)) continue;
    const BlockDev& B = c->blk[b];
    if (!qin[b] || !qout[b]) { c->err = "cfd_step_host: null host pointer"; return CFD_E_ARG; }
    const size_t N = (size_t)B.n[0] * B.n[1] * B.n[2];
    ProfScope ps(c, PK_COPY);
    for (int m = 0; m < 5; ++m) CUDA_TRY(c, copy3d(B, B.q + (size_t)m * B.M, const_cast<double*>(qin[b]) + m * N, true));
  }
  int rc;
  if ((rc = cfd_exchange_interfaces(c)) != 0) return rc;
  if ((rc = cfd_apply_bc(c)) != 0) return rc;
  for (int s = 1; s <= 3; ++s)
    if ((rc = cfd_stage_fused(c, s, dt, nullptr)) != 0) return rc;
  for (size_t b = 0; b < c->blk.size(); ++b) {
    if (!c->is_local(b)) continue;
    const BlockDev& B = c->blk[b];
    const size_t N = (size_t)B.n[0] * B.n[1] * B.n[2];
    ProfScope ps(c, PK_COPY);
    for (int m = 0; m < 5; ++m) CUDA_TRY(c, copy3d(B, B.q + (size_t)m * B.M, qout[b] + m * N, false));
  }
  if (res5) CUDA_TRY(c, cudaMemcpyAsync(res5, c->d_res, 5 * sizeof(double), cudaMemcpyDeviceToHost, c->stream));
  CUDA_TRY(c, cudaStreamSynchronize(c->stream));
  return CFD_OK;
}

static const char* k_prof_names[CFD_PROF_NCLASS] = {"inviscid_xi", "inviscid_eta", "inviscid_zeta", "visc_flux", "visc_phi", "rk_stage",
                                                    "residual_final", "ghost_fill", "phys_bc", "metrics", "host_copy", "other"};

extern "C" const char* cfd_profile_name(int id) { return (id >= 0 && id < CFD_PROF_NCLASS) ? k_prof_names[id] : ""; }

extern "C" int cfd_profile_enable(cfd_ctx* c, int on) {
  if (!c) return CFD_E_ARG;
  CUDA_TRY(c, cudaStreamSynchronize(c->stream));
  c->prof_on = on != 0;
  c->prof_used = 0;
  return CFD_OK;
}

extern "C" int cfd_profile_read(cfd_ctx* c, double* ms, long long* launches) {
  if (!c || !ms || !launches) return CFD_E_ARG;
  CUDA_TRY(c, cudaStreamSynchronize(c->stream));
  for (int i = 0; i < CFD_PROF_NCLASS; ++i) { ms[i] = 0.0; launches[i] = 0; }
  for (size_t t = 0; t + 1 < c->prof_used; t += 2) {
    float e = 0.f;
    CUDA_TRY(c, cudaEventElapsedTime(&e, c->prof_ev[t], c->prof_ev[t + 1]));
    const int id = c->prof_id[t / 2];
    ms[id] += e;
    launches[id] += 1;
  }
  c->prof_used = 0;
  return CFD_OK;
}

extern "C" int cfd_set_visc_tile(cfd_ctx* c, int tile) {
  if (!c) return CFD_E_ARG;
  if (tile < -1 || tile > 2) { c->err = "cfd_set_visc_tile: tile must be -1 (automatic), 0, 1 or 2"; return CFD_E_ARG; }
  c->visc_tile = tile;
  return CFD_OK;
}

extern "C" int cfd_profile_only(cfd_ctx* c, unsigned mask) {
  if (!c) return CFD_E_ARG;
  c->only_mask = mask;
  if ((mask & 0xFu) == 0xFu && c->err.rfind("cfd_profile_only mask active", 0) == 0) c->err.clear();  // warning of launch_rhs
  return CFD_OK;
}

extern "C" int cfd_set_sweep_plan(cfd_ctx* c, int plan) {
  if (!c) return CFD_E_ARG;
  if (plan != 0 && plan != 4 && plan != 5) { c->err = "cfd_set_sweep_plan: plan must be 0, 4 or 5"; return CFD_E_ARG; }
  c->xi_mode = plan == 4 ? 2 : (plan == 5 ? 1 : 0);
  return CFD_OK;
}

extern "C" int cfd_selftest_fastmath(int n, const double* x_host, double* rcp_host, double* rsqrt_host) {
  if (n < 1 || !x_host || !rcp_host || !rsqrt_host) return CFD_E_ARG;
  return launch_fastmath_selftest(n, x_host, rcp_host, rsqrt_host);
}

extern "C" int cfd_fp64_peak_probe(int iters, double* tflops) {
  if (!tflops || iters < 1) return CFD_E_ARG;
  return launch_fp64_probe(iters, tflops);
}
