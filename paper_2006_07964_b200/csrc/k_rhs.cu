// The launch sequence of cfd_rhs / cfd_stage_fused (S2 + S3, optionally S4 inside the last sweep).   sm_100a, fp64.
// P:L<n> = PAPER.md line; U<k> = DESIGN.md reading.  Shares no code with oracle/.
//
// Per block:  k_visc_march (Navier–Stokes only: S = d(Fv^xi)/d(xi) and the Fv^eta, Fv^zeta rows into the workspace)
//   -> xi sweep (r = X^xi) -> eta sweep (r += X^eta + S; differentiates Fv^eta) -> zeta sweep (r = J (r + X^zeta);
//   differentiates Fv^zeta; or the fused RK stage, Eq. 20).   X^d = d(Fv^d)/d(xi^d) - D^d  (Eq. 19).
#include "cfd_internal.cuh"

__global__ void k_res_final(const double* __restrict__ partials, int n, double* __restrict__ res);
int march_init();
int launch_march(cfd_ctx* c, const BlockDev& B, int dir, int acc, const RkFuse* rk, int* rk_ctas, bool sx, bool no_rows);
int launch_march_xi(cfd_ctx* c, const BlockDev& B);

int sweep_init() { return march_init(); }

// The three sweeps of block B.  The xi sweep, whose lanes sit on lines a row pitch apart, runs out of a per-warp chunk ring:
// k_xi_ldg (16-byte cp.async; default), k_xi_tma (xi_mode 1, cfd_set_sweep_plan(5)) or, for blocks with odd ni (row pitch not
// a multiple of 16 bytes) and xi_mode 2 (plan 4), k_march_xi (8-byte cp.async staging); scheme 1 (original AFWENO) has
// k_xi_ldg and, for odd ni, the plain marching kernel with strided lanes.
static int launch_sweeps(cfd_ctx* c, const BlockDev& B, const RkFuse* rk, int* rk_ctas) {
  int rc = 0;
  if (c->only_mask & (1u << PK_INV_XI)) {
    ProfScope ps(c, PK_INV_XI);
    const int b = (int)(&B - c->blk.data());
    const bool orig = c->prm.scheme == 1;
    if (!orig && c->xi_mode == 1 && xi_tma_ok(c, b)) rc = launch_xi_tma(c, b, true);
    else if ((orig || c->xi_mode != 2) && xi_ldg_ok(c, b)) rc = launch_xi_tma(c, b, false);
    else if (orig) rc = launch_march(c, B, 0, 0, nullptr, nullptr, false, true);
    else rc = launch_march_xi(c, B);
  }
  if (rc == 0 && (c->only_mask & (1u << PK_INV_ETA))) { ProfScope ps(c, PK_INV_ETA); rc = launch_march(c, B, 1, 1, nullptr, nullptr, true, false); }
  if (rc == 0 && (c->only_mask & (1u << PK_INV_ZETA))) { ProfScope ps(c, PK_INV_ZETA); rc = launch_march(c, B, 2, 2, rk, rk_ctas, false, false); }
  return rc;
}

// cfd_rhs (fused_stage 0) or, with fused_stage 1..3, the RHS with the RK stage fused into the last sweep
// (cfd_stage_fused): the new state lands in the r buffers and the caller exchanges the buffer roles.
int launch_rhs(cfd_ctx* c, int fused_stage, double dt) {
  RkFuse rk;
  rk.stage = fused_stage;
  rk.dt = dt;
  rk.a = fused_stage == 2 ? 3.0 / 4.0 : (fused_stage == 3 ? 1.0 / 3.0 : 0.0);
  rk.b = fused_stage == 2 ? 1.0 / 4.0 : (fused_stage == 3 ? 2.0 / 3.0 : 1.0);
  double* const partials = c->ws + ws_partials_offset_doubles(c);
  const long long cap = (long long)rk_max_partial_blocks() * (long long)c->blk.size();
  long long used = 0;
  // Blocks are independent until the ghost fill: with several blocks (and no per-kernel timing) each block's chain of
  // kernels goes to one of the library-owned side streams, forked from and joined back into the context's stream, so that
  // small blocks (C4: 8 x 96^3, about one wave of CTAs per kernel) fill the GPU together.  Every block has its own scratch.
  cudaStream_t const main_stream = c->stream;
  size_t nlocal = 0;
  for (size_t b = 0; b < c->blk.size(); ++b) nlocal += c->is_local(b) ? 1 : 0;
  const bool fork = nlocal > 1 && !c->prof_on && c->side[0] != nullptr;
  if (fork) {
    CUDA_TRY(c, cudaEventRecord(c->ev_fork, main_stream));
    for (int t = 0; t < cfd_ctx::NSIDE; ++t) CUDA_TRY(c, cudaStreamWaitEvent(c->side[t], c->ev_fork, 0));
  }
  int bi = 0, rc = 0;
  // the sweeps size their segments for the CTAs of all concurrently running blocks (C4: 3.31 -> 3.48 Gpts/s)
  c->conc = fork ? (int)(nlocal < (size_t)cfd_ctx::NSIDE ? nlocal : (size_t)cfd_ctx::NSIDE) : 1;
  for (size_t bx = 0; bx < c->blk.size(); ++bx) {
    if (!c->is_local(bx)) continue;  // NEXT-4: a peer GPU advances this block
    const BlockDev& B = c->blk[bx];
    if (fork) c->stream = c->side[bi++ % cfd_ctx::NSIDE];
    if (c->pd.viscous && (c->only_mask & (1u << PK_VISC_FLUX))) {
      ProfScope ps(c, PK_VISC_FLUX);
      rc = launch_visc_march(c, B);
    }
    rk.partials = partials + used * 5;
    rk.max_ctas = cap - used < rk_max_partial_blocks() ? cap - used : rk_max_partial_blocks();
    int ctas = 0;
    if (rc == 0) rc = launch_sweeps(c, B, fused_stage ? &rk : nullptr, &ctas);
    if (rc != 0) break;
    if (fused_stage == 1) used += ctas;
  }
  c->stream = main_stream;
  if (fork) {  // joined on every path: after an error the work already queued on the side streams stays ordered
    for (int t = 0; t < cfd_ctx::NSIDE; ++t) {
      CUDA_TRY(c, cudaEventRecord(c->ev_join[t], c->side[t]));
      CUDA_TRY(c, cudaStreamWaitEvent(main_stream, c->ev_join[t], 0));
    }
  }
  if (rc != 0) return rc;
  if (fused_stage == 1) {
    ProfScope ps(c, PK_RES);
    k_res_final<<<1, 160, 0, c->stream>>>(partials, (int)used, c->d_res);
    c->launches++;
  }
  CUDA_TRY(c, cudaGetLastError());
  // cfd_profile_only: with a hot kernel class masked out the call still returns 0 (the power probe loops it), but the
  // context says so in cfd_last_error, so that an invalid r / state can never pass for a valid one unnoticed
  if ((c->only_mask & 0xFu) != 0xFu)
    c->err = "cfd_profile_only mask active (a hot kernel class is switched off): the results of this call are INVALID";
  return CFD_OK;
}
