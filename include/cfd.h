/* =====================================================================================
 * cfd.h — C ABI of the B200-native (sm_100a) fp64 hot path of
 *   Ye, Zhang, Wan, Yan, Sun, "Accelerating CFD simulation with high order finite difference
 *   method on curvilinear coordinates for modern GPU clusters", Adv. Aerodyn. 4:7 (2022).
 * Citations: P:L<n> = line n of /root/reference/PAPER.md; U<k> = reading k in DESIGN.md §3.
 *
 * The path: right-hand side R(Q) of the compressible Navier–Stokes equations in strong
 * conservation form on curvilinear multi-block structured grids (Eq. 2) and the
 * TVD-RK3 stage update (Eq. 20), in the stage order of Fig. 2:
 *     cfd_rhs -> cfd_rk_stage -> cfd_exchange_interfaces -> cfd_apply_bc .
 *
 * General rules
 *  - Every function returns 0 (CFD_OK) on success and a negative cfd_status on error; nothing
 *    throws, nothing calls exit().  cfd_last_error() returns a message for the last failure.
 *  - All field buffers are DEVICE pointers OWNED BY THE CALLER (e.g. torch tensors) for the
 *    whole life of the context; the library keeps non-owning pointers and never frees them.
 *  - Layout of every field: fp64, structure-of-arrays [var][k][j][i], i fastest, each axis
 *    carrying CFD_NG = 6 ghost layers on both sides: extents (ni+12, nj+12, nk+12),
 *    M = (ni+12)(nj+12)(nk+12) doubles per variable.  Pointers must be 16-byte aligned.
 *  - All work is ordered on the CUDA stream given to cfd_create_blocks: it is enqueued there or, for contexts
 *    with more than one block, partly on eight library-owned non-blocking side streams that cfd_rhs /
 *    cfd_stage_fused fork from that stream and join back into it before they return (the blocks' kernel chains
 *    run concurrently; work enqueued on the caller's stream before or after a call is ordered with it).  No
 *    function synchronises the device unless documented ("returns host values").
 *  - No cudaMalloc/cudaFree after cfd_create_blocks (which allocates a few KB of descriptors and, for
 *    multi-block contexts, the side streams and their events).
 *  - There is no CPU fallback: without a CUDA device cfd_create_blocks fails with CFD_E_CUDA.
 * ===================================================================================== */
#ifndef CFD_B200_H
#define CFD_B200_H

#include <stddef.h>

#ifdef __cplusplus
extern "C" {
#endif

#define CFD_NG 6 /* ghost layers per face (U12; the paper has ghost cells, M != N, depth unstated) */

typedef enum {
  CFD_OK = 0,
  CFD_E_ARG = -1,       /* null / misaligned pointer, bad size, bad enum */
  CFD_E_TOPOLOGY = -2,  /* inconsistent face descriptor (perm/sign/extents) */
  CFD_E_JACOBIAN = -3,  /* J <= 0 at an interior node (cfd_compute_metrics) */
  CFD_E_STAGE = -4,     /* RK stage not in 1..3 */
  CFD_E_WORKSPACE = -5, /* workspace too small / null */
  CFD_E_CUDA = -6       /* a CUDA runtime call failed (message holds cudaGetErrorString) */
} cfd_status;

/* face types (S5/S6; the paper names bc_block / bc_phys only) */
#define CFD_FACE_PERIODIC 1
#define CFD_FACE_INTERFACE 2
#define CFD_FACE_WALL_NOSLIP_ADIABATIC 3 /* U13 */
#define CFD_FACE_FARFIELD_CHAR 4         /* U14 */

typedef struct cfd_ctx cfd_ctx; /* opaque, owned by the library */

typedef struct {
  int ni, nj, nk; /* interior sizes (>= 6 each); arrays are (n + 2*CFD_NG) per axis */
} cfd_dims;

typedef struct {
  double gamma;    /* ratio of specific heats (1.4 in the paper) */
  double mach;     /* Ma_inf  (viscous scaling Ma/Re of tau and q) */
  double reynolds; /* Re_inf */
  double prandtl;  /* Pr */
  double weno_eps; /* epsilon of Eq. 15 (1e-6) */
  int viscous;     /* 0 Euler, 1 Navier–Stokes */
  int scheme;      /* 0 modified AFWENO (Fig. 11); 1 original (Fig. 9; default sweep plan only) */
  double q_inf[5]; /* far-field conservative state (rho, rho u, rho v, rho w, e) */
  double sutherland; /* molecular viscosity (U11): > 0: Sutherland's law mu(T) = T^(3/2) (1+S)/(T+S) with
                        S = this value = 110.4 K / T_inf (T_inf = 1, mu(1) = 1); <= 0: constant mu = 1 */
} cfd_params;

typedef struct {
  int block, face;         /* face: 0 -xi, 1 +xi, 2 -eta, 3 +eta, 4 -zeta, 5 +zeta */
  int type;                /* CFD_FACE_* */
  int nbr_block, nbr_face; /* PERIODIC / INTERFACE only */
  int perm[3];             /* my axis a runs along the neighbour's axis perm[a] ... */
  int sign[3];             /* ... in direction sign[a] = +1 / -1 (proper rotations only) */
  double shift[3];         /* (x,y,z) translation added to the neighbour's coordinates when they
                              become my ghost coordinates (periodic images) */
} cfd_face;

typedef struct {
  double* q;    /* [5][M] conservative variables Q = (rho, rho u, rho v, rho w, e), no 1/J */
  double* qn;   /* [5][M] Q^n of Eq. 20 */
  double* r;    /* [5][M] R(Q) */
  double* xyz;  /* [3][M] node coordinates; the caller fills the interior, the library the ghosts */
  double* khat; /* [9][M] hatted metrics, index d*3+c = d(xi^d)/d(x_c) / J  (Eq. 7) */
  double* jac;  /* [1][M] J (Eq. 8) */
} cfd_block_ptrs;

/* Bytes of device scratch the caller must pass to cfd_create_blocks: 12 doubles per stored point of EVERY block
 * (each block has its own area, so that the per-block kernels of a multi-block case can run concurrently: the
 * viscous rows S = d(Fv^xi)/d(xi), Fv^eta, Fv^zeta; the 9 metric first derivatives during cfd_compute_metrics),
 * plus the partial sums of the residual / CFL reductions. */
size_t cfd_workspace_bytes(int nblocks, const cfd_dims* dims, const cfd_params* params);

/* Build a context over nblocks point-matched blocks (a patch is a whole block face).
 * Validates sizes, alignment and the face descriptors: all six faces of every block described exactly once,
 * permutation proper, normal-axis sign consistent with the face pair, tangential extents equal, the two sides of
 * a connection pointing at each other with inverse permutations, at least 7 nodes normal to a wall
 * (CFD_E_TOPOLOGY otherwise).  `workspace` is device memory of at
 * least cfd_workspace_bytes(), caller-owned.  `cuda_stream` is a cudaStream_t (may be 0). */
int cfd_create_blocks(cfd_ctx** out, int nblocks, const cfd_dims* dims, const cfd_block_ptrs* ptrs, int nfaces,
                      const cfd_face* faces, const cfd_params* params, void* workspace, size_t workspace_bytes,
                      void* cuda_stream);

/* NEXT-4 (the paper shards one sub-block set per GPU and exchanges halos over MPI / GPUDirect P2P on
 * PCIe): BLOCK SHARDING over the GPUs of one NVLink / NVSwitch node, one process per
 * GPU.  The same call as cfd_create_blocks over the WHOLE topology (all nblocks blocks, all faces), but this context
 * OWNS only the blocks with local[b] != 0 (local == NULL: all of them); the others are advanced by peer processes.
 * For a peer's block, ptrs[b].q, .qn, .r, .xyz are PEER-MAPPED device pointers to that process's buffers (CUDA IPC /
 * P2P over NVLink; khat, jac may be NULL), given in the same order as the owner passed them, and are only ever READ:
 * cfd_exchange_interfaces (and the xyz fill of cfd_compute_metrics) pull the ghost layers of the local blocks straight
 * out of the owner's interior cells with P2P loads through the same composed index maps -- no packing, no staging
 * buffer, no host copy (on NVSwitch every peer is equidistant, so the paper's topology-aware placement, P:L356–390,
 * has nothing left to decide).  Everything else (metrics, RHS, RK stage, BCs, CFL) runs on the local blocks
 * only; res5 and the CFL maximum are LOCAL sums / maxima: the caller reduces them over the processes.
 * The single-call stages cfd_stage, cfd_stage_fused and cfd_step_host are REFUSED (CFD_E_ARG, nothing enqueued) on a
 * context that has peer-owned blocks: they would run the P2P ghost fill right behind the local sweeps, with no way to
 * know that the peers have finished writing (or have rotated their buffer roles) -- a silent data race.  Use
 * cfd_stage_fused_local -> cross-process barrier -> cfd_exchange_interfaces -> barrier -> cfd_apply_bc instead
 * (paper_2006_07964_b200/sharded.py does).
 * Ordering is the caller's job (the binding does it with collectives on the compute stream): every process must have
 * finished the stage's last sweep before any process runs cfd_exchange_interfaces of that stage, all processes must call
 * the stage functions in lock step (the buffer roles of cfd_stage_fused rotate identically everywhere), and the
 * owners' xyz interiors must be in place before cfd_compute_metrics.  The workspace is sized by
 * cfd_workspace_bytes_sharded (local blocks only). */
int cfd_create_blocks_sharded(cfd_ctx** out, int nblocks, const cfd_dims* dims, const cfd_block_ptrs* ptrs, const int* local,
                              int nfaces, const cfd_face* faces, const cfd_params* params, void* workspace,
                              size_t workspace_bytes, void* cuda_stream);
size_t cfd_workspace_bytes_sharded(int nblocks, const cfd_dims* dims, const int* local, const cfd_params* params);

/* S1 (Eqs. 7–8): fills the ghost layers of xyz (interfaces / periodic shift, wall = odd
 * reflection, far field = linear extrapolation), then khat and jac by 6th-order central differences
 * in conservative form, valid on the index box [-3, n+3)^3 of every block.
 * Returns host values: synchronises the stream; CFD_E_JACOBIAN if J <= 0 at an interior node. */
int cfd_compute_metrics(cfd_ctx*);

/* S2 + S3 (Eqs. 9–19 with Steger–Warming splitting and the modified AFWENO of Fig. 11 -- or, with params.scheme = 1,
 * the original ordering of Fig. 9; Eqs. 5, 6, 21 with 6th-order central differences, mu = 1 or Sutherland's mu(T)):
 * r := J [ sum_d d(Fv^d)/d(xi^d) - sum_d D^d ] on interior points.
 * Requires valid ghost layers in q (cfd_exchange_interfaces + cfd_apply_bc).  Asynchronous. */
int cfd_rhs(cfd_ctx*);

/* S4 (Eq. 20): q <- a q^n + b (q + dt r) on interior points, (a,b) = (0,1), (3/4,1/4), (1/3,2/3) for
 * stage 1, 2, 3; stage 1 first saves q^n := q and accumulates res_m = sum over all blocks' INNER
 * points of r_m^2 ("summation of all inner grid points": every interior node except the node planes that a
 * WALL / FARFIELD face owns -- cfd_apply_bc overwrites those nodes after every stage, r there is never used; U17a)
 * with a fixed-order (run-to-run deterministic) reduction.
 * res5_host_or_null: if non-null (stage 1 only) receives the 5 sums and the stream is synchronised. */
int cfd_rk_stage(cfd_ctx*, int stage, double dt, double* res5_host_or_null);

/* S6: fills the ghost layers of q behind PERIODIC / INTERFACE faces from the
 * neighbour's interior through the signed index permutation, faces then edges then corners. */
int cfd_exchange_interfaces(cfd_ctx*);

/* S5: no-slip adiabatic wall (U13) and characteristic far field (U14) on q: boundary
 * node plane and the 6 ghost layers behind it, tangential index range [-3, n+3). */
int cfd_apply_bc(cfd_ctx*);

/* On-device CFL time step ("time step dt" per point, "reduced-dimensional operation", Fig. 2
 * timestep_gpu; reading U16): s_i = sum_d ( |k_d . u| + c |k_d| ), k_d = J khat^d, at every interior point of every
 * block from the current q; *dt_host = cfl / max_i s_i (MAX reduction: order-independent, deterministic).
 * dt_local_dev_or_null: if non-null, one DEVICE pointer per block to a caller-owned array of M doubles (field layout with
 * ghosts); the local time step cfl / s_i is written at interior points (ghost entries untouched).
 * Requires cfd_compute_metrics.  One bandwidth-bound pass over q, khat, jac (120 B per point).
 * Returns host values: synchronises the stream.  CFD_E_ARG if cfl <= 0 or the state is not physical: a single interior
 * point with rho <= 0, p < 0 or a NaN makes s_i NaN, the reduction keeps NaNs (it is not an fmax), and the call fails
 * instead of returning a dt from the remaining points (dt_local then holds NaN at the offending points). */
int cfd_cfl_dt(cfd_ctx*, double cfl, double* dt_host, double* const* dt_local_dev_or_null);

/* Convenience: the four calls above for one stage, in Fig. 2's order, on the context's stream. */
int cfd_stage(cfd_ctx*, int stage, double dt, double* res5_host_or_null);

/* The same stage with the RK update fused into the last inviscid sweep: the zeta sweep forms R = J (r + X) point by point and writes a q^n + b (q + dt R) (Eq. 20) straight
 * into the r buffer, so R is never stored and no separate RK pass runs; stage 1 also reduces res_m = sum R_m^2
 * (fixed order).  Because q cannot be overwritten while neighbouring points still read it, the three state
 * buffers of every block EXCHANGE ROLES instead of being copied: after stage 1 the old r buffer holds q, the old
 * q buffer holds q^n and the old q^n buffer is the scratch r; after stages 2 and 3 q and r swap.
 * cfd_buffer_roles tells which of the caller's buffers currently plays which role; every other entry point
 * (cfd_rhs, cfd_rk_stage, cfd_exchange_interfaces, cfd_apply_bc, cfd_step_host) follows the current roles.
 * The contents of the r buffer after this call are scratch.  res5_host_or_null as in cfd_rk_stage. */
int cfd_stage_fused(cfd_ctx*, int stage, double dt, double* res5_host_or_null);

/* The part of cfd_stage_fused that touches the context's own blocks only: S2 + S3 with S4 inside the last sweep and the
 * exchange of the buffer roles, WITHOUT the ghost fill and the physical BCs.  A sharded context (cfd_create_blocks_sharded)
 * calls this, lets every process reach the same point (a collective on the compute stream), and then calls
 * cfd_exchange_interfaces and cfd_apply_bc; on an unsharded context the three calls in a row are cfd_stage_fused. */
int cfd_stage_fused_local(cfd_ctx*, int stage, double dt, double* res5_host_or_null);

/* roles[0], roles[1], roles[2] = which buffer of cfd_block_ptrs (0 = the one passed as q, 1 = qn, 2 = r)
 * currently holds Q, Q^n and R / scratch.  (0, 1, 2) until cfd_stage_fused or cfd_step_host is used. */
int cfd_buffer_roles(const cfd_ctx*, int roles[3]);

/* End-to-end entry with HOST buffers (bench.py's e2e leg): for every block b, copies the interior state
 * q_in_host[b] (layout [5][nk][nj][ni], fp64, i fastest, no ghost layers; pinned memory recommended)
 * into the device q, fills ghosts (S6, S5), runs one TVD-RK3 step (three cfd_stage_fused calls, Eq. 20,
 * P:L173–180), copies the interior of q back into q_out_host[b] (same layout; may alias q_in_host[b])
 * and synchronises the stream.  res5_host_or_null as in cfd_rk_stage.  Returns host values. */
int cfd_step_host(cfd_ctx*, const double* const* q_in_host, double* const* q_out_host, double dt,
                  double* res5_host_or_null);

/* Per-kernel device timing (bench.py's roofline leg).  While enabled, every kernel launch of the hot
 * path is bracketed by CUDA events on the context's stream.  cfd_profile_read synchronises the stream,
 * writes, for each kernel class id < CFD_PROF_NCLASS, the summed device time in ms and the number of
 * launches since the last read, and resets the counters.  cfd_profile_name(id) is a static string. */
#define CFD_PROF_NCLASS 12
int cfd_profile_enable(cfd_ctx*, int on);
int cfd_profile_read(cfd_ctx*, double ms[CFD_PROF_NCLASS], long long launches[CFD_PROF_NCLASS]);
const char* cfd_profile_name(int id);

/* Measurement aid (power / clock measurements of one kernel class looped alone, profiles/r2_power.md): cfd_rhs and
 * cfd_stage_fused launch only the hot kernel classes whose bit (1 << class id: 0 xi sweep, 1 eta sweep, 2 zeta sweep,
 * 3 viscous point fluxes) is set in mask.  With any of these bits clear the RESULTS ARE INVALID; the default is all ones.
 * While such a mask is active every cfd_rhs / cfd_stage_fused[_local] call still returns 0 but leaves "cfd_profile_only mask
 * active ... INVALID" in cfd_last_error, so that a masked result cannot pass for a valid one; restoring all ones clears it. */
int cfd_profile_only(cfd_ctx*, unsigned mask);

/* ---- For callers that cannot allocate device memory --------------------------------------------------------------
 * S4, stage 1 (Eq. 20: q^n := q, q := q + dt r) with the residual res_m = sum over the interior points of
 * r_m^2 (U17) for ONE block, WITHOUT a context and without any workspace.
 *
 * Who needs it: everything else in this header goes through cfd_create_blocks, which calls cudaMalloc and wants a
 * caller-allocated workspace.  That is impossible for a solver plug-in whose host application has already reserved all of
 * the device memory for its own arena (cudaMalloc just returns out-of-memory there), for a coupling / in-situ loop that
 * may not stall the GPU (cudaMalloc and cudaFree synchronise against every stream of the device), and for a callback that
 * is simply handed q and r by somebody else and owns no allocator.  Such a caller passes only its inputs and outputs;
 * the per-CTA partial sums of the reduction live in a fixed array inside the library image.
 *
 * Arguments: q (in/out), qn (out), r (in): DEVICE pointers, fp64, layout [5][nk+12][nj+12][ni+12] with the CFD_NG ghost
 * layers like cfd_block_ptrs (ghost entries are neither read nor written), 8-byte aligned, caller-owned; ni, nj, nk >= 1;
 * res5_dev: DEVICE pointer to 5 doubles receiving res_m (read it back on the same stream when you need it);
 * cuda_stream: a cudaStream_t of the CURRENT device (may be 0).  Asynchronous; never synchronises.  For a block within
 * the limit the values of q, qn and res are those cfd_rk_stage(ctx, 1, dt, res) produces (same summation order) for a
 * block without WALL / FARFIELD faces; this call knows no face types and sums over ALL interior nodes, whereas
 * cfd_rk_stage leaves out the node planes such faces own.
 *
 * Limit: ni*nj*nk <= CFD_STATIC_MAX_POINTS (2 097 152 = 128^3 interior points); larger blocks are refused with
 * CFD_E_WORKSPACE and a message naming both numbers -- nothing is launched.  Cost: the built-in array takes
 * CFD_STATIC_SCRATCH_BYTES (320 KB) of device memory on every GPU that loads this library, from load until process exit.
 *
 * Set-up: the FIRST call on each device looks up that device's address of the built-in array (cudaGetSymbolAddress, with
 * the device current, which also makes the runtime load the library's kernels there) and caches it; make that first call
 * during start-up, before you begin any stream capture.  After it the call only launches two kernels: no cudaMalloc,
 * cudaFree or other allocating routine, ever.
 *
 * Sharing: there is ONE array per device and every call uses it.  It keeps whatever the previous call left in it; that is
 * harmless because each call overwrites every slot it later reads (nothing has to start at zero, so nothing is cleared).
 * Two calls that may run on the same GPU at the same time (different streams, or different host threads on different
 * streams) RACE on it and give wrong residuals: issue all calls for one device on one stream, or order them with events.
 *
 * Errors: CFD_E_ARG (null / misaligned pointer, size < 1), CFD_E_WORKSPACE (block too large), CFD_E_CUDA (runtime call
 * failed); cfd_static_last_error() returns the message of the calling thread's last failing call ("" after a success). */
#define CFD_STATIC_MAX_POINTS 2097152
#define CFD_STATIC_SCRATCH_BYTES 327680
int cfd_rk_stage1_static(double* q, double* qn, const double* r, int ni, int nj, int nk, double dt, double* res5_dev,
                         void* cuda_stream);
const char* cfd_static_last_error(void);

/* Frees the context (never the caller's buffers). */
int cfd_destroy(cfd_ctx*);

/* Message for the most recent failing call on this context (or on creation if ctx == NULL). */
const char* cfd_last_error(const cfd_ctx*);

/* Number of kernel launches enqueued by this context so far (for bench.py's gpu_launches). */
long long cfd_launch_count(const cfd_ctx*);

/* Register-resident DFMA loop on the context-free default stream: measures the plain FP64 FMA
 * throughput of the device (the "alu" roofline denominator).  Returns host values (TFLOP/s,
 * FMA = 2 flops) in *tflops; synchronises. */
int cfd_fp64_peak_probe(int iters, double* tflops);

/* Kernel of the xi sweep inside cfd_rhs / cfd_stage_fused (all choices compute the same R up to summation order).
 * All three sweeps are MARCHING sweeps (one thread walks a grid line segment; every operand staged once per point through
 * shared memory); the xi sweep, whose lanes sit on lines a row pitch apart, runs out of a per-warp ring of 4-position
 * chunks in shared memory:
 *   0 (default)  ring filled by warp-cooperative 16-byte cp.async with a hand-made 32-byte swizzle, r written with 16-byte
 *                stores (k_xi_ldg); blocks with odd ni (row pitch not a multiple of 16 bytes) use plan 4's kernel;
 *   4            8-byte cp.async staging into padded per-line rings (k_march_xi), any ni;
 *   5            ring filled by TMA boxes 4 x 32 x 1 x nvar with SWIZZLE_32B and written back by TMA stores (k_xi_tma;
 *                correct, kept for measurement: the TMA unit is the bottleneck for 32-byte box rows); scheme 0 only.
 * Other values (the tiled one-thread-per-point kernels of round 1, plans 1-3 and 6) are rejected with CFD_E_ARG: they were
 * retired after profiles/r1_*.md settled the comparison. */
int cfd_set_sweep_plan(cfd_ctx*, int plan);

/* Tile of the viscous point-flux kernel (k_visc_march; all choices compute the same values bit for bit): -1 (default) picks,
 * per block, the geometry with the fewest thread-planes; 0 = 64 x 8 threads (58 output columns per tile row), 1 = 70 x 7
 * (64 columns), 2 = 54 x 9 (48 columns).  For tests and measurements. */
int cfd_set_visc_tile(cfd_ctx*, int tile);

/* Device self-test of the branch-free fp64 reciprocal / reciprocal square root the hot kernels use instead
 * of IEEE division (csrc/fastmath.cuh): for n HOST values x > 0 writes 1/x and 1/sqrt(x) as the kernels compute
 * them into the HOST arrays rcp_out, rsqrt_out (tests compare with correctly rounded results).  Allocates
 * and frees its own scratch; synchronises.  Not on the hot path. */
int cfd_selftest_fastmath(int n, const double* x_host, double* rcp_out_host, double* rsqrt_out_host);

#ifdef __cplusplus
}
#endif
#endif /* CFD_B200_H */
