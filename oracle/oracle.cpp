// =====================================================================================
// ORACLE — TEST INFRASTRUCTURE, NOT PRODUCT CODE.  See oracle_core.hpp for the header
// statement, citations and parity status.  This file holds the block-level loops (ghost
// fill, metrics, RHS assembly, RK stage, boundary conditions) and the C entry points the
// tests load with ctypes.  Shares no code with paper_2006_07964_b200/csrc.
// =====================================================================================
#include "oracle_core.hpp"

#include <algorithm>
#include <cstdio>
#include <cstring>
#ifdef _OPENMP
#include <omp.h>
#endif

namespace orc {

static inline int axis_of(int face) { return face / 2; }
static inline int side_of(int face) { return face % 2; }
static inline bool is_connect(int t) { return t == FT_PERIODIC || t == FT_INTERFACE; }

int Solver::create(int nblocks, const int* dims, int nfaces, const Face* f, const Params* p) {
  prm = *p;
  blk.resize(nblocks);
  for (int b = 0; b < nblocks; ++b) {
    Block& B = blk[b];
    for (int a = 0; a < 3; ++a) {
      B.n[a] = dims[3 * b + a];
      if (B.n[a] < NG) { err = "block interior size must be >= 6 on every axis"; return -1; }
      B.m[a] = B.n[a] + 2 * NG;
    }
    B.M = size_t(B.m[0]) * B.m[1] * B.m[2];
    B.q.assign(5 * B.M, 0.0);
    B.qn.assign(5 * B.M, 0.0);
    B.r.assign(5 * B.M, 0.0);
    B.xyz.assign(3 * B.M, 0.0);
    B.khat.assign(9 * B.M, 0.0);
    B.jac.assign(B.M, 0.0);
    for (int s = 0; s < 6; ++s) { B.ftype[s] = FT_NONE; B.fidx[s] = -1; }
  }
  faces.assign(f, f + nfaces);
  for (int t = 0; t < nfaces; ++t) {
    const Face& F = faces[t];
    if (F.block < 0 || F.block >= nblocks || F.face < 0 || F.face > 5) { err = "face: bad block/face id"; return -2; }
    Block& B = blk[F.block];
    if (B.fidx[F.face] != -1) { err = "face described twice"; return -2; }
    B.ftype[F.face] = F.type;
    B.fidx[F.face] = t;
    if (is_connect(F.type)) {
      if (F.nbr_block < 0 || F.nbr_block >= nblocks || F.nbr_face < 0 || F.nbr_face > 5) { err = "face: bad neighbour"; return -2; }
      // perm must be a permutation, signs +-1, proper rotation
      int seen[3] = {0, 0, 0};
      for (int a = 0; a < 3; ++a) {
        if (F.perm[a] < 0 || F.perm[a] > 2 || (F.sign[a] != 1 && F.sign[a] != -1)) { err = "face: bad perm/sign"; return -2; }
        seen[F.perm[a]]++;
      }
      if (seen[0] != 1 || seen[1] != 1 || seen[2] != 1) { err = "face: perm is not a permutation"; return -2; }
      int par = ((F.perm[0] == 0 && F.perm[1] == 1) || (F.perm[0] == 1 && F.perm[1] == 2) || (F.perm[0] == 2 && F.perm[1] == 0)) ? 1 : -1;
      if (par * F.sign[0] * F.sign[1] * F.sign[2] != 1) { err = "face: not a proper rotation"; return -2; }
      int an = axis_of(F.face);
      if (F.perm[an] != axis_of(F.nbr_face)) { err = "face: nbr_face axis != perm[normal axis]"; return -2; }
      int want = (side_of(F.face) != side_of(F.nbr_face)) ? 1 : -1;
      if (F.sign[an] != want) { err = "face: normal-axis sign inconsistent with the face pair"; return -2; }
      const Block& N = blk[F.nbr_block];
      for (int a = 0; a < 3; ++a)
        if (a != an && N.n[F.perm[a]] != B.n[a]) { err = "face: interface extents do not match"; return -2; }
    } else if (F.type != FT_WALL && F.type != FT_FARFIELD) {
      err = "face: unknown type"; return -2;
    }
  }
  return 0;
}

// Index map through (perm, sign) — reading U15: ghost layer g of my face is the neighbour's
// interior layer g-1 counted from its matching face; tangential axes match over the whole face.
int Solver::map_index(const Face& F, const int me[3], int nb[3]) const {
  const Block& B = blk[F.block];
  const Block& N = blk[F.nbr_block];
  const int an = axis_of(F.face);
  for (int a = 0; a < 3; ++a) {
    const int ap = F.perm[a];
    if (a == an) {
      const int s = side_of(F.face), sp = side_of(F.nbr_face);
      if (s == 0 && sp == 1) nb[ap] = me[a] + N.n[ap];
      else if (s == 0 && sp == 0) nb[ap] = -me[a] - 1;
      else if (s == 1 && sp == 0) nb[ap] = me[a] - B.n[a];
      else nb[ap] = N.n[ap] + B.n[a] - 1 - me[a];
    } else {
      nb[ap] = (F.sign[a] > 0) ? me[a] : (B.n[a] - 1 - me[a]);
    }
  }
  return 0;
}

// S6 (P:L262 bc_block, L301 "exchanged on GPU without leaving the device"; reading U15).
// Three passes: pass p fills the ghost cells that have exactly p indices out of range from
// cells with p-1 indices out of range (faces, then edges, then corners).  A cell that lies
// beyond several faces is filled through the lowest axis whose face is PERIODIC/INTERFACE.
void Solver::fill_connect(int field) {
  const int nv = field == 0 ? 5 : 3;
  for (int pass = 1; pass <= 3; ++pass) {
    for (size_t b = 0; b < blk.size(); ++b) {
      Block& B = blk[b];
      std::vector<double>& dst = field == 0 ? B.q : B.xyz;
#pragma omp parallel for schedule(static) num_threads(nthreads)
      for (int k = -NG; k < B.n[2] + NG; ++k)
        for (int j = -NG; j < B.n[1] + NG; ++j)
          for (int i = -NG; i < B.n[0] + NG; ++i) {
            const int me[3] = {i, j, k};
            int nout = 0, fsel = -1;
            for (int a = 0; a < 3; ++a) {
              int fc = -1;
              if (me[a] < 0) fc = 2 * a;
              else if (me[a] >= B.n[a]) fc = 2 * a + 1;
              if (fc >= 0) {
                ++nout;
                if (fsel < 0 && is_connect(B.ftype[fc])) fsel = fc;
              }
            }
            if (nout != pass || fsel < 0) continue;
            const Face& F = faces[B.fidx[fsel]];
            int nb[3];
            map_index(F, me, nb);
            const Block& N = blk[F.nbr_block];
            const std::vector<double>& src = field == 0 ? N.q : N.xyz;
            const size_t id = B.idx(i, j, k), is = N.idx(nb[0], nb[1], nb[2]);
            for (int v = 0; v < nv; ++v) {
              double val = src[v * N.M + is];
              if (field == 1) val += F.shift[v];
              dst[v * B.M + id] = val;
            }
          }
    }
  }
}

// Ghost coordinates behind physical-boundary faces: WALL = odd (point) reflection about the
// boundary node (U13), FARFIELD = linear extrapolation (U14).  Whole tangential extent.
void Solver::bc_xyz() {
  for (const Face& F : faces) {
    if (F.type != FT_WALL && F.type != FT_FARFIELD) continue;
    Block& B = blk[F.block];
    const int an = axis_of(F.face), s = side_of(F.face);
    const int t1 = (an + 1) % 3, t2 = (an + 2) % 3;
    const int bnode = s == 0 ? 0 : B.n[an] - 1;
    const int dir = s == 0 ? 1 : -1;  // towards the interior
    for (int b2 = -NG; b2 < B.n[t2] + NG; ++b2)
      for (int b1 = -NG; b1 < B.n[t1] + NG; ++b1)
        for (int g = 1; g <= NG; ++g) {
          int pb[3], pg[3], pi[3];
          pb[an] = bnode; pb[t1] = b1; pb[t2] = b2;
          pg[an] = bnode - g * dir; pg[t1] = b1; pg[t2] = b2;
          pi[t1] = b1; pi[t2] = b2;
          for (int c = 0; c < 3; ++c) {
            double xb = B.xyz[c * B.M + B.idx(pb[0], pb[1], pb[2])];
            double val;
            if (F.type == FT_WALL) {
              pi[an] = bnode + g * dir;
              val = 2.0 * xb - B.xyz[c * B.M + B.idx(pi[0], pi[1], pi[2])];
            } else {
              pi[an] = bnode + dir;
              val = xb + double(g) * (xb - B.xyz[c * B.M + B.idx(pi[0], pi[1], pi[2])]);
            }
            B.xyz[c * B.M + B.idx(pg[0], pg[1], pg[2])] = val;
          }
        }
  }
}

// S1 / O1: conservative metrics Eq. 7 and Jacobian Eq. 8, 6th-order central.
// Valid on the box [-3, n+3)^3 of every block; untouched elsewhere.
int Solver::compute_metrics() {
  fill_connect(1);
  bc_xyz();
  for (Block& B : blk) {
    const size_t M = B.M;
    // first derivatives xd[c][d] = d x_c / d xi^d ; valid where the index along d is in [-3, n+3)
    std::vector<double> xd(9 * M, 0.0);
    for (int c = 0; c < 3; ++c)
      for (int d = 0; d < 3; ++d) {
        const size_t st = B.stride(d);
        const double* x = &B.xyz[c * M];
        double* o = &xd[(c * 3 + d) * M];
        int lo[3] = {-NG, -NG, -NG}, hi[3] = {B.n[0] + NG, B.n[1] + NG, B.n[2] + NG};
        lo[d] = -3; hi[d] = B.n[d] + 3;
#pragma omp parallel for schedule(static) num_threads(nthreads)
        for (int k = lo[2]; k < hi[2]; ++k)
          for (int j = lo[1]; j < hi[1]; ++j)
            for (int i = lo[0]; i < hi[0]; ++i) {
              const size_t p = B.idx(i, j, k);
              o[p] = d6(x[p - 3 * st], x[p - 2 * st], x[p - st], x[p + st], x[p + 2 * st], x[p + 3 * st]);
            }
      }
    // Eq. 7: khat^d_c = delta_{d2}( (x_{c1})_{d1} x_{c2} ) - delta_{d1}( (x_{c1})_{d2} x_{c2} ),
    // (d, d1, d2) and (c, c1, c2) cyclic.
    for (int d = 0; d < 3; ++d)
      for (int c = 0; c < 3; ++c) {
        const int d1 = (d + 1) % 3, d2 = (d + 2) % 3, c1 = (c + 1) % 3, c2 = (c + 2) % 3;
        const double* a1 = &xd[(c1 * 3 + d1) * M];  // (x_{c1})_{d1}
        const double* a2 = &xd[(c1 * 3 + d2) * M];  // (x_{c1})_{d2}
        const double* x2 = &B.xyz[c2 * M];
        const size_t s1 = B.stride(d1), s2 = B.stride(d2);
        double* o = &B.khat[(d * 3 + c) * M];
#pragma omp parallel for schedule(static) num_threads(nthreads)
        for (int k = -3; k < B.n[2] + 3; ++k)
          for (int j = -3; j < B.n[1] + 3; ++j)
            for (int i = -3; i < B.n[0] + 3; ++i) {
              const size_t p = B.idx(i, j, k);
              auto P1 = [&](ptrdiff_t off) { return a1[p + off] * x2[p + off]; };
              auto P2 = [&](ptrdiff_t off) { return a2[p + off] * x2[p + off]; };
              const ptrdiff_t S1 = ptrdiff_t(s1), S2 = ptrdiff_t(s2);
              double t1 = d6(P1(-3 * S2), P1(-2 * S2), P1(-S2), P1(S2), P1(2 * S2), P1(3 * S2));
              double t2 = d6(P2(-3 * S1), P2(-2 * S1), P2(-S1), P2(S1), P2(2 * S1), P2(3 * S1));
              o[p] = t1 - t2;
            }
      }
    // Eq. 8 in the printed order
    bool bad = false;
    for (int k = -3; k < B.n[2] + 3; ++k)
      for (int j = -3; j < B.n[1] + 3; ++j)
        for (int i = -3; i < B.n[0] + 3; ++i) {
          const size_t p = B.idx(i, j, k);
          auto X = [&](int c, int d) { return xd[(c * 3 + d) * M + p]; };
          double ji = X(0, 0) * X(1, 1) * X(2, 2) - X(0, 0) * X(1, 2) * X(2, 1) + X(0, 1) * X(1, 2) * X(2, 0) -
                      X(0, 1) * X(1, 0) * X(2, 2) + X(0, 2) * X(1, 0) * X(2, 1) - X(0, 2) * X(1, 1) * X(2, 0);
          B.jac[p] = 1.0 / ji;
          const bool interior = i >= 0 && i < B.n[0] && j >= 0 && j < B.n[1] && k >= 0 && k < B.n[2];
          if (interior && !(ji > 0.0)) bad = true;
        }
    if (bad) { err = "J <= 0 at an interior node"; return -3; }
  }
  return 0;
}

// S2 + S3 / O2 + O3: r := J [ (V^xi + V^eta + V^zeta) - (D^xi + D^eta + D^zeta) ] on interior
// points (Eq. 2 with U~ = Q/J on a static grid; accumulation order = reading U18).
int Solver::rhs() {
  const double gamma = prm.gamma, eps = prm.weno_eps;
  for (Block& B : blk) {
    const size_t M = B.M;
    std::vector<double> accD(5 * M, 0.0), accV(5 * M, 0.0);
    // ---- inviscid, d = xi, eta, zeta ------------------------------------------------
    for (int d = 0; d < 3; ++d) {
      const int t1 = (d + 1) % 3, t2 = (d + 2) % 3;
      const int n = B.n[d];
      const size_t st = B.stride(d);
#pragma omp parallel num_threads(nthreads)
      {
        std::vector<double> Qb(5 * (n + 2 * NG)), kb(3 * (n + 2 * NG)), Db(5 * n);
        const double* Ql[5]; const double* kl[3]; double* D[5];
        for (int m = 0; m < 5; ++m) { Ql[m] = &Qb[m * (n + 2 * NG)]; D[m] = &Db[m * n]; }
        for (int c = 0; c < 3; ++c) kl[c] = &kb[c * (n + 2 * NG)];
#pragma omp for schedule(static) collapse(2)
        for (int b2 = 0; b2 < B.n[t2]; ++b2)
          for (int b1 = 0; b1 < B.n[t1]; ++b1) {
            int p0[3]; p0[d] = 0; p0[t1] = b1; p0[t2] = b2;
            const size_t base = B.idx(p0[0], p0[1], p0[2]);
            for (int i = -NG; i < n + NG; ++i) {
              const size_t p = base + ptrdiff_t(i) * ptrdiff_t(st);
              for (int m = 0; m < 5; ++m) Qb[m * (n + 2 * NG) + NG + i] = B.q[m * M + p];
              // metrics are only valid to depth 3; deeper entries are never read by inviscid_line
              for (int c = 0; c < 3; ++c) kb[c * (n + 2 * NG) + NG + i] = B.khat[(d * 3 + c) * M + p];
            }
            inviscid_line<double>(n, Ql, kl, gamma, eps, prm.scheme, D);
            for (int i = 0; i < n; ++i) {
              const size_t p = base + size_t(i) * st;
              for (int m = 0; m < 5; ++m) accD[m * M + p] += Db[m * n + i];
            }
          }
      }
    }
    // ---- viscous ---------------------------------------------------------------------
    if (prm.viscous) {
      const double mu0 = prm.mach / prm.reynolds;                      // Ma/Re: the factor of tau and q (U9)
      // pass A (cuda_vars_derv_xyz, Fig. 12): Cartesian gradients of (u,v,w,T) on interior + 3 face layers
      std::vector<double> G(12 * M, 0.0);
#pragma omp parallel for schedule(static) num_threads(nthreads)
      for (int k = -3; k < B.n[2] + 3; ++k)
        for (int j = -3; j < B.n[1] + 3; ++j)
          for (int i = -3; i < B.n[0] + 3; ++i) {
            const int nout = (i < 0 || i >= B.n[0]) + (j < 0 || j >= B.n[1]) + (k < 0 || k >= B.n[2]);
            if (nout > 1) continue;
            const size_t p = B.idx(i, j, k);
            double dphi[3][4];
            for (int d = 0; d < 3; ++d) {
              const ptrdiff_t st = ptrdiff_t(B.stride(d));
              double ph[7][4];
              for (int s = -3; s <= 3; ++s) {
                if (s == 0) continue;
                double Q[5];
                for (int m = 0; m < 5; ++m) Q[m] = B.q[m * M + p + s * st];
                phi_point(Q, gamma, ph[s + 3]);
              }
              for (int f = 0; f < 4; ++f) dphi[d][f] = d6(ph[0][f], ph[1][f], ph[2][f], ph[4][f], ph[5][f], ph[6][f]);
            }
            double kh[3][3], g[3][4];
            for (int d = 0; d < 3; ++d)
              for (int c = 0; c < 3; ++c) kh[d][c] = B.khat[(d * 3 + c) * M + p];
            grad_point(dphi, kh, B.jac[p], g);
            for (int c = 0; c < 3; ++c)
              for (int f = 0; f < 4; ++f) G[(c * 4 + f) * M + p] = g[c][f];
          }
      // pass B (cuda_vflux_flux + cuda_vflux_df): point viscous flux along d, then its 6th-order derivative
      for (int d = 0; d < 3; ++d) {
        std::vector<double> Fv(5 * M, 0.0);
        int lo[3] = {0, 0, 0}, hi[3] = {B.n[0], B.n[1], B.n[2]};
        lo[d] = -3; hi[d] = B.n[d] + 3;
#pragma omp parallel for schedule(static) num_threads(nthreads)
        for (int k = lo[2]; k < hi[2]; ++k)
          for (int j = lo[1]; j < hi[1]; ++j)
            for (int i = lo[0]; i < hi[0]; ++i) {
              const size_t p = B.idx(i, j, k);
              double Q[5], ph[4], g[3][4], kd[3], F[5];
              for (int m = 0; m < 5; ++m) Q[m] = B.q[m * M + p];
              phi_point(Q, gamma, ph);
              for (int c = 0; c < 3; ++c) {
                kd[c] = B.khat[(d * 3 + c) * M + p];
                for (int f = 0; f < 4; ++f) g[c][f] = G[(c * 4 + f) * M + p];
              }
              const double mu = mu0 * sutherland_mu(ph[3], prm.sutherland);   // (Ma/Re) mu(T); mu = 1 without Sutherland (U11)
              const double kappa = mu / (prm.prandtl * (gamma - 1.0));
              visc_flux_point(ph, g, kd, mu, kappa, F);
              for (int m = 0; m < 5; ++m) Fv[m * M + p] = F[m];
            }
        const ptrdiff_t st = ptrdiff_t(B.stride(d));
#pragma omp parallel for schedule(static) num_threads(nthreads)
        for (int k = 0; k < B.n[2]; ++k)
          for (int j = 0; j < B.n[1]; ++j)
            for (int i = 0; i < B.n[0]; ++i) {
              const size_t p = B.idx(i, j, k);
              for (int m = 0; m < 5; ++m) {
                const double* f = &Fv[m * M];
                accV[m * M + p] += d6(f[p - 3 * st], f[p - 2 * st], f[p - st], f[p + st], f[p + 2 * st], f[p + 3 * st]);
              }
            }
      }
    }
#pragma omp parallel for schedule(static) num_threads(nthreads)
    for (int k = 0; k < B.n[2]; ++k)
      for (int j = 0; j < B.n[1]; ++j)
        for (int i = 0; i < B.n[0]; ++i) {
          const size_t p = B.idx(i, j, k);
          for (int m = 0; m < 5; ++m) B.r[m * M + p] = B.jac[p] * (accV[m * M + p] - accD[m * M + p]);
        }
  }
  return 0;
}

// S4 / O4: Eq. 20 written as Q <- a Q^n + b (Q + dt R), (a,b) = (0,1), (3/4,1/4), (1/3,2/3);
// stage 1 saves Q^n and returns res_m = sum of R_m^2 over the INNER grid points ("summation of all inner grid
// points"; readings U17, U17a): the node planes a physical boundary condition owns (WALL / FARFIELD faces: the BC
// overwrites those nodes after every stage, R there is never used) are not inner points and are left out of the sum.
int Solver::rk_stage(int stage, double dt, double* res5) {
  if (stage < 1 || stage > 3) { err = "stage must be 1..3"; return -4; }
  const double a = stage == 1 ? 0.0 : (stage == 2 ? 3.0 / 4.0 : 1.0 / 3.0);
  const double b = stage == 1 ? 1.0 : (stage == 2 ? 1.0 / 4.0 : 2.0 / 3.0);
  double res[5] = {0, 0, 0, 0, 0};
  for (size_t bi = 0; bi < blk.size(); ++bi) {
    Block& B = blk[bi];
    const size_t M = B.M;
    bool owned[6] = {false, false, false, false, false, false};  // faces of this block with a physical BC (types 3, 4)
    for (const Face& F : faces)
      if (F.block == (int)bi && (F.type == 3 || F.type == 4)) owned[F.face] = true;
    for (int k = 0; k < B.n[2]; ++k)
      for (int j = 0; j < B.n[1]; ++j)
        for (int i = 0; i < B.n[0]; ++i) {
          const size_t p = B.idx(i, j, k);
          for (int m = 0; m < 5; ++m) {
            const size_t e = m * M + p;
            if (stage == 1) {
              const bool bc_node = (owned[0] && i == 0) || (owned[1] && i == B.n[0] - 1) || (owned[2] && j == 0) ||
                                   (owned[3] && j == B.n[1] - 1) || (owned[4] && k == 0) || (owned[5] && k == B.n[2] - 1);
              B.qn[e] = B.q[e];
              if (!bc_node) res[m] += B.r[e] * B.r[e];
              B.q[e] = B.q[e] + dt * B.r[e];
            } else {
              B.q[e] = a * B.qn[e] + b * (B.q[e] + dt * B.r[e]);
            }
          }
        }
  }
  if (res5 && stage == 1) for (int m = 0; m < 5; ++m) res5[m] = res[m];
  return 0;
}

int Solver::exchange_interfaces() { fill_connect(0); return 0; }

// S5: physical boundary conditions (the paper gives no formulas; readings U13, U14).
// Applied on the tangential range [-3, n+3) so that the edge ghosts the viscous terms read are set.
int Solver::apply_bc() {
  const double gamma = prm.gamma, g1 = gamma - 1.0;
  for (const Face& F : faces) {
    if (F.type != FT_WALL && F.type != FT_FARFIELD) continue;
    Block& B = blk[F.block];
    const size_t M = B.M;
    const int an = axis_of(F.face), s = side_of(F.face);
    const int t1 = (an + 1) % 3, t2 = (an + 2) % 3;
    const int bnode = s == 0 ? 0 : B.n[an] - 1;
    const int dir = s == 0 ? 1 : -1;
    for (int b2 = -3; b2 < B.n[t2] + 3; ++b2)
      for (int b1 = -3; b1 < B.n[t1] + 3; ++b1) {
        auto at = [&](int off) {
          int p[3]; p[an] = bnode + off * dir; p[t1] = b1; p[t2] = b2;
          return B.idx(p[0], p[1], p[2]);
        };
        const size_t pb = at(0);
        if (F.type == FT_WALL) {
          // U13: no-slip adiabatic wall on the node plane; dp/dn = dT/dn = 0 to 4th order
          double pp[5], TT[5];
          for (int l = 1; l <= 4; ++l) {
            double Q[5];
            for (int m = 0; m < 5; ++m) Q[m] = B.q[m * M + at(l)];
            Prim<double> st = prims(Q, gamma);
            pp[l] = st.p; TT[l] = gamma * st.p / st.rho;
          }
          const double p0 = (48.0 * pp[1] - 36.0 * pp[2] + 16.0 * pp[3] - 3.0 * pp[4]) / 25.0;
          const double T0 = (48.0 * TT[1] - 36.0 * TT[2] + 16.0 * TT[3] - 3.0 * TT[4]) / 25.0;
          const double r0 = gamma * p0 / T0;
          B.q[0 * M + pb] = r0; B.q[1 * M + pb] = 0.0; B.q[2 * M + pb] = 0.0; B.q[3 * M + pb] = 0.0;
          B.q[4 * M + pb] = p0 / g1;
          for (int g = 1; g <= NG; ++g) {
            const size_t pg = at(-g), pi = at(g);
            B.q[0 * M + pg] = B.q[0 * M + pi];
            B.q[1 * M + pg] = -B.q[1 * M + pi];
            B.q[2 * M + pg] = -B.q[2 * M + pi];
            B.q[3 * M + pg] = -B.q[3 * M + pi];
            B.q[4 * M + pg] = B.q[4 * M + pi];
          }
        } else {
          // U14: characteristic far field from Riemann invariants along the outward normal
          double kn[3];
          for (int c = 0; c < 3; ++c) kn[c] = B.khat[(an * 3 + c) * M + pb];
          const double kl = std::sqrt(kn[0] * kn[0] + kn[1] * kn[1] + kn[2] * kn[2]);
          const double so = s == 1 ? 1.0 : -1.0;
          const double nx = so * kn[0] / kl, ny = so * kn[1] / kl, nz = so * kn[2] / kl;
          double Qi[5];
          for (int m = 0; m < 5; ++m) Qi[m] = B.q[m * M + at(1)];
          Prim<double> si = prims(Qi, gamma), sf = prims(prm.q_inf, gamma);
          const double uni = si.u * nx + si.v * ny + si.w * nz;
          const double unf = sf.u * nx + sf.v * ny + sf.w * nz;
          const double Rp = uni + 2.0 * si.c / g1;
          const double Rm = unf - 2.0 * sf.c / g1;
          const double Vn = 0.5 * (Rp + Rm);
          const double cb = 0.25 * g1 * (Rp - Rm);
          double rho, u, v, w, p;
          if (Vn >= cb) {            // supersonic outflow: everything from the interior
            rho = si.rho; u = si.u; v = si.v; w = si.w; p = si.p;
          } else if (Vn <= -cb) {    // supersonic inflow: everything from the far field
            rho = sf.rho; u = sf.u; v = sf.v; w = sf.w; p = sf.p;
          } else {
            const Prim<double>& sr = (Vn >= 0.0) ? si : sf;
            const double unr = (Vn >= 0.0) ? uni : unf;
            const double ent = sr.p / std::pow(sr.rho, gamma);
            u = sr.u + (Vn - unr) * nx; v = sr.v + (Vn - unr) * ny; w = sr.w + (Vn - unr) * nz;
            rho = std::pow(cb * cb / (gamma * ent), 1.0 / g1);
            p = rho * cb * cb / gamma;
          }
          double Qb[5] = {rho, rho * u, rho * v, rho * w, p / g1 + 0.5 * rho * (u * u + v * v + w * w)};
          for (int m = 0; m < 5; ++m) B.q[m * M + pb] = Qb[m];
          for (int g = 1; g <= NG; ++g)
            for (int m = 0; m < 5; ++m) B.q[m * M + at(-g)] = Qb[m];
        }
      }
  }
  return 0;
}

// Harness helper (reading U16): dt = CFL / max_interior sum_d ( |k.u| + c |k| ), k = J khat^d.
double Solver::cfl_dt(double cfl) const {
  double mx = 0.0;
  for (const Block& B : blk)
    for (int k = 0; k < B.n[2]; ++k)
      for (int j = 0; j < B.n[1]; ++j)
        for (int i = 0; i < B.n[0]; ++i) {
          const size_t p = B.idx(i, j, k);
          double Q[5];
          for (int m = 0; m < 5; ++m) Q[m] = B.q[m * B.M + p];
          Prim<double> s = prims(Q, prm.gamma);
          double sum = 0.0;
          for (int d = 0; d < 3; ++d) {
            const double kx = B.jac[p] * B.khat[(d * 3 + 0) * B.M + p], ky = B.jac[p] * B.khat[(d * 3 + 1) * B.M + p],
                         kz = B.jac[p] * B.khat[(d * 3 + 2) * B.M + p];
            sum += std::fabs(kx * s.u + ky * s.v + kz * s.w) + s.c * std::sqrt(kx * kx + ky * ky + kz * kz);
          }
          mx = std::max(mx, sum);
        }
  return cfl / mx;
}

}  // namespace orc

// =====================================================================================
// C entry points (ctypes)
// =====================================================================================
using namespace orc;
extern "C" {

void* orc_create(int nblocks, const int* dims, int nfaces, const Face* faces, const Params* p) {
  Solver* s = new Solver();
  if (s->create(nblocks, dims, nfaces, faces, p) != 0) {
    std::fprintf(stderr, "orc_create: %s\n", s->err.c_str());
    delete s;
    return nullptr;
  }
  return s;
}
void orc_destroy(void* h) { delete static_cast<Solver*>(h); }
void orc_set_threads(void* h, int n) { static_cast<Solver*>(h)->nthreads = n < 1 ? 1 : n; }
int orc_max_threads() {
#ifdef _OPENMP
  return omp_get_max_threads();
#else
  return 1;
#endif
}
// field: 0 q, 1 qn, 2 r, 3 xyz, 4 khat, 5 jac
double* orc_field(void* h, int block, int field) {
  Block& B = static_cast<Solver*>(h)->blk[block];
  switch (field) {
    case 0: return B.q.data();
    case 1: return B.qn.data();
    case 2: return B.r.data();
    case 3: return B.xyz.data();
    case 4: return B.khat.data();
    case 5: return B.jac.data();
  }
  return nullptr;
}
const char* orc_last_error(void* h) { return static_cast<Solver*>(h)->err.c_str(); }
int orc_compute_metrics(void* h) { return static_cast<Solver*>(h)->compute_metrics(); }
int orc_rhs(void* h) { return static_cast<Solver*>(h)->rhs(); }
int orc_rk_stage(void* h, int stage, double dt, double* res5) { return static_cast<Solver*>(h)->rk_stage(stage, dt, res5); }
int orc_exchange_interfaces(void* h) { return static_cast<Solver*>(h)->exchange_interfaces(); }
int orc_apply_bc(void* h) { return static_cast<Solver*>(h)->apply_bc(); }
double orc_cfl_dt(void* h, double cfl) { return static_cast<Solver*>(h)->cfl_dt(cfl); }

// ---- per-point routines, exported for the pins -------------------------------------
double orc_d6(const double* a7) { return d6(a7[0], a7[1], a7[2], a7[4], a7[5], a7[6]); }
void orc_weno5(const double* s5, double eps, double* vL, double* vR) { weno5_LR(s5[0], s5[1], s5[2], s5[3], s5[4], eps, *vL, *vR); }
void orc_weno5_beta(const double* s5, double* b3) { weno5_beta(s5[0], s5[1], s5[2], s5[3], s5[4], b3[0], b3[1], b3[2]); }
void orc_eig(const double* Q, const double* n, double gamma, double* L25, double* R25) {
  double L[5][5], R[5][5];
  eig_LR(Q, n, gamma, L, R);
  std::memcpy(L25, L, sizeof(L));
  std::memcpy(R25, R, sizeof(R));
}
void orc_sw_flux(const double* Q, const double* k, double gamma, int sgn, double* F) { sw_flux(Q, k, gamma, sgn, F); }
void orc_point_flux(const double* Q, const double* k, double gamma, double* F) { point_flux(Q, k, gamma, F); }
double orc_khat_half(const double* a6) { return khat_half(a6[0], a6[1], a6[2], a6[3], a6[4], a6[5]); }
// Ql: [5][n+12], kl: [3][n+12], D: [5][n]
void orc_inviscid_line(int n, const double* Ql, const double* kl, double gamma, double eps, int scheme, double* D) {
  const double* q[5]; const double* k[3]; double* d[5];
  for (int m = 0; m < 5; ++m) { q[m] = Ql + m * (n + 2 * NG); d[m] = D + m * n; }
  for (int c = 0; c < 3; ++c) k[c] = kl + c * (n + 2 * NG);
  inviscid_line<double>(n, q, k, gamma, eps, scheme, d);
}
// g: [3][4] (d phi_f / d x_c), vel[3], k[3]
void orc_visc_flux_point(const double* vel, const double* g, const double* k, double mu, double kappa, double* Fv) {
  double gg[3][4];
  std::memcpy(gg, g, sizeof(gg));
  visc_flux_point(vel, gg, k, mu, kappa, Fv);
}
double orc_sutherland_mu(double T, double S) { return sutherland_mu(T, S); }
void orc_grad_point(const double* dphi, const double* kh, double J, double* g) {
  double a[3][4], b[3][3], o[3][4];
  std::memcpy(a, dphi, sizeof(a));
  std::memcpy(b, kh, sizeof(b));
  grad_point(a, b, J, o);
  std::memcpy(g, o, sizeof(o));
}

}  // extern "C"
