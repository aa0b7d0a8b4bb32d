// =====================================================================================
// ORACLE — TEST INFRASTRUCTURE.  Exact algorithmic flop count of one grid point per RK stage
// ("the contract value is the exact count obtained by running the oracle's
// per-point routine with a counting scalar type").  Convention: add, sub, mul, div, sqrt = 1
// each; negation, abs, comparisons, copies and index arithmetic = 0; each point's work is
// counted once (no credit for anything an implementation recomputes redundantly).
// Prints one JSON object.  Built by oracle/build.py; run by tests and quoted in DESIGN.md.
// =====================================================================================
#include "oracle_core.hpp"

#include <cstdio>

namespace cnt {
struct C {
  double v;
  C() : v(0) {}
  C(double x) : v(x) {}
};
static long n_add = 0, n_mul = 0, n_div = 0, n_sqrt = 0;
inline C operator+(const C& a, const C& b) { ++n_add; return C(a.v + b.v); }
inline C operator-(const C& a, const C& b) { ++n_add; return C(a.v - b.v); }
inline C operator*(const C& a, const C& b) { ++n_mul; return C(a.v * b.v); }
inline C operator/(const C& a, const C& b) { ++n_div; return C(a.v / b.v); }
inline C operator-(const C& a) { return C(-a.v); }
inline C sqrt(const C& a) { ++n_sqrt; return C(std::sqrt(a.v)); }
inline C fabs(const C& a) { return C(std::fabs(a.v)); }
struct Snap { long a, m, d, s; long total() const { return a + m + d + s; } };
inline Snap snap() { return Snap{n_add, n_mul, n_div, n_sqrt}; }
inline Snap diff(const Snap& x, const Snap& y) { return Snap{y.a - x.a, y.m - x.m, y.d - x.d, y.s - x.s}; }
}  // namespace cnt

using cnt::C;

static cnt::Snap inviscid_line_cost(int n, int scheme) {
  const int m = n + 2 * orc::NG;
  std::vector<C> Q(5 * m), K(3 * m), D(5 * n);
  for (int i = 0; i < m; ++i) {
    double x = 0.3 * i;
    double rho = 1.0 + 0.1 * std::sin(x), u = 0.3 + 0.1 * std::cos(x), p = 0.7 + 0.05 * std::sin(2 * x);
    Q[0 * m + i] = rho; Q[1 * m + i] = rho * u; Q[2 * m + i] = 0.1 * rho; Q[3 * m + i] = -0.2 * rho;
    Q[4 * m + i] = p / 0.4 + 0.5 * rho * (u * u + 0.05);
    K[0 * m + i] = 1.0 + 0.01 * std::sin(x); K[1 * m + i] = 0.1; K[2 * m + i] = -0.05;
  }
  const C* Ql[5]; const C* kl[3]; C* Dl[5];
  for (int v = 0; v < 5; ++v) { Ql[v] = &Q[v * m]; Dl[v] = &D[v * n]; }
  for (int c = 0; c < 3; ++c) kl[c] = &K[c * m];
  cnt::Snap s0 = cnt::snap();
  orc::inviscid_line<C>(n, Ql, kl, C(1.4), C(1e-6), scheme, Dl);
  return cnt::diff(s0, cnt::snap());
}

static void print(const char* name, const cnt::Snap& s, bool last = false) {
  std::printf("  \"%s\": {\"add\": %ld, \"mul\": %ld, \"div\": %ld, \"sqrt\": %ld, \"total\": %ld}%s\n", name, s.a, s.m,
              s.d, s.s, s.total(), last ? "" : ",");
}

int main() {
  std::printf("{\n");
  cnt::Snap tot_ns{0, 0, 0, 0}, tot_eu{0, 0, 0, 0};
  auto acc = [](cnt::Snap& t, const cnt::Snap& s, long k = 1) { t.a += k * s.a; t.m += k * s.m; t.d += k * s.d; t.s += k * s.s; };
  for (int scheme = 0; scheme < 2; ++scheme) {
    // marginal cost of one more point on a line (removes the two end points' extra work)
    cnt::Snap a = inviscid_line_cost(10, scheme), b = inviscid_line_cost(30, scheme);
    cnt::Snap per{(b.a - a.a) / 20, (b.m - a.m) / 20, (b.d - a.d) / 20, (b.s - a.s) / 20};
    print(scheme == 0 ? "S2_per_direction_modified" : "S2_per_direction_original", per);
    if (scheme == 0) { acc(tot_ns, per, 3); acc(tot_eu, per, 3); }
  }
  // accumulate D^xi + D^eta + D^zeta : 5 adds per direction
  cnt::Snap accD{15, 0, 0, 0};
  acc(tot_ns, accD); acc(tot_eu, accD);
  // ---- viscous, one point ----
  cnt::Snap visc{0, 0, 0, 0};
  {
    C Q[5] = {1.1, 0.3, 0.1, -0.2, 2.0}, phi[4];
    cnt::Snap s0 = cnt::snap();
    orc::phi_point(Q, C(1.4), phi);                       // (u,v,w,T) once per point
    C dphi[3][4];
    for (int d = 0; d < 3; ++d)
      for (int f = 0; f < 4; ++f) dphi[d][f] = orc::d6(C(0.1), C(0.2), C(0.3), C(0.5), C(0.6), C(0.7));  // 12 derivatives
    C kh[3][3] = {{1, .1, .2}, {.1, 1, .3}, {.2, .1, 1}}, g[3][4];
    orc::grad_point(dphi, kh, C(2.0), g);                 // chain rule, Eq. 21
    for (int d = 0; d < 3; ++d) {                         // three point fluxes, Eqs. 5-6
      C Fv[5];
      orc::visc_flux_point(phi, g, kh[d], C(1e-3), C(2e-3), Fv);
    }
    for (int d = 0; d < 3; ++d)                           // derivative of rows 2..5 (row 1 is identically 0)
      for (int m = 1; m < 5; ++m) (void)orc::d6(C(0.1), C(0.2), C(0.3), C(0.5), C(0.6), C(0.7));
    visc = cnt::diff(s0, cnt::snap());
    visc.a += 8;                                          // V^xi + V^eta + V^zeta on 4 rows
  }
  print("S3_viscous", visc);
  acc(tot_ns, visc);
  cnt::Snap fin{5, 5, 0, 0};                              // r = J * (accV - accD)
  acc(tot_ns, fin); acc(tot_eu, fin);
  cnt::Snap rk{10, 15, 0, 0};                             // q = a*qn + b*(q + dt*r), 5 equations
  print("S4_rk_stage", rk);
  acc(tot_ns, rk); acc(tot_eu, rk);
  print("total_navier_stokes_per_point_stage", tot_ns);
  print("total_euler_per_point_stage", tot_eu, true);
  std::printf("}\n");
  return 0;
}
